"""Tidally locked hot-Jupiter benchmark driver (section 7.2): base HE-VI step + NEXT-1 + the
forcing of Eq. 59-61.

    python examples/hot_jupiter_run.py [days] [level] [layers]

The paper's set-up (L529): Table 1's planet, level 5 x 37 layers from 0 to 4875 km, dt = 600 s, D = 0.01992
(Table 1: 941.2 s), isothermal 1600 K in (discrete) hydrostatic balance, at rest.  n = 6 and the surface pressure
1e5 Pa are not printed in the paper.  Prints the zonal-mean zonal wind every 50 Earth days.  Everything runs in
the CUDA library."""
import os
import sys
import time

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import numpy as np
import torch

import paper_1607_05535_b200 as thor
import thor_inputs as ti

PLANET = ti.PAPER_HOT_JUPITER
FORCING = ti.HOT_JUPITER_FORCING


def main():
    days = int(sys.argv[1]) if len(sys.argv) > 1 else 300
    level = int(sys.argv[2]) if len(sys.argv) > 2 else 5
    nv = int(sys.argv[3]) if len(sys.argv) > 3 else 37
    g = thor.Grid(level, nv, PLANET)
    xyz, N = g.view["xyz"], g.n_cols
    rho, _, _, p = ti.rest_state(PLANET, nv, N, 1.0e5, 1600.0)
    stream = torch.cuda.Stream()
    st = thor.State(g, rho, np.zeros((N, nv, 3)), np.zeros((N, nv + 1)), p, cuda_stream=stream.cuda_stream)
    st.set_diffusion(0.01992)
    st.set_hot_jupiter(FORCING)
    dt, n = 600.0, 6
    lat = np.degrees(np.arcsin(xyz[:, 2]))
    lon = np.arctan2(xyz[:, 1], xyz[:, 0])
    east = np.stack([-np.sin(lon), np.cos(lon), np.zeros(N)], axis=-1)
    bins = np.linspace(-90, 90, 37)
    ib = np.clip(np.digitize(lat, bins) - 1, 0, 35)
    m0 = st.diagnostics()[0]
    t0, done = time.time(), 0
    for d in range(50, days + 1, 50):
        nsteps = int(round(d * 86400.0 / dt)) - done
        done += nsteps
        st.step(nsteps, dt, n)
        rho, V, W, p = st.get()
        if not np.all(np.isfinite(p)):
            print("day", d, "not finite")
            break
        u = np.sum(V * east[:, None, :], axis=-1) / rho
        ubar = np.array([[u[ib == b, k].mean() for k in range(nv)] for b in range(36)])
        pbar = p.mean(axis=0)
        kj, bj = np.unravel_index(np.argmax(ubar.T), ubar.T.shape)
        Tk = p / (PLANET["Rd"] * rho)
        print("day %4d  max zonal-mean u %.0f m/s at lat %.0f, p %.0f hPa | min %.0f m/s | equatorial u at that level %.0f | "
              "T %.0f..%.0f K | mass drift %.1e | %.0f s wall" % (d, ubar.max(), 0.5 * (bins[bj] + bins[bj + 1]), pbar[kj] / 100,
                                                                 ubar.min(), ubar[17:19, kj].mean(), Tk.min(), Tk.max(),
                                                                 st.diagnostics()[0] / m0 - 1, time.time() - t0), flush=True)


if __name__ == "__main__":
    main()
