"""Held-Suarez benchmark driver (section 7.1): the base HE-VI step + the hyper-diffusion and
divergence damping of section 4 (NEXT-1) + the forcing of Eq. 51-55 from the evolving sigma (NEXT-2).

    python examples/held_suarez_run.py [days] [level] [layers]

The paper's set-up (L452-L454): level 5 x 37 layers from 0 to 32 km, dt = 1000 s, D = 0.004837 (Table 1: 6.46e3 s),
at rest, every column with the temperature profile of T_eq at the equator in (discrete) hydrostatic balance.
n = 6 acoustic substeps (L252's example) and p_s = 1e5 Pa are not printed for this run.  Prints the zonal-mean
zonal wind maximum every 50 days.  Everything runs in the CUDA library; this file only sets the run up and bins
the output by latitude."""
import os
import sys
import time

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

import numpy as np
import torch

import paper_1607_05535_b200 as thor
import thor_inputs as ti

EARTH = dict(ti.EARTH, z_top=32.0e3)
HELD_SUAREZ = ti.HELD_SUAREZ


def main():
    days = int(sys.argv[1]) if len(sys.argv) > 1 else 300
    level = int(sys.argv[2]) if len(sys.argv) > 2 else 5
    nv = int(sys.argv[3]) if len(sys.argv) > 3 else 37
    g = thor.Grid(level, nv, EARTH)
    xyz, N = g.view["xyz"], g.n_cols
    # L452: the equatorial T_eq profile in discrete hydrostatic balance, the same in every column, at rest
    _, _, z_h = ti.vertical_grid(EARTH, nv)
    pcol, Tcol = ti.benchmark_column(EARTH, z_h, 1.0e5, ti.held_suarez_equator_profile(EARTH, HELD_SUAREZ))
    p = np.tile(pcol, (N, 1))
    rho = p / (EARTH["Rd"] * np.tile(Tcol, (N, 1)))
    stream = torch.cuda.Stream()
    st = thor.State(g, rho, np.zeros((N, nv, 3)), np.zeros((N, nv + 1)), p, cuda_stream=stream.cuda_stream)
    st.set_diffusion(0.004837)
    st.set_held_suarez(HELD_SUAREZ)
    dt, n = 1000.0, 6
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
        Tk = p / (EARTH["Rd"] * rho)
        print("day %4d  max zonal-mean u %.1f m/s at lat %.0f, p %.0f hPa | equatorial surface u %.1f | T %.0f..%.0f K | "
              "mass drift %.1e | %.0f s wall" % (d, ubar.max(), 0.5 * (bins[bj] + bins[bj + 1]), pbar[kj] / 100,
                                               ubar[17:19, 0].mean(), Tk.min(), Tk.max(), st.diagnostics()[0] / m0 - 1,
                                               time.time() - t0), flush=True)


if __name__ == "__main__":
    main()
