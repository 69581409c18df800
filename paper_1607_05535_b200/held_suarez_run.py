"""Held-Suarez benchmark driver (section 7.1): the base HE-VI step + the hyper-diffusion and
divergence damping of section 4 (NEXT-1) + the forcing of Eq. 51-55 from the evolving sigma (NEXT-2).

    python -m paper_1607_05535_b200.held_suarez_run [days] [level] [layers]

Level 5 x 32 layers, dt = 1000 s, n = 6 acoustic substeps, D = 0.004837 (Table 1), rest state at 300 K
with 0.1 K noise, lid at 32 km.  Prints the zonal-mean zonal wind maximum every 50 days.  Everything
runs in the CUDA library; this file only sets the run up and bins the output by latitude."""
import sys
import time

import numpy as np
import torch

import paper_1607_05535_b200 as thor

EARTH = dict(radius=6.371e6, omega=7.292e-5, gravity=9.8, Rd=287.0, Cp=1005.0, p_ref=1.0e5, z_top=32.0e3)
HELD_SUAREZ = dict(T_surf=315.0, dT_y=60.0, dth_z=10.0, T_min=200.0, k_a=1.0 / (40 * 86400.0), k_s=1.0 / (4 * 86400.0),
                   k_f=1.0 / 86400.0, sigma_b=0.7, p_star=1.0e5)


def main():
    days = int(sys.argv[1]) if len(sys.argv) > 1 else 300
    level = int(sys.argv[2]) if len(sys.argv) > 2 else 5
    nv = int(sys.argv[3]) if len(sys.argv) > 3 else 32
    g = thor.Grid(level, nv, EARTH)
    xyz, N = g.view["xyz"], g.n_cols
    # isothermal column in discrete hydrostatic balance, 300 K, p_s = 1e5 Pa, plus 0.1 K noise
    dz = EARTH["z_top"] / nv
    q = EARTH["gravity"] * dz / (2.0 * EARTH["Rd"] * 300.0)
    pcol = np.empty(nv)
    pcol[0] = 1.0e5 * np.exp(-EARTH["gravity"] * 0.5 * dz / (EARTH["Rd"] * 300.0))
    for k in range(1, nv):
        pcol[k] = pcol[k - 1] * (1.0 - q) / (1.0 + q)
    p = np.tile(pcol, (N, 1))
    T = 300.0 + np.random.default_rng(1).uniform(-0.1, 0.1, size=p.shape)
    rho = p / (EARTH["Rd"] * T)
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
