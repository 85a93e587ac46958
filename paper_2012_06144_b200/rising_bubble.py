"""Single rising bubble of section 6.1 on one GPU: set-up from the dimensionless groups, time stepping
with libacm, rise velocity and drag coefficient against the correlation of eq. 35.

    python -m paper_2012_06144_b200.rising_bubble --re 35 --eo 30 [--scale 1.0] [--tstar 10]

Set-up of the paper: 256 x 1024 x 256 cells, bubble of radius 16 at (128, 256, 128), no-slip walls at the top and
bottom (y), periodic otherwise, D3Q19 MRT for both LB steps, rho* = 1000, mu* = 100, t_ref = 18 000, xi = 5,
M = 0.04, run to t* = 10.  `--scale s` shrinks the domain, the bubble and t_ref by s (the groups stay the same).
Prints one JSON line per sample (t*, bubble centroid, rise velocity, Reynolds number of the rise) and a final line
with the terminal velocity, C_D^LBM (eq. 34) and C_D^exp (eq. 35).  Everything numerical runs in the library's
kernels; this module only sets parameters and records diagnostics.
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np
import torch

from . import binding, inputs


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--re", type=float, default=35.0, help="gravity Reynolds number Re_Gr (eq. 31)")
    ap.add_argument("--eo", type=float, default=30.0, help="Eotvos number (eq. 32)")
    ap.add_argument("--scale", type=float, default=1.0, help="1.0 = the paper's 256 x 1024 x 256 with R = 16")
    ap.add_argument("--tstar", type=float, default=10.0, help="run until t/t_ref = tstar (P:407)")
    ap.add_argument("--samples", type=int, default=100)
    ap.add_argument("--mobility", type=float, default=0.04)
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"])
    args = ap.parse_args(argv)

    s = args.scale
    nx, ny, nz = int(round(256 * s)), int(round(1024 * s)), int(round(256 * s))
    R, t_ref = 16.0 * s, 18000.0 * s
    D = 2.0 * R
    q = binding.bubble_params(args.re, args.eo, D, t_ref, 1.0, 1000.0, 100.0)
    p = inputs.Params(nx=nx, ny=ny, nz=nz, stencil_phase=19, stencil_hydro=19, rho_H=1.0, rho_L=q["rho_L"], sigma=q["sigma"],
                      M=args.mobility, nu_H=q["nu_H"], nu_L=q["nu_L"], gravity=(0.0, -q["gy"], 0.0), wall_flags=inputs.WALL_Y)
    phi = inputs.sphere_phi(p, (nx / 2.0, ny / 4.0, nz / 2.0), R, heavy_inside=False)
    dt = np.float64 if args.precision == "f64" else np.float32
    sim = binding.ACM.from_params(p, precision=args.precision)
    sim.init(torch.from_numpy(phi.astype(dt)).cuda(), torch.zeros((3,) + p.shape, dtype=sim.dtype, device="cuda"))
    del phi
    total = int(round(args.tstar * t_ref))
    every = max(1, total // args.samples)
    print(json.dumps({"setup": {"grid": [nx, ny, nz], "R": R, "t_ref": t_ref, "Re_Gr": args.re, "Eo": args.eo, **q,
                                "tau_H": 3 * q["nu_H"], "tau_L": 3 * q["nu_L"], "steps": total}}), flush=True)
    m0 = sim.phi_mass()
    t0 = time.time()
    hist = []
    done = 0
    while done < total:
        n = min(every, total - done)
        sim.step(n)
        done += n
        V, X, U = sim.bubble_diag()
        rec = {"t_star": done / t_ref, "step": done, "y": X[1], "u_y": U[1], "V": V,
               "Re_rise": U[1] * D / q["nu_H"], "mass_drift": sim.phi_mass() / m0 - 1.0}
        hist.append(rec)
        print(json.dumps(rec), flush=True)
        if not np.isfinite(U[1]):
            raise SystemExit("diverged")
    wall = time.time() - t0
    # terminal velocity: mean rise velocity over the last fifth of the run
    tail = [r["u_y"] for r in hist[-max(1, len(hist) // 5):]]
    u_t = float(np.mean(tail))
    out = {"u_t": u_t, "u_t_spread": float(np.max(tail) - np.min(tail)), "C_D_LBM": binding.drag_lbm(q["gy"], 1.0, q["rho_L"], D, u_t),
           "C_D_exp": binding.drag_exp(args.re), "wall_s": wall, "MLUPS": p.ncells * total / wall / 1e6}
    out["ratio"] = out["C_D_LBM"] / out["C_D_exp"]
    print(json.dumps({"result": out}), flush=True)


if __name__ == "__main__":
    main()
