"""Taylor-Green vortex decay with the library (App. E): 2D periodic unit square, n x n particles,
delta-SPH (delta_form 1 = the term of [43] the paper runs, or 0), RK4 with dt = 0.25 H / c0, optional particle shifting
at the end of every step.  Prints KE(t)/KE(0) against the analytic exp(-16 pi^2 nu t) (velocity
amplitude exp(-8 pi^2 nu t), R12) as a markdown table and the effective viscosity fitted on t <= t_fit.

    python -m paper_2507_21684_b200.tgv_decay [--n 128] [--t-end 1.0] [--delta-form 1] [--shift 0.5] [--nu 0.01]

Needs a CUDA device (the library has no CPU fallback).  Input generation: workloads.make(1, n_axis=n) without jitter.
"""
from __future__ import annotations

import argparse
import math

import numpy as np


def run(n=128, t_end=1.0, delta_form=1, shift=0.5, nu=0.01, jitter=0.0, every=0.1, skin=0.08):
    import torch
    from . import workloads as W
    from .binding import Sph

    wl = W.make(0, n_axis=n) if jitter == 0.0 else W.make(1, n_axis=n)
    par = W.Params(**{**wl.params.__dict__, "nu": nu, "delta_form": delta_form, "renorm_rcond": 1e-4})
    dom = W.rk_domain(wl, skin)
    dev = "cuda:0"
    t = lambda a: torch.from_numpy(a).to(dev)
    x, v, rho, m, h, kind = t(wl.x), t(wl.v), t(wl.rho), t(wl.m), t(wl.h), t(wl.kind)
    sph = Sph(0, wl.n)
    ke = lambda: 0.5 * float((m.double()[:, None] * v.double() ** 2).sum())
    ke0 = ke()
    nsteps = int(round(t_end / wl.dt))
    rows = [(0.0, 1.0, 1.0)]
    next_out = every
    for s in range(1, nsteps + 1):
        sph.rk_step(dom, par, wl.dt, skin, x, v, rho, m, h, kind)
        if shift > 0.0:
            sph.shift(shift, x, m, rho, kind)
        tt = s * wl.dt
        if tt + 1e-12 >= next_out or s == nsteps:
            rows.append((tt, ke() / ke0, math.exp(-16.0 * math.pi ** 2 * nu * tt)))
            next_out += every
    sph.check()
    sph.close()
    return rows, wl.dt, nsteps


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=128)
    ap.add_argument("--t-end", type=float, default=1.0)
    ap.add_argument("--delta-form", type=int, default=1)
    ap.add_argument("--shift", type=float, default=0.5, help="shifting coefficient theta (0 = no shifting)")
    ap.add_argument("--nu", type=float, default=0.01)
    ap.add_argument("--t-fit", type=float, default=0.5)
    args = ap.parse_args()
    rows, dt, nsteps = run(args.n, args.t_end, args.delta_form, args.shift, args.nu)
    print(f"Taylor-Green {args.n}x{args.n}, nu = {args.nu}, delta_form = {args.delta_form}, shift theta = {args.shift}, "
          f"dt = {dt:.3e}, {nsteps} RK4 steps")
    print("| t | KE/KE0 | exp(-16 pi^2 nu t) | ratio |")
    print("|---|---|---|---|")
    for tt, k, a in rows:
        print(f"| {tt:.3f} | {k:.5f} | {a:.5f} | {k / a:.4f} |")
    fit = [(tt, k) for tt, k, _ in rows if 0.0 < tt <= args.t_fit + 1e-9 and k > 0]
    if len(fit) >= 2:
        ts, ks = np.array([f[0] for f in fit]), np.array([f[1] for f in fit])
        slope = np.polyfit(ts, np.log(ks), 1)[0]
        nu_eff = -slope / (16.0 * math.pi ** 2)
        print(f"effective viscosity from KE decay on t <= {args.t_fit}: nu_eff = {nu_eff:.5f} (nu = {args.nu}; ratio {nu_eff / args.nu:.3f}); "
              f"Re = U L / nu_eff = {1.0 / nu_eff:.1f} against {1.0 / args.nu:.1f}")


if __name__ == "__main__":
    main()
