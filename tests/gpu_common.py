"""Helpers for the -m gpu parity tests: move a workload to the device, run the oracle on the same fp32 inputs."""
import numpy as np
import torch

import oracle
from paper_2507_21684_b200 import workloads as W
from paper_2507_21684_b200.binding import Sph


class Dev:
    def __init__(self, wl):
        dev = "cuda:0"
        self.x = torch.from_numpy(wl.x).to(dev)
        self.v = torch.from_numpy(wl.v).to(dev)
        self.rho = torch.from_numpy(wl.rho).to(dev)
        self.m = torch.from_numpy(wl.m).to(dev)
        self.h = torch.from_numpy(wl.h).to(dev)
        self.kind = torch.from_numpy(wl.kind).to(dev)


def build(wl, scale=1.0, sph=None, dev=None):
    sph = sph or Sph(0)
    dev = dev or Dev(wl)
    sph.build_cells(wl.domain, dev.x, dev.h)
    nnz = sph.neighbors(scale)
    return sph, dev, nnz


def oracle_lists(wl, scale=1.0, method=1):
    return oracle.neighbors(wl.domain, wl.x, wl.h, search_scale=scale, method=method)


def fuzz_workload(seed, scale=None, dt_cfl=0.0, tiny=False):
    """seeded random small problem: dimension, periodicity per axis, box aspect, clustered positions (some cells empty),
    uniform or log-normal h, cell size with or without slack, search scale (drawn unless `scale` is given).  dt =
    dt_cfl * min(h) / c0.  Returns (workload, search_scale)."""
    rng = np.random.default_rng(1234 + seed)
    dim = int(rng.integers(2, 4))
    per = tuple(int(rng.integers(0, 2)) for _ in range(dim)) + (0,) * (3 - dim)
    Lbox = rng.uniform(0.6, 1.6, size=dim)
    lo = rng.uniform(-1.0, 1.0, size=dim)
    n = int(rng.integers(300, 3000))
    if tiny:
        n = 1 + n % 40
    hbar = float(rng.uniform(0.08, 0.16)) * float(Lbox.min())
    varh = bool(rng.integers(0, 2))
    h = (hbar * np.exp(rng.normal(0, 0.1, size=n)) if varh else np.full(n, hbar)).astype(np.float32)
    # clustered positions: a mixture of a uniform background and a few blobs, so that some cells are empty
    x = rng.uniform(0.0, 1.0, size=(n, dim))
    nb = n // 2
    centres = rng.uniform(0.2, 0.8, size=(3, dim))
    x[:nb] = centres[rng.integers(0, 3, size=nb)] + rng.normal(0, 0.07, size=(nb, dim))
    x = np.clip(x, 1e-4, 1.0 - 1e-4) * Lbox + lo
    drawn = float(rng.choice([1.0, 1.15]))
    scale = drawn if scale is None else float(scale)
    cell = float(np.float32(h.max()) * np.float32(scale) * np.float32(rng.choice([1.0001, 1.3])))
    lo3 = tuple(lo) + (0.0,) * (3 - dim)
    hi3 = tuple(lo + Lbox) + (0.0,) * (3 - dim)
    if any(per[k] and Lbox[k] / cell < 3.0 for k in range(dim)):
        cell = float(min(Lbox[k] for k in range(dim) if per[k]) / 3.0001)
        h = np.minimum(h, np.float32(cell / scale / 1.0001)).astype(np.float32)
    dom = W.Domain(dim=dim, periodic=per, lo=lo3, hi=hi3, cell_size=cell)
    base = W.make(3 if dim == 3 else 0, **(dict(n_axis=8) if dim == 3 else {})).params
    par = W.Params(**{**base.__dict__, "alpha": 0.02, "g": (0.1, -0.2, 0.05)})
    wl = W.Workload(name=f"fuzz{seed}", domain=dom, params=par, x=x.astype(np.float32),
                    v=rng.normal(0, 0.3, size=(n, dim)).astype(np.float32),
                    rho=(1.0 + 0.03 * rng.normal(size=n)).astype(np.float32),
                    m=(np.full(n, 1.0 / n) * np.exp(rng.normal(0, 0.05, size=n))).astype(np.float32), h=h,
                    kind=(rng.uniform(size=n) < 0.05).astype(np.uint8), dt=dt_cfl * float(h.min()) / par.c0, dx=0.05,
                    seed=seed)
    return wl, scale


def renorm_errors(L_gpu, grad_gpu, L_o, grad_o, M_o, rcond):
    """Per-row errors of the renormalisation outputs against the oracle, for the rows where the comparison is meaningful.
    The pseudo-inverse takes a rank decision (eigenvalue against rcond * largest): rows with an eigenvalue within a
    factor 3 of the cutoff are left out (fp32 and fp64 may decide differently there; both results are valid).
    What fp32 bounds is the ABSOLUTE error of the sums M_i, b_i, about 1e-6 of the size a full neighbourhood gives
    them (as for drho/dt, reading R10: sums are judged against the size of the summed terms).  The inverse turns it
    into a relative error dL/|L| ~ dM / lambda_min, so a row is measured against its own size times
        amp_i = max(1, s_i / (50 lambda_min_i)),   s_i = max(lambda_max_i, half the median lambda_max),
    i.e. the plain bar for rows with condition number <= 50 and a typical M; a row whose few neighbours all sit at the
    very edge of the support (M_i orders of magnitude below typical, (1-q)^5 cancelling in fp32) is relaxed in
    proportion.  Returns (err_L, err_grad, rows compared)."""
    lam = np.abs(np.linalg.eigvalsh(M_o))
    lmax = np.maximum(lam.max(axis=1), 1e-300)
    ratio = lam / lmax[:, None]
    near = np.any((ratio > rcond / 3.0) & (ratio < rcond * 3.0), axis=1)
    lmin = np.where(ratio > rcond, lam, np.inf).min(axis=1)                # smallest retained eigenvalue
    s_i = np.maximum(lmax, 0.5 * np.median(lmax))
    amp = np.maximum(1.0, s_i / (50.0 * lmin))          # rows without a retained eigenvalue (L = 0 exactly): amp = 1
    ok = ~near
    sL = np.abs(L_o).reshape(len(L_o), -1).max(axis=1)
    sL = np.maximum(np.maximum(sL, np.median(sL)), 1e-300)
    eL = np.abs(L_gpu.astype(np.float64) - L_o).reshape(len(L_o), -1).max(axis=1) / (sL * amp)
    sg = np.maximum(np.maximum(np.abs(grad_o).max(axis=1), np.median(np.abs(grad_o).max(axis=1))), 1e-300)
    eg = np.abs(grad_gpu.astype(np.float64) - grad_o).max(axis=1) / (sg * amp)
    return float(eL[ok].max()), float(eg[ok].max()), int(ok.sum())


def renorm_good_rows(M_o, rcond):
    """rows on which the renormalisation is well-posed in fp32: no eigenvalue within a factor 3 of the rank cutoff,
    condition number of the retained part <= 50, and M_i not orders of magnitude below the typical one (see
    renorm_errors).  The adjoint tests put their cotangent on these rows only."""
    lam = np.abs(np.linalg.eigvalsh(M_o))
    lmax = np.maximum(lam.max(axis=1), 1e-300)
    ratio = lam / lmax[:, None]
    near = np.any((ratio > rcond / 3.0) & (ratio < rcond * 3.0), axis=1)
    lmin = np.where(ratio > rcond, lam, np.inf).min(axis=1)
    return (~near) & (lmax / lmin <= 50.0) & (lmax >= 1e-2 * np.median(lmax))
