"""ctypes front-end of the fp64 CPU oracle (oracle/sph_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package.  It imports nothing from the
CUDA package.  Argument marshalling only -- all arithmetic is in sph_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import numpy as np

from .build import build as _build

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.orc_w.restype = C.c_double
        _lib.orc_w.argtypes = [C.c_double, C.c_double, C.c_int]
        _lib.orc_gfac.restype = C.c_double
        _lib.orc_gfac.argtypes = [C.c_double, C.c_double, C.c_int]
        _lib.orc_kfac.restype = C.c_double
        _lib.orc_kfac.argtypes = [C.c_double, C.c_double, C.c_int]
        _lib.orc_neighbors.restype = C.c_int64
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None else None


def _dom(domain):
    per = np.ascontiguousarray(list(domain.periodic)[:3] + [0] * (3 - len(domain.periodic)), dtype=np.int32)
    lo = _d(list(domain.lo)[:3] + [0.0] * (3 - len(domain.lo)))
    hi = _d(list(domain.hi)[:3] + [0.0] * (3 - len(domain.hi)))
    # the C ABI carries lo/hi as binary32
    lo = lo.astype(np.float32).astype(np.float64)
    hi = hi.astype(np.float32).astype(np.float64)
    return int(domain.dim), per, lo, hi


def _par(params):
    # the C ABI carries the scalars as binary32
    vals = np.asarray(params.as_list(), dtype=np.float32).astype(np.float64)
    return _d(list(vals) + [float(params.pressure_form)])


def _par_raw(values, form=0):
    """parameters given directly as 10 doubles (for finite differences in the scalars)"""
    return _d(list(values) + [float(form)])


def w(r, H, dim):
    return lib().orc_w(float(r), float(H), int(dim))


def gfac(r, H, dim):
    return lib().orc_gfac(float(r), float(H), int(dim))


def kfac(r, H, dim):
    return lib().orc_kfac(float(r), float(H), int(dim))


def num_threads():
    return int(lib().orc_num_threads())


def wrap32(domain, x):
    dim, per, lo, hi = _dom(domain)
    x = _d(x)
    n = x.shape[0]
    xw = np.empty_like(x)
    bad = C.c_int64(0)
    lib().orc_wrap32(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(x), _p(xw), C.byref(bad))
    return xw, int(bad.value)


def neighbors(domain, x, h, search_scale=1.0, method=0, prewrapped=False):
    """CSR neighbour lists (row_ptr int64 [n+1], col_idx int32 [nnz], rows ascending, self included)
    of the binary32 positions ``x``.  method 0 = brute force, 1 = oracle grid."""
    dim, per, lo, hi = _dom(domain)
    if prewrapped:
        xw = _d(x)
    else:
        xw, _ = wrap32(domain, np.asarray(x, dtype=np.float32))
    h = _d(np.asarray(h, dtype=np.float32))
    n = xw.shape[0]
    row_ptr = np.zeros(n + 1, dtype=np.int64)
    args = [C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(xw), _p(h), C.c_double(float(np.float32(search_scale))),
            C.c_int(method), _p(row_ptr)]
    nnz = lib().orc_neighbors(*args, None)
    if nnz < 0:
        raise MemoryError("oracle neighbour search")
    col = np.empty(max(int(nnz), 1), dtype=np.int32)
    lib().orc_neighbors(*args, _p(col))
    return row_ptr, col[:nnz]


def density(domain, x, h, m, row_ptr, col_idx):
    dim, per, lo, hi = _dom(domain)
    x, h, m = _d(x), _d(h), _d(m)
    n = x.shape[0]
    rho = np.empty(n, dtype=np.float64)
    lib().orc_density(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(x), _p(h), _p(m),
                      _p(np.ascontiguousarray(row_ptr, np.int64)), _p(np.ascontiguousarray(col_idx, np.int32)), _p(rho))
    return rho


def max_displacement(domain, x, x_build):
    """largest minimum-image displacement of a particle since the positions of the neighbour query"""
    dim, per, lo, hi = _dom(domain)
    x, xb = _d(x), _d(x_build)
    f = lib().orc_max_displacement
    f.restype = C.c_double
    return float(f(C.c_int64(x.shape[0]), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(x), _p(xb)))


def grad_sum(domain, x, h, a, row_ptr, col_idx):
    """g_i = sum_j a_j grad_i W_ij (the gradient term of PAPER.md:379 Eq.24 with a = m/rho)"""
    dim, per, lo, hi = _dom(domain)
    x, h, a = _d(x), _d(h), _d(a)
    n = x.shape[0]
    g = np.empty((n, dim), dtype=np.float64)
    lib().orc_grad_sum(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(x), _p(h), _p(a),
                       _p(np.ascontiguousarray(row_ptr, np.int64)), _p(np.ascontiguousarray(col_idx, np.int32)), _p(g))
    return g


def shift(domain, x, h, m, rho, kind, theta, row_ptr, col_idx):
    """Particle shifting at the end of a step (reading R18, Fickian form):
    x_i <- x_i - theta l_i^2 sum_j (m_j/rho_j) grad_i W_ij for fluid kinds, l = h/kappa_d."""
    dim = int(domain.dim)
    kap = 2.171239 if dim == 2 else 2.207940
    g = grad_sum(domain, x, h, _d(m) / _d(rho), row_ptr, col_idx)
    ell = _d(np.asarray(h, dtype=np.float32)) / kap
    out = _d(x).copy()
    fluid = np.asarray(kind) == 0
    out[fluid] -= theta * (ell[fluid] ** 2)[:, None] * g[fluid]
    return out


def grad_sum_vjp(domain, x, h, a, row_ptr, col_idx, g_bar):
    """(x_bar, a_bar) = J^T g_bar of grad_sum() with the adjacency held fixed"""
    dim, per, lo, hi = _dom(domain)
    x, h, a, gb = _d(x), _d(h), _d(a), _d(g_bar)
    n = x.shape[0]
    xb = np.empty((n, dim), dtype=np.float64)
    ab = np.empty(n, dtype=np.float64)
    lib().orc_grad_sum_vjp(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(x), _p(h), _p(a),
                           _p(np.ascontiguousarray(row_ptr, np.int64)), _p(np.ascontiguousarray(col_idx, np.int32)),
                           _p(gb), _p(xb), _p(ab))
    return xb, ab


def density_vjp(domain, x, h, m, row_ptr, col_idx, rho_bar):
    """(x_bar, m_bar) = J^T rho_bar of density() with the adjacency held fixed (Eq.21)"""
    dim, per, lo, hi = _dom(domain)
    x, h, m, rb = _d(x), _d(h), _d(m), _d(rho_bar)
    n = x.shape[0]
    xb = np.empty((n, dim), dtype=np.float64)
    mb = np.empty(n, dtype=np.float64)
    lib().orc_density_vjp(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(x), _p(h), _p(m),
                          _p(np.ascontiguousarray(row_ptr, np.int64)), _p(np.ascontiguousarray(col_idx, np.int32)),
                          _p(rb), _p(xb), _p(mb))
    return xb, mb


def renorm_gradient(domain, x, h, vol, A, row_ptr, col_idx, rcond=1e-4):
    """Kernel renormalisation (Eq.44, Eq.45): L_i = [sum_j V_j (x_j - x_i) (x) grad_i W_ij]^+ and the
    corrected gradient <grad A>_i = sum_j V_j (A_j - A_i) L_i grad_i W_ij.  The pseudo-inverse is the Moore-Penrose
    inverse with eigenvalues below rcond * (largest |eigenvalue|) dropped (numpy.linalg.pinv; the matrix is symmetric
    because grad W is parallel to x_i - x_j).  Returns (L [n,d,d], grad [n,d], M [n,d,d])."""
    dim, per, lo, hi = _dom(domain)
    x, h, vol, A = _d(x), _d(h), _d(vol), _d(A)
    n = x.shape[0]
    M = np.empty((n, dim, dim), dtype=np.float64)
    b = np.empty((n, dim), dtype=np.float64)
    lib().orc_renorm_moments(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(x), _p(h), _p(vol), _p(A),
                             _p(np.ascontiguousarray(row_ptr, np.int64)), _p(np.ascontiguousarray(col_idx, np.int32)),
                             _p(M), _p(b))
    L = np.linalg.pinv(M, rcond=rcond, hermitian=True)
    grad = np.einsum("nkl,nl->nk", L, b)
    return L, grad, M


def renorm_gradient_vjp(domain, x, h, vol, A, row_ptr, col_idx, grad_bar, rcond=1e-4):
    """(x_bar, vol_bar, A_bar) = J^T grad_bar of the corrected gradient of renorm_gradient(), adjacency fixed.
    Per particle, with g = L b, L = M^+ (symmetric), P = M L the projector on the range of M:
        b_bar = L g_bar,   L_bar = g_bar b^T,
        M_bar = -L L_bar L + (I - P) L_bar L L        (differential of the pseudo-inverse at constant rank,
              = -b_bar g^T + ((I - P) g_bar) (L g)^T    Golub & Pereyra 1973; the third term of that formula
                                                         vanishes because b lies in the range of M)
    then the pair terms by orc_renorm_moments_vjp."""
    dim, per, lo, hi = _dom(domain)
    x, h, vol, A, gb = _d(x), _d(h), _d(vol), _d(A), _d(grad_bar)
    n = x.shape[0]
    rp = np.ascontiguousarray(row_ptr, np.int64)
    ci = np.ascontiguousarray(col_idx, np.int32)
    L, g, M = renorm_gradient(domain, x, h, vol, A, rp, ci, rcond=rcond)
    bbar = np.einsum("nkl,nl->nk", L, gb)
    P = np.einsum("nkl,nlm->nkm", M, L)
    c = gb - np.einsum("nkl,nl->nk", P, gb)
    u = np.einsum("nkl,nl->nk", L, g)
    Mbar = -np.einsum("nk,nl->nkl", bbar, g) + np.einsum("nk,nl->nkl", c, u)
    Mbar = np.ascontiguousarray(Mbar)
    bbar = np.ascontiguousarray(bbar)
    xb = np.empty((n, dim), dtype=np.float64)
    vb = np.empty(n, dtype=np.float64)
    ab = np.empty(n, dtype=np.float64)
    lib().orc_renorm_moments_vjp(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(x), _p(h), _p(vol), _p(A),
                                 _p(rp), _p(ci), _p(Mbar), _p(bbar), _p(xb), _p(vb), _p(ab))
    return xb, vb, ab


def _delta_form(params, delta_form):
    if delta_form is not None:
        return int(delta_form)
    return int(getattr(params, "delta_form", 0)) if params is not None else 0


def _rcond(params, rcond):
    if rcond is not None:
        return float(rcond)
    return float(getattr(params, "renorm_rcond", 1e-4)) if params is not None else 1e-4


def rhs(domain, params, x, v, rho, m, h, kind, row_ptr, col_idx, rows=None, with_scales=False, par_raw=None,
        delta_form=None, rcond=None):
    """drho/dt and acceleration.  delta_form 1 (params.delta_form or the argument): the delta-term of
    [43] with the renormalised density gradient -- orc_rhs's Molteni-Colagrossi term plus orc_delta_renorm_term, with
    <grad rho>^L from renorm_gradient(vol = m/rho, A = rho)."""
    dim, per, lo, hi = _dom(domain)
    par = _par(params) if par_raw is None else par_raw
    x, v, rho, m, h = _d(x), _d(v), _d(rho), _d(m), _d(h)
    kind = np.ascontiguousarray(kind, dtype=np.uint8)
    n = x.shape[0]
    drho = np.zeros(n)
    acc = np.zeros((n, dim))
    dform = _delta_form(params, delta_form)
    sd = np.zeros(n) if (with_scales or dform) else None
    sa = np.zeros(n) if with_scales else None
    rp = np.ascontiguousarray(row_ptr, np.int64)
    ci = np.ascontiguousarray(col_idx, np.int32)
    rows_a = None if rows is None else np.ascontiguousarray(rows, np.int64)
    lib().orc_rhs(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(par), _p(x), _p(v), _p(rho), _p(m), _p(h),
                  _p(kind), _p(rp), _p(ci), _p(rows_a), C.c_int64(0 if rows is None else len(rows_a)),
                  _p(drho), _p(acc), _p(sd), _p(sa))
    if dform == 1:
        _, g, _ = renorm_gradient(domain, x, h, m / rho, rho, rp, ci, rcond=_rcond(params, rcond))
        g = np.ascontiguousarray(g)
        lib().orc_delta_renorm_term(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(par), _p(x), _p(rho), _p(m),
                                    _p(h), _p(rp), _p(ci), _p(g), _p(rows_a), C.c_int64(0 if rows is None else len(rows_a)),
                                    _p(drho), _p(sd))
    if with_scales:
        return drho, acc, sd, sa
    return drho, acc


def rhs_vjp(domain, params, x, v, rho, m, h, kind, row_ptr, col_idx, drho_bar, acc_bar, rows=None, par_raw=None,
            delta_form=None, rcond=None):
    """(x_bar, v_bar, rho_bar, params_bar) = J^T (drho_bar, acc_bar) of rhs(), adjacency held fixed.  delta_form 1 adds the
    adjoint of orc_delta_renorm_term: its direct dependences (orc_delta_renorm_term_vjp) and, through the cotangent of
    the gradient field, the adjoint of the renormalised gradient with vol = m/rho and A = rho (full rows only)."""
    dim, per, lo, hi = _dom(domain)
    par = _par(params) if par_raw is None else par_raw
    x, v, rho, m, h = _d(x), _d(v), _d(rho), _d(m), _d(h)
    lam, mu = _d(drho_bar), _d(acc_bar)
    kind = np.ascontiguousarray(kind, dtype=np.uint8)
    n = x.shape[0]
    xb = np.zeros((n, dim))
    vb = np.zeros((n, dim))
    rb = np.zeros(n)
    pb = np.zeros(10)
    rp = np.ascontiguousarray(row_ptr, np.int64)
    ci = np.ascontiguousarray(col_idx, np.int32)
    rows_a = None if rows is None else np.ascontiguousarray(rows, np.int64)
    lib().orc_rhs_vjp(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(par), _p(x), _p(v), _p(rho), _p(m), _p(h),
                      _p(kind), _p(rp), _p(ci), _p(lam), _p(mu), _p(rows_a), C.c_int64(0 if rows is None else len(rows_a)),
                      _p(xb), _p(vb), _p(rb), _p(pb))
    if _delta_form(params, delta_form) == 1:
        if rows is not None:
            raise ValueError("delta_form 1: the adjoint is computed for all rows")
        rc = _rcond(params, rcond)
        vol = m / rho
        _, g, _ = renorm_gradient(domain, x, h, vol, rho, rp, ci, rcond=rc)
        g = np.ascontiguousarray(g)
        gbar = np.zeros((n, dim))
        lib().orc_delta_renorm_term_vjp(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(par), _p(x), _p(rho),
                                        _p(m), _p(h), _p(rp), _p(ci), _p(g), _p(lam), _p(xb), _p(rb), _p(gbar), _p(pb))
        xb2, volb, Ab = renorm_gradient_vjp(domain, x, h, vol, rho, rp, ci, gbar, rcond=rc)
        xb += xb2
        rb += Ab - volb * m / (rho * rho)                 # A = rho;  vol = m / rho
    return xb, vb, rb, pb


def _wrap64(domain, x):
    """binary64 wrap of stage positions into the periodic box (same formula as wrap64 in sph_oracle.c)"""
    dim, per, lo, hi = _dom(domain)
    xw = _d(x).copy()
    for k in range(dim):
        if per[k]:
            Lk = float(np.float32(hi[k]) - np.float32(lo[k]))       # the one binary32 L of readings R3/R4
            xw[:, k] = xw[:, k] - Lk * np.floor((xw[:, k] - lo[k]) / Lk)
            xw[xw[:, k] >= hi[k], k] -= Lk
            xw[xw[:, k] < lo[k], k] += Lk
    return xw


def _f_eval(domain, params, X, V, R, m, h, kind, method, par_raw):
    """k = f(Y) with exact neighbours of the stage positions; returns (kx, kv, kr, lists)"""
    lists = neighbors(domain, _wrap64(domain, X), h, method=method, prewrapped=True)
    kr, kv = rhs(domain, params, X, V, R, m, h, kind, *lists, par_raw=par_raw)
    kx = np.where(np.asarray(kind)[:, None] != 0, 0.0, V)
    return kx, kv, kr, lists


def _rk4_step_py(domain, params, dt, x, v, rho, m, h, kind, method, par_raw):
    """classic RK4 written out in Python on top of rhs() -- used for delta_form 1, whose right-hand side is composed in
    this module"""
    c = (0.0, 0.5, 0.5, 1.0)
    b = (1.0 / 6.0, 1.0 / 3.0, 1.0 / 3.0, 1.0 / 6.0)
    x, v, rho = _d(x), _d(v), _d(rho)
    ax, av, ar = np.zeros_like(x), np.zeros_like(v), np.zeros_like(rho)
    kx = kv = kr = None
    for s in range(4):
        X = x if s == 0 else x + c[s] * dt * kx
        V = v if s == 0 else v + c[s] * dt * kv
        R = rho if s == 0 else rho + c[s] * dt * kr
        kx, kv, kr, _ = _f_eval(domain, params, X, V, R, m, h, kind, method, par_raw)
        ax, av, ar = ax + b[s] * kx, av + b[s] * kv, ar + b[s] * kr
    return x + dt * ax, v + dt * av, rho + dt * ar


def _rk4_step_vjp_py(domain, params, dt, x0, v0, r0, m, h, kind, xb, vb, rb, pb, method, par_raw):
    """discrete adjoint of _rk4_step_py with recomputed stages"""
    c = (0.0, 0.5, 0.5, 1.0)
    b = (1.0 / 6.0, 1.0 / 3.0, 1.0 / 3.0, 1.0 / 6.0)
    x0, v0, r0 = _d(x0), _d(v0), _d(r0)
    Y, lists = [], []
    kx = kv = kr = None
    for s in range(4):
        X = x0 if s == 0 else x0 + c[s] * dt * kx
        V = v0 if s == 0 else v0 + c[s] * dt * kv
        R = r0 if s == 0 else r0 + c[s] * dt * kr
        Y.append((X, V, R))
        kx, kv, kr, l = _f_eval(domain, params, X, V, R, m, h, kind, method, par_raw)
        lists.append(l)
    fluid = (np.asarray(kind) == 0)[:, None]
    Ybx, Ybv, Ybr = np.zeros_like(x0), np.zeros_like(v0), np.zeros_like(r0)
    sx, sv, sr = np.zeros_like(x0), np.zeros_like(v0), np.zeros_like(r0)
    for s in (3, 2, 1, 0):
        a_next = 0.0 if s == 3 else c[s + 1]
        kbx = b[s] * dt * xb + a_next * dt * Ybx
        kbv = b[s] * dt * vb + a_next * dt * Ybv
        kbr = b[s] * dt * rb + a_next * dt * Ybr
        Ybx, Ybv, Ybr, pk = rhs_vjp(domain, params, *Y[s], m, h, kind, *lists[s], kbr, kbv, par_raw=par_raw)
        Ybv = Ybv + np.where(fluid, kbx, 0.0)             # dx/dt = v for fluid kinds
        sx, sv, sr = sx + Ybx, sv + Ybv, sr + Ybr
        pb = pb + pk
    return xb + sx, vb + sv, rb + sr, pb


def rk4_step(domain, params, dt, x, v, rho, m, h, kind, method=0, par_raw=None):
    if _delta_form(params, None) == 1:
        return _rk4_step_py(domain, params, dt, x, v, rho, m, h, kind, method, par_raw)
    dim, per, lo, hi = _dom(domain)
    par = _par(params) if par_raw is None else par_raw
    x, v, rho = _d(x).copy(), _d(v).copy(), _d(rho).copy()
    m, h = _d(m), _d(h)
    kind = np.ascontiguousarray(kind, dtype=np.uint8)
    n = x.shape[0]
    lib().orc_rk4_step(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(par), C.c_double(dt),
                       _p(x), _p(v), _p(rho), _p(m), _p(h), _p(kind), C.c_int(method))
    return x, v, rho


def rk4_step_vjp(domain, params, dt, x0, v0, rho0, m, h, kind, x_bar, v_bar, rho_bar, params_bar=None, method=0,
                 par_raw=None):
    if _delta_form(params, None) == 1:
        pb0 = np.zeros(10) if params_bar is None else _d(params_bar).copy()
        return _rk4_step_vjp_py(domain, params, dt, x0, v0, rho0, m, h, kind, _d(x_bar).copy(), _d(v_bar).copy(),
                                _d(rho_bar).copy(), pb0, method, par_raw)
    dim, per, lo, hi = _dom(domain)
    par = _par(params) if par_raw is None else par_raw
    x0, v0, rho0, m, h = _d(x0), _d(v0), _d(rho0), _d(m), _d(h)
    xb, vb, rb = _d(x_bar).copy(), _d(v_bar).copy(), _d(rho_bar).copy()
    pb = np.zeros(10) if params_bar is None else _d(params_bar).copy()
    kind = np.ascontiguousarray(kind, dtype=np.uint8)
    n = x0.shape[0]
    lib().orc_rk4_step_vjp(C.c_int64(n), C.c_int(dim), _p(per), _p(lo), _p(hi), _p(par), C.c_double(dt),
                           _p(x0), _p(v0), _p(rho0), _p(m), _p(h), _p(kind), C.c_int(method),
                           _p(xb), _p(vb), _p(rb), _p(pb))
    return xb, vb, rb, pb
