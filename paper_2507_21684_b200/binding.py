"""Thin ctypes binding of the C ABI in include/sph.h (argument marshalling only).

PyTorch is used for device memory and streams; every step of the path runs in the CUDA library
``libsph_b200.so`` built from ``csrc/``.  There is no CPU fallback: if the library is missing, cannot be
loaded, or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libsph_b200.so")

EXPORTS = ("sph_create", "sph_destroy", "sph_build_cells", "sph_neighbors", "sph_neighbors_export", "sph_density",
           "sph_density_vjp", "sph_lists_valid", "sph_grad_sum", "sph_grad_sum_vjp", "sph_renorm_gradient", "sph_renorm_gradient_vjp",
           "sph_rhs", "sph_rhs_vjp", "sph_rk_step", "sph_rk_step_vjp", "sph_forward_backward_host", "sph_step_host",
           "sph_check", "sph_debug_bounds_violations", "sph_strerror", "sph_get_info", "sph_get_layout", "sph_profile_enable", "sph_profile_read",
           "sph_set_option", "sph_shift", "sph_prefix_sum_noalloc")

# keys of sph_set_option (enum SPH_OPT_* in include/sph.h)
OPT_PAIR_GROUP, OPT_LIST_MODE, OPT_TILE_EDGE, OPT_PAIR_WARPS, OPT_FILL_MASKS, OPT_RK_EXTRA_SKIN = 1, 2, 3, 4, 5, 6
OPT_UNIFORM_MASS_PATH, OPT_BUILD_FUSED, OPT_STAGE_BULK, OPT_VJP_SPLIT, OPT_TILE_TABLES = 7, 8, 9, 10, 11
LIST_AUTO, LIST_GENERIC, LIST_TILE = 0, 1, 2

# kernel classes of sph_profile_read (enum SPH_K_* in include/sph.h)
KERNEL_CLASSES = ("key", "sort", "reorder", "count", "scan", "fill", "export", "density", "pack", "rhs", "vjp",
                  "reduce", "rk")


class SphDomain(C.Structure):
    _fields_ = [("dim", C.c_int), ("periodic", C.c_int * 3), ("lo", C.c_float * 3), ("hi", C.c_float * 3),
                ("cell_size", C.c_float)]


class SphParams(C.Structure):
    _fields_ = [("c0", C.c_float), ("rho0", C.c_float), ("gamma", C.c_float), ("delta", C.c_float),
                ("alpha", C.c_float), ("nu", C.c_float), ("eps", C.c_float), ("g", C.c_float * 3),
                ("pressure_form", C.c_int), ("delta_form", C.c_int), ("renorm_rcond", C.c_float)]


class SphError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"sph error {code}: {msg}")
        self.code = code


_lib = None


def load_library(path: str = LIB_PATH):
    """dlopen the CUDA library.  Raises if it has not been built (python -m paper_2507_21684_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(path):
        raise FileNotFoundError(f"{path} is missing: build it with `python -m paper_2507_21684_b200.build` "
                                "(there is no CPU fallback)")
    lib = C.CDLL(path)
    vp, i64, f32 = C.c_void_p, C.c_int64, C.c_float
    lib.sph_create.argtypes = [C.POINTER(vp), C.c_int, i64]
    lib.sph_destroy.argtypes = [vp]
    lib.sph_build_cells.argtypes = [vp, C.POINTER(SphDomain), vp, vp, i64, vp]
    lib.sph_neighbors.argtypes = [vp, f32, C.POINTER(i64), vp]
    lib.sph_neighbors_export.argtypes = [vp, vp, vp, vp]
    lib.sph_density.argtypes = [vp, vp, vp, vp]
    lib.sph_density_vjp.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.sph_grad_sum.argtypes = [vp, vp, vp, vp]
    lib.sph_grad_sum_vjp.argtypes = [vp, vp, vp, vp, vp, vp]
    lib.sph_renorm_gradient.argtypes = [vp, vp, vp, C.c_float, vp, vp, vp]
    lib.sph_renorm_gradient_vjp.argtypes = [vp, vp, vp, C.c_float, vp, vp, vp, vp, vp]
    lib.sph_shift.argtypes = [vp, f32, vp, vp, vp, vp, vp]
    lib.sph_lists_valid.argtypes = [vp, vp, f32, C.POINTER(C.c_int32), C.POINTER(f32), vp]
    lib.sph_rhs.argtypes = [vp, C.POINTER(SphParams)] + [vp] * 7 + [vp]
    lib.sph_rhs_vjp.argtypes = [vp, C.POINTER(SphParams)] + [vp] * 11 + [vp]
    lib.sph_rk_step.argtypes = [vp, C.POINTER(SphDomain), C.POINTER(SphParams), f32, f32, i64] + [vp] * 6 + [vp]
    lib.sph_rk_step_vjp.argtypes = [vp, C.POINTER(SphDomain), C.POINTER(SphParams), f32, f32, i64] + [vp] * 10 + [vp]
    lib.sph_forward_backward_host.argtypes = [vp, C.POINTER(SphDomain), C.POINTER(SphParams), f32, i64] + [vp] * 14 + \
                                             [C.POINTER(i64)]
    lib.sph_step_host.argtypes = [vp, C.POINTER(SphDomain), C.POINTER(SphDomain), C.POINTER(SphParams), f32, f32, i64] + \
                                 [vp] * 15 + [C.POINTER(i64)]
    lib.sph_profile_enable.argtypes = [vp, C.c_int]
    lib.sph_set_option.argtypes = [vp, C.c_int, C.c_int]
    lib.sph_profile_read.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(i64)]
    lib.sph_check.argtypes = [vp]
    lib.sph_prefix_sum_noalloc.argtypes = [C.c_int, vp, vp, i64, vp]
    lib.sph_debug_bounds_violations.argtypes = [vp, C.POINTER(C.c_int64)]
    lib.sph_strerror.argtypes = [C.c_int]
    lib.sph_strerror.restype = C.c_char_p
    lib.sph_get_info.argtypes = [vp, C.POINTER(C.c_int32 * 3), C.POINTER(i64), C.POINTER(i64), C.POINTER(i64)]
    lib.sph_get_layout.argtypes = [vp, C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(i64), C.POINTER(i64)]
    for name in EXPORTS:
        if name != "sph_strerror":
            getattr(lib, name).restype = C.c_int
    _lib = lib
    return lib


def make_domain(domain) -> SphDomain:
    d = SphDomain()
    d.dim = int(domain.dim)
    for k in range(3):
        d.periodic[k] = int(domain.periodic[k]) if k < len(domain.periodic) else 0
        d.lo[k] = float(domain.lo[k]) if k < len(domain.lo) else 0.0
        d.hi[k] = float(domain.hi[k]) if k < len(domain.hi) else 0.0
    d.cell_size = float(domain.cell_size)
    return d


def make_params(params) -> SphParams:
    p = SphParams()
    p.c0, p.rho0, p.gamma, p.delta = params.c0, params.rho0, params.gamma, params.delta
    p.alpha, p.nu, p.eps = params.alpha, params.nu, params.eps
    for k in range(3):
        p.g[k] = float(params.g[k])
    p.pressure_form = int(params.pressure_form)
    p.delta_form = int(getattr(params, "delta_form", 0))
    p.renorm_rcond = float(getattr(params, "renorm_rcond", 1e-4))
    return p


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _f32(t, shape=None):
    assert t.is_cuda and t.dtype == torch.float32 and t.is_contiguous(), "need a contiguous float32 CUDA tensor"
    if shape is not None:
        assert tuple(t.shape) == tuple(shape), (tuple(t.shape), shape)
    return t


PREFIX_SUM_NOALLOC_MAX = 1 << 26      # SPH_PREFIX_SUM_NOALLOC_MAX of include/sph.h


def prefix_sum_noalloc(counts, offsets):
    """sph_prefix_sum_noalloc: exclusive prefix sum of a uint32 count array (viewed through an int32 / uint32 CUDA tensor
    of n entries) into the caller's int64 tensor of n + 1 entries, on the current stream.  Allocates nothing -- neither
    here (both tensors are the caller's) nor in the library; raises SphError(-6) beyond PREFIX_SUM_NOALLOC_MAX."""
    lib = load_library()
    assert counts.is_cuda and counts.is_contiguous() and counts.dtype in (torch.int32, torch.uint32)
    n = int(counts.numel())
    assert offsets.is_cuda and offsets.is_contiguous() and offsets.dtype == torch.int64 and offsets.numel() == n + 1
    rc = lib.sph_prefix_sum_noalloc(int(counts.device.index or 0), _ptr(counts), _ptr(offsets), n, _stream())
    if rc != 0:
        raise SphError(rc, lib.sph_strerror(rc).decode())
    return offsets


class Sph:
    """One ``sph_ctx``.  Method names mirror the C calls (sph_<name>)."""

    def __init__(self, device: int = 0, n_max: int = 0):
        self.lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the SPH library has no CPU fallback")
        self.device = device
        self._ctx = C.c_void_p()
        self._chk(self.lib.sph_create(C.byref(self._ctx), device, n_max))
        self.n = 0
        self.dim = 0

    def close(self):
        if self._ctx:
            self.lib.sph_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _chk(self, code):
        if code != 0:
            raise SphError(code, self.lib.sph_strerror(code).decode())

    # ------------------------------------------------------------------ calls
    def build_cells(self, domain, x, h):
        self.dim = int(domain.dim)
        self.n = int(x.shape[0])
        self._dom = make_domain(domain)
        _f32(x, (self.n, self.dim))
        _f32(h, (self.n,))
        self._chk(self.lib.sph_build_cells(self._ctx, C.byref(self._dom), _ptr(x), _ptr(h), self.n, _stream()))

    def neighbors(self, search_scale: float = 1.0) -> int:
        nnz = C.c_int64(0)
        self._chk(self.lib.sph_neighbors(self._ctx, float(search_scale), C.byref(nnz), _stream()))
        self.nnz = int(nnz.value)
        return self.nnz

    def neighbors_export(self):
        row_ptr = torch.empty(self.n + 1, dtype=torch.int64, device=f"cuda:{self.device}")
        col = torch.empty(max(self.nnz, 1), dtype=torch.int32, device=f"cuda:{self.device}")
        self._chk(self.lib.sph_neighbors_export(self._ctx, _ptr(row_ptr), _ptr(col), _stream()))
        return row_ptr, col[: self.nnz]

    def shift(self, theta, x, m, rho, kind):
        """particle shifting at the end of a step: x <- x - theta l^2 sum_j V_j grad_i W_ij for fluid
        kinds, at the current positions, on the lists of the last build; x in place"""
        _f32(x, (self.n, self.dim)); _f32(m, (self.n,)); _f32(rho, (self.n,))
        assert kind.dtype == torch.uint8 and kind.is_cuda and kind.is_contiguous()
        self._chk(self.lib.sph_shift(self._ctx, float(theta), _ptr(x), _ptr(m), _ptr(rho), _ptr(kind), _stream()))
        return x

    def lists_valid(self, x, skin_needed: float = 0.0):
        """(valid, max displacement since the build): the Verlet-list test of PAPER.md:568"""
        _f32(x, (self.n, self.dim))
        ok, D = C.c_int32(0), C.c_float(0.0)
        self._chk(self.lib.sph_lists_valid(self._ctx, _ptr(x), float(skin_needed), C.byref(ok), C.byref(D), _stream()))
        return bool(ok.value), float(D.value)

    def density(self, m, out=None):
        _f32(m, (self.n,))
        out = torch.empty_like(m) if out is None else out
        self._chk(self.lib.sph_density(self._ctx, _ptr(m), _ptr(out), _stream()))
        return out

    def density_vjp(self, m, rho_bar, x_bar=None, m_bar=None, want_m_bar=True):
        """(x_bar, m_bar) = J^T rho_bar of density() at the build positions"""
        import torch
        m, rho_bar = _f32(m, (self.n,)), _f32(rho_bar, (self.n,))
        x_bar = torch.empty((self.n, self.dim), dtype=torch.float32, device=m.device) if x_bar is None else _f32(x_bar, (self.n, self.dim))
        if m_bar is None and want_m_bar:
            m_bar = torch.empty(self.n, dtype=torch.float32, device=m.device)
        self._chk(self.lib.sph_density_vjp(self._ctx, _ptr(m), _ptr(rho_bar), _ptr(x_bar),
                                           _ptr(m_bar) if m_bar is not None else None, _stream()))
        return x_bar, m_bar

    def grad_sum(self, a, out=None):
        """g_i = sum_j a_j grad_i W_ij at the build positions (Eq.24 with a = m/rho)"""
        a = _f32(a, (self.n,))
        out = torch.empty((self.n, self.dim), dtype=torch.float32, device=a.device) if out is None else _f32(out, (self.n, self.dim))
        self._chk(self.lib.sph_grad_sum(self._ctx, _ptr(a), _ptr(out), _stream()))
        return out

    def grad_sum_vjp(self, a, g_bar, x_bar=None, a_bar=None, want_a_bar=True):
        """(x_bar, a_bar) = J^T g_bar of grad_sum()"""
        a, g_bar = _f32(a, (self.n,)), _f32(g_bar, (self.n, self.dim))
        x_bar = torch.empty((self.n, self.dim), dtype=torch.float32, device=a.device) if x_bar is None else _f32(x_bar, (self.n, self.dim))
        if a_bar is None and want_a_bar:
            a_bar = torch.empty(self.n, dtype=torch.float32, device=a.device)
        self._chk(self.lib.sph_grad_sum_vjp(self._ctx, _ptr(a), _ptr(g_bar), _ptr(x_bar),
                                            _ptr(a_bar) if a_bar is not None else None, _stream()))
        return x_bar, a_bar

    def renorm_gradient(self, vol, A, rcond=1e-4, L=None, grad=None, want_L=True):
        """(L [n,d,d], grad [n,d]): renormalisation matrix and corrected gradient of the scalar field A"""
        vol, A = _f32(vol, (self.n,)), _f32(A, (self.n,))
        if L is None and want_L:
            L = torch.empty((self.n, self.dim, self.dim), dtype=torch.float32, device=A.device)
        grad = torch.empty((self.n, self.dim), dtype=torch.float32, device=A.device) if grad is None else _f32(grad, (self.n, self.dim))
        self._chk(self.lib.sph_renorm_gradient(self._ctx, _ptr(vol), _ptr(A), C.c_float(rcond),
                                               _ptr(L) if L is not None else None, _ptr(grad), _stream()))
        return L, grad

    def renorm_gradient_vjp(self, vol, A, grad_bar, rcond=1e-4, x_bar=None, vol_bar=None, A_bar=None):
        """(x_bar, vol_bar, A_bar) = J^T grad_bar of the corrected gradient of renorm_gradient()"""
        vol, A, grad_bar = _f32(vol, (self.n,)), _f32(A, (self.n,)), _f32(grad_bar, (self.n, self.dim))
        x_bar = torch.empty((self.n, self.dim), dtype=torch.float32, device=A.device) if x_bar is None else _f32(x_bar, (self.n, self.dim))
        vol_bar = torch.empty(self.n, dtype=torch.float32, device=A.device) if vol_bar is None else _f32(vol_bar, (self.n,))
        A_bar = torch.empty(self.n, dtype=torch.float32, device=A.device) if A_bar is None else _f32(A_bar, (self.n,))
        self._chk(self.lib.sph_renorm_gradient_vjp(self._ctx, _ptr(vol), _ptr(A), C.c_float(rcond), _ptr(grad_bar),
                                                   _ptr(x_bar), _ptr(vol_bar), _ptr(A_bar), _stream()))
        return x_bar, vol_bar, A_bar

    def rhs(self, params, x, v, rho, m, kind, drho_dt=None, acc=None):
        p = make_params(params)
        _f32(x, (self.n, self.dim)); _f32(v, (self.n, self.dim)); _f32(rho, (self.n,)); _f32(m, (self.n,))
        assert kind.dtype == torch.uint8 and kind.is_cuda and kind.is_contiguous()
        drho_dt = torch.empty_like(rho) if drho_dt is None else drho_dt
        acc = torch.empty_like(v) if acc is None else acc
        self._chk(self.lib.sph_rhs(self._ctx, C.byref(p), _ptr(x), _ptr(v), _ptr(rho), _ptr(m), _ptr(kind),
                                   _ptr(drho_dt), _ptr(acc), _stream()))
        return drho_dt, acc

    def rhs_vjp(self, params, x, v, rho, m, kind, drho_bar, acc_bar, out=None):
        p = make_params(params)
        _f32(x, (self.n, self.dim)); _f32(v, (self.n, self.dim)); _f32(rho, (self.n,)); _f32(m, (self.n,))
        _f32(drho_bar, (self.n,)); _f32(acc_bar, (self.n, self.dim))
        if out is None:
            out = (torch.empty_like(x), torch.empty_like(v), torch.empty_like(rho),
                   torch.empty(10, dtype=torch.float32, device=x.device))
        xb, vb, rb, pb = out
        self._chk(self.lib.sph_rhs_vjp(self._ctx, C.byref(p), _ptr(x), _ptr(v), _ptr(rho), _ptr(m), _ptr(kind),
                                       _ptr(drho_bar), _ptr(acc_bar), _ptr(xb), _ptr(vb), _ptr(rb), _ptr(pb), _stream()))
        return xb, vb, rb, pb

    def rk_step(self, domain, params, dt, skin, x, v, rho, m, h, kind):
        """in place on x, v, rho"""
        d, p = make_domain(domain), make_params(params)
        n = int(x.shape[0])
        self.n, self.dim = n, int(domain.dim)
        self._chk(self.lib.sph_rk_step(self._ctx, C.byref(d), C.byref(p), float(dt), float(skin), n, _ptr(x), _ptr(v),
                                       _ptr(rho), _ptr(m), _ptr(h), _ptr(kind), _stream()))

    def rk_step_vjp(self, domain, params, dt, skin, x0, v0, rho0, m, h, kind, x_bar, v_bar, rho_bar, params_bar=None):
        """in place on x_bar, v_bar, rho_bar; params_bar (10 floats, device) is accumulated into"""
        d, p = make_domain(domain), make_params(params)
        n = int(x0.shape[0])
        self.n, self.dim = n, int(domain.dim)
        self._chk(self.lib.sph_rk_step_vjp(self._ctx, C.byref(d), C.byref(p), float(dt), float(skin), n, _ptr(x0), _ptr(v0),
                                           _ptr(rho0), _ptr(m), _ptr(h), _ptr(kind), _ptr(x_bar), _ptr(v_bar),
                                           _ptr(rho_bar), _ptr(params_bar), _stream()))

    def forward_backward_host(self, domain, params, search_scale, x, v, rho, m, h, kind, drho_bar, acc_bar, outs=None):
        """HOST numpy arrays (or pinned torch CPU tensors) in and out; copies are inside the C call."""
        d, p = make_domain(domain), make_params(params)
        n, dim = int(x.shape[0]), int(domain.dim)

        def hp(a):
            if isinstance(a, torch.Tensor):
                assert not a.is_cuda and a.is_contiguous()
                return C.c_void_p(a.data_ptr())
            assert a.flags["C_CONTIGUOUS"]
            return a.ctypes.data_as(C.c_void_p)

        if outs is None:
            outs = dict(drho_dt=np.empty(n, np.float32), acc=np.empty((n, dim), np.float32),
                        x_bar=np.empty((n, dim), np.float32), v_bar=np.empty((n, dim), np.float32),
                        rho_bar=np.empty(n, np.float32), params_bar=np.empty(10, np.float32))
        nnz = C.c_int64(0)
        self._chk(self.lib.sph_forward_backward_host(
            self._ctx, C.byref(d), C.byref(p), float(search_scale), n, hp(x), hp(v), hp(rho), hp(m), hp(h), hp(kind),
            hp(drho_bar), hp(acc_bar), hp(outs["drho_dt"]), hp(outs["acc"]), hp(outs["x_bar"]), hp(outs["v_bar"]),
            hp(outs["rho_bar"]), hp(outs["params_bar"]), C.byref(nnz)))
        self.n, self.dim, self.nnz = n, dim, int(nnz.value)
        return outs

    def step_host(self, domain, domain_rk, params, dt, skin, x, v, rho, m, h, kind, drho_bar, acc_bar, outs):
        """One whole step of the hot path on HOST arrays (pinned torch CPU tensors or numpy); x, v, rho are advanced in
        place; ``outs`` maps density, drho_dt, acc, x_bar, v_bar, rho_bar, params_bar to host arrays (or None)."""
        d, drk, p = make_domain(domain), make_domain(domain_rk), make_params(params)
        n = int(x.shape[0])

        def hp(a):
            if a is None:
                return None
            if isinstance(a, torch.Tensor):
                assert not a.is_cuda and a.is_contiguous()
                return C.c_void_p(a.data_ptr())
            assert a.flags["C_CONTIGUOUS"]
            return a.ctypes.data_as(C.c_void_p)

        nnz = (C.c_int64 * 2)()
        self._chk(self.lib.sph_step_host(
            self._ctx, C.byref(d), C.byref(drk), C.byref(p), float(dt), float(skin), n, hp(x), hp(v), hp(rho), hp(m),
            hp(h), hp(kind), hp(drho_bar), hp(acc_bar), hp(outs.get("density")), hp(outs.get("drho_dt")),
            hp(outs.get("acc")), hp(outs.get("x_bar")), hp(outs.get("v_bar")), hp(outs.get("rho_bar")),
            hp(outs.get("params_bar")), C.cast(nnz, C.POINTER(C.c_int64))))
        self.n, self.dim = n, int(domain.dim)
        return int(nnz[0]), int(nnz[1])

    def set_option(self, key, value):
        self._chk(self.lib.sph_set_option(self._ctx, int(key), int(value)))

    def profile_enable(self, on=True):
        self._chk(self.lib.sph_profile_enable(self._ctx, 1 if on else 0))

    def profile_read(self):
        """{class: (ms_sum, launches)} since the last read (synchronises the device)"""
        k = len(KERNEL_CLASSES)
        ms, cnt = (C.c_double * k)(), (C.c_int64 * k)()
        self._chk(self.lib.sph_profile_read(self._ctx, C.cast(ms, C.POINTER(C.c_double)), C.cast(cnt, C.POINTER(C.c_int64))))
        return {name: (float(ms[i]), int(cnt[i])) for i, name in enumerate(KERNEL_CLASSES)}

    def check(self):
        self._chk(self.lib.sph_check(self._ctx))

    def debug_bounds_violations(self) -> int:
        """violations counted by a --bounds debug build of the library; -1 for a normal build"""
        c = C.c_int64(0)
        self._chk(self.lib.sph_debug_bounds_violations(self._ctx, C.byref(c)))
        return int(c.value)

    def layout(self):
        """layout of the lists of the last neighbors(): mode 1 generic / 2 tile-local, tile edge, largest halo / rows"""
        mode, edge, hm, rm = C.c_int32(0), C.c_int32(0), C.c_int64(0), C.c_int64(0)
        self._chk(self.lib.sph_get_layout(self._ctx, C.byref(mode), C.byref(edge), C.byref(hm), C.byref(rm)))
        return dict(mode=int(mode.value), tile_edge=int(edge.value), halo_max=int(hm.value), rows_max=int(rm.value))

    def info(self):
        nc = (C.c_int32 * 3)()
        n, nnz, launches = C.c_int64(0), C.c_int64(0), C.c_int64(0)
        self._chk(self.lib.sph_get_info(self._ctx, C.byref(nc), C.byref(n), C.byref(nnz), C.byref(launches)))
        return dict(ncell=tuple(nc), n=int(n.value), nnz=int(nnz.value), launches=int(launches.value))
