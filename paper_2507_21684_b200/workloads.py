"""Seeded synthetic inputs for the five BASELINE.json configs (C0..C4).

This module only *generates inputs* (particle lattices, initial fields, parameter
sets).  It holds none of the method's arithmetic (no kernel, no neighbour search,
no SPH sums) and imports neither ``oracle/`` nor the CUDA binding, so both sides
can be fed the very same fp32 arrays.  Recipe: SURVEY.md §8(d) table; stands in
for the paper's "fully occupied domains, with random noise added to the particle
positions, with the usual neighbourhood sizes".

Every array is created on the host with ``numpy.random.Generator(PCG64(seed))``,
``seed = 1000 + config index``, in float64, then cast ONCE to float32.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

__all__ = ["Domain", "Params", "Workload", "make", "CONFIG_NAMES"]

CONFIG_NAMES = ("C0_tgv2d_32", "C1_tgv2d_256", "C2_dambreak2d", "C3_tgv3d_128", "C4_box3d_256_varh")


@dataclass
class Domain:
    """Mirror of ``sph_domain`` (include/sph.h)."""
    dim: int
    periodic: tuple
    lo: tuple
    hi: tuple
    cell_size: float


@dataclass
class Params:
    """Mirror of ``sph_params`` (include/sph.h). Order of ``as_list`` = order of params_bar."""
    c0: float = 10.0
    rho0: float = 1.0
    gamma: float = 7.0
    delta: float = 0.1
    alpha: float = 0.0
    nu: float = 0.01
    eps: float = 0.01
    g: tuple = (0.0, 0.0, 0.0)
    pressure_form: int = 0
    delta_form: int = 0          # 0 = Molteni-Colagrossi delta-term; 1 = with the renormalised density gradient of [43]
    renorm_rcond: float = 1e-4   # relative eigenvalue cutoff of the pseudo-inverse L_i, delta_form 1 only

    def as_list(self):
        return [self.c0, self.rho0, self.gamma, self.delta, self.alpha, self.nu, self.eps,
                self.g[0], self.g[1], self.g[2]]


@dataclass
class Workload:
    name: str
    domain: Domain
    params: Params
    x: np.ndarray      # [n, dim] f32
    v: np.ndarray      # [n, dim] f32
    rho: np.ndarray    # [n] f32
    m: np.ndarray      # [n] f32
    h: np.ndarray      # [n] f32   support radius H ("h" is the support)
    kind: np.ndarray   # [n] u8    0 fluid, 1 fixed boundary
    dt: float
    dx: float
    seed: int
    notes: dict = field(default_factory=dict)

    @property
    def n(self):
        return int(self.x.shape[0])

    @property
    def dim(self):
        return int(self.domain.dim)


def _f32(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64).astype(np.float32))


def _lattice(n_axis, dim):
    """Cell-centred lattice on the unit box, x fastest.  Returns [n_axis**dim, dim] f64."""
    dx = 1.0 / n_axis
    c = (np.arange(n_axis, dtype=np.float64) + 0.5) * dx
    if dim == 2:
        yy, xx = np.meshgrid(c, c, indexing="ij")
        return np.stack([xx.ravel(), yy.ravel()], axis=1)
    zz, yy, xx = np.meshgrid(c, c, c, indexing="ij")
    return np.stack([xx.ravel(), yy.ravel(), zz.ravel()], axis=1)


def _tgv(x, dim):
    """Taylor-Green initial velocity on the unit box (BASELINE.json configs 0,1,3)."""
    tp = 2.0 * np.pi
    if dim == 2:
        u = np.sin(tp * x[:, 0]) * np.cos(tp * x[:, 1])
        w = -np.cos(tp * x[:, 0]) * np.sin(tp * x[:, 1])
        return np.stack([u, w], axis=1)
    u = np.sin(tp * x[:, 0]) * np.cos(tp * x[:, 1]) * np.cos(tp * x[:, 2])
    w = -np.cos(tp * x[:, 0]) * np.sin(tp * x[:, 1]) * np.cos(tp * x[:, 2])
    return np.stack([u, w, np.zeros_like(u)], axis=1)


def _periodic_box(dim, cell):
    return Domain(dim=dim, periodic=(1,) * dim + (0,) * (3 - dim), lo=(0.0,) * 3,
                  hi=(1.0,) * dim + (0.0,) * (3 - dim), cell_size=float(cell))


def _tgv_case(idx, name, n_axis, dim, support_in_dx, jitter, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    dx = 1.0 / n_axis
    x = _lattice(n_axis, dim)
    if jitter > 0.0:
        x = x + rng.uniform(-jitter * dx, jitter * dx, size=x.shape)
        x = x - np.floor(x)            # wrap into [0,1)
    x32 = _f32(x)
    x32[x32 >= 1.0] = 0.0              # a value that rounded up to the box edge is the same point as 0
    v = _tgv(x32.astype(np.float64), dim)   # fields evaluated at the (jittered) fp32 positions
    n = x32.shape[0]
    H = np.float32(support_in_dx * dx)
    par = Params(c0=10.0, rho0=1.0, gamma=7.0, delta=0.1, alpha=0.0, nu=0.01, eps=0.01)
    return Workload(
        name=name, domain=_periodic_box(dim, float(H)), params=par,
        x=x32, v=_f32(v), rho=np.ones(n, np.float32), m=np.full(n, dx ** dim, np.float32),
        h=np.full(n, H, np.float32), kind=np.zeros(n, np.uint8),
        dt=0.25 * float(H) / par.c0, dx=dx, seed=seed,
        notes={"config": idx, "n_axis": n_axis, "support_in_dx": support_in_dx, "jitter_dx": jitter})


def _dambreak(dx, seed, name="C2_dambreak2d"):
    """BASELINE.json config 2. Fluid block 1.0 x 2.0 in a 4.0 x 3.0 tank, 3 layers of fixed
    boundary particles outside bottom / left / right walls (open top)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    nfx, nfy = int(round(1.0 / dx)), int(round(2.0 / dx))
    cx = (np.arange(nfx) + 0.5) * dx
    cy = (np.arange(nfy) + 0.5) * dx
    yy, xx = np.meshgrid(cy, cx, indexing="ij")
    xf = np.stack([xx.ravel(), yy.ravel()], axis=1)
    layers = -(np.arange(3) + 0.5) * dx
    # bottom: x from -3dx .. 4+3dx
    nbx = int(round(4.0 / dx)) + 6
    bx = (np.arange(nbx) - 3 + 0.5) * dx
    by, bxx = np.meshgrid(layers, bx, indexing="ij")
    bottom = np.stack([bxx.ravel(), by.ravel()], axis=1)
    nwy = int(round(3.0 / dx))
    wy = (np.arange(nwy) + 0.5) * dx
    wyy, wxx = np.meshgrid(wy, layers, indexing="ij")
    left = np.stack([wxx.ravel(), wyy.ravel()], axis=1)
    right = np.stack([4.0 - wxx.ravel(), wyy.ravel()], axis=1)
    xb = np.concatenate([bottom, left, right], axis=0)
    x = np.concatenate([xf, xb], axis=0)
    nf, nb = xf.shape[0], xb.shape[0]
    n = nf + nb
    g = 9.81
    Hw = 2.0
    c0 = 10.0 * np.sqrt(2.0 * g * Hw)
    rho0, gamma = 1000.0, 7.0
    depth = np.clip(Hw - x[:, 1], 0.0, None)      # boundary below y=0 continues the column
    depth = np.where(x[:, 1] < 0.0, Hw - x[:, 1], depth)
    rho = rho0 * (1.0 + gamma * g * depth / c0 ** 2) ** (1.0 / gamma)
    v = np.zeros((n, 2))
    v[:nf] = rng.normal(0.0, 0.01 * c0, size=(nf, 2))
    kind = np.zeros(n, np.uint8)
    kind[nf:] = 1
    H = np.float32(4.0 * dx)
    lo = (np.float32(-3.0 * dx), np.float32(-3.0 * dx), 0.0)
    hi = (np.float32(4.0 + 3.0 * dx), np.float32(3.0), 0.0)
    dom = Domain(dim=2, periodic=(0, 0, 0), lo=tuple(float(a) for a in lo),
                 hi=tuple(float(a) for a in hi), cell_size=float(H))
    par = Params(c0=float(np.float32(c0)), rho0=rho0, gamma=gamma, delta=0.1, alpha=0.01, nu=0.0,
                 eps=0.01, g=(0.0, -g, 0.0))
    return Workload(
        name=name, domain=dom, params=par, x=_f32(x), v=_f32(v), rho=_f32(rho),
        m=np.full(n, rho0 * dx * dx, np.float32), h=np.full(n, H, np.float32), kind=kind,
        dt=0.25 * float(H) / float(c0), dx=dx, seed=seed,
        notes={"config": 2, "n_fluid": nf, "n_boundary": nb})


def _box3d_varh(n_axis, seed, name="C4_box3d_256_varh"):
    """BASELINE.json config 4: jittered lattice, Gaussian velocities, log-normal support."""
    rng = np.random.Generator(np.random.PCG64(seed))
    dx = 1.0 / n_axis
    x = _lattice(n_axis, 3)
    x = x + rng.uniform(-0.1 * dx, 0.1 * dx, size=x.shape)
    x = x - np.floor(x)
    x32 = _f32(x)
    x32[x32 >= 1.0] = 0.0
    n = x32.shape[0]
    v = rng.normal(0.0, 0.1, size=(n, 3))
    h = 3.0 * dx * np.exp(rng.normal(0.0, 0.1, size=n))
    h32 = _f32(h)
    par = Params(c0=10.0, rho0=1.0, gamma=7.0, delta=0.1, alpha=0.0, nu=0.01, eps=0.01)
    return Workload(
        name=name, domain=_periodic_box(3, float(h32.max())), params=par,
        x=x32, v=_f32(v), rho=np.ones(n, np.float32), m=np.full(n, dx ** 3, np.float32),
        h=h32, kind=np.zeros(n, np.uint8), dt=0.25 * 3.0 * dx / par.c0, dx=dx, seed=seed,
        notes={"config": 4, "n_axis": n_axis})


def make(config: int, n_axis: int | None = None, dx: float | None = None) -> Workload:
    """Build config ``config`` (0..4).  ``n_axis`` / ``dx`` shrink the same recipe for tests
    (parity cases at sizes the oracle finishes in seconds); ``None`` = BASELINE.json's size."""
    seed = 1000 + config
    if config == 0:
        return _tgv_case(0, CONFIG_NAMES[0], n_axis or 32, 2, 4.0, 0.0, seed)
    if config == 1:
        return _tgv_case(1, CONFIG_NAMES[1], n_axis or 256, 2, 4.0, 0.05, seed)
    if config == 2:
        return _dambreak(dx or 0.002, seed)
    if config == 3:
        return _tgv_case(3, CONFIG_NAMES[3], n_axis or 128, 3, 3.0, 0.0, seed)
    if config == 4:
        return _box3d_varh(n_axis or 256, seed)
    raise ValueError("config must be 0..4")


RK_SKIN = 0.06      # Verlet skin of the RK4 list: skin*H >= 2*dt*max|v| = 0.05 H for dt = 0.25 H/c0, |v| <= c0/10


def rk_domain(wl: Workload, skin: float = RK_SKIN) -> Domain:
    """grid for sph_rk_step: the same box with cell_size >= (1 + skin) * max h (input generation only)"""
    d = wl.domain
    cs = float(np.float32(np.float32(wl.h.max()) * np.float32(1.0 + skin) * np.float32(1.0001)))
    return Domain(dim=d.dim, periodic=d.periodic, lo=d.lo, hi=d.hi, cell_size=max(cs, float(d.cell_size)))


def random_cotangents(wl: Workload, seed_offset: int = 500):
    """lambda = dL/d(drho/dt), mu = dL/d(acc) ~ N(0,1) (C2, C3, C4)."""
    rng = np.random.Generator(np.random.PCG64(wl.seed + seed_offset))
    lam = rng.normal(size=wl.n).astype(np.float32)
    mu = rng.normal(size=(wl.n, wl.dim)).astype(np.float32)
    return lam, mu


def perturbed(wl: Workload, amp_x: float = 0.2, amp_rho: float = 0.02, seed_offset: int = 77) -> Workload:
    """A disordered variant of ``wl`` for parity tests that must exercise every term:
    positions jittered by ``amp_x*dx`` (then wrapped on periodic axes), densities scaled by
    ``1 + amp_rho*U(-1,1)``.  Input generation only."""
    rng = np.random.Generator(np.random.PCG64(wl.seed + seed_offset))
    x = wl.x.astype(np.float64) + rng.uniform(-amp_x * wl.dx, amp_x * wl.dx, size=wl.x.shape)
    for k in range(wl.dim):
        if wl.domain.periodic[k]:
            L = wl.domain.hi[k] - wl.domain.lo[k]
            x[:, k] = wl.domain.lo[k] + np.mod(x[:, k] - wl.domain.lo[k], L)
    x32 = _f32(x)
    for k in range(wl.dim):
        if wl.domain.periodic[k]:
            x32[x32[:, k] >= np.float32(wl.domain.hi[k]), k] = np.float32(wl.domain.lo[k])
        else:
            x32[:, k] = np.clip(x32[:, k], np.float32(wl.domain.lo[k]),
                                np.nextafter(np.float32(wl.domain.hi[k]), np.float32(-np.inf)))
    rho = wl.rho.astype(np.float64) * (1.0 + amp_rho * rng.uniform(-1.0, 1.0, size=wl.n))
    out = Workload(**{**wl.__dict__})
    out.x = x32
    out.rho = _f32(rho)
    out.name = wl.name + "_perturbed"
    return out
