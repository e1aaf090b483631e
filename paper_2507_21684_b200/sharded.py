"""Domain-decomposed sph_rhs / sph_rhs_vjp over several GPUs: host-side plumbing only.

One process per GPU.  The box is cut into `world` slabs along one axis; a rank owns the particles of its slab and
borrows, from its two neighbours, the particles within one halo width (>= the search radius) of the shared faces.
Every step of the arithmetic still runs in the library's kernels, on the local problem "owned + ghost particles in the
slab extended by the halo, bounded along the cut axis":

  * one exchange per RHS (x, v, rho, m, h, kind of the ghosts) and one per VJP (their cotangents lambda, mu);
  * NO reverse halo reduction: the lists are symmetric and row i of the adjoint kernels evaluates both ordered pairs
    (i<-j), (j<-i) and keeps what lands on i, so x_bar, v_bar, rho_bar of an owned row are complete once the states and
    cotangents of its neighbours are there;
  * params_bar is linear in the cotangents and the terms of row i carry only lambda_i, mu_i: the local adjoint with the
    ghost cotangents zeroed gives this rank's share, one 10-float all-reduce (sum) gives the total;
  * ghost rows are computed and thrown away (their neighbourhoods are truncated).
Periodic images across the cut axis are resolved when a ghost is received (+-L on that coordinate); the other axes keep
their periodicity inside the library.  Particles that have left their slab move to their new owner in `migrate`.

The collectives are torch.distributed point-to-point calls (NCCL over NVLink on GPUs; gloo in the CPU tests, which plug
the fp64 oracle in as the local solver -- tests/test_multirank_cpu.py).  Nothing here computes a pair term.
"""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist

from .workloads import Domain

__all__ = ["ShardedSph", "CudaSolver"]


class CudaSolver:
    """Local solver = the C-ABI library on this rank's GPU (paper_2507_21684_b200.binding.Sph)."""

    def __init__(self, device: int = 0):
        from .binding import Sph
        self.sph = Sph(device)
        self.device = torch.device(f"cuda:{device}")

    def build(self, domain, x, h, search_scale):
        self.sph.build_cells(domain, x, h)
        return self.sph.neighbors(search_scale)

    def density(self, m):
        return self.sph.density(m)

    def rhs(self, params, x, v, rho, m, h, kind):
        return self.sph.rhs(params, x, v, rho, m, kind)

    def rhs_vjp(self, params, x, v, rho, m, h, kind, lam, mu):
        return self.sph.rhs_vjp(params, x, v, rho, m, kind, lam, mu)

    def close(self):
        self.sph.close()


class ShardedSph:
    """Slab decomposition along `axis` (default: the longest axis of the box).

    halo_width: >= search_scale * max(h) over ALL ranks, <= the slab width (so that a neighbour is never two ranks away).
    solver: an object with build / density / rhs / rhs_vjp as CudaSolver has them, working on tensors of `device`.
    """

    def __init__(self, domain: Domain, halo_width: float, solver, axis: int | None = None, group=None):
        self.domain, self.solver, self.group = domain, solver, group
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        dim = int(domain.dim)
        ext = [float(domain.hi[k]) - float(domain.lo[k]) for k in range(dim)]
        self.axis = int(np.argmax(ext)) if axis is None else int(axis)
        a = self.axis
        self.periodic = bool(domain.periodic[a])
        self.lo, self.L, self.w = float(domain.lo[a]), ext[a], float(halo_width)
        width = self.L / self.world
        if not (self.w > 0.0) or self.w > width:
            raise ValueError(f"halo width {self.w} must be positive and at most the slab width {width}")
        if self.periodic and self.L < 2.0 * self.w:
            raise ValueError("a periodic axis must be at least two halo widths long")
        self.lo_r = self.lo + self.L * self.rank / self.world
        self.hi_r = self.lo + self.L * (self.rank + 1) / self.world
        wrap = self.periodic
        self.left = (self.rank - 1) % self.world if (wrap or self.rank > 0) else None
        self.right = (self.rank + 1) % self.world if (wrap or self.rank < self.world - 1) else None
        # +-L on the cut coordinate of a ghost that arrives across the periodic face
        self.shift_left = -self.L if (wrap and self.rank == 0) else 0.0
        self.shift_right = self.L if (wrap and self.rank == self.world - 1) else 0.0
        pad = 1e-3 * self.w                                   # the shifted ghosts are rounded to binary32
        lo3, hi3, per3 = list(domain.lo), list(domain.hi), list(domain.periodic)
        lo3[a], hi3[a], per3[a] = self.lo_r - self.w - pad, self.hi_r + self.w + pad, 0
        self.local_domain = Domain(dim=dim, periodic=tuple(per3), lo=tuple(lo3), hi=tuple(hi3),
                                   cell_size=float(domain.cell_size))
        self.n_own = 0
        self._built_scale = None

    # ------------------------------------------------------------------------------------------ ownership
    def wrapped(self, x: torch.Tensor) -> torch.Tensor:
        """cut-axis coordinate in [lo, lo + L) (binary64) -- identity on a bounded axis"""
        xa = x[:, self.axis].double()
        if not self.periodic:
            return xa
        xw = xa - self.L * torch.floor((xa - self.lo) / self.L)
        return torch.where(xw >= self.lo + self.L, xw - self.L, xw)

    def owner(self, x: torch.Tensor) -> torch.Tensor:
        """rank that owns each position (int64); the same formula on every rank"""
        r = torch.floor((self.wrapped(x) - self.lo) / self.L * self.world).long()
        return r.clamp_(0, self.world - 1)

    def select_owned(self, x: torch.Tensor) -> torch.Tensor:
        """indices of the rows of a replicated array that this rank owns (no communication)"""
        return torch.nonzero(self.owner(x) == self.rank).flatten()

    # ------------------------------------------------------------------------------------------ communication
    def _all_counts(self, mine: torch.Tensor) -> torch.Tensor:
        """[world, k] int64 table of every rank's small integer record"""
        if self.world == 1:
            return mine.view(1, -1).clone()
        out = [torch.empty_like(mine) for _ in range(self.world)]
        dist.all_gather(out, mine, group=self.group)
        return torch.stack(out)

    def _p2p(self, sends: dict, recv_rows: dict, cols: int, like: torch.Tensor) -> dict:
        """sends: {peer: tensor [rows, cols]}, recv_rows: {peer: rows}.  Returns {peer: tensor}.  A message to oneself is
        a copy; everything else is one isend/irecv per peer, posted together."""
        got, ops, keep = {}, [], []
        for peer, rows in recv_rows.items():
            if peer == self.rank:
                got[peer] = sends[peer].clone()
                continue
            buf = torch.empty((rows, cols), dtype=like.dtype, device=like.device)
            got[peer] = buf
            if rows:
                ops.append(dist.P2POp(dist.irecv, buf, peer, group=self.group))
        for peer, t in sends.items():
            if peer != self.rank and t.shape[0]:
                t = t.contiguous()
                keep.append(t)
                ops.append(dist.P2POp(dist.isend, t, peer, group=self.group))
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()
        return got

    # ------------------------------------------------------------------------------------------ halo plan
    def plan(self, x: torch.Tensor):
        """Decide, from the owned positions x [n_own, dim], which rows each neighbour borrows.  Collective (counts)."""
        if not bool((self.owner(x) == self.rank).all()):
            raise ValueError("plan(): some positions belong to another slab -- call migrate() first")
        xw = self.wrapped(x)
        none = torch.empty(0, dtype=torch.long, device=x.device)
        self.idx_L = torch.nonzero(xw < self.lo_r + self.w).flatten() if self.left is not None else none
        self.idx_R = torch.nonzero(xw >= self.hi_r - self.w).flatten() if self.right is not None else none
        mine = torch.tensor([self.idx_L.numel(), self.idx_R.numel()], dtype=torch.long, device=x.device)
        counts = self._all_counts(mine).cpu()
        self.n_own = int(x.shape[0])
        self.n_from_left = int(counts[self.left][1]) if self.left is not None else 0      # their right-face rows
        self.n_from_right = int(counts[self.right][0]) if self.right is not None else 0   # their left-face rows
        self.n_local = self.n_own + self.n_from_left + self.n_from_right
        self._xw32 = xw.to(torch.float32)
        self._built_scale = None
        return self.n_from_left, self.n_from_right

    def exchange(self, fields, positions: bool = False):
        """fields: list of tensors with n_own rows (any float/uint8 dtype, 1-D or 2-D).  ONE message per neighbour
        carries all of them (as float32 columns).  Returns the list extended to n_local rows: owned, ghosts from the left
        neighbour, ghosts from the right neighbour.  positions=True: fields[0] is x; its cut coordinate is put into the
        slab's frame (wrapped for the owned rows, shifted by -+L for ghosts from across the periodic face)."""
        dev = fields[0].device
        cols2d = [f.reshape(self.n_own, -1).to(torch.float32) for f in fields]
        if positions:
            cols2d[0] = cols2d[0].clone()
            cols2d[0][:, self.axis] = self._xw32
        widths = [c.shape[1] for c in cols2d]
        packed = torch.cat(cols2d, dim=1) if len(cols2d) > 1 else cols2d[0]
        ncol = packed.shape[1]
        partL, partR = packed[self.idx_L], packed[self.idx_R]
        sends, recv_rows = {}, {}
        if self.left is not None and self.left == self.right:
            sends[self.left] = torch.cat([partL, partR])
            recv_rows[self.left] = self.n_from_right + self.n_from_left
        else:
            if self.left is not None:
                sends[self.left], recv_rows[self.left] = partL, self.n_from_left
            if self.right is not None:
                sends[self.right], recv_rows[self.right] = partR, self.n_from_right
        got = self._p2p(sends, recv_rows, ncol, packed)
        empty = packed[:0]
        if self.left is not None and self.left == self.right:
            buf = got[self.left]                               # [their L part -> my right ghosts, their R part -> my left ghosts]
            from_right, from_left = buf[:self.n_from_right], buf[self.n_from_right:]
        else:
            from_left = got[self.left] if self.left is not None else empty
            from_right = got[self.right] if self.right is not None else empty
        if positions:
            for g, sh in ((from_left, self.shift_left), (from_right, self.shift_right)):
                if sh != 0.0 and g.shape[0]:
                    g[:, self.axis] = (g[:, self.axis].double() + sh).to(torch.float32)
        full = torch.cat([packed, from_left, from_right])
        out, c0 = [], 0
        for f, wd in zip(fields, widths):
            col = full[:, c0:c0 + wd]
            c0 += wd
            col = col.reshape((self.n_local,) + tuple(f.shape[1:])).contiguous()
            out.append(col.to(f.dtype) if f.dtype != torch.float32 else col)
        return out

    # ------------------------------------------------------------------------------------------ the path
    def _prepare(self, x, v, rho, m, h, kind, search_scale):
        X, V, RHO, M, H, K = self.exchange([x, v, rho, m, h, kind], positions=True)       # the one exchange of a RHS
        self.solver.build(self.local_domain, X, H, search_scale)
        self._built_scale = search_scale
        return X, V, RHO, M, H, K

    def density(self, x, m, h, search_scale: float = 1.0):
        X, M, H = self.exchange([x, m, h], positions=True)
        self.solver.build(self.local_domain, X, H, search_scale)
        return self.solver.density(M)[:self.n_own]

    def rhs(self, params, x, v, rho, m, h, kind, search_scale: float = 1.0):
        """(drho_dt, acc) of the owned rows; plan(x) must have been called for these positions"""
        X, V, RHO, M, H, K = self._prepare(x, v, rho, m, h, kind, search_scale)
        self._state = (X, V, RHO, M, H, K)
        drho, acc = self.solver.rhs(params, X, V, RHO, M, H, K)
        return drho[:self.n_own], acc[:self.n_own]

    def rhs_vjp(self, params, drho_bar, acc_bar, state=None):
        """(x_bar, v_bar, rho_bar) of the owned rows and the all-reduced params_bar, for the state of the last rhs() (or
        `state` = (x, v, rho, m, h, kind, search_scale), which costs the RHS exchange again)."""
        if state is not None:
            self._state = self._prepare(*state)
        X, V, RHO, M, H, K = self._state
        LAM, MU = self.exchange([drho_bar, acc_bar])                                     # the one exchange of a VJP
        xb, vb, rb, _ = self.solver.rhs_vjp(params, X, V, RHO, M, H, K, LAM, MU)
        # this rank's share of params_bar: the rows it owns, i.e. ghost cotangents zeroed (linear in the cotangents)
        LAM0, MU0 = LAM.clone(), MU.clone()
        LAM0[self.n_own:] = 0
        MU0[self.n_own:] = 0
        pb = self.solver.rhs_vjp(params, X, V, RHO, M, H, K, LAM0, MU0)[3].clone()
        if self.world > 1:
            dist.all_reduce(pb, op=dist.ReduceOp.SUM, group=self.group)
        return xb[:self.n_own], vb[:self.n_own], rb[:self.n_own], pb

    # ------------------------------------------------------------------------------------------ migration
    def migrate(self, x, fields):
        """Particles whose position left the slab move to their new owner.  x [n, dim] and every tensor of `fields`
        (n rows each) are returned for the new set of owned particles: the stayers in their old order, then the arrivals
        ordered by source rank.  Collective."""
        own = self.owner(x)
        stay = torch.nonzero(own == self.rank).flatten()
        allf = [x] + list(fields)
        cols2d = [f.reshape(x.shape[0], -1).to(torch.float32) for f in allf]
        widths = [c.shape[1] for c in cols2d]
        packed = torch.cat(cols2d, dim=1)
        out_idx = {p: torch.nonzero(own == p).flatten() for p in range(self.world) if p != self.rank}
        mine = torch.tensor([out_idx[p].numel() if p != self.rank else 0 for p in range(self.world)], dtype=torch.long,
                            device=x.device)
        table = self._all_counts(mine).cpu()                                              # table[src][dst]
        sends = {p: packed[i] for p, i in out_idx.items() if i.numel()}
        recv_rows = {p: int(table[p][self.rank]) for p in range(self.world) if p != self.rank and int(table[p][self.rank])}
        got = self._p2p(sends, recv_rows, packed.shape[1], packed)
        full = torch.cat([packed[stay]] + [got[p] for p in sorted(got)])
        out, c0 = [], 0
        for f, wd in zip(allf, widths):
            col = full[:, c0:c0 + wd].reshape((full.shape[0],) + tuple(f.shape[1:])).contiguous()
            c0 += wd
            out.append(col.to(f.dtype) if f.dtype != torch.float32 else col)
        return out[0], out[1:]
