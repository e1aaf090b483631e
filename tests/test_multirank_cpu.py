"""world_size-2 (and 3) gloo tests (CPU) of the N > 1 paths.  bench.py runs replicas only: its only
collectives are the barrier and the max / sum all-reduces of the timing contract -- covered first.  The sharded path
(paper_2507_21684_b200/sharded.py, slab decomposition with halo exchange) is covered below with the fp64 oracle as the
local solver: the halo bookkeeping is what runs here, the CUDA kernels are covered by the -m gpu tests."""
import json
import os
import socket
import subprocess
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    dist.barrier()
    # rank r took (10 + 5 r) ms for (100 + r) units: the job took the slowest rank's time for the sum of the units
    ms, units = bench.reduce_over_ranks(10.0 + 5.0 * rank, 100 + rank, "cpu")
    from paper_2507_21684_b200 import workloads as W
    wl = bench.make_workload(0, rank)                     # replicas differ by their seed only
    out[rank] = (ms, units, wl.seed, wl.n)
    dist.destroy_process_group()


def test_max_time_and_summed_work_over_two_ranks():
    world, port = 2, _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][:2] == (15.0, 201.0) and res[1][:2] == (15.0, 201.0)
    assert res[0][2] != res[1][2] and res[0][3] == res[1][3]


def test_reference_arm_under_torchrun_prints_one_line_from_rank_0():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--config", "0", "--ref-rows", "256"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = lines[0]
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["value"] > 0


# ------------------------------------------------------------------------------------------ NEXT-4: slab decomposition
class OracleSolver:
    """local solver for the CPU tests of paper_2507_21684_b200.sharded: the fp64 oracle on the local (owned + ghost)
    problem.  Same interface as sharded.CudaSolver."""

    def build(self, domain, x, h, search_scale):
        import oracle
        self.domain, self.x, self.h = domain, x.numpy(), h.numpy()
        self.lists = oracle.neighbors(domain, self.x, self.h, search_scale=search_scale, method=1)
        return int(self.lists[0][-1])

    def density(self, m):
        import oracle
        return torch.from_numpy(oracle.density(self.domain, self.x, self.h, m.numpy(), *self.lists))

    def rhs(self, params, x, v, rho, m, h, kind):
        import oracle
        d, a = oracle.rhs(self.domain, params, x.numpy(), v.numpy(), rho.numpy(), m.numpy(), h.numpy(), kind.numpy(),
                          *self.lists)
        return torch.from_numpy(d), torch.from_numpy(a)

    def rhs_vjp(self, params, x, v, rho, m, h, kind, lam, mu):
        import oracle
        out = oracle.rhs_vjp(self.domain, params, x.numpy(), v.numpy(), rho.numpy(), m.numpy(), h.numpy(), kind.numpy(),
                             *self.lists, lam.numpy(), mu.numpy())
        return tuple(torch.from_numpy(np.asarray(o)) for o in out)


def _sharded_case(name):
    from paper_2507_21684_b200 import workloads as W
    if name == "periodic3d":
        wl = W.perturbed(W.make(3, n_axis=12), amp_x=0.3, amp_rho=0.03)
    elif name == "periodic2d_varh":
        wl = W.perturbed(W.make(1, n_axis=28), amp_x=0.3, amp_rho=0.03)
        rng = np.random.default_rng(3)
        wl.h = (wl.h * np.exp(rng.normal(0, 0.05, size=wl.n))).astype(np.float32)
        wl.domain = W.Domain(dim=2, periodic=wl.domain.periodic, lo=wl.domain.lo, hi=wl.domain.hi,
                             cell_size=float(wl.h.max()) * 1.0001)
        wl.x = (wl.x + np.float32(2.0) * (rng.integers(-1, 2, size=wl.x.shape))).astype(np.float32)   # out-of-box images
    else:
        wl = W.perturbed(W.make(2, dx=0.04), amp_x=0.2, amp_rho=0.01)                  # bounded box, boundary kinds
    return wl


def _sharded_worker(rank, world, port, name, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from paper_2507_21684_b200 import workloads as W
    from paper_2507_21684_b200.sharded import ShardedSph
    torch.set_num_threads(1)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = _sharded_case(name)
    lam, mu = W.random_cotangents(wl)
    sh = ShardedSph(wl.domain, float(wl.h.max()) * 1.0001, OracleSolver())
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a))
    own = sh.select_owned(t(wl.x))
    x, v, rho, m, h, kind = (t(a)[own] for a in (wl.x, wl.v, wl.rho, wl.m, wl.h, wl.kind))
    ghosts = sh.plan(x)
    dens = sh.density(x, m, h)
    drho, acc = sh.rhs(wl.params, x, v, rho, m, h, kind)
    xb, vb, rb, pb = sh.rhs_vjp(wl.params, t(lam)[own], t(mu)[own])
    # migration: push every particle by a quarter of a slab along the cut axis, re-own, and check that nothing is lost
    x2 = x.clone()
    x2[:, sh.axis] += np.float32(0.25 * sh.L / world)
    ids = own.to(torch.float32)
    x3, (ids3, rho3) = sh.migrate(x2, [ids, rho])
    ok_owner = bool((sh.owner(x3) == rank).all())
    out[rank] = dict(own=own.numpy(), ghosts=ghosts, dens=dens.numpy(), drho=drho.numpy(), acc=acc.numpy(), xb=xb.numpy(),
                     vb=vb.numpy(), rb=rb.numpy(), pb=pb.numpy(), ids3=ids3.numpy().astype(np.int64), rho3=rho3.numpy(),
                     ok_owner=ok_owner, axis=sh.axis)
    dist.destroy_process_group()


def _check_sharded(name, world):
    import oracle
    from paper_2507_21684_b200 import workloads as W
    port = _free_port()
    with mp.Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_sharded_worker, args=(world, port, name, out), nprocs=world, join=True)
        res = dict(out)
    wl = _sharded_case(name)
    lam, mu = W.random_cotangents(wl)
    lists = oracle.neighbors(wl.domain, wl.x, wl.h, method=1)
    dens = oracle.density(wl.domain, wl.x, wl.h, wl.m, *lists)
    drho, acc, sd, sa = oracle.rhs(wl.domain, wl.params, wl.x, wl.v, wl.rho, wl.m, wl.h, wl.kind, *lists, with_scales=True)
    xb, vb, rb, pb = oracle.rhs_vjp(wl.domain, wl.params, wl.x, wl.v, wl.rho, wl.m, wl.h, wl.kind, *lists, lam, mu)
    owned = np.concatenate([res[r]["own"] for r in range(world)])
    assert np.array_equal(np.sort(owned), np.arange(wl.n))                 # every particle has exactly one owner
    assert all(sum(res[r]["ghosts"]) > 0 for r in range(world))            # and every rank borrowed some
    # positions are rounded once more when a ghost is shifted by L, so agreement is to binary32 round-off of the box
    # size relative to the summed terms, not bitwise
    def close(key, ref, scale):
        got = np.concatenate([res[r][key] for r in range(world)])
        err = np.max(np.abs(got - ref[owned])) / scale
        if os.environ.get("SPH_VERBOSE"):
            print(name, key, "err", err)
        assert err < 2e-6, (name, key, err)
    close("dens", dens, np.max(np.abs(dens)))
    close("drho", drho, np.max(sd))
    close("acc", acc, np.max(sa))
    close("xb", xb, np.max(np.abs(xb)))
    close("vb", vb, np.max(np.abs(vb)))
    close("rb", rb, np.max(np.abs(rb)))
    for r in range(world):                                                 # the all-reduced parameter gradient, on every rank
        assert np.max(np.abs(res[r]["pb"] - pb) / (np.abs(pb) + 1e-6 * np.max(np.abs(pb)))) < 2e-4, (res[r]["pb"], pb)
    ids = np.concatenate([res[r]["ids3"] for r in range(world)])
    assert np.array_equal(np.sort(ids), np.arange(wl.n)) and all(res[r]["ok_owner"] for r in range(world))
    assert np.array_equal(np.concatenate([res[r]["rho3"] for r in range(world)]), wl.rho[ids])
    assert any(not np.array_equal(np.sort(res[r]["ids3"]), np.sort(res[r]["own"])) for r in range(world))   # some did move


def test_slab_decomposition_two_ranks_periodic_3d():
    _check_sharded("periodic3d", 2)


def test_slab_decomposition_two_ranks_periodic_2d_variable_h_and_out_of_box_positions():
    _check_sharded("periodic2d_varh", 2)


def test_slab_decomposition_two_ranks_bounded_box_with_boundary_kinds():
    _check_sharded("bounded", 2)


def test_slab_decomposition_three_ranks_periodic():
    _check_sharded("periodic2d_varh", 3)
