#!/usr/bin/env python
"""bench.py -- throughput of the delta-SPH hot path on B200 (BASELINE.json config 3 by default).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

One "step" is one pass of the whole hot path (every SURVEY.md 8(a) row) over the current particle state:

    sph_build_cells + sph_neighbors(1.0)      N1-N7  rebuild, exact radius, grid of cell size H
    sph_density                               D
    sph_rhs                                   R0, R1
    sph_rhs_vjp (lambda, mu ~ N(0,1))         R0, B1, B2
    sph_rk_step(dt, skin)                     N1-N7 again on the skin grid, 4 x (R0, R1), T  -> advances the state

`value` = pair interactions per second, a pair interaction being one pair with r < H processed by one pair pass
(self pairs included): per step 7 x nnz(exact list), summed over all ranks, divided by the
max-over-ranks device time.  The RK list carries a Verlet skin; its entries beyond H contribute exactly 0, are no work
of the method and are NOT counted (`value_on_list_entries` = 3 nnz(exact) + 4 nnz(skin) is printed beside it).
The headline loop runs with the library's per-class profiling OFF; `kernels` comes from a second, untimed loop.
The north-star figure "ms per forward+backward RHS step" and its HBM / FP32 fractions sit inside `roofline`
(`ms_fwd_bwd`, `hbm_frac_fwd_bwd`, `hbm_frac_fwd_bwd_of_8TBs`, `fp32_frac_fwd_bwd`).  `roofline.traffic` is NOT
measured in the run: it is the ncu capture named by `roofline.traffic_source` (profiles/traffic.json), printed only
for the workload and layout it was taken on.  `--opt KEY=VALUE` passes sph_set_option knobs (A/B runs, sweeps).

N > 1: the path does not shard in this round ("replicas only"): every rank runs an
independent replica of the workload (different seed), no data-path collective; weak scaling.

--impl reference: the fp64 CPU oracle (oracle/), as it stands, on the host cores, on a bounded sample of rows.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "pair_interactions_per_s"
UNIT = "pair-interactions/s"
from paper_2507_21684_b200.workloads import RK_SKIN as SKIN, rk_domain   # noqa: E402  (input generation only)


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)", float(d.get("sm_max_mhz", 1965.0))
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)", 1965.0


def make_workload(config, seed_shift, n_axis=None):
    from paper_2507_21684_b200 import workloads as W
    wl = W.make(config, n_axis=n_axis) if config != 2 else W.make(config)
    if seed_shift:
        # replicas: same recipe, different random cotangents / jitter stream
        wl.seed += 7919 * seed_shift
    return wl


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)"""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20",
                                       "-i", str(gpu_index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            c = [t.strip() for t in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2])); pw.append(float(c[3]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if c[5 + k].lower().startswith("active"):
                    reasons.add(nm)
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            # under load = samples whose power is above the idle floor; fall back to all samples
            thr = 0.5 * max(pw)
            load = [s for s, p in zip(sm, pw) if p >= thr] or sm
            out = {"sm_mhz": float(np.median(load)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                   "samples": len(sm), "power_w_max": float(max(pw))}
        return out


# --------------------------------------------------------------------------------------------------------------
# algorithmic bytes / flops per launch
FLOP_PER_PAIR = {"rhs": 60.0, "vjp": 170.0, "density": 25.0}     # FMA = 2 flop, MUFU = 1
FP32_LANES_PER_SM, N_SM = 128, 148                               # B200_PROFILING.md / B300_MICROARCH.md unit counts


def algorithmic_bytes(cls, n, nnz, dim, idx_bytes):
    """HBM bytes one launch has to move: the index stream (2 B per entry in the tile-local layout, 4 B in the generic
    one), row_ptr, the per-particle state read once and the outputs written once.  Neighbour state is served from
    shared memory / L2 and is not HBM traffic."""
    state = 40 if dim == 3 else 32                   # sorted SoA s0,s1(,s2) read once per row
    if cls == "rhs":
        return idx_bytes * nnz + 8 * (n + 1) + n * (state + 1 + 16)              # + kind + {a, drho/dt}
    if cls == "vjp":
        return idx_bytes * nnz + 8 * (n + 1) + n * (state + 16 + 16 + 32)        # + cotangents + EOS derivs + {xbar,rhobar},{vbar}
    if cls == "density":
        return idx_bytes * nnz + 8 * (n + 1) + n * (16 + 4 + 4 + 4)              # pos, m, perm, rho
    if cls == "fill":                                # the one-kernel list build: positions in, lists + row_ptr + cnt out
        return idx_bytes * nnz + n * (16 + 8 + 4)
    return None


def measured_traffic(workload, layout_mode):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full captures
    (profiles/traffic.json).  NOT measured in this run: returned with its source, and only for the workload and list
    layout the captures were taken on."""
    p = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        d = json.load(open(p))
    except Exception:
        return {}
    if d.get("workload") != workload or d.get("layout") != layout_mode:
        return {}
    return {k: v for k, v in d.items() if isinstance(v, dict)}


def reduce_over_ranks(ms_local, units_local, device="cpu"):
    """Timing contract for N > 1 (replicas only): the job's time is the MAX over ranks of the
    device time, the job's work the SUM over ranks of the units processed.  Returns (ms_max, units_sum); a plain
    pass-through when torch.distributed is not initialised.  The only collectives of the bench."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(ms_local), float(units_local)
    tt = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    pp = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    dist.all_reduce(pp, op=dist.ReduceOp.SUM)
    return float(tt.item()), float(pp.item())


def cpu_sample(wl, budget_s=12.0, seed=3):
    """The oracle, as it stands, on a bounded sample: forward RHS + VJP of `rows` sampled rows of the workload (lists
    from the oracle's own grid search over all particles, timed separately)."""
    import oracle
    from paper_2507_21684_b200 import workloads as W
    lam, mu = W.random_cotangents(wl)
    t0 = time.perf_counter()
    rp, ci = oracle.neighbors(wl.domain, wl.x, wl.h, method=1)
    t_lists = time.perf_counter() - t0
    rng = np.random.default_rng(seed)

    def run(nrows):
        rows = np.sort(rng.choice(wl.n, size=min(nrows, wl.n), replace=False)).astype(np.int64)
        t0 = time.perf_counter()
        oracle.rhs(wl.domain, wl.params, wl.x, wl.v, wl.rho, wl.m, wl.h, wl.kind, rp, ci, rows=rows)
        oracle.rhs_vjp(wl.domain, wl.params, wl.x, wl.v, wl.rho, wl.m, wl.h, wl.kind, rp, ci, lam, mu, rows=rows)
        dt = time.perf_counter() - t0
        pairs = 2 * int((rp[rows + 1] - rp[rows]).sum())
        return pairs, dt, len(rows)

    pairs, dt, nr = run(20000)                       # calibration
    want = int(min(wl.n, max(20000, 20000 * budget_s / max(dt, 1e-3))))
    pairs, dt, nr, passes = 0, 0.0, 0, 0
    while dt < 0.8 * budget_s and passes < 16:       # a sample capped by the workload size is repeated
        p1, d1, nr = run(want)
        pairs, dt, passes = pairs + p1, dt + d1, passes + 1
    return {"value": pairs / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "note": "the parity oracle as it stands (plain fp64 C, OpenMP over rows), NOT a tuned CPU implementation; it runs "
                    "the two pair passes sph_rhs + sph_rhs_vjp only (no neighbour search, no RK4), so it is a stated "
                    "baseline for the pair-pass rate and no like-for-like ratio to `value` is claimed",
            "sample": f"oracle.rhs + oracle.rhs_vjp (fp64, OpenMP) on {passes} x {nr} sampled rows of {wl.name} "
                      f"({pairs} pair interactions in {dt:.2f} s); oracle grid neighbour search over all "
                      f"{wl.n} particles took {t_lists:.2f} s and is not in the figure"}, (rp, ci)


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores; rank 0 only."""
    if rank != 0:
        return
    import oracle
    from paper_2507_21684_b200 import workloads as W
    wl = make_workload(args.config, 0, args.n_axis)
    lam, mu = W.random_cotangents(wl)
    rp, ci = oracle.neighbors(wl.domain, wl.x, wl.h, method=1)
    rng = np.random.default_rng(11)
    nrows = args.ref_rows

    def step():
        rows = np.sort(rng.choice(wl.n, size=min(nrows, wl.n), replace=False)).astype(np.int64)
        oracle.rhs(wl.domain, wl.params, wl.x, wl.v, wl.rho, wl.m, wl.h, wl.kind, rp, ci, rows=rows)
        oracle.rhs_vjp(wl.domain, wl.params, wl.x, wl.v, wl.rho, wl.m, wl.h, wl.kind, rp, ci, lam, mu, rows=rows)
        return 2 * int((rp[rows + 1] - rp[rows]).sum())

    for _ in range(args.warmup):
        step()
    t0 = time.perf_counter()
    pairs = 0
    for _ in range(args.steps):
        pairs += step()
    dt = time.perf_counter() - t0
    val = pairs / dt
    sample = (f"per step: oracle.rhs + oracle.rhs_vjp (fp64, OpenMP) on {min(nrows, wl.n)} sampled rows of {wl.name}; "
              f"lists prebuilt by the oracle grid search")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "n_particles": wl.n, "dim": wl.dim},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config index (3 = 3D 128^3, the metric's)")
    ap.add_argument("--n-axis", type=int, default=None, help="shrink the lattice (debugging only; invalid as a result)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE",
                    help="sph_set_option before the run (integer keys of include/sph.h, e.g. 9=1: bulk-copy staging of the halo); "
                         "repeatable.  For A/B measurements: the line records it in config.options")
    ap.add_argument("--ref-rows", type=int, default=100000)
    ap.add_argument("--cpu-budget", type=float, default=12.0)
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = max(args.warmup, 0)            # the driver passes W; W >= 3 is the rule for reported numbers

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_2507_21684_b200 import workloads as W
    from paper_2507_21684_b200.binding import Sph

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the SPH library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    wl = make_workload(args.config, rank, args.n_axis)
    dom, dom_rk, par = wl.domain, rk_domain(wl), wl.params
    lam_h, mu_h = W.random_cotangents(wl)
    n, dim = wl.n, wl.dim
    t = lambda a: torch.from_numpy(a).to(dev)
    x, v, rho, m, h, kind = t(wl.x), t(wl.v), t(wl.rho), t(wl.m), t(wl.h), t(wl.kind)
    lam, mu = t(lam_h), t(mu_h)
    dens = torch.empty_like(rho); drho = torch.empty_like(rho); acc = torch.empty_like(v)
    vjp_out = (torch.empty_like(x), torch.empty_like(v), torch.empty_like(rho), torch.empty(10, dtype=torch.float32, device=dev))
    sph = Sph(local_rank, n)
    for kv in args.opt:
        k_, v_ = kv.split("=")
        sph.set_option(int(k_), int(v_))
    ev = lambda: torch.cuda.Event(enable_timing=True)
    phases = ("rebuild", "density", "fwd", "bwd", "rk4")
    marks = []                                       # per timed step: 6 events
    counts = {"nnz": 0, "nnz_rk": 0}

    def step(timed):
        e = [ev() for _ in range(6)] if timed else None
        if timed: e[0].record()
        sph.build_cells(dom, x, h)
        nnz = sph.neighbors(1.0)
        if timed: e[1].record()
        sph.density(m, dens)
        if timed: e[2].record()
        sph.rhs(par, x, v, rho, m, kind, drho, acc)
        if timed: e[3].record()
        sph.rhs_vjp(par, x, v, rho, m, kind, lam, mu, vjp_out)
        if timed: e[4].record()
        sph.rk_step(dom_rk, par, wl.dt, SKIN, x, v, rho, m, h, kind)
        if timed: e[5].record()
        nnz_rk = sph.info()["nnz"]
        if timed:
            marks.append(e)
            counts["nnz"] += nnz
            counts["nnz_rk"] += nnz_rk
        return nnz, nnz_rk

    for _ in range(args.warmup):
        step(False)
    sph.check()
    layout = sph.layout()
    idx_bytes = 2 if layout["mode"] == 2 else 4
    # headline loop: class profiling OFF (its ~60 event records per step stay out of the timed region)
    sph.profile_enable(False)
    launches0 = sph.info()["launches"]
    barrier()
    clocks = ClockSampler(local_rank) if rank == 0 else None
    t_start, t_stop = ev(), ev()
    t_start.record()
    for _ in range(args.steps):
        nnz_last, nnz_rk_last = step(True)
    t_stop.record()
    barrier()
    clk = clocks.stop() if clocks else None
    ms_total = t_start.elapsed_time(t_stop)
    launches = sph.info()["launches"] - launches0
    sph.check()
    # second loop, not part of `value`: per-class device times (sph_profile_enable brackets every launch with events)
    prof_steps = max(1, min(args.steps, 5))
    sph.profile_read()                               # clear accumulators
    sph.profile_enable(True)
    for _ in range(prof_steps):
        step(False)
    torch.cuda.synchronize()
    sph.profile_enable(False)
    prof = sph.profile_read()
    assert torch.isfinite(vjp_out[0]).all() and torch.isfinite(x).all(), "non-finite state after the timed steps"

    # work of a step.  list_entries: CSR entries the seven pair passes walk (3 on the exact list, 4 on the RK list with
    # its Verlet skin).  pairs_in_support: pairs with r < H only -- the entries of the skin list beyond H contribute
    # exactly 0 and are no work of the method; the four RK stages are counted with the exact list's size (the state moves
    # by < 3 % of H within a step).  `value` is quoted on pairs_in_support.
    entries_rank = 3 * counts["nnz"] + 4 * counts["nnz_rk"]
    pairs_rank = 7 * counts["nnz"]
    ph_ms = {p: float(np.mean([mk[i].elapsed_time(mk[i + 1]) for mk in marks])) for i, p in enumerate(phases)}
    fb_ms = ph_ms["fwd"] + ph_ms["bwd"]
    nnz_mean = counts["nnz"] / args.steps

    ms_max, pairs_all = reduce_over_ranks(ms_total, pairs_rank, dev)
    _, entries_all = reduce_over_ranks(ms_total, entries_rank, dev)
    value = pairs_all / (ms_max * 1e-3)

    # ---- NEXT-1 row, outside the timed step: adjoint of the summation density (the paper's
    # own backward benchmark) on the exact-radius list of the current state
    sph.build_cells(dom, x, h)
    nnz_x = sph.neighbors(1.0)
    rb_dev = lam                                          # any cotangent: reuse lambda ~ N(0,1)
    xb_dev, mb_dev = torch.empty_like(x), torch.empty_like(rho)
    sph.density_vjp(m, rb_dev, xb_dev, mb_dev)
    e0, e1 = ev(), ev()
    e0.record()
    for _ in range(5):
        sph.density_vjp(m, rb_dev, xb_dev, mb_dev)
    e1.record()
    torch.cuda.synchronize()
    dvjp_ms = e0.elapsed_time(e1) / 5.0
    extras = {"density_vjp": {"ms": dvjp_ms, "pair_interactions_per_s": nnz_x / (dvjp_ms * 1e-3), "nnz": int(nnz_x),
                              "note": "sph_density_vjp (x_bar and m_bar), not part of the timed step"}}
    # kernel-gradient sum and its adjoint (gradient term of the shifting loss, Eq.24), a = m/rho
    a_dev = (m / rho).contiguous()
    gs_dev, ab_dev = torch.empty_like(x), torch.empty_like(rho)
    # kernel renormalisation (Eq.44/45): L_i and the corrected density gradient, V = m/rho
    L_dev = torch.empty((x.shape[0], x.shape[1], x.shape[1]), dtype=torch.float32, device=x.device)
    for name, call in (("grad_sum", lambda: sph.grad_sum(a_dev, gs_dev)),
                       ("grad_sum_vjp", lambda: sph.grad_sum_vjp(a_dev, mu, xb_dev, ab_dev)),
                       ("renorm_gradient", lambda: sph.renorm_gradient(a_dev, rho, 1e-4, L_dev, gs_dev)),
                       ("renorm_gradient_vjp", lambda: sph.renorm_gradient_vjp(a_dev, rho, mu, 1e-4, xb_dev, mb_dev, ab_dev))):
        call()
        e0, e1 = ev(), ev()
        e0.record()
        for _ in range(5):
            call()
        e1.record()
        torch.cuda.synchronize()
        ms_x = e0.elapsed_time(e1) / 5.0
        extras[name] = {"ms": ms_x, "pair_interactions_per_s": nnz_x / (ms_x * 1e-3), "nnz": int(nnz_x)}

    # ---- e2e: the same step through sph_step_host with pinned host buffers, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        hx, hv, hr = pin(wl.x.copy()), pin(wl.v.copy()), pin(wl.rho.copy())
        hm, hh, hk, hl, hmu = pin(wl.m), pin(wl.h), pin(wl.kind), pin(lam_h), pin(mu_h)
        outs = {"density": pin(np.empty(n, np.float32)), "drho_dt": pin(np.empty(n, np.float32)),
                "acc": pin(np.empty((n, dim), np.float32)), "x_bar": pin(np.empty((n, dim), np.float32)),
                "v_bar": pin(np.empty((n, dim), np.float32)), "rho_bar": pin(np.empty(n, np.float32)),
                "params_bar": pin(np.empty(10, np.float32))}
        h2d = sum(a.numel() * a.element_size() for a in (hx, hv, hr, hm, hh, hk, hl, hmu))
        d2h = sum(a.numel() * a.element_size() for a in outs.values()) + sum(a.numel() * a.element_size() for a in (hx, hv, hr))
        ke = max(3, min(args.steps, 10))
        for _ in range(2):
            sph.step_host(dom, dom_rk, par, wl.dt, SKIN, hx, hv, hr, hm, hh, hk, hl, hmu, outs)
        barrier()
        pairs_e = 0
        t0 = time.perf_counter()
        for _ in range(ke):
            a, b = sph.step_host(dom, dom_rk, par, wl.dt, SKIN, hx, hv, hr, hm, hh, hk, hl, hmu, outs)
            pairs_e += 7 * a                          # pairs in support, as for `value`
        torch.cuda.synchronize()
        dt_e = time.perf_counter() - t0
        te_max, pe_sum = reduce_over_ranks(dt_e, pairs_e, dev)
        assert np.isfinite(outs["params_bar"].numpy()).all()
        e2e = {"value": pe_sum / te_max, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "steps": ke, "ms_per_step": 1e3 * te_max / ke,
               "call": "sph_step_host (pinned host buffers; H2D + whole step + D2H inside the timed region)"}

    if rank == 0:
        hbm, hbm_src, sm_max = peaks()
        kern = {}
        tot_k = sum(ms for ms, _ in prof.values()) or 1.0
        for name, (ms, cnt) in prof.items():
            if cnt:
                kern[name] = {"ms_per_step": ms / prof_steps, "launches_per_step": cnt / prof_steps,
                              "share": ms / tot_k}
        # dominant kernel among the classes with a stated byte model
        cand = [c for c in ("rhs", "vjp", "density", "fill") if c in kern]
        dom_cls = max(cand, key=lambda c: kern[c]["ms_per_step"])
        # algorithmic work per launch is counted on pairs in support (see above), also for the four RK launches
        nnz_for = {"rhs": nnz_mean, "vjp": nnz_mean, "density": nnz_mean,
                   "fill": (counts["nnz"] + counts["nnz_rk"]) / (2.0 * args.steps)}    # entries written per build
        roof = {}
        traffic = measured_traffic(wl.name, layout["mode"])
        fp32_peak = N_SM * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12       # TFLOP/s, FMA = 2 flop
        for c in cand:
            ms_launch = prof[c][0] / max(prof[c][1] / (2 if c == "density" else 1), 1)
            by = algorithmic_bytes(c, n, nnz_for[c], dim, idx_bytes)
            tr = traffic.get(c, {}).get("bytes")
            tr_src = traffic.get(c, {}).get("source")
            hbm_view = {"bound": "hbm", "achieved": by / (ms_launch * 1e-3) / 1e9, "peak": hbm, "unit": "GB/s",
                        "frac": by / (ms_launch * 1e-3) / 1e9 / hbm, "traffic": tr, "traffic_source": tr_src, "kernel": c,
                        "ms_per_launch": ms_launch, "algorithmic_bytes_per_launch": int(by), "peak_source": hbm_src}
            if c in FLOP_PER_PAIR:
                # the pair kernels are bound by FP32 issue / shared-memory gathers, not by HBM (profiles/): their
                # roofline is the plain-ALU one; the HBM view north_star asks for is kept beside it
                fl = FLOP_PER_PAIR[c] * nnz_for[c]
                ach = fl / (ms_launch * 1e-3) / 1e12
                roof[c] = {"bound": "alu", "achieved": ach, "peak": fp32_peak, "unit": "TFLOP/s", "frac": ach / fp32_peak,
                           "traffic": tr, "traffic_source": tr_src, "kernel": c, "ms_per_launch": ms_launch,
                           "algorithmic_flop_per_launch": fl, "flop_per_pair": FLOP_PER_PAIR[c],
                           "peak_source": f"{N_SM} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 flop x {sm_max:.0f} MHz "
                                          "(unit counts of the guides, clocks.max.sm of MEASURED_PEAKS.json)",
                           "hbm": hbm_view}
            else:
                roof[c] = hbm_view
        fb_bytes = algorithmic_bytes("rhs", n, nnz_mean, dim, idx_bytes) + algorithmic_bytes("vjp", n, nnz_mean, dim, idx_bytes)
        fb_flop = (FLOP_PER_PAIR["rhs"] + FLOP_PER_PAIR["vjp"]) * nnz_mean
        # BASELINE.json's metric -- ms per forward+backward RHS step at this config and the fraction of the HBM peak --
        # rides inside `roofline` so that it is part of every parsed record; the FP32 fraction is the binding roof
        # (with 2-byte indices the arithmetic needs 3.5x the time of the bytes)
        fwd_bwd = {"ms_fwd_bwd": fb_ms, "pairs_per_s_fwd_bwd": 2.0 * nnz_mean / (fb_ms * 1e-3),
                   "hbm_frac_fwd_bwd": fb_bytes / (fb_ms * 1e-3) / 1e9 / hbm,
                   "hbm_frac_fwd_bwd_of_8TBs": fb_bytes / (fb_ms * 1e-3) / 1e9 / 8000.0,
                   "fp32_frac_fwd_bwd": fb_flop / (fb_ms * 1e-3) / 1e12 / fp32_peak,
                   "algorithmic_bytes_fwd_bwd": int(fb_bytes), "algorithmic_flop_fwd_bwd": fb_flop}
        roof_main = dict(roof[dom_cls])
        roof_main.update(fwd_bwd)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": wl.name, "n_particles": n, "dim": dim, "nnz_exact_list": int(nnz_last),
                       "nnz_skin_list": int(nnz_rk_last), "skin": SKIN, "replicas": world,
                       "pairs_in_support_per_step": int(pairs_all / args.steps),
                       "list_entries_per_step": int(entries_all / args.steps),
                       "value_counts": "pairs in support (r < H): 7 x nnz of the exact list per step; the RK list's "
                                       "entries beyond H contribute exactly 0 and are not counted",
                       "options": list(args.opt),
                       "list_layout": {1: "generic int32 ids", 2: "tile-local uint16"}[layout["mode"]],
                       "tile_edge_cells": layout["tile_edge"], "tile_halo_max": layout["halo_max"],
                       "step": "build_cells+neighbors, density, rhs, rhs_vjp, rk_step(rebuild + 4 rhs)",
                       "l2": "inputs larger than L2: every pair pass streams its 0.45-0.55 GB list (2 B per entry) and the "
                             "rebuild writes it; per step > 4 GB of list traffic against L2 = 126 MB"},
            "value_on_list_entries": entries_all / (ms_max * 1e-3),
            "ms_fwd_bwd": fb_ms, "pairs_per_s_fwd_bwd": 2.0 * nnz_mean / (fb_ms * 1e-3),
            "hbm_frac_fwd_bwd": fwd_bwd["hbm_frac_fwd_bwd"],
            "hbm_frac_fwd_bwd_of_8TBs": fwd_bwd["hbm_frac_fwd_bwd_of_8TBs"],
            "phase_ms": ph_ms, "kernels": kern, "kernels_note": f"per-class device times from a second loop of {prof_steps} "
            "steps with sph_profile_enable(1); the headline loop runs with profiling off",
            "roofline": roof_main, "roofline_all": roof,
            "gpu_launches": int(launches), "clocks": clk, "next_rows": extras,
        }
        if e2e:
            line["e2e"] = e2e
        if world == 1 and not args.no_cpu:
            wl0 = make_workload(args.config, 0, args.n_axis)
            line["cpu_baseline"], _ = cpu_sample(wl0, args.cpu_budget)
        print(json.dumps(line))
    sph.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
