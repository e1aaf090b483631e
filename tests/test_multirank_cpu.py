"""world_size-2 gloo tests (CPU) of the N > 1 path.  The hot path does not shard in this round ("replicas only",
DESIGN.md section 9): every rank runs an independent replica, and the only collectives are the barrier and the
max / sum all-reduces of bench.py's timing contract -- that logic is what is covered here."""
import json
import os
import socket
import subprocess
import sys

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
