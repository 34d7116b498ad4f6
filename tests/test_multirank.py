"""N > 1 host logic of bench.py on CPU (gloo, world size 2): DESIGN.md §9 "replicas only".

The path has no data-path collective; what the ranks share is the timing rule (max over ranks, whole-job rate) and
the rule that under torchrun only rank 0 runs and prints the reference arm.
"""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench

    ms = 10.0 + 5.0 * rank  # rank 1 is the slow one
    dist.barrier()
    mx = bench.max_over_ranks(dist, ms, torch.device("cpu"))
    out.put((rank, mx, bench.aggregate_rate(world, 1e9, mx)))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, mx, rate in res:
        assert mx == 15.0  # every rank sees the slowest rank's time
        assert abs(rate - 2 * 1e9 / 15e-3 / 1e9) < 1e-9  # 2 replicas x 1e9 pairs in 15 ms


def test_single_rank_is_identity():
    import bench

    assert bench.max_over_ranks(None, 3.25, torch.device("cpu")) == 3.25
    assert bench.aggregate_rate(1, 2e9, 1000.0) == 2.0


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--workload", "1",
           "--steps", "1", "--warmup", "0", "--ref-obs", "64"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    js = json.loads(lines[0])
    assert js["impl"] == "reference" and js["n_gpus"] == 2 and js["cpu_baseline"]["kind"] == "oracle"
    assert js["value"] > 0 and js["e2e"]["h2d_bytes_per_step"] == 0 and js["config"]["workload"].startswith("cfg1")
