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


def test_gpus_flag_without_torchrun_starts_n_ranks():
    """`python bench.py --gpus 2` with no WORLD_SIZE in the environment (how the driver ran N = 1 in round 1) must not
    silently measure one rank: bench.py re-executes itself under torch.distributed.run with 2 ranks, rank 0 prints the one
    JSON line with n_gpus = 2 and rank 1 really ran (it reports itself idle in the reference arm)."""
    import bench

    cmd = bench.spawn_command(["--gpus", "3", "--steps", "2"], 3, 29512)
    assert cmd[1:4] == ["-m", "torch.distributed.run", "--nnodes=1"] and "--nproc-per-node=3" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[-4:] == ["--gpus", "3", "--steps", "2"]
    assert os.path.samefile(cmd[cmd.index("29512") + 1], os.path.join(ROOT, "bench.py"))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--impl", "reference", "--workload", "1",
                        "--steps", "1", "--warmup", "0", "--ref-obs", "64"], capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    js = json.loads(lines[0])
    assert js["impl"] == "reference" and js["n_gpus"] == 2
    assert "rank 1 of 2: idle" in r.stderr


def test_slab_range_partitions_every_layer():
    """Host logic of the observation-slab sharding (bench.py --shard obs)."""
    from paper_2209_07944_b200.jefi import slab_range

    for nz in (1, 7, 8, 9, 96, 100, 128):
        for world in (1, 2, 3, 4, 8, 16):
            r = [slab_range(nz, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == nz
            assert all(a[1] == b[0] for a, b in zip(r, r[1:])) and all(a[0] % 8 == 0 for a in r)
            r32 = [slab_range(nz, k, world, edge=32) for k in range(world)]  # x-thin tile geometry: 32-plane layers
            assert r32[0][0] == 0 and r32[-1][1] == nz and all(a[1] == b[0] for a, b in zip(r32, r32[1:])) and all(a[0] % 32 == 0 for a in r32)
    assert [slab_range(96, k, 8) for k in range(8)] == [(0, 8), (8, 24), (24, 32), (32, 48), (48, 56), (56, 72), (72, 80), (80, 96)]


def _slab_worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from paper_2209_07944_b200.jefi import slab_range

    nx, ny, nz = 5, 4, 20
    full = torch.arange(6 * nx * ny * nz, dtype=torch.float32).reshape(6, -1) + 1.0  # what a 1-GPU field step would give
    ranges = [slab_range(nz, r, world) for r in range(world)]  # (0, 8) and (8, 20): unequal slabs, the gather pads the narrow one
    k0, k1 = ranges[rank]
    mine = torch.full_like(full, 123.0)  # stale values outside the slab must not leak into the result
    mine[:, nx * ny * k0:nx * ny * k1] = full[:, nx * ny * k0:nx * ny * k1]
    bench.assemble_slabs(dist, mine, nx * ny, ranges, rank)
    out.put((rank, bool(torch.equal(mine, full))))
    dist.barrier()
    dist.destroy_process_group()


def test_slab_assembly_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_slab_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, True), (1, True)]


def test_deal_range_covers_every_particle_once():
    """Host logic of the sharded PIC step (paper_2209_07944_b200/sharded.py): particles are dealt to ranks in contiguous blocks."""
    import numpy as np

    from paper_2209_07944_b200.sharded import deal_particles, deal_range

    for count in (0, 1, 7, 4096, 1000003):
        for world in (1, 2, 3, 8):
            r = [deal_range(count, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == count and all(a[1] == b[0] for a, b in zip(r, r[1:]))
            assert max(b - a for a, b in r) - min(b - a for a, b in r) <= 1
    part = {"x": np.arange(10.0), "alive": np.ones(10, np.uint8)}
    a, b = deal_particles(part, 0, 2), deal_particles(part, 1, 2)
    assert np.array_equal(np.concatenate([a["x"], b["x"]]), part["x"]) and a["alive"].size == 5
    a["x"][0] = -1.0
    assert part["x"][0] == 0.0  # copies, not views


def _sharded_step_worker(rank: int, world: int, port: int, out):
    """The six stages of ShardedPic.step with a stand-in context that records the calls and does integer-valued 'physics', so the
    exchanges can be checked exactly on CPU tensors: what each rank deposits, that sources are summed, slabs gathered."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2209_07944_b200.jefi import GridSpec, slab_range
    from paper_2209_07944_b200.sharded import ShardedPic

    class FakeCtx:
        def __init__(self):
            self.grid = GridSpec(3, 2, 20, 1.0, 1.0, 1.0, 1.0)
            self.N = self.grid.N
            self.src = torch.zeros((4, self.N))
            self.EB = torch.full((6, self.N), -7.0)
            self.calls = []

        def slab_range(self, r, w):
            return slab_range(self.grid.nz, r, w)

        def deposit(self, part):
            self.calls.append("deposit")
            self.src.zero_()
            self.src[:, part["cell"]] += part["q"]  # each rank's own particles only

        def push_sources(self):
            self.calls.append("push_sources")
            self.pushed = self.src.clone()

        def field_step_slab(self, k0, k1):
            self.calls.append(("slab", k0, k1))
            p = self.grid.nx * self.grid.ny
            comp = torch.arange(6.0).reshape(6, 1)
            self.EB[:, p * k0:p * k1] = self.pushed[0, p * k0:p * k1] * 10.0 + comp  # a function of the SUMMED sources

        def push_particles(self, part):
            self.calls.append("push_particles")
            part["seen_E"] = self.EB[0, part["cell"]].clone()

    ctx = FakeCtx()
    sp = ShardedPic(ctx, dist, rank, world)
    part = {"cell": torch.tensor([5 + rank, 100]), "q": torch.tensor([1.0 + rank, 2.0])}  # cell 100 gets charge from both ranks
    sp.step(part)
    expect_src = torch.zeros(ctx.N)
    expect_src[5], expect_src[6], expect_src[100] = 1.0, 2.0, 4.0
    ok = torch.equal(ctx.pushed[0], expect_src)
    ok &= torch.equal(ctx.EB, expect_src * 10.0 + torch.arange(6.0).reshape(6, 1))  # whole grid, both slabs, on every rank
    ok &= ctx.calls == ["deposit", "push_sources", ("slab",) + slab_range(20, rank, world), "push_particles"]
    ok &= torch.equal(part["seen_E"], torch.tensor([10.0 * (1.0 + rank), 40.0]))  # the push sees fields of cells the OTHER rank solved
    ok &= sp.bytes_per_step == {"all_reduce_rho_J": 16 * ctx.N, "all_gather_E_B": 24 * ctx.N}
    out.put((rank, bool(ok)))
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_pic_step_exchanges_gloo_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_sharded_step_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res == [(0, True), (1, True)]
