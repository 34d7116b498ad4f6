"""The sharded PIC step (paper_2209_07944_b200/sharded.py) with real contexts.

This pool gives one GPU per call, so the two ranks are two PROCESSES on cuda:0 that talk through gloo (which carries CUDA tensors
through the host; NCCL refuses two ranks on one device).  No rank's kernel waits on another rank's: every collective is a host-
side exchange between whole kernels, so sharing one GPU only serialises them.  What is checked is the data path - who deposits
what, that the sources are summed before they enter the ring, that the slabs of E, B reach every rank - against the fp64
oracle's one-domain closed loop, at the bars of tests/test_gpu_parity.py.
"""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

pytestmark = pytest.mark.gpu

STEPS = 10


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _rank(rank: int, world: int, port: int, config: int, out):
    import torch
    import torch.distributed as dist

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2209_07944_b200 import jefi as J
    from paper_2209_07944_b200 import workloads as wl
    from paper_2209_07944_b200.sharded import ShardedPic, deal_particles, deal_range

    w = wl.WORKLOADS[config]
    part = wl.particles(config)
    ctx = J.JefiContext(J.GridSpec(w.n, w.n, w.n, w.dx, w.dx, w.dx, w.dt), device="cuda:0", packed_fields=False)
    mine = {k: torch.from_numpy(np.ascontiguousarray(v)).to(ctx.device) for k, v in deal_particles(part, rank, world).items()}
    sp = ShardedPic(ctx, dist, rank, world)
    for _ in range(STEPS):
        sp.step(mine)
    torch.cuda.synchronize()
    res = {k: v.cpu().numpy() for k, v in mine.items()}
    res.update(rank=rank, EB=ctx.EB.cpu().numpy(), src=ctx.src.cpu().numpy(), impl=ctx.info["field_impl"], ranges=sp.ranges,
               own=deal_range(len(part["x"]), rank, world), step=J.jefi_get_info(ctx.handle)["step"])
    out.put(res)
    dist.barrier()
    ctx.close()
    dist.destroy_process_group()


@pytest.mark.parametrize("config", [1, 2])
def test_two_ranks_closed_loop_against_the_one_domain_oracle(cuda_device, config):
    import torch.multiprocessing as mp

    import oracle
    from oracle import OracleConfig
    from paper_2209_07944_b200 import workloads as wl

    world = 2
    mpc = mp.get_context("spawn")
    q = mpc.Queue()
    port = _free_port()
    procs = [mpc.Process(target=_rank, args=(r, world, port, config, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=600) for _ in procs), key=lambda r: r["rank"])
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    w = wl.WORKLOADS[config]
    part = wl.particles(config)
    cfg = OracleConfig(w.n, w.n, w.n, w.dx, w.dx, w.dx, w.dt)
    orc = oracle.OracleJefi(cfg)
    po = {k: v.astype(np.float64) for k, v in part.items() if k != "alive"}
    po["alive"] = part["alive"].copy()
    for _ in range(STEPS):
        So, Eo, Bo = orc.pic_step(po)
    r0, r1 = res
    assert r0["step"] == r1["step"] == STEPS - 1
    assert r0["ranges"] == r1["ranges"] and r0["ranges"][0][0] == 0 and r0["ranges"][-1][1] == w.n and r0["ranges"][0][1] == r0["ranges"][1][0]
    assert 0 < r0["ranges"][0][1] < w.n  # both ranks really solved a slab
    # every rank ends up with the same sources and the same whole-grid fields, bit for bit
    assert np.array_equal(r0["src"], r1["src"]) and np.array_equal(r0["EB"], r1["EB"])
    for a in range(4):
        assert np.linalg.norm(r0["src"][a] - So[a]) <= 1e-5 * max(np.linalg.norm(So[a]), 1e-300), a
    for name, F, Fo in (("E", r0["EB"][:3], Eo), ("B", r0["EB"][3:], Bo)):
        d = F.astype(np.float64) - Fo
        nrm = np.linalg.norm(Fo)
        assert np.linalg.norm(d) / nrm <= 1e-4, (name, np.linalg.norm(d) / nrm)
        assert np.abs(d).max() / (nrm / np.sqrt(Fo.size)) <= 1e-3, name
    # trajectories: rank r owns the particles [lo, hi) of the one-domain list
    for r in res:
        lo, hi = r["own"]
        both = (r["alive"] == 1) & (po["alive"][lo:hi] == 1)
        assert (r["alive"] != po["alive"][lo:hi]).sum() <= 2 and both.sum() > 0.9 * (hi - lo)
        for k in "xyz":
            assert np.abs(r[k][both] - po[k][lo:hi][both]).max() / w.n <= 1e-5, (r["rank"], k)
    assert res[0]["own"][1] == res[1]["own"][0] and res[1]["own"][1] == len(part["x"])
