#!/usr/bin/env python
"""bench.py — Jefimenko field-solve throughput on B200 (BASELINE.json metric), one JSON line on stdout.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 4|analytic20|slab251] [--no-pic] [--impl reference]

Product arm: the timed "step" is one pass of the field path over the 96^3 field-only workload (BASELINE.json
configs[3], the one the metric "G source-obs pairs/s and % FP32 peak" is quoted on): jefi_push_sources of a fresh
seeded source slice already resident in HBM + jefi_field_step.  The ring (9.5 GB) is far larger than L2, so no
L2 flush is needed between iterations (workloads whose ring would fit in L2 are timed step by step with a 512 MB fill
in between).  `e2e` repeats it through jefi_field_step_host with pinned HOST buffers.
`pic` adds PIC steps/s (deposit -> push_sources -> field_step -> push_particles) over BASELINE.json's whole runs of configs
1, 2, 3, 5 from t0, and the field-kernel time with the history at full depth;
`paper_workloads` the pairs/s of the paper's own shapes (20^3 at kappa = 6, the 1x251x111 slab); `paper_run` the paper's one
printed whole-run set-up (1x251x111, 1e7 macro-particles, 1e4 steps) as a whole.
Reference arm (--impl reference): the fp64 CPU oracle, as it stands, on a bounded sample of the same workload.
N > 1: one process per GPU.  Under torchrun (WORLD_SIZE set) this process is one rank; without it `--gpus N` re-executes
itself under `python -m torch.distributed.run --nproc-per-node N` so that N ranks really run.  Default for N > 1: `--shard obs`
(DESIGN.md section 9): the observation planes of ONE field step are split over the ranks, E, B are
assembled with an NCCL all-gather, `"scaling": "strong"`; the `pic_sharded` leg runs whole PIC steps that way (particles dealt
to ranks, all-reduce of rho, J, slab solve, all-gather of E, B: paper_2209_07944_b200/sharded.py).  `--shard replicas`: every
rank runs the same workload on its own GPU with no data-path collective (`"scaling": "weak"`).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2209_07944_b200 import workloads as wl  # noqa: E402

# FP32 roofline of the field kernel ("bound": "alu"): 148 SMs x 128 FP32 lanes x 2 FLOP x max SM clock.
N_SM, LANES = 148, 128
FLOP_PER_PAIR = 48.0  # 24 FMA per source-observation pair
# dram__bytes_read.sum + dram__bytes_write.sum of ONE k_field_tiled launch, per (workload, delay rule), each from a committed
# `ncu --set full` capture under profiles/ and valid only for the kernel source it was taken from: the entry names the file
# and the sha1 (first 12 hex digits) of csrc/jefi_field.cu + csrc/jefi_ctx.h of that build.  With a different kernel source
# `traffic` is null and `traffic_source` says the capture is stale.
FIELD_DRAM_BYTES = {
    # (workload name, rule): (bytes, profile, kernel source sha)
    ("cfg4_96c_field_only", "nearest"): (91.143151e9 + 707.036928e6, "profiles/r3b_field_tiled_ncu_full.md", "cece236078a7"),
    ("cfg4_96c_field_only", "linear"): (53.111260e9 + 706.341376e6, "profiles/r3b_field_tiled_ncu_full.md", "cece236078a7"),
}
# From the same captures: how busy the FMA pipe and the shared-memory data pipe were (sm__pipe_fma_cycles_active and
# l1tex__data_pipe_lsu_wavefronts_mem_shared, % of peak sustained elapsed) and the FP32 lane-operations the kernel EXECUTES per
# source-observation pair ((64 FFMA2 + 32 (FFMA + FMUL + FADD)) thread-instructions / pairs).  `roofline.achieved` counts the
# survey's 48 FLOP per pair whatever the kernel executes, so it is an ALGORITHMIC rate: the dyad geometry evaluates distance,
# delay and geometric factors once for two pairs and executes fewer.  These figures say how full the pipes really were.
FIELD_PIPES = {
    ("cfg4_96c_field_only", "nearest"): {"fma_pipe_busy": 0.679, "smem_data_pipe_busy": 0.947, "fp32_lane_ops_per_pair": 20.2},
    ("cfg4_96c_field_only", "linear"): {"fma_pipe_busy": 0.698, "smem_data_pipe_busy": 0.778, "fp32_lane_ops_per_pair": None},
}


def kernel_source_sha() -> str:
    h = hashlib.sha1()
    for f in ("jefi_field.cu", "jefi_ctx.h"):
        with open(os.path.join(ROOT, "paper_2209_07944_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:12]


def field_traffic(name: str, rule: str):
    ent = FIELD_DRAM_BYTES.get((name, rule))
    if ent is None:
        return None, "no ncu --set full capture of this workload / rule under profiles/"
    nbytes, prof, sha = ent
    if sha != kernel_source_sha():
        return None, f"stale: {prof} was captured on kernel source {sha}, this build is {kernel_source_sha()}"
    return nbytes, prof


def field_pipes(name: str, rule: str):
    """Pipe utilisation of the field kernel from the sha-matched ncu capture (None when there is none for this source)."""
    ent = FIELD_DRAM_BYTES.get((name, rule))
    if ent is None or ent[2] != kernel_source_sha():
        return None
    return FIELD_PIPES.get((name, rule))


def log(*a):
    print(*a, file=sys.stderr, flush=True)


class ClockSampler:
    """Samples SM clock and throttle reasons during the timed region (NVML, every 100 ms)."""

    REASONS = {0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x10: "sync_boost",
               0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown",
               0x100: "display_clock_setting"}

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # noqa: BLE001
            log("clock sampler unavailable:", e)
            self.nv = None

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                for bit, name in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:  # noqa: BLE001
                pass
            self._stop.wait(0.1)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def visible_gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:  # noqa: BLE001
            return local_rank
    return local_rank


# --------------------------------------------------------------------------------------------------- reference arm
def oracle_config(w: wl.FieldWorkload, rule: int = 0):
    import oracle

    kw = dict(c=w.c, eps0=w.eps0) if w.c > 0 else {}
    return oracle.OracleConfig(*w.shape, *w.h, w.dt, delay_rule=rule, **kw)


def oracle_sample_rate(w: wl.FieldWorkload, ring_host: np.ndarray, n_obs: int, seed_tag: int, rule: int = 0):
    """Oracle pairs/s on n_obs seeded observation cells against all sources (fp64, all host cores)."""
    import oracle

    cfg = oracle_config(w, rule)
    obs = np.random.default_rng([w.seed, seed_tag]).integers(0, w.N, size=n_obs, dtype=np.int64)
    t0 = time.perf_counter()
    oracle.field(cfg, w.H - 1, ring_host, obs)
    dt = time.perf_counter() - t0
    return n_obs * (w.N - 1) / dt, dt


def host_ring(w: wl.FieldWorkload) -> np.ndarray:
    ring = np.empty((w.H, 4, w.N), dtype=np.float32)
    for t in range(w.H):
        ring[t] = w.slice(t)
    return ring


def workload_config(w: wl.FieldWorkload, rule: str) -> dict:
    """The `config` object both arms print (same keys, so that the driver can match the two lines)."""
    ring_gb = 32.0 * w.H * w.N / 1e9  # the device ring of the product arm (32 B per cell-slot, before tile padding)
    return {"workload": w.name, "grid": list(w.shape), "H": w.H, "dx": w.h[0], "dt": w.dt, "kappa": round(w.kappa, 6),
            "pairs_per_step": float(w.N) * float(w.N - 1), "delay_rule": rule,
            "l2": (f"inputs ({ring_gb:.1f} GB ring) larger than L2, no flush" if not ring_needs_flush(32 * w.H * w.N)
                   else "512 MB fill between timed steps")}


def ring_needs_flush(ring_bytes: float) -> bool:
    """Inputs larger than L2 need no flush; a ring that would (nearly) fit in the 126 MB L2 is flushed between timed steps."""
    return ring_bytes < 512 * 1024 * 1024


def run_reference(args, w: wl.FieldWorkload) -> dict:
    import oracle

    cores = oracle.num_threads()
    log(f"[reference] building the {w.H}-slot host history of {w.name} ...")
    ring = host_ring(w)
    n_obs = min(args.ref_obs, w.N)
    rates = []
    for i in range(args.warmup + args.steps):
        r, dt = oracle_sample_rate(w, ring, n_obs, i, 1 if args.delay_rule == "linear" else 0)
        log(f"[reference] step {i}: {n_obs} obs cells x {w.N - 1} sources in {dt:.2f} s -> {r / 1e9:.4f} Gpairs/s")
        if i >= args.warmup:
            rates.append((r, dt))
    tot_pairs = sum(r * dt for r, dt in rates)
    tot_t = sum(dt for _, dt in rates)
    val = tot_pairs / tot_t / 1e9
    sample = f"{n_obs} seeded observation cells x all {w.N - 1} source cells per step (of {w.N} cells)"
    return {"impl": "reference", "metric": "jefimenko_source_obs_pairs_per_s", "value": val, "unit": "Gpairs/s",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / len(rates),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(w, args.delay_rule),
            "cpu_baseline": {"value": val, "unit": "Gpairs/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": "Gpairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


# --------------------------------------------------------------------------------------------------- product arm
def max_over_ranks(dist, ms: float, device) -> float:
    """Multi-GPU timing rule: a step takes as long as the slowest rank (all-reduce MAX; identity at world size 1)."""
    import torch

    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def assemble_slabs(dist, EB, plane: int, ranges, rank: int) -> None:
    """--shard obs: rank r has computed the observation planes ranges[r] = [k0, k1) of EB ([6][N], plane = nx*ny cells per
    z-plane); one all-gather over the slabs (24 N bytes per rank) leaves every rank with the whole E, B."""
    from paper_2209_07944_b200.sharded import gather_slabs

    gather_slabs(dist, EB, plane, ranges, rank)


def aggregate_rate(world: int, pairs_per_rank: float, ms_max: float) -> float:
    """Whole-job Gpairs/s: every rank processed pairs_per_rank pairs (replicas) in ms_max."""
    return world * pairs_per_rank / (ms_max * 1e-3) / 1e9


def time_pic_sharded(J, torch, device, dist, rank: int, world: int, config: int, steps: int, warmup: int) -> dict:
    """Whole PIC steps of one config over `world` ranks (paper_2209_07944_b200/sharded.py): particles dealt
    to the ranks, per step one all-reduce of rho, J (16 N bytes) and one all-gather of E, B (24 N bytes), each rank solving its
    observation slab.  `steps` steps from t0 on a fresh context, CUDA events on every rank, max over ranks.  Every rank calls this."""
    from paper_2209_07944_b200.sharded import ShardedPic, deal_particles

    w = wl.WORKLOADS[config]
    mine0 = deal_particles(wl.particles(config), rank, world)

    def run(nsteps: int):
        ctx = J.JefiContext(J.GridSpec(w.n, w.n, w.n, w.dx, w.dx, w.dx, w.dt), device=device, packed_fields=False)
        dp = {k: torch.from_numpy(np.ascontiguousarray(v)).to(device) for k, v in mine0.items()}
        sp = ShardedPic(ctx, dist, rank, world)
        dist.barrier()
        torch.cuda.synchronize(device)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(nsteps):
            sp.step(dp)
        e1.record()
        dist.barrier()
        torch.cuda.synchronize(device)
        alive = dp["alive"].sum().to(torch.float64).reshape(1)
        dist.all_reduce(alive)
        res = (e0.elapsed_time(e1), int(alive.item()), sp.ranges, sp.bytes_per_step, ctx.info["field_impl"])
        ctx.close()
        return res

    run(warmup)
    ms, alive, ranges, nbytes, impl = run(steps)
    ms = max_over_ranks(dist, ms, device)
    return {"workload": w.name, "ranks": world, "steps": steps, "from": "t0", "total_ms": ms, "steps_per_s": 1e3 * steps / ms,
            "alive_at_end": alive, "slabs": ranges, "bytes_per_step_per_rank": nbytes, "field_impl": impl,
            "how": "ShardedPic.step: deposit, all-reduce(rho, J), push_sources, field_step_slab, all-gather(E, B), push_particles"}


def time_pic(J, torch, device, config: int, steps: int, warmup: int) -> dict:
    """PIC steps/s of one config through JefiContext.pic_step = jefi_pic_step: on its own (non-default) stream, so that a step
    is ONE CUDA-graph launch (deposit, history push, field solve with packed E/B output, particle push), particles re-sorted
    by cell every 8 steps.  CUDA events on that stream.
    `steps` = BASELINE.json's run length for the config, FROM t0 (a fresh context: empty history).  The field kernel skips
    tile pairs whose whole slot window lies before t0 (their sources are exactly zero), so a step costs what its
    light cone holds: the whole run is timed (`steps_per_s`, the figure SURVEY.md section 8(d)(4) asks for), the last step alone
    (`last_step_ms`), and one field step with the history filled to its full depth (`field_kernel_ms_full_history`: the rate a
    run longer than H steps settles at).  `warmup` steps run first on a throw-away context (graph capture, module load)."""
    w = wl.WORKLOADS[config]
    side = torch.cuda.Stream(device)
    with torch.cuda.stream(side):
        if warmup > 0:
            wctx = J.JefiContext(J.GridSpec(w.n, w.n, w.n, w.dx, w.dx, w.dx, w.dt), device=device, sort_every=8)
            wpart = {k: torch.from_numpy(v).to(device) for k, v in wl.particles(config).items()}
            for _ in range(warmup):
                wctx.pic_step(wpart)
            side.synchronize()
            wctx.close()
            del wpart
        ctx = J.JefiContext(J.GridSpec(w.n, w.n, w.n, w.dx, w.dx, w.dx, w.dt), device=device, sort_every=8)
        part = {k: torch.from_numpy(v).to(device) for k, v in wl.particles(config).items()}
        side.synchronize()
        evs = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
        l0 = ctx.launch_count()
        evs[0].record(side)
        for i in range(steps):
            ctx.pic_step(part)
            evs[i + 1].record(side)
        side.synchronize()
        total_ms = evs[0].elapsed_time(evs[steps])
        per_step = [evs[i].elapsed_time(evs[i + 1]) for i in range(steps)]
        launches = ctx.launch_count() - l0
        alive = int(part["alive"].sum().item())
        # the field kernel alone with the history at full depth: H more pushes of the last deposited sources, then timed steps
        for _ in range(ctx.H):
            ctx.push_sources()
        kms = []
        for _ in range(2):
            ctx.push_sources()
            ctx.field_step()
            kms.append(ctx.last_field_kernel_ms())
        side.synchronize()
    full_ms = float(np.mean(kms))
    out = {"workload": w.name, "steps": steps, "from": "t0 (empty history)", "warmup": warmup, "total_ms": total_ms,
           "ms_per_step": total_ms / steps, "steps_per_s": 1e3 * steps / total_ms, "first_step_ms": per_step[0], "last_step_ms": per_step[-1],
           "particles": int(part["x"].numel()), "alive_at_end": alive, "H": ctx.H,
           "field_kernel_ms_full_history": full_ms,
           "launches": launches, "graph": "one CUDA-graph launch per step (jefi_pic_step)", "field_impl": ctx.info["field_impl"], "tiles": ctx.tile_info}
    ctx.close()
    return out


# Table 1 of the paper, JefiPIC column: step -> (maximum displacement / m, maximum velocity / (m/s)) at 0.4 and 0.6 ns
TABLE1 = {4000: (8.43e-4, 2.20e6), 6000: (1.29e-3, 2.25e6)}


def time_paper_run(J, torch, device, count: int = 10_000_000, steps: int = 10_000) -> dict:
    """The one whole-run time the paper prints for the method (section 3.3.2): the planar
    emission in a 10 T B_y on 1 x 251 x 111 cells, dx = 1e-5 m, dt = 1e-13 s, 1 ns = 1e4 steps, 1e7 macro-particles, "within only
    half an hour" on one A100 in fp64.  The same set-up (seeded stand-in for the unknown initial placement, reading A23) through
    jefi_pic_step, timed as a whole with CUDA events: context only, another machine and precision."""
    w = wl.SLABS["planar_emission"]
    nx, ny, nz = w.shape
    side = torch.cuda.Stream(device)
    with torch.cuda.stream(side):
        ctx = J.JefiContext(J.GridSpec(nx, ny, nz, w.dx, w.dx, w.dx, w.dt, Bext=w.Bext), device=device, sort_every=8)
        part = {k: torch.from_numpy(v).to(device) for k, v in wl.slab_particles("planar_emission", count).items()}
        part["tag"] = torch.arange(count, dtype=torch.int32, device=device)  # permuted along by the cell sort: particle identity
        y0 = part["y"].clone()
        side.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        table1 = {}
        e0.record(side)
        for i in range(steps):
            ctx.pic_step(part)
            if i + 1 in TABLE1:  # the paper's two read-out times (Table 1), with the paper's own particle count
                al = part["alive"].bool()
                dy = (part["y"][al].double() - y0[part["tag"][al].long()].double()).max() * w.dx
                u = [part[k][al].double() for k in ("ux", "uy", "uz")]
                vy = (u[1] / (1 + u[0] ** 2 + u[1] ** 2 + u[2] ** 2).sqrt()).max() * wl.C_SI
                table1[i + 1] = (dy, vy)  # device scalars: read back after the timed region
        e1.record(side)
        side.synchronize()
        ms = e0.elapsed_time(e1)
        alive = int(part["alive"].sum().item())
        # what a step of this workload is made of: 200 further steps through the five individual calls
        # (the graph's contents, issued one by one) with a CUDA event between calls; the state is the run's own at its end
        names = ("sort_every_8", "deposit", "push_sources", "field_step_packed", "push_particles_packed")
        tot = {k: 0.0 for k in names}
        bsteps = 200
        evs = []
        for i in range(bsteps):
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(6)]
            ev[0].record(side)
            if i % 8 == 0:
                ctx.sort_particles(part)
            ev[1].record(side)
            ctx.deposit(part)
            ev[2].record(side)
            ctx.push_sources()
            ev[3].record(side)
            ctx.field_step_packed()
            ev[4].record(side)
            ctx.push_particles_packed(part)
            ev[5].record(side)
            evs.append(ev)
        side.synchronize()
        for ev in evs:
            for j, k in enumerate(names):
                tot[k] += ev[j].elapsed_time(ev[j + 1])
        breakdown = {k: v / bsteps for k, v in tot.items()}
        breakdown["sum_ms_per_step"] = sum(tot.values()) / bsteps
        breakdown["how"] = f"{bsteps} steps after the run, the five C-ABI calls issued one by one on the same stream, CUDA events between them (ms per step)"
    out = {"workload": w.name, "grid": [nx, ny, nz], "particles": count, "steps": steps, "simulated_ns": steps * w.dt * 1e9,
           "total_s": ms * 1e-3, "steps_per_s": 1e3 * steps / ms, "alive_at_end": alive, "field_impl": ctx.info["field_impl"], "tiles": ctx.tile_info,
           "ms_per_call": breakdown,
           "table1": {f"{k * w.dt * 1e9:.1f} ns": {"max_displacement_m": float(d), "paper_jefipic_m": TABLE1[k][0], "ratio": float(d) / TABLE1[k][0],
                                                   "max_vy_m_per_s": float(v), "paper_jefipic_m_per_s": TABLE1[k][1], "ratio_v": float(v) / TABLE1[k][1]}
                      for k, (d, v) in table1.items()},
           "paper": "JefiPIC: 'within only half an hour' on one A100, fp64 (PAPER.md:372); UNIPIC: 'over 6 hours' on a Xeon workstation"}
    ctx.close()
    return out


def hbm_peak_gbs():
    """Measured HBM copy bandwidth of this pool's B200s (MEASURED_PEAKS.json, driver-written), else the guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "of measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:  # noqa: BLE001
        return 6650.0, "of fallback (B200_PROFILING.md, 6.65 TB/s)"


def time_particle_kernels(J, torch, device, config: int = 5, reps: int = 5) -> dict:
    """HBM roofline of the particle kernels: jefi_deposit (direct and cell-sorted) and
    jefi_push_particles on the particle set of a config (default 5: 8e6 macro-particles on 128^3), each call timed
    alone with CUDA events.  The context uses H = 2 (these kernels never touch the ring); E, B are seeded random
    fields scaled so that nothing leaves the grid.  Particle arrays (232 MB) exceed L2; a 512 MB fill between
    repetitions flushes it anyway.  Algorithmic bytes per call are stated in DESIGN.md §6.3-6.4."""
    w = wl.WORKLOADS[config]
    part_h = wl.particles(config)
    P, N = int(part_h["x"].shape[0]), w.N
    peak, peak_src = hbm_peak_gbs()
    flush = torch.empty(128 * 1024 * 1024, dtype=torch.float32, device=device)
    g = torch.Generator(device=device)
    g.manual_seed(w.seed)
    out = {"workload": w.name + "_particles", "particles": P, "grid": [w.n] * 3, "hbm_peak_gbs": peak, "peak_source": peak_src,
           "l2": "512 MB fill between repetitions", "kernels": {}}

    def timed(fn):
        ms = []
        for _ in range(reps + 1):
            flush.fill_(1.0)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            torch.cuda.synchronize(device)
            ms.append(e0.elapsed_time(e1))
        return float(np.median(ms[1:]))

    def entry(ms, nbytes, launches):
        return {"ms": ms, "algorithmic_bytes": nbytes, "gbs": nbytes / (ms * 1e-3) / 1e9, "frac": nbytes / (ms * 1e-3) / 1e9 / peak,
                "mparticles_per_s": P / (ms * 1e-3) / 1e6, "launches_per_call": launches}

    EB = (torch.rand((6, N), device=device, generator=g) - 0.5)
    EB[:3] *= 1e3   # V/m: u changes by ~1e-7 per step, nobody leaves
    EB[3:] *= 1e-3  # tesla
    dep_bytes = 29.0 * P + 32.0 * N   # 7 floats + alive per particle; zero-fill and final write-back of the four grids
    push_bytes = 53.0 * P + 24.0 * N  # 29 B read + 24 B written per particle; every field value read at least once
    ctxs = {m: J.JefiContext(J.GridSpec(w.n, w.n, w.n, w.dx, w.dx, w.dx, w.dt, H=2), device=device,
                             field_impl=J.JEFI_FIELD_REFERENCE, deposit_mode=getattr(J, "JEFI_DEPOSIT_" + m))
            for m in ("DIRECT", "RUNS", "SORTED")}
    part = {k: torch.from_numpy(v).to(device) for k, v in part_h.items()}
    for order in ("caller_order", "cell_sorted"):
        if order == "cell_sorted":
            c0 = ctxs["RUNS"]
            scratch = {k: v.clone() for k, v in part.items()}
            c0.sort_particles(scratch)  # allocates the scratch
            l0 = c0.launch_count()
            ms = timed(lambda: c0.sort_particles(part))
            # keys 13 B in + 8 out; scatter 8 in + 4 out; gather 4 + 37 in, 37 out; copy back 37 in + 37 out
            out["kernels"]["sort_particles"] = entry(ms, 222.0 * P, (c0.launch_count() - l0) // (reps + 1))
            del scratch
        for m, extra in (("DIRECT", 0.0), ("RUNS", 0.0), ("SORTED", 41.0)):
            if order == "cell_sorted" and m == "SORTED":
                continue
            ctx = ctxs[m]
            l0 = ctx.launch_count()
            ms = timed(lambda: ctx.deposit(part))
            out["kernels"][f"deposit_{m.lower()}_{order}"] = entry(ms, dep_bytes + extra * P, (ctx.launch_count() - l0) // (reps + 1))
        pp = {k: v.clone() for k, v in part.items()}
        ms = timed(lambda: ctxs["RUNS"].push_particles(pp, EB))
        out["kernels"][f"push_{order}"] = entry(ms, push_bytes, 1)
        del pp
    for ctx in ctxs.values():
        ctx.close()
    del part
    del flush
    torch.cuda.empty_cache()
    return out


def fp32_peak_tflops(sm_max_mhz) -> float:
    return N_SM * LANES * 2 * (sm_max_mhz or 1965.0) * 1e6 / 1e12


def time_field_workload(J, torch, device, w: wl.FieldWorkload, rule: str, steps: int, warmup: int, sm_max_mhz) -> dict:
    """pairs/s of one field-only workload on one GPU (the `paper_workloads` leg): H pushes fill the history, then `steps`
    steps of jefi_push_sources + jefi_field_step, each timed with its own CUDA events; the ring of these small grids would
    fit in L2, so a 512 MB fill runs between steps."""
    ctx = J.JefiContext(J.GridSpec(*w.shape, *w.h, w.dt, c=w.c, eps0=w.eps0), device=device,
                        delay_rule=J.JEFI_DELAY_LINEAR if rule == "linear" else J.JEFI_DELAY_NEAREST)
    for t in range(w.H):
        ctx.push_sources(torch.from_numpy(w.slice(t)).to(device))
    fresh = [torch.from_numpy(w.slice(w.H + i)).to(device) for i in range(4)]
    flush = torch.empty(128 * 1024 * 1024, dtype=torch.float32, device=device)
    ms, kms = [], []
    for i in range(warmup + steps):
        flush.fill_(float(i))
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        ctx.push_sources(fresh[i % 4])
        ctx.field_step()
        e1.record()
        torch.cuda.synchronize(device)
        if i >= warmup:
            ms.append(e0.elapsed_time(e1))
            kms.append(ctx.last_field_kernel_ms())
    pairs = float(w.N) * float(w.N - 1)
    step_ms, kernel_ms = float(np.mean(ms)), float(np.mean(kms))
    peak = fp32_peak_tflops(sm_max_mhz)
    achieved = FLOP_PER_PAIR * pairs / (kernel_ms * 1e-3) / 1e12
    out = {"config": workload_config(w, rule), "value": pairs / (step_ms * 1e-3) / 1e9, "unit": "Gpairs/s", "ms_per_step": step_ms,
           "steps": steps, "warmup": warmup, "l2": "512 MB fill between steps",
           "field_impl": ctx.info["field_impl"], "field_impl_reason": ctx.info["field_impl_reason"], "tiles": ctx.tile_info,
           "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                        "kernel_ms": kernel_ms, "peak_source": PEAK_SOURCE}}
    ctx.close()
    del flush
    return out


PEAK_SOURCE = ("of derived: 148 SM x 128 FP32 lanes x 2 FLOP x clocks.max.sm (MEASURED_PEAKS.json has no FP32 figure; the FFMA-chain "
               "probe of this run is in peak_measured, the derived figure is the larger, i.e. conservative, denominator)")


def run_product(args, w: wl.FieldWorkload) -> dict:
    import torch

    from paper_2209_07944_b200 import jefi as J

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    device = torch.device(f"cuda:{local}")
    torch.cuda.set_device(device)
    dist = None
    if world > 1 or "TORCHELASTIC_RUN_ID" in os.environ:  # under torchrun NCCL is initialised even with one rank (plumbing check)
        import torch.distributed as dist

        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("NCCL_DEBUG", "INFO")  # the rank count is visible in the log
        dist.init_process_group("nccl", device_id=device)
    J.load_library()

    ctx = J.JefiContext(J.GridSpec(*w.shape, *w.h, w.dt, c=w.c, eps0=w.eps0), device=device,
                        delay_rule=J.JEFI_DELAY_LINEAR if args.delay_rule == "linear" else J.JEFI_DELAY_NEAREST)
    N, H = w.N, ctx.H
    assert H == w.H
    keep_host = (rank == 0 and not args.no_cpu_baseline)  # rank 0 times the oracle at every N (after the timed region; the other ranks wait)
    ring_host = np.empty((H, 4, N), dtype=np.float32) if keep_host else None
    log(f"[rank {rank}/{world}] {w.name}: N={N} H={H} ring={ctx.info['ring_bytes'] / 1e9:.2f} GB; {ctx.info['field_impl_reason']}")
    t0 = time.perf_counter()
    for t in range(H):  # fill the history so that every delay is valid at the timed steps
        s = w.slice(t)
        if keep_host:
            ring_host[t] = s
        ctx.push_sources(torch.from_numpy(s).to(device, non_blocking=False))
    torch.cuda.synchronize(device)
    log(f"[rank {rank}] history filled in {time.perf_counter() - t0:.1f} s")

    nfresh = args.warmup + args.steps
    fresh = [torch.from_numpy(w.slice(H + i)).to(device) for i in range(min(nfresh, 8))]
    pairs = float(N) * float(N - 1)
    # inputs larger than L2 need no flush; a ring that would (nearly) fit in the 126 MB L2 is flushed between steps
    need_flush = ring_needs_flush(32 * H * N)  # the same rule workload_config() states in `config.l2` (both arms print it)
    flush = torch.empty(128 * 1024 * 1024, dtype=torch.float32, device=device) if need_flush else None

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(device)

    # --shard obs (N > 1): every rank holds the whole history and solves its slab of observation planes, then E, B are
    # assembled over NVLink (strong scaling of ONE field step).  Default: replicas.
    shard = args.shard == "obs" and dist is not None
    nz = w.shape[2]
    ranges = [ctx.slab_range(r, world) for r in range(world)] if shard else [(0, nz)]
    k0, k1 = ranges[rank] if shard else (0, nz)
    plane = w.shape[0] * w.shape[1]

    def field_step():
        if shard:
            ctx.field_step_slab(k0, k1)
            assemble_slabs(dist, ctx.EB, plane, ranges, rank)
        else:
            ctx.field_step()

    # ---- device-resident timing ----
    for i in range(args.warmup):
        ctx.push_sources(fresh[i % len(fresh)])
        field_step()
    barrier()
    sampler = ClockSampler(visible_gpu_index(local))
    sampler.start()
    l0 = ctx.launch_count()
    barrier()
    if not need_flush:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for i in range(args.steps):
            ctx.push_sources(fresh[(args.warmup + i) % len(fresh)])
            field_step()
        e1.record()
        barrier()
        step_ms = e0.elapsed_time(e1) / args.steps
    else:
        evs = []
        for i in range(args.steps):
            flush.fill_(float(i))
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.push_sources(fresh[(args.warmup + i) % len(fresh)])
            field_step()
            e1.record()
            evs.append((e0, e1))
        barrier()
        step_ms = float(np.mean([a.elapsed_time(b) for a, b in evs]))
    clocks = sampler.stop()
    launches = ctx.launch_count() - l0
    # per-launch duration of the dominant kernel FROM THE TIMED LAUNCHES: the library records CUDA events on its stream around
    # the field kernel of every step (it keeps the last 64); they are read back here, after the timed region
    kms = [ctx.field_kernel_ms(i) for i in range(min(args.steps, 64))]
    kernel_ms = float(np.mean(kms))
    step_ms_max = max_over_ranks(dist, step_ms, device)
    value = aggregate_rate(1 if shard else world, pairs, step_ms_max)  # sharded: the job is ONE step of N^2 pairs
    pairs_per_launch = pairs * (k1 - k0) / nz if shard else pairs

    # ---- end to end through the C-ABI with host buffers ----
    src_pin = torch.empty(4 * N, dtype=torch.float32).pin_memory()
    eb_pin = torch.empty(6 * N, dtype=torch.float32).pin_memory()
    src_pin.copy_(torch.from_numpy(w.slice(H + 100).reshape(-1)))
    J.jefi_field_step_host(ctx.handle, N, src_pin, eb_pin)  # warm-up (allocates the staging buffers)
    barrier()
    e2e_steps = max(1, min(args.steps, 3))
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        J.jefi_field_step_host(ctx.handle, N, src_pin, eb_pin)
    torch.cuda.synchronize(device)
    e2e_ms = (time.perf_counter() - t0) * 1e3 / e2e_steps
    e2e_ms_max = max_over_ranks(dist, e2e_ms, device)
    e2e_val = aggregate_rate(1 if shard else world, pairs, e2e_ms_max)  # sharded runs: one rank's own full step
    checksum = float(eb_pin[:N].double().abs().sum())

    # measured FP32 pipe throughput of this GPU, in this run (scalar FFMA chains and packed FFMA2 chains)
    probe = ({"ffma": J.jefi_debug_fp32_peak(ctx.handle, 0), "ffma2": J.jefi_debug_fp32_peak(ctx.handle, 1),
              "ffma_3reg": J.jefi_debug_fp32_peak(ctx.handle, 2), "ffma2_3reg": J.jefi_debug_fp32_peak(ctx.handle, 3)} if rank == 0 else None)
    lds = ({k: J.jefi_debug_lds128_cycles(ctx.handle, i) for i, k in enumerate(("broadcast", "lane_pairs_share", "32_rows", "one_pair_differs",
                                                                                "pairs_share_rows_8_apart"))} if rank == 0 else None)
    impl, reason, tiles, ring_bytes = ctx.info["field_impl"], ctx.info["field_impl_reason"], ctx.tile_info, ctx.info["ring_bytes"]
    ctx.close()
    del flush
    torch.cuda.empty_cache()

    pic_sharded = None
    if dist is not None and shard and not args.no_pic:  # every rank takes part; BASELINE.json's config 3 for its 200 steps from t0
        pic_sharded = time_pic_sharded(J, torch, device, dist, rank, world, 3, 200, 3)

    out = None
    if rank == 0:
        sm_max = clocks.get("sm_max_mhz") or 1965.0
        peak = fp32_peak_tflops(sm_max)
        achieved = FLOP_PER_PAIR * pairs_per_launch / (kernel_ms * 1e-3) / 1e12
        traffic, traffic_src = field_traffic(w.name, args.delay_rule)
        cfg = workload_config(w, args.delay_rule)  # identical in both arms; what only this arm has goes to `launch`
        launch = {"parallelism": ("obs_slabs" if shard else "replicas") if dist is not None else "single", "field_impl": impl,
                  "field_impl_reason": reason, "tiles": tiles, "ring_bytes": ring_bytes}
        pipes = field_pipes(w.name, args.delay_rule)
        out = {"metric": "jefimenko_source_obs_pairs_per_s", "value": value, "unit": "Gpairs/s", "n_gpus": world,
               "steps": args.steps, "warmup": args.warmup, "ms_per_step": step_ms_max, "higher_is_better": True,
               "scaling": "strong" if shard else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
               "config": cfg, "launch": launch,
               "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                            "traffic": traffic, "traffic_source": traffic_src,
                            "achieved_kind": "algorithmic: 48 FLOP (24 FMA, SURVEY.md 8(d)) per source-observation pair x pairs / kernel time, "
                                             "whatever the kernel executes; fma_pipe_busy is the pipe's own utilisation",
                            "fma_pipe_busy": pipes["fma_pipe_busy"] if pipes else None,
                            "smem_data_pipe_busy": pipes["smem_data_pipe_busy"] if pipes else None,
                            "fp32_lane_ops_per_pair_executed": pipes["fp32_lane_ops_per_pair"] if pipes else None,
                            "kernel": "k_field_tiled" if impl == 2 else "k_field_reference",
                            "kernel_ms": kernel_ms, "kernel_ms_source": f"CUDA events around the field kernel of the {len(kms)} timed steps",
                            "flop_per_pair": FLOP_PER_PAIR, "peak_source": PEAK_SOURCE, "kernel_source_sha": kernel_source_sha(),
                            "peak_measured": {"ffma_tflops": probe["ffma"]["tflops"], "ffma2_tflops": probe["ffma2"]["tflops"],
                                              "ffma_3reg_tflops": probe["ffma_3reg"]["tflops"], "ffma2_3reg_tflops": probe["ffma2_3reg"]["tflops"],
                                              "sm_count": probe["ffma"]["sm_count"],
                                              "how": "jefi_debug_fp32_peak: 2048 threads/SM x 16 independent FMA chains, CUDA events, best of 3; ffma/ffma2: multiplier "
                                                     "and addend shared by the chains, *_3reg: three registers of its own per FMA (register-file bound)",
                                              "frac_of_measured": achieved / max(probe["ffma"]["tflops"], probe["ffma2"]["tflops"])}},
               "smem_probe": {"lds128_sm_cycles": lds, "how": "jefi_debug_lds128_cycles: 16 warps/SM issuing LDS.128 only, rows per lane as named; "
                                     "the field kernel issues 2 LDS.128 per source-observation pair"},
               "e2e": {"value": e2e_val, "unit": "Gpairs/s", "h2d_bytes_per_step": 16 * N, "d2h_bytes_per_step": 24 * N,
                       "ms_per_step": e2e_ms_max, "checksum_abs_ex": checksum},
               "gpu_launches": int(launches), "clocks": clocks}
        if pic_sharded is not None:
            out["pic_sharded"] = pic_sharded
        if not args.no_pic and world == 1:
            out["pic"] = []
            for cfgno, st, wu in ((1, 64, 3), (2, 100, 3), (3, 200, 3), (5, 50, 2)):  # BASELINE.json's run lengths
                try:
                    out["pic"].append(time_pic(J, torch, device, cfgno, st, wu))
                except Exception as e:  # noqa: BLE001
                    out["pic"].append({"workload": wl.WORKLOADS[cfgno].name, "error": str(e)})
            out["paper_workloads"] = []
            for key in ("analytic20", "slab251"):
                if wl.field_workload(key).name == w.name:
                    continue
                try:
                    out["paper_workloads"].append(time_field_workload(J, torch, device, wl.field_workload(key), "nearest", 20, 3, sm_max))
                except Exception as e:  # noqa: BLE001
                    out["paper_workloads"].append({"config": {"workload": key}, "error": str(e)})
            try:
                out["paper_run"] = time_paper_run(J, torch, device)
            except Exception as e:  # noqa: BLE001
                out["paper_run"] = {"error": str(e)}
            try:
                out["particle_kernels"] = time_particle_kernels(J, torch, device)
            except Exception as e:  # noqa: BLE001
                out["particle_kernels"] = {"error": str(e)}
        if keep_host:
            import oracle

            nobs = min(args.cpu_obs, N)
            r, dt = oracle_sample_rate(w, ring_host, nobs, 0, 1 if args.delay_rule == "linear" else 0)
            out["cpu_baseline"] = {"value": r / 1e9, "unit": "Gpairs/s", "cores": oracle.num_threads(), "kind": "oracle",
                                   "sample": f"{nobs} seeded observation cells x all {N - 1} source cells "
                                             f"({dt:.1f} s of fp64 CPU work)"}
        else:
            out["cpu_baseline"] = None
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    return out


def spawn_command(argv, gpus: int, port: int):
    """`python bench.py --gpus N` outside torchrun: the command that re-runs this file with N ranks, one per GPU."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={gpus}", "--master-addr", "127.0.0.1",
            "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def free_port() -> int:
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        return sk.getsockname()[1]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="jefi", choices=["jefi", "reference"])
    ap.add_argument("--workload", default="4", help="field workload: BASELINE.json config number (4 = 96^3, the default), or one of "
                    "the paper's own shapes: analytic20 (20^3, kappa = 6), slab251 (1x251x111), slab101")
    ap.add_argument("--no-pic", action="store_true", help="skip the PIC steps/s, paper-workload and particle-kernel legs")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--shard", default="obs", choices=["replicas", "obs"],
                    help="N > 1: observation z-slabs of one field step (default, strong scaling) or replicas (weak scaling)")
    ap.add_argument("--delay-rule", default="nearest", choices=["nearest", "linear"],
                    help="retarded-time rule: nearest = BASELINE.json's configs (reading A1); linear = second rule (A22)")
    ap.add_argument("--particles-only", action="store_true", help="only the deposit/push HBM-roofline leg (for ncu captures)")
    ap.add_argument("--paper-run-only", action="store_true", help="only the paper_run leg (1x251x111, 1e7 macro-particles, 1e4 steps)")
    ap.add_argument("--cpu-obs", type=int, default=4096, help="observation cells of the cpu_baseline sample")
    ap.add_argument("--ref-obs", type=int, default=1024, help="observation cells per step of --impl reference")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not under torchrun: start the N ranks ourselves (their stdout/stderr pass through; rank 0 prints the one JSON line)
        rc = subprocess.call(spawn_command(sys.argv[1:], args.gpus, free_port()))
        sys.exit(rc)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus:
        log(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}; the launcher's world size is what runs and is reported")
    args.warmup = max(args.warmup, 3) if args.impl == "jefi" else max(args.warmup, 0)
    w = wl.field_workload(args.workload)
    rank = int(os.environ.get("RANK", "0"))
    if args.particles_only:
        import torch

        from paper_2209_07944_b200 import jefi as J

        J.load_library()
        res = time_particle_kernels(J, torch, torch.device("cuda:0"), reps=max(1, args.steps))
    elif args.paper_run_only:
        import torch

        from paper_2209_07944_b200 import jefi as J

        J.load_library()
        res = {"paper_run": time_paper_run(J, torch, torch.device("cuda:0"))}
    elif args.impl == "reference":
        if rank != 0:
            log(f"[reference] rank {rank} of {world}: idle (rank 0 alone runs the CPU oracle)")
            return
        res = run_reference(args, w)
    else:
        res = run_product(args, w)
    if res is not None:
        print(json.dumps(res), flush=True)


if __name__ == "__main__":
    main()
