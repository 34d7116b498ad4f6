"""One PIC step over several GPUs ("accomplish the parallel computing").

Rank bookkeeping only: every number is computed by the kernels of libjefi through the C-ABI calls of ``jefi.py``; this module
decides which rank does what and moves whole arrays between ranks with ``torch.distributed``.

The partition.  The Jefimenko sum of an observation cell needs the history of ALL source cells, so every rank keeps the full
ring (32 H N bytes; 30 GB at 128^3) and the OBSERVATION cells are what is split: rank r solves the z-planes
``slab_range(nz, r, world)``.  The particles are dealt to the ranks by index once, at the start; a particle stays with its
rank whatever cell it moves to (every rank has E, B and deposits on the whole grid), so nothing migrates.  One step n
 is then

    1. jefi_deposit            each rank deposits ITS particles into its own rho, J  ([4][N] floats)
    2. all-reduce (sum)        rho, J over ranks: 16 N bytes per rank       <- the first of the two exchanges of a step
    3. jefi_push_sources       every rank stores the same summed sources in its ring
    4. jefi_field_step_slab    each rank solves its observation planes against all sources
    5. all-gather              E, B slabs -> every rank has the whole E, B: 24 N bytes      <- the second exchange
    6. jefi_push_particles     each rank pushes ITS particles

Both exchanges are plain NCCL collectives on the context's stream order; there is no kernel to fuse them with: the all-reduce
follows a deposit whose atomics finish in no particular order, and the gather follows a kernel whose CTAs each finish a whole
observation tile at the very end of their run.  The field solve is > 99 % of a step from 64^3 up, which is what the slabs split.

What differs from a one-GPU step: rho, J are sums of per-rank partial deposits (a different order of the fp32 additions, inside
the 1e-5 rel-L2 the deposit is held to anyway); E, B of a cell are the sums one rank formed, bit-identical on every rank after
the gather, and - given the same sources - bit-identical to the one-GPU result (jefi_field_step_slab).
"""
from __future__ import annotations

from typing import Dict, List, Tuple

from . import jefi as J


def deal_range(count: int, rank: int, world: int) -> Tuple[int, int]:
    """Particles [lo, hi) of `count` that rank `rank` of `world` owns: contiguous blocks by index, sizes differing by at most 1."""
    return (count * rank) // world, (count * (rank + 1)) // world


def deal_particles(part: Dict, rank: int, world: int) -> Dict:
    """The rank's share of every per-particle array of `part` (numpy arrays or tensors), as contiguous copies."""
    n = len(part["x"])
    lo, hi = deal_range(n, rank, world)
    out = {}
    for k, v in part.items():
        s = v[lo:hi]
        out[k] = s.clone() if hasattr(s, "clone") else s.copy()
    return out


def gather_slabs(dist, EB, plane: int, ranges: List[Tuple[int, int]], rank: int) -> None:
    """All-gather of the observation slabs (step 5): on entry rank r holds its planes ranges[r] = [k0, k1) of EB ([6][N],
    `plane` = nx*ny cells per z-plane), on return every rank holds all of E, B.  Slabs need not be equal (whole layers of
    observation tiles), so each rank sends a [6][plane * widest] block, zero-padded, and copies the valid part of every
    block it receives: 24 N bytes per rank up to the padding.  dist = None (one rank): nothing to do."""
    import torch

    if dist is None or len(ranges) == 1:
        return
    widest = max(k1 - k0 for k0, k1 in ranges)
    k0, k1 = ranges[rank]
    send = torch.zeros((6, plane * widest), dtype=EB.dtype, device=EB.device)
    send[:, :plane * (k1 - k0)] = EB[:, plane * k0:plane * k1]
    recv = [torch.empty_like(send) for _ in ranges]
    dist.all_gather(recv, send)
    for r, (a, b) in enumerate(ranges):
        if r != rank and b > a:
            EB[:, plane * a:plane * b] = recv[r][:, :plane * (b - a)]


class ShardedPic:
    """The six-stage step above for one rank.  `ctx` is this rank's JefiContext on the full grid; `part` this rank's particles
    (deal_particles).  dist: the torch.distributed module with an initialised default group (NCCL on one GPU per rank; gloo
    works too and moves the tensors through the host), or None for a single rank."""

    def __init__(self, ctx: "J.JefiContext", dist, rank: int = 0, world: int = 1):
        self.ctx, self.dist, self.rank, self.world = ctx, (dist if world > 1 else None), rank, world
        g = ctx.grid
        self.plane = g.nx * g.ny
        self.ranges = [ctx.slab_range(r, world) for r in range(world)]
        self.bytes_per_step = {"all_reduce_rho_J": 16 * ctx.N, "all_gather_E_B": 24 * ctx.N} if world > 1 else {}

    def step(self, part: Dict) -> None:
        ctx = self.ctx
        ctx.deposit(part)                                         # 1
        if self.dist is not None:
            self.dist.all_reduce(ctx.src, op=self.dist.ReduceOp.SUM)  # 2
        ctx.push_sources()                                        # 3
        k0, k1 = self.ranges[self.rank]
        if k1 > k0:
            ctx.field_step_slab(k0, k1)                           # 4
        gather_slabs(self.dist, ctx.EB, self.plane, self.ranges, self.rank)  # 5
        ctx.push_particles(part)                                  # 6
