"""jefi_deposit_static: the deposit for callers that may not allocate device memory.

Some users of libjefi cannot call cudaMalloc at the point where they deposit charge: their application took all device memory
into its own pool at start-up and permits no driver allocation afterwards, or their step loop cannot tolerate the device-wide
synchronisation an allocation may cause.  For them the library has one entry point, jefi_deposit_static, whose sort scratch is
a fixed 16 MiB array inside the library's CUDA module instead of context memory: it needs no context and never allocates, at
the price of a size limit (JEFI_STATIC_MAX_PARTICLES particles, JEFI_STATIC_MAX_BINS sort bins) and of one array shared by
every call on a device.

This file checks that entry point against the path everybody else uses (jefi_deposit on a context in JEFI_DEPOSIT_SORTED
mode, same kernels, context-owned scratch) at the tolerance of the other deposit tests, rel-L2 <= 1e-5 per quantity (the sums
are fp32 atomics, so the order of the additions is free), and against the fp64 oracle.  It makes several calls in a row on
one stream with different grids and list lengths, because the shared array keeps the previous call's contents: a long list on
a large grid first, then a short list on a small grid (stale keys, counts and offsets beyond its own range must not matter),
then the first input again.  The file is named so that pytest collects it last; it passes alone in a fresh process (then it
is the first user of the array on the device) and after the other GPU tests.
"""
import ctypes

import numpy as np
import pytest

C_LIGHT = 299792458.0


def make_particles(shape, count, seed):
    """Seeded particles over the whole box including the half-cell border (virtual nodes), some dead, a few hand-placed on
    cell faces, corners and just outside the grid."""
    rng = np.random.default_rng(seed)
    pos = [rng.uniform(0, n, count) for n in shape]
    special = np.array([[0.0, 0.0, 0.0], [0.49999, 0.5, 0.50001], [shape[0] - 1e-4, shape[1] - 0.5, shape[2] - 0.50001],
                        [0.25, shape[1] / 2, shape[2] / 2], [shape[0] + 3.0, 1.0, 1.0]])
    x, y, z = (np.concatenate([a, special[:, i]]) for i, a in enumerate(pos))
    P = x.shape[0]
    u = rng.normal(0, 0.3, (3, P))
    part = dict(x=x, y=y, z=z, ux=u[0], uy=u[1], uz=u[2], qw=rng.uniform(-2, 2, P) * 1e-13)
    part = {k: v.astype(np.float32) for k, v in part.items()}
    alive = np.ones(P, dtype=np.uint8)
    alive[::13] = 0
    alive[-1] = 1  # marked alive but outside the grid: deposits nothing
    part["alive"] = alive
    return part


def to_dev(part, device):
    import torch

    return {k: torch.from_numpy(np.ascontiguousarray(v)).to(device) for k, v in part.items()}


def assert_same_sums(S, Sref, what):
    for a in range(4):
        assert np.linalg.norm(S[a].astype(np.float64) - Sref[a]) <= 1e-5 * np.linalg.norm(Sref[a]), (what, a)


@pytest.mark.gpu
def test_static_deposit_matches_the_context_deposit_on_calls_in_a_row(cuda_device):
    import torch

    import oracle
    from oracle import OracleConfig
    from paper_2209_07944_b200 import jefi as J

    J.load_library()  # fails loudly if libjefi.so was not built
    dx = 1e-4
    dt = dx / (2 * C_LIGHT)
    cases = [((40, 33, 21), 300000, 101),  # 28 k cells, 3e5 particles: many scan tiles, long runs per cell
             ((7, 5, 3), 900, 102),        # tiny grid, short list: reads only its own part of the stale scratch
             ((40, 33, 21), 300000, 101),  # the first input again
             ((16, 16, 16), 0, 103)]       # empty list: outputs zeroed, nothing else runs
    first = None
    for shape, count, seed in cases:
        N = shape[0] * shape[1] * shape[2]
        part = make_particles(shape, count, seed) if count else {k: np.zeros(0, np.float32) for k in ("x", "y", "z", "ux", "uy", "uz", "qw")}
        if not count:
            part["alive"] = np.zeros(0, np.uint8)
        dp = to_dev(part, cuda_device)
        # the existing path: a context in JEFI_DEPOSIT_SORTED mode (context-owned, cudaMalloc'ed scratch)
        ctx = J.JefiContext(J.GridSpec(*shape, dx, dx, dx, dt), field_impl=J.JEFI_FIELD_REFERENCE, deposit_mode=J.JEFI_DEPOSIT_SORTED)
        Sref = ctx.deposit(dp).cpu().numpy().astype(np.float64)
        ctx.close()
        # the entry point under test; outputs pre-filled with junk to see that it overwrites them
        out = torch.full((4, N), 7.0, dtype=torch.float32, device=cuda_device)
        before = {k: v.clone() for k, v in dp.items()}
        J.jefi_deposit_static(*shape, dx, dx, dx, dp["x"], dp["y"], dp["z"], dp["ux"], dp["uy"], dp["uz"], dp["qw"], dp["alive"],
                              out[0], out[1], out[2], out[3])
        S = out.cpu().numpy()
        assert all(torch.equal(dp[k], before[k]) for k in dp)  # the caller's particle arrays are inputs only
        if count == 0:
            assert not S.any() and not Sref.any()
            continue
        assert_same_sums(S, Sref, ("static vs context", shape, count))
        assert np.array_equal(S[0] != 0, Sref[0] != 0)  # the same set of nodes received charge
        cfg = OracleConfig(*shape, dx, dx, dx, dt)
        So = oracle.deposit(cfg, part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"], part["qw"], part["alive"])
        assert_same_sums(S, So, ("static vs oracle", shape, count))
        if first is None:
            first = S
        elif shape == cases[0][0]:
            assert_same_sums(S, first.astype(np.float64), "third call vs first call")
    # alive == NULL is allowed, as in jefi_deposit
    shape = (9, 8, 7)
    part = make_particles(shape, 5000, 104)
    dp = to_dev(part, cuda_device)
    out = torch.empty((4, shape[0] * shape[1] * shape[2]), dtype=torch.float32, device=cuda_device)
    J.jefi_deposit_static(*shape, dx, dx, dx, dp["x"], dp["y"], dp["z"], dp["ux"], dp["uy"], dp["uz"], dp["qw"], None,
                          out[0], out[1], out[2], out[3])
    cfg = OracleConfig(*shape, dx, dx, dx, dt)
    So = oracle.deposit(cfg, part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"], part["qw"], np.ones_like(part["alive"]))
    assert_same_sums(out.cpu().numpy(), So, "alive = NULL")


def test_static_deposit_rejects_sizes_beyond_its_fixed_scratch():
    """The scratch cannot grow, so inputs over either limit are refused with the limit named, before any CUDA call (which is
    why this part runs on a box without a GPU): nothing is launched and nothing is written."""
    from paper_2209_07944_b200 import build, jefi as J

    build.build_lib()
    lib = J.load_library()
    err = ctypes.create_string_buffer(512)
    one = ctypes.c_void_p(256)  # never dereferenced: the checks come first
    args_tail = [one] * 7 + [None] + [one] * 4 + [err, len(err)]
    rc = lib.jefi_deposit_static(0, None, 16, 16, 16, 1e-4, 1e-4, 1e-4, 0.0, J.JEFI_STATIC_MAX_PARTICLES + 1, *args_tail)
    assert rc == J.JEFI_EINVAL and b"JEFI_STATIC_MAX_PARTICLES" in err.value
    rc = lib.jefi_deposit_static(0, None, 80, 80, 80, 1e-4, 1e-4, 1e-4, 0.0, 10, *args_tail)  # 81^3 + 1 bins > 524288
    assert rc == J.JEFI_EINVAL and b"JEFI_STATIC_MAX_BINS" in err.value
    rc = lib.jefi_deposit_static(0, None, 0, 16, 16, 1e-4, 1e-4, 1e-4, 0.0, 10, *args_tail)
    assert rc == J.JEFI_EINVAL and err.value
    rc = lib.jefi_deposit_static(0, None, 16, 16, 16, 1e-4, 1e-4, 1e-4, 0.0, 10, *([None] + args_tail[1:]))
    assert rc == J.JEFI_EINVAL and b"NULL" in err.value
    assert lib.jefi_deposit_static(0, None, 16, 16, 16, 1e-4, 1e-4, 1e-4, 0.0, J.JEFI_STATIC_MAX_PARTICLES + 1, *(args_tail[:-2] + [None, 0])) == J.JEFI_EINVAL
    assert (79 + 1) ** 3 + 1 <= J.JEFI_STATIC_MAX_BINS  # the grid size include/jefi.h quotes as fitting
