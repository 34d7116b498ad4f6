"""GPU parity: libjefi (through the C-ABI binding) against the fp64 oracle, element by element, same seeded inputs.

Tolerances (BASELINE.json north_star, reading A20 in DESIGN.md §3):
  fields     ||d||_2 / ||F_oracle||_2 <= 1e-4 over all 3N components, and max|d| <= 1e-3 * ||F_oracle||_2 / sqrt(3N)
  positions  max_p |dr|_inf / (n cells) <= 1e-5 after 10 steps, over particles alive in both
  indices    delay table, cell indices, history slots: bit-exact
  deposit    rel-L2 <= 1e-5 (fp32 atomics: summation order is not defined)
"""
import math

import numpy as np
import pytest

import oracle
from oracle import OracleConfig
from paper_2209_07944_b200 import workloads as wl

pytestmark = pytest.mark.gpu

C = 299792458.0


def field_err(F, Fo):
    """(relative L2, max-abs / RMS) of a [3][n] field against the oracle's."""
    d = F.astype(np.float64) - Fo
    nrm = np.linalg.norm(Fo)
    rms = nrm / math.sqrt(Fo.size)
    return np.linalg.norm(d) / nrm, np.abs(d).max() / rms


def assert_field_parity(E, B, Eo, Bo, tag=""):
    for name, F, Fo in (("E", E, Eo), ("B", B, Bo)):
        if np.linalg.norm(Fo) == 0.0:
            assert np.all(F == 0.0), f"{tag}{name}: oracle is exactly zero"
            continue
        l2, mx = field_err(F, Fo)
        assert l2 <= 1e-4, f"{tag}{name}: rel-L2 {l2:.3e}"
        assert mx <= 1e-3, f"{tag}{name}: max-abs/rms {mx:.3e}"


@pytest.fixture(scope="module")
def J(cuda_device):
    from paper_2209_07944_b200 import jefi

    jefi.load_library()  # fails loudly if libjefi.so was not built
    return jefi


def make_ctx(J, shape, h, dt, impl, **kw):
    g = J.GridSpec(shape[0], shape[1], shape[2], h[0], h[1], h[2], dt, **kw)
    return J.JefiContext(g, field_impl=impl)


def run_history(J, ctx, slices):
    """Push [4][N] fp32 slices one by one; return E, B (float32 numpy [3][N]) at the last step."""
    import torch

    for s in slices:
        t = torch.from_numpy(np.ascontiguousarray(s)).to(ctx.device)
        ctx.push_sources(t)
    eb = ctx.field_step().cpu().numpy()
    return eb[:3], eb[3:]


def oracle_history(cfg, slices, obs=None):
    orc = oracle.OracleJefi(cfg)
    for s in slices:
        orc.push_sources(*s.astype(np.float64))
    return orc.field_step(obs)


# ------------------------------------------------------------------------------------------- delay table (a2)
@pytest.mark.parametrize("shape,h,kappa", [((16, 16, 16), (1e-4, 1e-4, 1e-4), 2.0), ((13, 10, 7), (1e-4, 0.7e-4, 1.3e-4), 1.37),
                                           ((32, 32, 32), (1e-4, 1e-4, 1e-4), 2.0)])
def test_delay_table_bit_exact(J, shape, h, kappa):
    dt = h[0] / (kappa * C)
    ctx = make_ctx(J, shape, h, dt, J.JEFI_FIELD_REFERENCE)
    cfg = OracleConfig(*shape, *h, dt)
    tab = J.jefi_debug_delay_table(ctx.handle, *shape)
    assert np.array_equal(tab, oracle.delay_table(cfg))
    assert ctx.H == cfg.H and ctx.info["ndt"] == oracle.num_dt(cfg)
    ctx.close()


def test_tiled_kernel_is_selected_for_benchmark_grids(J):
    """kappa = 2 grids: the fp32 delay arithmetic is proven equal to the fp64 table, so AUTO picks the tiled kernel."""
    for n, dx in ((16, 1e-4), (32, 1e-4), (64, 5e-5)):
        ctx = make_ctx(J, (n, n, n), (dx, dx, dx), dx / (2 * C), J.JEFI_FIELD_AUTO)
        assert ctx.info["field_impl"] == J.JEFI_FIELD_TILED
        ctx.close()


# ------------------------------------------------------------------------------------------- field (a1 + a3)
FIELD_CASES = [
    # shape, spacing, kappa, number of pushed steps (relative to H): spans several tiles and ragged tails
    ((16, 16, 16), (1e-4, 1e-4, 1e-4), 2.0, "full"),
    ((16, 16, 16), (1e-4, 1e-4, 1e-4), 2.0, "early"),
    ((16, 16, 16), (1e-4, 1e-4, 1e-4), 2.0, "wrapped"),
    ((13, 10, 7), (1e-4, 1e-4, 1e-4), 2.0, "wrapped"),
    ((9, 5, 3), (1e-4, 1e-4, 1e-4), 2.0, "full"),
    ((1, 1, 1), (1e-4, 1e-4, 1e-4), 2.0, "full"),
    ((2, 1, 1), (1e-4, 1e-4, 1e-4), 2.0, "full"),
    ((20, 12, 8), (1e-4, 2e-4, 1e-4), 2.0, "wrapped"),
]


@pytest.mark.parametrize("impl", ["reference", "tiled"])
@pytest.mark.parametrize("shape,h,kappa,fill", FIELD_CASES)
def test_field_parity_random_history(J, impl, shape, h, kappa, fill):
    dt = h[0] / (kappa * C)
    cfg = OracleConfig(*shape, *h, dt)
    nsteps = {"full": cfg.H, "early": max(2, cfg.H // 3), "wrapped": 2 * cfg.H + 3}[fill]
    # J in [-c, c] so that all three terms of Eq. (2.4) are comparable (SURVEY.md §8(d) config-4 caveat)
    slices = [wl.history_slice(cfg.N, t, 4242, j_scale=C) for t in range(nsteps)]
    ctx = make_ctx(J, shape, h, dt, J.JEFI_FIELD_TILED if impl == "tiled" else J.JEFI_FIELD_REFERENCE)
    E, B = run_history(J, ctx, slices)
    Eo, Bo = oracle_history(cfg, slices)
    if cfg.N == 1:
        assert np.all(E == 0) and np.all(B == 0) and np.all(Eo == 0)
    else:
        assert_field_parity(E, B, Eo, Bo, f"{impl} {shape} {fill}: ")
    ctx.close()


@pytest.mark.parametrize("impl", ["reference", "tiled"])
@pytest.mark.parametrize("shape,h,kappa,fill", [FIELD_CASES[0], FIELD_CASES[1], FIELD_CASES[3], FIELD_CASES[6], FIELD_CASES[7]])
def test_field_parity_linear_delay_rule(J, impl, shape, h, kappa, fill):
    """JEFI_DELAY_LINEAR (reading A22) against the oracle's RULE_LINEAR; it must also differ from the nearest rule."""
    dt = h[0] / (kappa * C)
    cfg = OracleConfig(*shape, *h, dt, delay_rule=oracle.RULE_LINEAR)
    nsteps = {"full": cfg.H, "early": max(2, cfg.H // 3), "wrapped": 2 * cfg.H + 3}[fill]
    slices = [wl.history_slice(cfg.N, t, 777, j_scale=C) for t in range(nsteps)]
    g = J.GridSpec(*shape, *h, dt)
    ctx = J.JefiContext(g, field_impl=J.JEFI_FIELD_TILED if impl == "tiled" else J.JEFI_FIELD_REFERENCE,
                        delay_rule=J.JEFI_DELAY_LINEAR)
    E, B = run_history(J, ctx, slices)
    Eo, Bo = oracle_history(cfg, slices)
    assert_field_parity(E, B, Eo, Bo, f"linear {impl} {shape} {fill}: ")
    if cfg.N > 8:
        En, Bn = oracle_history(OracleConfig(*shape, *h, dt), slices)
        assert field_err(E, En)[0] > 1e-3  # the two rules are visibly different on this input
    ctx.close()


def analytic_sources(cfg, t):
    """PAPER.md:421-425 Eqs. (3.4)-(3.5): Jx = Jy = Jz = sin(x+y+z) sin(t), rho = 3 (cos(t) - 1) cos(x+y+z) at the cell
    centres, time t = step * dt; fp32 [4][N] as the C-ABI takes them."""
    k, j, i = np.meshgrid(np.arange(cfg.nz), np.arange(cfg.ny), np.arange(cfg.nx), indexing="ij")
    u = ((i + 0.5) * cfg.dx + (j + 0.5) * cfg.dy + (k + 0.5) * cfg.dz).ravel()
    tt = t * cfg.dt
    jv = np.sin(u) * math.sin(tt)
    return np.stack([3.0 * (math.cos(tt) - 1.0) * np.cos(u), jv, jv, jv]).astype(np.float32)


@pytest.mark.parametrize("rule", ["NEAREST", "LINEAR"])
def test_paper_analytic_sources_ndt_scan(J, rule):
    """The paper's N_dt experiment: 20^3 cells, dx = 0.3, dt = 0.05, c = eps0 = mu0 = 1 (kappa = 6), ring
    depths below and above the ~207 steps light needs to cross the diagonal.  Every depth is compared with the oracle
    at the same depth; depths >= N_dt + 2 agree with one another bit for bit on the GPU as they do in the oracle (P9),
    a truncated history visibly does not."""
    n = 20
    base = OracleConfig(n, n, n, 0.3, 0.3, 0.3, 0.05, c=1.0, eps0=1.0)
    ndt = oracle.num_dt(base)
    assert ndt == 208
    step = 260
    res = {}
    for depth in (ndt + 2, ndt + 42, 101, 31):
        cfg = OracleConfig(n, n, n, 0.3, 0.3, 0.3, 0.05, c=1.0, eps0=1.0, H=depth, delay_rule=getattr(oracle, "RULE_" + rule))
        slices = [analytic_sources(cfg, t) for t in range(step + 1)]
        ctx = J.JefiContext(J.GridSpec(n, n, n, 0.3, 0.3, 0.3, 0.05, c=1.0, eps0=1.0, H=depth),
                            delay_rule=getattr(J, "JEFI_DELAY_" + rule))
        assert ctx.H == depth
        # kappa = 6: the slot window of a tile pair (61+ rows) exceeds the largest compiled pitch (48), so the tiled kernel
        # serves it in two passes (MODE_MULTI) instead of falling back to the reference kernel
        assert ctx.info["field_impl"] == J.JEFI_FIELD_TILED, ctx.info["field_impl_reason"]
        ti = ctx.tile_info
        assert ti["window_slots"] > ti["window_pitch"] == 48 and ti["obs_tile"] == (8, 8, 8)
        E, B = run_history(J, ctx, slices)
        Eo, Bo = oracle_history(cfg, slices)
        assert_field_parity(E, B, Eo, Bo, f"analytic sources, depth {depth}: ")
        res[depth] = (E, B, ctx.info["field_impl"])
        ctx.close()
    E0, B0, _ = res[ndt + 2]
    assert np.array_equal(res[ndt + 42][0], E0) and np.array_equal(res[ndt + 42][1], B0)
    for depth in (101, 31):
        assert field_err(res[depth][0], E0.astype(np.float64))[0] > 1e-2


@pytest.mark.parametrize("impl", ["reference", "tiled"])
@pytest.mark.parametrize("shape,world", [((16, 16, 16), 2), ((13, 10, 20), 3), ((9, 5, 3), 2), ((24, 24, 40), 4)])
def test_field_step_slabs_add_up_to_the_full_step_bitwise(J, impl, shape, world):
    """observation slabs are independent; `world` slab calls (what `world` GPUs would each do) assemble the
    full jefi_field_step bit for bit, and each call writes nothing outside its slab."""
    import torch

    h = (1e-4,) * 3
    dt = h[0] / (2 * C)
    cfg = OracleConfig(*shape, *h, dt)
    ctx = make_ctx(J, shape, h, dt, J.JEFI_FIELD_TILED if impl == "tiled" else J.JEFI_FIELD_REFERENCE)
    for t in range(min(cfg.H, 40)):
        ctx.push_sources(torch.from_numpy(wl.history_slice(cfg.N, t, 99, j_scale=C)).to(ctx.device))
    full = ctx.field_step().clone()
    asm = torch.full_like(full, float("nan"))
    plane = shape[0] * shape[1]
    covered = 0
    for r in range(world):
        k0, k1 = J.slab_range(shape[2], r, world)
        assert k0 % 8 == 0 and 0 <= k0 <= k1 <= shape[2]
        part = torch.full_like(full, -7.0)
        ctx.field_step_slab(k0, k1, part)
        assert bool((part[:, :plane * k0] == -7.0).all()) and bool((part[:, plane * k1:] == -7.0).all())
        asm[:, plane * k0:plane * k1] = part[:, plane * k0:plane * k1]
        covered += k1 - k0
    assert covered == shape[2]
    # bit for bit, also when the source range is split over CTAs (the pieces are added in a fixed order)
    assert torch.equal(asm, full), (impl, shape, ctx.tile_info)
    with pytest.raises(J.JefiError):
        ctx.field_step_slab(4, shape[2])  # k0 not a multiple of 8
    # the last rank's slab against the oracle itself, on its own cells only (not through the full step)
    k0, k1 = J.slab_range(shape[2], world - 1, world)
    slices = [wl.history_slice(cfg.N, t, 99, j_scale=C) for t in range(min(cfg.H, 40))]
    obs = np.arange(plane * k0, plane * k1, dtype=np.int64)
    Eo, Bo = oracle_history(cfg, slices, obs)
    part = torch.zeros_like(full)
    ctx.field_step_slab(k0, k1, part)
    got = part.cpu().numpy()[:, plane * k0:plane * k1]
    assert_field_parity(got[:3], got[3:], Eo, Bo, f"slab [{k0},{k1}) of {shape} vs oracle: ")
    ctx.close()


@pytest.mark.parametrize("impl", ["reference", "tiled"])
def test_field_light_cone_exact_zero(J, impl):
    """A single source cell switched on at step n0: cells outside the light cone are exactly zero on the GPU too."""
    import torch

    n = 16
    dx = 1e-4
    dt = dx / (2 * C)
    cfg = OracleConfig(n, n, n, dx, dx, dx, dt)
    ctx = make_ctx(J, (n, n, n), (dx, dx, dx), dt, J.JEFI_FIELD_TILED if impl == "tiled" else J.JEFI_FIELD_REFERENCE)
    src = 3 + n * (5 + n * 2)
    rng = np.random.default_rng(5)
    slices = []
    for t in range(12):
        s = np.zeros((4, cfg.N), dtype=np.float32)
        if t >= 4:
            s[:, src] = rng.uniform(-1, 1, 4) * np.array([1, C, C, C])
        slices.append(s)
    E, B = run_history(J, ctx, slices)
    Eo, Bo = oracle_history(cfg, slices)
    zero = (np.abs(Eo).sum(0) == 0) & (np.abs(Bo).sum(0) == 0)
    assert zero.sum() > 1000
    assert np.all(E[:, zero] == 0) and np.all(B[:, zero] == 0)
    assert_field_parity(E, B, Eo, Bo, impl + " light cone: ")
    ctx.close()


def test_field_shallow_history_a15(J):
    """H smaller than N_dt + 2: delays beyond the stored history contribute zero (reading A15) in both kernels."""
    n, dx = 12, 1e-4
    dt = dx / (2 * C)
    cfg = OracleConfig(n, n, n, dx, dx, dx, dt, H=9)
    slices = [wl.history_slice(cfg.N, t, 99, j_scale=C) for t in range(25)]
    Eo, Bo = oracle_history(cfg, slices)
    for impl in (J.JEFI_FIELD_REFERENCE, J.JEFI_FIELD_TILED):
        ctx = make_ctx(J, (n, n, n), (dx, dx, dx), dt, impl, H=9)
        E, B = run_history(J, ctx, slices)
        assert_field_parity(E, B, Eo, Bo, f"impl {impl} shallow: ")
        ctx.close()


def test_history_slots_bit_exact_indices(J):
    """The ring returns, for every steps_back, the slice pushed at that step (index parity); values survive the
    J/c storage scaling to 1 ulp."""
    import torch

    n, dx = 8, 1e-4
    dt = dx / (2 * C)
    ctx = make_ctx(J, (n, n, n), (dx, dx, dx), dt, J.JEFI_FIELD_REFERENCE)
    H = ctx.H
    slices = [wl.history_slice(n ** 3, t, 7, j_scale=1e6) for t in range(2 * H + 5)]
    for s in slices:
        ctx.push_sources(torch.from_numpy(s).to(ctx.device))
    last = len(slices) - 1
    for back in (0, 1, 2, H // 2, H - 1):
        got = J.jefi_debug_history_slot(ctx.handle, n ** 3, back, ctx.device).cpu().numpy()
        want = slices[last - back]
        assert np.array_equal(got[0], want[0])  # rho is stored unscaled
        assert np.allclose(got[1:], want[1:], rtol=2.5e-7, atol=0)
        # it is this step and not a neighbour
        assert not np.allclose(got[0], slices[last - back - 1][0])
    with pytest.raises(J.JefiError):
        J.jefi_debug_history_slot(ctx.handle, n ** 3, H, ctx.device)
    ctx.close()


# ------------------------------------------------------------------------------------------- particles (a4, a5)
def to_dev(part, device):
    import torch

    return {k: torch.from_numpy(np.ascontiguousarray(v)).to(device) for k, v in part.items()}


def edge_particles(n, seed, count):
    """Uniform over the whole grid including the half-cell border (virtual nodes) + hand-placed edge cases."""
    rng = np.random.default_rng(seed)
    x, y, z = (rng.uniform(0, n, count) for _ in range(3))
    special = np.array([[0.0, 0.0, 0.0], [0.49999, 0.5, 0.50001], [n - 1e-4, n - 0.5, n - 0.50001], [0.25, n / 2, n / 2],
                        [n / 2 + 0.5, n / 2 + 0.5, n / 2 + 0.5]])
    x, y, z = (np.concatenate([a, special[:, i]]) for i, a in enumerate((x, y, z)))
    P = x.shape[0]
    u = rng.normal(0, 0.3, (3, P))
    part = dict(x=x, y=y, z=z, ux=u[0], uy=u[1], uz=u[2], qw=rng.uniform(-2, 2, P) * 1e-13,
                qm=np.where(rng.uniform(size=P) < 0.5, -1.75882001076e11, 9.5788331560e7))
    part = {k: v.astype(np.float32) for k, v in part.items()}
    alive = np.ones(P, dtype=np.uint8)
    alive[::17] = 0
    part["alive"] = alive
    return part


@pytest.mark.parametrize("shape", [(16, 16, 16), (13, 10, 7)])
def test_deposit_parity_and_indices(J, shape):
    dx = 1e-4
    dt = dx / (2 * C)
    cfg = OracleConfig(*shape, dx, dx, dx, dt)
    ctx = make_ctx(J, shape, (dx, dx, dx), dt, J.JEFI_FIELD_REFERENCE)
    part = edge_particles(min(shape), 11, 20000)
    for k, lim in zip("xyz", shape):  # stretch to the actual box
        part[k] = (part[k] * (lim / min(shape))).astype(np.float32)
        part[k] = np.minimum(part[k], np.nextafter(np.float32(lim), np.float32(0)))
    dp = to_dev(part, ctx.device)
    idx = J.jefi_debug_cell_index(ctx.handle, dp["x"], dp["y"], dp["z"]).cpu().numpy()
    assert np.array_equal(idx, oracle.cell_index(part["x"], part["y"], part["z"]))  # bit-exact
    S = ctx.deposit(dp).cpu().numpy()
    So = oracle.deposit(cfg, part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"], part["qw"], part["alive"])
    for a in range(4):
        assert np.linalg.norm(S[a] - So[a]) <= 1e-5 * np.linalg.norm(So[a]), a
    assert np.array_equal(S[0] != 0, So[0] != 0)  # the same set of nodes received charge
    # cell-sorted input (the case the warp aggregation is for) gives the same answer
    order = np.lexsort((idx[:, 0], idx[:, 1], idx[:, 2]))
    ps = to_dev({k: v[order] for k, v in part.items()}, ctx.device)
    S2 = ctx.deposit(ps).cpu().numpy()
    for a in range(4):
        assert np.linalg.norm(S2[a] - So[a]) <= 1e-5 * np.linalg.norm(So[a]), a
    ctx.close()


@pytest.mark.parametrize("shape,count", [((16, 16, 16), 20000), ((13, 10, 7), 50000), ((5, 4, 3), 7), ((8, 8, 8), 300000)])
def test_deposit_sorted_mode_order_and_parity(J, shape, count):
    """JEFI_DEPOSIT_SORTED: the internal order is a valid cell sort of exactly the depositing particles (keys compared
    bit-exactly with the oracle's cell indices; the order inside a cell is free), and the sums match the oracle."""
    dx = 1e-4
    dt = dx / (2 * C)
    cfg = OracleConfig(*shape, dx, dx, dx, dt)
    g = J.GridSpec(*shape, dx, dx, dx, dt)
    ctx = J.JefiContext(g, field_impl=J.JEFI_FIELD_REFERENCE, deposit_mode=J.JEFI_DEPOSIT_SORTED)
    part = edge_particles(min(shape), 5, count)
    for k, lim in zip("xyz", shape):
        part[k] = (part[k] * (lim / min(shape))).astype(np.float32)
        part[k] = np.minimum(part[k], np.nextafter(np.float32(lim), np.float32(0)))
    dp = to_dev(part, ctx.device)
    order, na = J.jefi_debug_cell_order(ctx.handle, dp["x"], dp["y"], dp["z"], dp["alive"])
    order = order.cpu().numpy()
    P = part["x"].shape[0]
    alive_idx = np.flatnonzero(part["alive"])
    assert np.array_equal(np.sort(order), np.arange(P))                          # a permutation of all particles
    assert na == alive_idx.size and np.array_equal(np.sort(order[:na]), alive_idx)  # depositing particles first
    idx = oracle.cell_index(part["x"], part["y"], part["z"])                    # [P][3], int
    key = (idx[:, 0] + 1) + (shape[0] + 1) * ((idx[:, 1] + 1) + (shape[1] + 1) * (idx[:, 2] + 1))
    assert np.all(np.diff(key[order[:na]]) >= 0)                                  # grouped by cell, ascending
    S = ctx.deposit(dp).cpu().numpy()
    So = oracle.deposit(cfg, part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"], part["qw"], part["alive"])
    for a in range(4):
        assert np.linalg.norm(S[a] - So[a]) <= 1e-5 * np.linalg.norm(So[a]), a
    assert np.array_equal(S[0] != 0, So[0] != 0)
    # a second call with fewer particles reuses the scratch; a particle marked alive but outside the grid adds nothing
    sub = {k: v[:1000].copy() for k, v in part.items()}
    sub["x"][0] = np.float32(shape[0] + 3.0)
    sub["alive"][0] = 1
    S2 = ctx.deposit(to_dev(sub, ctx.device)).cpu().numpy()
    So2 = oracle.deposit(cfg, sub["x"], sub["y"], sub["z"], sub["ux"], sub["uy"], sub["uz"], sub["qw"], sub["alive"])
    for a in range(4):
        assert np.linalg.norm(S2[a] - So2[a]) <= 1e-5 * np.linalg.norm(So2[a]), a
    ctx.close()


def test_deposit_modes_agree_on_config3_particles(J):
    """1e6 beam electrons of config 3 on the 64^3 grid: direct, sorted and auto deposits against the oracle."""
    w = wl.WORKLOADS[3]
    part = wl.particles(3)
    cfg = OracleConfig(w.n, w.n, w.n, w.dx, w.dx, w.dx, w.dt)
    So = oracle.deposit(cfg, part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"], part["qw"], part["alive"])
    for mode in (J.JEFI_DEPOSIT_DIRECT, J.JEFI_DEPOSIT_SORTED, J.JEFI_DEPOSIT_RUNS, J.JEFI_DEPOSIT_AUTO):
        ctx = J.JefiContext(J.GridSpec(w.n, w.n, w.n, w.dx, w.dx, w.dx, w.dt), field_impl=J.JEFI_FIELD_REFERENCE, deposit_mode=mode)
        S = ctx.deposit(to_dev(part, ctx.device)).cpu().numpy()
        for a in range(4):
            assert np.linalg.norm(S[a] - So[a]) <= 1e-5 * np.linalg.norm(So[a]), (mode, a)
        ctx.close()


@pytest.mark.parametrize("mode", ["DIRECT", "RUNS"])
def test_sort_particles_in_place(J, mode):
    """jefi_sort_particles permutes all arrays consistently (checked through the tag), groups the depositing particles
    by cell, and changes neither the deposit (to summation order) nor any particle's push (bit for bit)."""
    import torch

    shape, dx = (13, 10, 7), 1e-4
    dt = dx / (2 * C)
    cfg = OracleConfig(*shape, dx, dx, dx, dt)
    ctx = J.JefiContext(J.GridSpec(*shape, dx, dx, dx, dt), field_impl=J.JEFI_FIELD_REFERENCE,
                        deposit_mode=getattr(J, "JEFI_DEPOSIT_" + mode))
    part = edge_particles(min(shape), 21, 40000)
    for k, lim in zip("xyz", shape):
        part[k] = (part[k] * (lim / min(shape))).astype(np.float32)
        part[k] = np.minimum(part[k], np.nextafter(np.float32(lim), np.float32(0)))
    P = part["x"].shape[0]
    dp = to_dev(part, ctx.device)
    dp["tag"] = torch.arange(P, dtype=torch.int32, device=ctx.device)
    ctx.sort_particles(dp)
    tag = dp["tag"].cpu().numpy()
    assert np.array_equal(np.sort(tag), np.arange(P))
    for k, v in part.items():
        assert np.array_equal(dp[k].cpu().numpy(), v[tag]), k  # every array moved with its particle
    na = int(part["alive"].sum())
    assert np.all(dp["alive"].cpu().numpy()[:na] == 1) and np.all(dp["alive"].cpu().numpy()[na:] == 0)
    idx = oracle.cell_index(part["x"], part["y"], part["z"])
    key = (idx[:, 0] + 1) + (shape[0] + 1) * ((idx[:, 1] + 1) + (shape[1] + 1) * (idx[:, 2] + 1))
    assert np.all(np.diff(key[tag[:na]]) >= 0)
    S = ctx.deposit(dp).cpu().numpy()
    So = oracle.deposit(cfg, part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"], part["qw"], part["alive"])
    for a in range(4):
        assert np.linalg.norm(S[a] - So[a]) <= 1e-5 * np.linalg.norm(So[a]), a
    # push: sorted and unsorted copies give bit-identical particles
    rng = np.random.default_rng(9)
    EB = torch.from_numpy(rng.normal(0, 1, (6, cfg.N)).astype(np.float32) * np.array([[1e4]] * 3 + [[1e-2]] * 3, dtype=np.float32)).to(ctx.device)
    du = to_dev(part, ctx.device)
    ctx.push_particles(du, EB)
    ctx.push_particles(dp, EB)
    for k in ("x", "y", "z", "ux", "uy", "uz", "alive"):
        assert np.array_equal(dp[k].cpu().numpy(), du[k].cpu().numpy()[tag]), k
    ctx.close()


def test_deposit_empty_and_all_dead(J):
    import torch

    n, dx = 8, 1e-4
    ctx = make_ctx(J, (n, n, n), (dx, dx, dx), dx / (2 * C), J.JEFI_FIELD_REFERENCE)
    ctx.src.fill_(7.0)
    empty = {k: torch.empty(0, dtype=torch.float32, device=ctx.device) for k in ("x", "y", "z", "ux", "uy", "uz", "qw")}
    empty["alive"] = torch.empty(0, dtype=torch.uint8, device=ctx.device)
    assert float(ctx.deposit(empty).abs().sum()) == 0.0  # outputs are overwritten even with no particles
    part = edge_particles(n, 3, 100)
    part["alive"][:] = 0
    assert float(ctx.deposit(to_dev(part, ctx.device)).abs().sum()) == 0.0
    ctx.close()


def test_push_parity_one_step_with_external_fields(J):
    n, dx = 16, 1e-4
    dt = dx / (2 * C)
    ext = dict(Eext=(1e5, -2e5, 3e4), Bext=(0.0, 10.0, 0.5))
    cfg = OracleConfig(n, n, n, dx, dx, dx, dt, **ext)
    ctx = make_ctx(J, (n, n, n), (dx, dx, dx), dt, J.JEFI_FIELD_REFERENCE, **ext)
    part = edge_particles(n, 21, 30000)
    rng = np.random.default_rng(22)
    F = rng.normal(0, 1, (6, cfg.N))
    F[:3] *= 1e7
    F[3:] *= 0.05
    F = F.astype(np.float32)
    import torch

    dp = to_dev(part, ctx.device)
    ctx.push_particles(dp, torch.from_numpy(F).to(ctx.device))
    po = {k: v.astype(np.float64) for k, v in part.items() if k != "alive"}
    alive_o = part["alive"].copy()
    oracle.push(cfg, po["x"], po["y"], po["z"], po["ux"], po["uy"], po["uz"], po["qm"], alive_o, F[:3].astype(np.float64),
                F[3:].astype(np.float64))
    got = {k: v.cpu().numpy() for k, v in dp.items()}
    both = (got["alive"] == 1) & (alive_o == 1)
    assert (got["alive"] != alive_o).sum() <= 2  # a particle within 1 ulp of a face may differ
    was_alive = part["alive"] == 1
    for k in "xyz":
        assert np.abs(got[k][was_alive] - po[k][was_alive]).max() / n <= 1e-6
    for k in ("ux", "uy", "uz"):
        assert np.abs(got[k][both] - po[k][both]).max() <= 2e-6 * max(1.0, np.abs(po[k]).max())
    dead = part["alive"] == 0
    assert np.array_equal(got["x"][dead], part["x"][dead]) and np.array_equal(got["ux"][dead], part["ux"][dead])
    ctx.close()


def test_push_parity_strongly_relativistic_crossed_fields(J):
    """u ~ 1, h E/c ~ 1 and h B/gamma ~ 1 per step (units c = 1): the regime in which the gamma of Eq. (2.10) matters (oracle pin
    P16: gamma of u^-, reading A6); a push that took gamma from u^{n-1/2} would be off by O(0.1) here."""
    import torch

    n, dx, dt = 12, 50.0, 1.0
    kw = dict(c=1.0, eps0=1.0, Eext=(0.3, -0.2, 0.1), Bext=(0.0, 0.5, -0.4))
    cfg = OracleConfig(n, n, n, dx, dx, dx, dt, **kw)
    ctx = make_ctx(J, (n, n, n), (dx, dx, dx), dt, J.JEFI_FIELD_REFERENCE, **kw)
    rng = np.random.default_rng(160)
    P = 20000
    part = dict(x=rng.uniform(0, n, P), y=rng.uniform(0, n, P), z=rng.uniform(0, n, P), ux=rng.normal(0, 0.7, P),
                uy=rng.normal(0, 0.7, P), uz=rng.normal(0, 0.7, P), qw=np.ones(P), qm=np.where(rng.uniform(size=P) < 0.5, -2.0, 2.0))
    part = {k: v.astype(np.float32) for k, v in part.items()}
    part["alive"] = np.ones(P, dtype=np.uint8)
    F = rng.normal(0, 1.0, (6, cfg.N)).astype(np.float32)
    F[3:] *= 1.5
    dp = to_dev(part, ctx.device)
    ctx.push_particles(dp, torch.from_numpy(F).to(ctx.device))
    po = {k: v.astype(np.float64) for k, v in part.items() if k != "alive"}
    alive_o = part["alive"].copy()
    oracle.push(cfg, po["x"], po["y"], po["z"], po["ux"], po["uy"], po["uz"], po["qm"], alive_o, F[:3].astype(np.float64),
                F[3:].astype(np.float64))
    got = {k: v.cpu().numpy() for k, v in dp.items()}
    assert (got["alive"] != alive_o).sum() <= 1
    umax = max(np.abs(po[k]).max() for k in ("ux", "uy", "uz"))
    assert umax > 2.0  # strongly relativistic
    for k in ("ux", "uy", "uz"):
        assert np.abs(got[k] - po[k]).max() <= 2e-6 * umax, k
    for k in "xyz":
        assert np.abs(got[k] - po[k]).max() / n <= 1e-6, k
    ctx.close()


# ------------------------------------------------------------------------------------------- closed loop (config 1)
def run_closed_loop(J, config, steps, scale=1.0, impl=None, sort_every=0):
    import torch

    w = wl.WORKLOADS[config]
    part = wl.particles(config, scale)
    cfg = OracleConfig(w.n, w.n, w.n, w.dx, w.dx, w.dx, w.dt)
    assert cfg.H == w.H
    ctx = make_ctx(J, (w.n,) * 3, (w.dx,) * 3, w.dt, J.JEFI_FIELD_AUTO if impl is None else impl)
    ctx.sort_every = sort_every  # 0: particles keep their array positions (JefiContext's default is 8)
    dp = to_dev(part, ctx.device)
    if sort_every:
        dp["tag"] = torch.arange(part["x"].shape[0], dtype=torch.int32, device=ctx.device)
    orc = oracle.OracleJefi(cfg)
    po = {k: v.astype(np.float64) for k, v in part.items() if k != "alive"}
    po["alive"] = part["alive"].copy()
    hist = []
    for s in range(steps):
        ctx.pic_step(dp)
        So, Eo, Bo = orc.pic_step(po)
        if s in (0, steps // 2, steps - 1):
            eb = ctx.EB.cpu().numpy()
            hist.append((s, eb[:3].copy(), eb[3:].copy(), Eo, Bo, ctx.src.cpu().numpy().copy(), So))
    got = {k: v.cpu().numpy() for k, v in dp.items()}
    if sort_every:  # back to the oracle's particle numbering
        inv = np.argsort(got.pop("tag"))
        got = {k: v[inv] for k, v in got.items()}
    ctx.close()
    return w, got, po, hist


def test_closed_loop_config1_10_steps(J):
    w, got, po, hist = run_closed_loop(J, 1, 10)
    both = (got["alive"] == 1) & (po["alive"] == 1)
    assert (got["alive"] != po["alive"]).sum() <= 1
    for k in "xyz":
        assert np.abs(got[k][both] - po[k][both]).max() / w.n <= 1e-5
    for s, E, B, Eo, Bo, S, So in hist:
        assert_field_parity(E, B, Eo, Bo, f"cfg1 step {s}: ")
        for a in range(4):
            assert np.linalg.norm(S[a] - So[a]) <= 1e-5 * max(np.linalg.norm(So[a]), 1e-300)


def test_closed_loop_config1_10_steps_with_periodic_cell_sort(J):
    """Same loop with jefi_sort_particles every 3 steps: trajectories (matched through the tag) keep the 1e-5 bar."""
    w, got, po, hist = run_closed_loop(J, 1, 10, sort_every=3)
    both = (got["alive"] == 1) & (po["alive"] == 1)
    assert (got["alive"] != po["alive"]).sum() <= 1
    for k in "xyz":
        assert np.abs(got[k][both] - po[k][both]).max() / w.n <= 1e-5
    s, E, B, Eo, Bo, S, So = hist[-1]
    assert_field_parity(E, B, Eo, Bo, "cfg1 step 9 (sorted): ")


def test_closed_loop_config1_full_64_steps(J):
    w, got, po, hist = run_closed_loop(J, 1, 64)
    both = (got["alive"] == 1) & (po["alive"] == 1)
    assert (got["alive"] != po["alive"]).sum() <= 2
    for k in "xyz":
        assert np.abs(got[k][both] - po[k][both]).max() / w.n <= 1e-5
    s, E, B, Eo, Bo, S, So = hist[-1]
    assert_field_parity(E, B, Eo, Bo, "cfg1 step 63: ")


# ------------------------------------------------------------------------------------------- errors
def test_error_paths(J):
    import torch

    with pytest.raises(J.JefiError):
        J.jefi_create(0, 4, 4, 1e-4, 1e-4, 1e-4, 1e-13)
    with pytest.raises(J.JefiError):
        J.jefi_create(4, 4, 4, 1e-4, 1e-4, 1e-4, -1.0)
    n, dx = 4, 1e-4
    ctx = make_ctx(J, (n, n, n), (dx, dx, dx), dx / (2 * C), J.JEFI_FIELD_AUTO)
    with pytest.raises(J.JefiError, match="before any"):
        ctx.field_step()
    lib = J.load_library()
    assert lib.jefi_push_sources(ctx.handle, None, None, None, None) == J.JEFI_EINVAL
    assert lib.jefi_field_step(None, None, None, None, None, None, None) == J.JEFI_EINVAL
    lib.jefi_destroy(None)  # NULL is a no-op
    ctx.close()


def test_roofline_probes_report_plausible_numbers(J):
    """jefi_debug_fp32_peak / jefi_debug_lds128_cycles (the denominators bench.py prints next to the derived FP32 peak): the FMA
    pipe delivers most of 148 x 128 x 2 x clock, an LDS.128 costs the data pipe about 2 cycles when every lane pair shares a quad
    and about 4 when one pair differs, and out-of-range modes are refused."""
    n, dx = 4, 1e-4
    ctx = make_ctx(J, (n, n, n), (dx, dx, dx), dx / (2 * C), J.JEFI_FIELD_AUTO)
    derived = 148 * 128 * 2 * 1.965e9 / 1e12
    for mode in range(4):
        r = J.jefi_debug_fp32_peak(ctx.handle, mode)
        assert r["sm_count"] >= 100 and 0.5 * derived < r["tflops"] < 1.1 * derived, (mode, r)
    cyc = [J.jefi_debug_lds128_cycles(ctx.handle, p) for p in range(5)]
    assert 1.5 < cyc[0] < 2.8 and 1.5 < cyc[1] < 2.8 and 3.2 < cyc[2] < 5.5 and 3.2 < cyc[3] < 5.5 and cyc[4] > cyc[1], cyc
    lib = J.load_library()
    import ctypes

    out = ctypes.c_double()
    assert lib.jefi_debug_fp32_peak(ctx.handle, 4, ctypes.byref(out), None) == J.JEFI_EINVAL
    assert lib.jefi_debug_lds128_cycles(ctx.handle, 5, ctypes.byref(out)) == J.JEFI_EINVAL
    ctx.close()
