"""Pins of the fp64 field oracle: closed forms, invariants, brute force.

None of these re-call the oracle to check itself: each expectation is a textbook formula, an invariant, a
value the paper prints, or a separately written dense numpy enumeration.
"""
import math
import os

import numpy as np
import pytest

import oracle
from oracle import OracleConfig

C = 299792458.0
EPS0 = 8.8541878128e-12
MU0 = 1.0 / (EPS0 * C * C)
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def make_cfg(n, dx=1e-4, kappa=2.0, **kw):
    if isinstance(n, int):
        n = (n, n, n)
    return OracleConfig(n[0], n[1], n[2], dx, dx, dx, dx / (kappa * C), **kw)


def centres(cfg):
    k, j, i = np.meshgrid(np.arange(cfg.nz), np.arange(cfg.ny), np.arange(cfg.nx), indexing="ij")
    return np.stack([(i.ravel() + 0.5) * cfg.dx, (j.ravel() + 0.5) * cfg.dy, (k.ravel() + 0.5) * cfg.dz], 0)


def static_ring(cfg, S):
    """The same [4][N] source in every slot (held since long before step n)."""
    return np.ascontiguousarray(np.broadcast_to(S, (cfg.H, 4, cfg.N)))


def cidx(cfg, i, j, k):
    return i + cfg.nx * (j + cfg.ny * k)


# ---------------------------------------------------------------- golden values the paper / BASELINE print
def test_golden_ndt_values():
    """PAPER.md:432 (§3.4): 20^3 cells, dx = 0.3, dt = 0.05, c = 1 -> sqrt(3*(20*0.3)^2)/dt ~ 207 steps;
    BASELINE.json configs: H = 58, 113, 224, 335, 446 for the five grids."""
    rows = [l.split() for l in open(os.path.join(GOLDEN, "ndt_values.txt")) if l.strip() and not l.startswith("#")]
    for n, dx, dt, c, lo, hi, H in rows:
        n, dx, dt, c = int(n), float(dx), float(dt) if dt != "dx/2c" else None, float(c)
        if dt is None:
            dt = dx / (2 * c)
        cfg = OracleConfig(n, n, n, dx, dx, dx, dt, c=c, eps0=1.0 if c == 1.0 else EPS0)
        ndt = oracle.num_dt(cfg)
        assert int(lo) <= ndt <= int(hi), (n, ndt)
        assert cfg.H == int(H)


def test_hist_cap_limits_ndt():
    """N_dt = min(N_dt, 10000)."""
    cfg = OracleConfig(8, 8, 8, 1.0, 1.0, 1.0, 1e-4, c=1.0, eps0=1.0, H=4)
    assert oracle.num_dt(cfg) == 10000
    cfg2 = OracleConfig(8, 8, 8, 1.0, 1.0, 1.0, 1e-4, c=1.0, eps0=1.0, H=4, hist_cap=50)
    assert oracle.num_dt(cfg2) == 50


# ---------------------------------------------------------------- P1 Coulomb
def test_p1_static_charge_is_coulomb_direct_sum():
    cfg = make_cfg((7, 6, 5))
    rng = np.random.default_rng(1)
    S = np.zeros((4, cfg.N))
    S[0] = rng.uniform(-1, 1, cfg.N)
    E, B = oracle.field(cfg, 10 * cfg.H, static_ring(cfg, S))
    r = centres(cfg)
    d = r[:, :, None] - r[:, None, :]  # [3][obs][src]
    R = np.sqrt((d ** 2).sum(0))
    np.fill_diagonal(R, np.inf)
    dV = cfg.dx * cfg.dy * cfg.dz
    Ec = dV / (4 * math.pi * EPS0) * (d * S[0][None, None, :] / R ** 3).sum(2)
    assert np.allclose(E, Ec, rtol=1e-12, atol=1e-12 * np.abs(Ec).max())
    assert np.all(B == 0.0)


def test_p1_single_cell_point_charge_magnitude_and_direction():
    cfg = make_cfg(9)
    S = np.zeros((4, cfg.N))
    src = (4, 4, 4)
    rho = 3.5e-3
    S[0, cidx(cfg, *src)] = rho
    E, _ = oracle.field(cfg, 5 * cfg.H, static_ring(cfg, S))
    Q = rho * cfg.dx ** 3
    for obs in [(8, 4, 4), (4, 0, 4), (6, 7, 1), (0, 0, 0), (5, 4, 4)]:
        d = (np.array(obs) - np.array(src)) * cfg.dx
        R = np.linalg.norm(d)
        e = E[:, cidx(cfg, *obs)]
        assert np.isclose(np.linalg.norm(e), Q / (4 * math.pi * EPS0 * R * R), rtol=1e-13)
        assert np.allclose(e / np.linalg.norm(e), d / R, atol=1e-13)  # radial, pointing away from +Q
    assert np.all(E[:, cidx(cfg, *src)] == 0.0)  # self cell skipped


# ---------------------------------------------------------------- P2 Biot-Savart
def test_p2_steady_current_is_biot_savart_direct_sum():
    cfg = make_cfg((5, 7, 6))
    rng = np.random.default_rng(2)
    S = np.zeros((4, cfg.N))
    S[1:] = rng.uniform(-1, 1, (3, cfg.N))
    E, B = oracle.field(cfg, 10 * cfg.H, static_ring(cfg, S))
    r = centres(cfg)
    d = r[:, :, None] - r[:, None, :]
    R = np.sqrt((d ** 2).sum(0))
    np.fill_diagonal(R, np.inf)
    dV = cfg.dx ** 3
    J = S[1:][:, None, :]
    # Biot-Savart: B = mu0/(4 pi) sum J x (r - r') / R^3 dV
    JxD = np.stack([J[1] * d[2] - J[2] * d[1], J[2] * d[0] - J[0] * d[2], J[0] * d[1] - J[1] * d[0]], 0)
    Bc = MU0 / (4 * math.pi) * dV * (JxD / R ** 3).sum(2)
    assert np.allclose(B, Bc, rtol=1e-12, atol=1e-12 * np.abs(Bc).max())
    assert np.all(E == 0.0)  # rho = 0 and J steady -> no E at all


def test_p2_line_current_right_handed_mu0_I_over_2_pi_r():
    """A z-directed line of current cells: B_phi -> mu0 I / (2 pi r) (finite-wire formula), right-handed."""
    n = (9, 9, 61)
    cfg = make_cfg(n)
    S = np.zeros((4, cfg.N))
    Jz = 2.0
    for k in range(n[2]):
        S[3, cidx(cfg, 4, 4, k)] = Jz
    _, B = oracle.field(cfg, 10 * cfg.H, static_ring(cfg, S))
    I = Jz * cfg.dx * cfg.dy
    kmid = n[2] // 2
    for r_cells in (2, 3, 4):
        obs = cidx(cfg, 4 + r_cells, 4, kmid)  # on the +x side: phi-hat = +y
        r = r_cells * cfg.dx
        half = (n[2] / 2) * cfg.dz
        exact_finite = MU0 * I / (2 * math.pi * r) * half / math.hypot(half, r)
        assert B[1, obs] > 0  # right-handed about +z
        assert abs(B[0, obs]) < 1e-12 * abs(B[1, obs]) and abs(B[2, obs]) < 1e-12 * abs(B[1, obs])
        assert np.isclose(B[1, obs], exact_finite, rtol=0.03)  # midpoint-rule discretisation error
    obs = cidx(cfg, 4, 4 + 3, kmid)  # on the +y side: phi-hat = -x
    assert B[0, obs] < 0


# ---------------------------------------------------------------- P3 light cone
def test_p3_outside_light_cone_is_bitwise_zero():
    cfg = make_cfg(10)
    src = (2, 3, 1)
    n0, n = 5, 17
    ring = np.zeros((cfg.H, 4, cfg.N))
    rng = np.random.default_rng(3)
    for t in range(n0, n + 1):  # source switched on at step n0 (zero before)
        ring[t % cfg.H, :, cidx(cfg, *src)] = rng.uniform(-1, 1, 4)
    E, B = oracle.field(cfg, n, ring)
    nin = nout = 0
    for k in range(10):
        for j in range(10):
            for i in range(10):
                R = cfg.dx * math.sqrt((i - src[0]) ** 2 + (j - src[1]) ** 2 + (k - src[2]) ** 2)
                m = math.floor(R / (C * cfg.dt) + 0.5)
                o = cidx(cfg, i, j, k)
                if m > n - n0:
                    assert np.all(E[:, o] == 0.0) and np.all(B[:, o] == 0.0)
                    nout += 1
                elif (i, j, k) != src:
                    assert np.any(E[:, o] != 0.0)
                    nin += 1
    assert nin > 50 and nout > 50


# ---------------------------------------------------------------- P4 linearity
def test_p4_linearity_in_the_sources():
    cfg = make_cfg((6, 5, 4))
    rng = np.random.default_rng(4)
    r1 = rng.integers(-8, 9, (cfg.H, 4, cfg.N)).astype(np.float64)
    r2 = rng.integers(-8, 9, (cfg.H, 4, cfg.N)).astype(np.float64)
    a, b = 3.0, -0.5
    n = 3 * cfg.H + 1
    E1, B1 = oracle.field(cfg, n, r1)
    E2, B2 = oracle.field(cfg, n, r2)
    E3, B3 = oracle.field(cfg, n, a * r1 + b * r2)
    assert np.allclose(E3, a * E1 + b * E2, rtol=1e-12, atol=1e-12 * np.abs(E3).max())
    assert np.allclose(B3, a * B1 + b * B2, rtol=1e-12, atol=1e-12 * np.abs(B3).max())


# ---------------------------------------------------------------- P5 symmetry
def test_p5_octahedral_static_rho_gives_radial_E_and_zero_B():
    n = 9
    cfg = make_cfg(n)
    k, j, i = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    r2 = (i - 4) ** 2 + (j - 4) ** 2 + (k - 4) ** 2
    S = np.zeros((4, cfg.N))
    S[0] = np.exp(-r2 / 6.0).ravel()  # depends on |r - centre| only -> full cubic symmetry
    E, B = oracle.field(cfg, 10 * cfg.H, static_ring(cfg, S))
    assert np.all(B == 0.0)
    Emax = np.abs(E).max()
    assert np.all(np.abs(E[:, cidx(cfg, 4, 4, 4)]) < 1e-13 * Emax)
    for a in range(1, 5):  # on the axes and the body diagonal E is exactly radial
        e = E[:, cidx(cfg, 4 + a, 4, 4)]
        assert e[0] > 0 and abs(e[1]) < 1e-13 * Emax and abs(e[2]) < 1e-13 * Emax
        e = E[:, cidx(cfg, 4 - a, 4 - a, 4 - a)]
        assert e[0] < 0 and np.allclose(e, e[0], rtol=1e-12)
    r = centres(cfg) - np.array([4.5, 4.5, 4.5])[:, None] * cfg.dx  # everywhere: radial to discretisation error
    rn = np.linalg.norm(r, axis=0)
    en = np.linalg.norm(E, axis=0)
    sel = rn > 0
    cosang = (E * r).sum(0)[sel] / (en[sel] * rn[sel])
    assert cosang.min() > 0.99


# ---------------------------------------------------------------- P6 translation and mirror
def test_p6_translation_and_mirror():
    cfg = make_cfg((8, 7, 6))
    rng = np.random.default_rng(6)
    n = 2 * cfg.H
    hist = np.zeros((cfg.H, 4, cfg.nz, cfg.ny, cfg.nx))
    hist[:, :, 1:4, 1:4, 1:4] = rng.uniform(-1, 1, (cfg.H, 4, 3, 3, 3))
    shift = (3, 2, 1)  # lattice vector (x, y, z)
    hist2 = np.roll(hist, (shift[2], shift[1], shift[0]), axis=(2, 3, 4))
    E1, B1 = oracle.field(cfg, n, hist.reshape(cfg.H, 4, cfg.N))
    E2, B2 = oracle.field(cfg, n, hist2.reshape(cfg.H, 4, cfg.N))
    for obs in [(0, 0, 0), (2, 2, 2), (4, 3, 1), (1, 4, 4)]:
        o1 = cidx(cfg, *obs)
        o2 = cidx(cfg, obs[0] + shift[0], obs[1] + shift[1], obs[2] + shift[2])
        assert np.allclose(E1[:, o1], E2[:, o2], rtol=1e-12) and np.allclose(B1[:, o1], B2[:, o2], rtol=1e-12)
    # mirror x -> -x: rho even, Jx odd; E is polar (Ex flips), B is axial (By, Bz flip)
    hm = hist[:, :, :, :, ::-1].copy()
    hm[:, 1] *= -1.0
    Em, Bm = oracle.field(cfg, n, hm.reshape(cfg.H, 4, cfg.N))
    E1g = E1.reshape(3, cfg.nz, cfg.ny, cfg.nx)[:, :, :, ::-1]
    B1g = B1.reshape(3, cfg.nz, cfg.ny, cfg.nx)[:, :, :, ::-1]
    Emg, Bmg = Em.reshape(3, cfg.nz, cfg.ny, cfg.nx), Bm.reshape(3, cfg.nz, cfg.ny, cfg.nx)
    sE, sB = np.array([-1, 1, 1.0])[:, None, None, None], np.array([1, -1, -1.0])[:, None, None, None]
    assert np.allclose(Emg, sE * E1g, rtol=1e-11, atol=1e-12 * np.abs(E1).max())
    assert np.allclose(Bmg, sB * B1g, rtol=1e-11, atol=1e-12 * np.abs(B1).max())


# ---------------------------------------------------------------- P7 / P8 time-dependent single cell, by hand
def test_p7_rho_sequence_two_sample_formula():
    """One cell with rho(t) a known sequence: E at distance R from Eq. (2.4) written out by hand."""
    cfg = make_cfg(12)
    src, obs = (1, 2, 3), (7, 2, 3)  # R = 6 dx -> s = 12.0 -> m = 12
    n = 40
    seq = lambda t: 0.25 * t * t - 3.0 * t + 1.0
    ring = np.zeros((cfg.H, 4, cfg.N))
    for t in range(n - cfg.H + 1, n + 1):
        if t >= 0:
            ring[t % cfg.H, 0, cidx(cfg, *src)] = seq(t)
    E, B = oracle.field(cfg, n, ring, np.array([cidx(cfg, *obs)]))
    R = 6 * cfg.dx
    m = 12
    rho0, rho1 = seq(n - m), seq(n - m - 1)
    dV = cfg.dx ** 3
    Ex = dV / (4 * math.pi * EPS0) * (R * rho0 / R ** 3 + R * ((rho0 - rho1) / cfg.dt) / (C * R ** 2))
    assert np.isclose(E[0, 0], Ex, rtol=1e-13)
    assert E[1, 0] == 0.0 and E[2, 0] == 0.0 and np.all(B == 0.0)
    # a non-integer delay: R = sqrt(5) dx -> s = 4.472 -> nearest step m = 4 (reading A1)
    obs2 = (2, 4, 3)
    E2, _ = oracle.field(cfg, n, ring, np.array([cidx(cfg, *obs2)]))
    d = np.array([1, 2, 0]) * cfg.dx
    R2 = np.linalg.norm(d)
    r0, r1 = seq(n - 4), seq(n - 5)
    e = dV / (4 * math.pi * EPS0) * (d * r0 / R2 ** 3 + d * ((r0 - r1) / cfg.dt) / (C * R2 ** 2))
    assert np.allclose(E2[:, 0], e, rtol=1e-13)


def test_p8_current_ramp_radiation_terms():
    """One cell with J ramping linearly: E = -(mu0/4pi) dV Jdot / R, B = -(mu0/4pi) dV d x (J/R^3 + Jdot/(c R^2))."""
    cfg = make_cfg(12)
    src, obs = (5, 5, 5), (8, 9, 5)  # d = (3, 4, 0) dx, R = 5 dx, m = 10
    n = 50
    slope = np.array([0.3, -0.2, 0.7])  # per step
    ring = np.zeros((cfg.H, 4, cfg.N))
    for t in range(n - cfg.H + 1, n + 1):
        ring[t % cfg.H, 1:, cidx(cfg, *src)] = slope * t
    E, B = oracle.field(cfg, n, ring, np.array([cidx(cfg, *obs)]))
    d = np.array([3, 4, 0]) * cfg.dx
    R = 5 * cfg.dx
    Jdot = slope / cfg.dt
    J0 = slope * (n - 10)
    dV = cfg.dx ** 3
    Eh = -(MU0 / (4 * math.pi)) * dV * Jdot / R
    Bh = -(MU0 / (4 * math.pi)) * dV * np.cross(d, J0 / R ** 3 + Jdot / (C * R ** 2))
    assert np.allclose(E[:, 0], Eh, rtol=1e-12)
    assert np.allclose(B[:, 0], Bh, rtol=1e-12)


# ---------------------------------------------------------------- P9 the paper's analytic-source example
def analytic_ring(cfg, n, depth):
    """Eqs. (3.4)-(3.5), sampled at cell centres, steps max(0, n-depth+1)..n."""
    r = centres(cfg)
    ph = r.sum(0)
    ring = np.zeros((depth, 4, cfg.N))
    for t in range(max(0, n - depth + 1), n + 1):
        tt = t * cfg.dt
        ring[t % depth, 0] = 3.0 * (math.cos(tt) - 1.0) * np.cos(ph)
        ring[t % depth, 1:] = np.sin(ph) * math.sin(tt)
    return ring


def test_p9_history_depth_insensitivity_above_ndt():
    """20^3, dx=0.3, dt=0.05, c=eps0=mu0=1; depths >= N_dt+2 agree, depths well below differ."""
    n = 10  # grid 10^3 keeps the CPU suite fast; same dx, dt, units as the paper's example
    cfg0 = OracleConfig(n, n, n, 0.3, 0.3, 0.3, 0.05, c=1.0, eps0=1.0)
    ndt = oracle.num_dt(cfg0)
    assert ndt == math.ceil(math.sqrt(3) * n * 0.3 / 0.05)
    step = 400
    obs = np.array([0, 5 + 10 * (5 + 10 * 5), 999, 37])
    res = {}
    for depth in (ndt + 2, ndt + 30, 2 * ndt, ndt // 2, ndt // 4):
        cfg = OracleConfig(n, n, n, 0.3, 0.3, 0.3, 0.05, c=1.0, eps0=1.0, H=depth)
        res[depth] = oracle.field(cfg, step, analytic_ring(cfg, step, depth), obs)
    E0, B0 = res[ndt + 2]
    for depth in (ndt + 30, 2 * ndt):
        assert np.array_equal(res[depth][0], E0) and np.array_equal(res[depth][1], B0)  # bitwise
    for depth in (ndt // 2, ndt // 4):
        assert np.abs(res[depth][0] - E0).max() > 1e-3 * np.abs(E0).max()  # truncated history visibly differs


# ---------------------------------------------------------------- P10 brute force on tiny grids
def dense_jefimenko(shape, h, dt, c, eps0, n, hist):
    """Separately written dense (N_obs x N_src) numpy evaluation; hist[t] = [4][N] for absolute steps t>=0."""
    nx, ny, nz = shape
    N = nx * ny * nz
    ids = np.arange(N)
    pos = np.stack([ids % nx, (ids // nx) % ny, ids // (nx * ny)], 1) * np.array(h)  # [N][3]
    D = pos[:, None, :] - pos[None, :, :]  # obs - src
    R = np.linalg.norm(D, axis=2)
    lag = np.floor(R / (c * dt) + 0.5).astype(int)
    mask = ~np.eye(N, dtype=bool)
    src = np.broadcast_to(ids[None, :], (N, N))

    def sample(t):
        out = np.zeros((4, N, N))
        ok = t >= 0
        tt = np.where(ok, t, 0)
        for comp in range(4):
            out[comp] = np.where(ok, hist[tt, comp, src], 0.0)
        return out

    S0, S1 = sample(n - lag), sample(n - lag - 1)
    dS = (S0 - S1) / dt
    Rs = np.where(mask, R, 1.0)
    mu0 = 1.0 / (eps0 * c * c)
    dV = h[0] * h[1] * h[2]
    E = np.zeros((3, N))
    W = np.zeros((3, N, N))
    for a in range(3):
        term = D[:, :, a] * S0[0] / Rs ** 3 + D[:, :, a] * dS[0] / (c * Rs ** 2) - dS[1 + a] / (c * c * Rs)
        E[a] = dV / (4 * np.pi * eps0) * (term * mask).sum(1)
        W[a] = (S0[1 + a] / Rs ** 3 + dS[1 + a] / (c * Rs ** 2)) * mask
    Bv = np.stack([D[:, :, 1] * W[2] - D[:, :, 2] * W[1], D[:, :, 2] * W[0] - D[:, :, 0] * W[2],
                   D[:, :, 0] * W[1] - D[:, :, 1] * W[0]], 0).sum(2)
    return E, -mu0 * dV / (4 * np.pi) * Bv


@pytest.mark.parametrize("shape,h,kappa", [((2, 2, 2), (1.0, 1.0, 1.0), 2.0), ((3, 3, 3), (1.0, 1.0, 1.0), 2.0),
                                           ((4, 4, 4), (1.0, 1.0, 1.0), 2.0), ((4, 3, 2), (1.0, 0.7, 1.3), 1.37),
                                           ((3, 4, 2), (0.5, 1.0, 2.0), 0.4)])
def test_p10_brute_force_tiny_grids(shape, h, kappa):
    c, eps0 = 1.0, 1.0
    dt = h[0] / (kappa * c)
    cfg = OracleConfig(shape[0], shape[1], shape[2], h[0], h[1], h[2], dt, c=c, eps0=eps0)
    rng = np.random.default_rng(10)
    nsteps = 3 * cfg.H
    hist = rng.uniform(-1, 1, (nsteps, 4, cfg.N))
    for n in (0, 1, 2, cfg.H // 2, nsteps - 1):
        ring = np.zeros((cfg.H, 4, cfg.N))
        for t in range(max(0, n - cfg.H + 1), n + 1):
            ring[t % cfg.H] = hist[t]
        E, B = oracle.field(cfg, n, ring)
        Ed, Bd = dense_jefimenko(shape, h, dt, c, eps0, n, hist)
        assert np.allclose(E, Ed, rtol=1e-11, atol=1e-12 * max(1e-300, np.abs(Ed).max()))
        assert np.allclose(B, Bd, rtol=1e-11, atol=1e-12 * max(1e-300, np.abs(Bd).max()))


def test_p10_two_cell_case_enumerated_by_hand():
    """2x1x1 grid, c = eps0 = 1, dx = 1, dt = 0.5 (kappa = 2 -> m = 2).  Cell 0 observes cell 1 only."""
    cfg = OracleConfig(2, 1, 1, 1.0, 1.0, 1.0, 0.5, c=1.0, eps0=1.0)
    assert oracle.delay(cfg, 1, 0, 0) == 2
    hist = {3: (2.0, 1.0, -1.0, 0.5), 2: (1.0, 3.0, 2.0, -2.0)}  # cell 1 at steps n-2=3 and n-3=2
    ring = np.zeros((cfg.H, 4, 2))
    for t, v in hist.items():
        ring[t % cfg.H, :, 1] = v
    ring[5 % cfg.H, :, 1] = (9.0, 9.0, 9.0, 9.0)  # step n itself: not yet visible at cell 0
    E, B = oracle.field(cfg, 5, ring)
    # d = r0 - r1 = (-1, 0, 0), R = 1; rho0 = 2, rho_dot = (2-1)/0.5 = 2; J0 = (1,-1,.5), J_dot = ((1-3),(-1-2),(.5+2))/0.5
    k = 1.0 / (4 * math.pi)
    jd = np.array([-4.0, -6.0, 5.0])
    assert np.allclose(E[:, 0], k * np.array([-1 * 2.0 + -1 * 2.0 - jd[0], -jd[1], -jd[2]]), rtol=1e-14)
    w = np.array([1.0, -1.0, 0.5]) + jd  # J0/R^3 + J_dot/(c R^2)
    assert np.allclose(B[:, 0], -k * np.cross([-1.0, 0, 0], w), rtol=1e-14)
    assert np.all(E[:, 1] == 0.0) and np.all(B[:, 1] == 0.0)  # cell 0 holds no sources


def test_a15_delays_beyond_stored_history_contribute_zero():
    cfg = make_cfg(8, H=6)  # far too shallow on purpose: only m <= 4 is stored
    S = np.zeros((4, cfg.N))
    S[0, cidx(cfg, 0, 0, 0)] = 1.0
    E, _ = oracle.field(cfg, 100, static_ring(cfg, S))
    assert np.any(E[:, cidx(cfg, 2, 0, 0)] != 0.0)  # m = 4 <= H-2
    assert np.all(E[:, cidx(cfg, 3, 0, 0)] == 0.0)  # m = 6 > H-2


def test_delay_table_nearest_step_and_no_ties_at_kappa_2():
    """Reading A1: m = floor(s + 1/2); at kappa = 2, s = 2 sqrt(q) is never a half-integer (16 q is even)."""
    cfg = make_cfg(24)
    tab = oracle.delay_table(cfg)
    a = np.arange(24)
    q = (a[None, None, :] ** 2 + a[None, :, None] ** 2 + a[:, None, None] ** 2).astype(np.int64)
    # exact integer characterisation: m is the unique integer with (2m-1)^2 <= 16 q < (2m+1)^2
    m = tab.astype(np.int64)
    assert np.all((m == 0) | ((2 * m - 1) ** 2 <= 16 * q)) and np.all(16 * q < (2 * m + 1) ** 2)
    assert not np.any((2 * m + 1) ** 2 == 16 * q) and not np.any((2 * m - 1) ** 2 == 16 * q)  # no ties
    assert tab[0, 0, 1] == 2 and tab[0, 1, 1] == 3 and tab[1, 1, 1] == 3 and tab[0, 0, 2] == 4
    assert tab.max() <= oracle.num_dt(cfg)


# ---------------------------------------------------------------- the float32-history entry (orc_field_f32)
@pytest.mark.parametrize("rule", [oracle.RULE_NEAREST, oracle.RULE_LINEAR])
def test_f32_history_entry_is_the_f64_entry_on_the_same_values(rule):
    """oracle.field dispatches on the ring's dtype: float32 rings (what the full-size GPU parity tests and bench.py's
    cpu_baseline pass, to keep a 335-446-slot history in host memory) go to orc_field_f32, the same Eqs. 2.4-2.6 body on a
    `const float*` history.  Every sample is promoted to double before any arithmetic, so on float32-representable values the
    two entries must agree BIT FOR BIT: for all cells and for a list of observation cells, on a ring that has wrapped and on
    one still filling (zero before t0), and against the separately written dense enumeration, which never sees a float."""
    shape, h, kappa = (5, 4, 3), (1.0, 0.8, 1.25), 1.7
    c, eps0 = 1.0, 1.0
    dt = h[0] / (kappa * c)
    cfg = OracleConfig(*shape, *h, dt, c=c, eps0=eps0, delay_rule=rule)
    rng = np.random.default_rng(32)
    nsteps = 2 * cfg.H + 3
    hist32 = rng.uniform(-1, 1, (nsteps, 4, cfg.N)).astype(np.float32)
    obs = np.array([0, 7, cfg.N - 1, 13, 13], dtype=np.int64)
    for n in (0, 2, cfg.H - 1, nsteps - 1):
        ring32 = np.zeros((cfg.H, 4, cfg.N), dtype=np.float32)
        for t in range(max(0, n - cfg.H + 1), n + 1):
            ring32[t % cfg.H] = hist32[t]
        ring64 = ring32.astype(np.float64)
        E32, B32 = oracle.field(cfg, n, ring32)
        E64, B64 = oracle.field(cfg, n, ring64)
        assert E32.dtype == np.float64 and np.array_equal(E32, E64) and np.array_equal(B32, B64)
        Eo32, Bo32 = oracle.field(cfg, n, ring32, obs)
        assert np.array_equal(Eo32, E64[:, obs]) and np.array_equal(Bo32, B64[:, obs])
        if rule == oracle.RULE_NEAREST:
            Ed, Bd = dense_jefimenko(shape, h, dt, c, eps0, n, hist32.astype(np.float64))
            assert np.allclose(E32, Ed, rtol=1e-11, atol=1e-12 * max(1e-300, np.abs(Ed).max()))
            assert np.allclose(B32, Bd, rtol=1e-11, atol=1e-12 * max(1e-300, np.abs(Bd).max()))
    # the two entries are told apart by dtype alone: a float32 ring whose values are NOT what the float64 ring holds must differ
    ring64 = rng.uniform(-1, 1, (cfg.H, 4, cfg.N))
    Ea, _ = oracle.field(cfg, 3 * cfg.H, ring64)
    Eb, _ = oracle.field(cfg, 3 * cfg.H, ring64.astype(np.float32))
    assert not np.array_equal(Ea, Eb) and np.allclose(Ea, Eb, rtol=0, atol=1e-6 * np.abs(Ea).max())
