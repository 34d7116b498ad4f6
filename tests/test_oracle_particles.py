"""Pins of the fp64 particle oracle: Boris invariants, deposit/interp identities."""
import math

import numpy as np

import oracle
from oracle import OracleConfig

C = 299792458.0
EPS0 = 8.8541878128e-12
QE = -1.602176634e-19
ME = 9.1093837015e-31


def make_cfg(n=8, dx=1e-4, **kw):
    return OracleConfig(n, n, n, dx, dx, dx, dx / (2 * C), **kw)


def one_particle(x, u, qm):
    f = lambda v: np.array([v], dtype=np.float64)
    return [f(x[0]), f(x[1]), f(x[2]), f(u[0]), f(u[1]), f(u[2]), f(qm), np.ones(1, dtype=np.uint8)]


# ---------------------------------------------------------------- P11 pure B
def test_p11_boris_pure_B_preserves_speed_gyroradius_and_angle():
    Bz = 10.0  # tesla
    cfg = make_cfg(64, dx=1e-6, Bext=(0.0, 0.0, Bz))
    qm = QE / ME
    u0 = np.array([0.3, 0.0, 0.1])  # relativistic on purpose
    gamma = math.sqrt(1 + u0 @ u0)
    st = one_particle((32.0, 32.0, 32.0), u0, qm)
    zero = np.zeros((3, cfg.N))
    umag, ang = [], []
    prev = u0[:2].copy()
    xs, ys = [], []
    for _ in range(200):
        oracle.push(cfg, *st, zero, zero)
        u = np.array([st[3][0], st[4][0], st[5][0]])
        umag.append(np.linalg.norm(u))
        cur = u[:2]
        ang.append(math.atan2(prev[0] * cur[1] - prev[1] * cur[0], prev @ cur))
        prev = cur.copy()
        xs.append(st[0][0] * cfg.dx)
        ys.append(st[1][0] * cfg.dy)
    assert st[7][0] == 1
    assert np.allclose(umag, np.linalg.norm(u0), rtol=1e-13)  # |u| (hence |v|) constant to rounding
    assert np.isclose(st[5][0], u0[2], rtol=1e-14)  # parallel momentum untouched
    omega_c = qm * Bz  # signed
    expect = 2 * math.atan(omega_c * cfg.dt / (2 * gamma))  # Boris rotation angle per step (sign: d phi = -qB/(gamma m) dt)
    assert np.allclose(ang, -expect, rtol=1e-10)
    # gyroradius: positions lie on a circle of radius gamma m v_perp/(|q| B) * (Boris factor 1/cos(theta/2)... ) -> fit
    xs, ys = np.array(xs), np.array(ys)
    A = np.stack([2 * xs, 2 * ys, np.ones_like(xs)], 1)
    sol, *_ = np.linalg.lstsq(A, xs ** 2 + ys ** 2, rcond=None)
    rad = math.sqrt(sol[2] + sol[0] ** 2 + sol[1] ** 2)
    r_l = C * abs(u0[0]) / (abs(qm) * Bz)  # gamma m v_perp / (|q| B) = c u_perp / (|q/m| B)
    # Boris: radius = v dt / (2 sin(theta/2)) with tan(theta/2) = omega_c dt / (2 gamma)
    th = abs(expect)
    r_boris = (C * abs(u0[0]) / gamma) * cfg.dt / (2 * math.sin(th / 2))
    assert np.isclose(rad, r_boris, rtol=1e-9)
    assert np.isclose(rad, r_l, rtol=1e-3)  # and within O((omega dt)^2) of the physical Larmor radius
    resid = np.sqrt((xs - sol[0]) ** 2 + (ys - sol[1]) ** 2) - rad
    assert np.abs(resid).max() < 1e-9 * rad


# ---------------------------------------------------------------- P12 pure E, and E x B drift
def test_p12_boris_pure_E_momentum_growth_exact():
    Ex = 2.5e6
    cfg = make_cfg(64, dx=1e-3, Eext=(Ex, 0.0, 0.0))
    qm = QE / ME
    st = one_particle((32.0, 32.0, 32.0), (0.0, 0.01, 0.0), qm)
    zero = np.zeros((3, cfg.N))
    for s in range(1, 40):
        oracle.push(cfg, *st, zero, zero)
        assert np.isclose(st[3][0], s * qm * Ex * cfg.dt / C, rtol=1e-13)
        assert st[4][0] == 0.01 and st[5][0] == 0.0


def test_p12_crossed_fields_drift_velocity():
    Ey, Bz = 1.0e5, 0.5  # drift v = E x B / B^2 = (Ey/Bz) x-hat = 2e5 m/s
    cfg = make_cfg(64, dx=1e-3, Eext=(0.0, Ey, 0.0), Bext=(0.0, 0.0, Bz))
    qm = QE / ME
    st = one_particle((20.0, 32.0, 32.0), (0.0, 0.0, 0.0), qm)
    zero = np.zeros((3, cfg.N))
    period = 2 * math.pi / (abs(qm) * Bz)
    nper = 20
    nsteps = int(round(nper * period / cfg.dt))
    x0 = st[0][0]
    for _ in range(nsteps):
        oracle.push(cfg, *st, zero, zero)
    vd = (st[0][0] - x0) * cfg.dx / (nsteps * cfg.dt)
    assert st[7][0] == 1
    assert np.isclose(vd, Ey / Bz, rtol=2e-3)


def test_p12_kill_rule_open_boundary():
    """PAPER.md:205, 239 / reading A13: alive iff every coordinate in [0, n) after the position update; a dead
    particle is neither pushed nor deposited."""
    cfg = make_cfg(8)
    beta = 0.6
    u = beta / math.sqrt(1 - beta * beta)
    step = beta * C * cfg.dt / cfg.dx  # 0.3 cells per step
    st = one_particle((7.5, 4.0, 4.0), (u, 0.0, 0.0), QE / ME)
    zero = np.zeros((3, cfg.N))
    oracle.push(cfg, *st, zero, zero)
    assert st[7][0] == 1 and np.isclose(st[0][0], 7.5 + step, rtol=1e-14)
    oracle.push(cfg, *st, zero, zero)
    assert st[7][0] == 0 and st[0][0] >= 8.0
    frozen = st[0][0]
    oracle.push(cfg, *st, zero, zero)
    assert st[0][0] == frozen  # no longer pushed
    S = oracle.deposit(cfg, st[0], st[1], st[2], st[3], st[4], st[5], np.array([QE]), st[7])
    assert np.all(S == 0.0)  # no longer a source


# ---------------------------------------------------------------- P13 deposit
def test_p13_deposit_charge_conservation_and_cell_centre():
    cfg = make_cfg(8)
    rng = np.random.default_rng(13)
    P = 500
    x, y, z = (rng.uniform(0.5, 7.5, P) for _ in range(3))  # interior: all 8 nodes inside
    u = rng.normal(0, 0.2, (3, P))
    qw = rng.uniform(-2, 2, P) * 1e-13
    S = oracle.deposit(cfg, x, y, z, u[0], u[1], u[2], qw)
    dV = cfg.dx ** 3
    assert np.isclose(S[0].sum() * dV, qw.sum(), rtol=1e-12)
    v = C * u / np.sqrt(1 + (u ** 2).sum(0))
    for a in range(3):
        assert np.isclose(S[1 + a].sum() * dV, (qw * v[a]).sum(), rtol=1e-11)
    # particle exactly at a cell centre -> everything in that cell
    S1 = oracle.deposit(cfg, [3.5], [2.5], [6.5], [0.1], [0.0], [0.0], [1e-13])
    c = 3 + 8 * (2 + 8 * 6)
    assert np.isclose(S1[0, c], 1e-13 / dV, rtol=1e-15) and np.count_nonzero(S1[0]) == 1
    assert np.isclose(S1[1, c], S1[0, c] * C * 0.1 / math.sqrt(1.01), rtol=1e-14)


def test_p13_deposit_weights_and_virtual_nodes():
    cfg = make_cfg(8)
    dV = cfg.dx ** 3
    q = 1e-13
    # alpha = 0.25, beta = 0.5, chi = 0.75 around node (2,3,4): hand-written trilinear weights (Eq. 2.16)
    S = oracle.deposit(cfg, [2.75], [4.0], [5.25], [0.0], [0.0], [0.0], [q])
    al, be, ch = 0.25, 0.5, 0.75
    for a in (0, 1):
        for b in (0, 1):
            for c in (0, 1):
                w = (al if a else 1 - al) * (be if b else 1 - be) * (ch if c else 1 - ch)
                assert np.isclose(S[0, (2 + a) + 8 * ((3 + b) + 8 * (4 + c))], q * w / dV, rtol=1e-13)
    assert np.count_nonzero(S[0]) == 8
    # within half a cell of the x=0 face: i = -1 is virtual, its share (1-alpha) is lost
    S = oracle.deposit(cfg, [0.2], [4.5], [4.5], [0.0], [0.0], [0.0], [q])
    alpha = 0.2 - 0.5 + 1.0
    assert np.isclose(S[0].sum() * dV, q * alpha, rtol=1e-13) and np.count_nonzero(S[0]) == 1
    # corner: only one of the eight nodes is real
    S = oracle.deposit(cfg, [7.9], [7.8], [0.1], [0.0], [0.0], [0.0], [q])
    assert np.count_nonzero(S[0]) == 1
    assert np.isclose(S[0, 7 + 8 * (7 + 8 * 0)] * dV, q * (1 - 0.4) * (1 - 0.3) * 0.6, rtol=1e-12)
    idx = oracle.cell_index([0.2, 0.5, 7.9, 0.49999, 3.5], [4.5] * 5, [0.1] * 5)
    assert idx[:, 0].tolist() == [-1, 0, 7, -1, 3] and idx[0, 2] == -1 and idx[0, 1] == 4


# ---------------------------------------------------------------- P14 interpolation
def test_p14_interpolation_reproduces_uniform_and_linear_fields():
    cfg = make_cfg(8)
    k, j, i = np.meshgrid(np.arange(8), np.arange(8), np.arange(8), indexing="ij")
    xc, yc, zc = i.ravel() + 0.5, j.ravel() + 0.5, k.ravel() + 0.5  # cell centres in grid units
    F = np.stack([np.full(cfg.N, 3.0), 2.0 * xc - yc + 0.5 * zc + 1.0, -xc + 4.0 * zc], 0)
    rng = np.random.default_rng(14)
    P = 200
    x, y, z = (rng.uniform(0.5, 7.5, P) for _ in range(3))
    out = oracle.interp(cfg, x, y, z, F)
    assert np.allclose(out[:, 0], 3.0, rtol=1e-14)
    assert np.allclose(out[:, 1], 2.0 * x - y + 0.5 * z + 1.0, rtol=1e-13)
    assert np.allclose(out[:, 2], -x + 4.0 * z, rtol=1e-13, atol=1e-13)
    # reading A12: near a face the virtual nodes count as zero and weights are not renormalised
    out = oracle.interp(cfg, [0.25], [4.5], [4.5], F)
    assert np.isclose(out[0, 0], 3.0 * 0.75, rtol=1e-14)


# ---------------------------------------------------------------- P15 loop wiring
def test_p15_two_macro_charges_first_step_is_coulomb_between_clouds():
    n = 12
    cfg = make_cfg(n)
    q = -1.602176634e-13
    pa, pb = np.array([3.5, 5.5, 5.5]), np.array([8.5, 5.5, 5.5])  # at cell centres, 5 cells apart, at rest
    part = dict(x=np.array([pa[0], pb[0]]), y=np.array([pa[1], pb[1]]), z=np.array([pa[2], pb[2]]),
                ux=np.zeros(2), uy=np.zeros(2), uz=np.zeros(2), qw=np.array([q, q]),
                qm=np.array([QE / ME, QE / ME]), alive=np.ones(2, dtype=np.uint8))
    orc = oracle.OracleJefi(cfg)
    # hold the charges fixed until the retarded field of one has reached the other (m = 10), then push once
    for _ in range(12):
        S = orc.deposit(part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"], part["qw"], part["alive"])
        orc.push_sources(*S)
    E, B = orc.field_step()
    orc.push_particles(part["x"], part["y"], part["z"], part["ux"], part["uy"], part["uz"], part["qm"], part["alive"], E, B)
    R = 5 * cfg.dx
    Ecoul = q / (4 * math.pi * EPS0 * R * R)  # field of the other macro-charge at this one (each fills one cell)
    du = (QE / ME) * Ecoul * cfg.dt / C
    assert np.isclose(part["ux"][0], -du, rtol=1e-12)  # like charges repel: particle a is pushed to -x
    assert np.isclose(part["ux"][1], +du, rtol=1e-12)
    assert part["uy"][0] == 0.0 and part["uz"][1] == 0.0
    v = C * part["ux"][1] / math.sqrt(1 + part["ux"][1] ** 2)
    assert np.isclose(part["x"][1], pb[0] + v * cfg.dt / cfg.dx, rtol=1e-15)


# ---------------------------------------------------------------- P16 which gamma the rotation uses when E != 0 and B != 0
def _rotated(ux, uy, ang):
    return ux * math.cos(ang) - uy * math.sin(ang), ux * math.sin(ang) + uy * math.cos(ang)


def _p16_case(sign, E, u0, via_grid):
    """Heaviside-Lorentz-like units c = 1, dt = 2, q/m = sign (h = (q/m) dt/2 = sign), B = (0, 0, 2).  Expected values are
    written out by hand from Eqs. (2.9)-(2.11) in the relativistic reading A6:
      u^- = u + h E/c;  gamma^- = sqrt(1 + |u^-|^2);  the rotation of Eq. (2.10) turns the part of u^- perpendicular to B by
      theta = 2 atan(h B/gamma^-) (clockwise about B for h B > 0, the pinned direction of P11);  u^{n+1/2} = u^+ + h E/c.
    The numbers are chosen so that |u^-|^2 = 3 exactly: gamma^- = 2, |h| B/gamma^- = 1, theta = 90 degrees, i.e. the
    perpendicular part goes (a, b) -> (b, -a) for h > 0 and (a, b) -> (-b, a) for h < 0.  Taking gamma from u^{n-1/2}
    instead (sqrt(2) or sqrt(3) here) turns by 109.5 / 98.2 degrees: every component is then off by > 0.1."""
    n, dx, dt = 8, 100.0, 2.0
    kw = dict(c=1.0, eps0=1.0)
    Bz = 2.0
    if via_grid:
        cfg = OracleConfig(n, n, n, dx, dx, dx, dt, **kw)
        Eg = np.repeat(np.array(E, dtype=np.float64)[:, None], cfg.N, 1)
        Bg = np.repeat(np.array([0.0, 0.0, Bz])[:, None], cfg.N, 1)
    else:
        cfg = OracleConfig(n, n, n, dx, dx, dx, dt, Eext=tuple(E), Bext=(0.0, 0.0, Bz), **kw)
        Eg = Bg = np.zeros((3, cfg.N))
    r0 = (4.0, 4.0, 4.0)  # interior: all 8 nodes inside, weights sum to 1 (P14), so a uniform grid field is exact
    st = one_particle(r0, u0, float(sign))
    oracle.push(cfg, *st, Eg, Bg)
    return cfg, r0, np.array([st[0][0], st[1][0], st[2][0]]), np.array([st[3][0], st[4][0], st[5][0]]), st[7][0]


def test_p16_boris_gamma_of_u_minus_E_parallel_B():
    """E || B (both along z), u^{n-1/2} = (0.6, 0.8, 0), h E/c = +-sqrt(2): u^- = (0.6, 0.8, +-sqrt 2), |u^-|^2 = 3."""
    r2 = math.sqrt(2.0)
    for sign in (+1.0, -1.0):
        for via_grid in (False, True):
            cfg, r0, r1, u1, alive = _p16_case(sign, (0.0, 0.0, r2), (0.6, 0.8, 0.0), via_grid)
            # perpendicular part (0.6, 0.8) turned by -+90 degrees; parallel part kicked twice by h E/c = sign sqrt 2
            want_u = np.array([0.8, -0.6, 2 * r2]) if sign > 0 else np.array([-0.8, 0.6, -2 * r2])
            assert np.allclose(u1, want_u, rtol=0, atol=1e-14), (sign, via_grid, u1)
            g1 = math.sqrt(1.0 + 1.0 + 8.0)  # |u_new|^2 = 0.64 + 0.36 + 8
            want_r = np.array(r0) + want_u / g1 * cfg.dt / cfg.dx  # Eq. (2.8), v = c u/gamma, grid units
            assert np.allclose(r1, want_r, rtol=0, atol=1e-14) and alive == 1
            # the misreading gamma(u^{n-1/2}) = sqrt 2 would turn by 2 atan(2/sqrt 2) instead: far outside 1e-6
            bad = _rotated(0.6, 0.8, -sign * 2 * math.atan(2.0 / r2))
            assert abs(bad[0] - want_u[0]) > 0.1


def test_p16_boris_gamma_of_u_minus_E_perpendicular_B():
    """E along x, B along z, u^{n-1/2} = (0, 1, 1), h E/c = +-1: u^- = (+-1, 1, 1), |u^-|^2 = 3, gamma^- = 2."""
    for sign in (+1.0, -1.0):
        for via_grid in (False, True):
            cfg, r0, r1, u1, alive = _p16_case(sign, (1.0, 0.0, 0.0), (0.0, 1.0, 1.0), via_grid)
            # h > 0: u^- = (1, 1, 1) -> u^+ = (1, -1, 1) -> + (1, 0, 0);  h < 0: u^- = (-1, 1, 1) -> u^+ = (-1, -1, 1) -> + (-1, 0, 0)
            want_u = np.array([2.0, -1.0, 1.0]) if sign > 0 else np.array([-2.0, -1.0, 1.0])
            assert np.allclose(u1, want_u, rtol=0, atol=1e-14), (sign, via_grid, u1)
            g1 = math.sqrt(7.0)
            want_r = np.array(r0) + want_u / g1 * cfg.dt / cfg.dx
            assert np.allclose(r1, want_r, rtol=0, atol=1e-14) and alive == 1
            # gamma(u^{n-1/2}) = sqrt 3 would give tan(theta/2) = 2/sqrt 3
            bad = _rotated(sign * 1.0, 1.0, -sign * 2 * math.atan(2.0 / math.sqrt(3.0)))
            assert abs(bad[1] - (-1.0)) > 0.1
