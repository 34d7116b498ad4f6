"""Pins of the oracle's linear-in-time retarded rule (reading A22 in DESIGN.md §3).

Rule: m = floor(R/(c dt) + 1/2) as in reading A1, phi = R/(c dt) - m in [-1/2, 1/2); values on the line through the two
samples A1 uses, S^{n-m} - phi (S^{n-m} - S^{n-m-1}); derivatives (S^{n-m} - S^{n-m-1})/dt.
As for the nearest rule, nothing here re-calls the oracle to check itself:
  L1  sources linear in time: the line is exact, and Jefimenko's retardation and derivative terms cancel, so E is the
      Coulomb sum of the PRESENT charge, B the Biot-Savart sum of the PRESENT current, plus -mu0/(4 pi) J_dot/R
  L2  where R/(c dt) is an exact integer (axis-aligned offsets at kappa = 2) phi = 0: bitwise the nearest rule
  L3  one source cell with a known sequence: the two-sample formula with phi written by hand (phi > 0 and phi < 0)
  L4  separately written dense numpy enumeration on tiny and anisotropic grids
  L5  light cone: an observation cell with m > n - n0 sees exactly zero
  L6  a smooth source: the value error falls 4x when dt is halved (second order), the nearest rule's only 2x
"""
import math

import numpy as np
import pytest

import oracle
from oracle import OracleConfig, RULE_LINEAR, RULE_NEAREST

C = 299792458.0
EPS0 = 8.8541878128e-12
MU0 = 1.0 / (EPS0 * C * C)


def make_cfg(n, dx=1e-4, kappa=2.0, **kw):
    if isinstance(n, int):
        n = (n, n, n)
    return OracleConfig(n[0], n[1], n[2], dx, dx, dx, dx / (kappa * C), delay_rule=RULE_LINEAR, **kw)


def centres(cfg):
    k, j, i = np.meshgrid(np.arange(cfg.nz), np.arange(cfg.ny), np.arange(cfg.nx), indexing="ij")
    return np.stack([(i.ravel() + 0.5) * cfg.dx, (j.ravel() + 0.5) * cfg.dy, (k.ravel() + 0.5) * cfg.dz], 0)


def ring_of(cfg, n, fn):
    """ring[t mod H] = fn(t) for the H most recent steps t <= n (older steps are not stored)."""
    ring = np.zeros((cfg.H, 4, cfg.N))
    for t in range(max(0, n - cfg.H + 1), n + 1):
        ring[t % cfg.H] = fn(t)
    return ring


# ---------------------------------------------------------------- L1
def test_L1_sources_linear_in_time_give_present_time_coulomb_and_biot_savart():
    cfg = make_cfg((7, 6, 5), kappa=2.0)
    rng = np.random.default_rng(1)
    a = rng.normal(size=(4, cfg.N))
    b = rng.normal(size=(4, cfg.N)) / (100 * cfg.dt)  # per second
    a[1:] *= C
    b[1:] *= C
    n = cfg.H + 5  # every sample any pair uses lies on the linear ramp (no step before 0 is touched)
    ring = ring_of(cfg, n, lambda t: a + b * (t * cfg.dt))
    E, B = oracle.field(cfg, n, ring)
    # independent closed form: present-time sources S(t_n); only the radiation term of E keeps the derivative
    Sn = a + b * (n * cfg.dt)
    pos = centres(cfg)
    dV = cfg.dx * cfg.dy * cfg.dz
    Ex = np.zeros((3, cfg.N))
    Bx = np.zeros((3, cfg.N))
    for o in range(cfg.N):
        d = pos[:, o:o + 1] - pos  # r - r'
        R = np.linalg.norm(d, axis=0)
        R[o] = np.inf
        Ex[:, o] = dV / (4 * math.pi * EPS0) * ((d * Sn[0] / R ** 3).sum(1)) - MU0 * dV / (4 * math.pi) * (b[1:] / R).sum(1)
        J = Sn[1:]
        cr = np.cross(J.T, d.T).T  # J x d
        Bx[:, o] = MU0 * dV / (4 * math.pi) * (cr / R ** 3).sum(1)
    assert np.abs(E - Ex).max() <= 1e-9 * np.abs(Ex).max()
    assert np.abs(B - Bx).max() <= 1e-9 * np.abs(Bx).max()
    # the nearest rule does NOT have this property (it mis-times every non-integer delay)
    En, _ = oracle.field(cfg, n, ring, rule=RULE_NEAREST)
    assert np.abs(En - Ex).max() > 1e-4 * np.abs(Ex).max()


# ---------------------------------------------------------------- L2
def test_L2_integer_delays_reduce_to_nearest_rule_bitwise():
    cfg = make_cfg(9, kappa=2.0)  # s = 2 |offset|: integer on the axes
    rng = np.random.default_rng(2)
    n = 60
    src = 4 + 9 * (4 + 9 * 4)
    hist = rng.normal(size=(n + 1, 4))

    def fn(t):
        S = np.zeros((4, cfg.N))
        S[:, src] = hist[t]
        return S

    ring = ring_of(cfg, n, fn)
    axis_obs = np.array([i + 9 * (4 + 9 * 4) for i in range(9) if i != 4] + [4 + 9 * (j + 9 * 4) for j in range(9) if j != 4]
                        + [4 + 9 * (4 + 9 * k) for k in range(9) if k != 4])
    El, Bl = oracle.field(cfg, n, ring, axis_obs, rule=RULE_LINEAR)
    En, Bn = oracle.field(cfg, n, ring, axis_obs, rule=RULE_NEAREST)
    assert np.array_equal(El, En) and np.array_equal(Bl, Bn)
    diag = np.array([5 + 9 * (5 + 9 * 5), 0])
    El, _ = oracle.field(cfg, n, ring, diag, rule=RULE_LINEAR)
    En, _ = oracle.field(cfg, n, ring, diag, rule=RULE_NEAREST)
    assert not np.array_equal(El, En)


# ---------------------------------------------------------------- L3
@pytest.mark.parametrize("off,kappa", [((3, 1, 0), 2.0), ((1, 2, 2), 0.7), ((0, 0, 1), 3.3), ((2, 1, 1), 2.0)])
def test_L3_two_sample_formula_with_theta_by_hand(off, kappa):
    cfg = make_cfg(6, kappa=kappa)
    n = 40
    rng = np.random.default_rng(3)
    hist = rng.normal(size=(n + 1, 4))
    hist[:, 1:] *= C
    s_i, o_i = (1, 1, 1), (1 + off[0], 1 + off[1], 1 + off[2])
    src = s_i[0] + 6 * (s_i[1] + 6 * s_i[2])
    obs = o_i[0] + 6 * (o_i[1] + 6 * o_i[2])

    def fn(t):
        S = np.zeros((4, cfg.N))
        S[:, src] = hist[t]
        return S

    E, B = oracle.field(cfg, n, ring_of(cfg, n, fn), np.array([obs]))
    d = np.array(off, dtype=float) * cfg.dx
    R = float(np.linalg.norm(d))
    s = R / (C * cfg.dt)
    m = math.floor(s + 0.5)
    phi = s - m
    S0, S1 = hist[n - m], hist[n - m - 1]
    val = S0 - phi * (S0 - S1)
    dot = (S0 - S1) / cfg.dt
    dV = cfg.dx ** 3
    Eh = dV / (4 * math.pi * EPS0) * (d * val[0] / R ** 3 + d * dot[0] / (C * R ** 2) - dot[1:] / (C * C * R))
    Bh = -MU0 * dV / (4 * math.pi) * np.cross(d, val[1:] / R ** 3 + dot[1:] / (C * R ** 2))
    assert np.allclose(E[:, 0], Eh, rtol=1e-12, atol=0)
    assert np.allclose(B[:, 0], Bh, rtol=1e-12, atol=1e-30)


# ---------------------------------------------------------------- L4
def dense_linear(shape, h, dt, c, eps0, n, hist):
    """Separately written dense (N_obs x N_src) numpy evaluation of the linear rule; hist[t] = [4][N], t >= 0."""
    nx, ny, nz = shape
    N = nx * ny * nz
    ids = np.arange(N)
    pos = np.stack([ids % nx, (ids // nx) % ny, ids // (nx * ny)], 1) * np.array(h)
    D = pos[:, None, :] - pos[None, :, :]
    R = np.linalg.norm(D, axis=2)
    sdel = R / (c * dt)
    lag = np.floor(sdel + 0.5).astype(int)
    phi = sdel - lag
    src = np.broadcast_to(ids[None, :], (N, N))

    def sample(t):
        ok = t >= 0
        tt = np.where(ok, t, 0)
        return np.stack([np.where(ok, hist[tt, comp, src], 0.0) for comp in range(4)])

    S0, S1 = sample(n - lag), sample(n - lag - 1)
    dS = (S0 - S1) / dt
    V = S0 - phi * dt * dS
    Rs = np.where(np.eye(N, dtype=bool), 1.0, R)
    off = ~np.eye(N, dtype=bool)
    mu0 = 1.0 / (eps0 * c * c)
    dV = h[0] * h[1] * h[2]
    E = np.zeros((3, N))
    W = np.zeros((3, N, N))
    for a in range(3):
        term = D[:, :, a] * V[0] / Rs ** 3 + D[:, :, a] * dS[0] / (c * Rs ** 2) - dS[1 + a] / (c * c * Rs)
        E[a] = dV / (4 * math.pi * eps0) * np.where(off, term, 0.0).sum(1)
        W[a] = np.where(off, V[1 + a] / Rs ** 3 + dS[1 + a] / (c * Rs ** 2), 0.0)
    B = np.zeros((3, N))
    B[0] = (D[:, :, 1] * W[2] - D[:, :, 2] * W[1]).sum(1)
    B[1] = (D[:, :, 2] * W[0] - D[:, :, 0] * W[2]).sum(1)
    B[2] = (D[:, :, 0] * W[1] - D[:, :, 1] * W[0]).sum(1)
    return E, -mu0 * dV / (4 * math.pi) * B


@pytest.mark.parametrize("shape,h,kappa,n", [((2, 2, 2), (1e-4,) * 3, 2.0, 9), ((3, 3, 3), (1e-4,) * 3, 2.0, 3),
                                             ((4, 3, 2), (1e-4, 2e-4, 1.5e-4), 1.3, 20), ((4, 4, 4), (0.3,) * 3, 6.0, 50)])
def test_L4_dense_brute_force(shape, h, kappa, n):
    unit = shape == (4, 4, 4)
    c, eps0 = (1.0, 1.0) if unit else (C, EPS0)
    dt = h[0] / (kappa * c)
    cfg = OracleConfig(*shape, *h, dt, c=c, eps0=eps0, delay_rule=RULE_LINEAR)
    rng = np.random.default_rng(4)
    hist = rng.normal(size=(n + 1, 4, cfg.N))
    hist[:, 1:] *= c
    E, B = oracle.field(cfg, n, ring_of(cfg, n, lambda t: hist[t]))
    Ed, Bd = dense_linear(shape, h, dt, c, eps0, n, hist)
    assert np.allclose(E, Ed, rtol=1e-10, atol=1e-12 * np.abs(Ed).max())
    assert np.allclose(B, Bd, rtol=1e-10, atol=1e-12 * np.abs(Bd).max())


# ---------------------------------------------------------------- L5
def test_L5_light_cone_zero_is_exact():
    cfg = make_cfg(8, kappa=2.0)
    n0, n = 5, 12
    src = 0
    rng = np.random.default_rng(5)

    def fn(t):
        S = np.zeros((4, cfg.N))
        if t >= n0:
            S[:, src] = rng.normal(size=4)
        return S

    E, B = oracle.field(cfg, n, ring_of(cfg, n, fn))
    idx = np.arange(cfg.N)
    i, j, k = idx % 8, (idx // 8) % 8, idx // 64
    q = i ** 2 + j ** 2 + k ** 2
    m = np.floor(2 * np.sqrt(q) + 0.5).astype(int)  # kappa = 2; no ties (16 q is even, (2k+1)^2 odd)
    outside = m > n - n0  # both samples of the pair are older than the switch-on
    assert outside.any() and (~outside).sum() > 1
    assert np.all(E[:, outside] == 0.0) and np.all(B[:, outside] == 0.0)
    inside = (~outside) & (idx != src)
    assert np.all(np.abs(E[:, inside]).sum(0) > 0)


# ---------------------------------------------------------------- L6
def test_L6_value_error_is_second_order_with_the_textbook_constant():
    """One pair, rho(t) = sin(w t), J = 0.  Eq. (2.4) gives E_x = dV/(4 pi eps0) d_x [rho(t_r)/R^3 + rho_dot/(c R^2)], and
    the derivative both rules use is the hand-computable backward difference of the two samples, so the retarded VALUE
    the rule used can be solved for.  With tau = t_r - t^{n-m} = -phi dt, Taylor's theorem gives
        nearest rule:  rho^{n-m} - rho(t_r)                    = -tau rho'            + O(dt^2)      (first order)
        linear rule:   rho^{n-m} + tau (backward difference) - rho(t_r) = -(tau/2)(tau + dt) rho'' + O(dt^3)  (second order)
    """
    off = (2, 1, 1)
    dx = 1e-4
    R = dx * math.sqrt(6.0)
    w = 2 * math.pi * C / (80 * dx)  # period = 80 cells of light travel: w dt = 0.039 at kappa = 2
    T = 300 * dx / (2 * C)           # same physical time for every dt
    for kappa in (2.0, 4.0, 8.0):
        cfg = OracleConfig(4, 4, 4, dx, dx, dx, dx / (kappa * C))
        dt = cfg.dt
        n = int(round(T / dt))
        src, obs = 0, off[0] + 4 * (off[1] + 4 * off[2])

        def fn(t):
            S = np.zeros((4, cfg.N))
            S[0, src] = math.sin(w * t * dt)
            return S

        ring = ring_of(cfg, n, fn)
        s = R / (C * dt)
        m = math.floor(s + 0.5)
        tau = (m - s) * dt
        t_r = n * dt - R / C
        dot = (math.sin(w * (n - m) * dt) - math.sin(w * (n - m - 1) * dt)) / dt  # what both rules use
        exact = math.sin(w * t_r)
        pref = dx ** 3 / (4 * math.pi * EPS0) * off[0] * dx
        err = {}
        for rule in (RULE_NEAREST, RULE_LINEAR):
            E, _ = oracle.field(cfg, n, ring, np.array([obs]), rule=rule)
            err[rule] = (E[0, 0] / pref - dot / (C * R ** 2)) * R ** 3 - exact  # value the rule used - exact value
        lead_near = -tau * w * math.cos(w * t_r)
        lead_lin = -(tau / 2) * (tau + dt) * (-w * w * math.sin(w * t_r))
        assert abs(err[RULE_NEAREST] - lead_near) <= 0.15 * abs(lead_near), kappa
        assert abs(err[RULE_LINEAR] - lead_lin) <= 0.15 * abs(lead_lin), kappa
        assert abs(err[RULE_LINEAR]) < 0.1 * abs(err[RULE_NEAREST])
