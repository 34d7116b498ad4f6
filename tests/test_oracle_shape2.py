"""Pins of the oracle's second-order shape function S^(2) (Eq. 2.14, reading A11).

None of these re-types the oracle's piecewise formula: they use the closed-form three weights of the quadratic B-spline
written out by hand, its moments, conservation, adjointness of deposit and interpolation, and a separately written dense
numpy enumeration.
"""
import math

import numpy as np
import pytest

import oracle
from oracle import OracleConfig

C = 299792458.0
N8 = 8


def cfg2(n=N8, dx=1e-4, **kw):
    return OracleConfig(n, n, n, dx, dx, dx, dx / (2 * C), shape_order=2, **kw)


def dep1(cfg, pos, u=(0.0, 0.0, 0.0), q=1.0):
    f = lambda v: np.array([v], dtype=np.float64)
    return oracle.deposit(cfg, f(pos[0]), f(pos[1]), f(pos[2]), f(u[0]), f(u[1]), f(u[2]), f(q))


def hand_w(delta):
    """Quadratic B-spline weights of the nodes at -1, 0, +1 for a particle at offset delta in [-1/2, 1/2] from the
    centre node (hand algebra from Eq. 2.14 with |x| = 1 + delta, |delta|, 1 - delta)."""
    return np.array([0.5 * (0.5 - delta) ** 2, 0.75 - delta * delta, 0.5 * (0.5 + delta) ** 2])


# Q1 ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("delta,wx", [(0.0, (1 / 8, 3 / 4, 1 / 8)), (0.25, (1 / 32, 11 / 16, 9 / 32)), (-0.25, (9 / 32, 11 / 16, 1 / 32)),
                                      (0.5 - 1e-13, (0.0, 0.5, 0.5))])
def test_q1_hand_weights(delta, wx):
    """A particle at the centre of cell (4,3,2) in y and z and at offset delta in x: node (4+a, 3+b, 2+c) gets
    wx[a] * wc[b] * wc[c] with wc = (1/8, 3/4, 1/8), the printed numbers of the three S^(2) weights."""
    cfg = cfg2()
    q = 3.0e-13
    S = dep1(cfg, (4.5 + delta, 3.5, 2.5), q=q)
    rho = S[0].reshape(N8, N8, N8)  # [k][j][i]
    dV = cfg.dx ** 3
    wc = (1 / 8, 3 / 4, 1 / 8)
    want = np.zeros_like(rho)
    for c in range(3):
        for b in range(3):
            for a in range(3):
                want[2 + c - 1, 3 + b - 1, 4 + a - 1] = q * wx[a] * wc[b] * wc[c] / dV
    assert np.allclose(rho, want, rtol=1e-11, atol=1e-12 * q / dV)
    assert np.count_nonzero(rho) <= 27


# Q2 ------------------------------------------------------------------------------------------------------------
def test_q2_interior_particles_conserve_charge_and_current():
    cfg = cfg2()
    rng = np.random.default_rng(2)
    P = 500
    pos = rng.uniform(1.0, N8 - 1.0, (3, P))  # all 27 nodes inside
    u = rng.normal(0, 0.4, (3, P))
    qw = rng.uniform(-2, 2, P) * 1e-13
    S = oracle.deposit(cfg, *pos, *u, qw)
    dV = cfg.dx ** 3
    assert np.isclose(S[0].sum() * dV, qw.sum(), rtol=1e-12)
    v = C * u / np.sqrt(1 + (u * u).sum(0))
    for a in range(3):
        assert np.isclose(S[1 + a].sum() * dV, (qw * v[a]).sum(), rtol=1e-11)
    # first moment: the deposited charge has its centroid at the particle (the spline reproduces linear functions)
    S1 = dep1(cfg, (3.3, 4.8, 2.1), q=1.0)[0].reshape(N8, N8, N8) * dV
    k, j, i = np.meshgrid(np.arange(N8), np.arange(N8), np.arange(N8), indexing="ij")
    assert np.isclose((S1 * (i + 0.5)).sum(), 3.3, rtol=1e-13) and np.isclose((S1 * (j + 0.5)).sum(), 4.8, rtol=1e-13)
    # second moment: variance 1/4 cell^2 per axis, whatever the offset (first order: alpha (1 - alpha))
    assert np.isclose((S1 * (i + 0.5 - 3.3) ** 2).sum(), 0.25, rtol=1e-12)
    assert np.isclose((S1 * (k + 0.5 - 2.1) ** 2).sum(), 0.25, rtol=1e-12)


# Q3 ------------------------------------------------------------------------------------------------------------
def test_q3_virtual_node_loss():
    """A particle in the first cell of x at offset delta loses exactly the share 1/2 (1/2 - delta)^2 of the virtual node
    i = -1; in the corner cell the three losses multiply."""
    cfg = cfg2()
    dV = cfg.dx ** 3
    for delta in (-0.5, -0.2, 0.0, 0.3):
        lost = 0.5 * (0.5 - delta) ** 2
        S = dep1(cfg, (0.5 + delta, 4.5, 4.5))
        assert np.isclose(S[0].sum() * dV, 1.0 - lost, rtol=1e-12)
        S = dep1(cfg, (N8 - 0.5 - delta, 4.5, 4.5))  # mirror: the node i = n is virtual
        assert np.isclose(S[0].sum() * dV, 1.0 - lost, rtol=1e-12)
    S = dep1(cfg, (0.5, 0.5, N8 - 0.5))
    assert np.isclose(S[0].sum() * dV, (1 - 1 / 8) ** 3, rtol=1e-12)
    # dead particles are not sources
    f = lambda v: np.array([v], dtype=np.float64)
    Sd = oracle.deposit(cfg, f(4.2), f(4.2), f(4.2), f(0), f(0), f(0), f(1.0), np.zeros(1, dtype=np.uint8))
    assert np.all(Sd == 0)


# Q4 ------------------------------------------------------------------------------------------------------------
def test_q4_interpolation_moments():
    cfg = cfg2()
    k, j, i = np.meshgrid(np.arange(N8), np.arange(N8), np.arange(N8), indexing="ij")
    xc, yc, zc = (i + 0.5).ravel(), (j + 0.5).ravel(), (k + 0.5).ravel()  # cell centres, grid units
    rng = np.random.default_rng(4)
    pos = rng.uniform(1.0, N8 - 1.0, (3, 300))
    lin = np.stack([2.0 + 0.0 * xc, 1.0 - 3.0 * xc + 0.5 * yc + 2.0 * zc, xc * 0 + yc])
    got = oracle.interp(cfg, *pos, lin)
    assert np.allclose(got[:, 0], 2.0, rtol=1e-14)
    assert np.allclose(got[:, 1], 1.0 - 3.0 * pos[0] + 0.5 * pos[1] + 2.0 * pos[2], rtol=1e-13, atol=1e-13)
    assert np.allclose(got[:, 2], pos[1], rtol=1e-13)
    # a quadratic field comes back shifted by the spline's variance 1/4: x^2 -> x^2 + 1/4 (first order: + alpha(1-alpha))
    quad = np.stack([xc ** 2, yc * zc, zc ** 2])
    got = oracle.interp(cfg, *pos, quad)
    assert np.allclose(got[:, 0], pos[0] ** 2 + 0.25, rtol=1e-13)
    assert np.allclose(got[:, 1], pos[1] * pos[2], rtol=1e-13)  # mixed term: product of two exact first moments
    assert np.allclose(got[:, 2], pos[2] ** 2 + 0.25, rtol=1e-13)
    c1 = OracleConfig(N8, N8, N8, 1e-4, 1e-4, 1e-4, 1e-4 / (2 * C))
    got1 = oracle.interp(c1, *pos, quad)
    al = (pos[0] - 0.5) - np.floor(pos[0] - 0.5)
    assert np.allclose(got1[:, 0], pos[0] ** 2 + al * (1 - al), rtol=1e-13)  # and the two orders are told apart
    # virtual nodes count as zero, weights not renormalised (reading A12): uniform field 1 near a face
    one = np.ones((3, cfg.N))
    g = oracle.interp(cfg, np.array([0.5 + 0.3]), np.array([4.5]), np.array([4.5]), one)
    assert np.allclose(g, 1.0 - 0.5 * (0.5 - 0.3) ** 2, rtol=1e-13)


# Q5 ------------------------------------------------------------------------------------------------------------
def dense_s2(shape, dx, pos, u, qw, alive):
    """Separately written 27-node enumeration with the closed-form weights (numpy, fp64)."""
    nx, ny, nz = shape
    out = np.zeros((4, nz, ny, nx))
    dV = dx[0] * dx[1] * dx[2]
    for p in range(pos.shape[1]):
        if not alive[p]:
            continue
        ic = np.floor(pos[:, p]).astype(int)
        d = pos[:, p] - ic - 0.5
        W = [hand_w(d[a]) for a in range(3)]
        g = math.sqrt(1 + u[:, p] @ u[:, p])
        v = C * u[:, p] / g
        for c in (-1, 0, 1):
            for b in (-1, 0, 1):
                for a in (-1, 0, 1):
                    ii, jj, kk = ic[0] + a, ic[1] + b, ic[2] + c
                    if 0 <= ii < nx and 0 <= jj < ny and 0 <= kk < nz:
                        r = qw[p] * W[0][a + 1] * W[1][b + 1] * W[2][c + 1] / dV
                        out[0, kk, jj, ii] += r
                        out[1:, kk, jj, ii] += r * v
    return out.reshape(4, -1)


@pytest.mark.parametrize("shape,h", [((5, 4, 3), (1e-4, 1e-4, 1e-4)), ((7, 2, 9), (1e-4, 2e-4, 0.5e-4)), ((1, 6, 5), (1e-5, 1e-5, 1e-5))])
def test_q5_dense_enumeration(shape, h):
    cfg = OracleConfig(*shape, *h, h[0] / (2 * C), shape_order=2)
    rng = np.random.default_rng(55)
    P = 400
    pos = np.stack([rng.uniform(0, n, P) for n in shape])
    pos[:, 0] = (0.0, 0.0, 0.0)
    pos[:, 1] = [n - 1e-9 for n in shape]
    pos[:, 2] = (0.5, 0.5, 0.5)
    u = rng.normal(0, 0.5, (3, P))
    qw = rng.uniform(-1, 1, P) * 1e-13
    alive = (rng.uniform(size=P) < 0.9).astype(np.uint8)
    S = oracle.deposit(cfg, *pos, *u, qw, alive)
    want = dense_s2(shape, h, pos, u, qw, alive)
    for a in range(4):
        assert np.allclose(S[a], want[a], rtol=1e-11, atol=1e-13 * np.abs(want[a]).max())
    idx = oracle.cell_index(*pos, shape_order=2)
    assert np.array_equal(idx, np.floor(pos).T.astype(np.int32))


# Q6 ------------------------------------------------------------------------------------------------------------
def test_q6_continuous_across_cell_faces():
    """Crossing xi = 3 swaps the centre node from 2 to 3: weights (0, 1/2, 1/2) on nodes 1..3 become (1/2, 1/2, 0) on 2..4.
    The deposit must not jump (the first-order weights are continuous too, but change node at xi = k + 1/2)."""
    cfg = cfg2()
    a = dep1(cfg, (3.0 - 1e-12, 4.3, 4.7))
    b = dep1(cfg, (3.0 + 1e-12, 4.3, 4.7))
    assert np.allclose(a, b, rtol=0, atol=1e-10 * np.abs(a).max())
    rho = a[0].reshape(N8, N8, N8)
    assert rho[:, :, 1].sum() < 1e-10 * rho.sum() and rho[:, :, 4].sum() < 1e-10 * rho.sum()
    assert np.isclose(rho[:, :, 2].sum(), rho[:, :, 3].sum(), rtol=1e-9)


# Q7 ------------------------------------------------------------------------------------------------------------
def test_q7_deposit_and_interpolation_are_adjoint_and_the_push_uses_s2():
    """Same weights in both directions: sum_nodes rho[node] F[node] dV = q * interp(F)(particle), also next to faces."""
    cfg = cfg2()
    rng = np.random.default_rng(7)
    F = rng.normal(0, 1, (3, cfg.N))
    dV = cfg.dx ** 3
    for pos in [(3.3, 4.8, 2.1), (0.1, 7.9, 4.0), (0.6, 0.4, 7.5)]:
        rho = dep1(cfg, pos, q=2.5)[0]
        g = oracle.interp(cfg, np.array([pos[0]]), np.array([pos[1]]), np.array([pos[2]]), F)[0]
        for a in range(3):
            assert np.isclose((rho * F[a]).sum() * dV, 2.5 * g[a], rtol=1e-12)
    # push with shape_order 2: pure E kick with the S^(2)-interpolated field, u_new = u + (q/m) dt E_p / c (P12)
    pos = (3.3, 4.8, 2.1)
    Ep = oracle.interp(cfg, np.array([pos[0]]), np.array([pos[1]]), np.array([pos[2]]), F)[0]
    c1 = OracleConfig(N8, N8, N8, 1e-4, 1e-4, 1e-4, 1e-4 / (2 * C))
    E1 = oracle.interp(c1, np.array([pos[0]]), np.array([pos[1]]), np.array([pos[2]]), F)[0]
    assert np.abs(Ep - E1).max() > 1e-2  # the two orders differ on a rough field
    f = lambda v: np.array([v], dtype=np.float64)
    qm = -1.75882001076e11
    st = [f(pos[0]), f(pos[1]), f(pos[2]), f(0.0), f(0.0), f(0.0), f(qm), np.ones(1, dtype=np.uint8)]
    oracle.push(cfg, *st, F, np.zeros((3, cfg.N)))
    for a in range(3):
        assert np.isclose(st[3 + a][0], qm * cfg.dt * Ep[a] / C, rtol=1e-12)
