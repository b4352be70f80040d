"""Pins for the oracle's kernel / direct sum O1 (no GPU).  SURVEY.md 8(c) pins P1-P4.

Each test checks oracle/ against something the paper or textbook physics fixes, written
independently here in numpy -- never against the oracle's own formula.
"""
import numpy as np
import pytest

import oracle

EPS0 = 8.8541878128e-12
C0 = 299792458.0
QE = -1.602176634e-19


def _golden_rows(name):
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", name)
    rows = []
    with open(path) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                rows.append([float(v) for v in line.split()])
    return np.array(rows)


def test_p1_uniformly_moving_charge_closed_form():
    """P1, eq. (3.1)-(3.2) PAPER.md:143-153 == textbook field of a uniformly moving charge:
    E = q/(4 pi eps0) * gamma R / (Rx^2 + Ry^2 + gamma^2 Rz^2)^(3/2) for motion along z."""
    for gamma, R in [(10.0, (1e-3, -2e-3, 3e-4)), (50.0, (2e-4, 1e-4, -1e-5)), (1.5, (0.3, 0.1, 0.2))]:
        pzv = np.sqrt(gamma * gamma - 1.0)
        R = np.array(R)
        x = np.array([R[0], 0.0]); y = np.array([R[1], 0.0]); z = np.array([R[2], 0.0])
        px = np.zeros(2); py = np.zeros(2); pz = np.full(2, pzv)
        E, B = oracle.direct(x, y, z, px, py, pz, q=QE)
        gb = np.sqrt(1.0 + pzv * pzv)
        den = (R[0] ** 2 + R[1] ** 2 + gb ** 2 * R[2] ** 2) ** 1.5
        E_exp = QE / (4 * np.pi * EPS0) * gb * R / den
        np.testing.assert_allclose(E[0], E_exp, rtol=2e-15)
        np.testing.assert_allclose(E[1], -E_exp, rtol=2e-15)
        # B = (1/c0) beta x E with beta = (0,0,pz/gamma)
        beta = np.array([0, 0, pzv / gb])
        np.testing.assert_allclose(B[0], np.cross(beta, E_exp) / C0, rtol=4e-15, atol=1e-40)


def test_p1_golden_values():
    """Hand-computed values (tests/golden/moving_charge.txt, derived there from eq. (3.1)-(3.2))."""
    rows = _golden_rows("moving_charge.txt")
    for gamma, rx, ry, rz, ex, ey, ez, bx, by, bz in rows:
        pzv = np.sqrt(gamma * gamma - 1.0)
        E, B = oracle.direct([rx, 0], [ry, 0], [rz, 0], [0, 0], [0, 0], [pzv, pzv], q=QE)
        np.testing.assert_allclose(E[0], [ex, ey, ez], rtol=1e-12)
        np.testing.assert_allclose(B[0], [bx, by, bz], rtol=1e-12, atol=1e-40)


def test_p2_coulomb_limit():
    """P2: p = 0 -> gamma = 1, g = R/|R|^3 (Coulomb), B = 0."""
    rng = np.random.default_rng(7)
    N = 50
    X = rng.normal(size=(N, 3))
    Z = np.zeros(N)
    q = rng.normal(size=N)
    E, B = oracle.direct(X[:, 0], X[:, 1], X[:, 2], Z, Z, Z, q=q)
    E_exp = np.zeros((N, 3))
    for i in range(N):
        for j in range(N):
            if i != j:
                R = X[i] - X[j]
                E_exp[i] += q[j] * R / np.linalg.norm(R) ** 3
    E_exp /= 4 * np.pi * EPS0
    np.testing.assert_allclose(E, E_exp, rtol=1e-12)
    assert np.all(B == 0.0)


def test_p3_b_equals_beta_cross_e():
    """P3: all sources share one p -> B = (p/gamma) x E / c0 for whole sums (eq. (3.1))."""
    rng = np.random.default_rng(11)
    N = 300
    X = rng.normal(size=(N, 3)) * [1e-3, 1e-3, 1e-4]
    p = np.array([0.3, -0.2, 25.0])
    P = np.tile(p, (N, 1))
    E, B = oracle.direct(X[:, 0], X[:, 1], X[:, 2], P[:, 0], P[:, 1], P[:, 2], q=QE)
    gam = np.sqrt(1 + p @ p)
    B_exp = np.cross(np.tile(p / gam, (N, 1)), E) / C0
    assert oracle.err2(B, B_exp) < 1e-13
    # sign of the cross product: p along +z, E along +x -> B along +y
    E1, B1 = oracle.direct([1e-3, 0], [0, 0], [0, 0], [0, 0], [0, 0], [5.0, 5.0], q=1.0)
    assert E1[0, 0] > 0 and B1[0, 1] > 0 and abs(B1[0, 0]) == 0 and abs(B1[0, 2]) == 0


def test_p3_per_source_momentum_enters_b_and_gamma():
    """Different momenta per source: E uses gamma_j, B uses p_j (eq. (3.1)), kernel uses gamma_bar."""
    x = np.array([0.0, 1e-3, -2e-3]); y = np.array([0.0, 2e-3, 1e-3]); z = np.array([0.0, 1e-4, 3e-4])
    P = np.array([[0.0, 0.0, 9.0], [0.1, 0.0, 10.0], [0.0, -0.2, 11.0]])
    E, B = oracle.direct(x, y, z, P[:, 0], P[:, 1], P[:, 2], q=2.0)
    pbar = P.mean(axis=0)
    g2 = 1 + pbar @ pbar
    assert oracle.gamma_bar(P[:, 0], P[:, 1], P[:, 2]) == pytest.approx(np.sqrt(g2), rel=1e-15)
    Ee = np.zeros(3); Be = np.zeros(3)
    for j in (1, 2):
        d = np.array([x[0] - x[j], y[0] - y[j], z[0] - z[j]])
        g = d / (d[0] ** 2 + d[1] ** 2 + g2 * d[2] ** 2) ** 1.5
        Ee += 2.0 * np.sqrt(1 + P[j] @ P[j]) * g
        Be += 2.0 * np.cross(P[j], g)
    np.testing.assert_allclose(E[0], Ee / (4 * np.pi * EPS0), rtol=1e-13)
    np.testing.assert_allclose(B[0], Be / (4 * np.pi * EPS0 * C0), rtol=1e-13)


def test_p4_symmetry():
    """P4: identical p and q -> sum_i E_i = 0 (g odd); mirrored bunch -> Ex(-x) = -Ex(x)."""
    rng = np.random.default_rng(3)
    N = 200
    X = rng.normal(size=(N, 3)) * [1e-3, 1e-3, 1e-4]
    X = np.concatenate([X, X * [-1, 1, 1]])  # mirror in x
    pz = np.full(2 * N, 20.0)
    Zp = np.zeros(2 * N)
    E, B = oracle.direct(X[:, 0], X[:, 1], X[:, 2], Zp, Zp, pz, q=QE)
    scale = np.abs(E).sum(axis=0)
    assert np.all(np.abs(E.sum(axis=0)) < 1e-12 * scale)
    np.testing.assert_allclose(E[N:, 0], -E[:N, 0], rtol=1e-10, atol=1e-12 * np.abs(E[:, 0]).max())
    np.testing.assert_allclose(E[N:, 1], E[:N, 1], rtol=1e-10, atol=1e-12 * np.abs(E[:, 1]).max())


def test_self_and_coincident_particles_contribute_zero():
    """G17: contribution is 0 iff D == 0 (covers i == j)."""
    x = [0.0, 0.0, 1e-3]; y = [0.0, 0.0, 0.0]; z = [0.0, 0.0, 0.0]
    E, B = oracle.direct(x, y, z, [0] * 3, [0] * 3, [3.0] * 3, q=1.0)
    assert np.all(np.isfinite(E)) and np.all(np.isfinite(B))
    np.testing.assert_array_equal(E[0], E[1])
    E1, _ = oracle.direct([7.0], [1.0], [2.0], [0.0], [0.0], [3.0], q=1.0)
    assert np.all(E1 == 0)


def test_raw_and_targets_subset():
    rng = np.random.default_rng(5)
    N = 64
    X = rng.normal(size=(N, 3)); P = rng.normal(size=(N, 3)) + [0, 0, 5]
    a = [X[:, 0], X[:, 1], X[:, 2], P[:, 0], P[:, 1], P[:, 2]]
    E, B = oracle.direct(*a, q=QE)
    Er, Br = oracle.direct(*a, q=QE, raw=True)
    np.testing.assert_allclose(E, Er / (4 * np.pi * EPS0), rtol=1e-15)
    np.testing.assert_allclose(B, Br / (4 * np.pi * EPS0 * C0), rtol=1e-15)
    t = np.array([5, 0, 63, 5])
    Et, Bt = oracle.direct(*a, q=QE, targets=t)
    np.testing.assert_array_equal(Et, E[t]); np.testing.assert_array_equal(Bt, B[t])


# ---------------------------------------------------------------------------------------------
# Source-momentum near field (alternative reading of Alg 5.10, G6)
# ---------------------------------------------------------------------------------------------
def _heaviside_field(q, R, p):
    """Textbook (Heaviside / Lienard-Wiechert, uniform motion) field at R from a charge with momentum p = gamma beta,
    in the cross-product form  E = q (1 - beta^2) R / (4 pi eps0 (R^2 - |R x beta|^2)^(3/2)),  B = beta x E / c0."""
    gam = np.sqrt(1.0 + p @ p)
    beta = p / gam
    den = (R @ R - np.sum(np.cross(R, beta) ** 2)) ** 1.5
    E = q / (4 * np.pi * EPS0) * (1.0 - beta @ beta) * R / den
    return E, np.cross(beta, E) / C0


def test_source_momentum_is_the_exact_field_of_each_moving_charge():
    """Each source's near field is stretched along ITS OWN momentum (any direction): for two particles with
    different momenta the field at one is the exact field of the other as a uniformly moving charge."""
    rng = np.random.default_rng(7)
    for _ in range(5):
        X = rng.normal(size=(2, 3)) * 1e-3
        Pm = np.stack([rng.normal(size=3) * [0.5, 0.5, 20.0], rng.normal(size=3) * [2.0, 1.0, 5.0]])
        E, B = oracle.direct(X[:, 0].copy(), X[:, 1].copy(), X[:, 2].copy(), Pm[:, 0].copy(), Pm[:, 1].copy(),
                             Pm[:, 2].copy(), q=QE, source_momentum=True)
        for i, j in ((0, 1), (1, 0)):
            E_exp, B_exp = _heaviside_field(QE, X[i] - X[j], Pm[j])
            # (1 - beta^2) and R^2 - |R x beta|^2 cancel to ~1/gamma^2: allow gamma^2 ulps in the textbook form
            tol = 1e-13 * (1.0 + Pm[j] @ Pm[j])
            np.testing.assert_allclose(E[i], E_exp, rtol=tol)
            np.testing.assert_allclose(B[i], B_exp, rtol=tol, atol=1e-30)


def test_source_momentum_reduces_to_mean_gamma_for_identical_momenta():
    """All p_j = (0, 0, p): D = dx^2 + dy^2 + (1 + p^2) dz^2 = eq. (3.2) with gamma_bar: both readings coincide
    ('they coincide when all momenta are identical', the only case the paper measures)."""
    rng = np.random.default_rng(8)
    N = 300
    x, y, z = rng.random(N), rng.random(N), rng.random(N)
    pz = np.full(N, np.sqrt(50.0 ** 2 - 1.0))
    zero = np.zeros(N)
    Ea, Ba = oracle.direct(x, y, z, zero, zero, pz, q=QE)
    Eb, Bb = oracle.direct(x, y, z, zero, zero, pz, q=QE, source_momentum=True)
    assert oracle.err2(Eb, Ea) < 1e-13 and oracle.err2(Bb, Ba) < 1e-13


def test_source_momentum_differs_for_an_energy_spread_and_fmm_near_field_uses_it():
    """With an energy spread the two readings differ at the 1e-3 level; the serial FMM in this mode
    equals the source-momentum direct sum when the far list is empty (pin P9 for the new near field)."""
    from paper_2302_07567_b200 import workloads
    w = workloads.config(1, N=1500)
    Ea, _ = oracle.direct(*w.arrays(), w.q)
    Eb, Bb = oracle.direct(*w.arrays(), w.q, source_momentum=True)
    d = oracle.err2(Eb, Ea)
    assert 1e-4 < d < 5e-2, d
    op = oracle.Plan(*w.arrays(), w.q, order_n=3, leaf_size=64, theta=0.05, source_momentum=True)
    assert op.n_m2l == 0
    E, B = op.eval()
    assert oracle.err2(E, Eb) < 1e-13 and oracle.err2(B, Bb) < 1e-13
    # with a far field: near part in the new mode, far part unchanged (mean gamma)
    op2 = oracle.Plan(*w.arrays(), w.q, order_n=4, leaf_size=64, theta=0.5, source_momentum=True)
    op3 = oracle.Plan(*w.arrays(), w.q, order_n=4, leaf_size=64, theta=0.5)
    assert op2.n_m2l > 0
    Ef2, _ = op2.eval(part="far")
    Ef3, _ = op3.eval(part="far")
    assert np.array_equal(Ef2, Ef3)
    En2, _ = op2.eval(part="near")
    En3, _ = op3.eval(part="near")
    assert oracle.err2(En2, En3) > 1e-5
