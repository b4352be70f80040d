"""Pins for the oracle's serial FMM O2 (no GPU).  SURVEY.md 8(c) pins P5-P12.

Everything here is checked against mathematics the paper states (Theorem 1, eq. (2.9),
Lemma 1, Alg 5.1/5.2/9.1 invariants) re-derived in numpy, or against the oracle's own O1
(already pinned by test_oracle_kernel_pins.py) where the paper says the two must agree.
"""
import numpy as np
import pytest

import oracle
from paper_2302_07567_b200 import workloads


def small(N=4096, seed=1001, **kw):
    w = workloads.config(1, N=N)
    for k, v in kw.items():
        setattr(w, k, v)
    return w


def plan_of(w, **kw):
    args = dict(order_n=w.order_n, leaf_size=w.leaf_size, theta=w.theta)
    args.update(kw)
    return oracle.Plan(*w.arrays(), q=w.q, **args)


# ---------------------------------------------------------------- interpolation (P5)
def test_cheb_nodes_are_second_kind_and_antisymmetric():
    for n in (1, 2, 3, 4, 6, 7, 10):
        c = oracle.cheb_nodes(n)
        np.testing.assert_allclose(c, np.cos(np.arange(n + 1) * np.pi / n), atol=2e-16)
        assert c[0] == 1.0 and c[n] == -1.0
        np.testing.assert_array_equal(c, -c[::-1])


@pytest.mark.parametrize("n", [1, 2, 4, 6, 8, 10])
def test_p5_theorem1_polynomial_reproduction(n):
    """Theorem 1: sum_k P(xi_k) l_k(x) = P(x) for deg P <= n."""
    rng = np.random.default_rng(n)
    a, b = -0.3, 1.7
    xi = (a + b) * 0.5 + (b - a) * 0.5 * np.cos(np.arange(n + 1) * np.pi / n)
    coef = rng.normal(size=n + 1)
    for x in np.concatenate([rng.uniform(a, b, 20), [a, b, 0.5 * (a + b)]]):
        ell = oracle.basis_1d(n, a, b, x)
        assert abs(ell.sum() - 1.0) < 1e-13
        assert abs(ell @ np.polyval(coef, xi) - np.polyval(coef, x)) < 1e-12 * (1 + abs(np.polyval(coef, x)))
    # a degree n+1 polynomial is NOT reproduced (the pin can fail)
    x = 0.4321
    ell = oracle.basis_1d(n, a, b, x)
    assert abs(ell @ xi ** (n + 1) - x ** (n + 1)) > 1e-8


def test_p5_lagrange_basis_matches_product_formula():
    """l_k(x) = prod_{m != k} (x - xi_m)/(xi_k - xi_m) (PAPER.md:51-53 definition)."""
    n, a, b = 5, 2.0, 3.0
    xi = (a + b) * 0.5 + (b - a) * 0.5 * np.cos(np.arange(n + 1) * np.pi / n)
    for x in (2.1, 2.5, 2.99):
        ell = oracle.basis_1d(n, a, b, x)
        for k in range(n + 1):
            ref = np.prod([(x - xi[m]) / (xi[k] - xi[m]) for m in range(n + 1) if m != k])
            assert ell[k] == pytest.approx(ref, rel=1e-12, abs=1e-15)


def test_exact_hit_and_degenerate_box():
    """I-4: x == xi_k -> l_k = 1, others 0; degenerate box b == a -> l_0 = 1."""
    n, a, b = 4, -1.0, 1.0
    c = oracle.cheb_nodes(n)
    for k in range(n + 1):
        ell = oracle.basis_1d(n, a, b, c[k])
        e = np.zeros(n + 1); e[k] = 1.0
        np.testing.assert_array_equal(ell, e)
    ell = oracle.basis_1d(n, 0.7, 0.7, 0.7)
    e = np.zeros(n + 1); e[0] = 1.0
    np.testing.assert_array_equal(ell, e)


# ---------------------------------------------------------------- tree (P11)
@pytest.mark.parametrize("N,N0", [(4096, 64), (1000, 37), (5, 64), (129, 1), (2048, 2048)])
@pytest.mark.parametrize("mode", [oracle.TREE_KD, oracle.TREE_MORTON_MEDIAN])
def test_p11_tree_invariants(N, N0, mode):
    w = small(N=N)
    p = plan_of(w, leaf_size=N0, tree_mode=mode)
    kappa = 0
    while N0 * 2 ** kappa < N:
        kappa += 1
    assert p.kappa == kappa and p.nodes == 2 ** (kappa + 1) - 1 and p.leaves == 2 ** kappa
    perm = p.perm()
    assert sorted(perm.tolist()) == list(range(N))
    lo, hi, bb = p.node_arrays()
    X = np.stack([w.x, w.y, w.z], axis=1)
    s = np.array([1.0, 1.0, p.gamma_bar])
    assert lo[0] == 0 and hi[0] == N
    for i in range(1, p.nodes + 1):
        l, h = lo[i - 1], hi[i - 1]
        if h > l:
            mem = X[perm[l:h]]
            np.testing.assert_array_equal(bb[i - 1, :3], mem.min(axis=0))  # tight bbox PAPER.md:45-49
            np.testing.assert_array_equal(bb[i - 1, 3:], mem.max(axis=0))
        if i < p.leaves:  # internal
            mid = l + (h - l + 1) // 2
            assert (lo[2 * i - 1], hi[2 * i - 1]) == (l, mid) and (lo[2 * i], hi[2 * i]) == (mid, h)
            if mode == oracle.TREE_KD and h - l >= 2:
                ext = s * (bb[i - 1, 3:] - bb[i - 1, :3])
                k = int(np.argmax(ext))  # first maximiser (G9)
                left, right = X[perm[l:mid], k], X[perm[mid:h], k]
                assert left.max() <= right.min()  # Alg 5.2: S1 = {k_i <= k_split}
        else:
            assert h - l <= N0
            assert h - l in (N // p.leaves, N // p.leaves + 1)
            if mode == oracle.TREE_KD:
                assert np.all(np.diff(perm[l:h]) > 0)  # canonical order in a leaf (T-3)


def test_kd_tie_break_by_index():
    """G8: equal coordinates -> membership decided by original index."""
    N = 16
    x = np.zeros(N); y = np.zeros(N); z = np.zeros(N)
    x[:] = np.repeat([0.0, 1.0], 8)[np.random.default_rng(0).permutation(N)]
    pz = np.full(N, 5.0)
    p = oracle.Plan(x, y, z, np.zeros(N), np.zeros(N), pz, order_n=2, leaf_size=2, theta=0.5)
    perm = p.perm(); lo, hi, _ = p.node_arrays()
    zeros = np.flatnonzero(x == 0.0); ones = np.flatnonzero(x == 1.0)
    np.testing.assert_array_equal(np.sort(perm[:8]), zeros)
    # level 2: all x equal inside -> extent 0 on every axis -> axis x, rank by index
    np.testing.assert_array_equal(perm[:8], zeros)
    np.testing.assert_array_equal(perm[8:], ones)


def test_morton_order_matches_numpy_restatement():
    """T-3': key = interleave(floor((s o x - lo)/L * 2^21)), z most significant."""
    w = small(N=777)
    p = plan_of(w, tree_mode=oracle.TREE_MORTON_MEDIAN)
    s = np.array([1.0, 1.0, p.gamma_bar])
    U = np.stack([w.x, w.y, w.z], axis=1) * s
    lo = U.min(axis=0); L = (U.max(axis=0) - lo).max()
    q = np.minimum(np.floor((U - lo) / L * 2097152.0), 2097151).astype(np.uint64)
    key = np.zeros(len(U), dtype=np.uint64)
    for b in range(21):
        for k in range(3):
            key |= ((q[:, k] >> np.uint64(b)) & np.uint64(1)) << np.uint64(3 * b + k)
    order = np.lexsort((np.arange(len(U)), key))
    np.testing.assert_array_equal(p.perm(), order)


# ---------------------------------------------------------------- traversal (P10)
@pytest.mark.parametrize("mode", [oracle.TREE_KD, oracle.TREE_MORTON_MEDIAN])
@pytest.mark.parametrize("theta", [0.3, 0.5])
def test_p10_coverage_exactly_once(mode, theta):
    """Alg 9.1: every ordered leaf pair is covered by exactly one (ancestor, ancestor) pair."""
    w = small(N=4096)
    p = plan_of(w, theta=theta, tree_mode=mode)
    p2p, m2l = p.lists()
    Lf = p.leaves
    cover = np.zeros((Lf, Lf), dtype=np.int32)

    def span(i):  # leaf range below heap node i
        lvl = int(np.log2(i)); width = Lf >> lvl
        first = (i - (1 << lvl)) * width
        return first, first + width
    for t, s in np.concatenate([p2p, m2l]):
        t0, t1 = span(t); s0, s1 = span(s)
        cover[t0:t1, s0:s1] += 1
    assert np.all(cover == 1)
    assert np.all(p2p >= Lf)  # P2P only between leaves (D-1)
    for arr in (p2p, m2l):  # sorted by (target, source), no duplicates (D-4)
        k = arr[:, 0].astype(np.int64) * (1 << 32) + arr[:, 1]
        assert np.all(np.diff(k) > 0)


def test_admissibility_rule_on_lists():
    """Alg 5.6-5.8 restated in numpy: every M2L pair is admissible, its parent pair was not."""
    w = small(N=4096)
    p = plan_of(w)
    _, _, bb = p.node_arrays()
    s = np.array([1.0, 1.0, p.gamma_bar])

    def r(i): return np.linalg.norm(s * (bb[i - 1, 3:] - bb[i - 1, :3]) / 2)   # Alg 5.6
    def d(i, j): return np.linalg.norm(s * ((bb[i - 1, :3] + bb[i - 1, 3:]) / 2 - (bb[j - 1, :3] + bb[j - 1, 3:]) / 2))  # Alg 5.7
    p2p, m2l = p.lists()
    assert len(m2l) > 0
    for t, sidx in m2l:
        assert max(r(t), r(sidx)) / d(t, sidx) < w.theta * (1 + 1e-12)   # Alg 5.8
    n_near_inadmissible = sum(1 for t, sidx in p2p if t == sidx or max(r(t), r(sidx)) >= w.theta * d(t, sidx))
    assert n_near_inadmissible > 0
    # the stretch matters: with gamma_bar forced to 1 the lists differ
    p1 = plan_of(w, gamma_bar_value=1.0)
    assert (p1.n_p2p, p1.n_m2l) != (p.n_p2p, p.n_m2l)


# ---------------------------------------------------------------- upward (P6, P7)
@pytest.mark.parametrize("mode", [oracle.TREE_KD, oracle.TREE_MORTON_MEDIAN])
def test_p6_moment_conservation_and_p7_m2m_equals_p2m(mode):
    w = small(N=2048, order_n=3)
    p = plan_of(w, leaf_size=32, tree_mode=mode)
    M = p.upward()
    perm = p.perm(); lo, hi, bb = p.node_arrays()
    gam = np.sqrt(1 + w.px ** 2 + w.py ** 2 + w.pz ** 2)
    m = w.q * np.stack([gam, w.px, w.py, w.pz], axis=1)
    X = np.stack([w.x, w.y, w.z], axis=1)
    n1 = p.n + 1
    c = np.cos(np.arange(n1) * np.pi / p.n)
    worst = 0.0
    for i in range(1, p.nodes + 1):
        mem = perm[lo[i - 1]:hi[i - 1]]
        tot = m[mem].sum(axis=0)
        np.testing.assert_allclose(M[i - 1].sum(axis=0), tot, rtol=1e-11, atol=1e-13 * np.abs(tot).max())  # P6 (2.4)
        # first moments (n >= 1): sum_nu xi_nu M_nu = sum_j x_j m_j
        a, b = bb[i - 1, :3], bb[i - 1, 3:]
        xi = [(a[g] + b[g]) / 2 + (b[g] - a[g]) / 2 * c for g in range(3)]
        G = np.stack(np.meshgrid(xi[0], xi[1], xi[2], indexing="ij"), axis=-1).reshape(-1, 3)
        first = G.T @ M[i - 1][:, 0]
        ref = X[mem].T @ m[mem, 0]
        np.testing.assert_allclose(first, ref, rtol=1e-9, atol=1e-12 * np.abs(X[mem]).max() * abs(tot[0]))
        direct_M = p.p2m_node(i)   # eq. (2.4) at this node from its particles
        scale = np.abs(direct_M).max()
        worst = max(worst, np.abs(M[i - 1] - direct_M).max() / scale)
    assert worst < 1e-12  # P7, eq. (2.9)


def test_p2m_against_numpy_restatement():
    """eq. (2.4) PAPER.md:74-76 for one leaf, with the product-form Lagrange basis."""
    w = small(N=512, order_n=2)
    p = plan_of(w, leaf_size=64)
    perm = p.perm(); lo, hi, bb = p.node_arrays()
    i = p.leaves + 3
    mem = perm[lo[i - 1]:hi[i - 1]]
    n = p.n
    c = np.cos(np.arange(n + 1) * np.pi / n)
    gam = np.sqrt(1 + w.px ** 2 + w.py ** 2 + w.pz ** 2)
    m = w.q * np.stack([gam, w.px, w.py, w.pz], axis=1)
    X = np.stack([w.x, w.y, w.z], axis=1)

    def basis(g, x):
        a, b = bb[i - 1, g], bb[i - 1, 3 + g]
        xi = (a + b) / 2 + (b - a) / 2 * c
        return np.array([np.prod([(x - xi[q]) / (xi[k] - xi[q]) for q in range(n + 1) if q != k]) for k in range(n + 1)])
    Mref = np.zeros(((n + 1) ** 3, 4))
    for j in mem:
        l = np.einsum("a,b,c->abc", basis(0, X[j, 0]), basis(1, X[j, 1]), basis(2, X[j, 2])).reshape(-1)
        Mref += np.outer(l, m[j])
    np.testing.assert_allclose(p.p2m_node(i), Mref, rtol=1e-9, atol=1e-12 * np.abs(Mref).max())


# ---------------------------------------------------------------- downward (P8) and whole (P9, P12)
def test_p8_lemma1_cumulative_local_field():
    """Lemma 1: L2L + L2P == sum over levels of sum_mu l_{S^l,mu}(x_i) L^raw_{S^l,mu}."""
    w = small(N=1024, order_n=3)
    p = plan_of(w, leaf_size=32)
    Lraw = p.m2l_raw()
    Efar, Bfar = p.eval(part="far")
    Efar_raw, Bfar_raw = _strip_prefactors(Efar, Bfar)
    perm = p.perm(); lo, hi, bb = p.node_arrays()
    n1 = p.n + 1
    X = np.stack([w.x, w.y, w.z], axis=1)
    rng = np.random.default_rng(0)
    for leaf in rng.choice(np.arange(p.leaves, p.nodes + 1), 6, replace=False):
        for k in range(lo[leaf - 1], min(hi[leaf - 1], lo[leaf - 1] + 4)):
            j = perm[k]
            acc = np.zeros(6)
            i = leaf
            while i >= 1:
                a, b = bb[i - 1, :3], bb[i - 1, 3:]
                l = [oracle.basis_1d(p.n, a[g], b[g], X[j, g]) for g in range(3)]
                l3 = np.einsum("a,b,c->abc", *l).reshape(-1)
                acc += l3 @ Lraw[i - 1]
                i //= 2
            got = np.concatenate([Efar_raw[j], Bfar_raw[j]])
            np.testing.assert_allclose(got, acc, rtol=1e-10, atol=1e-12 * np.abs(acc).max())


def _strip_prefactors(E, B):
    cE = 1.0 / (4 * np.pi * 8.8541878128e-12)
    return E / cE, B / (cE / 299792458.0)


def test_p9_empty_far_list_equals_direct():
    """P9: eta so small that nothing is admissible -> FMM == direct to rounding."""
    w = small(N=2048)
    p = plan_of(w, theta=1e-3)
    assert p.n_m2l == 0 and p.n_p2p == p.leaves ** 2
    E, B = p.eval()
    Ed, Bd = oracle.direct(*w.arrays(), q=w.q, gamma_bar_value=p.gamma_bar)
    assert oracle.err2(E, Ed) < 1e-13 and oracle.err2(B, Bd) < 1e-13


def test_single_leaf_is_direct():
    """G23: N <= N0 -> root is a leaf, FMM == direct."""
    w = small(N=50)
    p = plan_of(w, leaf_size=64)
    assert p.kappa == 0 and p.n_p2p == 1 and p.n_m2l == 0
    E, B = p.eval()
    Ed, Bd = oracle.direct(*w.arrays(), q=w.q)
    assert oracle.err2(E, Ed) < 1e-14 and oracle.err2(B, Bd) < 1e-14


def test_near_plus_far_is_all_and_leaf_selection():
    w = small(N=1024, order_n=2)
    p = plan_of(w, leaf_size=32)
    E, B = p.eval()
    En, Bn = p.eval(part="near"); Ef, Bf = p.eval(part="far")
    np.testing.assert_allclose(En + Ef, E, rtol=1e-12, atol=1e-14 * np.abs(E).max())
    sel = [p.leaves + 1, p.nodes]
    Es, Bs = p.eval(leaves=sel)
    perm = p.perm(); lo, hi, _ = p.node_arrays()
    for leaf in sel:
        mem = perm[lo[leaf - 1]:hi[leaf - 1]]
        np.testing.assert_array_equal(Es[mem], E[mem]); np.testing.assert_array_equal(Bs[mem], B[mem])
    assert np.isnan(Es).sum() == 3 * (w.N - sum(hi[l - 1] - lo[l - 1] for l in sel))


@pytest.mark.parametrize("mode", [oracle.TREE_KD])
def test_p12_convergence_in_n_and_eta(mode):
    """PAPER.md:504-506 (trend only; absolute values are 'parity unpinned')."""
    w = small(N=4096)
    Ed, Bd = oracle.direct(*w.arrays(), q=w.q)
    errs = {}
    for theta in (0.5, 0.4):
        for n in (2, 4, 6, 8):
            p = plan_of(w, order_n=n, theta=theta, tree_mode=mode)
            E, B = p.eval()
            errs[(theta, n)] = max(oracle.err2(E, Ed), oracle.err2(B, Bd))
    for theta in (0.5, 0.4):
        e = [errs[(theta, n)] for n in (2, 4, 6, 8)]
        assert all(e[k + 1] < 0.5 * e[k] for k in range(3)), e
    for n in (2, 4, 6, 8):
        assert errs[(0.4, n)] < errs[(0.5, n)]
    assert errs[(0.5, 2)] < 0.1 and errs[(0.5, 8)] < 1e-3 and errs[(0.5, 8)] > 1e-9


def test_paper_shaped_input_identical_momenta():
    """PAPER.md:380 workload shape (uniform cube, identical p): B == beta x E / c0 survives the FMM."""
    w = workloads.paper_cube(N=4000, gamma0=50.0, order_n=4)
    p = plan_of(w)
    E, B = p.eval()
    beta = np.array([0, 0, np.sqrt(1 - 1 / 50.0 ** 2)])
    Bexp = np.cross(np.tile(beta, (w.N, 1)), E) / 299792458.0
    assert oracle.err2(B, Bexp) < 1e-12
    Ed, Bd = oracle.direct(*w.arrays(), q=w.q)
    assert oracle.err2(E, Ed) < 5e-3


# ---------------------------------------------------------------------------------------------
# Tree over a given particle order (refit of an existing partition)
# ---------------------------------------------------------------------------------------------
def test_given_order_equal_to_kd_order_reproduces_the_kd_plan():
    """Fed the KD plan's own permutation, the given-order plan is the KD plan: same ranges, boxes, lists, fields."""
    w = small(N=3000)
    a = plan_of(w, theta=0.5)
    b = oracle.Plan(*w.arrays(), w.q, order_n=4, leaf_size=64, theta=0.5, gamma_bar_value=a.gamma_bar, given_order=a.perm())
    assert np.array_equal(a.perm(), b.perm())
    for u, v in zip(a.node_arrays(), b.node_arrays()):
        assert np.array_equal(u, v)
    for u, v in zip(a.lists(), b.lists()):
        assert np.array_equal(u, v)
    Ea, Ba = a.eval()
    Eb, Bb = b.eval()
    assert np.array_equal(Ea, Eb) and np.array_equal(Ba, Bb)


def test_given_order_after_a_drift_is_a_valid_tree_with_the_same_accuracy():
    """Particles drift (a tracker step); the OLD order is kept.  The plan is still a partition with tight boxes, every
    leaf pair is covered exactly once (P10), and the FMM error against the direct sum stays at the KD tree's level."""
    w = small(N=4096)
    old = plan_of(w, theta=0.5)
    rng = np.random.default_rng(3)
    x2 = w.x + 2e-5 * rng.standard_normal(w.N)       # 2 % of sigma_x
    y2 = w.y + 2e-5 * rng.standard_normal(w.N)
    z2 = w.z + 2e-6 * rng.standard_normal(w.N)
    args = (x2, y2, z2, w.px, w.py, w.pz)
    p = oracle.Plan(*args, w.q, order_n=4, leaf_size=64, theta=0.5, given_order=old.perm())
    assert np.array_equal(p.perm(), old.perm())
    lo, hi, bb = p.node_arrays()
    lo0, hi0, _ = old.node_arrays()
    assert np.array_equal(lo, lo0) and np.array_equal(hi, hi0)           # T-2 ranges depend on (N, N0) only
    perm = p.perm()
    for i in (1, 2, 37, p.nodes):                                         # tight boxes (T-4)
        m = perm[lo[i - 1]:hi[i - 1]]
        assert np.array_equal(bb[i - 1], [x2[m].min(), y2[m].min(), z2[m].min(), x2[m].max(), y2[m].max(), z2[m].max()])
    p2p, m2l = p.lists()
    Lf = p.leaves
    cover = np.zeros((Lf, Lf), dtype=np.int32)
    for t, s in np.concatenate([p2p, m2l]):
        lt, ls = int(np.log2(t)), int(np.log2(s))
        wt, ws = Lf >> lt, Lf >> ls
        cover[(t - (1 << lt)) * wt:(t - (1 << lt) + 1) * wt, (s - (1 << ls)) * ws:(s - (1 << ls) + 1) * ws] += 1
    assert np.all(cover == 1)
    Ed, Bd = oracle.direct(*args, w.q, gamma_bar_value=p.gamma_bar)
    E, B = p.eval()
    fresh = oracle.Plan(*args, w.q, order_n=4, leaf_size=64, theta=0.5, gamma_bar_value=p.gamma_bar)
    Ef, _ = fresh.eval()
    e_refit, e_fresh = oracle.err2(E, Ed), oracle.err2(Ef, Ed)
    assert e_refit < 3 * e_fresh and e_refit < 5e-3, (e_refit, e_fresh)


# ---------------------------------------------------------------------------------------------
# Treecode variant (particle-cluster; Fig. 1a)
# ---------------------------------------------------------------------------------------------
def _leaf_span(i, Lf):
    lvl = int(np.log2(i)); width = Lf >> lvl
    first = (i - (1 << lvl)) * width
    return first, first + width


@pytest.mark.parametrize("theta", [0.3, 0.5])
def test_treecode_lists_cover_every_source_leaf_once_per_target_leaf(theta):
    w = small(N=4096)
    p = plan_of(w, theta=theta)
    pp, pc = p.treecode_lists()
    Lf = p.leaves
    cover = np.zeros((Lf, Lf), dtype=np.int32)
    assert np.all(pp >= Lf) and np.all(pc[:, 0] >= Lf)           # targets are leaves; PP sources are leaves
    for t, s in np.concatenate([pp, pc]):
        s0, s1 = _leaf_span(s, Lf)
        cover[t - Lf, s0:s1] += 1
    assert np.all(cover == 1)
    assert len(pc) > 0 or theta < 0.5                            # (theta = 0.3 leaves no admissible cluster at this size)
    lo, hi, bb = p.node_arrays()                                 # every PC pair satisfies Alg 5.8, no PP pair was tested
    s = np.array([1.0, 1.0, p.gamma_bar])
    for t, c in pc[:: max(1, len(pc) // 200)]:
        bt, bc = bb[t - 1], bb[c - 1]
        rt = np.linalg.norm(s * (bt[3:] - bt[:3]) * 0.5); rc = np.linalg.norm(s * (bc[3:] - bc[:3]) * 0.5)
        d = np.linalg.norm(s * ((bt[:3] + bt[3:]) * 0.5 - (bc[:3] + bc[3:]) * 0.5))
        assert max(rt, rc) < theta * d * (1 + 1e-12)


def test_treecode_equals_numpy_restatement_and_direct_without_clusters():
    """PC interaction restated in numpy from the exported moments, boxes and Chebyshev points; with a tiny theta the
    PC list is empty and the treecode is the direct sum."""
    w = small(N=600)
    p = oracle.Plan(*w.arrays(), w.q, order_n=3, leaf_size=40, theta=0.5, raw=True)
    pp, pc = p.treecode_lists()
    M = p.upward()
    lo, hi, bb = p.node_arrays()
    perm = p.perm()
    c = oracle.cheb_nodes(3)
    g2 = p.gamma_bar ** 2
    X = np.stack([w.x, w.y, w.z], axis=1)
    gam = np.sqrt(1 + w.px ** 2 + w.py ** 2 + w.pz ** 2)
    W = np.stack([w.q * gam, w.q * w.px, w.q * w.py, w.q * w.pz], axis=1)
    E = np.zeros((w.N, 3)); B = np.zeros((w.N, 3))

    def add(tidx, src_x, src_w):
        d = X[tidx][:, None, :] - src_x[None, :, :]
        D = d[..., 0] ** 2 + d[..., 1] ** 2 + g2 * d[..., 2] ** 2
        wgt = np.where(D > 0, 1.0 / np.where(D > 0, D, 1.0) ** 1.5, 0.0)
        g = wgt[..., None] * d
        E[tidx] += np.einsum("ts,tsk->tk", src_w[None, :, 0] * np.ones_like(wgt), g)
        B[tidx] += np.einsum("tsk->tk", np.cross(np.broadcast_to(src_w[None, :, 1:], g.shape), g))
    for t, s in pp:
        add(perm[lo[t - 1]:hi[t - 1]], X[perm[lo[s - 1]:hi[s - 1]]], W[perm[lo[s - 1]:hi[s - 1]]])
    for t, s in pc:
        b = bb[s - 1]
        ax = [(b[k] + b[3 + k]) * 0.5 + (b[3 + k] - b[k]) * 0.5 * c for k in range(3)]
        xi = np.stack(np.meshgrid(*ax, indexing="ij"), axis=-1).reshape(-1, 3)      # nu = (nu1 (n+1) + nu2)(n+1) + nu3
        add(perm[lo[t - 1]:hi[t - 1]], xi, M[s - 1])
    Et, Bt = p.eval_treecode()
    assert len(pc) > 0
    assert oracle.err2(Et, E) < 1e-13 and oracle.err2(Bt, B) < 1e-13
    q = oracle.Plan(*w.arrays(), w.q, order_n=3, leaf_size=40, theta=0.01, raw=True)
    assert len(q.treecode_lists()[1]) == 0
    Ed, Bd = oracle.direct(*w.arrays(), w.q, raw=True)
    Eq, Bq = q.eval_treecode()
    assert oracle.err2(Eq, Ed) < 1e-13 and oracle.err2(Bq, Bd) < 1e-13


def test_treecode_converges_and_is_at_least_as_accurate_as_the_fmm():
    w = small(N=4096)
    Ed, _ = oracle.direct(*w.arrays(), w.q)
    errs = []
    for n in (2, 4, 6):
        p = oracle.Plan(*w.arrays(), w.q, order_n=n, leaf_size=64, theta=0.5)
        Et, _ = p.eval_treecode()
        Ef, _ = p.eval()
        et, ef = oracle.err2(Et, Ed), oracle.err2(Ef, Ed)
        errs.append(et)
        assert et < 1.5 * ef, (n, et, ef)        # only the source side is interpolated
    assert errs[0] > errs[1] > errs[2] and errs[2] < 1e-3
