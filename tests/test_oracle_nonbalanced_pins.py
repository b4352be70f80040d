"""Pins for the oracle's non-balanced tree option (ORC_TREE_STOP_AT_N0; no GPU).

Alg 5.2 as printed splits a cluster only while |S| > N0.  With median splits the sizes of a level
differ by at most one, so this differs from the complete tree of reading T-1 exactly when some clusters of level
kappa-1 hold N0 particles: those stay leaves, the tree has leaves on two levels.  Pinned here by

* a restatement of Alg 5.1 / 5.2 on plain Python index sets (recursion as printed, no arrays, no levels) whose
  clusters, leaves and particle order must equal the oracle's, and Alg 5.11 restated over that tree (children(S)
  empty <=> leaf) whose two lists must equal the oracle's exactly;
* the invariants of Alg 5.2 (a leaf holds at most N0, a split cluster more than N0, the leaves partition the bunch);
* identity with the complete tree whenever no cluster of level kappa-1 holds exactly N0 particles;
* exactly-once coverage of every ordered leaf pair by P2P + M2L (brute force over the leaf x leaf matrix);
* M2M == P2M at the parent of a level-(kappa-1) leaf (its moments must come from P2M at that leaf), empty far list
  => FMM == direct, FMM -> direct as n grows, treecode == direct trend.
"""
import sys

import numpy as np
import pytest

import oracle
from paper_2302_07567_b200 import workloads


def alg52_tree(x, y, z, s, N0):
    """Alg 5.2 with Alg 5.1 on index sets.  Readings G7 (left child gets
    ceil(|S|/2)), G8 (members ranked by (coordinate, index)), G9 (first maximiser).  Returns
    {heap id: (members, is_leaf)} with the members of a leaf in ascending index (T-3)."""
    coord = (x, y, z)
    tree = {}

    def subdivide(node, S):
        if len(S) > N0:                                   # "if |S| > N0 then"
            ext = [s[k] * (max(coord[k][i] for i in S) - min(coord[k][i] for i in S)) for k in range(3)]
            k = 0
            for c in (1, 2):
                if ext[c] > ext[k]:
                    k = c
            ranked = sorted(S, key=lambda i: (coord[k][i], i))
            half = (len(S) + 1) // 2
            tree[node] = (sorted(S), False)
            subdivide(2 * node, ranked[:half])
            subdivide(2 * node + 1, ranked[half:])
        else:                                             # "children(S) = {}"
            tree[node] = (sorted(S), True)

    old = sys.getrecursionlimit()
    sys.setrecursionlimit(10000)
    try:
        subdivide(1, list(range(len(x))))
    finally:
        sys.setrecursionlimit(old)
    return tree


def alg511_on_tree(tree, x, y, z, s, eta):
    """Alg 5.11 over a tree given as {id: (members, is_leaf)}; Alg 5.6-5.8 squared in the order
    of reading D-2 (Python floats: every operation rounded separately)."""
    coord = (x, y, z)
    box = {}
    for i, (S, _) in tree.items():
        if S:
            box[i] = ([min(float(coord[k][j]) for j in S) for k in range(3)], [max(float(coord[k][j]) for j in S) for k in range(3)])
    p2p, m2l = [], []
    eta2 = eta * eta

    def diam2(i):
        a, b = box[i]
        e = [s[k] * ((b[k] - a[k]) * 0.5) for k in range(3)]
        return (e[0] * e[0] + e[1] * e[1]) + e[2] * e[2]

    def dist2(i, j):
        (ai, bi), (aj, bj) = box[i], box[j]
        e = [s[k] * ((ai[k] + bi[k]) * 0.5 - (aj[k] + bj[k]) * 0.5) for k in range(3)]
        return (e[0] * e[0] + e[1] * e[1]) + e[2] * e[2]

    def rec(t, src):
        if not tree[t][0] or not tree[src][0]:
            return
        leaf_t, leaf_s = tree[t][1], tree[src][1]
        if leaf_t and leaf_s:
            p2p.append((t, src))
            return
        rt, rs = diam2(t), diam2(src)
        if max(rt, rs) < eta2 * dist2(t, src):
            m2l.append((t, src))
        elif leaf_t:
            rec(t, 2 * src); rec(t, 2 * src + 1)
        elif leaf_s:
            rec(2 * t, src); rec(2 * t + 1, src)
        elif rt > rs:
            rec(2 * t, src); rec(2 * t + 1, src)
        else:
            rec(t, 2 * src); rec(t, 2 * src + 1)

    rec(1, 1)
    return (np.array(sorted(p2p), dtype=np.int32).reshape(-1, 2), np.array(sorted(m2l), dtype=np.int32).reshape(-1, 2))


def bunch(N):
    return workloads.config(1, N=N)


# (N, N0) with floor(N / 2^(kappa-1)) == N0: clusters of exactly N0 particles exist one level above kappa
EARLY = [(4097, 64), (1030, 16), (2500, 39), (300, 37), (3, 1), (129, 64)]


@pytest.mark.parametrize("N,N0", EARLY)
def test_alg52_as_printed_restated_on_sets(N, N0):
    """Clusters, leaves, particle order and both lists of the oracle equal those of Alg 5.2 / 5.11 restated on sets."""
    w = bunch(N)
    p = oracle.Plan(*w.arrays(), q=w.q, order_n=2, leaf_size=N0, theta=0.5, stop_at_n0=True)
    x, y, z = (np.asarray(a, dtype=float) for a in w.arrays()[:3])
    s = (1.0, 1.0, p.gamma_bar)
    tree = alg52_tree(x, y, z, s, N0)
    lo, hi, bb = p.node_arrays()
    flags, perm = p.leaf_flags(), p.perm()
    assert set(np.flatnonzero(flags != 2) + 1) == set(tree)              # the same clusters exist
    for i, (S, is_leaf) in tree.items():
        assert flags[i - 1] == (1 if is_leaf else 0)
        members = perm[lo[i - 1]:hi[i - 1]]
        assert sorted(members.tolist()) == S
        if is_leaf:
            assert members.tolist() == S                                   # T-3: ascending index inside a leaf
    # leaves on two levels, and the early ones hold exactly N0
    leaf_ids = p.leaf_ids()
    levels = np.floor(np.log2(leaf_ids)).astype(int)
    assert set(levels) == {p.kappa - 1, p.kappa}
    early = leaf_ids[levels == p.kappa - 1]
    assert len(early) > 0 and all(hi[i - 1] - lo[i - 1] == N0 for i in early)
    # unused slots are exactly the children of those leaves: empty range, zero box
    unused = np.flatnonzero(flags == 2) + 1
    assert sorted(unused.tolist()) == sorted([2 * i for i in early] + [2 * i + 1 for i in early])
    assert not lo[unused - 1].any() and not hi[unused - 1].any() and not bb[unused - 1].any()
    p2p_r, m2l_r = alg511_on_tree(tree, x, y, z, s, 0.5)
    p2p_o, m2l_o = p.lists()
    np.testing.assert_array_equal(p2p_o, p2p_r)
    np.testing.assert_array_equal(m2l_o, m2l_r)
    if N >= 1000:
        assert len(m2l_o) > 0
        # the two trees really differ here: the complete tree has other lists
        q = oracle.Plan(*w.arrays(), q=w.q, order_n=2, leaf_size=N0, theta=0.5)
        assert q.lists()[0].shape != p2p_o.shape


@pytest.mark.parametrize("mode", [oracle.TREE_KD, oracle.TREE_MORTON_MEDIAN])
@pytest.mark.parametrize("N,N0", EARLY + [(4096, 64), (5003, 37), (1000, 1000), (17, 64)])
def test_alg52_invariants_and_coverage(N, N0, mode):
    """A leaf holds at most N0, a split cluster more than N0, the leaves partition the bunch (Alg 5.2), and every
    ordered pair of leaves is covered exactly once by P2P or by an M2L pair of ancestors (P10, brute force)."""
    w = bunch(N)
    p = oracle.Plan(*w.arrays(), q=w.q, order_n=2, leaf_size=N0, theta=0.5, tree_mode=mode, stop_at_n0=True)
    lo, hi, _ = p.node_arrays()
    flags = p.leaf_flags()
    size = hi - lo
    assert (size[flags == 1] <= N0).all() and (size[flags == 0] > N0).all()
    leaf_ids = p.leaf_ids()
    order = np.argsort(lo[leaf_ids - 1], kind="stable")
    cover = np.concatenate([np.arange(lo[i - 1], hi[i - 1]) for i in leaf_ids[order]])
    np.testing.assert_array_equal(cover, np.arange(N))
    for i in np.flatnonzero(flags == 0) + 1:                              # children tile the parent, left gets the ceiling
        assert lo[2 * i - 1] == lo[i - 1] and hi[2 * i] == hi[i - 1] and hi[2 * i - 1] == lo[2 * i]
        assert size[2 * i - 1] == (size[i - 1] + 1) // 2
    # coverage: count[a, b] over non-empty leaves
    live = [int(i) for i in leaf_ids if size[i - 1] > 0]
    pos = {i: k for k, i in enumerate(live)}

    def leaves_below(i):
        if flags[i - 1] == 1:
            return [i] if i in pos else []
        return leaves_below(2 * i) + leaves_below(2 * i + 1)

    count = np.zeros((len(live), len(live)), dtype=np.int64)
    p2p, m2l = p.lists()
    for t, s_ in p2p:
        assert flags[t - 1] == 1 and flags[s_ - 1] == 1
        count[pos[int(t)], pos[int(s_)]] += 1
    for t, s_ in m2l:
        a = [pos[i] for i in leaves_below(int(t))]
        b = [pos[i] for i in leaves_below(int(s_))]
        count[np.ix_(a, b)] += 1
    assert (count == 1).all()


@pytest.mark.parametrize("mode", [oracle.TREE_KD, oracle.TREE_MORTON_MEDIAN])
@pytest.mark.parametrize("N,N0", [(4096, 64), (5003, 37), (4160, 64), (1000, 1000)])
def test_same_tree_when_no_cluster_holds_exactly_n0(N, N0, mode):
    """floor(N / 2^(kappa-1)) != N0 (or kappa = 0): Alg 5.2 as printed gives the complete tree of reading T-1 (G13)."""
    w = bunch(N)
    a = oracle.Plan(*w.arrays(), q=w.q, order_n=2, leaf_size=N0, theta=0.5, tree_mode=mode, stop_at_n0=True)
    b = oracle.Plan(*w.arrays(), q=w.q, order_n=2, leaf_size=N0, theta=0.5, tree_mode=mode)
    assert (a.leaf_flags() != 2).all()
    np.testing.assert_array_equal(a.leaf_ids(), np.arange(b.leaves, b.nodes + 1))
    np.testing.assert_array_equal(a.perm(), b.perm())
    for u, v in zip(a.lists(), b.lists()):
        np.testing.assert_array_equal(u, v)
    for u, v in zip(a.node_arrays(), b.node_arrays()):
        np.testing.assert_array_equal(u, v)


def test_moments_of_an_early_leaf_come_from_p2m():
    """P7 at the parent of a level-(kappa-1) leaf: M2M of (P2M at that leaf, M2M of its sibling's children) equals
    P2M evaluated directly at the parent (exact up to rounding, Theorem 1); the unused slots carry nothing."""
    N, N0 = 1030, 16
    w = bunch(N)
    p = oracle.Plan(*w.arrays(), q=w.q, order_n=3, leaf_size=N0, theta=0.5, stop_at_n0=True, raw=True)
    M = p.upward()
    flags = p.leaf_flags()
    early = [int(i) for i in p.leaf_ids() if i < p.leaves]
    assert early
    for i in early[:8]:
        np.testing.assert_array_equal(M[i - 1], p.p2m_node(i))
        assert not M[2 * i - 1].any() and not M[2 * i].any()
        par = i // 2
        ref = p.p2m_node(par)
        assert np.max(np.abs(M[par - 1] - ref)) <= 1e-12 * np.max(np.abs(ref))
    ref = p.p2m_node(1)
    assert np.max(np.abs(M[0] - ref)) <= 1e-12 * np.max(np.abs(ref))
    assert (flags == 2).sum() == 2 * len(early)


@pytest.mark.parametrize("N,N0", [(1030, 16), (300, 37), (3, 1)])
def test_empty_far_list_is_direct(N, N0):
    """P9 on the non-balanced tree: eta so small that nothing is admissible => FMM == direct sum."""
    w = bunch(N)
    p = oracle.Plan(*w.arrays(), q=w.q, order_n=2, leaf_size=N0, theta=1e-6, stop_at_n0=True)
    assert p.n_m2l == 0
    E, B = p.eval()
    Ed, Bd = oracle.direct(*w.arrays(), w.q, gamma_bar_value=p.gamma_bar)
    assert oracle.err2(E, Ed) <= 1e-13 and oracle.err2(B, Bd) <= 1e-13


def test_convergence_on_the_non_balanced_tree():
    """P12: the FMM on the non-balanced tree converges to the direct sum as n grows; so does its treecode variant;
    selected-leaf evaluation accepts an early leaf and agrees with the full one."""
    N, N0 = 2500, 39
    w = bunch(N)
    Ed, Bd = None, None
    errs, errs_tc = [], []
    for n in (2, 4, 6):
        p = oracle.Plan(*w.arrays(), q=w.q, order_n=n, leaf_size=N0, theta=0.5, stop_at_n0=True)
        if Ed is None:
            Ed, Bd = oracle.direct(*w.arrays(), w.q, gamma_bar_value=p.gamma_bar)
        E, B = p.eval()
        errs.append(oracle.err2(E, Ed))
        Et, Bt = p.eval_treecode()
        errs_tc.append(oracle.err2(Et, Ed))
    assert errs[0] > 2 * errs[1] > 4 * errs[2] and errs[2] < 1e-3, errs
    assert errs_tc[0] > 2 * errs_tc[1] > 4 * errs_tc[2] and errs_tc[2] < 1e-3, errs_tc
    q = oracle.Plan(*w.arrays(), q=w.q, order_n=6, leaf_size=N0, theta=0.5)   # the complete tree: same error level
    assert errs[2] / 3 < oracle.err2(q.eval()[0], Ed) < errs[2] * 3
    early = [int(i) for i in p.leaf_ids() if i < p.leaves][:3]
    Es, Bs = p.eval(leaves=early)
    lo, hi, _ = p.node_arrays()
    perm = p.perm()
    for i in early:
        idx = perm[lo[i - 1]:hi[i - 1]]
        np.testing.assert_array_equal(Es[idx], E[idx])
        np.testing.assert_array_equal(Bs[idx], B[idx])
    with pytest.raises(ValueError):
        p.eval(leaves=[2 * early[0]])                                     # an unused slot is not a leaf
