"""Pins for the oracle's dual tree traversal and split-axis choice (no GPU).

The GPU lists are compared bit for bit with whatever the oracle emits, so the oracle's own
traversal needs a pin that is not itself: here Alg 5.11 (same logic as
Alg 9.1) is restated as a plain recursive Python function over the oracle's
exported bounding boxes, with Alg 5.6-5.8 evaluated in the order of reading
D-2 in IEEE doubles (Python floats: every product and sum rounded separately, no FMA).  The
restated lists must equal ``Plan.lists()`` exactly.  A wrong split choice (always the source,
``>=`` instead of ``>``, the target on a tie) changes these lists on the inputs below; each test
first shows, with the restatement itself, that the alternative rule gives different lists, so the
pin can fail.

Also here: Alg 5.1 with two and three axes tied on a NON-ZERO stretched
extent (reading G9: first maximiser in the order x, y, z).
"""
import sys

import numpy as np
import pytest

import oracle
from paper_2302_07567_b200 import workloads


def alg511_lists(bb, leaves, sizes, s, eta, split_target_rule="gt"):
    """Alg 5.11 with P2P / M2L replaced by list appends (= Alg 9.1).  bb[i-1] = bbox of heap node i.
    split_target_rule: 'gt' = the paper's `diam(S_t) > diam(S_s)` (ties split the source, D-3);
    'ge' and 'never' are the wrong rules used to show that the pin discriminates."""
    p2p, m2l = [], []
    eta2 = eta * eta

    def diam2(i):  # Alg 5.6 squared, D-2 order
        a, b = bb[i - 1, :3], bb[i - 1, 3:]
        e = [s[k] * ((float(b[k]) - float(a[k])) * 0.5) for k in range(3)]
        return (e[0] * e[0] + e[1] * e[1]) + e[2] * e[2]

    def dist2(i, j):  # Alg 5.7 squared, D-2 order
        e = []
        for k in range(3):
            ci = (float(bb[i - 1, k]) + float(bb[i - 1, 3 + k])) * 0.5
            cj = (float(bb[j - 1, k]) + float(bb[j - 1, 3 + k])) * 0.5
            e.append(s[k] * (ci - cj))
        return (e[0] * e[0] + e[1] * e[1]) + e[2] * e[2]

    def rec(t, src):
        if sizes[t - 1] == 0 or sizes[src - 1] == 0:   # an empty cluster takes part in nothing
            return
        leaf_t, leaf_s = t >= leaves, src >= leaves    # children(S) == {} (complete tree, T-1)
        if leaf_t and leaf_s:
            p2p.append((t, src))
            return
        rt, rs = diam2(t), diam2(src)
        if max(rt, rs) < eta2 * dist2(t, src):          # Alg 5.8 squared (D-2)
            m2l.append((t, src))
        elif leaf_t:
            rec(t, 2 * src); rec(t, 2 * src + 1)
        elif leaf_s:
            rec(2 * t, src); rec(2 * t + 1, src)
        else:
            split_target = {"gt": rt > rs, "ge": rt >= rs, "never": False}[split_target_rule]
            if split_target:
                rec(2 * t, src); rec(2 * t + 1, src)
            else:
                rec(t, 2 * src); rec(t, 2 * src + 1)

    old = sys.getrecursionlimit()
    sys.setrecursionlimit(10000)
    try:
        rec(1, 1)
    finally:
        sys.setrecursionlimit(old)
    return (np.array(sorted(p2p), dtype=np.int32).reshape(-1, 2), np.array(sorted(m2l), dtype=np.int32).reshape(-1, 2))


def restate(p, eta, rule="gt"):
    lo, hi, bb = p.node_arrays()
    return alg511_lists(bb, p.leaves, hi - lo, (1.0, 1.0, p.gamma_bar), eta, rule)


@pytest.mark.parametrize("mode", [oracle.TREE_KD, oracle.TREE_MORTON_MEDIAN])
@pytest.mark.parametrize("theta", [0.3, 0.5])
@pytest.mark.parametrize("N,N0", [(4096, 64), (4096, 16), (5003, 37)])
def test_alg511_restatement_equals_oracle_lists(N, N0, theta, mode):
    """The oracle's lists are exactly those of Alg 5.11 restated in Python (full N and a ragged N)."""
    w = workloads.config(1, N=N)
    p = oracle.Plan(*w.arrays(), q=w.q, order_n=2, leaf_size=N0, theta=theta, tree_mode=mode)
    p2p_o, m2l_o = p.lists()
    p2p_r, m2l_r = restate(p, theta)
    np.testing.assert_array_equal(p2p_o, p2p_r)
    np.testing.assert_array_equal(m2l_o, m2l_r)
    if N0 == 64 and theta == 0.3:
        assert len(m2l_r) == 0      # pin P9's case: nothing is admissible, every leaf pair is near field
        return
    assert len(m2l_r) > 0
    # the pin can fail: never splitting the target (the mutant `else if (0)`) gives other lists
    p2p_n, m2l_n = restate(p, theta, "never")
    assert m2l_n.shape != m2l_r.shape or not np.array_equal(m2l_n, m2l_r)


def mirrored_cloud(N_half, seed):
    """A cloud that is mirror-symmetric in x: siblings (and all mirrored node pairs) then have bit-identical
    stretched radii, which is the tie of reading D-3."""
    rng = np.random.default_rng(seed)
    x = rng.uniform(0.01, 4.0, N_half)          # long in x: the root splits along x
    y = rng.uniform(-0.5, 0.5, N_half)
    z = rng.uniform(-0.05, 0.05, N_half)
    X = np.concatenate([x, -x]); Y = np.concatenate([y, y]); Z = np.concatenate([z, z])
    return X, Y, Z


@pytest.mark.parametrize("theta,seed,N_half,N0", [(0.5, 7, 512, 16), (0.5, 8, 512, 16), (0.5, 9, 1024, 8), (0.3, 7, 1024, 8)])
def test_d3_tie_splits_the_source(theta, seed, N_half, N0):
    """diam(S_t) == diam(S_s) (not >) => the source is split (Alg 5.11 `else` branch)."""
    X, Y, Z = mirrored_cloud(N_half, seed)
    N = 2 * N_half
    pz = np.full(N, 3.0)
    p = oracle.Plan(X, Y, Z, np.zeros(N), np.zeros(N), pz, q=1.0, order_n=2, leaf_size=N0, theta=theta)
    lo, hi, bb = p.node_arrays()
    # the tie is really there: nodes 2 and 3 are mirror images with identical extents
    np.testing.assert_array_equal(bb[1, 3:] - bb[1, :3], bb[2, 3:] - bb[2, :3])
    p2p_o, m2l_o = p.lists()
    p2p_r, m2l_r = restate(p, theta, "gt")
    np.testing.assert_array_equal(p2p_o, p2p_r)
    np.testing.assert_array_equal(m2l_o, m2l_r)
    # splitting the target on a tie (`>=`) gives different lists on this input, so the equality above pins the tie rule
    p2p_g, m2l_g = restate(p, theta, "ge")
    assert m2l_g.shape != m2l_r.shape or not np.array_equal(m2l_g, m2l_r)


def test_d3_tie_minimal_example_by_hand():
    """Sixteen points worked by hand: x = +-(0.25, 1, 2, ..., 7), y alternating +-1.5, z = 0, leaves of 2, eta = 0.5.
    Level-1 nodes 2 (x in [-7,-0.25]) and 3 (x in [0.25,7]) are mirror images: r = sqrt(3.375^2 + 1.5^2) = 3.693 each
    (the tie), d = 7.25, r/d = 0.509: not admissible.  (3,2) must split the SOURCE: (3,4) with 4 = x in [-7,-4]:
    max r = 3.693, d = 9.125 -> 0.405 < 0.5, admissible, so M2L holds (3,4); and (3,5) -> target split -> (7,5) with
    7 = x in [4,7], 5 = x in [-3,-0.25]: max r = 2.12, d = 7.125 -> admissible.  Splitting the target on the tie would
    test (6,2) (r/d = 3.693/5.25: not admissible) and (7,2), and (3,4) could never be emitted."""
    ax = np.array([0.25, 1, 2, 3, 4, 5, 6, 7], dtype=float)
    xs = np.concatenate([-ax[::-1], ax])
    ys = np.where(np.arange(16) % 2 == 0, 1.5, -1.5)
    N = len(xs)
    p = oracle.Plan(xs, ys, np.zeros(N), np.zeros(N), np.zeros(N), np.zeros(N), q=1.0, order_n=1,
                    leaf_size=2, theta=0.5)
    lo, hi, bb = p.node_arrays()
    np.testing.assert_array_equal(bb[1], [-7, -1.5, 0, -0.25, 1.5, 0])
    np.testing.assert_array_equal(bb[2], [0.25, -1.5, 0, 7, 1.5, 0])
    np.testing.assert_array_equal(bb[3], [-7, -1.5, 0, -4, 1.5, 0])
    np.testing.assert_array_equal(bb[6], [4, -1.5, 0, 7, 1.5, 0])
    _, m2l = p.lists()
    pairs = set(map(tuple, m2l.tolist()))
    assert (2, 3) not in pairs and (3, 2) not in pairs
    assert (3, 4) in pairs and (2, 7) in pairs and (7, 5) in pairs and (4, 6) in pairs
    assert not any(t in (6, 7) and s == 2 for t, s in pairs) and not any(t in (4, 5) and s == 3 for t, s in pairs)
    assert (4, 3) not in pairs and (7, 2) not in pairs


# ---------------------------------------------------------------- Alg 5.1, reading G9
def _left_members(p):
    lo, hi, _ = p.node_arrays()
    return set(p.perm()[lo[1]:hi[1]].tolist())   # node 2 = left child of the root


def test_g9_two_axes_tie_on_nonzero_extent_first_wins():
    """x and y extents are both exactly 1 (z smaller): the split axis is x, the FIRST maximiser."""
    # 8 points; by x the lower half is {0,1,2,3}, by y it is {0,2,4,6}
    x = np.array([0.0, 0.1, 0.2, 0.3, 0.7, 0.8, 0.9, 1.0])
    y = np.array([0.0, 1.0, 0.1, 0.9, 0.2, 0.8, 0.3, 0.7])
    z = np.array([0.0, 0.01, 0.02, 0.03, 0.04, 0.05, 0.06, 0.07])
    N = 8
    p = oracle.Plan(x, y, z, np.zeros(N), np.zeros(N), np.zeros(N), q=1.0, order_n=1, leaf_size=4, theta=0.5,
                    gamma_bar_value=2.0)
    assert _left_members(p) == {0, 1, 2, 3}
    # y strictly larger -> y wins (the argmax is really taken)
    y2 = y * 1.5
    p = oracle.Plan(x, y2, z, np.zeros(N), np.zeros(N), np.zeros(N), q=1.0, order_n=1, leaf_size=4, theta=0.5,
                    gamma_bar_value=2.0)
    assert _left_members(p) == {0, 2, 4, 6}


def test_g9_stretched_z_ties_and_wins():
    """The extent that counts is s_k (b_k - a_k) with s = (1, 1, gamma_bar) (Alg 5.1):
    z extent 0.5 with gamma_bar = 2 ties x and y at 1.0 -> x; y and z tie above x -> y; gamma_bar = 2.5 -> z."""
    x = np.array([0.0, 0.1, 0.2, 0.3, 0.7, 0.8, 0.9, 1.0])
    y = np.array([0.0, 1.0, 0.1, 0.9, 0.2, 0.8, 0.3, 0.7])
    z = np.array([0.5, 0.4, 0.0, 0.1, 0.45, 0.35, 0.05, 0.15])   # by z the lower half is {2,3,6,7}
    N = 8
    mk = lambda xx, gb: oracle.Plan(xx, y, z, np.zeros(N), np.zeros(N), np.zeros(N), q=1.0, order_n=1, leaf_size=4,
                                    theta=0.5, gamma_bar_value=gb)
    assert _left_members(mk(x, 2.0)) == {0, 1, 2, 3}          # three-way tie at 1.0 -> x
    assert _left_members(mk(x * 0.5, 2.0)) == {0, 2, 4, 6}    # x extent 0.5; y and gamma z tie at 1.0 -> y
    assert _left_members(mk(x, 2.5)) == {2, 3, 6, 7}          # gamma z = 1.25 > 1 -> z
