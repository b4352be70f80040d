"""Pins for the oracle's list reuse (orc_plan_set_lists, orc_plan_eta_eff; no GPU).

A refit may keep the interaction lists of an earlier traversal while the particles move a little.  The oracle then
evaluates Alg 5.12 over lists it is handed, and reports how far the kept far pairs are from eq. (4.3).  Pinned by:
* lists of another plan over the same tree (eta = 0.3 handed to an eta = 0.5 plan) reproduce that plan's fields bit for bit,
  and the plan's own lists handed back change nothing;
* the all-near list (every ordered pair of leaves in P2P, no M2L) reproduces the direct sum;
* eta_eff equals a numpy restatement of Alg 5.6-5.8 on the exported boxes, is below theta for every list the oracle's own
  traversal made (Alg 5.8), and above it once a kept pair's boxes have moved enough;
* kept lists after a drift still cover every ordered pair of leaves exactly once, and the error against the direct sum
  of the moved particles stays at the level of a fresh traversal.
"""
import numpy as np
import pytest

import oracle
from paper_2302_07567_b200 import workloads


def eta_restated(p):
    """Alg 5.6-5.8 with s = (1, 1, gamma_bar) over the plan's M2L list, float64 numpy."""
    _, _, bb = p.node_arrays()
    _, m2l = p.lists()
    if len(m2l) == 0:
        return 0.0
    s = np.array([1.0, 1.0, p.gamma_bar])
    a, b = bb[:, :3], bb[:, 3:]
    r2 = (((b - a) * 0.5 * s) ** 2)
    r2 = (r2[:, 0] + r2[:, 1]) + r2[:, 2]
    c = (a + b) * 0.5
    e = (c[m2l[:, 0] - 1] - c[m2l[:, 1] - 1]) * s
    d2 = (e[:, 0] ** 2 + e[:, 1] ** 2) + e[:, 2] ** 2
    return float(np.sqrt(np.max(np.maximum(r2[m2l[:, 0] - 1], r2[m2l[:, 1] - 1]) / d2)))


@pytest.mark.parametrize("mode", [oracle.TREE_KD, oracle.TREE_MORTON_MEDIAN])
@pytest.mark.parametrize("cfg,N,N0,theta", [(1, 4096, 64, 0.5), (2, 5003, 37, 0.4), (4, 3000, 50, 0.3), (3, 2000, 100, 0.7)])
def test_eta_eff_restated_and_below_theta(cfg, N, N0, theta, mode):
    w = workloads.config(cfg, N=N)
    p = oracle.Plan(*w.arrays(), q=w.q, order_n=2, leaf_size=N0, theta=theta, tree_mode=mode)
    assert p.n_m2l > 0
    assert p.eta_eff() == eta_restated(p)
    assert 0.5 * theta < p.eta_eff() < theta        # Alg 5.8 holds for every emitted far pair, and some pair is close to it


def test_handed_lists_are_the_ones_evaluated():
    w = workloads.config(1, N=3000)
    kw = dict(order_n=3, leaf_size=40)
    a = oracle.Plan(*w.arrays(), q=w.q, theta=0.5, **kw)
    b = oracle.Plan(*w.arrays(), q=w.q, theta=0.3, gamma_bar_value=a.gamma_bar, **kw)
    Ea, Ba = a.eval()
    Eb, Bb = b.eval()
    assert a.n_m2l != b.n_m2l and not np.array_equal(Ea, Eb)
    a.set_lists(*a.lists())                          # its own lists: nothing changes
    E, B = a.eval()
    assert np.array_equal(E, Ea) and np.array_equal(B, Ba)
    a.set_lists(*[v[::-1] for v in b.lists()])       # the eta = 0.3 lists (any order): a becomes b
    for u, v in zip(a.lists(), b.lists()):
        np.testing.assert_array_equal(u, v)
    E, B = a.eval()
    assert np.array_equal(E, Eb) and np.array_equal(B, Bb)
    assert a.eta_eff() == b.eta_eff() < 0.3
    # all-near list: the direct sum
    leaves = [int(i) for i in a.leaf_ids()]
    allnear = np.array([(t, s) for t in leaves for s in leaves], dtype=np.int32)
    a.set_lists(allnear, np.zeros((0, 2), dtype=np.int32))
    assert a.eta_eff() == 0.0
    E, B = a.eval()
    Ed, Bd = oracle.direct(*w.arrays(), w.q, gamma_bar_value=a.gamma_bar)
    assert oracle.err2(E, Ed) <= 1e-13 and oracle.err2(B, Bd) <= 1e-13
    with pytest.raises(ValueError):
        a.set_lists(np.array([[1, leaves[0]]], dtype=np.int32), np.zeros((0, 2), dtype=np.int32))   # the root is no leaf
    with pytest.raises(ValueError):
        a.set_lists(allnear, np.array([[a.nodes + 1, 2]], dtype=np.int32))


@pytest.mark.parametrize("stop", [False, True])
def test_kept_lists_after_a_drift(stop):
    N, N0, theta = 4097, 64, 0.5
    w = workloads.config(1, N=N)
    kw = dict(order_n=4, leaf_size=N0, theta=theta, stop_at_n0=stop)
    p0 = oracle.Plan(*w.arrays(), q=w.q, **kw)
    rng = np.random.default_rng(12)
    etas, errs = [], []
    for sigma in (1e-6, 3e-5, 3e-4):                # drift as a fraction of sigma_x = 1 mm: 0.1 %, 3 %, 30 %
        x, y, z = (a + rng.normal(0.0, sigma * (0.1 if k == 2 else 1.0), N) for k, a in enumerate((w.x, w.y, w.z)))
        kept = oracle.Plan(x, y, z, w.px, w.py, w.pz, q=w.q, given_order=p0.perm(), **kw)
        fresh_lists = kept.lists()
        fresh_err = oracle.err2(kept.eval()[0], oracle.direct(x, y, z, w.px, w.py, w.pz, w.q, gamma_bar_value=kept.gamma_bar)[0])
        kept.set_lists(*p0.lists())
        # coverage: every ordered pair of non-empty leaves exactly once (P10), whatever the boxes are now
        lo, hi, _ = kept.node_arrays()
        flags = kept.leaf_flags()
        live = [int(i) for i in kept.leaf_ids() if hi[i - 1] > lo[i - 1]]
        pos = {i: k for k, i in enumerate(live)}

        def below(i):
            if flags[i - 1] == 1:
                return [pos[i]] if i in pos else []
            return below(2 * i) + below(2 * i + 1)

        count = np.zeros((len(live), len(live)), dtype=np.int64)
        p2p, m2l = kept.lists()
        for t, s in p2p:
            count[pos[int(t)], pos[int(s)]] += 1
        for t, s in m2l:
            count[np.ix_(below(int(t)), below(int(s)))] += 1
        assert (count == 1).all()
        E, B = kept.eval()
        Ed, Bd = oracle.direct(x, y, z, w.px, w.py, w.pz, w.q, gamma_bar_value=kept.gamma_bar)
        etas.append(kept.eta_eff())
        errs.append(oracle.err2(E, Ed) / fresh_err)
        assert kept.eta_eff() == eta_restated(kept)
        assert (len(fresh_lists[1]) != len(m2l)) or sigma < 1e-5
    assert etas[0] < etas[1] < etas[2] and etas[0] < 1.02 * theta and etas[2] > 1.2 * theta, etas
    # a small drift keeps the accuracy of a fresh traversal; the loss grows with eta_eff, which is what the caller watches
    assert errs[0] < 1.5 and errs[1] < 10.0 and errs[2] > errs[1], errs
