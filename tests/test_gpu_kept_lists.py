"""GPU parity (-m gpu) of fmm_plan_refit_keep_lists (plan reuse with the lists kept while the
particles move a little).  The oracle builds the same tree over the kept particle order on the moved particles, is
handed the lists of the first traversal (orc_plan_set_lists, pinned in tests/test_oracle_kept_lists_pins.py) and
evaluates Alg 5.12 over them; the GPU must give the same boxes bit for bit, the same lists, fields and expansions
within 1e-12, and the same eta_eff (the admissibility ratio of the kept far pairs) to rounding of the square root.
"""
import numpy as np
import pytest

import oracle
from paper_2302_07567_b200 import workloads

pytestmark = pytest.mark.gpu

TOL = 1e-12


@pytest.fixture(scope="module")
def fmm():
    from paper_2302_07567_b200 import binding, build
    build.build_library()
    binding.load_library()
    return binding


def assert_close(f, fref, what, tol=TOL):
    f, fref = np.asarray(f), np.asarray(fref)
    e2 = np.sqrt(np.sum((f - fref) ** 2) / np.sum(fref ** 2))
    d = np.linalg.norm(f - fref, axis=1).max() / np.linalg.norm(fref, axis=1).max()
    assert e2 <= tol and d <= tol, f"{what}: err2={e2:.3e} max={d:.3e} > {tol}"


def to_np(EB):
    E, B = EB
    return E.cpu().numpy().T.copy(), B.cpu().numpy().T.copy()


def pairs(ex, name, nodes):
    off, src = ex[name + "_off"], ex[name + "_src"]
    tgt = np.repeat(np.arange(1, nodes + 1, dtype=np.int32), np.diff(off))
    return np.stack([tgt, src], axis=1)


CASES = [  # (label, config, N, n, N0, theta, flags-name, drift as a fraction of the bunch size)
    ("config1_kd", 1, 4096, 4, 64, 0.5, "kd", 0.01),
    ("config2_ragged_morton", 2, 20011, 5, 128, 0.5, "morton", 0.003),
    ("nonbalanced", 1, 4097, 4, 64, 0.5, "stop", 0.01),
    ("gamma100", 4, 9000, 6, 256, 0.4, "kd", 0.02),
    ("big_drift", 3, 30000, 3, 100, 0.4, "kd", 0.2),
]


@pytest.mark.parametrize("case", CASES, ids=[c[0] for c in CASES])
def test_refit_keep_lists_matches_oracle(fmm, case):
    _, cfg, N, n, N0, theta, mode, drift = case
    w = workloads.config(cfg, N=N)
    flags = {"kd": fmm.FMM_TREE_KD, "morton": fmm.FMM_TREE_MORTON_MEDIAN, "stop": fmm.FMM_TREE_STOP_AT_N0}[mode]
    okw = dict(order_n=n, leaf_size=N0, theta=theta, stop_at_n0=(mode == "stop"))
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta, flags=flags)
    st0 = plan.stats()
    ex0 = plan.export()
    lists0 = (pairs(ex0, "p2p", st0["nodes"]), pairs(ex0, "m2l", st0["nodes"]))
    rng = np.random.default_rng(21)
    x, y, z = (a + rng.normal(0.0, drift * a.std(), N) for a in (w.x, w.y, w.z))
    px, py, pz = (a * (1.0 + rng.normal(0.0, 1e-3, N)) for a in (w.px, w.py, w.pz))
    for rep in range(2):                              # twice: a kept plan can be refitted again
        eta = plan.refit_keep_lists(x, y, z, px, py, pz, w.q)
        st = plan.stats()
        assert (st["n_p2p"], st["n_m2l"]) == (st0["n_p2p"], st0["n_m2l"])
        E, B = to_np(plan.eval())
        ex = plan.export(want_M=True, want_L=True)
        op = oracle.Plan(x, y, z, px, py, pz, w.q, gamma_bar_value=st["gamma_bar"], given_order=ex0["perm"], **okw)
        assert abs(st["gamma_bar"] - oracle.gamma_bar(px, py, pz)) <= 1e-13 * st["gamma_bar"]
        lo, hi, bb = op.node_arrays()
        assert np.array_equal(ex["perm"], ex0["perm"]) and np.array_equal(ex["node_lo"], lo) and np.array_equal(ex["node_hi"], hi)
        assert np.array_equal(ex["bbox"].view(np.uint64), bb.view(np.uint64)), "bounding boxes differ"
        fresh = op.lists()
        op.set_lists(*lists0)
        for name, ref in (("p2p", lists0[0]), ("m2l", lists0[1])):
            assert np.array_equal(pairs(ex, name, st["nodes"]), ref), f"kept {name} list changed"
        eta_o = op.eta_eff()
        assert abs(eta - eta_o) <= 4e-16 * eta_o, (eta, eta_o)
        if drift >= 0.2:                              # boxes moved a lot: kept far pairs violate eq. (4.3), and the caller is told
            assert eta > theta and len(fresh[1]) != len(lists0[1])
        Eo, Bo, Lo = op.eval(want_L=True)
        Mo = op.upward()
        assert_close(E, Eo, "kept-lists E")
        assert_close(B, Bo, "kept-lists B")
        live = hi > lo
        assert np.abs(ex["M"][live] - Mo[live]).max() <= TOL * np.abs(Mo).max()
        for f in (slice(0, 3), slice(3, 6)):
            scale = np.abs(Lo[live][..., f]).max()
            assert np.abs(ex["L"][live][..., f] - Lo[live][..., f]).max() <= TOL * scale
        x = x + rng.normal(0.0, 0.2 * drift * w.x.std(), N)
    # a full refit afterwards rebuilds the lists on the moved boxes, and eta_eff is below theta again
    plan.refit(x, y, z, px, py, pz, w.q)
    st = plan.stats()
    op = oracle.Plan(x, y, z, px, py, pz, w.q, gamma_bar_value=st["gamma_bar"], given_order=ex0["perm"], **okw)
    ex = plan.export()
    for name, ref in zip(("p2p", "m2l"), op.lists()):
        assert np.array_equal(pairs(ex, name, st["nodes"]), ref)
    assert plan.refit_keep_lists(x, y, z, px, py, pz, w.q) < theta
    E, B = to_np(plan.eval())
    Eo, Bo = op.eval()
    assert_close(E, Eo, "refit E")
    plan.close()


def test_keep_lists_refusals(fmm):
    w = workloads.config(1, N=3000)
    kw = dict(order_n=2, leaf_size=40, theta=0.5)
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, flags=fmm.FMM_METHOD_TREECODE, **kw)
    with pytest.raises(fmm.FmmError, match="-1"):
        plan.refit_keep_lists(*w.arrays(), w.q)
    plan.close()
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, **kw)
    E0, B0 = to_np(plan.eval())
    bad = w.x.copy()
    bad[7] = np.nan
    with pytest.raises(fmm.FmmError, match="-4"):
        plan.refit_keep_lists(bad, w.y, w.z, w.px, w.py, w.pz, w.q)
    with pytest.raises(fmm.FmmError, match="-1"):      # an invalid plan has no lists to keep
        plan.refit_keep_lists(*w.arrays(), w.q)
    plan.update(*w.arrays(), w.q)
    assert plan.refit_keep_lists(*w.arrays(), w.q) < 0.5
    E1, B1 = to_np(plan.eval())
    assert np.array_equal(E0, E1) and np.array_equal(B0, B1)   # same particles, same lists: the same result bit for bit
    plan.close()


def test_time_stepping_policy_keeps_the_accuracy_of_a_fresh_plan(fmm):
    """The loop of README.md: lists built with a margin (theta = 0.42), kept while eta_eff <= 0.5 (the eta whose accuracy is
    accepted), rebuilt otherwise.  After every step the error against the all-pairs sum of the moved particles must stay at
    the level of a plan freshly built with theta = 0.5 on those particles, and the policy must have used both branches."""
    w = workloads.config(2, N=20000)
    build_theta, accept, kw = 0.42, 0.5, dict(order_n=5, leaf_size=100)
    rng = np.random.default_rng(33)
    x, y, z = w.x.copy(), w.y.copy(), w.z.copy()
    vel = [rng.normal(0.0, 0.01 * a.std(), w.N) for a in (x, y, z)]       # a steady drift of 1 % of the bunch size per step
    plan = fmm.fmm_plan_create(x, y, z, w.px, w.py, w.pz, w.q, theta=build_theta, **kw)
    kept = rebuilt = 0
    for step in range(10):
        x, y, z = x + vel[0], y + vel[1], z + vel[2]
        eta = plan.refit_keep_lists(x, y, z, w.px, w.py, w.pz, w.q)
        if eta > accept:
            plan.refit(x, y, z, w.px, w.py, w.pz, w.q)
            rebuilt += 1
        else:
            kept += 1
        E, B = to_np(plan.eval())
        gb = plan.stats()["gamma_bar"]
        Ed, Bd = to_np(fmm.fmm_direct(x, y, z, w.px, w.py, w.pz, w.q, gamma_bar=gb))
        fresh = fmm.fmm_plan_create(x, y, z, w.px, w.py, w.pz, w.q, theta=accept, gamma_bar=gb, **kw)
        Ef, Bf = to_np(fresh.eval())
        fresh.close()
        assert oracle.err2(E, Ed) <= 1.5 * oracle.err2(Ef, Ed), (step, eta, oracle.err2(E, Ed), oracle.err2(Ef, Ed))
        assert oracle.err2(B, Bd) <= 1.5 * oracle.err2(Bf, Bd), (step, eta)
    assert kept >= 2 and rebuilt >= 1, (kept, rebuilt)
    plan.close()
