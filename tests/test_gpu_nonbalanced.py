"""GPU parity (-m gpu) of the non-balanced tree option FMM_TREE_STOP_AT_N0: Alg 5.2 as printed
 keeps a cluster of at most N0 particles as a leaf, so leaves sit on levels kappa-1 and kappa.
Same bars as tests/test_gpu_parity.py: tree order, node ranges, boxes and both lists bit-exact against the oracle
(ORC_TREE_STOP_AT_N0, pinned in tests/test_oracle_nonbalanced_pins.py), expansions and fields within 1e-12.
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


def measures(f, fref):
    f, fref = np.asarray(f), np.asarray(fref)
    e2 = np.sqrt(np.sum((f - fref) ** 2) / np.sum(fref ** 2))
    d = np.linalg.norm(f - fref, axis=1).max() / np.linalg.norm(fref, axis=1).max()
    return float(e2), float(d)


def assert_close(f, fref, what, tol=TOL):
    e2, d = measures(f, fref)
    assert e2 <= tol and d <= tol, f"{what}: err2={e2:.3e} max={d:.3e} > {tol}"


def to_np(EB):
    E, B = EB
    return E.cpu().numpy().T.copy(), B.cpu().numpy().T.copy()


# (label, config, N, n, N0, theta): floor(N / 2^(kappa-1)) == N0 in all but the last two
CASES = [
    ("early_63_of_64", 1, 4097, 4, 64, 0.5),          # 63 leaves of 64 on level 6, two leaves on level 7
    ("half_early", 2, 20000, 5, 78, 0.5),             # 20000 / 256 = 78.1: 224 leaves of 78 on level 8, 64 of 39/40 on level 9
    ("ragged_37", 3, 300, 3, 37, 0.4),
    ("gamma100", 4, 9217, 6, 72, 0.4),                # strongly stretched boxes; 9217 / 128 = 72.008
    ("three_particles", 1, 3, 2, 1, 0.5),             # leaf 3 on level 1, leaves 4 and 5 on level 2
    ("big_leaves_level_kernels", 2, 16402, 3, 4100, 0.5),   # nodes of level kappa-1 exceed KD_LOCAL: kd_mark / kd_split take the last level
    ("mutual_w4", 2, 40970, 4, 640, 0.5),             # 640-particle leaves beside 320 / 321
    ("no_early_power_of_two", 1, 4096, 4, 64, 0.5),   # the flag changes nothing (G13)
    ("no_early_ragged", 2, 5003, 3, 37, 0.5),
]
IDS = [c[0] for c in CASES]


def make(case):
    _, cfg, N, n, N0, theta = case
    return workloads.config(cfg, N=N), n, N0, theta


@pytest.mark.parametrize("mode", ["kd", "morton"])
@pytest.mark.parametrize("case", CASES, ids=IDS)
def test_tree_and_lists_bit_exact(fmm, case, mode):
    w, n, N0, theta = make(case)
    flags = (fmm.FMM_TREE_KD if mode == "kd" else fmm.FMM_TREE_MORTON_MEDIAN) | fmm.FMM_TREE_STOP_AT_N0
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta, flags=flags)
    st = plan.stats()
    ex = plan.export()
    op = oracle.Plan(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta, gamma_bar_value=st["gamma_bar"],
                     tree_mode=oracle.TREE_KD if mode == "kd" else oracle.TREE_MORTON_MEDIAN, stop_at_n0=True)
    assert (st["kappa"], st["nodes"], st["leaves"], st["P"]) == (op.kappa, op.nodes, op.leaves, op.P)
    n_early = int((op.leaf_ids() < op.leaves).sum()) if op.kappa > 0 else 0
    assert st["early_leaves"] == n_early
    assert (n_early > 0) == (not case[0].startswith("no_early"))
    assert np.array_equal(ex["perm"], op.perm()), "permutation differs"
    lo, hi, bb = op.node_arrays()
    assert np.array_equal(ex["node_lo"], lo) and np.array_equal(ex["node_hi"], hi)
    assert np.array_equal(ex["bbox"].view(np.uint64), bb.view(np.uint64)), "bounding boxes differ"
    p2p, m2l = op.lists()
    assert st["n_p2p"] == len(p2p) and st["n_m2l"] == len(m2l)
    for name, ref in (("p2p", p2p), ("m2l", m2l)):
        off, src = ex[name + "_off"], ex[name + "_src"]
        tgt = np.repeat(np.arange(1, st["nodes"] + 1, dtype=np.int32), np.diff(off))
        assert off[0] == 0 and off[-1] == len(ref)
        assert np.array_equal(tgt, ref[:, 0]) and np.array_equal(src, ref[:, 1]), f"{name} list differs"
    plan.close()


@pytest.mark.parametrize("mode", ["kd", "morton"])
@pytest.mark.parametrize("case", CASES[:7], ids=IDS[:7])
def test_fields_and_expansions(fmm, case, mode):
    w, n, N0, theta = make(case)
    flags = (fmm.FMM_TREE_KD if mode == "kd" else fmm.FMM_TREE_MORTON_MEDIAN) | fmm.FMM_TREE_STOP_AT_N0
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta, flags=flags)
    st = plan.stats()
    E, B = to_np(plan.eval())
    E2, B2 = to_np(plan.eval())
    assert np.array_equal(E, E2) and np.array_equal(B, B2)
    ex = plan.export(want_M=True, want_L=True)
    op = oracle.Plan(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta, gamma_bar_value=st["gamma_bar"],
                     tree_mode=oracle.TREE_KD if mode == "kd" else oracle.TREE_MORTON_MEDIAN, stop_at_n0=True)
    Eo, Bo, Lo = op.eval(want_L=True)
    Mo = op.upward()
    assert_close(E, Eo, "FMM E")
    assert_close(B, Bo, "FMM B")
    scale = np.abs(Mo).max()
    assert np.abs(ex["M"] - Mo).max() <= TOL * scale, "multipole moments differ (unused slots must be zero)"
    if st["n_m2l"] > 0:
        lo, hi, _ = op.node_arrays()
        live = hi > lo
        for f in (slice(0, 3), slice(3, 6)):
            scale = np.abs(Lo[live][..., f]).max()
            assert np.abs(ex["L"][live][..., f] - Lo[live][..., f]).max() <= TOL * scale, "local fields differ"
        assert not ex["L"][op.leaf_flags() == 2].any()
    plan.close()


def test_refit_update_and_host_entry(fmm):
    w = workloads.config(2, N=20000)
    kw = dict(order_n=4, leaf_size=78, theta=0.5)
    flags = fmm.FMM_TREE_STOP_AT_N0
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, flags=flags, **kw)
    perm0 = plan.export()["perm"].copy()
    rng = np.random.default_rng(5)
    x2, y2, z2 = (a + rng.normal(0, 2e-5, w.N) for a in (w.x, w.y, w.z))
    plan.refit(x2, y2, z2, w.px, w.py, w.pz, w.q)
    st = plan.stats()
    E, B = to_np(plan.eval())
    op = oracle.Plan(x2, y2, z2, w.px, w.py, w.pz, w.q, gamma_bar_value=st["gamma_bar"], given_order=perm0, stop_at_n0=True, **kw)
    ex = plan.export()
    p2p, m2l = op.lists()
    assert np.array_equal(ex["p2p_src"], p2p[:, 1]) and np.array_equal(ex["m2l_src"], m2l[:, 1])
    Eo, Bo = op.eval()
    assert_close(E, Eo, "refit E")
    assert_close(B, Bo, "refit B")
    plan.update(x2, y2, z2, w.px, w.py, w.pz, w.q)
    st = plan.stats()
    E, B = to_np(plan.eval())
    op = oracle.Plan(x2, y2, z2, w.px, w.py, w.pz, w.q, gamma_bar_value=st["gamma_bar"], stop_at_n0=True, **kw)
    Eo, Bo = op.eval()
    assert_close(E, Eo, "update E")
    assert_close(B, Bo, "update B")
    plan.close()
    E, B, st = fmm.fmm_field_host(*w.arrays(), w.q, flags=flags, **kw)
    op = oracle.Plan(*w.arrays(), w.q, gamma_bar_value=st["gamma_bar"], stop_at_n0=True, **kw)
    Eo, Bo = op.eval()
    assert_close(E.numpy().T, Eo, "host entry E")
    assert_close(B.numpy().T, Bo, "host entry B")


def test_source_momentum_and_treecode(fmm):
    w = workloads.config(1, N=4097)
    kw = dict(order_n=4, leaf_size=64, theta=0.5)
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, flags=fmm.FMM_TREE_STOP_AT_N0 | fmm.FMM_KERNEL_SOURCE_MOMENTUM, **kw)
    st = plan.stats()
    E, B = to_np(plan.eval())
    op = oracle.Plan(*w.arrays(), w.q, gamma_bar_value=st["gamma_bar"], stop_at_n0=True, source_momentum=True, **kw)
    Eo, Bo = op.eval()
    assert_close(E, Eo, "source-momentum E")
    assert_close(B, Bo, "source-momentum B")
    plan.close()
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, flags=fmm.FMM_TREE_STOP_AT_N0 | fmm.FMM_METHOD_TREECODE, **kw)
    st = plan.stats()
    ex = plan.export()
    op = oracle.Plan(*w.arrays(), w.q, gamma_bar_value=st["gamma_bar"], stop_at_n0=True, **kw)
    pp, pc = op.treecode_lists()
    for name, ref in (("p2p", pp), ("m2l", pc)):
        off, src = ex[name + "_off"], ex[name + "_src"]
        tgt = np.repeat(np.arange(1, st["nodes"] + 1, dtype=np.int32), np.diff(off))
        assert np.array_equal(tgt, ref[:, 0]) and np.array_equal(src, ref[:, 1]), f"treecode {name} list differs"
    E, B = to_np(plan.eval())
    Eo, Bo = op.eval_treecode()
    assert_close(E, Eo, "treecode E")
    assert_close(B, Bo, "treecode B")
    plan.close()
