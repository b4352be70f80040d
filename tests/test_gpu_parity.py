"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI (binding -> libfmm_b200.so),
against the CPU oracle on the same seeded inputs.

Bars:
  * tree permutation, node ranges, bounding boxes, both CSR lists: bit-exact;
  * fields (and M, L expansions): err2 (eq. (6.1)) <= 1e-12 and
    max_i |f_i - fref_i| / max_i |fref_i| <= 1e-12, for E and for B;
  * FMM-vs-direct error of the GPU equals the oracle's to 3 significant digits.
The oracle is given the plan's gamma_bar (reading D-5) so that both sides share every bit of it.
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
    """(err2 of eq. (6.1), max-norm relative error); f, fref are [N,3]."""
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


def small_cases():
    """(label, workload, n, N0, theta): several tiles, ragged tails, degenerate trees."""
    c1 = workloads.config(1)
    yield "config1", c1, 4, 64, 0.5
    w = workloads.config(2, N=20011)          # ragged: leaf sizes 78 / 79
    yield "config2_ragged", w, 5, 128, 0.5
    w = workloads.config(3, N=30000)
    yield "config3_small_n3", w, 3, 100, 0.4
    w = workloads.config(4, N=9000)           # gamma = 100: strongly stretched boxes
    yield "config4_small", w, 6, 256, 0.4
    w = workloads.paper_cube(N=6000, order_n=2)  # identical momenta, N0 = 27
    yield "paper_cube_n2", w, 2, 27, 0.5
    w = workloads.config(2, N=3000)           # n = 8: P = 729, M2L threads = 736 (one block per SM)
    yield "order8", w, 8, 200, 0.5
    w = workloads.config(2, N=2000)           # n = 9: P = 1000 = two batches of 500 (1024 threads would leave no room for the producer warp)
    yield "order9", w, 9, 150, 0.5
    w = workloads.config(3, N=2500)           # n = 10: P = 1331 > 1024 -> two proxy batches per target node, 2 pipeline stages
    yield "order10_batches", w, 10, 300, 0.5
    w = workloads.config(1, N=1500)           # n = 12 (FMM_MAX_ORDER): P = 2197, three batches, single-stage pipeline
    yield "order12_max", w, 12, 200, 0.45
    w = workloads.config(1, N=50)             # N <= N0: the root is a leaf (G23)
    yield "single_leaf", w, 4, 64, 0.5
    w = workloads.config(1, N=3)              # N0 = 1: an empty leaf appears
    yield "three_particles", w, 2, 1, 0.5
    w = workloads.config(1, N=1)
    yield "one_particle", w, 2, 8, 0.5


CASES = list(small_cases())
IDS = [c[0] for c in CASES]


# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,targets", [(4096, None), (5003, 777), (1, None), (300, None)])
def test_direct_matches_oracle(fmm, N, targets):
    w = workloads.config(1, N=N)
    gb = oracle.gamma_bar(w.px, w.py, w.pz)
    tidx = None
    if targets:
        tidx = np.random.default_rng(5).choice(N, size=targets, replace=False).astype(np.int64)
    E, B = to_np(fmm.fmm_direct(*w.arrays(), w.q, gamma_bar=gb, targets=tidx))
    Eo, Bo = oracle.direct(*w.arrays(), w.q, gamma_bar_value=gb, targets=tidx)
    if N == 1:
        assert np.all(E == 0) and np.all(B == 0) and np.all(Eo == 0)
        return
    assert_close(E, Eo, "direct E")
    assert_close(B, Bo, "direct B")


def test_direct_own_gamma_bar_and_charges(fmm):
    w = workloads.config(2, N=3000)
    q = np.random.default_rng(11).uniform(0.5, 2.0, w.N) * workloads.ELECTRON_CHARGE
    E, B = to_np(fmm.fmm_direct(*w.arrays(), q))          # gamma_bar computed on the device
    Eo, Bo = oracle.direct(*w.arrays(), q)                # and by the oracle (serial sum)
    assert_close(E, Eo, "direct E (own gamma_bar, per-particle q)", 1e-11)
    assert_close(B, Bo, "direct B (own gamma_bar, per-particle q)", 1e-11)


# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("mode", ["kd", "morton"])
@pytest.mark.parametrize("case", CASES, ids=IDS)
def test_tree_and_lists_bit_exact(fmm, case, mode):
    _, w, n, N0, theta = case
    flags = fmm.FMM_TREE_KD if mode == "kd" else fmm.FMM_TREE_MORTON_MEDIAN
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta, flags=flags)
    st = plan.stats()
    ex = plan.export()
    op = oracle.Plan(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta, gamma_bar_value=st["gamma_bar"],
                     tree_mode=oracle.TREE_KD if mode == "kd" else oracle.TREE_MORTON_MEDIAN)
    assert (st["kappa"], st["nodes"], st["leaves"], st["P"]) == (op.kappa, op.nodes, op.leaves, op.P)
    assert abs(st["gamma_bar"] - oracle.gamma_bar(w.px, w.py, w.pz)) <= 1e-13 * st["gamma_bar"]
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
@pytest.mark.parametrize("case", CASES, ids=IDS)
def test_fmm_fields_match_serial_oracle(fmm, case, mode):
    _, w, n, N0, theta = case
    flags = fmm.FMM_TREE_KD if mode == "kd" else fmm.FMM_TREE_MORTON_MEDIAN
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta, flags=flags)
    st = plan.stats()
    E, B = to_np(plan.eval())
    ex = plan.export(want_M=True, want_L=True)
    op = oracle.Plan(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta, gamma_bar_value=st["gamma_bar"],
                     tree_mode=oracle.TREE_KD if mode == "kd" else oracle.TREE_MORTON_MEDIAN)
    Eo, Bo, Lo = op.eval(want_L=True)
    Mo = op.upward()
    if w.N == 1:
        assert np.all(E == 0) and np.all(B == 0)
        return
    assert_close(E, Eo, "FMM E")
    assert_close(B, Bo, "FMM B")
    lo, hi, _ = op.node_arrays()
    live = hi > lo
    scale = np.abs(Mo).max()
    assert np.abs(ex["M"][live] - Mo[live]).max() <= TOL * scale, "multipole moments differ"
    if st["n_m2l"] > 0:
        for f in (slice(0, 3), slice(3, 6)):
            scale = np.abs(Lo[live][..., f]).max()
            assert np.abs(ex["L"][live][..., f] - Lo[live][..., f]).max() <= TOL * scale, "local fields differ"
    # FMM-vs-direct error: the GPU's equals the oracle's to 3 significant digits
    Ed, Bd = oracle.direct(*w.arrays(), w.q, gamma_bar_value=st["gamma_bar"])
    if st["n_m2l"] > 0:
        for f, fo, fd in ((E, Eo, Ed), (B, Bo, Bd)):
            a, b = oracle.err2(f, fd), oracle.err2(fo, fd)
            assert abs(a - b) <= 5e-3 * b + 1e-13
    else:  # pin P9: empty far list => FMM == direct
        assert_close(E, Ed, "FMM(no far field) vs direct E", 1e-11)
    plan.close()


def test_raw_sums_and_charges(fmm):
    w = workloads.config(1, N=3000)
    q = np.random.default_rng(3).uniform(-2.0, 2.0, w.N)
    plan = fmm.fmm_plan_create(*w.arrays(), q, order_n=3, leaf_size=50, theta=0.5, flags=fmm.FMM_RAW_SUMS)
    st = plan.stats()
    E, B = to_np(plan.eval())
    op = oracle.Plan(*w.arrays(), q, order_n=3, leaf_size=50, theta=0.5, gamma_bar_value=st["gamma_bar"], raw=True)
    Eo, Bo = op.eval()
    assert_close(E, Eo, "raw E")
    assert_close(B, Bo, "raw B")
    plan.close()


def test_deterministic_and_update(fmm):
    w = workloads.config(2, N=12000)
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=4, leaf_size=64, theta=0.5)
    E1, B1 = to_np(plan.eval())
    E2, B2 = to_np(plan.eval())
    assert np.array_equal(E1, E2) and np.array_equal(B1, B2), "not bit-reproducible run to run"
    w2 = workloads.gaussian_bunch(12000, 20.0, 0.01, 77, order_n=4, leaf_size=64, theta=0.5)
    plan.update(*w2.arrays(), w2.q)
    st = plan.stats()
    E3, B3 = to_np(plan.eval())
    op = oracle.Plan(*w2.arrays(), w2.q, order_n=4, leaf_size=64, theta=0.5, gamma_bar_value=st["gamma_bar"])
    Eo, Bo = op.eval()
    assert_close(E3, Eo, "updated plan E")
    assert_close(B3, Bo, "updated plan B")
    plan.close()


def test_field_host_entry(fmm):
    w = workloads.config(1)
    E, B, st = fmm.fmm_field_host(*w.arrays(), w.q, order_n=w.order_n, leaf_size=w.leaf_size, theta=w.theta)
    op = oracle.Plan(*w.arrays(), w.q, order_n=w.order_n, leaf_size=w.leaf_size, theta=w.theta,
                     gamma_bar_value=st["gamma_bar"])
    Eo, Bo = op.eval()
    assert_close(E.numpy().T, Eo, "host entry E")
    assert_close(B.numpy().T, Bo, "host entry B")


def test_bad_arguments(fmm):
    w = workloads.config(1, N=100)
    for kw in (dict(order_n=0, leaf_size=8, theta=0.5), dict(order_n=13, leaf_size=8, theta=0.5),
               dict(order_n=2, leaf_size=0, theta=0.5), dict(order_n=2, leaf_size=8, theta=0.0),
               dict(order_n=2, leaf_size=8, theta=float("nan"))):
        with pytest.raises(fmm.FmmError):
            fmm.fmm_plan_create(*w.arrays(), w.q, **kw)
    bad = w.pz.copy()
    bad[3] = np.nan
    with pytest.raises(fmm.FmmError):
        fmm.fmm_plan_create(w.x, w.y, w.z, w.px, w.py, bad, w.q, order_n=2, leaf_size=8, theta=0.5)


def test_non_finite_inputs_are_refused(fmm):
    """FMM_ENONFINITE (include/fmm.h): one fused scan in step a0 finds NaN / Inf in x, y, z, px, py, pz or q, also when
    gamma_bar is given; a plan whose update failed refuses fmm_eval until an update succeeds."""
    w = workloads.config(1, N=5000)
    base = dict(order_n=2, leaf_size=40, theta=0.5)
    names = ["x", "y", "z", "px", "py", "pz"]
    for k, name in enumerate(names):
        for val in (np.nan, np.inf, -np.inf):
            arrs = [a.copy() for a in w.arrays()]
            arrs[k][(17 * k + 3) % w.N] = val
            for gb in (0.0, 10.0):
                with pytest.raises(fmm.FmmError, match="-4"):
                    fmm.fmm_plan_create(*arrs, w.q, gamma_bar=gb, **base)
    q = np.full(w.N, workloads.ELECTRON_CHARGE)
    q[-1] = np.nan
    with pytest.raises(fmm.FmmError, match="-4"):
        fmm.fmm_plan_create(*w.arrays(), q, **base)
    # a failed update invalidates the plan, a good one revives it
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, **base)
    E0, B0 = to_np(plan.eval())
    arrs = [a.copy() for a in w.arrays()]
    arrs[0][5] = np.inf
    with pytest.raises(fmm.FmmError, match="-4"):
        plan.update(*arrs, w.q)
    with pytest.raises(fmm.FmmError, match="-1"):
        plan.eval()
    plan.update(*w.arrays(), w.q)
    E1, B1 = to_np(plan.eval())
    assert np.array_equal(E0, E1) and np.array_equal(B0, B1)
    plan.close()


# ---------------------------------------------------------------------------------------------
# FMM_KERNEL_SOURCE_MOMENTUM: near field stretched along each source's own momentum (G6 alternative,
# SURVEY.md 8(f) rank 2).  Same bars as the default kernel.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,targets", [(4096, None), (3001, 500)])
def test_direct_source_momentum_matches_oracle(fmm, N, targets):
    w = workloads.config(4, N=N)                      # gamma = 100, 2 % spread: the two readings differ most here
    tg = None if targets is None else np.sort(np.random.default_rng(5).choice(N, targets, replace=False)).astype(np.int64)
    E, B = to_np(fmm.fmm_direct(*w.arrays(), w.q, flags=fmm.FMM_KERNEL_SOURCE_MOMENTUM, targets=tg))
    Eo, Bo = oracle.direct(*w.arrays(), w.q, source_momentum=True, targets=tg)
    assert_close(E, Eo, "direct E (source momentum)")
    assert_close(B, Bo, "direct B (source momentum)")
    Em, _ = oracle.direct(*w.arrays(), w.q, targets=tg)
    assert oracle.err2(Eo, Em) > 1e-4                 # ... and it is a different kernel


@pytest.mark.parametrize("case", [c for c in CASES if c[0] in ("config1", "config2_ragged", "config4_small", "paper_cube_n2",
                                                              "single_leaf")], ids=lambda c: c[0])
def test_fmm_source_momentum_matches_serial_oracle(fmm, case):
    _, w, n, N0, theta = case
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta,
                               flags=fmm.FMM_TREE_KD | fmm.FMM_KERNEL_SOURCE_MOMENTUM)
    st = plan.stats()
    E, B = to_np(plan.eval())
    ex = plan.export()
    op = oracle.Plan(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta, gamma_bar_value=st["gamma_bar"],
                     source_momentum=True)
    p2p, m2l = op.lists()                              # the kernel mode does not touch tree or lists
    assert np.array_equal(ex["perm"], op.perm())
    assert np.array_equal(ex["p2p_src"], p2p[:, 1]) and np.array_equal(ex["m2l_src"], m2l[:, 1])
    Eo, Bo = op.eval()
    assert_close(E, Eo, "FMM E (source momentum)")
    assert_close(B, Bo, "FMM B (source momentum)")
    plan.close()


# ---------------------------------------------------------------------------------------------
# fmm_plan_refit: the particle order of the last build is kept
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("sm", [False, True], ids=["mean_gamma", "source_momentum"])
def test_refit_matches_oracle_over_the_same_order(fmm, sm):
    w = workloads.config(2, N=20011)
    flags = fmm.FMM_TREE_KD | (fmm.FMM_KERNEL_SOURCE_MOMENTUM if sm else 0)
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=4, leaf_size=128, theta=0.5, flags=flags)
    perm0 = plan.export()["perm"].copy()
    rng = np.random.default_rng(17)
    x2 = w.x + 3e-5 * rng.standard_normal(w.N)
    y2 = w.y + 3e-5 * rng.standard_normal(w.N)
    z2 = w.z + 3e-6 * rng.standard_normal(w.N)
    pz2 = w.pz * (1.0 + 1e-3 * rng.standard_normal(w.N))
    args = (x2, y2, z2, w.px, w.py, pz2)
    plan.refit(*args, w.q)
    st = plan.stats()
    ex = plan.export()
    assert np.array_equal(ex["perm"], perm0), "refit must keep the particle order"
    op = oracle.Plan(*args, w.q, order_n=4, leaf_size=128, theta=0.5, gamma_bar_value=st["gamma_bar"], given_order=perm0,
                     source_momentum=sm)
    assert abs(st["gamma_bar"] - oracle.gamma_bar(w.px, w.py, pz2)) <= 1e-13 * st["gamma_bar"]
    lo, hi, bb = op.node_arrays()
    assert np.array_equal(ex["bbox"].view(np.uint64), bb.view(np.uint64)), "bounding boxes differ"
    p2p, m2l = op.lists()
    assert np.array_equal(ex["p2p_src"], p2p[:, 1]) and np.array_equal(ex["m2l_src"], m2l[:, 1])
    E, B = to_np(plan.eval())
    Eo, Bo = op.eval()
    assert_close(E, Eo, "refit E")
    assert_close(B, Bo, "refit B")
    # a full update afterwards re-sorts: back to the KD tree of the new positions
    plan.update(*args, w.q)
    ok = oracle.Plan(*args, w.q, order_n=4, leaf_size=128, theta=0.5, gamma_bar_value=plan.stats()["gamma_bar"], source_momentum=sm)
    assert np.array_equal(plan.export()["perm"], ok.perm())
    plan.close()


def test_overlap_is_bit_identical_to_serial_and_stable(fmm):
    """fmm_plan_set_overlap: P2P on the plan's side stream beside P2M/M2M/M2L/L2L.  Regression for a cross-proxy
    write-after-read hazard in the M2L source ring (generic reads of a stage vs. the next bulk-TMA copy into it) that
    only showed with concurrent kernels: 25 evaluations in each mode must be bit-identical."""
    import torch
    # n = 3: two consumer warps + producer warp; n = 5 and n = 6: 7 / 11 consumer warps + the helper warp that also
    # refills the ring (anonymous `empty` arrivals: every warp must wait for a stage before releasing it)
    for cfg, N, n, N0, theta in ((3, 30000, 3, 100, 0.4), (2, 20000, 5, 128, 0.5), (3, 40000, 6, 256, 0.5)):
        w = workloads.config(cfg, N=N)
        plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta)
        plan.set_overlap(False)
        E0, B0 = plan.eval()
        E0, B0 = E0.clone(), B0.clone()
        for ov in (True, False, True):
            plan.set_overlap(ov)
            for _ in range(25):
                E, B = plan.eval()
                assert torch.equal(E, E0) and torch.equal(B, B0), f"n={n} overlap={ov}: result changed between evaluations"
        plan.close()


# ---------------------------------------------------------------------------------------------
# FMM_METHOD_TREECODE: particle-cluster variant (Fig. 1a)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("case", [c for c in CASES if c[0] in ("config1", "config2_ragged", "config3_small_n3", "config4_small",
                                                              "paper_cube_n2", "order8", "single_leaf", "three_particles")],
                         ids=lambda c: c[0])
def test_treecode_matches_oracle(fmm, case):
    _, w, n, N0, theta = case
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta,
                               flags=fmm.FMM_TREE_KD | fmm.FMM_METHOD_TREECODE)
    st = plan.stats()
    ex = plan.export()
    op = oracle.Plan(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=theta, gamma_bar_value=st["gamma_bar"])
    assert np.array_equal(ex["perm"], op.perm())
    pp, pc = op.treecode_lists()
    assert st["n_p2p"] == len(pp) and st["n_m2l"] == len(pc)
    for name, ref in (("p2p", pp), ("m2l", pc)):          # "m2l" slots carry the particle-cluster list in this mode
        off, src = ex[name + "_off"], ex[name + "_src"]
        tgt = np.repeat(np.arange(1, st["nodes"] + 1, dtype=np.int32), np.diff(off))
        assert np.array_equal(tgt, ref[:, 0]) and np.array_equal(src, ref[:, 1]), f"{name} list differs"
    E, B = to_np(plan.eval())
    Eo, Bo = op.eval_treecode()
    assert_close(E, Eo, "treecode E")
    assert_close(B, Bo, "treecode B")
    E2, B2 = to_np(plan.eval())
    assert np.array_equal(E, E2) and np.array_equal(B, B2)
    plan.close()


def test_treecode_cross_checks_the_fmm(fmm):
    """Two independently structured approximations of the same sum agree at the level of their error against it."""
    w = workloads.config(2, N=30000)
    kw = dict(order_n=6, leaf_size=128, theta=0.5)
    a = fmm.fmm_plan_create(*w.arrays(), w.q, **kw)
    b = fmm.fmm_plan_create(*w.arrays(), w.q, flags=fmm.FMM_METHOD_TREECODE, **kw)
    Ea, _ = to_np(a.eval())
    Eb, _ = to_np(b.eval())
    Ed, _ = to_np(fmm.fmm_direct(*w.arrays(), w.q, gamma_bar=a.stats()["gamma_bar"]))
    ea, eb = oracle.err2(Ea, Ed), oracle.err2(Eb, Ed)
    assert eb < 1.5 * ea and oracle.err2(Ea, Eb) < 2 * ea, (ea, eb)
    a.close(); b.close()


# ---------------------------------------------------------------------------------------------
# mutual near field: one block evaluates a pair of leaves for both directions; entries whose reverse pair is
# missing from the list (after a radius tie in Alg 5.11, reading D-3) must take the one-sided path
# ---------------------------------------------------------------------------------------------
def _mirrored_bunch(N_half, seed):
    rng = np.random.default_rng(seed)
    x = rng.uniform(0.01, 4.0, N_half)
    y = rng.uniform(-0.5, 0.5, N_half)
    z = rng.uniform(-0.05, 0.05, N_half)
    X = np.concatenate([x, -x]); Y = np.concatenate([y, y]); Z = np.concatenate([z, z])
    N = 2 * N_half
    px, py = 1e-2 * rng.standard_normal(N), 1e-2 * rng.standard_normal(N)
    pz = 3.0 * (1.0 + 0.05 * rng.standard_normal(N))
    q = rng.uniform(0.5, 2.0, N)
    return X, Y, Z, px, py, pz, q


@pytest.mark.parametrize("theta,seed,N_half,N0", [(0.5, 7, 512, 16), (0.3, 7, 1024, 8), (0.5, 3, 2048, 32), (0.5, 9, 1024, 8)])
def test_mutual_near_field_handles_one_sided_entries(fmm, theta, seed, N_half, N0):
    X, Y, Z, px, py, pz, q = _mirrored_bunch(N_half, seed)
    plan = fmm.fmm_plan_create(X, Y, Z, px, py, pz, q, order_n=3, leaf_size=N0, theta=theta, flags=fmm.FMM_RAW_SUMS)
    st = plan.stats()
    ex = plan.export()
    op = oracle.Plan(X, Y, Z, px, py, pz, q, order_n=3, leaf_size=N0, theta=theta, gamma_bar_value=st["gamma_bar"], raw=True)
    p2p, _ = op.lists()
    tgt = np.repeat(np.arange(1, st["nodes"] + 1, dtype=np.int32), np.diff(ex["p2p_off"]))
    assert np.array_equal(tgt, p2p[:, 0]) and np.array_equal(ex["p2p_src"], p2p[:, 1])
    pairs = set(map(tuple, p2p))
    mateless = sum((s, t) not in pairs for t, s in pairs)
    if (theta, seed) != (0.5, 9):
        assert mateless > 0, "this input is meant to contain entries without a reverse pair"
    E, B = to_np(plan.eval())
    Eo, Bo = op.eval()
    assert_close(E, Eo, f"mutual near field E ({mateless} one-sided entries)")
    assert_close(B, Bo, f"mutual near field B ({mateless} one-sided entries)")
    plan.close()


@pytest.mark.parametrize("N,N0,n", [(5000, 300, 2), (7001, 700, 2), (2500, 1000, 3), (1300, 1300, 2), (20000, 33, 2)])
def test_mutual_near_field_leaf_shapes(fmm, N, N0, n):
    """Leaves of 157 / 438 / 625 / 1300 (one leaf, more than 1024 particles: one-sided kernel) / 20 particles: every
    (targets per thread, warps per block) shape of the near-field kernels, ragged last tiles, many entries per tile."""
    w = workloads.config(2, N=N)
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=0.5)
    st = plan.stats()
    E, B = to_np(plan.eval())
    Eo, Bo = oracle.Plan(*w.arrays(), w.q, order_n=n, leaf_size=N0, theta=0.5, gamma_bar_value=st["gamma_bar"]).eval()
    assert_close(E, Eo, "E")
    assert_close(B, Bo, "B")
    plan.close()


def test_plan_on_one_stream_evaluated_under_another(fmm):
    """the library works on the stream given at fmm_plan_create and frees scratch right after enqueueing; the
    binding must therefore run every later call on that stream, whatever torch's current stream is."""
    import torch
    w = workloads.config(2, N=15000)
    dev = torch.device("cuda", 0)
    ref_plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=4, leaf_size=64, theta=0.5)
    Eref, Bref = to_np(ref_plan.eval())
    ref_plan.close()
    sa, sb = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    with torch.cuda.stream(sa):
        plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=4, leaf_size=64, theta=0.5)
    assert plan.stream == sa
    d_in = [torch.as_tensor(a).to(dev) for a in w.arrays()]
    junk = []
    with torch.cuda.stream(sb):
        for _ in range(3):
            plan.update(*d_in, w.q)
            junk.append(torch.full((1 << 22,), 7.0, device=dev))   # allocator pressure on stream B's pool
            E, B = plan.eval()
            E2 = E * 1.0                                          # consumer on stream B right after the call
        sb.synchronize()
    assert np.array_equal(E2.cpu().numpy().T, Eref)
    assert np.array_equal(to_np((E, B))[1], Bref)
    plan.close()


@pytest.mark.parametrize("kind", ["short_runs", "long_run", "all_equal_axis", "duplicates"])
def test_kd_sort_key_ties(fmm, kind):
    """The KD build sorts by a 32-bit quantisation of the coordinates and repairs runs of equal keys afterwards
    (kernels_kd.cu): runs of up to 64 entries in place, longer ones by a rebuild with exact keys.  The particle order must be
    the oracle's (coordinate, index) order in every case."""
    rng = np.random.default_rng(42)
    N = 6000
    y = rng.normal(0, 1e-3, N)
    z = rng.normal(0, 1e-4, N)
    if kind == "short_runs":      # 300 clusters of 20 points 1e-13 apart: 20 entries per sort key, out of order
        x = np.repeat(rng.uniform(-1, 1, 300), 20) + 1e-13 * rng.standard_normal(N)
    elif kind == "long_run":      # one tight cluster and two far outliers: thousands of entries per sort key
        x = 1e-9 * rng.random(N)
        x[7], x[4000] = -1e3, 1e3
    elif kind == "all_equal_axis":
        x = np.full(N, 0.25)
    else:                          # exact duplicates: ties go to the index
        x = np.repeat(rng.uniform(-1, 1, N // 4), 4)
        rng.shuffle(x)
    px, py, pz = np.zeros(N), np.zeros(N), np.full(N, 5.0)
    plan = fmm.fmm_plan_create(x, y, z, px, py, pz, 1.0, order_n=2, leaf_size=40, theta=0.5)
    st = plan.stats()
    ex = plan.export()
    op = oracle.Plan(x, y, z, px, py, pz, 1.0, order_n=2, leaf_size=40, theta=0.5, gamma_bar_value=st["gamma_bar"])
    assert np.array_equal(ex["perm"], op.perm()), "permutation differs"
    _, _, bb = op.node_arrays()
    assert np.array_equal(ex["bbox"].view(np.uint64), bb.view(np.uint64))
    E, B = to_np(plan.eval())
    Eo, Bo = op.eval()
    assert_close(E, Eo, "E")
    plan.close()


@pytest.mark.parametrize("N", [2048, 5003, 70001])
def test_direct_all_targets_mutual_form(fmm, N):
    """fmm_direct with all N targets evaluates every particle pair once for both directions (tiles of 256 in super-tiles,
    kernels_pairs.cu direct_mutual_kernel): ragged last tile, ragged last super-tile, first / diagonal / off-diagonal blocks.
    Compared with the oracle's direct sum on a seeded sample of targets."""
    w = workloads.config(4, N=N)
    q = np.random.default_rng(17).uniform(0.5, 2.0, N) * workloads.ELECTRON_CHARGE
    gb = oracle.gamma_bar(w.px, w.py, w.pz)
    E, B = to_np(fmm.fmm_direct(*w.arrays(), q, gamma_bar=gb))
    idx = np.sort(np.random.default_rng(18).choice(N, size=min(N, 1500), replace=False)).astype(np.int64)
    idx[:4] = [0, 255, 256, N - 1][: len(idx[:4])]
    Eo, Bo = oracle.direct(*w.arrays(), q, gamma_bar_value=gb, targets=idx)
    assert_close(E[idx], Eo, "direct (mutual form) E")
    assert_close(B[idx], Bo, "direct (mutual form) B")
    # and identical to the one-sided kernel (targets given explicitly) up to summation order
    E1, B1 = to_np(fmm.fmm_direct(*w.arrays(), q, gamma_bar=gb, targets=idx))
    assert_close(E[idx], E1, "mutual vs one-sided direct E")
    assert_close(B[idx], B1, "mutual vs one-sided direct B")


@pytest.mark.parametrize("shift,axis,tol", [(1.0, 2, 1e-12), (1.0, 0, 1e-12), (100.0, 2, 1e-10), (100.0, 0, 1e-10)])
def test_displaced_bunch(fmm, shift, axis, tol):
    """positions far from the origin (a lab-frame offset of metres for a millimetre bunch).  The fields depend on
    differences only, but the M2L z trick works with box-centre-relative proxy offsets whose rounding grows with |z0|
    (DESIGN.md section 9): 1e-12 holds for |offset| / extent up to about 1e3, at 1e5 the documented bound is 1e-10."""
    w = workloads.config(2, N=20000)
    pos = [w.x.copy(), w.y.copy(), w.z.copy()]
    pos[axis] += shift
    plan = fmm.fmm_plan_create(*pos, w.px, w.py, w.pz, w.q, order_n=5, leaf_size=128, theta=0.5)
    st = plan.stats()
    E, B = to_np(plan.eval())
    ex = plan.export()
    op = oracle.Plan(*pos, w.px, w.py, w.pz, w.q, order_n=5, leaf_size=128, theta=0.5, gamma_bar_value=st["gamma_bar"])
    assert np.array_equal(ex["perm"], op.perm())
    p2p, m2l = op.lists()
    assert np.array_equal(ex["p2p_src"], p2p[:, 1]) and np.array_equal(ex["m2l_src"], m2l[:, 1])
    Eo, Bo = op.eval()
    assert_close(E, Eo, f"E, bunch displaced by {shift} m along axis {axis}", tol)
    assert_close(B, Bo, f"B, bunch displaced by {shift} m along axis {axis}", tol)
    plan.close()


@pytest.mark.parametrize("n", [7, 11])
def test_orders_at_the_shared_memory_opt_in_boundary(fmm, n):
    """n = 7: the L2P kernel needs exactly 48 KB of dynamic shared memory beside 1 KB of static (the default limit counts
    both); n = 11 sits between the other cases of the order sweep."""
    w = workloads.config(3, N=4000)
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=n, leaf_size=256, theta=0.5)
    st = plan.stats()
    E, B = to_np(plan.eval())
    Eo, Bo = oracle.Plan(*w.arrays(), w.q, order_n=n, leaf_size=256, theta=0.5, gamma_bar_value=st["gamma_bar"]).eval()
    assert_close(E, Eo, "E")
    assert_close(B, Bo, "B")
    plan.close()


def test_one_sided_fallback_when_the_reaction_segments_do_not_fit(fmm, monkeypatch):
    """The mutual near field needs 48 bytes per particle of half the P2P list; if the allocator refuses that block the plan
    falls back to the one-sided kernel (same fields up to summation order) instead of failing."""
    w = workloads.config(2, N=20000)
    kw = dict(order_n=3, leaf_size=64, theta=0.5)
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, **kw)
    st = plan.stats()
    assert st["p2p_mutual"] == 1 and st["react_particles"] > 0
    E0, B0 = to_np(plan.eval())
    plan.close()
    refused = 48 * st["react_particles"]
    orig = fmm._TorchAllocator._alloc

    def picky(self, nbytes, user):
        return None if int(nbytes) == refused else orig(self, nbytes, user)

    monkeypatch.setattr(fmm._TorchAllocator, "_alloc", picky)
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, **kw)
    st1 = plan.stats()
    assert st1["p2p_mutual"] == 0 and st1["n_p2p"] == st["n_p2p"]
    E1, B1 = to_np(plan.eval())
    assert_close(E1, E0, "one-sided fallback E")
    assert_close(B1, B0, "one-sided fallback B")
    plan.close()


def test_traversal_spill_path(fmm, monkeypatch):
    """The warp walks of the traversal keep their pairs in a 512-entry stack and hand what does not fit to a second
    launch; with the stack shrunk to 64 entries (FMM_TEST_WALK_STACK) many walks spill and the lists must still be the oracle's."""
    monkeypatch.setenv("FMM_TEST_WALK_STACK", "64")
    w = workloads.config(2, N=60000)
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=2, leaf_size=8, theta=0.5)
    st = plan.stats()
    ex = plan.export()
    op = oracle.Plan(*w.arrays(), w.q, order_n=2, leaf_size=8, theta=0.5, gamma_bar_value=st["gamma_bar"])
    p2p, m2l = op.lists()
    assert st["n_p2p"] == len(p2p) and st["n_m2l"] == len(m2l)
    assert np.array_equal(ex["p2p_src"], p2p[:, 1]) and np.array_equal(ex["m2l_src"], m2l[:, 1])
    plan.close()


@pytest.mark.parametrize("N,N0,stop", [(20011, 128, False), (65536, 128, False), (9000, 7, False), (40970, 640, True), (5000, 300, False),
                                       (16402, 4100, True)])
def test_kd_order_with_li_rebuilt_by_the_leaf_blocks(fmm, monkeypatch, N, N0, stop):
    """From 2^19 particles on the level kernels of the KD build split three lists and kd_local rebuilds the index-ordered list
    of its node by sorting the member ids in shared memory; FMM_TEST_KD_SORT_LI takes that route on small bunches (ragged node
    sizes, nodes of 2,500 .. 4,096 particles, leaves of 7, the non-balanced option; the last case has leaves beyond KD_LOCAL and
    must keep all four lists).  The particle order must be the oracle's either way."""
    w = workloads.config(2, N=N)
    flags = fmm.FMM_TREE_STOP_AT_N0 if stop else 0
    ref = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=2, leaf_size=N0, theta=0.5, flags=flags)
    perm_ref = ref.export()["perm"]
    gb = ref.stats()["gamma_bar"]
    ref.close()
    monkeypatch.setenv("FMM_TEST_KD_SORT_LI", "1")
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=2, leaf_size=N0, theta=0.5, flags=flags)
    perm = plan.export()["perm"]
    plan.close()
    op = oracle.Plan(*w.arrays(), w.q, order_n=2, leaf_size=N0, theta=0.5, gamma_bar_value=gb, stop_at_n0=stop)
    assert np.array_equal(perm, op.perm()) and np.array_equal(perm_ref, perm)


@pytest.mark.parametrize("N,N0,cube", [(10000, 729, True), (40000, 729, True), (5003, 640, False), (200000, 900, True), (9000, 1000, False),
                                       (5008, 343, True),
                                       # leaves of 1025 .. 2048 particles: two target passes per block (1250, 2048, 1025 / 1026, 1563)
                                       (20000, 1331, True), (8192, 2048, False), (4101, 1100, False), (100000, 1600, True),
                                       # every warp's share ends in more than 15 particles: still the RAGGED kernels (700; 1400 in two passes)
                                       (11200, 700, False), (5600, 1400, True), (44800, 700, True)])
def test_ragged_leaves_in_the_mutual_near_field(fmm, N, N0, cube):
    """Leaves that leave whole warp-slots of an eight-warp near-field block empty (625 particles in 8 x 32 x 3 slots, 782 or 879
    in 8 x 32 x 4, ...): the warps with an empty last slot run the shorter loops and the slot assignment rotates with the block
    index (p2p_mutual_kernel, RAGGED); with and without the row split; (313 in 4 x 32 x 3) keeps the plain kernel; leaves of
    more than 1,024 particles are worked on in two passes whose reaction sums add up in the same segments.  Where every warp's
    equal share of the leaf ends in 1 .. 15 particles (313 = 4 x 79, 625 = 8 x 79, 782 = 8 x 98, ...) the half-rate last slot
    of test_half_rate_tail_slot_of_one_warp_leaves is used instead, with per-warp shares.
    Fields against the oracle, and the same bits from one evaluation to the next."""
    w = workloads.paper_cube(N=N, order_n=2) if cube else workloads.config(2, N=N)
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=2, leaf_size=N0, theta=0.5)
    st = plan.stats()
    assert st["p2p_mutual"] == 1
    E, B = to_np(plan.eval())
    E2, B2 = to_np(plan.eval())
    assert np.array_equal(E, E2) and np.array_equal(B, B2)
    op = oracle.Plan(*w.arrays(), w.q, order_n=2, leaf_size=N0, theta=0.5, gamma_bar_value=st["gamma_bar"])
    Eo, Bo = op.eval()
    assert_close(E, Eo, "ragged leaves E")
    assert_close(B, Bo, "ragged leaves B")
    plan.close()


@pytest.mark.parametrize("N,N0,cfg", [(5000, 40, 1), (10000, 110, 2), (13000, 110, 3), (20011, 128, 2), (80000, 125, 0), (4200, 47, 1), (1100, 79, 4)])
def test_half_rate_tail_slot_of_one_warp_leaves(fmm, N, N0, cfg):
    """One-warp leaves whose last target slot holds at most 15 particles (39 / 40 = 32 + 8, 78 / 79 = 64 + 15, 101 / 102 = 96 + 6,
    33 = 32 + 1, 69 = 64 + 5): the tail sits in two lanes of opposite parity and the slot is worked on at every second step of the
    rotation (p2p_mutual_kernel, HALF).  Fields against the oracle, the same bits from one evaluation to the next, and against the
    all-pairs sum when nothing is admissible (every pair of leaves then goes through the near field)."""
    w = workloads.paper_cube(N=N, order_n=3) if cfg == 0 else workloads.config(cfg, N=N)
    for theta in (0.5, 1e-3):
        plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=3, leaf_size=N0, theta=theta)
        st = plan.stats()
        assert st["p2p_mutual"] == 1
        E, B = to_np(plan.eval())
        E2, B2 = to_np(plan.eval())
        assert np.array_equal(E, E2) and np.array_equal(B, B2)
        if theta == 0.5:
            op = oracle.Plan(*w.arrays(), w.q, order_n=3, leaf_size=N0, theta=theta, gamma_bar_value=st["gamma_bar"])
            Eo, Bo = op.eval()
        elif N <= 20011:
            assert st["n_m2l"] == 0
            Eo, Bo = oracle.direct(*w.arrays(), w.q, gamma_bar_value=st["gamma_bar"])
        else:
            plan.close()
            continue
        assert_close(E, Eo, f"half-rate tail E (theta {theta})")
        assert_close(B, Bo, f"half-rate tail B (theta {theta})")
        plan.close()


@pytest.mark.parametrize("kind", ["coplanar_z", "coplanar_x", "collinear_z", "at_rest", "wide_theta", "gamma_1e4"])
def test_degenerate_geometry_and_momenta(fmm, kind):
    """Boxes with zero extent along one or two axes (their proxy points coincide there and every particle hits a node of the
    barycentric form exactly), a bunch at rest (gamma_bar = 1: B = 0), theta = 0.9 (large boxes still admissible) and
    gamma_bar = 1e4 (z extents stretched far beyond x and y): structures bit-exact, fields as everywhere else."""
    w = workloads.config(3, N=6000)
    theta = 0.5
    if kind == "coplanar_z":
        w.z[:] = 0.25
    elif kind == "coplanar_x":
        w.x[:] = -1.0
    elif kind == "collinear_z":
        w.x[:] = 0.0
        w.y[:] = 3.0
    elif kind == "at_rest":
        w.px[:] = 0.0; w.py[:] = 0.0; w.pz[:] = 0.0
    elif kind == "wide_theta":
        theta = 0.9
    elif kind == "gamma_1e4":
        w.pz[:] = w.pz * (1e4 / np.sqrt(1.0 + np.mean(w.pz) ** 2))
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=4, leaf_size=50, theta=theta)
    st, ex = plan.stats(), plan.export()
    E, B = to_np(plan.eval())
    op = oracle.Plan(*w.arrays(), w.q, order_n=4, leaf_size=50, theta=theta, gamma_bar_value=st["gamma_bar"])
    assert np.array_equal(ex["perm"], op.perm())
    p2p, m2l = op.lists()
    assert np.array_equal(ex["p2p_src"], p2p[:, 1]) and np.array_equal(ex["m2l_src"], m2l[:, 1])
    assert st["n_m2l"] > 0
    Eo, Bo = op.eval()
    assert np.isfinite(E).all() and np.isfinite(B).all()
    assert_close(E, Eo, "E " + kind)
    if kind == "at_rest":
        assert st["gamma_bar"] == 1.0 and np.all(B == 0.0) and np.all(Bo == 0.0)
    else:
        assert_close(B, Bo, "B " + kind)
    plan.close()
    op.close()


@pytest.mark.parametrize("method", ["fmm", "treecode"])
def test_upward_pass_of_the_build_and_stage_timers(fmm, method):
    """A build enqueues P2M + M2M itself, behind its one host wait, and fmm_eval reuses the moments:
    repeated evaluations, evaluations with the stage timers switched on or off in between (which makes fmm_eval run the
    upward pass again, between its own events) and an update under running timers all give the same bits, and the six
    stage times are there whenever the timers were on for the evaluation."""
    w = workloads.config(2, N=9000)
    flags = fmm.FMM_TREE_KD | (fmm.FMM_METHOD_TREECODE if method == "treecode" else 0)
    plan = fmm.fmm_plan_create(*w.arrays(), w.q, order_n=3, leaf_size=50, theta=0.5, flags=flags)
    E0, B0 = to_np(plan.eval())
    plan.set_timing(True)
    E1, B1 = to_np(plan.eval())
    st = plan.stats()
    assert st["timing_valid"] == 1 and st["ms_p2m"] > 0 and st["ms_m2m"] > 0 and st["ms_l2p"] > 0
    E2, B2 = to_np(plan.eval())      # moments of the evaluation before
    plan.update(*w.arrays(), w.q)    # same particles: the build runs the upward pass under the timers
    E3, B3 = to_np(plan.eval())
    st = plan.stats()
    assert st["timing_valid"] == 1 and st["ms_p2m"] > 0 and st["ms_m2m"] > 0 and st["ms_m2l"] > 0 and st["ms_p2p"] > 0
    plan.set_timing(False)
    E4, B4 = to_np(plan.eval())
    for E, B in ((E1, B1), (E2, B2), (E3, B3), (E4, B4)):
        assert np.array_equal(E, E0) and np.array_equal(B, B0)
    w2 = workloads.config(2, N=9000)
    w2.x[:] = w2.x * 1.5             # a different tree: the moments must be those of the new build
    plan.update(*w2.arrays(), w2.q)
    st = plan.stats()
    E5, B5 = to_np(plan.eval())
    op = oracle.Plan(*w2.arrays(), w2.q, order_n=3, leaf_size=50, theta=0.5, gamma_bar_value=st["gamma_bar"])
    Eo, Bo = op.eval_treecode() if method == "treecode" else op.eval()
    assert_close(E5, Eo, "E after update")
    assert_close(B5, Bo, "B after update")
    plan.close()
    op.close()
