"""Seeded randomised parity (-m gpu): random sizes, orders 1..9, leaf sizes, theta, tree mode, kernel, method, per-particle
charges and coincident particles, each compared with the oracle exactly as in test_gpu_parity.py (structures bit-exact,
fields 1e-12 in both measures).  A wider sweep of the same generator (several hundred cases) found the n = 9 launch shape."""
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


def _measures(f, fo):
    s = np.sum(fo ** 2)
    if s == 0:
        return float(np.abs(f).max()), 0.0
    return (float(np.sqrt(np.sum((f - fo) ** 2) / s)),
            float(np.linalg.norm(f - fo, axis=1).max() / np.linalg.norm(fo, axis=1).max()))


@pytest.mark.parametrize("seed", range(30))
def test_random_case_matches_oracle(fmm, seed):
    rng = np.random.default_rng(1000 + seed)
    N = int(rng.choice([1, 2, 7, 33, 200, 1000, 3000, 8000]))
    n = int(rng.integers(1, 10))
    N0 = int(rng.choice([1, 3, 16, 40, 64, 100, 128, 256, 300]))
    theta = float(rng.choice([0.2, 0.3, 0.4, 0.5]))
    cfg = int(rng.choice([1, 3, 4]))
    morton, sm, tc = bool(rng.integers(0, 2)), bool(rng.integers(0, 2)), bool(rng.integers(0, 3) == 0)
    if N0 < 16 and N > 1000:
        N0 = 64
    w = workloads.config(cfg, N=N)
    if rng.integers(0, 4) == 0:                      # coincident particles (G17: they contribute nothing to each other)
        k = max(1, N // 10)
        w.x[:k], w.y[:k], w.z[:k] = w.x[-k:].copy(), w.y[-k:].copy(), w.z[-k:].copy()
    q = rng.uniform(-2.0, 2.0, N) if rng.integers(0, 2) else w.q
    flags = ((fmm.FMM_TREE_MORTON_MEDIAN if morton else fmm.FMM_TREE_KD) | (fmm.FMM_KERNEL_SOURCE_MOMENTUM if sm else 0)
             | (fmm.FMM_METHOD_TREECODE if tc else 0))
    plan = fmm.fmm_plan_create(*w.arrays(), q, order_n=n, leaf_size=N0, theta=theta, flags=flags)
    st, ex = plan.stats(), plan.export()
    E, B = plan.eval()
    E, B = E.cpu().numpy().T, B.cpu().numpy().T
    op = oracle.Plan(*w.arrays(), q, order_n=n, leaf_size=N0, theta=theta, gamma_bar_value=st["gamma_bar"],
                     tree_mode=oracle.TREE_MORTON_MEDIAN if morton else oracle.TREE_KD, source_momentum=sm)
    assert np.array_equal(ex["perm"], op.perm())
    if tc:
        near, far = op.treecode_lists()
        Eo, Bo = op.eval_treecode()
    else:
        near, far = op.lists()
        Eo, Bo = op.eval()
    assert np.array_equal(ex["p2p_src"], near[:, 1]) and np.array_equal(ex["m2l_src"], far[:, 1])
    assert np.isfinite(E).all() and np.isfinite(B).all()
    for f, fo, what in ((E, Eo, "E"), (B, Bo, "B")):
        e2, d = _measures(f, fo)
        assert e2 <= TOL and d <= TOL, f"{what}: err2={e2:.3e} max={d:.3e} case={dict(N=N, n=n, N0=N0, theta=theta, cfg=cfg, morton=morton, sm=sm, tc=tc)}"
    plan.close()
    op.close()
