"""GPU test (-m gpu) of fmm_direct_noalloc, the one entry point that allocates nothing (include/fmm.h): its scratch is a
fixed device array inside the library.  Collected last on purpose (the file name sorts after every other test file).

Checked against the existing path, fmm_direct, within the 1e-12 of the other GPU tests (eq. (6.1) norm and max norm), on
calls made in a row that share the array: different sizes, target subsets, per-particle charges, both kernels; a repeat of
the first call must reproduce it bit for bit (nothing of the calls in between leaks through the shared scratch); the size
limit is refused with a clear text; torch's allocator and the device's free memory see no allocation across the calls.
Stands alone: builds / loads the library itself and depends on no state left by other tests.
"""
import numpy as np
import pytest

from paper_2302_07567_b200 import workloads

pytestmark = pytest.mark.gpu

TOL = 1e-12


@pytest.fixture(scope="module")
def fmm():
    from paper_2302_07567_b200 import binding, build
    build.build_library()
    binding.load_library()
    return binding


def assert_close(got, ref, what, tol=TOL):
    f, fref = got.cpu().numpy().T, ref.cpu().numpy().T
    e2 = np.sqrt(np.sum((f - fref) ** 2) / np.sum(fref ** 2))
    d = np.linalg.norm(f - fref, axis=1).max() / np.linalg.norm(fref, axis=1).max()
    assert e2 <= tol and d <= tol, f"{what}: err2={e2:.3e} max={d:.3e} > {tol}"


def mean_gamma(w):
    return float(np.sqrt(1.0 + np.mean(w.px) ** 2 + np.mean(w.py) ** 2 + np.mean(w.pz) ** 2))


def test_no_alloc_direct_matches_fmm_direct_on_calls_in_a_row(fmm):
    import torch
    dev = torch.device("cuda:0")
    w1 = workloads.config(1, N=5003)
    w2 = workloads.config(2, N=3000)
    gb1, gb2 = mean_gamma(w1), mean_gamma(w2)
    q2 = np.random.default_rng(3).uniform(0.5, 2.0, w2.N) * workloads.ELECTRON_CHARGE
    tidx = np.random.default_rng(5).choice(w2.N, size=777, replace=False).astype(np.int64)

    # call 1: all targets, scalar charge
    E1, B1 = fmm.fmm_direct_noalloc(*w1.arrays(), w1.q, gamma_bar=gb1)
    E1, B1 = E1.clone(), B1.clone()
    Er, Br = fmm.fmm_direct(*w1.arrays(), w1.q, gamma_bar=gb1)
    assert_close(E1, Er, "call 1 E")
    assert_close(B1, Br, "call 1 B")
    # call 2, right behind it: another bunch, a target subset, per-particle charges (fewer sources and targets than call 1,
    # so the array still holds call 1's weights and partial sums beyond what this call writes)
    E2, B2 = fmm.fmm_direct_noalloc(*w2.arrays(), q2, gamma_bar=gb2, targets=tidx)
    Er, Br = fmm.fmm_direct(*w2.arrays(), q2, gamma_bar=gb2, targets=tidx)
    assert_close(E2, Er, "call 2 E")
    assert_close(B2, Br, "call 2 B")
    # call 3: the source-momentum kernel (needs no gamma_bar), raw sums
    fl = fmm.FMM_KERNEL_SOURCE_MOMENTUM | fmm.FMM_RAW_SUMS
    E3, B3 = fmm.fmm_direct_noalloc(*w2.arrays(), q2, gamma_bar=0.0, flags=fl, targets=tidx)
    Er, Br = fmm.fmm_direct(*w2.arrays(), q2, flags=fl, targets=tidx)
    assert_close(E3, Er, "call 3 E")
    assert_close(B3, Br, "call 3 B")
    # call 4 = call 1 again: bit for bit what call 1 gave
    E4, B4 = fmm.fmm_direct_noalloc(*w1.arrays(), w1.q, gamma_bar=gb1)
    assert torch.equal(E4, E1) and torch.equal(B4, B1)

    # with inputs and outputs already on the device the calls allocate nothing that torch or the driver can see
    d_in = [torch.as_tensor(a, dtype=torch.float64).to(dev) for a in w1.arrays()]
    out = torch.empty((6, w1.N), dtype=torch.float64, device=dev)
    fmm.fmm_direct_noalloc(*d_in, w1.q, gamma_bar=gb1, out=out)
    torch.cuda.synchronize()
    for _ in range(2):
        out.zero_()
        torch.cuda.synchronize()
        # (the counters bracket the library call alone: torch.equal and friends below allocate their own temporaries)
        before = (torch.cuda.memory_allocated(dev), torch.cuda.memory_reserved(dev),
                  torch.cuda.memory_stats(dev)["allocation.all.allocated"], torch.cuda.mem_get_info(dev)[0])
        fmm.fmm_direct_noalloc(*d_in, w1.q, gamma_bar=gb1, out=out)
        torch.cuda.synchronize()
        after = (torch.cuda.memory_allocated(dev), torch.cuda.memory_reserved(dev),
                 torch.cuda.memory_stats(dev)["allocation.all.allocated"], torch.cuda.mem_get_info(dev)[0])
        assert after[:3] == before[:3] and after[3] >= before[3], (before, after)
        assert torch.equal(out[:3], E1) and torch.equal(out[3:], B1)


def test_no_alloc_direct_at_its_size_limit_and_beyond(fmm):
    N = fmm.FMM_NOALLOC_MAX_N
    w = workloads.config(3, N=N)
    gb = mean_gamma(w)
    E, B = fmm.fmm_direct_noalloc(*w.arrays(), w.q, gamma_bar=gb)
    Er, Br = fmm.fmm_direct(*w.arrays(), w.q, gamma_bar=gb)    # (all targets at this size: the pair-sharing kernel)
    assert_close(E, Er, "limit E")
    assert_close(B, Br, "limit B")
    big = workloads.config(3, N=N + 1)
    with pytest.raises(fmm.FmmError, match=r"-1.*exceed the fixed scratch"):
        fmm.fmm_direct_noalloc(*big.arrays(), big.q, gamma_bar=gb)
    with pytest.raises(fmm.FmmError, match=r"-1.*gamma_bar must be given"):
        fmm.fmm_direct_noalloc(*w.arrays(), w.q, gamma_bar=0.0)
    # a refused call leaves the entry point usable
    E2, B2 = fmm.fmm_direct_noalloc(*w.arrays(), w.q, gamma_bar=gb)
    import torch
    assert torch.equal(E2, E) and torch.equal(B2, B)


def test_no_alloc_direct_tiny_inputs(fmm):
    """One particle (no pair: zero fields), 33 particles (one ragged tile), a single target out of many."""
    import torch
    w = workloads.config(1, N=1)
    E, B = fmm.fmm_direct_noalloc(*w.arrays(), w.q, gamma_bar=10.0)
    assert E.shape == (3, 1) and not E.any() and not B.any()
    w = workloads.config(1, N=33)
    E, B = fmm.fmm_direct_noalloc(*w.arrays(), w.q, gamma_bar=10.0)
    Er, Br = fmm.fmm_direct(*w.arrays(), w.q, gamma_bar=10.0)
    assert_close(E, Er, "33 particles E")
    assert_close(B, Br, "33 particles B")
    w = workloads.config(2, N=20000)
    one = np.array([12345], dtype=np.int64)
    E, B = fmm.fmm_direct_noalloc(*w.arrays(), w.q, gamma_bar=10.0, targets=one)
    Er, Br = fmm.fmm_direct(*w.arrays(), w.q, gamma_bar=10.0, targets=one)
    assert E.shape == (3, 1)
    assert_close(E, Er, "single target E")
    assert_close(B, Br, "single target B")
