"""Thin ctypes binding over libfmm_b200.so (include/fmm.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels.  PyTorch supplies device memory (the
library's workspace comes from torch's caching allocator through the fmm_alloc_fn callback) and the
stream.  There is no CPU fallback: if the library is missing or there is no CUDA device, calls raise.

The functions carry the names of the C entry points: ``fmm_plan_create``, ``fmm_plan_update``,
``fmm_eval``, ``fmm_direct``, ``fmm_field_host``, ``fmm_plan_stats``, ``fmm_plan_export``,
``fmm_plan_destroy``.  ``Plan`` is a small convenience wrapper around them.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np
import torch

HERE = Path(__file__).resolve().parent
LIB_PATH = HERE / "libfmm_b200.so"

FMM_MAX_ORDER = 12
FMM_TREE_KD = 0
FMM_TREE_MORTON_MEDIAN = 1
FMM_TREE_STOP_AT_N0 = 32
FMM_RAW_SUMS = 4
FMM_KERNEL_MEAN_GAMMA = 0
FMM_KERNEL_SOURCE_MOMENTUM = 8
FMM_METHOD_FMM = 0
FMM_METHOD_TREECODE = 16

_dp = C.POINTER(C.c_double)
_i64p = C.POINTER(C.c_int64)
_i32p = C.POINTER(C.c_int32)
ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class fmm_particles_t(C.Structure):
    _fields_ = [("N", C.c_int64), ("x", C.c_void_p), ("y", C.c_void_p), ("z", C.c_void_p),
                ("px", C.c_void_p), ("py", C.c_void_p), ("pz", C.c_void_p), ("q", C.c_void_p),
                ("q_scalar", C.c_double)]


class fmm_params_t(C.Structure):
    _fields_ = [("order_n", C.c_int), ("leaf_size", C.c_int), ("theta", C.c_double),
                ("gamma_bar", C.c_double), ("flags", C.c_uint32)]


class fmm_stats_t(C.Structure):
    _fields_ = [("N", C.c_int64), ("order_n", C.c_int32), ("P", C.c_int32), ("leaf_size", C.c_int32),
                ("kappa", C.c_int32), ("nodes", C.c_int64), ("leaves", C.c_int64), ("n_p2p", C.c_int64),
                ("n_m2l", C.c_int64), ("p2p_pairs", C.c_int64), ("m2l_pairs", C.c_int64),
                ("gamma_bar", C.c_double), ("theta", C.c_double), ("flags", C.c_uint32),
                ("timing_valid", C.c_int32), ("ms_tree", C.c_float), ("ms_lists", C.c_float),
                ("ms_p2m", C.c_float), ("ms_m2m", C.c_float), ("ms_m2l", C.c_float), ("ms_l2l", C.c_float),
                ("ms_p2p", C.c_float), ("ms_l2p", C.c_float), ("workspace_bytes", C.c_int64),
                ("p2p_split", C.c_int32), ("m2l_split", C.c_int32), ("p2p_mutual", C.c_int32), ("early_leaves", C.c_int32),
                ("react_particles", C.c_int64)]

    def as_dict(self) -> dict:
        return {k: getattr(self, k) for k, _ in self._fields_}


class fmm_export_t(C.Structure):
    _fields_ = [("perm", C.c_void_p), ("node_lo", C.c_void_p), ("node_hi", C.c_void_p), ("bbox", C.c_void_p),
                ("p2p_off", C.c_void_p), ("p2p_src", C.c_void_p), ("m2l_off", C.c_void_p), ("m2l_src", C.c_void_p),
                ("M", C.c_void_p), ("L", C.c_void_p)]


EXPORTED_SYMBOLS = ["fmm_plan_create", "fmm_plan_update", "fmm_plan_refit", "fmm_plan_refit_keep_lists", "fmm_eval", "fmm_direct", "fmm_direct_noalloc", "fmm_field_host",
                    "fmm_plan_set_timing", "fmm_plan_set_overlap", "fmm_plan_stats", "fmm_plan_export", "fmm_plan_destroy",
                    "fmm_launch_count", "fmm_strerror", "fmm_last_error", "fmm_version"]

_lib = None


class FmmError(RuntimeError):
    pass


def load_library():
    """dlopen libfmm_b200.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not LIB_PATH.exists():
        raise FmmError(f"{LIB_PATH} is missing: build it with `python -m paper_2302_07567_b200.build` "
                       "(there is no CPU fallback)")
    lib = C.CDLL(str(LIB_PATH))
    vp = C.c_void_p
    lib.fmm_plan_create.restype = C.c_int
    lib.fmm_plan_create.argtypes = [C.POINTER(vp), C.POINTER(fmm_particles_t), C.POINTER(fmm_params_t),
                                    ALLOC_FN, FREE_FN, vp, vp]
    lib.fmm_plan_update.restype = C.c_int
    lib.fmm_plan_update.argtypes = [vp, C.POINTER(fmm_particles_t)]
    lib.fmm_plan_refit.restype = C.c_int
    lib.fmm_plan_refit.argtypes = [vp, C.POINTER(fmm_particles_t)]
    lib.fmm_plan_refit_keep_lists.restype = C.c_int
    lib.fmm_plan_refit_keep_lists.argtypes = [vp, C.POINTER(fmm_particles_t), C.POINTER(C.c_double)]
    lib.fmm_eval.restype = C.c_int
    lib.fmm_eval.argtypes = [vp] + [vp] * 6
    lib.fmm_direct.restype = C.c_int
    lib.fmm_direct.argtypes = [C.POINTER(fmm_particles_t), C.c_double, C.c_uint32, C.c_int64, vp] + [vp] * 6 + \
                              [ALLOC_FN, FREE_FN, vp, vp]
    lib.fmm_direct_noalloc.restype = C.c_int
    lib.fmm_direct_noalloc.argtypes = [C.POINTER(fmm_particles_t), C.c_double, C.c_uint32, C.c_int64, vp] + [vp] * 6 + [vp]
    lib.fmm_field_host.restype = C.c_int
    lib.fmm_field_host.argtypes = [C.POINTER(fmm_particles_t), C.POINTER(fmm_params_t)] + [vp] * 6 + \
                                  [C.POINTER(fmm_stats_t), ALLOC_FN, FREE_FN, vp, vp]
    lib.fmm_plan_set_timing.restype = C.c_int
    lib.fmm_plan_set_timing.argtypes = [vp, C.c_int]
    lib.fmm_plan_set_overlap.restype = C.c_int
    lib.fmm_plan_set_overlap.argtypes = [vp, C.c_int]
    lib.fmm_plan_stats.restype = C.c_int
    lib.fmm_plan_stats.argtypes = [vp, C.POINTER(fmm_stats_t)]
    lib.fmm_plan_export.restype = C.c_int
    lib.fmm_plan_export.argtypes = [vp, C.POINTER(fmm_export_t)]
    lib.fmm_plan_destroy.restype = None
    lib.fmm_plan_destroy.argtypes = [vp]
    lib.fmm_launch_count.restype = C.c_int64
    lib.fmm_strerror.restype = C.c_char_p
    lib.fmm_strerror.argtypes = [C.c_int]
    lib.fmm_last_error.restype = C.c_char_p
    lib.fmm_last_error.argtypes = [vp]
    lib.fmm_version.restype = C.c_char_p
    _lib = lib
    return lib


def _require_cuda():
    if not torch.cuda.is_available():
        raise FmmError("no CUDA device: the FMM path runs only on the GPU (there is no CPU fallback)")


def _check(rc: int, plan=None):
    if rc != 0:
        lib = load_library()
        msg = lib.fmm_strerror(rc).decode()
        detail = lib.fmm_last_error(plan).decode()
        raise FmmError(f"libfmm_b200: {msg} ({rc}){': ' + detail if detail else ''}")


# ---- workspace allocator backed by torch's caching allocator --------------------------------
class _TorchAllocator:
    def __init__(self, device):
        self.device = device
        self.live = {}
        self.alloc_cb = ALLOC_FN(self._alloc)
        self.free_cb = FREE_FN(self._free)

    def _alloc(self, nbytes, _user):
        try:
            t = torch.empty(int(nbytes), dtype=torch.uint8, device=self.device)
        except Exception:  # out of memory -> NULL -> FMM_ENOMEM
            return None
        self.live[t.data_ptr()] = t
        return t.data_ptr()

    def _free(self, ptr, _user):
        self.live.pop(ptr, None)


def _dev_f64(a, device):
    t = torch.as_tensor(a, dtype=torch.float64)
    return t.to(device).contiguous()


def _particles(x, y, z, px, py, pz, q, device):
    arrs = [_dev_f64(a, device) for a in (x, y, z, px, py, pz)]
    N = arrs[0].numel()
    for a in arrs:
        if a.numel() != N or a.dim() != 1:
            raise ValueError("x, y, z, px, py, pz must be 1-D arrays of equal length")
    s = fmm_particles_t()
    s.N = N
    s.x, s.y, s.z, s.px, s.py, s.pz = (a.data_ptr() for a in arrs)
    keep = arrs
    if q is None or np.isscalar(q):
        s.q = None
        s.q_scalar = float(-1.602176634e-19 if q is None else q)
    else:
        qt = _dev_f64(q, device)
        if qt.numel() != N:
            raise ValueError("q must have length N")
        s.q = qt.data_ptr()
        s.q_scalar = 0.0
        keep = arrs + [qt]
    return s, keep


def _stream_ptr():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


class _on_plan_stream:
    """Run a block on the plan's stream: the plan stream first waits for the caller's current stream (inputs the
    caller has just produced), and on exit the caller's stream waits for the plan stream (outputs).  Workspace and
    outputs allocated inside belong to the plan stream's pool; ``keep`` tensors are recorded on the caller's stream."""

    def __init__(self, plan):
        self.plan = plan

    def __enter__(self):
        self.caller = torch.cuda.current_stream(self.plan.device)
        self.same = self.caller == self.plan.stream
        if not self.same:
            self.plan.stream.wait_stream(self.caller)
        self.ctx = torch.cuda.stream(self.plan.stream)
        self.ctx.__enter__()
        return self

    def hand_over(self, *tensors):
        if not self.same:
            for t in tensors:
                t.record_stream(self.caller)

    def __exit__(self, *exc):
        self.ctx.__exit__(*exc)
        if not self.same:
            self.caller.wait_stream(self.plan.stream)
        return False


# ---- the C calls --------------------------------------------------------------------------------
class Plan:
    """Handle of an fmm_plan_t (tree + interaction lists).  Create with ``fmm_plan_create``."""

    def __init__(self, handle, allocator, N, device, stream):
        self._h = handle
        self._alloc = allocator
        self.N = N
        self.device = device
        # The library enqueues everything on the stream given to fmm_plan_create and frees scratch right after
        # enqueueing (stream-ordered).  Torch's caching allocator is per stream, so every later call runs under
        # this stream (``_on_plan_stream``) and the caller's current stream is ordered with it on both sides.
        self.stream = stream

    def update(self, x, y, z, px, py, pz, q=None):
        return fmm_plan_update(self, x, y, z, px, py, pz, q)

    def refit_keep_lists(self, x, y, z, px, py, pz, q=None) -> float:
        """fmm_plan_refit_keep_lists: returns eta_eff, the largest admissibility ratio of the kept far pairs."""
        return fmm_plan_refit_keep_lists(self, x, y, z, px, py, pz, q)

    def refit(self, x, y, z, px, py, pz, q=None):
        return fmm_plan_refit(self, x, y, z, px, py, pz, q)

    def eval(self, out=None):
        return fmm_eval(self, out)

    def stats(self) -> dict:
        return fmm_plan_stats(self)

    def export(self, want_M=False, want_L=False) -> dict:
        return fmm_plan_export(self, want_M, want_L)

    def set_overlap(self, on=True):
        _check(load_library().fmm_plan_set_overlap(self._h, int(bool(on))), self._h)

    def set_timing(self, on=True):
        _check(load_library().fmm_plan_set_timing(self._h, int(bool(on))), self._h)

    def close(self):
        fmm_plan_destroy(self)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def fmm_plan_create(x, y, z, px, py, pz, q=None, *, order_n, leaf_size, theta, gamma_bar=0.0,
                    flags=FMM_TREE_KD, device="cuda:0") -> Plan:
    """a0-a3: gamma_bar, tree order, bounding boxes, dual tree traversal -> CSR lists."""
    _require_cuda()
    lib = load_library()
    device = torch.device(device)
    with torch.cuda.device(device):
        parts, keep = _particles(x, y, z, px, py, pz, q, device)
        prm = fmm_params_t(int(order_n), int(leaf_size), float(theta), float(gamma_bar), int(flags))
        alloc = _TorchAllocator(device)
        h = C.c_void_p()
        rc = lib.fmm_plan_create(C.byref(h), C.byref(parts), C.byref(prm), alloc.alloc_cb, alloc.free_cb, None,
                                 _stream_ptr())
        _check(rc)
        stream = torch.cuda.current_stream(device)
        del keep
    return Plan(h, alloc, parts.N, device, stream)


def fmm_plan_update(plan: Plan, x, y, z, px, py, pz, q=None):
    lib = load_library()
    with torch.cuda.device(plan.device), _on_plan_stream(plan):
        parts, keep = _particles(x, y, z, px, py, pz, q, plan.device)
        _check(lib.fmm_plan_update(plan._h, C.byref(parts)), plan._h)
        del keep


def fmm_plan_refit(plan: Plan, x, y, z, px, py, pz, q=None):
    """Keeps the particle order of the last build; new boxes and lists on the moved particles (no sort)."""
    lib = load_library()
    with torch.cuda.device(plan.device), _on_plan_stream(plan):
        parts, keep = _particles(x, y, z, px, py, pz, q, plan.device)
        _check(lib.fmm_plan_refit(plan._h, C.byref(parts)), plan._h)
        del keep


def fmm_plan_refit_keep_lists(plan: Plan, x, y, z, px, py, pz, q=None) -> float:
    """Keeps the particle order AND both lists of the last build; new gamma_bar, boxes and moments.  Returns eta_eff."""
    lib = load_library()
    eta = C.c_double(0.0)
    with torch.cuda.device(plan.device), _on_plan_stream(plan):
        parts, keep = _particles(x, y, z, px, py, pz, q, plan.device)
        _check(lib.fmm_plan_refit_keep_lists(plan._h, C.byref(parts), C.byref(eta)), plan._h)
        del keep
    return float(eta.value)


def fmm_eval(plan: Plan, out=None):
    """a4-a10.  Returns (E[3,N], B[3,N]) device tensors in caller order (rows x, y, z).  Enqueue only."""
    lib = load_library()
    with torch.cuda.device(plan.device), _on_plan_stream(plan) as s:
        if out is None:
            out = torch.empty((6, plan.N), dtype=torch.float64, device=plan.device)
            s.hand_over(out)
        ptrs = [C.c_void_p(out[k].data_ptr()) for k in range(6)]
        _check(lib.fmm_eval(plan._h, *ptrs), plan._h)
    return out[:3], out[3:]


def fmm_plan_stats(plan: Plan) -> dict:
    s = fmm_stats_t()
    _check(load_library().fmm_plan_stats(plan._h, C.byref(s)), plan._h)
    return s.as_dict()


def fmm_plan_export(plan: Plan, want_M=False, want_L=False) -> dict:
    """Host copies of perm, node ranges, bounding boxes, CSR lists and optionally M / L."""
    st = fmm_plan_stats(plan)
    N, nodes, P = st["N"], st["nodes"], st["P"]
    out = {
        "perm": np.empty(N, dtype=np.int64), "node_lo": np.empty(nodes, dtype=np.int64),
        "node_hi": np.empty(nodes, dtype=np.int64), "bbox": np.empty((nodes, 6)),
        "p2p_off": np.empty(nodes + 1, dtype=np.int32), "p2p_src": np.empty(st["n_p2p"], dtype=np.int32),
        "m2l_off": np.empty(nodes + 1, dtype=np.int32), "m2l_src": np.empty(st["n_m2l"], dtype=np.int32),
    }
    if want_M:
        out["M"] = np.empty((nodes, P, 4))
    if want_L:
        out["L"] = np.empty((nodes, P, 6))
    e = fmm_export_t()
    for k, v in out.items():
        setattr(e, k, v.ctypes.data if v.size else None)
    with torch.cuda.device(plan.device), _on_plan_stream(plan):
        _check(load_library().fmm_plan_export(plan._h, C.byref(e)), plan._h)
    return out


def fmm_plan_destroy(plan: Plan):
    if getattr(plan, "_h", None):
        load_library().fmm_plan_destroy(plan._h)
        plan._h = None
        plan._alloc.live.clear()


def fmm_direct(x, y, z, px, py, pz, q=None, *, gamma_bar=0.0, flags=0, targets=None, device="cuda:0"):
    """a11: direct summation at ``targets`` (index array; None = all).  Returns (E[3,nt], B[3,nt])."""
    _require_cuda()
    lib = load_library()
    device = torch.device(device)
    with torch.cuda.device(device):
        parts, keep = _particles(x, y, z, px, py, pz, q, device)
        if targets is None:
            nt, tptr, tkeep = parts.N, None, None
        else:
            tkeep = torch.as_tensor(np.ascontiguousarray(targets, dtype=np.int64)).to(device)
            nt, tptr = tkeep.numel(), C.c_void_p(tkeep.data_ptr())
        out = torch.empty((6, nt), dtype=torch.float64, device=device)
        alloc = _TorchAllocator(device)
        rc = lib.fmm_direct(C.byref(parts), float(gamma_bar), int(flags), nt, tptr,
                            *[C.c_void_p(out[k].data_ptr()) for k in range(6)],
                            alloc.alloc_cb, alloc.free_cb, None, _stream_ptr())
        _check(rc)
        torch.cuda.current_stream().synchronize()  # inputs (keep, tkeep) must outlive the enqueued work
        del keep, tkeep
    return out[:3], out[3:]


FMM_NOALLOC_MAX_N = 32768


def fmm_direct_noalloc(x, y, z, px, py, pz, q=None, *, gamma_bar, flags=0, targets=None, out=None, device="cuda:0"):
    """a11 through the entry point that allocates nothing (scratch in a fixed device array of the library; N and the number
    of targets at most FMM_NOALLOC_MAX_N; one call at a time per device).  Inputs already on the device are used in place and
    ``out`` ([6, nt] float64 device tensor) is written in place, so that a caller who passes both makes no allocation at all.
    Returns (E[3,nt], B[3,nt]) as views of ``out``.  Enqueue only when the inputs are device tensors."""
    _require_cuda()
    lib = load_library()
    device = torch.device(device)
    with torch.cuda.device(device):
        parts, keep = _particles(x, y, z, px, py, pz, q, device)
        if targets is None:
            nt, tptr, tkeep = parts.N, None, None
        else:
            tkeep = targets if (torch.is_tensor(targets) and targets.is_cuda and targets.dtype == torch.int64) else \
                torch.as_tensor(np.ascontiguousarray(targets, dtype=np.int64)).to(device)
            nt, tptr = tkeep.numel(), C.c_void_p(tkeep.data_ptr())
        if out is None:
            out = torch.empty((6, nt), dtype=torch.float64, device=device)
        if out.shape != (6, nt) or out.dtype != torch.float64 or not out.is_cuda or not out.is_contiguous():
            raise ValueError("out must be a contiguous [6, n_targets] float64 device tensor")
        rc = lib.fmm_direct_noalloc(C.byref(parts), float(gamma_bar), int(flags), nt, tptr,
                                    *[C.c_void_p(out[k].data_ptr()) for k in range(6)], _stream_ptr())
        _check(rc)
        torch.cuda.current_stream().synchronize()  # inputs (keep, tkeep) must outlive the enqueued work
        del keep, tkeep
    return out[:3], out[3:]


def fmm_field_host(x, y, z, px, py, pz, q=None, *, order_n, leaf_size, theta, gamma_bar=0.0,
                   flags=FMM_TREE_KD, out=None, device="cuda:0"):
    """Whole of Alg 5.12 from HOST arrays (numpy or pinned CPU tensors) to host arrays.

    Returns (E[3,N], B[3,N]) as a host tensor pair plus the plan statistics."""
    _require_cuda()
    lib = load_library()
    device = torch.device(device)
    host = [torch.as_tensor(a, dtype=torch.float64).contiguous() for a in (x, y, z, px, py, pz)]
    N = host[0].numel()
    s = fmm_particles_t()
    s.N = N
    s.x, s.y, s.z, s.px, s.py, s.pz = (a.data_ptr() for a in host)
    if q is None or np.isscalar(q):
        s.q, s.q_scalar = None, float(-1.602176634e-19 if q is None else q)
    else:
        qh = torch.as_tensor(q, dtype=torch.float64).contiguous()
        host.append(qh)
        s.q, s.q_scalar = qh.data_ptr(), 0.0
    if out is None:
        out = torch.empty((6, N), dtype=torch.float64).pin_memory()
    prm = fmm_params_t(int(order_n), int(leaf_size), float(theta), float(gamma_bar), int(flags))
    st = fmm_stats_t()
    with torch.cuda.device(device):
        alloc = _TorchAllocator(device)
        rc = lib.fmm_field_host(C.byref(s), C.byref(prm), *[C.c_void_p(out[k].data_ptr()) for k in range(6)],
                                C.byref(st), alloc.alloc_cb, alloc.free_cb, None, _stream_ptr())
        _check(rc)
    return out[:3], out[3:], st.as_dict()


def fmm_launch_count() -> int:
    return int(load_library().fmm_launch_count())
