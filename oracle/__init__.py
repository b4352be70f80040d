"""CPU oracle (TEST INFRASTRUCTURE, NOT THE PRODUCT) -- ctypes wrapper around fmm_oracle.c.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2302_07567_b200`` and shares no code with the CUDA path.

What it computes is stated in ``fmm_oracle.h``: O1 = direct O(N^2) sum of eq. (3.1)-(3.2)
(PAPER.md:143-153), O2 = the serial FMM of Alg 5.12.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "fmm_oracle.c"
_HDR = _HERE / "fmm_oracle.h"
_LIB = _HERE / "libfmm_oracle.so"

TREE_KD = 0
TREE_MORTON_MEDIAN = 1


def build(force: bool = False) -> Path:
    """Compile fmm_oracle.c with gcc (-O2, no FMA contraction, OpenMP over targets)."""
    newest = max(_SRC.stat().st_mtime, _HDR.stat().st_mtime)
    if force or not _LIB.exists() or _LIB.stat().st_mtime < newest:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["gcc", "-std=gnu99", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
               "-fPIC", "-shared", "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None
_dp = C.POINTER(C.c_double)
_i64p = C.POINTER(C.c_int64)
_i32p = C.POINTER(C.c_int32)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        _lib.orc_gamma_bar.restype = C.c_double
        _lib.orc_gamma_bar.argtypes = [C.c_int64, _dp, _dp, _dp]
        _lib.orc_cheb_nodes.argtypes = [C.c_int, _dp]
        _lib.orc_basis_1d.argtypes = [C.c_int, C.c_double, C.c_double, C.c_double, _dp]
        _lib.orc_direct.restype = C.c_int
        _lib.orc_direct.argtypes = [C.c_int64] + [_dp] * 7 + [C.c_double, C.c_double, C.c_int,
                                                               C.c_int64, _i64p] + [_dp] * 6
        _lib.orc_plan_create.restype = C.c_void_p
        _lib.orc_plan_create.argtypes = [C.c_int64] + [_dp] * 7 + [C.c_double, C.c_int, C.c_int,
                                                                    C.c_double, C.c_double, C.c_int, C.c_int]
        _lib.orc_plan_create_given_order.restype = C.c_void_p
        _lib.orc_plan_create_given_order.argtypes = list(_lib.orc_plan_create.argtypes[:13]) + [C.c_int, _i64p]
        _lib.orc_plan_destroy.argtypes = [C.c_void_p]
        _lib.orc_plan_sizes.argtypes = [C.c_void_p, _i64p]
        _lib.orc_plan_gamma_bar.restype = C.c_double
        _lib.orc_plan_gamma_bar.argtypes = [C.c_void_p]
        _lib.orc_plan_perm.argtypes = [C.c_void_p, _i64p]
        _lib.orc_plan_nodes.argtypes = [C.c_void_p, _i64p, _i64p, _dp]
        _lib.orc_plan_lists.argtypes = [C.c_void_p, _i32p, _i32p, _i32p, _i32p]
        _lib.orc_plan_leaf_flags.argtypes = [C.c_void_p, C.POINTER(C.c_int8)]
        _lib.orc_plan_set_lists.restype = C.c_int
        _lib.orc_plan_set_lists.argtypes = [C.c_void_p, C.c_int64, _i32p, _i32p, C.c_int64, _i32p, _i32p]
        _lib.orc_plan_eta_eff.restype = C.c_double
        _lib.orc_plan_eta_eff.argtypes = [C.c_void_p]
        _lib.orc_upward.argtypes = [C.c_void_p, _dp]
        _lib.orc_p2m_node.argtypes = [C.c_void_p, C.c_int64, _dp]
        _lib.orc_eval.restype = C.c_int
        _lib.orc_eval.argtypes = [C.c_void_p, C.c_int64, _i64p, C.c_int] + [_dp] * 7
        _lib.orc_m2l_raw.argtypes = [C.c_void_p, _dp]
        _lib.orc_treecode_sizes.argtypes = [C.c_void_p, _i64p]
        _lib.orc_treecode_lists.argtypes = [C.c_void_p, _i32p, _i32p, _i32p, _i32p]
        _lib.orc_eval_treecode.restype = C.c_int
        _lib.orc_eval_treecode.argtypes = [C.c_void_p] + [_dp] * 6
        _lib.orc_num_threads.restype = C.c_int
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def num_threads() -> int:
    return int(lib().orc_num_threads())


def gamma_bar(px, py, pz) -> float:
    px, ppx = _d(px)
    py, ppy = _d(py)
    pz, ppz = _d(pz)
    return float(lib().orc_gamma_bar(len(px), ppx, ppy, ppz))


def cheb_nodes(n: int) -> np.ndarray:
    c = np.empty(n + 1)
    lib().orc_cheb_nodes(n, c.ctypes.data_as(_dp))
    return c


def basis_1d(n: int, a: float, b: float, x: float) -> np.ndarray:
    ell = np.empty(n + 1)
    lib().orc_basis_1d(n, float(a), float(b), float(x), ell.ctypes.data_as(_dp))
    return ell


def _charges(q, N):
    if q is None or np.isscalar(q):
        return None, None, float(-1.602176634e-19 if q is None else q)
    qa, qp = _d(q)
    assert len(qa) == N
    return qa, qp, 0.0


def direct(x, y, z, px, py, pz, q=None, gamma_bar_value=None, raw=False, targets=None, source_momentum=False):
    """O1: returns (E[nt,3], B[nt,3]) at ``targets`` (default: all particles)."""
    arrs = [_d(a) for a in (x, y, z, px, py, pz)]
    N = len(arrs[0][0])
    qa, qp, qs = _charges(q, N)
    gb = gamma_bar(px, py, pz) if gamma_bar_value is None else float(gamma_bar_value)
    if targets is None:
        nt, tp = N, None
    else:
        t = np.ascontiguousarray(targets, dtype=np.int64)
        nt, tp = len(t), t.ctypes.data_as(_i64p)
    out = [np.empty(nt) for _ in range(6)]
    rc = lib().orc_direct(N, *[p for _, p in arrs], qp, qs, gb, int(bool(raw)) | (2 if source_momentum else 0), nt, tp,
                          *[o.ctypes.data_as(_dp) for o in out])
    assert rc == 0
    return np.stack(out[:3], axis=1), np.stack(out[3:], axis=1)


class Plan:
    """O2: tree + interaction lists, then upward / eval (serial FMM of Alg 5.12)."""

    def __init__(self, x, y, z, px, py, pz, q=None, *, order_n, leaf_size, theta,
                 gamma_bar_value=None, tree_mode=TREE_KD, raw=False, source_momentum=False, given_order=None,
                 stop_at_n0=False):
        """stop_at_n0: Alg 5.2 as printed -- a cluster of at most N0 particles is a leaf wherever it is (leaves on two
        levels, ORC_TREE_STOP_AT_N0); default: every node of level kappa is a leaf (reading T-1).
        given_order: particle order (tree position -> particle index) to build the tree over instead of sorting
        (refit of an existing partition); tree_mode is then ignored."""
        arrs = [_d(a) for a in (x, y, z, px, py, pz)]
        self.N = len(arrs[0][0])
        qa, qp, qs = _charges(q, self.N)
        gb = -1.0 if gamma_bar_value is None else float(gamma_bar_value)
        flags = int(bool(raw)) | (2 if source_momentum else 0) | (4 if stop_at_n0 else 0)
        if given_order is None:
            self._h = lib().orc_plan_create(self.N, *[p for _, p in arrs], qp, qs, int(order_n),
                                            int(leaf_size), float(theta), gb, int(tree_mode), flags)
        else:
            go = np.ascontiguousarray(given_order, dtype=np.int64)
            if go.shape != (self.N,) or not np.array_equal(np.sort(go), np.arange(self.N)):
                raise ValueError("given_order must be a permutation of range(N)")
            self._h = lib().orc_plan_create_given_order(self.N, *[p for _, p in arrs], qp, qs, int(order_n),
                                                        int(leaf_size), float(theta), gb, flags, go.ctypes.data_as(_i64p))
        if not self._h:
            raise ValueError("orc_plan_create: invalid arguments")
        s = np.empty(6, dtype=np.int64)
        lib().orc_plan_sizes(self._h, s.ctypes.data_as(_i64p))
        self.kappa, self.nodes, self.leaves, self.P, self.n_p2p, self.n_m2l = (int(v) for v in s)
        self.n = int(order_n)
        self.gamma_bar = float(lib().orc_plan_gamma_bar(self._h))

    def close(self):
        if getattr(self, "_h", None):
            lib().orc_plan_destroy(self._h)
            self._h = None

    __del__ = close

    def perm(self) -> np.ndarray:
        p = np.empty(self.N, dtype=np.int64)
        lib().orc_plan_perm(self._h, p.ctypes.data_as(_i64p))
        return p

    def node_arrays(self):
        """(lo[nodes], hi[nodes], bbox[nodes,6]); row i-1 is heap node i."""
        lo = np.empty(self.nodes, dtype=np.int64)
        hi = np.empty(self.nodes, dtype=np.int64)
        bb = np.empty((self.nodes, 6))
        lib().orc_plan_nodes(self._h, lo.ctypes.data_as(_i64p), hi.ctypes.data_as(_i64p),
                             bb.ctypes.data_as(_dp))
        return lo, hi, bb

    def leaf_flags(self) -> np.ndarray:
        """[nodes] int8, row i-1 is heap node i: 1 leaf, 0 has children, 2 unused slot (stop_at_n0 only)."""
        f = np.empty(self.nodes, dtype=np.int8)
        lib().orc_plan_leaf_flags(self._h, f.ctypes.data_as(C.POINTER(C.c_int8)))
        return f

    def leaf_ids(self) -> np.ndarray:
        """heap ids of the leaves, ascending"""
        return np.flatnonzero(self.leaf_flags() == 1).astype(np.int64) + 1

    def lists(self):
        """(p2p[np2p,2], m2l[nm2l,2]) as (target, source) heap ids sorted by (target, source)."""
        a = [np.empty(self.n_p2p, dtype=np.int32), np.empty(self.n_p2p, dtype=np.int32),
             np.empty(self.n_m2l, dtype=np.int32), np.empty(self.n_m2l, dtype=np.int32)]
        lib().orc_plan_lists(self._h, *[v.ctypes.data_as(_i32p) for v in a])
        return np.stack(a[:2], axis=1), np.stack(a[2:], axis=1)

    def set_lists(self, p2p, m2l):
        """Replace both lists by (target, source) pairs kept from an earlier traversal (refit with list reuse)."""
        a = [np.ascontiguousarray(np.asarray(v, dtype=np.int32).reshape(-1, 2)[:, k]) for v in (p2p, m2l) for k in (0, 1)]
        rc = lib().orc_plan_set_lists(self._h, len(a[0]), a[0].ctypes.data_as(_i32p), a[1].ctypes.data_as(_i32p),
                                      len(a[2]), a[2].ctypes.data_as(_i32p), a[3].ctypes.data_as(_i32p))
        if rc != 0:
            raise ValueError("orc_plan_set_lists: bad node id")
        self.n_p2p, self.n_m2l = len(a[0]), len(a[2])

    def eta_eff(self) -> float:
        """max over the M2L list of max(diam S_t, diam S_s) / dist(S_t, S_s) with the plan's boxes (Alg 5.6-5.8)."""
        return float(lib().orc_plan_eta_eff(self._h))

    def upward(self) -> np.ndarray:
        M = np.empty((self.nodes, self.P, 4))
        lib().orc_upward(self._h, M.ctypes.data_as(_dp))
        return M

    def p2m_node(self, node: int) -> np.ndarray:
        M = np.empty((self.P, 4))
        lib().orc_p2m_node(self._h, int(node), M.ctypes.data_as(_dp))
        return M

    def m2l_raw(self) -> np.ndarray:
        L = np.empty((self.nodes, self.P, 6))
        lib().orc_m2l_raw(self._h, L.ctypes.data_as(_dp))
        return L

    def treecode_lists(self):
        """(pp[npp,2], pc[npc,2]) as (target leaf, source) heap ids sorted by (target, source)."""
        s = np.empty(2, dtype=np.int64)
        lib().orc_treecode_sizes(self._h, s.ctypes.data_as(_i64p))
        a = [np.empty(int(s[0]), dtype=np.int32), np.empty(int(s[0]), dtype=np.int32),
             np.empty(int(s[1]), dtype=np.int32), np.empty(int(s[1]), dtype=np.int32)]
        lib().orc_treecode_lists(self._h, *[v.ctypes.data_as(_i32p) for v in a])
        return np.stack(a[:2], axis=1), np.stack(a[2:], axis=1)

    def eval_treecode(self):
        """Treecode variant (particle-cluster): (E[N,3], B[N,3]) in caller order."""
        out = [np.empty(self.N) for _ in range(6)]
        lib().orc_eval_treecode(self._h, *[o.ctypes.data_as(_dp) for o in out])
        return np.stack(out[:3], axis=1), np.stack(out[3:], axis=1)

    def eval(self, leaves=None, part="all", want_L=False):
        """Returns (E[N,3], B[N,3]) in caller order (rows of unselected leaves are NaN)."""
        code = {"all": 0, "near": 1, "far": 2}[part]
        out = [np.full(self.N, np.nan) for _ in range(6)]
        if leaves is None:
            nsel, sp = 0, None
        else:
            sel = np.ascontiguousarray(leaves, dtype=np.int64)
            nsel, sp = len(sel), sel.ctypes.data_as(_i64p)
        L = np.empty((self.nodes, self.P, 6)) if want_L else None
        rc = lib().orc_eval(self._h, nsel, sp, code, *[o.ctypes.data_as(_dp) for o in out],
                            L.ctypes.data_as(_dp) if want_L else None)
        if rc != 0:
            raise ValueError("orc_eval: bad leaf selection")
        E, B = np.stack(out[:3], axis=1), np.stack(out[3:], axis=1)
        return (E, B, L) if want_L else (E, B)


def err2(f, f_ref) -> float:
    """eq. (6.1) for one field: (sum_i |f_i - fref_i|^2 / sum_i |fref_i|^2)^(1/2)."""
    f, f_ref = np.asarray(f), np.asarray(f_ref)
    return float(np.sqrt(np.sum((f - f_ref) ** 2) / np.sum(f_ref ** 2)))
