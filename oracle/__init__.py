"""TEST INFRASTRUCTURE ONLY -- ctypes front-end of the CPU fp64 oracle.

The arithmetic lives in ``oracle/qmcd_oracle.c`` (plain C, fp64, no BLAS); this
file only compiles it with gcc and marshals numpy arrays.  It shares nothing
with, and never imports, ``paper_1708_00744_b200`` (the CUDA path).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.

Paths (citations: /root/reference/PAPER.md):
  * path 0 -- explicit LU determinant ratio / inverse
  * path 1 -- rank-1 Sherman-Morrison, Eqs. 1-2
  * path 2 -- delayed rank-K, Eqs. 3-4
  * path 3 -- lock-step variant; path 4 -- path 2 with the slot-replacement
    accept for an electron accepted twice inside one window (reading G7)
Pins: tests/test_oracle_pins.py (every function, incl. the residual on known non-zero
cases).  Parity unpinned: nothing.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "qmcd_oracle.c")
_LIB = os.path.join(_HERE, "libqmcd_oracle.so")
_lock = threading.Lock()
_lib = None

ORC_OK, ORC_ESINGULAR, ORC_EINVAL, ORC_ENOMEM = 0, -1, -2, -3


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, strict fp64, OpenMP over walkers)."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp",
                   "-fno-fast-math", "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True, capture_output=True)
            os.replace(tmp, _LIB)
    return _LIB


_dp = ctypes.POINTER(ctypes.c_double)
_ip = ctypes.POINTER(ctypes.c_int)
_up = ctypes.POINTER(ctypes.c_ubyte)


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build()
    L = ctypes.CDLL(_LIB)
    L.orc_slogdet.argtypes = [ctypes.c_int, _dp, _ip, _dp]
    L.orc_slogdet.restype = ctypes.c_int
    L.orc_inverse.argtypes = [ctypes.c_int, _dp, _dp]
    L.orc_inverse.restype = ctypes.c_int
    L.orc_ratio_bruteforce.argtypes = [ctypes.c_int, _dp, ctypes.c_int, _dp, _dp]
    L.orc_ratio_bruteforce.restype = ctypes.c_int
    L.orc_sm_ratio.argtypes = [ctypes.c_int, _dp, ctypes.c_int, _dp]
    L.orc_sm_ratio.restype = ctypes.c_double
    L.orc_sm_accept.argtypes = [ctypes.c_int, _dp, ctypes.c_int, _dp]
    L.orc_sm_accept.restype = ctypes.c_int
    L.orc_delayed_create.argtypes = [ctypes.c_int, ctypes.c_int, _dp]
    L.orc_delayed_create.restype = ctypes.c_void_p
    L.orc_delayed_destroy.argtypes = [ctypes.c_void_p]
    L.orc_delayed_destroy.restype = None
    L.orc_delayed_pending.argtypes = [ctypes.c_void_p]
    L.orc_delayed_pending.restype = ctypes.c_int
    L.orc_delayed_flush_count.argtypes = [ctypes.c_void_p]
    L.orc_delayed_flush_count.restype = ctypes.c_long
    L.orc_delayed_ratio.argtypes = [ctypes.c_void_p, ctypes.c_int, _dp, _dp]
    L.orc_delayed_ratio.restype = ctypes.c_int
    L.orc_delayed_accept.argtypes = [ctypes.c_void_p]
    L.orc_delayed_accept.restype = ctypes.c_int
    L.orc_delayed_reject.argtypes = [ctypes.c_void_p]
    L.orc_delayed_reject.restype = None
    L.orc_delayed_flush.argtypes = [ctypes.c_void_p]
    L.orc_delayed_flush.restype = ctypes.c_int
    L.orc_delayed_S.argtypes = [ctypes.c_void_p]
    L.orc_delayed_S.restype = _dp
    L.orc_delayed_J.argtypes = [ctypes.c_void_p]
    L.orc_delayed_J.restype = _ip
    L.orc_run.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                          ctypes.c_int, _dp, _dp, _up, _dp, ctypes.c_int, ctypes.c_int,
                          _dp, _up, _ip]
    L.orc_run.restype = ctypes.c_int
    L.orc_run_lockstep.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                   _dp, _dp, _dp, _up, _dp, ctypes.c_int, ctypes.c_int,
                                   _dp, _up, ctypes.POINTER(ctypes.c_long), _ip]
    L.orc_run_lockstep.restype = ctypes.c_int
    L.orc_delayed_set_replace.argtypes = [ctypes.c_void_p, ctypes.c_int]
    L.orc_delayed_set_replace.restype = None
    L.orc_run_jseq.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, _ip, ctypes.c_int,
                               _dp, _dp, _up, _dp, ctypes.c_int, ctypes.c_int,
                               _dp, _up, ctypes.POINTER(ctypes.c_long), _ip]
    L.orc_run_jseq.restype = ctypes.c_int
    L.orc_residual.argtypes = [ctypes.c_int, _dp, _dp]
    L.orc_residual.restype = ctypes.c_double
    L.orc_max_threads.argtypes = []
    L.orc_max_threads.restype = ctypes.c_int
    _lib = L
    return L


class OracleError(RuntimeError):
    pass


def _chk(rc: int, what: str):
    if rc < 0:
        raise OracleError(f"{what}: oracle error {rc}")
    return rc


def _f64(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None and a.shape != tuple(shape):
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def _p(a):
    return a.ctypes.data_as(_dp)


# ---------------------------------------------------------------- path 0
def slogdet(A):
    """(sign, log|det A|) by the oracle's own LU."""
    A = _f64(A)
    n = A.shape[0]
    s = ctypes.c_int()
    la = ctypes.c_double()
    _chk(_load().orc_slogdet(n, _p(A), ctypes.byref(s), ctypes.byref(la)), "slogdet")
    return s.value, la.value


def inverse(A):
    """Explicit LU inverse."""
    A = _f64(A)
    n = A.shape[0]
    out = np.empty((n, n), dtype=np.float64)
    _chk(_load().orc_inverse(n, _p(A), _p(out)), "inverse")
    return out


def ratio_bruteforce(A, j, v):
    """det(A with column j := v) / det(A) by explicit LU."""
    A = _f64(A)
    n = A.shape[0]
    v = _f64(v, (n,))
    R = ctypes.c_double()
    _chk(_load().orc_ratio_bruteforce(n, _p(A), int(j), _p(v), ctypes.byref(R)), "ratio_bruteforce")
    return R.value


def residual(A, B):
    """max |A B - I| (BASELINE.json north_star)."""
    A = _f64(A)
    n = A.shape[0]
    B = _f64(B, (n, n))
    return _load().orc_residual(n, _p(A), _p(B))


# ---------------------------------------------------------------- path 1
def sm_ratio(B, j, v):
    """R = B[j,:].v, Eq. 1."""
    B = _f64(B)
    n = B.shape[0]
    v = _f64(v, (n,))
    return _load().orc_sm_ratio(n, _p(B), int(j), _p(v))


def sm_accept(B, j, v):
    """In-place Sherman-Morrison update of B (must be a C-contiguous float64 array), Eq. 2."""
    if not (isinstance(B, np.ndarray) and B.dtype == np.float64 and B.flags.c_contiguous):
        raise ValueError("B must be a C-contiguous float64 ndarray (updated in place)")
    n = B.shape[0]
    v = _f64(v, (n,))
    rc = _load().orc_sm_accept(n, _p(B), int(j), _p(v))
    if rc == ORC_ESINGULAR:
        raise OracleError("sm_accept: singular move (R == 0 or non-finite)")
    _chk(rc, "sm_accept")


# ---------------------------------------------------------------- path 2
class Delayed:
    """One walker's delayed rank-K state.  ``B`` is borrowed and
    updated in place at every flush."""

    def __init__(self, B, K, replace=False):
        """replace=True: path 4 -- an electron accepted again inside one window replaces the column of
        its queue slot instead of flushing first (reading G7, second alternative)."""
        if not (isinstance(B, np.ndarray) and B.dtype == np.float64 and B.flags.c_contiguous):
            raise ValueError("B must be a C-contiguous float64 ndarray (updated in place)")
        self.B = B
        self.n = B.shape[0]
        self.K = int(K)
        self._L = _load()
        self._h = self._L.orc_delayed_create(self.n, self.K, _p(B))
        if not self._h:
            raise OracleError("delayed_create: bad arguments (need 1 <= K <= N)")
        if replace:
            self._L.orc_delayed_set_replace(self._h, 1)

    def __del__(self):
        h, self._h = getattr(self, "_h", None), None
        if h:
            self._L.orc_delayed_destroy(h)

    @property
    def pending(self) -> int:
        return self._L.orc_delayed_pending(self._h)

    @property
    def flush_count(self) -> int:
        return self._L.orc_delayed_flush_count(self._h)

    def ratio(self, j, v) -> float:
        v = _f64(v, (self.n,))
        R = ctypes.c_double()
        _chk(self._L.orc_delayed_ratio(self._h, int(j), _p(v), ctypes.byref(R)), "delayed_ratio")
        return R.value

    def accept(self) -> bool:
        """Queue the staged move; returns True if a flush happened inside."""
        rc = self._L.orc_delayed_accept(self._h)
        if rc == ORC_ESINGULAR:
            raise OracleError("delayed_accept: singular move")
        return bool(_chk(rc, "delayed_accept"))

    def reject(self):
        self._L.orc_delayed_reject(self._h)

    def flush(self):
        _chk(self._L.orc_delayed_flush(self._h), "delayed_flush")

    def S(self):
        m, K = self.pending, self.K
        full = np.ctypeslib.as_array(self._L.orc_delayed_S(self._h), shape=(K, K))
        return full[:m, :m].copy()

    def J(self):
        m = self.pending
        return np.ctypeslib.as_array(self._L.orc_delayed_J(self._h), shape=(self.K,))[:m].copy()


# ---------------------------------------------------------------- batch driver
def run(path, B, K, proposals, j_begin=0, mask=None, uniforms=None, final_flush=True):
    """Run n_moves proposals on every walker (sequential electrons from j_begin).

    B          [batch][N][N] float64, C-contiguous, updated IN PLACE
    proposals  [n_moves][batch][N]
    mask       [n_moves][batch] uint8  -> accept iff mask            (mode 0)
    uniforms   [n_moves][batch] f64    -> accept iff u < min(1,R^2)  (mode 1)
    Returns (R [n_moves][batch], acc [n_moves][batch] uint8, threads_used).
    """
    if not (isinstance(B, np.ndarray) and B.dtype == np.float64 and B.flags.c_contiguous and B.ndim == 3):
        raise ValueError("B must be a C-contiguous float64 [batch][N][N] ndarray")
    batch, n, _ = B.shape
    proposals = _f64(proposals)
    n_moves = proposals.shape[0]
    if proposals.shape != (n_moves, batch, n):
        raise ValueError("proposals must be [n_moves][batch][N]")
    if (mask is None) == (uniforms is None):
        raise ValueError("exactly one of mask / uniforms")
    R = np.zeros((n_moves, batch), dtype=np.float64)
    acc = np.zeros((n_moves, batch), dtype=np.uint8)
    thr = ctypes.c_int()
    if mask is not None:
        mask = np.ascontiguousarray(mask, dtype=np.uint8)
        assert mask.shape == (n_moves, batch)
        mp, up, mode = mask.ctypes.data_as(_up), None, 0
    else:
        uniforms = _f64(uniforms, (n_moves, batch))
        mp, up, mode = None, _p(uniforms), 1
    rc = _load().orc_run(int(path), batch, n, int(K), n_moves, int(j_begin), _p(B), _p(proposals),
                         mp, up, mode, int(bool(final_flush)), _p(R), acc.ctypes.data_as(_up),
                         ctypes.byref(thr))
    _chk(rc, "run")
    return R, acc, thr.value


def run_lockstep(A, B, K, proposals, j_begin=0, mask=None, uniforms=None, final_flush=True):
    """Path 3, the lock-step variant: every proposal takes a queue slot
    (a rejected one with the unchanged column of A), Eq. 4 every K proposals.

    A, B       [batch][N][N] float64, C-contiguous, both updated IN PLACE
    other arguments as in run().  Returns (R, acc, flushes [batch], threads_used).
    """
    for X in (A, B):
        if not (isinstance(X, np.ndarray) and X.dtype == np.float64 and X.flags.c_contiguous and X.ndim == 3):
            raise ValueError("A and B must be C-contiguous float64 [batch][N][N] ndarrays")
    if A.shape != B.shape:
        raise ValueError("A and B differ in shape")
    batch, n, _ = B.shape
    proposals = _f64(proposals)
    n_moves = proposals.shape[0]
    if proposals.shape != (n_moves, batch, n):
        raise ValueError("proposals must be [n_moves][batch][N]")
    if (mask is None) == (uniforms is None):
        raise ValueError("exactly one of mask / uniforms")
    R = np.zeros((n_moves, batch), dtype=np.float64)
    acc = np.zeros((n_moves, batch), dtype=np.uint8)
    fl = (ctypes.c_long * batch)()
    thr = ctypes.c_int()
    if mask is not None:
        mask = np.ascontiguousarray(mask, dtype=np.uint8)
        assert mask.shape == (n_moves, batch)
        mp, up, mode = mask.ctypes.data_as(_up), None, 0
    else:
        uniforms = _f64(uniforms, (n_moves, batch))
        mp, up, mode = None, _p(uniforms), 1
    rc = _load().orc_run_lockstep(batch, n, int(K), n_moves, int(j_begin), _p(A), _p(B), _p(proposals),
                                  mp, up, mode, int(bool(final_flush)), _p(R), acc.ctypes.data_as(_up),
                                  fl, ctypes.byref(thr))
    _chk(rc, "run_lockstep")
    return R, acc, np.array(list(fl), dtype=np.int64), thr.value


def run_jseq(B, K, proposals, jseq, replace, mask=None, uniforms=None, final_flush=True):
    """Delayed rank-K run with an ARBITRARY electron sequence jseq [n_moves] (the same for every
    walker).  replace=False: path 2 (a repeated electron flushes first); replace=True: path 4
    (slot replacement).  Returns (R, acc, flushes [batch], threads_used); B updated in place."""
    if not (isinstance(B, np.ndarray) and B.dtype == np.float64 and B.flags.c_contiguous and B.ndim == 3):
        raise ValueError("B must be a C-contiguous float64 [batch][N][N] ndarray")
    batch, n, _ = B.shape
    proposals = _f64(proposals)
    n_moves = proposals.shape[0]
    if proposals.shape != (n_moves, batch, n):
        raise ValueError("proposals must be [n_moves][batch][N]")
    jseq = np.ascontiguousarray(jseq, dtype=np.int32)
    if jseq.shape != (n_moves,):
        raise ValueError("jseq must be [n_moves]")
    if (mask is None) == (uniforms is None):
        raise ValueError("exactly one of mask / uniforms")
    R = np.zeros((n_moves, batch), dtype=np.float64)
    acc = np.zeros((n_moves, batch), dtype=np.uint8)
    fl = (ctypes.c_long * batch)()
    thr = ctypes.c_int()
    if mask is not None:
        mask = np.ascontiguousarray(mask, dtype=np.uint8)
        assert mask.shape == (n_moves, batch)
        mp, up, mode = mask.ctypes.data_as(_up), None, 0
    else:
        uniforms = _f64(uniforms, (n_moves, batch))
        mp, up, mode = None, _p(uniforms), 1
    rc = _load().orc_run_jseq(batch, n, int(K), n_moves, jseq.ctypes.data_as(_ip), int(bool(replace)),
                              _p(B), _p(proposals), mp, up, mode, int(bool(final_flush)), _p(R),
                              acc.ctypes.data_as(_up), fl, ctypes.byref(thr))
    _chk(rc, "run_jseq")
    return R, acc, np.array(list(fl), dtype=np.int64), thr.value


def max_threads() -> int:
    return _load().orc_max_threads()
