"""Thin ctypes binding of ``libqmcd.so`` (include/qmcd.h): same names, argument
marshalling only -- every step of the hot path runs in the CUDA kernels.  torch is
used for device memory and streams.  There is NO CPU fallback: a missing library
or a missing CUDA device raises.
"""
from __future__ import annotations

import ctypes
import os

from . import buildlib

OK, EINVAL, ESTATE, ECUDA, ESINGULAR, ENOMEM, ELIMIT = 0, -1, -2, -3, -4, -5, -6

# name -> (restype, argtypes); mirrors include/qmcd.h one to one
_vp, _ci, _sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
SYMBOLS = {
    "qmcd_workspace_bytes": (_sz, [_ci, _ci, _ci]),
    "qmcd_create": (_ci, [ctypes.POINTER(_vp), _ci, _ci, _ci, _vp, _sz, _vp]),
    "qmcd_destroy": (_ci, [_vp]),
    "qmcd_set_inverse": (_ci, [_vp, _vp]),
    "qmcd_ratio": (_ci, [_vp, _ci, _vp, _vp]),
    "qmcd_ratio_jv": (_ci, [_vp, _vp, _vp, _vp]),
    "qmcd_accept": (_ci, [_vp, _vp]),
    "qmcd_accept_metropolis": (_ci, [_vp, _vp, _vp]),
    "qmcd_reject": (_ci, [_vp]),
    "qmcd_flush": (_ci, [_vp]),
    "qmcd_pending": (_ci, [_vp, _vp]),
    "qmcd_status": (_ci, [_vp, ctypes.POINTER(_ci), ctypes.POINTER(_ci)]),
    "qmcd_counters": (_ci, [_vp, _vp]),
    "qmcd_worker_stats": (_ci, [_vp, _vp, _vp]),
    "qmcd_sweep": (_ci, [_vp, _ci, _ci, _vp, _vp, _vp, _vp, _vp]),
    "qmcd_sweep_host": (_ci, [_vp, _ci, _ci, _vp, _vp, _vp, _vp, _vp, _vp, _sz]),
    "qmcd_sweep_host_min_staging": (_sz, [_ci, _ci]),
    "qmcd_invert_scratch_bytes": (_sz, [_ci, _ci]),
    "qmcd_invert": (_ci, [_vp, _vp, _vp, _vp, _sz, _vp]),
    "qmcd_invert_static_max_bytes": (_sz, []),
    "qmcd_invert_static": (_ci, [_vp, _vp, _vp, _vp]),
    "qmcd_set_option": (_ci, [_vp, ctypes.c_char_p, _ci]),
    "qmcd_get_option": (_ci, [_vp, ctypes.c_char_p]),
    "qmcd_probe_fp64": (_ci, [_ci, _ci, _vp, ctypes.POINTER(ctypes.c_double)]),
    "qmcd_strerror": (ctypes.c_char_p, [_ci]),
    "qmcd_version": (ctypes.c_char_p, []),
}

_lib = None


class QmcdError(RuntimeError):
    def __init__(self, code, what):
        self.code = code
        msg = _lib.qmcd_strerror(code).decode() if _lib is not None else "?"
        super().__init__(f"{what}: {msg} ({code})")


def load(path: str | None = None):
    """dlopen the library (building is the job of buildlib.build / __graft_entry__.build)."""
    global _lib
    if _lib is not None:
        return _lib
    path = path or buildlib.LIB
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is missing: run `python -m paper_1708_00744_b200.buildlib` "
                           "(there is no CPU fallback)")
    L = ctypes.CDLL(path)
    for name, (res, args) in SYMBOLS.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


def _chk(rc, what):
    if rc < 0:
        raise QmcdError(rc, what)
    return rc


def _ptr(t, dtype=None, device="cuda"):
    """data_ptr of a contiguous tensor (None -> NULL)."""
    if t is None:
        return None
    import torch
    if not isinstance(t, torch.Tensor):
        raise TypeError("expected a torch.Tensor")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"expected dtype {dtype}, got {t.dtype}")
    if device == "cuda" and not t.is_cuda:
        raise ValueError("expected a CUDA tensor")
    if device == "cpu" and t.is_cuda:
        raise ValueError("expected a host tensor")
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    return t.data_ptr()


def workspace_bytes(N, K, batch) -> int:
    return load().qmcd_workspace_bytes(N, K, batch)


def probe_fp64(kind: int, iters: int = 4096) -> float:
    """TFLOP/s of a register-resident DFMA (kind 0) / DMMA (kind 1) loop on this GPU."""
    import torch
    out = ctypes.c_double()
    st = torch.cuda.current_stream().cuda_stream
    _chk(load().qmcd_probe_fp64(kind, iters, st, ctypes.byref(out)), "qmcd_probe_fp64")
    return out.value


class Qmcd:
    """One handle = `batch` walkers of order N with delay K on the current CUDA stream."""

    def __init__(self, N: int, K: int, batch: int, stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("qmcd needs a CUDA device (no CPU fallback)")
        self._L = load()
        self.N, self.K, self.batch = int(N), int(K), int(batch)
        nbytes = self._L.qmcd_workspace_bytes(self.N, self.K, self.batch)
        if nbytes == 0:
            raise QmcdError(EINVAL, "qmcd_workspace_bytes")
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
        off = (-self.workspace.data_ptr()) % 256
        self._ws_ptr = self.workspace.data_ptr() + off
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        h = _vp()
        _chk(self._L.qmcd_create(ctypes.byref(h), self.N, self.K, self.batch, self._ws_ptr, nbytes,
                                 self.stream.cuda_stream), "qmcd_create")
        self._h = h
        self._Ainv = None

    def close(self):
        h, self._h = getattr(self, "_h", None), None
        if h:
            self._L.qmcd_destroy(h)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the calls of include/qmcd.h
    def set_inverse(self, Ainv):
        import torch
        if tuple(Ainv.shape) != (self.batch, self.N, self.N):
            raise ValueError("Ainv must be [batch][N][N]")
        _chk(self._L.qmcd_set_inverse(self._h, _ptr(Ainv, torch.float64)), "qmcd_set_inverse")
        self._Ainv = Ainv                      # keep the borrowed tensor alive

    def ratio(self, j, v, R):
        import torch
        if isinstance(j, int):
            _chk(self._L.qmcd_ratio(self._h, j, _ptr(v, torch.float64), _ptr(R, torch.float64)), "qmcd_ratio")
        else:
            _chk(self._L.qmcd_ratio_jv(self._h, _ptr(j, torch.int32), _ptr(v, torch.float64),
                                       _ptr(R, torch.float64)), "qmcd_ratio_jv")

    def accept(self, mask=None):
        import torch
        _chk(self._L.qmcd_accept(self._h, _ptr(mask, torch.uint8)), "qmcd_accept")

    def accept_metropolis(self, uniforms, acc_out=None):
        import torch
        _chk(self._L.qmcd_accept_metropolis(self._h, _ptr(uniforms, torch.float64),
                                            _ptr(acc_out, torch.uint8)), "qmcd_accept_metropolis")

    def reject(self):
        _chk(self._L.qmcd_reject(self._h), "qmcd_reject")

    def flush(self):
        _chk(self._L.qmcd_flush(self._h), "qmcd_flush")

    def pending(self, m_out=None):
        import torch
        if m_out is None:
            m_out = torch.empty(self.batch, dtype=torch.int32, device="cuda")
        _chk(self._L.qmcd_pending(self._h, _ptr(m_out, torch.int32)), "qmcd_pending")
        return m_out

    def counters(self):
        import torch
        out = torch.empty((self.batch, 8), dtype=torch.int64, device="cuda")
        _chk(self._L.qmcd_counters(self._h, _ptr(out, torch.int64)), "qmcd_counters")
        return out

    def worker_stats(self):
        """-> (stats [512][4] int64 per CTA of the grid, flush_rank_sum [batch] int64); see qmcd.h."""
        import torch
        st = torch.empty((512, 4), dtype=torch.int64, device="cuda")
        fr = torch.empty(self.batch, dtype=torch.int64, device="cuda")
        _chk(self._L.qmcd_worker_stats(self._h, _ptr(st, torch.int64), _ptr(fr, torch.int64)), "qmcd_worker_stats")
        return st, fr

    def status(self):
        st, info = _ci(), (_ci * 2)()
        _chk(self._L.qmcd_status(self._h, ctypes.byref(st), info), "qmcd_status")
        return st.value, (info[0], info[1])

    def sweep(self, j_begin, proposals, mask=None, uniforms=None, R_out=None, acc_out=None):
        import torch
        n_moves = int(proposals.shape[0])
        if tuple(proposals.shape) != (n_moves, self.batch, self.N):
            raise ValueError("proposals must be [n_moves][batch][N]")
        _chk(self._L.qmcd_sweep(self._h, int(j_begin), n_moves, _ptr(proposals, torch.float64),
                                _ptr(mask, torch.uint8), _ptr(uniforms, torch.float64),
                                _ptr(R_out, torch.float64), _ptr(acc_out, torch.uint8)), "qmcd_sweep")

    def sweep_host(self, j_begin, proposals, mask=None, uniforms=None, R_out=None, acc_out=None,
                   staging=None):
        """Host-buffer (end-to-end) run; `staging` is a CUDA uint8 scratch tensor."""
        import torch
        n_moves = int(proposals.shape[0])
        if staging is None:
            need = self._L.qmcd_sweep_host_min_staging(self.N, self.batch)
            staging = torch.empty(max(need, 64 << 20) + 256, dtype=torch.uint8, device="cuda")
        off = (-staging.data_ptr()) % 256
        _chk(self._L.qmcd_sweep_host(self._h, int(j_begin), n_moves,
                                     _ptr(proposals, torch.float64, "cpu"), _ptr(mask, torch.uint8, "cpu"),
                                     _ptr(uniforms, torch.float64, "cpu"), _ptr(R_out, torch.float64, "cpu"),
                                     _ptr(acc_out, torch.uint8, "cpu"),
                                     staging.data_ptr() + off, staging.numel() - off), "qmcd_sweep_host")

    def invert(self, A, Ainv=None, info=None):
        """Ainv[b] <- A[b]^-1 on the device (qmcd_invert); returns (Ainv, info [batch] int32).
        Does not adopt the result: call set_inverse(Ainv)."""
        import torch
        if tuple(A.shape) != (self.batch, self.N, self.N):
            raise ValueError("A must be [batch][N][N]")
        if Ainv is None:
            Ainv = torch.empty_like(A)
        if info is None:
            info = torch.empty(self.batch, dtype=torch.int32, device="cuda")
        need = self._L.qmcd_invert_scratch_bytes(self.N, self.batch)
        if need == 0:
            raise ValueError("qmcd_invert: N too large")
        scratch = torch.empty(need + 256, dtype=torch.uint8, device="cuda")
        off = (-scratch.data_ptr()) % 256
        _chk(self._L.qmcd_invert(self._h, _ptr(A, torch.float64), _ptr(Ainv, torch.float64),
                                 scratch.data_ptr() + off, need, _ptr(info, torch.int32)), "qmcd_invert")
        self._keep = scratch          # alive until the next call (the work is only enqueued)
        return Ainv, info

    def invert_static(self, A, Ainv, info):
        """qmcd_invert_static: the same inversion with the library's static device scratch (allocates nothing --
        neither does this wrapper: Ainv and info come from the caller).  Raises QmcdError(ELIMIT) past 1 MiB."""
        import torch
        if tuple(A.shape) != (self.batch, self.N, self.N) or tuple(Ainv.shape) != tuple(A.shape):
            raise ValueError("A and Ainv must be [batch][N][N]")
        _chk(self._L.qmcd_invert_static(self._h, _ptr(A, torch.float64), _ptr(Ainv, torch.float64),
                                        _ptr(info, torch.int32)), "qmcd_invert_static")

    def set_option(self, key: str, value: int):
        _chk(self._L.qmcd_set_option(self._h, key.encode(), int(value)), f"qmcd_set_option({key})")

    def get_option(self, key: str) -> int:
        return _chk(self._L.qmcd_get_option(self._h, key.encode()), f"qmcd_get_option({key})")
