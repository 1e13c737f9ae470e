"""Thin ctypes binding of libapd_b200.so (include/apd.h).  Argument marshalling only: every step
of the path runs in the library's CUDA kernels.  PyTorch supplies device memory and the stream.

There is NO fallback: if the shared library is missing or fails to load, importing a compute
entry point raises.  This module never imports ``oracle/``.
"""
from __future__ import annotations

import ctypes
import dataclasses
import os
from typing import Optional, Sequence

import torch

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libapd_b200.so")

APD_OK = 0
APD_NOT_CONVERGED = 1
APD_E_ARG = -1
APD_E_CUDA = -2
APD_E_ARCH = -3

KERNEL_AUTO = 0
KERNEL_DIRECT = 1
KERNEL_ROWPOLY = 2
KERNEL_TENSOR = 3
BAD_X_NONFINITE, BAD_A_NONFINITE, BAD_A_NOT_SYMMETRIC, BAD_A_NOT_POSITIVE_DEFINITE = 1, 2, 4, 8
BAD_W_NONFINITE, BAD_TARGET_VOL_NOT_POSITIVE, BAD_TARGET_VOL_SUM = 16, 32, 64


class ApdError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"libapd_b200 status {status}: {msg}")
        self.status = status


class apd_grid(ctypes.Structure):
    _fields_ = [("dim", ctypes.c_int32), ("n", ctypes.c_int32 * 3),
                ("lo", ctypes.c_double * 3), ("hi", ctypes.c_double * 3)]


class apd_opts(ctypes.Structure):
    _fields_ = [("kernel", ctypes.c_int32), ("cull", ctypes.c_int32), ("lbfgs_history", ctypes.c_int32),
                ("max_iters", ctypes.c_int32), ("max_evals", ctypes.c_int32), ("reserved", ctypes.c_int32 * 3)]


class apd_slab(ctypes.Structure):
    _fields_ = [("lo", ctypes.c_int32), ("n", ctypes.c_int32)]


REDUCE_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p)      # apd_reduce_fn(user, cuda_stream)

_lib = None
_P = ctypes.c_void_p


def load_library() -> ctypes.CDLL:
    """Loads libapd_b200.so; raises (never falls back) when it is absent."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2403_03571_b200.build` "
                          "(there is no CPU or PyTorch fallback)")
    lib = ctypes.CDLL(LIB_PATH)
    lib.apd_default_opts.restype = None
    lib.apd_default_opts.argtypes = [ctypes.POINTER(apd_opts)]
    lib.apd_create.restype = ctypes.c_int
    lib.apd_create.argtypes = [ctypes.POINTER(_P), ctypes.c_int32, ctypes.c_int32, ctypes.c_int32]
    lib.apd_destroy.restype = None
    lib.apd_destroy.argtypes = [_P]
    lib.apd_last_error.restype = ctypes.c_char_p
    lib.apd_last_error.argtypes = [_P]
    lib.apd_assign.restype = ctypes.c_int
    lib.apd_assign.argtypes = [_P, ctypes.POINTER(apd_grid), ctypes.c_int32] + [_P] * 10 + [ctypes.POINTER(apd_opts), _P]
    lib.apd_solve.restype = ctypes.c_int
    lib.apd_solve.argtypes = ([_P, ctypes.POINTER(apd_grid), ctypes.c_int32, _P, _P, _P, ctypes.c_double]
                              + [_P] * 5 + [ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32),
                                            ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double),
                                            ctypes.POINTER(apd_opts), _P])
    lib.apd_assign_host.restype = ctypes.c_int
    lib.apd_assign_host.argtypes = [_P, ctypes.POINTER(apd_grid), ctypes.c_int32] + [_P] * 10 + [ctypes.POINTER(apd_opts)]
    lib.apd_solve_host.restype = ctypes.c_int
    lib.apd_solve_host.argtypes = ([_P, ctypes.POINTER(apd_grid), ctypes.c_int32, _P, _P, _P, ctypes.c_double]
                                   + [_P] * 5 + [ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32),
                                                 ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double),
                                                 ctypes.POINTER(apd_opts)])
    lib.apd_assign_points.restype = ctypes.c_int
    lib.apd_assign_points.argtypes = [_P, ctypes.c_int64, _P, _P, ctypes.c_int32] + [_P] * 10
    lib.apd_solve_points.restype = ctypes.c_int
    lib.apd_solve_points.argtypes = ([_P, ctypes.c_int64, _P, _P, ctypes.c_double, ctypes.c_int32, _P, _P, _P,
                                      ctypes.c_double] + [_P] * 4
                                     + [ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32),
                                        ctypes.POINTER(ctypes.c_double), ctypes.POINTER(apd_opts), _P])
    lib.apd_solve_stats.restype = ctypes.c_int
    lib.apd_solve_stats.argtypes = [_P, ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32)]
    lib.apd_lloyd.restype = ctypes.c_int
    lib.apd_lloyd.argtypes = ([_P, ctypes.POINTER(apd_grid), ctypes.c_int32, _P, _P, _P, ctypes.c_double, ctypes.c_int32]
                              + [_P] * 4 + [ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32),
                                            ctypes.POINTER(ctypes.c_double), ctypes.POINTER(apd_opts), _P])
    lib.apd_solve_refine.restype = ctypes.c_int
    lib.apd_solve_refine.argtypes = ([_P, ctypes.POINTER(apd_grid), ctypes.c_int32, _P, _P, _P, ctypes.c_double, ctypes.c_int32]
                                     + [_P] * 3 + [ctypes.POINTER(ctypes.c_int32)] * 3
                                     + [ctypes.POINTER(ctypes.c_double), ctypes.POINTER(apd_opts), _P])
    lib.apd_solve_continuation.restype = ctypes.c_int
    lib.apd_solve_continuation.argtypes = ([_P, ctypes.POINTER(apd_grid), ctypes.c_int32, ctypes.c_int32, _P, _P, _P,
                                            ctypes.c_double] + [_P] * 4
                                           + [ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32),
                                              ctypes.POINTER(ctypes.c_double), ctypes.POINTER(apd_opts), _P])
    lib.apd_resolution_bound.restype = ctypes.c_double
    lib.apd_resolution_bound.argtypes = [ctypes.c_int32, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int32]
    lib.apd_choose_resolution.restype = ctypes.c_int32
    lib.apd_choose_resolution.argtypes = [ctypes.c_int32, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int32]
    lib.apd_solve_history.restype = ctypes.c_int
    lib.apd_solve_history.argtypes = [_P, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double), ctypes.c_int32]
    lib.apd_slab_align.restype = ctypes.c_int32
    lib.apd_slab_align.argtypes = [ctypes.c_int32]
    lib.apd_counter_words.restype = ctypes.c_int64
    lib.apd_counter_words.argtypes = [ctypes.POINTER(apd_grid), ctypes.c_int32, ctypes.c_int32]
    lib.apd_assign_slab.restype = ctypes.c_int
    lib.apd_assign_slab.argtypes = ([_P, ctypes.POINTER(apd_grid), ctypes.POINTER(apd_slab), ctypes.c_int32] + [_P] * 5
                                    + [ctypes.c_int32, ctypes.POINTER(apd_opts), _P])
    lib.apd_finalize_counters.restype = ctypes.c_int
    lib.apd_finalize_counters.argtypes = [_P, ctypes.POINTER(apd_grid), ctypes.c_int32, _P, ctypes.c_int32] + [_P] * 8
    lib.apd_solve_slab.restype = ctypes.c_int
    lib.apd_solve_slab.argtypes = ([_P, ctypes.POINTER(apd_grid), ctypes.POINTER(apd_slab), ctypes.c_int32, _P, _P, _P,
                                    ctypes.c_double] + [_P] * 5 + [REDUCE_FN, _P, ctypes.POINTER(ctypes.c_int32),
                                                                   ctypes.POINTER(ctypes.c_int32),
                                                                   ctypes.POINTER(ctypes.c_double),
                                                                   ctypes.POINTER(ctypes.c_double),
                                                                   ctypes.POINTER(apd_opts), _P])
    lib.apd_reserve.restype = ctypes.c_int
    lib.apd_reserve.argtypes = [_P, ctypes.POINTER(apd_grid), ctypes.POINTER(apd_opts)]
    lib.apd_assign_stats.restype = ctypes.c_int
    lib.apd_assign_stats.argtypes = [_P] + [ctypes.POINTER(ctypes.c_int32)] * 4 + [ctypes.POINTER(ctypes.c_double)]
    lib.apd_assign_static.restype = ctypes.c_int
    lib.apd_assign_static.argtypes = [ctypes.POINTER(apd_grid), ctypes.c_int32] + [_P] * 9
    lib.apd_static_scratch_bytes.restype = ctypes.c_int64
    lib.apd_static_scratch_bytes.argtypes = []
    lib.apd_static_last_error.restype = ctypes.c_char_p
    lib.apd_static_last_error.argtypes = []
    lib.apd_lloyd_points.restype = ctypes.c_int
    lib.apd_lloyd_points.argtypes = ([_P, ctypes.c_int64, _P, _P, ctypes.c_double, ctypes.c_int32, _P, _P, _P,
                                      ctypes.c_double, ctypes.c_int32] + [_P] * 4 +
                                     [ctypes.POINTER(ctypes.c_int32), ctypes.POINTER(ctypes.c_int32),
                                      ctypes.POINTER(ctypes.c_double), ctypes.POINTER(apd_opts), _P])
    lib.apd_validate.restype = ctypes.c_int
    lib.apd_validate.argtypes = [_P, ctypes.POINTER(apd_grid), ctypes.c_int32, _P, _P, _P, _P,
                                 ctypes.POINTER(ctypes.c_uint32), _P]
    _lib = lib
    return lib


EXPORTED_SYMBOLS = ["apd_default_opts", "apd_create", "apd_destroy", "apd_last_error", "apd_assign", "apd_solve",
                    "apd_assign_host", "apd_solve_host", "apd_solve_history", "apd_assign_points", "apd_solve_points", "apd_solve_stats", "apd_lloyd", "apd_solve_refine", "apd_resolution_bound",
                    "apd_choose_resolution", "apd_reserve", "apd_assign_stats", "apd_slab_align", "apd_counter_words",
                    "apd_assign_slab", "apd_finalize_counters", "apd_solve_slab", "apd_solve_continuation",
                    "apd_assign_static", "apd_static_scratch_bytes", "apd_static_last_error", "apd_validate", "apd_lloyd_points"]


def make_grid(dim: int, n: Sequence[int], lo: Sequence[float], hi: Sequence[float]) -> apd_grid:
    g = apd_grid()
    g.dim = dim
    for k in range(3):
        g.n[k] = int(n[k]) if k < dim else 1
        g.lo[k] = float(lo[k]) if k < dim else 0.0
        g.hi[k] = float(hi[k]) if k < dim else 1.0
    return g


def slab_align(dim: int) -> int:
    return int(load_library().apd_slab_align(dim))


def counter_words(grid: apd_grid, M: int, with_idxsum: bool = False) -> int:
    return int(load_library().apd_counter_words(ctypes.byref(grid), M, int(with_idxsum)))


def slab_partition(n_last: int, world: int, align: int):
    """Splits the n_last planes of a grid's last axis into `world` contiguous slabs whose boundaries are multiples of
    `align` (apd_slab_align), as evenly as the alignment allows.  Returns [(lo, n)] per rank.  Needs at least one layer
    of `align` planes per rank."""
    layers = (n_last + align - 1) // align
    if layers < world:
        raise ValueError(f"{n_last} planes are {layers} layers of {align}: fewer than the {world} ranks")
    out, lo = [], 0
    for r in range(world):
        nl = layers // world + (1 if r < layers % world else 0)
        n = min(nl * align, n_last - lo)
        out.append((lo, max(n, 0)))
        lo += max(n, 0)
    return out


def make_opts(kernel: int = KERNEL_AUTO, cull: int = 0, lbfgs_history: int = 10, max_iters: int = 1000,
              max_evals: int = 0) -> apd_opts:
    o = apd_opts()
    load_library().apd_default_opts(ctypes.byref(o))
    o.kernel, o.cull, o.lbfgs_history, o.max_iters, o.max_evals = kernel, cull, lbfgs_history, max_iters, max_evals
    return o


def _dev(t: Optional[torch.Tensor], dtype, name: str, numel: Optional[int] = None):
    if t is None:
        return None
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous CUDA tensor of dtype {dtype}")
    if numel is not None and t.numel() != numel:
        raise ValueError(f"{name}: expected {numel} elements, got {t.numel()}")
    return ctypes.c_void_p(t.data_ptr())


def _host(a, dtype, name: str, numel: Optional[int] = None):
    if a is None:
        return None
    if not (isinstance(a, torch.Tensor) and not a.is_cuda and a.dtype == dtype and a.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous CPU tensor of dtype {dtype}")
    if numel is not None and a.numel() != numel:
        raise ValueError(f"{name}: expected {numel} elements, got {a.numel()}")
    return ctypes.c_void_p(a.data_ptr())


@dataclasses.dataclass
class SolveInfo:
    status: int
    iters: int
    evals: int
    max_rel_err: float
    dual: float


class ApdContext:
    """Owns an apd_ctx (workspace on one B200)."""

    def __init__(self, dim: int, max_seeds: int, device: int = 0):
        self._lib = load_library()
        self._h = _P()
        rc = self._lib.apd_create(ctypes.byref(self._h), dim, max_seeds, device)
        if rc != APD_OK:
            raise ApdError(rc, (self._lib.apd_last_error(None) or b"").decode())
        self.dim, self.max_seeds, self.device = dim, max_seeds, device

    def close(self):
        if getattr(self, "_h", None):
            self._lib.apd_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc: int, allow=(APD_OK,)):
        if rc not in allow:
            raise ApdError(rc, (self._lib.apd_last_error(self._h) or b"").decode())
        return rc

    def _stream(self):
        return ctypes.c_void_p(torch.cuda.current_stream(self.device).cuda_stream)

    # -- device-pointer calls -----------------------------------------------------------------
    def apd_assign(self, grid: apd_grid, X, A, w, target_vol=None, labels=None, vol=None, dual=None,
                   max_rel_err=None, centroids=None, pairs_evaluated=None, opts: Optional[apd_opts] = None):
        """apd_assign of include/apd.h on CUDA tensors; asynchronous on torch's current stream."""
        d = grid.dim
        M = X.shape[0]
        rc = self._lib.apd_assign(
            self._h, ctypes.byref(grid), M, _dev(X, torch.float32, "X", M * d), _dev(A, torch.float32, "A", M * d * d),
            _dev(w, torch.float32, "w", M), _dev(target_vol, torch.float32, "target_vol", M),
            _dev(labels, torch.int32, "labels"), _dev(vol, torch.float64, "vol", M),
            _dev(dual, torch.float64, "dual", 1), _dev(max_rel_err, torch.float64, "max_rel_err", 1),
            _dev(centroids, torch.float64, "centroids", M * d), _dev(pairs_evaluated, torch.int64, "pairs_evaluated", 1),
            ctypes.byref(opts) if opts is not None else None, self._stream())
        self._check(rc)

    def apd_assign_points(self, Y, pvol, X, A, w, target_vol=None, labels=None, vol=None, dual=None,
                          max_rel_err=None, centroids=None):
        """apd_assign_points of include/apd.h on CUDA tensors (user-supplied points and volumes)."""
        d = self.dim
        N, M = Y.shape[0], X.shape[0]
        rc = self._lib.apd_assign_points(
            self._h, N, _dev(Y, torch.float32, "Y", N * d), _dev(pvol, torch.float32, "pvol", N), M,
            _dev(X, torch.float32, "X", M * d), _dev(A, torch.float32, "A", M * d * d), _dev(w, torch.float32, "w", M),
            _dev(target_vol, torch.float32, "target_vol", M), _dev(labels, torch.int32, "labels", N),
            _dev(vol, torch.float64, "vol", M), _dev(dual, torch.float64, "dual", 1),
            _dev(max_rel_err, torch.float64, "max_rel_err", 1), _dev(centroids, torch.float64, "centroids", M * d),
            self._stream())
        self._check(rc)

    def apd_solve_points(self, Y, pvol, total_volume: float, X, A, target_vol, tol: float, w_init=None, w=None,
                         labels=None, vol=None, opts: Optional[apd_opts] = None) -> SolveInfo:
        """apd_solve_points of include/apd.h on CUDA tensors; blocks until finished."""
        d = self.dim
        N, M = Y.shape[0], X.shape[0]
        it, ev = ctypes.c_int32(0), ctypes.c_int32(0)
        err = ctypes.c_double(0.0)
        rc = self._lib.apd_solve_points(
            self._h, N, _dev(Y, torch.float32, "Y", N * d), _dev(pvol, torch.float32, "pvol", N), float(total_volume), M,
            _dev(X, torch.float32, "X", M * d), _dev(A, torch.float32, "A", M * d * d),
            _dev(target_vol, torch.float32, "target_vol", M), float(tol), _dev(w_init, torch.float32, "w_init", M),
            _dev(w, torch.float32, "w", M), _dev(labels, torch.int32, "labels", N), _dev(vol, torch.float64, "vol", M),
            ctypes.byref(it), ctypes.byref(ev), ctypes.byref(err), ctypes.byref(opts) if opts is not None else None,
            self._stream())
        self._check(rc, allow=(APD_OK, APD_NOT_CONVERGED))
        return SolveInfo(rc, it.value, ev.value, err.value, float("nan"))

    def apd_solve(self, grid: apd_grid, X, A, target_vol, tol: float, w_init=None, w=None, labels=None, vol=None,
                  w64=None, opts: Optional[apd_opts] = None) -> SolveInfo:
        """apd_solve of include/apd.h on CUDA tensors; blocks until finished."""
        d = grid.dim
        M = X.shape[0]
        it, ev = ctypes.c_int32(0), ctypes.c_int32(0)
        err, dual = ctypes.c_double(0.0), ctypes.c_double(0.0)
        rc = self._lib.apd_solve(
            self._h, ctypes.byref(grid), M, _dev(X, torch.float32, "X", M * d), _dev(A, torch.float32, "A", M * d * d),
            _dev(target_vol, torch.float32, "target_vol", M), float(tol), _dev(w_init, torch.float32, "w_init", M),
            _dev(w, torch.float32, "w", M), _dev(labels, torch.int32, "labels"), _dev(vol, torch.float64, "vol", M),
            _dev(w64, torch.float64, "w64", M), ctypes.byref(it), ctypes.byref(ev), ctypes.byref(err),
            ctypes.byref(dual), ctypes.byref(opts) if opts is not None else None, self._stream())
        self._check(rc, allow=(APD_OK, APD_NOT_CONVERGED))
        return SolveInfo(rc, it.value, ev.value, err.value, dual.value)

    # -- voxel-slab sharding (f4) ---------------------------------------------------------------
    def apd_assign_slab(self, grid: apd_grid, slab, X, A, w, labels=None, counters=None, with_idxsum: bool = False,
                        opts: Optional[apd_opts] = None):
        """apd_assign_slab of include/apd.h: raw counters of planes [lo, lo + n) of the last axis (slab = (lo, n));
        counters: CUDA int64 tensor of counter_words(grid, M, with_idxsum) words."""
        d = grid.dim
        M = X.shape[0]
        sl = apd_slab(int(slab[0]), int(slab[1]))
        rc = self._lib.apd_assign_slab(
            self._h, ctypes.byref(grid), ctypes.byref(sl), M, _dev(X, torch.float32, "X", M * d),
            _dev(A, torch.float32, "A", M * d * d), _dev(w, torch.float32, "w", M), _dev(labels, torch.int32, "labels"),
            _dev(counters, torch.int64, "counters", counter_words(grid, M, with_idxsum)), int(with_idxsum),
            ctypes.byref(opts) if opts is not None else None, self._stream())
        self._check(rc)

    def apd_finalize_counters(self, grid: apd_grid, counters, X, w, target_vol=None, vol=None, dual=None,
                              max_rel_err=None, centroids=None, with_idxsum: bool = False):
        """apd_finalize_counters of include/apd.h: vol / dual / error / centroids from REDUCED counters."""
        d = grid.dim
        M = X.shape[0]
        rc = self._lib.apd_finalize_counters(
            self._h, ctypes.byref(grid), M, _dev(counters, torch.int64, "counters", counter_words(grid, M, with_idxsum)),
            int(with_idxsum), _dev(X, torch.float32, "X", M * d), _dev(w, torch.float32, "w", M),
            _dev(target_vol, torch.float32, "target_vol", M), _dev(vol, torch.float64, "vol", M),
            _dev(dual, torch.float64, "dual", 1), _dev(max_rel_err, torch.float64, "max_rel_err", 1),
            _dev(centroids, torch.float64, "centroids", M * d), self._stream())
        self._check(rc)

    def apd_solve_slab(self, grid: apd_grid, slab, X, A, target_vol, tol: float, counters, reduce=None, w_init=None,
                       w=None, labels=None, vol=None, opts: Optional[apd_opts] = None) -> SolveInfo:
        """apd_solve_slab of include/apd.h.  `reduce`: a Python callable () -> None that sums `counters` (CUDA int64
        tensor, counter_words(grid, M) words) over all ranks in place, in order with torch's current stream -- e.g.
        lambda: torch.distributed.all_reduce(counters).  Blocks until finished."""
        d = grid.dim
        M = X.shape[0]
        sl = apd_slab(int(slab[0]), int(slab[1]))
        it, ev = ctypes.c_int32(0), ctypes.c_int32(0)
        err, dual = ctypes.c_double(0.0), ctypes.c_double(0.0)
        failure = []

        def _cb(user, stream):
            try:
                reduce()
                return 0
            except Exception as e:        # an exception must not cross the C ABI
                failure.append(e)
                return 1
        cb = REDUCE_FN(_cb) if reduce is not None else ctypes.cast(None, REDUCE_FN)
        rc = self._lib.apd_solve_slab(
            self._h, ctypes.byref(grid), ctypes.byref(sl), M, _dev(X, torch.float32, "X", M * d),
            _dev(A, torch.float32, "A", M * d * d), _dev(target_vol, torch.float32, "target_vol", M), float(tol),
            _dev(w_init, torch.float32, "w_init", M), _dev(w, torch.float32, "w", M), _dev(labels, torch.int32, "labels"),
            _dev(vol, torch.float64, "vol", M), _dev(counters, torch.int64, "counters", counter_words(grid, M, False)),
            cb, None, ctypes.byref(it), ctypes.byref(ev), ctypes.byref(err), ctypes.byref(dual),
            ctypes.byref(opts) if opts is not None else None, self._stream())
        if failure:
            raise failure[0]
        self._check(rc, allow=(APD_OK, APD_NOT_CONVERGED))
        return SolveInfo(rc, it.value, ev.value, err.value, dual.value)

    # -- host-pointer calls -------------------------------------------------------------------
    def apd_assign_host(self, grid: apd_grid, X, A, w, target_vol=None, labels=None, vol=None, centroids=None,
                        opts: Optional[apd_opts] = None):
        """apd_assign_host on CPU tensors (pinned or not); returns (dual, max_rel_err, pairs)."""
        d = grid.dim
        M = X.shape[0]
        dual, err = ctypes.c_double(0.0), ctypes.c_double(0.0)
        pairs = ctypes.c_uint64(0)
        rc = self._lib.apd_assign_host(
            self._h, ctypes.byref(grid), M, _host(X, torch.float32, "X", M * d), _host(A, torch.float32, "A", M * d * d),
            _host(w, torch.float32, "w", M), _host(target_vol, torch.float32, "target_vol", M),
            _host(labels, torch.int32, "labels"), _host(vol, torch.float64, "vol", M),
            ctypes.cast(ctypes.byref(dual), _P), ctypes.cast(ctypes.byref(err), _P),
            _host(centroids, torch.float64, "centroids", M * d), ctypes.cast(ctypes.byref(pairs), _P),
            ctypes.byref(opts) if opts is not None else None)
        self._check(rc)
        return dual.value, err.value, pairs.value

    def apd_solve_host(self, grid: apd_grid, X, A, target_vol, tol: float, w_init=None, w=None, labels=None,
                       vol=None, w64=None, opts: Optional[apd_opts] = None) -> SolveInfo:
        d = grid.dim
        M = X.shape[0]
        it, ev = ctypes.c_int32(0), ctypes.c_int32(0)
        err, dual = ctypes.c_double(0.0), ctypes.c_double(0.0)
        rc = self._lib.apd_solve_host(
            self._h, ctypes.byref(grid), M, _host(X, torch.float32, "X", M * d), _host(A, torch.float32, "A", M * d * d),
            _host(target_vol, torch.float32, "target_vol", M), float(tol), _host(w_init, torch.float32, "w_init", M),
            _host(w, torch.float32, "w", M), _host(labels, torch.int32, "labels"), _host(vol, torch.float64, "vol", M),
            _host(w64, torch.float64, "w64", M), ctypes.byref(it), ctypes.byref(ev), ctypes.byref(err),
            ctypes.byref(dual), ctypes.byref(opts) if opts is not None else None)
        self._check(rc, allow=(APD_OK, APD_NOT_CONVERGED))
        return SolveInfo(rc, it.value, ev.value, err.value, dual.value)

    def apd_lloyd(self, grid: apd_grid, X, A, target_vol, tol: float, K: int, w_init=None, w=None, labels=None,
                  vol=None, opts: Optional[apd_opts] = None) -> SolveInfo:
        """apd_lloyd of include/apd.h (Algorithm 3) on CUDA tensors; X is updated in place; blocks until finished."""
        d = grid.dim
        M = X.shape[0]
        it, ev = ctypes.c_int32(0), ctypes.c_int32(0)
        err = ctypes.c_double(0.0)
        rc = self._lib.apd_lloyd(
            self._h, ctypes.byref(grid), M, _dev(X, torch.float32, "X", M * d), _dev(A, torch.float32, "A", M * d * d),
            _dev(target_vol, torch.float32, "target_vol", M), float(tol), int(K),
            _dev(w_init, torch.float32, "w_init", M), _dev(w, torch.float32, "w", M), _dev(labels, torch.int32, "labels"),
            _dev(vol, torch.float64, "vol", M), ctypes.byref(it), ctypes.byref(ev), ctypes.byref(err),
            ctypes.byref(opts) if opts is not None else None, self._stream())
        self._check(rc, allow=(APD_OK, APD_NOT_CONVERGED))
        return SolveInfo(rc, it.value, ev.value, err.value, float("nan"))

    def apd_lloyd_points(self, Y, pvol, total_volume: float, X, A, target_vol, tol: float, K: int, w_init=None, w=None,
                         labels=None, vol=None, opts: Optional[apd_opts] = None) -> SolveInfo:
        """apd_lloyd_points of include/apd.h (Algorithm 3 on points with element volumes); X is updated in place."""
        d = self.dim
        N, M = int(Y.shape[0]), int(X.shape[0])
        it, ev = ctypes.c_int32(0), ctypes.c_int32(0)
        err = ctypes.c_double(0.0)
        rc = self._lib.apd_lloyd_points(
            self._h, N, _dev(Y, torch.float32, "Y", N * d), _dev(pvol, torch.float32, "pvol", N), float(total_volume), M,
            _dev(X, torch.float32, "X", M * d), _dev(A, torch.float32, "A", M * d * d),
            _dev(target_vol, torch.float32, "target_vol", M), float(tol), int(K),
            _dev(w_init, torch.float32, "w_init", M), _dev(w, torch.float32, "w", M),
            _dev(labels, torch.int32, "labels", N), _dev(vol, torch.float64, "vol", M), ctypes.byref(it), ctypes.byref(ev),
            ctypes.byref(err), ctypes.byref(opts) if opts is not None else None, self._stream())
        self._check(rc, allow=(APD_OK, APD_NOT_CONVERGED))
        return SolveInfo(rc, it.value, ev.value, err.value, float("nan"))

    def apd_solve_refine(self, grid: apd_grid, X, A, target_vol, tol: float, max_refinements: int, w_init=None,
                         w=None, vol=None, opts: Optional[apd_opts] = None):
        """apd_solve_refine of include/apd.h (Algorithm 2 incl. step 4); `grid.n` is updated in place.
        Returns (SolveInfo, refinements)."""
        d = grid.dim
        M = X.shape[0]
        rf, it, ev = ctypes.c_int32(0), ctypes.c_int32(0), ctypes.c_int32(0)
        err = ctypes.c_double(0.0)
        rc = self._lib.apd_solve_refine(
            self._h, ctypes.byref(grid), M, _dev(X, torch.float32, "X", M * d), _dev(A, torch.float32, "A", M * d * d),
            _dev(target_vol, torch.float32, "target_vol", M), float(tol), int(max_refinements),
            _dev(w_init, torch.float32, "w_init", M), _dev(w, torch.float32, "w", M), _dev(vol, torch.float64, "vol", M),
            ctypes.byref(rf), ctypes.byref(it), ctypes.byref(ev), ctypes.byref(err),
            ctypes.byref(opts) if opts is not None else None, self._stream())
        self._check(rc, allow=(APD_OK, APD_NOT_CONVERGED))
        return SolveInfo(rc, it.value, ev.value, err.value, float("nan")), rf.value

    def apd_solve_continuation(self, grid: apd_grid, levels: int, X, A, target_vol, tol: float, w_init=None, w=None,
                               labels=None, vol=None, opts: Optional[apd_opts] = None):
        """apd_solve_continuation of include/apd.h.  Returns (status, iters per level, evals per level, max_rel_err),
        coarsest level first."""
        d = grid.dim
        M = X.shape[0]
        it = (ctypes.c_int32 * (levels + 1))()
        ev = (ctypes.c_int32 * (levels + 1))()
        err = ctypes.c_double(0.0)
        rc = self._lib.apd_solve_continuation(
            self._h, ctypes.byref(grid), int(levels), M, _dev(X, torch.float32, "X", M * d),
            _dev(A, torch.float32, "A", M * d * d), _dev(target_vol, torch.float32, "target_vol", M), float(tol),
            _dev(w_init, torch.float32, "w_init", M), _dev(w, torch.float32, "w", M), _dev(labels, torch.int32, "labels"),
            _dev(vol, torch.float64, "vol", M), it, ev, ctypes.byref(err),
            ctypes.byref(opts) if opts is not None else None, self._stream())
        self._check(rc, allow=(APD_OK, APD_NOT_CONVERGED))
        return rc, list(it), list(ev), err.value

    def solve_stats(self):
        """(evaluations recorded, candidate-list rebuilds) of the most recent apd_solve."""
        n, r = ctypes.c_int32(0), ctypes.c_int32(0)
        self._check(self._lib.apd_solve_stats(self._h, ctypes.byref(n), ctypes.byref(r)))
        return n.value, r.value

    def solve_history(self, cap: int = 8192):
        """(dual, max_rel_err) numpy arrays, one entry per evaluation of the most recent apd_solve."""
        import numpy as np
        d = (ctypes.c_double * cap)()
        e = (ctypes.c_double * cap)()
        n = self._lib.apd_solve_history(self._h, d, e, cap)
        if n < 0:
            self._check(n)
        return np.array(d[:n], dtype=np.float64), np.array(e[:n], dtype=np.float64)

    def validate(self, grid: Optional[apd_grid], X, A, w=None, target_vol=None) -> int:
        """apd_validate of include/apd.h: 0, or the OR of the BAD_* flags."""
        M, d = int(X.shape[0]), self.dim
        out = ctypes.c_uint32(0)
        self._check(self._lib.apd_validate(self._h, ctypes.byref(grid) if grid is not None else None, M,
                                           _dev(X, torch.float32, "X", M * d), _dev(A, torch.float32, "A", M * d * d),
                                           _dev(w, torch.float32, "w", M), _dev(target_vol, torch.float32, "target_vol", M),
                                           ctypes.byref(out), self._stream()))
        return int(out.value)

    def reserve(self, grid: apd_grid, opts: Optional[apd_opts] = None):
        """apd_reserve of include/apd.h: grow the workspace ahead of time."""
        self._check(self._lib.apd_reserve(self._h, ctypes.byref(grid), ctypes.byref(opts) if opts is not None else None))

    def assign_stats(self) -> dict:
        """apd_assign_stats of include/apd.h: what the most recent evaluation launched."""
        k, rl, cu, nt = (ctypes.c_int32(0) for _ in range(4))
        ms = ctypes.c_double(0.0)
        self._check(self._lib.apd_assign_stats(self._h, ctypes.byref(k), ctypes.byref(rl), ctypes.byref(cu),
                                               ctypes.byref(nt), ctypes.byref(ms)))
        return dict(kernel=k.value, row_long=rl.value, cull=cu.value, n_tiles=nt.value, kernel_ms=ms.value)

    def last_kernel_ms(self) -> float:
        return float(self.assign_stats()["kernel_ms"])


STATIC_MAX_SEEDS = 4096        # APD_STATIC_MAX_SEEDS of include/apd.h
STATIC_MAX_TILES = 16384       # APD_STATIC_MAX_TILES


def apd_assign_static(grid: apd_grid, X, A, w, target_vol=None, labels=None, vol=None, dual=None, max_rel_err=None):
    """apd_assign_static of include/apd.h on CUDA tensors: no context, no allocation; runs on X's device (made
    current for the call), asynchronously on torch's current stream of that device."""
    lib = load_library()
    d, M = grid.dim, X.shape[0]
    with torch.cuda.device(X.device):
        rc = lib.apd_assign_static(
            ctypes.byref(grid), M, _dev(X, torch.float32, "X", M * d), _dev(A, torch.float32, "A", M * d * d),
            _dev(w, torch.float32, "w", M), _dev(target_vol, torch.float32, "target_vol", M),
            _dev(labels, torch.int32, "labels"), _dev(vol, torch.float64, "vol", M),
            _dev(dual, torch.float64, "dual", 1), _dev(max_rel_err, torch.float64, "max_rel_err", 1),
            ctypes.c_void_p(torch.cuda.current_stream(X.device).cuda_stream))
    if rc != APD_OK:
        raise ApdError(rc, (lib.apd_static_last_error() or b"").decode())


def static_scratch_bytes() -> int:
    return int(load_library().apd_static_scratch_bytes())


def apd_resolution_bound(dim: int, domain_volume: float, v_min: float, eps: float, practical: bool) -> float:
    return float(load_library().apd_resolution_bound(dim, domain_volume, v_min, eps, int(practical)))


def apd_choose_resolution(dim: int, domain_volume: float, v_min: float, eps: float, practical: bool) -> int:
    return int(load_library().apd_choose_resolution(dim, domain_volume, v_min, eps, int(practical)))
