"""paper_1204_6630_b200 -- thin Python binding of libtpcf.so (include/tpcf.h).

Argument marshalling only: every step of the path (RA/Dec -> unit vectors, pair distances, binning,
histogram merge) runs in the CUDA kernels behind the C ABI; the estimator is the library's own host
arithmetic.  The functions carry the names of the C entry points.  PyTorch is used here only for device
memory (CUDA tensors handed in by pointer) and streams.  There is no CPU fallback: if libtpcf.so cannot be
built or loaded this module raises, and every compute call fails with TpcfError(TPCF_ECUDA) without a GPU.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Tuple

import numpy as np

from . import build as _build

TPCF_OK, TPCF_EINVAL, TPCF_ENOMEM, TPCF_ECUDA, TPCF_ESTATE = 0, 1, 2, 3, 4
TPCF_LINEAR, TPCF_LOG, TPCF_EXPLICIT = 0, 1, 2
TPCF_D, TPCF_R, TPCF_D2 = 0, 1, 2
TPCF_F32, TPCF_F64 = 0, 1
TPCF_DD, TPCF_DR, TPCF_RR, TPCF_D1D2, TPCF_D2R = 0, 1, 2, 3, 4
TPCF_ENGINE_FAST, TPCF_ENGINE_EXACT64, TPCF_ENGINE_TENSOR = 0, 1, 2
_STATUS = {0: "TPCF_OK", 1: "TPCF_EINVAL", 2: "TPCF_ENOMEM", 3: "TPCF_ECUDA", 4: "TPCF_ESTATE"}
_MODES = {"linear": TPCF_LINEAR, "log": TPCF_LOG, "explicit": TPCF_EXPLICIT}
_KINDS = {"DD": TPCF_DD, "DR": TPCF_DR, "RR": TPCF_RR}
_ALL_KINDS = dict(_KINDS, D1D2=TPCF_D1D2, D2R=TPCF_D2R)
_CATS = {"D": TPCF_D, "R": TPCF_R, "D2": TPCF_D2}

# every symbol include/tpcf.h declares (tests check that the library exports them all)
EXPORTS = (
    "tpcf_create", "tpcf_get_edges", "tpcf_load", "tpcf_count", "tpcf_count_async", "tpcf_estimate",
    "tpcf_estimate_from", "tpcf_destroy", "tpcf_last_error", "tpcf_set_stream", "tpcf_set_engine",
    "tpcf_set_guard_scale", "tpcf_set_partition", "tpcf_get_stats", "tpcf_get_thresholds", "tpcf_classify_fast",
    "tpcf_plan", "tpcf_plan_item_pairs", "tpcf_set_kernel_timing", "tpcf_get_kernel_times", "tpcf_set_window",
    "tpcf_get_bands", "tpcf_window_host", "tpcf_tensor_probe", "tpcf_create_r", "tpcf_load_xyz", "tpcf_set_pruning", "tpcf_count_all", "tpcf_count_all_async",
    "tpcf_estimate_cross", "tpcf_set_weights", "tpcf_count_weighted", "tpcf_set_tensor_share_limit",
    "tpcf_count_static", "tpcf_count3",
)
TPCF_STATIC_MAX_ROWS, TPCF_STATIC_MAX_BINS = 65536, 4096
TPCF_COUNT3_MAX_ROWS, TPCF_COUNT3_MAX_BINS = 16384, 30


class TpcfError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS.get(status, status)}: {message}")
        self.status = status


class tpcf_stats(ctypes.Structure):
    _fields_ = [("pairs", ctypes.c_uint64), ("rechecked", ctypes.c_uint64), ("work_items", ctypes.c_uint64),
                ("launches", ctypes.c_int), ("grid", ctypes.c_int), ("block", ctypes.c_int),
                ("smem_bytes", ctypes.c_int), ("cells", ctypes.c_int), ("cell_bits", ctypes.c_int),
                ("kernel_ms", ctypes.c_float), ("win_blocks", ctypes.c_uint64 * 6),
                ("pruned_blocks", ctypes.c_uint64), ("lookup_share", ctypes.c_float)]

    def as_dict(self):
        d = {k: getattr(self, k) for k, _ in self._fields_}
        d["win_blocks"] = [int(x) for x in self.win_blocks]
        return d


_lib = None


def lib() -> ctypes.CDLL:
    """Load (building first if the sources are newer) the in-tree libtpcf.so.  Raises if that is impossible."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if _build.stale():
            path = _build.build()
        L = ctypes.CDLL(path)
        vp, i32, sz, u64, dbl = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t, ctypes.c_uint64, ctypes.c_double
        sig = {
            "tpcf_create": [ctypes.POINTER(vp), i32, vp, i32],
            "tpcf_create_r": [ctypes.POINTER(vp), i32, vp, i32, dbl],
            "tpcf_load_xyz": [vp, i32, vp, i32, sz, i32, vp],
            "tpcf_get_edges": [vp, vp],
            "tpcf_load": [vp, i32, vp, i32, sz, i32, vp],
            "tpcf_count": [vp, i32, vp, vp, vp, sz],
            "tpcf_count_async": [vp, i32, vp],
            "tpcf_count_all": [vp, vp, vp],
            "tpcf_count_all_async": [vp, vp],
            "tpcf_estimate": [vp, vp],
            "tpcf_estimate_cross": [vp, vp],
            "tpcf_set_weights": [vp, i32, vp, sz],
            "tpcf_count_weighted": [vp, i32, vp, vp],
            "tpcf_estimate_from": [vp, vp, vp, i32, u64, u64, vp],
            "tpcf_set_stream": [vp, vp],
            "tpcf_set_engine": [vp, i32],
            "tpcf_set_guard_scale": [vp, dbl],
            "tpcf_set_tensor_share_limit": [vp, dbl],
            "tpcf_set_window": [vp, i32],
            "tpcf_set_pruning": [vp, i32],
            "tpcf_get_bands": [vp, i32, vp, vp, vp, ctypes.POINTER(i32)],
            "tpcf_window_host": [vp, ctypes.c_float, ctypes.c_float, ctypes.POINTER(i32), ctypes.POINTER(i32)],
            "tpcf_tensor_probe": [vp, vp, vp, ctypes.c_size_t, vp],
            "tpcf_set_partition": [vp, i32, i32],
            "tpcf_get_stats": [vp, ctypes.POINTER(tpcf_stats)],
            "tpcf_set_kernel_timing": [vp, i32],
            "tpcf_get_kernel_times": [vp, vp, i32, ctypes.POINTER(i32)],
            "tpcf_get_thresholds": [vp, vp],
            "tpcf_classify_fast": [vp, ctypes.c_float, ctypes.POINTER(i32)],
            "tpcf_plan": [vp, i32, u64, u64, ctypes.POINTER(u64)],
            "tpcf_plan_item_pairs": [vp, i32, u64, u64, u64, ctypes.POINTER(u64)],
            "tpcf_count3": [vp, i32, vp],
            "tpcf_count_static": [i32, vp, i32, vp, sz, vp, sz, i32, vp, vp, ctypes.c_char_p, sz],
        }
        for name, args in sig.items():
            fn = getattr(L, name)
            fn.argtypes = args
            fn.restype = i32
        L.tpcf_destroy.argtypes = [vp]
        L.tpcf_destroy.restype = None
        L.tpcf_last_error.argtypes = [vp]
        L.tpcf_last_error.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _check(ctx, status: int):
    if status != TPCF_OK:
        msg = lib().tpcf_last_error(ctx).decode() if ctx else "invalid arguments"
        raise TpcfError(status, msg)


def _np_ptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def _is_torch(x) -> bool:
    return type(x).__module__.startswith("torch")


# ---- the C entry points, one Python function each --------------------------------------------------------
def tpcf_create(nbins: int, theta_deg, mode) -> ctypes.c_void_p:
    mode = _MODES.get(mode, mode)
    th = np.ascontiguousarray(theta_deg, dtype=np.float64)
    need = nbins + 1 if mode == TPCF_EXPLICIT else 2
    if th.ndim != 1 or th.shape[0] != need:
        raise TpcfError(TPCF_EINVAL, f"theta_deg must hold {need} values")
    ctx = ctypes.c_void_p()
    st = lib().tpcf_create(ctypes.byref(ctx), int(nbins), _np_ptr(th), int(mode))
    if st != TPCF_OK:
        raise TpcfError(st, "tpcf_create rejected the binning")
    return ctx


def tpcf_create_r(nbins: int, r_edges, mode, max_abs_coord: float) -> ctypes.c_void_p:
    mode = _MODES.get(mode, mode)
    e = np.ascontiguousarray(r_edges, dtype=np.float64)
    need = nbins + 1 if mode == TPCF_EXPLICIT else 2
    if e.ndim != 1 or e.shape[0] != need:
        raise TpcfError(TPCF_EINVAL, f"r_edges must hold {need} values")
    ctx = ctypes.c_void_p()
    st = lib().tpcf_create_r(ctypes.byref(ctx), int(nbins), _np_ptr(e), int(mode), float(max_abs_coord))
    if st != TPCF_OK:
        raise TpcfError(st, "tpcf_create_r rejected the binning")
    return ctx


def tpcf_destroy(ctx) -> None:
    lib().tpcf_destroy(ctx)


def tpcf_get_edges(ctx, nbins: int) -> np.ndarray:
    e = np.empty(nbins + 1, dtype=np.float64)
    _check(ctx, lib().tpcf_get_edges(ctx, _np_ptr(e)))
    return e


def tpcf_get_thresholds(ctx, nbins: int) -> np.ndarray:
    t = np.empty(nbins + 1, dtype=np.float64)
    _check(ctx, lib().tpcf_get_thresholds(ctx, _np_ptr(t)))
    return t


def tpcf_load_xyz(ctx, which: int, xyz, stream: int = 0) -> int:
    """xyz: (n, 3) float32/float64 numpy array, CPU torch tensor (pinned or not) or CUDA torch tensor."""
    return tpcf_load(ctx, which, xyz, stream, cols=3)


def tpcf_load(ctx, which: int, radec_deg, stream: int = 0, cols: int = 2) -> int:
    """radec_deg: (n, 2) float32/float64 numpy array, CPU torch tensor (pinned or not) or CUDA torch tensor."""
    if _is_torch(radec_deg):
        t = radec_deg
        if t.dim() != 2 or t.shape[1] != cols or not t.is_contiguous():
            raise TpcfError(TPCF_EINVAL, f"catalog must be a contiguous (n, {cols}) tensor")
        dt = {"torch.float32": TPCF_F32, "torch.float64": TPCF_F64}.get(str(t.dtype))
        if dt is None:
            raise TpcfError(TPCF_EINVAL, "catalog dtype must be float32 or float64")
        n, ptr, on_dev = t.shape[0], ctypes.c_void_p(t.data_ptr()), int(t.is_cuda)
        keep = t
    else:
        a = np.asarray(radec_deg)
        if a.dtype not in (np.float32, np.float64):
            raise TpcfError(TPCF_EINVAL, "catalog dtype must be float32 or float64")
        a = np.ascontiguousarray(a)
        if a.ndim != 2 or a.shape[1] != cols:
            raise TpcfError(TPCF_EINVAL, f"catalog must be an (n, {cols}) array")
        dt = TPCF_F32 if a.dtype == np.float32 else TPCF_F64
        n, ptr, on_dev, keep = a.shape[0], _np_ptr(a), 0, a
    fn = lib().tpcf_load_xyz if cols == 3 else lib().tpcf_load
    _check(ctx, fn(ctx, int(which), ptr, dt, n, on_dev, ctypes.c_void_p(stream)))
    del keep
    return n


def tpcf_count(ctx, kind: int, nbins: int, rows=None) -> Tuple[np.ndarray, int, int]:
    hist = np.zeros(nbins, dtype=np.uint64)
    uo = np.zeros(2, dtype=np.uint64)
    if rows is None:
        st = lib().tpcf_count(ctx, int(kind), _np_ptr(hist), _np_ptr(uo), None, 0)
    else:
        r = np.ascontiguousarray(rows, dtype=np.int64)
        st = lib().tpcf_count(ctx, int(kind), _np_ptr(hist), _np_ptr(uo), _np_ptr(r), r.shape[0])
    _check(ctx, st)
    return hist, int(uo[0]), int(uo[1])


def tpcf_count_async(ctx, kind: int, hist_dev_ptr: int) -> None:
    _check(ctx, lib().tpcf_count_async(ctx, int(kind), ctypes.c_void_p(hist_dev_ptr)))


def tpcf_count_static(nbins: int, theta_deg, mode, radec_i_dev_ptr: int, n_i: int, radec_j_dev_ptr: Optional[int], n_j: int,
                      dtype: int, hist_dev_ptr: int, stream_ptr: int = 0) -> None:
    """The count that never allocates device memory (include/tpcf.h): for callers whose GPU memory is already spoken for
    (a framework's pool owns it all, a fixed per-GPU budget) or who cannot take the device-wide stall of cudaMalloc.
    Inputs and the nbins + 2 uint64 output are DEVICE pointers the caller owns; radec_j_dev_ptr None/0 with n_j 0 counts
    the pairs i < j of the first catalog.  At most TPCF_STATIC_MAX_ROWS rows (n_i + n_j) and TPCF_STATIC_MAX_BINS bins;
    calls on one GPU must not overlap; returns when the stream has drained."""
    mode = _MODES.get(mode, mode)
    th = np.ascontiguousarray(theta_deg, dtype=np.float64)
    need = nbins + 1 if mode == TPCF_EXPLICIT else 2
    if th.ndim != 1 or th.shape[0] != need:
        raise TpcfError(TPCF_EINVAL, f"theta_deg must hold {need} values")
    err = ctypes.create_string_buffer(512)
    st = lib().tpcf_count_static(int(nbins), _np_ptr(th), int(mode), ctypes.c_void_p(radec_i_dev_ptr), int(n_i),
                                 ctypes.c_void_p(radec_j_dev_ptr or None), int(n_j), int(dtype), ctypes.c_void_p(hist_dev_ptr),
                                 ctypes.c_void_p(stream_ptr or None), err, len(err))
    if st != TPCF_OK:
        raise TpcfError(st, err.value.decode())


def tpcf_count_all(ctx, nbins: int):
    """{"DD": (hist, under, over), "DR": ..., "RR": ...} of one call that has the three counts in flight together."""
    hist = np.zeros((3, nbins), dtype=np.uint64)
    uo = np.zeros((3, 2), dtype=np.uint64)
    _check(ctx, lib().tpcf_count_all(ctx, _np_ptr(hist), _np_ptr(uo)))
    return {k: (hist[i].copy(), int(uo[i, 0]), int(uo[i, 1])) for k, i in _KINDS.items()}


def tpcf_count_all_async(ctx, hist_dev_ptr: int) -> None:
    _check(ctx, lib().tpcf_count_all_async(ctx, ctypes.c_void_p(hist_dev_ptr)))


def tpcf_estimate(ctx, nbins: int) -> np.ndarray:
    w = np.empty(nbins, dtype=np.float64)
    _check(ctx, lib().tpcf_estimate(ctx, _np_ptr(w)))
    return w


def tpcf_count3(ctx, which: int, nbins: int) -> np.ndarray:
    """Three-point counts of one loaded catalog: uint64 array [nbins+2]^3 over the ascending side slots (include/tpcf.h)."""
    m = nbins + 2
    h3 = np.zeros((m, m, m), dtype=np.uint64)
    _check(ctx, lib().tpcf_count3(ctx, int(which), _np_ptr(h3)))
    return h3


def tpcf_estimate_cross(ctx, nbins: int) -> np.ndarray:
    w = np.empty(nbins, dtype=np.float64)
    _check(ctx, lib().tpcf_estimate_cross(ctx, _np_ptr(w)))
    return w


def tpcf_set_weights(ctx, which: int, w) -> None:
    w = np.ascontiguousarray(w, dtype=np.float64)
    if w.ndim != 1:
        raise TpcfError(TPCF_EINVAL, "weights must be a 1-D array")
    _check(ctx, lib().tpcf_set_weights(ctx, int(which), _np_ptr(w), w.shape[0]))


def tpcf_count_weighted(ctx, kind: int, nbins: int) -> Tuple[np.ndarray, float, float]:
    h = np.zeros(nbins, dtype=np.float64)
    uo = np.zeros(2, dtype=np.float64)
    _check(ctx, lib().tpcf_count_weighted(ctx, int(kind), _np_ptr(h), _np_ptr(uo)))
    return h, float(uo[0]), float(uo[1])


def tpcf_estimate_from(dd, dr, rr, n_d: int, n_r: int) -> np.ndarray:
    dd = np.ascontiguousarray(dd, dtype=np.uint64)
    dr = np.ascontiguousarray(dr, dtype=np.uint64)
    rr = np.ascontiguousarray(rr, dtype=np.uint64)
    w = np.empty(dd.shape[0], dtype=np.float64)
    st = lib().tpcf_estimate_from(_np_ptr(dd), _np_ptr(dr), _np_ptr(rr), dd.shape[0], int(n_d), int(n_r), _np_ptr(w))
    if st != TPCF_OK:
        raise TpcfError(st, "tpcf_estimate_from: invalid arguments")
    return w


def tpcf_set_stream(ctx, stream: int) -> None:
    _check(ctx, lib().tpcf_set_stream(ctx, ctypes.c_void_p(stream)))


def tpcf_set_engine(ctx, engine: int) -> None:
    _check(ctx, lib().tpcf_set_engine(ctx, int(engine)))


def tpcf_set_guard_scale(ctx, scale: float) -> None:
    _check(ctx, lib().tpcf_set_guard_scale(ctx, float(scale)))


def tpcf_set_window(ctx, enabled: bool) -> None:
    _check(ctx, lib().tpcf_set_window(ctx, int(bool(enabled))))


def tpcf_set_tensor_share_limit(ctx, limit: float) -> None:
    _check(ctx, lib().tpcf_set_tensor_share_limit(ctx, float(limit)))


def tpcf_set_pruning(ctx, enabled: bool) -> None:
    _check(ctx, lib().tpcf_set_pruning(ctx, int(bool(enabled))))


def tpcf_get_bands(ctx):
    """(lo, hi, slot_below) arrays of the fast engine's guard bands."""
    n = ctypes.c_int()
    _check(ctx, lib().tpcf_get_bands(ctx, 0, None, None, None, ctypes.byref(n)))
    lo, hi = np.empty(n.value, dtype=np.float32), np.empty(n.value, dtype=np.float32)
    sb = np.empty(n.value, dtype=np.int32)
    _check(ctx, lib().tpcf_get_bands(ctx, n.value, _np_ptr(lo), _np_ptr(hi), _np_ptr(sb), ctypes.byref(n)))
    return lo, hi, sb


def tpcf_window_host(ctx, lo2: float, hi2: float) -> Tuple[int, int]:
    k, e = ctypes.c_int(), ctypes.c_int()
    _check(ctx, lib().tpcf_window_host(ctx, ctypes.c_float(lo2), ctypes.c_float(hi2), ctypes.byref(k), ctypes.byref(e)))
    return k.value, e.value


def tpcf_set_partition(ctx, part: int, nparts: int) -> None:
    _check(ctx, lib().tpcf_set_partition(ctx, int(part), int(nparts)))


def tpcf_get_stats(ctx) -> dict:
    s = tpcf_stats()
    _check(ctx, lib().tpcf_get_stats(ctx, ctypes.byref(s)))
    return s.as_dict()


def tpcf_set_kernel_timing(ctx, enabled: bool) -> None:
    _check(ctx, lib().tpcf_set_kernel_timing(ctx, int(bool(enabled))))


def tpcf_get_kernel_times(ctx) -> np.ndarray:
    ms = np.zeros(64, dtype=np.float32)
    n = ctypes.c_int()
    _check(ctx, lib().tpcf_get_kernel_times(ctx, _np_ptr(ms), 64, ctypes.byref(n)))
    return ms[: n.value].copy()


def tpcf_tensor_probe(ctx, s_rows: np.ndarray, b_rows: np.ndarray) -> np.ndarray:
    """q tiles of the tensor engine's MMA: s_rows, b_rows (ntiles, 128, 4) float32 -> (ntiles, 128, 128) float32."""
    s_rows = np.ascontiguousarray(s_rows, dtype=np.float32)
    b_rows = np.ascontiguousarray(b_rows, dtype=np.float32)
    if s_rows.ndim != 3 or s_rows.shape[1:] != (128, 4) or b_rows.shape != s_rows.shape:
        raise ValueError("s_rows and b_rows must both be (ntiles, 128, 4)")
    q = np.empty((s_rows.shape[0], 128, 128), dtype=np.float32)
    _check(ctx, lib().tpcf_tensor_probe(ctx, s_rows.ctypes.data_as(ctypes.c_void_p), b_rows.ctypes.data_as(ctypes.c_void_p),
                                        s_rows.shape[0], q.ctypes.data_as(ctypes.c_void_p)))
    return q


def tpcf_classify_fast(ctx, d2: float) -> int:
    out = ctypes.c_int()
    _check(ctx, lib().tpcf_classify_fast(ctx, ctypes.c_float(d2), ctypes.byref(out)))
    return out.value


def tpcf_plan(ctx, kind: int, n_d: int, n_r: int) -> int:
    out = ctypes.c_uint64()
    _check(ctx, lib().tpcf_plan(ctx, int(kind), int(n_d), int(n_r), ctypes.byref(out)))
    return out.value


def tpcf_plan_item_pairs(ctx, kind: int, n_d: int, n_r: int, w: int) -> int:
    out = ctypes.c_uint64()
    _check(ctx, lib().tpcf_plan_item_pairs(ctx, int(kind), int(n_d), int(n_r), int(w), ctypes.byref(out)))
    return out.value


class Context:
    """Owns one tpcf_ctx.  Convenience wrapper over the functions above; holds no arithmetic."""

    def __init__(self, nbins: int, theta_deg, mode="explicit", max_abs_coord: Optional[float] = None):
        """Angular context (tpcf_create); with max_abs_coord a 3-D context (tpcf_create_r: theta_deg holds r edges)."""
        self.nbins = int(nbins)
        self.spatial = max_abs_coord is not None
        self._ctx = tpcf_create_r(nbins, theta_deg, mode, max_abs_coord) if self.spatial else tpcf_create(nbins, theta_deg, mode)
        self.n = {TPCF_D: 0, TPCF_R: 0, TPCF_D2: 0}

    def close(self):
        if getattr(self, "_ctx", None):
            tpcf_destroy(self._ctx)
            self._ctx = None

    __del__ = close

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    @property
    def handle(self):
        return self._ctx

    def edges(self):
        return tpcf_get_edges(self._ctx, self.nbins)

    def thresholds(self):
        return tpcf_get_thresholds(self._ctx, self.nbins)

    def load(self, which, radec_deg, stream: int = 0):
        which = _CATS.get(which, which)
        self.n[which] = tpcf_load(self._ctx, which, radec_deg, stream, cols=3 if self.spatial else 2)

    def count(self, kind, rows=None):
        return tpcf_count(self._ctx, _ALL_KINDS.get(kind, kind), self.nbins, rows)

    def count_async(self, kind, out):
        """out: CUDA uint64/int64 tensor with nbins+2 elements, written {under, bins..., over} on the stream."""
        if not (_is_torch(out) and out.is_cuda and out.is_contiguous() and out.numel() >= self.nbins + 2
                and out.element_size() == 8):
            raise TpcfError(TPCF_EINVAL, "out must be a contiguous CUDA 64-bit tensor of nbins+2 elements")
        tpcf_count_async(self._ctx, _ALL_KINDS.get(kind, kind), out.data_ptr())

    def count_all(self):
        return tpcf_count_all(self._ctx, self.nbins)

    def count_all_async(self, out):
        """out: contiguous CUDA 64-bit tensor of 3 x (nbins+2) elements: {under, bins..., over} of DD, DR, RR."""
        if not (_is_torch(out) and out.is_cuda and out.is_contiguous() and out.numel() >= 3 * (self.nbins + 2)
                and out.element_size() == 8):
            raise TpcfError(TPCF_EINVAL, "out must be a contiguous CUDA 64-bit tensor of 3 x (nbins+2) elements")
        tpcf_count_all_async(self._ctx, out.data_ptr())

    def estimate(self):
        return tpcf_estimate(self._ctx, self.nbins)

    def count3(self, which="D"):
        return tpcf_count3(self._ctx, _CATS.get(which, which), self.nbins)

    def estimate_cross(self):
        return tpcf_estimate_cross(self._ctx, self.nbins)

    def set_weights(self, which, w):
        tpcf_set_weights(self._ctx, _CATS.get(which, which), w)

    def count_weighted(self, kind):
        return tpcf_count_weighted(self._ctx, _ALL_KINDS.get(kind, kind), self.nbins)

    def set_stream(self, stream: int):
        tpcf_set_stream(self._ctx, stream)

    def set_engine(self, engine):
        tpcf_set_engine(self._ctx, {"fast": TPCF_ENGINE_FAST, "exact64": TPCF_ENGINE_EXACT64, "tensor": TPCF_ENGINE_TENSOR}.get(engine, engine))

    def set_guard_scale(self, scale: float):
        tpcf_set_guard_scale(self._ctx, scale)

    def set_window(self, enabled: bool):
        tpcf_set_window(self._ctx, enabled)

    def set_tensor_share_limit(self, limit: float):
        tpcf_set_tensor_share_limit(self._ctx, limit)

    def set_pruning(self, enabled: bool):
        tpcf_set_pruning(self._ctx, enabled)

    def bands(self):
        return tpcf_get_bands(self._ctx)

    def window_host(self, lo2: float, hi2: float):
        return tpcf_window_host(self._ctx, lo2, hi2)

    def set_partition(self, part: int, nparts: int):
        tpcf_set_partition(self._ctx, part, nparts)

    def stats(self):
        return tpcf_get_stats(self._ctx)

    def set_kernel_timing(self, enabled: bool):
        tpcf_set_kernel_timing(self._ctx, enabled)

    def kernel_times_ms(self):
        return tpcf_get_kernel_times(self._ctx)

    def classify_fast(self, d2: float):
        return tpcf_classify_fast(self._ctx, d2)

    def plan(self, kind, n_d: int, n_r: int):
        return tpcf_plan(self._ctx, _KINDS.get(kind, kind), n_d, n_r)

    def plan_item_pairs(self, kind, n_d: int, n_r: int, w: int):
        return tpcf_plan_item_pairs(self._ctx, _KINDS.get(kind, kind), n_d, n_r, w)
