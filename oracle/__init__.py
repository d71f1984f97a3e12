"""ctypes front-end of the C oracle (oracle/tpcf_oracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package; it imports nothing from paper_1204_6630_b200.  The arithmetic is all in the C file (one
thread per call); this module marshals arrays and, when threads > 1, splits the outer i-rows over
Python threads that each call the same single-threaded C loop on a private histogram and sums the
integer results (order-independent).
"""
from __future__ import annotations

import ctypes
import os
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass
from typing import Optional

import numpy as np

from .build import build as _build

_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        L = ctypes.CDLL(_build())
        vp, sz, i32, i64p = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int, ctypes.c_void_p
        L.orc_radec_to_xyz.argtypes = [vp, sz, vp]
        L.orc_radec_to_xyz.restype = None
        L.orc_count_auto.argtypes = [vp, sz, sz, sz, vp, i32, vp, vp, vp]
        L.orc_count_auto.restype = i32
        L.orc_count_cross.argtypes = [vp, sz, sz, sz, vp, sz, vp, i32, vp, vp, vp]
        L.orc_count_cross.restype = i32
        L.orc_count_rows.argtypes = [vp, i64p, sz, sz, vp, sz, i32, vp, i32, vp, vp, vp]
        L.orc_count_rows.restype = i32
        f64 = ctypes.c_double
        L.orc_count_auto_xyz.argtypes = [vp, sz, sz, sz, vp, i32, f64, vp, vp]
        L.orc_count_auto_xyz.restype = i32
        L.orc_count_cross_xyz.argtypes = [vp, sz, sz, sz, vp, sz, vp, i32, f64, vp, vp]
        L.orc_count_cross_xyz.restype = i32
        L.orc_count_rows_xyz.argtypes = [vp, i64p, sz, sz, vp, sz, i32, vp, i32, f64, vp, vp]
        L.orc_count_rows_xyz.restype = i32
        L.orc_wsum_auto.argtypes = [vp, vp, sz, sz, sz, vp, i32, vp, vp]
        L.orc_wsum_auto.restype = i32
        L.orc_wsum_cross.argtypes = [vp, vp, sz, sz, sz, vp, vp, sz, vp, i32, vp, vp]
        L.orc_wsum_cross.restype = i32
        L.orc_estimate.argtypes = [vp, vp, vp, i32, ctypes.c_uint64, ctypes.c_uint64, vp]
        L.orc_estimate.restype = None
        L.orc_count_triples.argtypes = [vp, sz, sz, sz, vp, i32, vp]
        L.orc_count_triples.restype = i32
        L.orc_estimate_cross.argtypes = [vp, vp, vp, vp, i32, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64, vp]
        L.orc_estimate_cross.restype = None
        _lib = L
    return _lib


def host_threads() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:  # pragma: no cover
        return max(1, os.cpu_count() or 1)


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def radec_to_xyz(radec) -> np.ndarray:
    """O1+O2: rows of (RA, Dec) degrees, float32 widened exactly to float64 -> (n, 3) unit vectors."""
    rd = np.ascontiguousarray(np.asarray(radec, dtype=np.float64).reshape(-1, 2))
    out = np.empty((rd.shape[0], 3), dtype=np.float64)
    lib().orc_radec_to_xyz(_ptr(rd), rd.shape[0], _ptr(out))
    return out


@dataclass
class Counts:
    """One histogram: hist[k] for the nbins theta bins plus the out-of-range counters."""
    hist: np.ndarray          # uint64[nbins]
    under: int
    over: int
    near: Optional[np.ndarray] = None   # uint64[nbins+1], O6 near-edge counters (validation runs)
    mismatch: Optional[int] = None      # O8 self-check counter (validation runs)

    @property
    def total(self) -> int:
        return int(self.hist.sum(dtype=np.uint64)) + self.under + self.over

    def tol(self) -> np.ndarray:
        """Per-bin tolerance tol_k = near[k] + near[k+1] (BASELINE.json / SURVEY.md O6)."""
        assert self.near is not None
        return (self.near[:-1] + self.near[1:]).astype(np.int64)


def _run(kind: str, spans, call, nbins: int, validate: bool, threads: int) -> Counts:
    def one(span):
        h = np.zeros(nbins + 2, dtype=np.uint64)
        nr = np.zeros(nbins + 1, dtype=np.uint64) if validate else None
        mm = np.zeros(1, dtype=np.uint64) if validate else None
        rc = call(span[0], span[1], h, nr, mm)
        if rc != 0:
            raise ValueError(f"oracle {kind}: bad arguments (rc={rc})")
        return h, nr, mm

    if threads <= 1 or len(spans) == 1:
        parts = [one(s) for s in spans]
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            parts = list(ex.map(one, spans))
    h = np.sum([p[0] for p in parts], axis=0, dtype=np.uint64)
    near = np.sum([p[1] for p in parts], axis=0, dtype=np.uint64) if validate else None
    mm = int(np.sum([p[2] for p in parts], dtype=np.uint64)) if validate else None
    return Counts(h[1:-1].copy(), int(h[0]), int(h[-1]), near, mm)


def _even_spans(n: int, parts: int):
    cuts = np.linspace(0, n, max(1, min(parts, n)) + 1).astype(np.int64)
    return [(int(a), int(b)) for a, b in zip(cuts[:-1], cuts[1:]) if b > a] or [(0, 0)]


def _triangle_spans(n: int, parts: int):
    """Split rows 0..n so each span holds about the same number of i<j pairs."""
    parts = max(1, min(parts, n))
    total = n * (n - 1) / 2.0
    cuts = [0]
    for p in range(1, parts):
        # rows [0, c) hold c*n - c(c+1)/2 pairs; solve for the target
        t = total * p / parts
        c = int(n - 0.5 - np.sqrt(max((n - 0.5) ** 2 - 2.0 * t, 0.0)))
        cuts.append(min(max(c, cuts[-1]), n))
    cuts.append(n)
    return [(a, b) for a, b in zip(cuts[:-1], cuts[1:]) if b > a] or [(0, 0)]


def count_auto(xyz: np.ndarray, edges, validate: bool = False, threads: int = 1) -> Counts:
    """DD or RR: all unordered pairs i<j of one catalog (reading A3)."""
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    e = np.ascontiguousarray(edges, dtype=np.float64)
    nb, n = e.shape[0] - 1, xyz.shape[0]
    L = lib()
    call = lambda a, b, h, nr, mm: L.orc_count_auto(_ptr(xyz), n, a, b, _ptr(e), nb, _ptr(h), _ptr(nr), _ptr(mm))
    return _run("auto", _triangle_spans(n, threads * 4 if threads > 1 else 1), call, nb, validate, threads)


def count_cross(a: np.ndarray, b: np.ndarray, edges, validate: bool = False, threads: int = 1) -> Counts:
    """DR: all N_a * N_b ordered pairs."""
    a = np.ascontiguousarray(a, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    e = np.ascontiguousarray(edges, dtype=np.float64)
    nb = e.shape[0] - 1
    L = lib()
    call = lambda i0, i1, h, nr, mm: L.orc_count_cross(_ptr(a), a.shape[0], i0, i1, _ptr(b), b.shape[0], _ptr(e), nb,
                                                       _ptr(h), _ptr(nr), _ptr(mm))
    return _run("cross", _even_spans(a.shape[0], threads), call, nb, validate, threads)


def count_rows(a: np.ndarray, rows, b: np.ndarray, exclude_self: bool, edges, validate: bool = False,
               threads: int = 1) -> Counts:
    """Row-subset mode: sum_{i in rows} sum_j, skipping j == i when exclude_self."""
    a = np.ascontiguousarray(a, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    r = np.ascontiguousarray(rows, dtype=np.int64)
    if r.size and (r.min() < 0 or r.max() >= a.shape[0]):
        raise ValueError("row index out of range")
    e = np.ascontiguousarray(edges, dtype=np.float64)
    nb = e.shape[0] - 1
    L = lib()
    call = lambda r0, r1, h, nr, mm: L.orc_count_rows(_ptr(a), _ptr(r), r0, r1, _ptr(b), b.shape[0],
                                                      1 if exclude_self else 0, _ptr(e), nb, _ptr(h), _ptr(nr),
                                                      _ptr(mm))
    return _run("rows", _even_spans(r.shape[0], threads), call, nb, validate, threads)


def estimate(dd, dr, rr, n_d: int, n_r: int) -> np.ndarray:
    """O7: pair-normalised Landy-Szalay w_k (Eq. 1 as read in A1)."""
    dd = np.ascontiguousarray(dd, dtype=np.uint64)
    dr = np.ascontiguousarray(dr, dtype=np.uint64)
    rr = np.ascontiguousarray(rr, dtype=np.uint64)
    w = np.empty(dd.shape[0], dtype=np.float64)
    lib().orc_estimate(_ptr(dd), _ptr(dr), _ptr(rr), dd.shape[0], int(n_d), int(n_r), _ptr(w))
    return w


def count_triples(xyz: np.ndarray, edges, threads: int = 1) -> np.ndarray:
    """Three-point counts of one catalog (orc_count_triples): dense uint64 array [nbins+2]^3 over the ascending slots
    (a <= b <= c; 0 = under, 1..nbins = bins, nbins+1 = over) of the three sides of every triple i<j<k."""
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    e = np.ascontiguousarray(edges, dtype=np.float64)
    nb, n = e.shape[0] - 1, xyz.shape[0]
    m = nb + 2
    L = lib()
    # rows [0, c) hold about (c/n)-dependent shares of the triples; many short spans balance the threads well enough
    spans = _even_spans(n, threads * 16 if threads > 1 else 1)

    def one(span):
        h = np.zeros(m * m * m, dtype=np.uint64)
        if L.orc_count_triples(_ptr(xyz), n, span[0], span[1], _ptr(e), nb, _ptr(h)) != 0:
            raise ValueError("oracle triples: bad arguments")
        return h

    if threads <= 1 or len(spans) == 1:
        parts = [one(sp) for sp in spans]
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            parts = list(ex.map(one, spans))
    return np.sum(parts, axis=0, dtype=np.uint64).reshape(m, m, m)


def estimate_cross(d1d2, d1r, d2r, rr, n_1: int, n_2: int, n_r: int) -> np.ndarray:
    """Cross-correlation estimator w12_k = (D1D2/n12 - D1R/n1r - D2R/n2r + RR/nrr) / (RR/nrr) (orc_estimate_cross)."""
    a = [np.ascontiguousarray(x, dtype=np.uint64) for x in (d1d2, d1r, d2r, rr)]
    w = np.empty(a[0].shape[0], dtype=np.float64)
    lib().orc_estimate_cross(_ptr(a[0]), _ptr(a[1]), _ptr(a[2]), _ptr(a[3]), a[0].shape[0], int(n_1), int(n_2), int(n_r), _ptr(w))
    return w


# ---- 3-D variant: Euclidean separations of Cartesian rows, bins in r -------------------------------
def count_auto_xyz(xyz: np.ndarray, r_edges, near_tol: float = -1.0, threads: int = 1) -> Counts:
    """DD or RR of the 3-D variant: all unordered pairs i<j, r = |a - b| in fp64; near_tol >= 0 also fills `near`."""
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    e = np.ascontiguousarray(r_edges, dtype=np.float64)
    nb, n = e.shape[0] - 1, xyz.shape[0]
    L = lib()
    call = lambda a, b, h, nr, mm: L.orc_count_auto_xyz(_ptr(xyz), n, a, b, _ptr(e), nb, near_tol, _ptr(h), _ptr(nr))
    return _run("auto_xyz", _triangle_spans(n, threads * 4 if threads > 1 else 1), call, nb, near_tol >= 0, threads)


def count_cross_xyz(a: np.ndarray, b: np.ndarray, r_edges, near_tol: float = -1.0, threads: int = 1) -> Counts:
    """DR of the 3-D variant: all N_a * N_b ordered pairs."""
    a = np.ascontiguousarray(a, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    e = np.ascontiguousarray(r_edges, dtype=np.float64)
    nb = e.shape[0] - 1
    L = lib()
    call = lambda i0, i1, h, nr, mm: L.orc_count_cross_xyz(_ptr(a), a.shape[0], i0, i1, _ptr(b), b.shape[0], _ptr(e), nb,
                                                           near_tol, _ptr(h), _ptr(nr))
    return _run("cross_xyz", _even_spans(a.shape[0], threads), call, nb, near_tol >= 0, threads)


def count_rows_xyz(a: np.ndarray, rows, b: np.ndarray, exclude_self: bool, r_edges, near_tol: float = -1.0,
                   threads: int = 1) -> Counts:
    """Row-subset mode of the 3-D variant."""
    a = np.ascontiguousarray(a, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    r = np.ascontiguousarray(rows, dtype=np.int64)
    if r.size and (r.min() < 0 or r.max() >= a.shape[0]):
        raise ValueError("row index out of range")
    e = np.ascontiguousarray(r_edges, dtype=np.float64)
    nb = e.shape[0] - 1
    L = lib()
    call = lambda r0, r1, h, nr, mm: L.orc_count_rows_xyz(_ptr(a), _ptr(r), r0, r1, _ptr(b), b.shape[0],
                                                          1 if exclude_self else 0, _ptr(e), nb, near_tol, _ptr(h), _ptr(nr))
    return _run("rows_xyz", _even_spans(r.shape[0], threads), call, nb, near_tol >= 0, threads)


# ---- weighted counts (oracle/tpcf_oracle.c orc_wsum_*): sum of w_i * w_j per bin --------------------------------------
@dataclass
class WeightedSums:
    """Per theta bin the fp64 sum of w_i * w_j over its pairs, plus the out-of-range sums and the sums of |w_i * w_j|."""
    hist: np.ndarray          # float64[nbins]
    under: float
    over: float
    abs_hist: np.ndarray      # float64[nbins + 2]: sum |w_i w_j| for {under, bins, over}: the scale of the tolerance


def _run_w(spans, call, nbins: int, threads: int) -> WeightedSums:
    def one(span):
        h, a = np.zeros(nbins + 2), np.zeros(nbins + 2)
        if call(span[0], span[1], h, a) != 0:
            raise ValueError("oracle weighted sums: bad arguments")
        return h, a

    if threads <= 1 or len(spans) == 1:
        parts = [one(s) for s in spans]
    else:
        with ThreadPoolExecutor(max_workers=threads) as ex:
            parts = list(ex.map(one, spans))
    h = np.sum([p[0] for p in parts], axis=0)
    a = np.sum([p[1] for p in parts], axis=0)
    return WeightedSums(h[1:-1].copy(), float(h[0]), float(h[-1]), a)


def wsum_auto(xyz: np.ndarray, w, edges, threads: int = 1) -> WeightedSums:
    L = lib()
    xyz = np.ascontiguousarray(xyz, dtype=np.float64)
    w = np.ascontiguousarray(w, dtype=np.float64)
    e = np.ascontiguousarray(edges, dtype=np.float64)
    nb, n = e.shape[0] - 1, xyz.shape[0]
    assert w.shape == (n,)
    call = lambda a, b, h, ab: L.orc_wsum_auto(_ptr(xyz), _ptr(w), n, a, b, _ptr(e), nb, _ptr(h), _ptr(ab))
    return _run_w(_triangle_spans(n, threads * 4 if threads > 1 else 1), call, nb, threads)


def wsum_cross(a: np.ndarray, wa, b: np.ndarray, wb, edges, threads: int = 1) -> WeightedSums:
    L = lib()
    a = np.ascontiguousarray(a, dtype=np.float64)
    b = np.ascontiguousarray(b, dtype=np.float64)
    wa = np.ascontiguousarray(wa, dtype=np.float64)
    wb = np.ascontiguousarray(wb, dtype=np.float64)
    e = np.ascontiguousarray(edges, dtype=np.float64)
    nb = e.shape[0] - 1
    assert wa.shape == (a.shape[0],) and wb.shape == (b.shape[0],)
    call = lambda i0, i1, h, ab: L.orc_wsum_cross(_ptr(a), _ptr(wa), a.shape[0], i0, i1, _ptr(b), _ptr(wb), b.shape[0], _ptr(e), nb,
                                                  _ptr(h), _ptr(ab))
    return _run_w(_even_spans(a.shape[0], threads), call, nb, threads)
