"""CPU-side checks of libtpcf (no GPU): the library loads and exports every symbol of include/tpcf.h, argument
validation, edge/threshold generation, the fast engine's lookup tables against the thresholds, the tile work
plan and its partition, the estimator, and the no-fallback rule (compute calls fail loudly without a GPU)."""
import ctypes
import json
import math
import os
import re

import numpy as np
import pytest

import oracle
import paper_1204_6630_b200 as T
import synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def has_gpu():
    try:
        import torch
        return torch.cuda.is_available()
    except Exception:
        return False


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "tpcf.h")).read()
    declared = set(re.findall(r"\b(tpcf_[a-z0-9_]+)\s*\(", header))
    assert declared == set(T.EXPORTS), declared ^ set(T.EXPORTS)
    L = T.lib()
    for name in declared:
        assert getattr(L, name) is not None


def test_create_rejects_bad_binnings():
    bad = [(0, [0.1, 1.0], "log"), (5000, [0.1, 1.0], "log"), (4, [0.0, 1.0], "log"), (4, [1.0, 1.0], "linear"),
           (4, [2.0, 1.0], "linear"), (4, [-1.0, 1.0], "linear"), (4, [1.0, 181.0], "linear"),
           (4, [float("nan"), 1.0], "linear"), (2, [0.0, 1.0, 1.0], "explicit"), (2, [0.0, 2.0, 1.0], "explicit"),
           (2, [0.0, 1.0, 200.0], "explicit")]
    for nbins, th, mode in bad:
        with pytest.raises(T.TpcfError) as ei:
            T.tpcf_create(nbins, th, mode)
        assert ei.value.status == T.TPCF_EINVAL


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
def test_edges_match_the_input_recipe_and_thresholds_closed_form(idx):
    cfg = synth.CONFIGS[idx]
    with T.Context(cfg.nbins, [cfg.theta_min, cfg.theta_max], cfg.mode) as c:
        e = c.edges()
        ref = synth.config_edges(cfg)
        assert e[0] == cfg.theta_min and e[-1] == cfg.theta_max
        np.testing.assert_allclose(e, ref, rtol=1e-14, atol=0)
        thr = c.thresholds()
    # T_k = |a-b|^2 at separation e_k = 2 - 2 cos(e_k): checked with mpmath-free high precision via the
    # half-angle form in numpy longdouble
    el = np.asarray(ref, dtype=np.longdouble) * (np.pi / np.longdouble(360.0))
    want = (4 * np.sin(el) ** 2).astype(np.float64)
    np.testing.assert_allclose(thr, want, rtol=1e-15, atol=0)   # 3-4 fp64 roundings in 4 sin^2(e pi/360)
    big = ref > 5.0                                  # where 2 - 2 cos is not cancellation-limited
    np.testing.assert_allclose(thr[big], 2.0 - 2.0 * np.cos(np.radians(ref[big])), rtol=1e-13)


def test_create_r_binning_of_the_3d_variant():
    """tpcf_create_r: thresholds are (e_k * scale)^2 with scale the power of two that brings every
    position inside the unit ball; edges beyond the largest possible separation and bad edges are rejected."""
    with T.Context(40, [1.0, 200.0], "log", max_abs_coord=1000.0) as c:
        e = c.edges()
        np.testing.assert_allclose(e, synth.edges(40, 1.0, 200.0, "log"), rtol=1e-14)
        thr = c.thresholds()
        scale = 2.0 ** -11                                   # 2^11 = 2048 > sqrt(3) * 1000
        np.testing.assert_array_equal(thr, (e * scale) ** 2)
        assert c.classify_fast(float(np.float32(thr[10] * 1.01))) == 11 and c.classify_fast(5.5) == 42
    with T.Context(8, [0.0, 4096.0], "linear", max_abs_coord=1000.0) as c:      # up to 2 / scale = 4096 is allowed
        assert c.thresholds()[0] == 0.0 and c.thresholds()[-1] == 4.0
    for nbins, th, mode, mx in [(8, [0.0, 4097.0], "linear", 1000.0), (4, [0.0, 1.0], "log", 10.0), (4, [-1.0, 1.0], "linear", 10.0),
                                (4, [1.0, 2.0], "linear", 0.0), (4, [1.0, 2.0], "linear", float("inf")),
                                (2, [0.0, 1.0, 1.0], "explicit", 10.0), (2, [0.0, float("nan"), 1.0], "explicit", 10.0)]:
        with pytest.raises(T.TpcfError) as ei:
            T.tpcf_create_r(nbins, th, mode, mx)
        assert ei.value.status == T.TPCF_EINVAL


def expected_slot(v, thr, nbins):
    if v >= 5.0:
        return nbins + 2
    if v < thr[0]:
        return 0
    if v > thr[-1]:
        return nbins + 1
    return min(int(np.searchsorted(thr, v, side="right")) - 1, nbins - 1) + 1


def fp32_bound(t):
    """|q_fp32 - q| bound of DESIGN.md section 4 (without the safety margin of the implementation): the larger of the
    difference form (9 t + 10 r sqrt(t)) 2^-24 with r <= 0.1 and the expanded form 29.1 t 2^-24 (window loops from 2.5 r on)."""
    return 6.0e-8 * math.sqrt(t) + 1.74e-6 * t


def fp32_bound_lookup(t):
    """Bound of the difference form alone, (9 t + 10 r sqrt(t)) 2^-24 with r <= kRCap = 0.25: what the cell-lookup tables
    (tpcf_classify_fast) must cover."""
    return 1.5e-7 * math.sqrt(t) + 5.4e-7 * t


@pytest.mark.parametrize("idx", [1, 2, 3, 4, 5])
@pytest.mark.parametrize("scale", [1.0, 8.0])
def test_fast_tables_agree_with_thresholds_outside_the_guard_bands(idx, scale):
    cfg = synth.CONFIGS[idx]
    rng = np.random.default_rng(idx)
    with T.Context(cfg.nbins, synth.config_edges(cfg), "explicit") as c:
        c.set_guard_scale(scale)
        thr = c.thresholds()
        pos = thr[thr > 0]
        near = (pos[:, None] * (1.0 + rng.normal(0.0, 2e-6, (len(pos), 24)))).ravel()
        vals = np.concatenate([np.exp(rng.uniform(np.log(1e-13), np.log(4.0), 6000)), near,
                               [0.0, 1e-30, 4.0, 4.0000005, 6.07, 19.9, 48.0]]).astype(np.float32)
        n_amb = 0
        for v in vals:
            v = float(v)
            s = c.classify_fast(v)
            d = np.abs(thr - v)
            k = int(np.argmin(d))
            if s == -1:
                n_amb += 1
                # ambiguous only close to an edge: within the (scaled, margin-included) band
                assert d[k] <= scale * (2.51e-7 * math.sqrt(thr[k]) + 1.01e-6 * thr[k] + 1.1e-13) + 1e-7 * thr[k]
            else:
                assert s == expected_slot(v, thr, cfg.nbins), (v, s)
                # a decided value must be farther from every droppable edge than the fp32 rounding bound,
                # otherwise the true d2 could be on the other side
                live = np.ones(len(thr), bool)
                live[0] = thr[0] > 0
                live[-1] = thr[-1] < 4.0
                if v < 4.5:
                    assert np.all(d[live] > fp32_bound_lookup(v)), (v, k)
        assert n_amb > 0
        assert c.stats()["cells"] <= 8192


@pytest.mark.parametrize("idx", [1, 3, 5])
def test_guard_bands_and_window_selection(idx):
    """The guard bands the window loops compare against, and the host mirror of the kernel's window selection
    (tpcf_window_host) against a brute-force scan of the band list."""
    cfg = synth.CONFIGS[idx]
    rng = np.random.default_rng(100 + idx)
    with T.Context(cfg.nbins, synth.config_edges(cfg), "explicit") as c:
        thr = c.thresholds()
        lo, hi, below = c.bands()
        n = len(lo)
        assert np.all(lo[1:] >= hi[:-1]) and np.all(hi >= lo), "bands ascending and disjoint"
        assert lo[-1] == hi[-1] == 5.0 and below[-1] <= cfg.nbins + 1, "last band: the zero-width discard edge"
        live = [k for k in range(cfg.nbins + 1) if not (k == 0 and thr[0] == 0.0) and not (k == cfg.nbins and thr[-1] >= 4.0)]
        assert n == len(live) + 1, "one band per droppable edge (none merged on the BASELINE configs) + discard"
        for b, k in enumerate(live):
            g = fp32_bound(thr[k])
            assert lo[b] <= thr[k] - g and thr[k] + g <= hi[b], "band covers the edge by more than the fp32 bound"
            assert below[b] == k, "result slot just below band b is the bin below edge k"
        for _ in range(4000):
            a = float(np.float32(np.exp(rng.uniform(np.log(1e-9), np.log(4.0)))))
            w = float(np.float32(a * (1.0 + np.exp(rng.uniform(np.log(1e-4), np.log(3.0))))))
            k, e = T.tpcf_window_host(c._ctx, a, w)
            touch = [b for b in range(n) if hi[b] > a and lo[b] <= w]          # bands the interval [a, w] can reach
            assert all(hi[b] <= a for b in range(k)), "no band below the first one reaches the interval"
            if e <= 3:
                assert set(touch) <= set(range(k, k + e)), (a, w, k, e, touch)
            else:
                assert len(touch) > 3 or (touch and touch[-1] - k >= 3)


def _f32(x):
    return np.asarray(x, dtype=np.float32)


def _fma32(a, b, c):
    """fp32 fused multiply-add: the product of two fp32 numbers is exact in fp64; one rounding to fp32 follows."""
    return _f32(a.astype(np.float64) * b.astype(np.float64) + c.astype(np.float64))


def test_fp32_error_bounds_of_design_section_4():
    """DESIGN.md section 4 in numbers: the kernel's two fp32 evaluations of the squared chord, replayed here in numpy
    fp32 on random (group, subtile) geometry, against the fp64 value.  Expanded form (window loops, chord >= 2.5 r):
    |error| <= 29.1 u max(d^2, mid); difference form (cell lookup): |error| <= (9 d^2 + 10 d r) u; u = 2^-24."""
    rng = np.random.default_rng(7)
    u = 2.0 ** -24
    n = 400_000
    def unit(v):
        return v / np.linalg.norm(v, axis=1, keepdims=True)
    cq64 = unit(rng.normal(size=(n, 3)))
    ri = np.exp(rng.uniform(np.log(1e-6), np.log(0.04), n))
    rj = np.exp(rng.uniform(np.log(1e-6), np.log(0.05), n))
    sep = (ri + rj) * np.exp(rng.uniform(np.log(3.6), np.log(400.0), n))      # centre distance: blocks from 2.6 r out
    cs64 = unit(cq64 + unit(np.cross(cq64, rng.normal(size=(n, 3)))) * sep[:, None])
    cq, cs = _f32(cq64), _f32(cs64)                                            # fp32 centres (exact values from here on)
    a = cq.astype(np.float64) + unit(rng.normal(size=(n, 3))) * (ri * rng.uniform(0, 1, n))[:, None]    # fp64 rows
    b = cs.astype(np.float64) + unit(rng.normal(size=(n, 3))) * (rj * rng.uniform(0, 1, n))[:, None]
    r = np.linalg.norm(a - cq, axis=1) + np.linalg.norm(b - cs, axis=1)
    d2 = ((a - b) ** 2).sum(1)
    d = np.sqrt(d2)
    ok = d >= 2.5 * (ri + rj)
    ap, bp = _f32(a - cq), _f32(b - cs)                                        # stored offsets (rounded once)
    bw = _f32((bp.astype(np.float64) ** 2).sum(1))                             # |b'|^2 formed in fp64, rounded once
    t = _f32(cq - cs)
    s = _f32(ap + t)
    # expanded form around a band centre mid (any value within a factor of the chord: the bound uses max(d2, mid))
    mid = _f32(d2 * np.exp(rng.uniform(np.log(0.3), np.log(3.0), n)))
    n2 = _fma32(s[:, 2], s[:, 2], _fma32(s[:, 1], s[:, 1], _f32(s[:, 0] * s[:, 0])))
    nsm = _f32(n2 - mid)
    m2b = _f32(-2.0 * bp)
    q = _fma32(s[:, 0], m2b[:, 0], _fma32(s[:, 1], m2b[:, 1], _fma32(s[:, 2], m2b[:, 2], _f32(nsm + bw))))
    err = np.abs(q.astype(np.float64) - (d2 - mid.astype(np.float64)))
    ratio = err[ok] / (u * np.maximum(d2[ok], mid[ok]))
    assert ok.sum() > n // 2 and ratio.max() <= 29.1, ratio.max()
    # difference form
    df = _f32(s - bp)
    qd = _fma32(df[:, 2], df[:, 2], _fma32(df[:, 1], df[:, 1], _f32(df[:, 0] * df[:, 0])))
    errd = np.abs(qd.astype(np.float64) - d2)
    assert np.all(errd <= (9.0 * d2 + 10.0 * d * r) * u)
    # and both stay inside the guard band width the tables are built with (margin included)
    g = 1.0e-7 * d + 3.0e-6 * np.maximum(d2, mid)
    assert np.all(err[ok] < g[ok] / 1.5) and np.all(errd < (1.0e-7 * d + 3.0e-6 * d2) / 1.5)


def test_fast_tables_survive_pathological_edges():
    # bins far narrower than the fp32 guard bands: everything near them must come back ambiguous (-1), never wrong
    e = np.concatenate([[0.0], 1.0 + 1e-7 * np.arange(40), [90.0, 180.0]])
    with T.Context(len(e) - 1, e, "explicit") as c:
        thr = c.thresholds()
        for v in np.linspace(thr[1] * 0.999, thr[40] * 1.001, 400).astype(np.float32):
            s = c.classify_fast(float(v))
            assert s == -1 or s == expected_slot(float(v), thr, len(e) - 1)
        assert c.classify_fast(3.0) == len(e) - 1          # inside the last bin [90, 180]
        assert c.classify_fast(4.0000005) == len(e) - 1    # e_n = 180: nothing is ever "over"
        assert c.classify_fast(0.0) == 1                   # e_0 = 0: theta = 0 is in bin 0


@pytest.mark.parametrize("n_d,n_r", [(1, 1), (5, 3), (1024, 1024), (1025, 2047), (4096, 4096), (100_000, 70_001)])
def test_plan_covers_every_pair_exactly_once(n_d, n_r):
    with T.Context(4, [0.1, 10.0], "log") as c:
        for kind, total in (("DD", n_d * (n_d - 1) // 2), ("DR", n_d * n_r), ("RR", n_r * (n_r - 1) // 2)):
            n = c.plan(kind, n_d, n_r)
            pairs = [c.plan_item_pairs(kind, n_d, n_r, w) for w in range(n)]
            assert sum(pairs) == total
            for nparts in (2, 3):
                assert sum(sum(pairs[p::nparts]) for p in range(nparts)) == total
            with pytest.raises(T.TpcfError):
                c.plan_item_pairs(kind, n_d, n_r, n)


def test_plan_sizes_at_paper_scale():
    with T.Context(4, [0.1, 10.0], "log") as c:
        n = c.plan("DR", 430_000, 430_000)
        assert 148 * 40 <= n <= 2 ** 32
        assert c.plan("RR", 1_000_000, 2_000_000) < 2 ** 32


def test_estimator_hand_case_and_against_oracle():
    g = json.load(open(os.path.join(ROOT, "tests", "golden", "hand_catalogs.json")))["landy_szalay_hand"]
    w = T.tpcf_estimate_from(g["dd"], g["dr"], g["rr"], g["n_d"], g["n_r"])
    assert abs(w[0] - g["w"][0]) < 1e-15
    rng = np.random.default_rng(3)
    dd, dr, rr = (rng.integers(0, 10 ** 9, 50).astype(np.uint64) for _ in range(3))
    rr[7] = 0
    a = T.tpcf_estimate_from(dd, dr, rr, 430_000, 500_000)
    b = oracle.estimate(dd, dr, rr, 430_000, 500_000)
    assert math.isnan(a[7]) and math.isnan(b[7])
    ok = ~np.isnan(b)
    np.testing.assert_allclose(a[ok], b[ok], rtol=1e-15, atol=1e-15)


def test_setters_validate():
    with T.Context(4, [0.1, 10.0], "log") as c:
        for bad in (0.0, -1.0, float("nan")):
            with pytest.raises(T.TpcfError):
                c.set_guard_scale(bad)
        for part, nparts in ((0, 0), (2, 2), (-1, 2)):
            with pytest.raises(T.TpcfError):
                c.set_partition(part, nparts)
        with pytest.raises(T.TpcfError):
            c.set_engine(7)
        c.set_partition(1, 2)
        c.set_engine("exact64")


@pytest.mark.skipif(has_gpu(), reason="checks the behaviour on a box without a GPU")
def test_no_cpu_fallback_compute_calls_fail_loudly_without_a_gpu():
    D, R, e, cfg = synth.make_config(1, n_d=64, n_r=64)
    with T.Context(cfg.nbins, e, "explicit") as c:
        with pytest.raises(T.TpcfError) as ei:
            c.load("D", D)
        assert ei.value.status == T.TPCF_ECUDA
        with pytest.raises(T.TpcfError) as ei:
            c.count("DD")
        assert ei.value.status == T.TPCF_ECUDA
        with pytest.raises(T.TpcfError) as ei:
            c.estimate()
        assert ei.value.status == T.TPCF_ESTATE


def test_product_package_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1204_6630_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "tpcf_oracle" not in src, f


def test_plan_refuses_the_kinds_with_a_third_catalog_size():
    """tpcf_plan takes (n_d, n_r) only: D1D2 and D2R pair a third catalog whose size it is not told."""
    with T.Context(4, [0.1, 10.0], "log") as c:
        for kind in (T.TPCF_D1D2, T.TPCF_D2R, 7, -1):
            with pytest.raises(T.TpcfError):
                c.plan(kind, 1000, 1000)
            with pytest.raises(T.TpcfError):
                c.plan_item_pairs(kind, 1000, 1000, 0)


def test_plan_numbering_under_a_partition_is_the_fixed_one():
    """With nparts > 1 the chunking is balanced for the constant 148 SMs on every rank (ranks on GPUs with
    different SM counts must enumerate the same items).  Without a GPU the context has not seen a device, so both
    numberings coincide here; what this pins is that setting and clearing a partition leaves the plan arithmetic intact."""
    with T.Context(4, [0.1, 10.0], "log") as c:
        base = [(k, c.plan(k, 430_000, 300_000)) for k in ("DD", "DR", "RR")]
        c.set_partition(1, 3)
        assert [(k, c.plan(k, 430_000, 300_000)) for k in ("DD", "DR", "RR")] == base
        c.set_partition(0, 1)
        assert [(k, c.plan(k, 430_000, 300_000)) for k in ("DD", "DR", "RR")] == base
