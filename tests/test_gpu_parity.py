"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element, on the same
seeded inputs (BASELINE.json acceptance):

  * totals bit-exact (under + bins + over == number of pairs, as integers);
  * every bin within tol_k = number of pairs whose fp64 cos(theta) lies within 1e-6 of one of its edges
    (the oracle reports it) -- and, because the fast engine rechecks guard-band pairs in fp64, in fact equal
    up to the handful of pairs that sit within fp64 rounding of an edge (STRICT below);
  * |w_gpu - w_oracle| <= 1e-6;
  * configs too large for the oracle: seeded 2,000-row subset against all j, plus identities on the full run.
"""
import json
import math
import os

import numpy as np
import pytest

import oracle
import paper_1204_6630_b200 as T
import synth

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLD = json.load(open(os.path.join(ROOT, "tests", "golden", "hand_catalogs.json")))
STRICT = 4          # pairs per histogram allowed to differ (fp64 ties: acos(dot) vs chord within ~1e-15)
W_TOL = 1e-6        # BASELINE.json: |w_gpu - w_oracle| <= 1e-6 absolute
KINDS = ("DD", "DR", "RR")


@pytest.fixture(autouse=True)
def fast_engine_in_this_module(monkeypatch):
    """The tests of this file pin TPCF_ENGINE_FAST (the FFMA2 kernel); tests/test_gpu_tensor.py repeats them for the
    library's default engine, TPCF_ENGINE_TENSOR."""
    init = T.Context.__init__

    def init_fast(self, *a, **k):
        init(self, *a, **k)
        self.set_engine("fast")

    monkeypatch.setattr(T.Context, "__init__", init_fast)


def full(h, u, o):
    return np.concatenate([[u], np.asarray(h, dtype=np.int64), [o]]).astype(np.int64)


def gpu_all(ctx, rows=None):
    out = {}
    for k in KINDS:
        r = None if rows is None else rows[k]
        out[k] = full(*ctx.count(k, r))
    return out


def orc_full(c):
    return full(c.hist, c.under, c.over)


def orc_tol(c):
    """tol for [under, bins..., over]: pairs within 1e-6 (in cos) of the slot's edges."""
    near = c.near.astype(np.int64)
    return np.concatenate([[near[0]], near[:-1] + near[1:], [near[-1]]])


def assert_parity(g, oc, expect_total):
    o = orc_full(oc)
    assert int(g.sum()) == expect_total == int(o.sum())
    d = np.abs(g - o)
    assert np.all(d <= orc_tol(oc)), "bin differs by more than the pairs within 1e-6 of its edges"
    assert int(d.sum()) <= STRICT, f"{int(d.sum())} pairs differ; the fp64 recheck should leave only fp64 ties"


def assert_w(wg, wo):
    assert np.array_equal(np.isnan(wg), np.isnan(wo))
    ok = ~np.isnan(wo)
    assert np.all(np.abs(wg[ok] - wo[ok]) <= W_TOL)


def oracle_all(D, R, e, threads):
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    return {"DD": oracle.count_auto(d, e, validate=True, threads=threads),
            "DR": oracle.count_cross(d, r, e, validate=True, threads=threads),
            "RR": oracle.count_auto(r, e, validate=True, threads=threads)}


def totals(nd, nr):
    return {"DD": nd * (nd - 1) // 2, "DR": nd * nr, "RR": nr * (nr - 1) // 2}


# ---------------------------------------------------------------------------------- full histograms
@pytest.mark.parametrize("idx,nd,nr", [(1, None, None), (2, 20_000, 17_777), (5, 20_000, 20_000), (3, 9_000, 11_111),
                                       (4, 6_000, 12_345)])
def test_full_histograms_and_w_match_oracle(idx, nd, nr, oracle_threads):
    D, R, e, cfg = synth.make_config(idx, n_d=nd, n_r=nr)
    nd, nr = D.shape[0], R.shape[0]
    o = oracle_all(D, R, e, oracle_threads)
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.load("D", D)
        c.load("R", R)
        g = gpu_all(c)
        wg = c.estimate()
        c.set_engine("exact64")
        gx = gpu_all(c)
    for k in KINDS:
        assert_parity(g[k], o[k], totals(nd, nr)[k])
        np.testing.assert_array_equal(g[k], gx[k])            # fast engine == fp64 engine, bit for bit
        assert o[k].mismatch == 0                             # oracle's own acos-vs-asin self check (P9)
    wo = oracle.estimate(o["DD"].hist, o["DR"].hist, o["RR"].hist, nd, nr)
    assert_w(wg, wo)
    assert_w(T.tpcf_estimate_from(g["DD"][1:-1], g["DR"][1:-1], g["RR"][1:-1], nd, nr), wo)


@pytest.mark.slow
def test_config2_full_size_full_histograms(oracle_threads):
    """Config 2 at its full 100k x 100k (2e10 pairs): the oracle runs threaded on the host cores."""
    D, R, e, cfg = synth.make_config(2)
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.load("D", D)
        c.load("R", R)
        g = gpu_all(c)
        wg = c.estimate()
    o = {"DD": oracle.count_auto(d, e, threads=oracle_threads), "DR": oracle.count_cross(d, r, e, threads=oracle_threads),
         "RR": oracle.count_auto(r, e, threads=oracle_threads)}
    for k in KINDS:
        of = orc_full(o[k])
        assert int(g[k].sum()) == totals(100_000, 100_000)[k] == int(of.sum())
        assert int(np.abs(g[k] - of).sum()) <= STRICT          # stricter than tol_k, which would need validate=True
    assert_w(wg, oracle.estimate(o["DD"].hist, o["DR"].hist, o["RR"].hist, 100_000, 100_000))


# ---------------------------------------------------------------------------------- large configs: row subsets
@pytest.mark.parametrize("idx,nrows", [(3, 2000), (4, 2000), (5, 2000)])
def test_full_size_configs_on_row_subset_and_identities(idx, nrows, oracle_threads):
    D, R, e, cfg = synth.make_config(idx)
    nd, nr = D.shape[0], R.shape[0]
    rows_d, rows_r = synth.subset_rows(nd, nrows, 12345), synth.subset_rows(nr, nrows, 12346)
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.load("D", D)
        c.load("R", R)
        g = gpu_all(c, {"DD": rows_d, "DR": rows_d, "RR": rows_r})
        with pytest.raises(T.TpcfError) as ei:          # a subset count is not a full count
            c.estimate()
        assert ei.value.status == T.TPCF_ESTATE
        o = {"DD": oracle.count_rows(d, rows_d, d, True, e, validate=True, threads=oracle_threads),
             "DR": oracle.count_rows(d, rows_d, r, False, e, validate=True, threads=oracle_threads),
             "RR": oracle.count_rows(r, rows_r, r, True, e, validate=True, threads=oracle_threads)}
        want = {"DD": nrows * (nd - 1), "DR": nrows * nr, "RR": nrows * (nr - 1)}
        for k in KINDS:
            assert_parity(g[k], o[k], want[k])
        # the full run, in the launch configuration bench.py times: totals identity (P2) ...
        f = gpu_all(c)
        for k in KINDS:
            assert int(f[k].sum()) == totals(nd, nr)[k]
        stats = c.stats()
        assert stats["work_items"] == c.plan("RR", nd, nr)
        # ... the partition identity (P5: the histogram does not depend on how the work is split) ...
        parts = []
        for p in range(3):
            c.set_partition(p, 3)
            parts.append(full(*c.count("DR")))
        c.set_partition(0, 1)
        np.testing.assert_array_equal(sum(parts), f["DR"])
        # ... a wider guard band changes nothing (the band is wide enough) ...
        c.set_guard_scale(4.0)
        np.testing.assert_array_equal(full(*c.count("DD")), f["DD"])
        c.set_guard_scale(1.0)
        # ... and DR(D, R) == DR(R, D)
        c.load("D", R)
        c.load("R", D)
        np.testing.assert_array_equal(full(*c.count("DR")), f["DR"])
    # uniform randoms: RR pair fraction per bin vs the closed form for the footprint-free case (config 4, full sky)
    if idx == 4:
        exp = totals(nd, nr)["RR"] * (np.cos(np.radians(e[:-1])) - np.cos(np.radians(e[1:]))) / 2.0
        assert np.all(np.abs(f["RR"][1:-1] - exp) <= 6.0 * np.sqrt(exp) + 1.0)          # P6 at 2e12 pairs
        assert abs(int(f["RR"][-1]) - totals(nd, nr)["RR"] / 2) <= 6.0 * math.sqrt(totals(nd, nr)["RR"] / 2)


@pytest.mark.parametrize("idx,nd,nr", [(3, 60_000, 50_000), (5, 40_000, 30_000), (2, 30_000, 30_000)])
def test_every_kernel_path_gives_the_same_histogram(idx, nd, nr):
    """The window loops (1-3 candidate edges per block), the per-pair cell lookup, the fp64 blocks and the plain fp64
    engine are four ways to the same integers: bit-identical histograms, and the path
    statistics show that each of them was really exercised."""
    D, R, e, cfg = synth.make_config(idx, n_d=nd, n_r=nr)
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.load("D", D)
        c.load("R", R)
        win, used = {}, np.zeros(6, dtype=np.int64)
        for k in KINDS:
            win[k] = full(*c.count(k))
            st = c.stats()
            used += np.asarray(st["win_blocks"], dtype=np.int64)
            assert int(win[k].sum()) == totals(nd, nr)[k] == st["pairs"]
        assert used[0] + used[1] + used[2] > 0, "no block took a window loop"
        assert used[3] > 0, "no block took the cell-lookup path (diagonal chunks always do)"
        c.set_window(False)
        for k in KINDS:
            np.testing.assert_array_equal(full(*c.count(k)), win[k])
            assert sum(c.stats()["win_blocks"][:3]) == 0
        c.set_window(True)
        c.set_guard_scale(8.0)                       # 8x wider guard bands: more fp64 rechecks, same integers
        np.testing.assert_array_equal(full(*c.count("DR")), win["DR"])
        c.set_guard_scale(1.0)
        c.set_engine("exact64")
        for k in KINDS:
            np.testing.assert_array_equal(full(*c.count(k)), win[k])


@pytest.mark.parametrize("idx,nd,nr", [(3, 60_000, 50_000), (2, 30_000, 30_000), (5, 40_000, 30_000), (4, 50_000, 70_000)])
def test_pruning_mode_gives_the_same_histograms(idx, nd, nr):
    """SURVEY.md NEXT-3 (the k-tree idea, at block granularity, as a separately named mode): blocks whose
    windows reach no bin edge are added wholesale.  Same integers as the brute-force count; the statistics show that
    blocks really were skipped."""
    D, R, e, cfg = synth.make_config(idx, n_d=nd, n_r=nr)
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.load("D", D)
        c.load("R", R)
        brute = {k: full(*c.count(k)) for k in KINDS}
        assert c.stats()["pruned_blocks"] == 0
        c.set_pruning(True)
        pruned = 0
        for k in KINDS:
            np.testing.assert_array_equal(full(*c.count(k)), brute[k])
            st = c.stats()
            pruned += st["pruned_blocks"]
            assert st["pairs"] == totals(nd, nr)[k]
        assert pruned > 0                    # on config 5 only the blocks of padding rows: its bins are finer than any block
        rows = synth.subset_rows(nd, 500)
        a = full(*c.count("DD", rows))
        c.set_pruning(False)
        np.testing.assert_array_equal(full(*c.count("DD", rows)), a)


@pytest.mark.parametrize("engine", ["fast", "tensor"])
def test_count_all_equals_three_counts(engine):
    """tpcf_count_all / tpcf_count_all_async (the three pair kernels in flight together on three streams) against three
    tpcf_count calls: same integers, stored for tpcf_estimate, repeatable, and after a catalog was replaced."""
    import torch
    D, R, e, cfg = synth.make_config(2, n_d=30_000, n_r=25_000)
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.set_engine(engine)
        c.load("D", D)
        c.load("R", R)
        one = {k: c.count(k) for k in KINDS}
        w1 = c.estimate()
        for _ in range(2):
            al = c.count_all()
            for k in KINDS:
                np.testing.assert_array_equal(al[k][0], one[k][0])
                assert al[k][1:] == one[k][1:]
        np.testing.assert_array_equal(c.estimate(), w1)
        out = torch.zeros(3, cfg.nbins + 2, dtype=torch.int64, device="cuda")
        st = torch.cuda.Stream()
        c.set_stream(st.cuda_stream)
        for _ in range(3):
            c.count_all_async(out)
        st.synchronize()
        for i, k in enumerate(KINDS):
            np.testing.assert_array_equal(out[i].cpu().numpy(), full(*one[k]))
        c.load("D", R[:20_000], stream=st.cuda_stream)      # replace D: the next count_all sees the new catalog
        al = c.count_all()
        assert int(al["DD"][0].sum()) + al["DD"][1] + al["DD"][2] == 20_000 * 19_999 // 2
        np.testing.assert_array_equal(al["RR"][0], one["RR"][0])
        c.set_stream(0)


def test_sparse_catalogs_fall_back_to_fp64_blocks(oracle_threads):
    """A few hundred points on the whole sky: every bounding radius exceeds the cap of the fp32 error bound, so all
    blocks are classified from the fp64 coordinates -- and still match the oracle."""
    rng = np.random.default_rng(11)
    def sky(n):
        return np.stack([rng.uniform(0.0, 360.0, n), np.degrees(np.arcsin(rng.uniform(-1.0, 1.0, n)))], 1)
    D, R = sky(700), sky(900)
    e = np.linspace(0.0, 180.0, 37)
    with T.Context(36, e, "explicit") as c:
        c.load("D", D)
        c.load("R", R)
        g = gpu_all(c)
        assert c.stats()["win_blocks"][5] > 0
        o = oracle_all(D, R, c.edges(), oracle_threads)
        for k in KINDS:
            assert_parity(g[k], o[k], totals(700, 900)[k])


def test_config5_shuffled_rows_give_the_same_histogram():
    D, R, e, cfg = synth.make_config(5, n_d=60_000, n_r=1000)
    S, _, _, _ = synth.make_config(5, n_d=60_000, n_r=1000, shuffle_d=True)
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.load("D", D)
        a = full(*c.count("DD"))
        c.load("D", S)
        b = full(*c.count("DD"))
    np.testing.assert_array_equal(a, b)                      # P5 permutation invariance


# ---------------------------------------------------------------------------------- closed forms on the GPU
def test_ring_closed_form_at_paper_scale():
    """P4: N points equally spaced on a great circle: separation m*360/N occurs N times (N/2 times for the
    antipodal one).  360,000 points = 6.5e10 pairs, no oracle run needed; bins of 250 separations each."""
    n, per = 360_000, 250
    delta = 360.0 / n
    ring = synth.great_circle_ring(n)
    e = (np.arange(0, n // 2 + 1, per) + 0.5) * delta
    e[-1] = 180.0
    nb = len(e) - 1
    with T.Context(nb, e, "explicit") as c:
        c.load("D", ring)
        h, u, o = c.count("DD")
        want = np.full(nb, per * n, dtype=np.uint64)
        want[-1] = (per - 1) * n + n // 2
        np.testing.assert_array_equal(h, want)
        assert (u, o) == (0, 0)
    # cross version: second ring shifted by delta/2 -> separations (m + 1/2) delta, 2N each
    e2 = np.arange(0, n // 2 + 1, per) * delta
    e2[-1] = 180.0
    with T.Context(len(e2) - 1, e2, "explicit") as c:
        c.load("D", ring)
        c.load("R", synth.great_circle_ring(n, phase_deg=delta / 2))
        h, u, o = c.count("DR")
        np.testing.assert_array_equal(h, np.full(len(e2) - 1, 2 * per * n, dtype=np.uint64))
        assert (u, o) == (0, 0)


@pytest.mark.parametrize("name", ["equator", "meridian", "wrap", "poles"])
@pytest.mark.parametrize("engine", ["fast", "exact64"])
def test_hand_catalogs(name, engine):
    g = GOLD[name]
    e = np.arange(-0.5, 181.0, 1.0)
    e[0], e[-1] = 0.0, 180.0
    with T.Context(181, e, "explicit") as c:
        c.set_engine(engine)
        c.load("D", np.asarray(g["radec"], dtype=np.float64))
        h, u, o = c.count("DD")
    want = np.zeros(181, dtype=np.uint64)
    for s in g["separations"]:
        want[int(round(s))] += 1
    np.testing.assert_array_equal(h, want)
    assert (u, o) == (0, 0)


def test_octahedron_closed_last_bin_and_cross_counts():
    g = GOLD["octahedron"]
    with T.Context(3, np.array(g["edges"], dtype=np.float64), "explicit") as c:
        c.load("D", np.asarray(g["radec"], dtype=np.float64))
        h, u, o = c.count("DD")
        np.testing.assert_array_equal(h, np.array(g["hist"], dtype=np.uint64))
        assert (u, o) == (0, 0)
    e = np.arange(-0.5, 21.0, 1.0)
    e[0] = 0.0
    with T.Context(len(e) - 1, e, "explicit") as c:
        c.load("D", np.array([[0, 0], [1, 0]], dtype=np.float32))
        c.load("R", np.array([[3, 0], [7, 0], [15, 0]], dtype=np.float32))
        h, u, o = c.count("DR")
    want = np.zeros(21, dtype=np.uint64)
    for s in (3, 7, 15, 2, 6, 14):
        want[s] += 1
    np.testing.assert_array_equal(h, want)


def test_small_angle_pairs_fp32_rows():
    for name in ("small_ra", "small_dec"):
        g = GOLD[name]
        th = g["theta"]
        with T.Context(1, [th * (1 - 1e-6), th * (1 + 1e-6)], "explicit") as c:
            c.load("D", np.asarray(g["radec"], dtype=np.float64))
            h, u, o = c.count("DD")
            assert (int(h[0]), u, o) == (1, 0, 0)
            assert c.stats()["rechecked"] == 1        # bins this narrow are decided by the fp64 path


# ---------------------------------------------------------------------------------- edge cases
@pytest.mark.parametrize("nd,nr", [(1, 1), (2, 3), (1023, 1025), (1024, 1024), (2049, 1), (3000, 5000)])
def test_ragged_sizes_totals_and_oracle(nd, nr, oracle_threads):
    D, R, _, _ = synth.make_config(1, n_d=nd, n_r=nr)
    e = np.array([0.0, 0.05, 0.5, 2.0, 180.0])
    o = oracle_all(D, R, e, 1)
    with T.Context(4, e, "explicit") as c:
        c.load("D", D)
        c.load("R", R)
        g = gpu_all(c)
    for k in KINDS:
        assert_parity(g[k], o[k], totals(nd, nr)[k])
        assert g[k][0] == 0 and g[k][-1] == 0         # edges span [0, 180]: nothing under or over


def test_duplicate_rows_theta_zero():
    D = np.array([[10.0, 20.0], [10.0, 20.0], [10.0, 20.0], [50.0, -30.0]])
    with T.Context(2, [0.0, 1.0, 180.0], "explicit") as c:      # e_0 = 0: theta = 0 belongs to bin 0
        c.load("D", D)
        c.load("R", D)
        assert tuple(full(*c.count("DD"))) == (0, 3, 3, 0)
        assert tuple(full(*c.count("DR"))) == (0, 10, 6, 0)      # 4 self pairs + 6 duplicate pairs at 0
        assert tuple(full(*c.count("DD", rows=[0, 3]))) == (0, 2, 4, 0)
    with T.Context(2, [0.5, 1.0, 180.0], "explicit") as c:      # e_0 > 0: theta = 0 is "under"
        c.load("D", D)
        assert tuple(full(*c.count("DD"))) == (3, 0, 3, 0)


def test_max_bins_linear_over_the_whole_range(oracle_threads):
    D, R, _, _ = synth.make_config(4, n_d=3000, n_r=2000)
    e = synth.edges(4096, 0.0, 180.0, "linear")
    o = oracle_all(D, R, e, oracle_threads)
    with T.Context(4096, [0.0, 180.0], "linear") as c:
        np.testing.assert_allclose(c.edges(), e, rtol=1e-14)
        c.load("D", D)
        c.load("R", R)
        g = gpu_all(c)
    for k in KINDS:
        assert_parity(g[k], o[k], totals(3000, 2000)[k])


def test_error_paths():
    D, R, e, cfg = synth.make_config(1, n_d=100, n_r=50)
    with T.Context(cfg.nbins, e, "explicit") as c:
        for fn in (lambda: c.count("DD"), lambda: c.count("DR")):
            with pytest.raises(T.TpcfError) as ei:
                fn()
            assert ei.value.status == T.TPCF_ESTATE
        c.load("D", D)
        with pytest.raises(T.TpcfError) as ei:
            c.count("DR")
        assert ei.value.status == T.TPCF_ESTATE
        c.load("R", R)
        for rows in ([100], [-1], [0, 5, 1000]):
            with pytest.raises(T.TpcfError) as ei:
                c.count("DD", rows=rows)
            assert ei.value.status == T.TPCF_EINVAL
        c.count("DD")
        c.count("DR")
        with pytest.raises(T.TpcfError) as ei:
            c.estimate()
        assert ei.value.status == T.TPCF_ESTATE               # RR missing
        c.count("RR")
        c.estimate()
        c.load("R", R)                                        # reloading R invalidates DR and RR
        with pytest.raises(T.TpcfError):
            c.estimate()
        for bad in ([[0.0, 91.0]], [[float("nan"), 0.0]], [[float("inf"), 0.0]]):
            with pytest.raises(T.TpcfError) as ei:
                c.load("D", np.asarray(bad, dtype=np.float64))
            assert ei.value.status == T.TPCF_EINVAL
        with pytest.raises(T.TpcfError):
            c.load("D", np.zeros((0, 2)))


def test_device_resident_inputs_streams_and_async_count():
    import torch
    D, R, e, cfg = synth.make_config(2, n_d=5000, n_r=7000)        # float32 rows
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.load("D", D)
        c.load("R", R)
        ref = gpu_all(c)
    st = torch.cuda.Stream()
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.set_stream(st.cuda_stream)
        c.load("D", torch.from_numpy(D).cuda(), stream=st.cuda_stream)       # device pointer in
        c.load("R", torch.from_numpy(R).pin_memory(), stream=st.cuda_stream)  # pinned host pointer in
        outs = {k: torch.zeros(cfg.nbins + 2, dtype=torch.int64, device="cuda") for k in KINDS}
        for k in KINDS:
            c.count_async(k, outs[k])
        st.synchronize()
        for k in KINDS:
            np.testing.assert_array_equal(outs[k].cpu().numpy(), ref[k])
    # float64 copies of the float32 rows give the same unit vectors, hence the same histogram
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.load("D", D.astype(np.float64))
        c.load("R", R.astype(np.float64))
        np.testing.assert_array_equal(full(*c.count("DR")), ref["DR"])
