"""GPU parity of the 3-D variant ("our results are extendible to the 3-dimensional
variant as well"): tpcf_create_r + tpcf_load_xyz + the same count / estimate calls, against the fp64 oracle
orc_count_*_xyz (oracle/tpcf_oracle.c: r = sqrt(dx^2 + dy^2 + dz^2) against the r edges), element by element.
Tolerance as for the angular path: totals bit-exact; a bin may differ only by pairs within near_tol = 1e-9 r_max of one
of its edges (the oracle reports them; in practice only fp64 ties: at most STRICT pairs per histogram); |dw| <= 1e-6."""
import numpy as np
import pytest

import oracle
import paper_1204_6630_b200 as T
import synth
from test_gpu_parity import KINDS, STRICT, assert_w, full, totals

pytestmark = pytest.mark.gpu
ENGINES = ("tensor", "fast", "exact64")


def box_ctx(nbins, edges, max_abs, engine="tensor", mode="explicit"):
    c = T.Context(nbins, edges, mode, max_abs_coord=max_abs)
    c.set_engine(engine)
    c.set_tensor_share_limit(1.0)          # "tensor" means pair_tensor_kernel here, whatever the block mix
    return c


def assert_parity_xyz(g, oc, expect_total):
    o = full(oc.hist, oc.under, oc.over)
    assert int(g.sum()) == expect_total == int(o.sum())
    near = oc.near.astype(np.int64)
    tol = np.concatenate([[near[0]], near[:-1] + near[1:], [near[-1]]])
    d = np.abs(g - o)
    assert np.all(d <= tol) and int(d.sum()) <= STRICT, (d.sum(), d.max())


@pytest.mark.parametrize("engine", ENGINES)
def test_cubic_lattice_hand_multiplicities(engine):
    """3x3x3 lattice scaled by 2.5 and shifted: 54, 72, 32, 27, 72, 48, 18, 24, 4 pairs at r^2 / 6.25 = 1, 2, 3, 4, 5, 6, 8,
    9, 12 (tests/test_oracle_pins.py X1 derives them); edges on the distances 2.5 and 5.0 themselves test the inclusivity."""
    want = {1: 54, 2: 72, 3: 32, 4: 27, 5: 72, 6: 48, 8: 18, 9: 24, 12: 4}
    x = synth.cubic_lattice(3) * 2.5 + np.array([7.0, -3.0, 11.0])
    d2s = sorted(want)
    r = 2.5 * np.sqrt(np.array(d2s, dtype=np.float64))
    e = np.concatenate([[0.5 * r[0]], 0.5 * (r[:-1] + r[1:]), [r[-1] + 1.0]])
    with box_ctx(len(e) - 1, e, 20.0, engine) as c:
        c.load("D", x)
        h, u, o = c.count("DD")
        assert list(h) == [want[d] for d in d2s] and u == 0 and o == 0
    with box_ctx(1, [2.5, 5.0], 20.0, engine) as c:
        c.load("D", x)
        h, u, o = c.count("DD")
        assert h[0] == sum(v for d, v in want.items() if 1 <= d <= 4) and u == 0
        assert o == sum(v for d, v in want.items() if d > 4)


@pytest.mark.parametrize("nd,nr,side,nbins,rmin,rmax,mode", [(20_000, 17_777, 1000.0, 30, 1.0, 200.0, "log"),
                                                             (9_000, 6_000, 80.0, 64, 0.0, 40.0, "linear")])
def test_clustered_box_full_histograms_and_xi_match_oracle(nd, nr, side, nbins, rmin, rmax, mode, oracle_threads):
    D, R, e = synth.make_box_config(nd, nr, side=side, nbins=nbins, r_min=rmin, r_max=rmax, mode=mode)
    tol = 1e-9 * rmax
    o = {"DD": oracle.count_auto_xyz(D, e, near_tol=tol, threads=oracle_threads),
         "DR": oracle.count_cross_xyz(D, R, e, near_tol=tol, threads=oracle_threads),
         "RR": oracle.count_auto_xyz(R, e, near_tol=tol, threads=oracle_threads)}
    res = {}
    for engine in ENGINES:
        with box_ctx(nbins, [rmin, rmax], side, engine, mode) as c:
            np.testing.assert_allclose(c.edges(), e, rtol=1e-14)
            c.load("D", D)
            c.load("R", R)
            res[engine] = {k: full(*c.count(k)) for k in KINDS}
            w = c.estimate()
            if engine == "tensor":
                used = np.zeros(6, dtype=np.int64)
                for k in KINDS:
                    c.count(k)
                    used += np.asarray(c.stats()["win_blocks"], dtype=np.int64)
                assert used[:3].sum() > 0 and used[3] + used[4] > 0      # window loops and the cell lookup both ran
        for k in KINDS:
            assert_parity_xyz(res[engine][k], o[k], totals(nd, nr)[k])
        assert_w(w, oracle.estimate(o["DD"].hist, o["DR"].hist, o["RR"].hist, nd, nr))
    for k in KINDS:
        np.testing.assert_array_equal(res["tensor"][k], res["exact64"][k])
        np.testing.assert_array_equal(res["fast"][k], res["exact64"][k])


def test_paper_scale_box_on_row_subset_and_identities(oracle_threads):
    """430k + 430k rows in a 1000-box, 40 log bins 1-200: a seeded 2000-row subset against all j (the oracle needs
    ~1.7e9 pairs), totals of the full count, f32 rows."""
    D, R, e = synth.make_box_config()
    nd, nr = D.shape[0], R.shape[0]
    rows = {"DD": synth.subset_rows(nd, 2000), "DR": synth.subset_rows(nd, 2000), "RR": synth.subset_rows(nr, 2000)}
    tol = 1e-9 * 200.0
    o = {"DD": oracle.count_rows_xyz(D, rows["DD"], D, True, e, near_tol=tol, threads=oracle_threads),
         "DR": oracle.count_rows_xyz(D, rows["DR"], R, False, e, near_tol=tol, threads=oracle_threads),
         "RR": oracle.count_rows_xyz(R, rows["RR"], R, True, e, near_tol=tol, threads=oracle_threads)}
    want = {"DD": 2000 * (nd - 1), "DR": 2000 * nr, "RR": 2000 * (nr - 1)}
    with box_ctx(40, e, 1000.0) as c:
        c.load("D", D)
        c.load("R", R)
        for k in KINDS:
            assert_parity_xyz(full(*c.count(k, rows[k])), o[k], want[k])
        f = {k: full(*c.count(k)) for k in KINDS}
        for k in KINDS:
            assert int(f[k].sum()) == totals(nd, nr)[k]
        c.set_engine("fast")
        for k in KINDS:
            np.testing.assert_array_equal(full(*c.count(k)), f[k])


def test_unit_vectors_with_chord_edges_reproduce_the_angular_histogram():
    """The identity that ties the 3-D path to the angular one (oracle pin X4): unit vectors fed as xyz with r edges
    2 sin(theta_k / 2) give the angular histogram."""
    D, R, e, cfg = synth.make_config(2, n_d=30_000, n_r=20_000)
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.load("D", D)
        c.load("R", R)
        ang = {k: full(*c.count(k)) for k in KINDS}
    with box_ctx(cfg.nbins, 2.0 * np.sin(np.radians(e) / 2.0), 1.0) as c:
        c.load("D", d)
        c.load("R", r)
        for k in KINDS:
            g = full(*c.count(k))
            assert int(np.abs(g - ang[k]).sum()) <= STRICT and int(g.sum()) == int(ang[k].sum())


def test_xyz_error_paths():
    x = synth.uniform_box(100, 10.0, synth.SplitMix(3))
    for bad in ((4, [0.0, 1.0], "log"), (4, [2.0, 1.0], "linear"), (2, [0.0, 1.0, 1.0], "explicit"), (4, [1.0, 100.0], "linear")):
        with pytest.raises(T.TpcfError) as ei:
            T.tpcf_create_r(bad[0], bad[1], bad[2], 10.0)           # the last one: r_max beyond the largest separation
        assert ei.value.status == T.TPCF_EINVAL
    with pytest.raises(T.TpcfError):
        T.tpcf_create_r(4, [1.0, 2.0], "linear", 0.0)
    with box_ctx(4, [0.1, 5.0], 10.0, mode="log") as c:
        with pytest.raises(T.TpcfError) as ei:
            T.tpcf_load(c.handle, T.TPCF_D, np.zeros((5, 2)))       # angular rows into a 3-D context
        assert ei.value.status == T.TPCF_ESTATE
        y = x.copy()
        y[17, 1] = 10.5                                             # beyond max_abs_coord
        with pytest.raises(T.TpcfError) as ei:
            c.load("D", y)
        assert ei.value.status == T.TPCF_EINVAL
        y[17, 1] = np.nan
        with pytest.raises(T.TpcfError):
            c.load("D", y)
        c.load("D", x.astype(np.float32))
        h, u, o = c.count("DD")
        assert int(h.sum()) + u + o == 100 * 99 // 2
    with T.Context(4, [0.1, 5.0], "log") as c:
        with pytest.raises(T.TpcfError) as ei:
            T.tpcf_load_xyz(c.handle, T.TPCF_D, x)
        assert ei.value.status == T.TPCF_ESTATE
