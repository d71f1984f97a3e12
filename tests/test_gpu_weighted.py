"""GPU parity of SURVEY.md NEXT-4 (PAPER.md:16 cross-correlations, PAPER.md:83, 89 extensions): the cross-catalog counts
D1D2 / D2R with their Landy-Szalay cross estimator, and the weighted sums of tpcf_count_weighted, against the fp64
oracle (orc_count_cross, orc_wsum_auto / orc_wsum_cross).  Counts: the usual bar (totals bit-exact, bins up to fp64 ties,
|dw| <= 1e-6).  Weighted sums: fp64 additions in an order that is not fixed, partial sums of at most 2^25 terms, so
|sum_gpu - sum_oracle| <= 2^-27 sum |w_i w_j| per bin plus the products of the <= STRICT pairs that
sit within fp64 rounding of an edge."""
import numpy as np
import pytest

import oracle
import paper_1204_6630_b200 as T
import synth
from test_gpu_parity import STRICT, assert_parity, assert_w, full

pytestmark = pytest.mark.gpu


def catalogs(nd, nr, n2):
    D, R, e, cfg = synth.make_config(2, n_d=nd, n_r=nr)
    D2 = synth.make_config(1, n_d=n2, n_r=16)[0] * np.array([3.0, 3.0])      # clumps on the same 30 x 30 deg patch
    return D, R, D2, e, cfg


@pytest.mark.parametrize("engine", ["tensor", "fast"])
def test_cross_catalog_counts_and_estimator(engine, oracle_threads):
    nd, nr, n2 = 20_000, 17_777, 9_000
    D, R, D2, e, cfg = catalogs(nd, nr, n2)
    d, r, d2 = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R), oracle.radec_to_xyz(D2)
    o = {"D1D2": oracle.count_cross(d, d2, e, validate=True, threads=oracle_threads),
         "DR": oracle.count_cross(d, r, e, validate=True, threads=oracle_threads),
         "D2R": oracle.count_cross(d2, r, e, validate=True, threads=oracle_threads),
         "RR": oracle.count_auto(r, e, validate=True, threads=oracle_threads)}
    want = {"D1D2": nd * n2, "DR": nd * nr, "D2R": n2 * nr, "RR": nr * (nr - 1) // 2}
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.set_engine(engine)
        c.set_tensor_share_limit(1.0)
        with pytest.raises(T.TpcfError) as ei:
            c.count("D1D2")
        assert ei.value.status == T.TPCF_ESTATE                       # D2 not loaded yet
        c.load("D", D)
        c.load("R", R)
        c.load("D2", D2)
        with pytest.raises(T.TpcfError):
            c.estimate_cross()
        g = {k: full(*c.count(k)) for k in want}
        for k in want:
            assert_parity(g[k], o[k], want[k])
        w12 = c.estimate_cross()
        rows = synth.subset_rows(n2, 300)
        sub = full(*c.count("D2R", rows))                             # rows index D2
        osub = oracle.count_rows(d2, rows, r, False, e, validate=True, threads=oracle_threads)
        assert_parity(sub, osub, 300 * nr)
    ref = oracle.estimate_cross(o["D1D2"].hist, o["DR"].hist, o["D2R"].hist, o["RR"].hist, nd, n2, nr)      # pinned in test_oracle_pins.py
    assert_w(w12, ref)


def test_weighted_sums_match_oracle(oracle_threads):
    nd, nr, n2 = 12_000, 9_000, 3_000
    D, R, D2, e, cfg = catalogs(nd, nr, n2)
    d, r, d2 = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R), oracle.radec_to_xyz(D2)
    rng = synth.SplitMix(97)
    wd, wr, w2 = 0.5 + rng.uniform(nd), rng.normal(nr), np.exp(rng.normal(n2))          # positive, signed, heavy-tailed
    o = {"DD": oracle.wsum_auto(d, wd, e, threads=oracle_threads), "DR": oracle.wsum_cross(d, wd, r, wr, e, threads=oracle_threads),
         "RR": oracle.wsum_auto(r, wr, e, threads=oracle_threads), "D1D2": oracle.wsum_cross(d, wd, d2, w2, e, threads=oracle_threads)}
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.load("D", D)
        c.load("R", R)
        with pytest.raises(T.TpcfError) as ei:
            c.count_weighted("DD")
        assert ei.value.status == T.TPCF_ESTATE                       # no weights yet
        with pytest.raises(T.TpcfError) as ei:
            c.set_weights("D", wd[:-1])
        assert ei.value.status == T.TPCF_EINVAL
        bad = wd.copy()
        bad[5] = np.inf
        with pytest.raises(T.TpcfError):
            c.set_weights("D", bad)
        c.set_weights("D", wd)
        c.set_weights("R", wr)
        c.load("D2", D2)
        c.set_weights("D2", w2)
        wmax = {"DD": wd.max() ** 2, "DR": wd.max() * np.abs(wr).max(), "RR": np.abs(wr).max() ** 2, "D1D2": wd.max() * w2.max()}
        for k in o:
            h, u, ov = c.count_weighted(k)
            got = np.concatenate([[u], h, [ov]])
            ref = np.concatenate([[o[k].under], o[k].hist, [o[k].over]])
            tol = 2.0 ** -27 * o[k].abs_hist + STRICT * wmax[k]
            assert np.all(np.abs(got - ref) <= tol), (k, float(np.max(np.abs(got - ref) / np.maximum(o[k].abs_hist, 1e-300))))
        # unit weights: the sums are the pair counts, exactly (integers below 2^53 in any order)
        c.set_weights("D", np.ones(nd))
        c.set_weights("R", np.ones(nr))
        for k in ("DD", "DR", "RR"):
            h, u, ov = c.count_weighted(k)
            hc, uc, oc = c.count(k)
            assert np.array_equal(h, hc.astype(np.float64)) and (u, ov) == (float(uc), float(oc)), k
        c.load("D", D)                                                # a reload drops the weights of that slot
        with pytest.raises(T.TpcfError) as ei:
            c.count_weighted("DR")
        assert ei.value.status == T.TPCF_ESTATE
