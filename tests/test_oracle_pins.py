"""Pins for the fp64 oracle against things that are NOT the oracle.

Every pin is chosen so that a plausible slip in oracle/tpcf_oracle.c (dropped term, wrong sign or
index, transposed operand, wrong edge convention, wrong normalisation in Eq. 1) fails at least one.
None of these tests touches the CUDA library.
"""
import json
import math
import os

import numpy as np
import pytest

import oracle
import synth

GOLD = json.load(open(os.path.join(os.path.dirname(__file__), "golden", "hand_catalogs.json")))


def xyz_of(radec):
    return oracle.radec_to_xyz(np.asarray(radec, dtype=np.float64))


def unit_bins(lo, hi):
    """Unit-width bins centred on the integers lo..hi: edges lo-0.5, ..., hi+0.5."""
    return np.arange(lo - 0.5, hi + 1.0, 1.0)


# ------------------------------------------------------------------ P1 hand catalogs
@pytest.mark.parametrize("name", ["equator", "meridian", "wrap", "poles"])
def test_p1_hand_separations(name):
    g = GOLD[name]
    e = unit_bins(0, 180)                      # bins centred on 0..180 deg
    e[0] = 0.0
    e[-1] = 180.0
    c = oracle.count_auto(xyz_of(g["radec"]), e)
    want = np.zeros(181, dtype=np.uint64)
    for s in g["separations"]:
        want[int(round(s))] += 1
    assert c.under == 0 and c.over == 0
    np.testing.assert_array_equal(c.hist, want)
    n = len(g["radec"])
    assert c.total == n * (n - 1) // 2


def test_p1_octahedron_closed_last_bin_and_clamp():
    g = GOLD["octahedron"]
    c = oracle.count_auto(xyz_of(g["radec"]), np.array(g["edges"], dtype=np.float64))
    np.testing.assert_array_equal(c.hist, np.array(g["hist"], dtype=np.uint64))
    assert (c.under, c.over) == (0, 0)         # 180 deg lands IN the closed last bin, not in 'over'


def test_p1_interior_edge_is_lower_inclusive():
    """A5: bin k = [e_k, e_{k+1}), last bin closed.  The +x, +y, +z axes are pairwise exactly 90 deg apart
    in fp64 (dot products 6e-17 or 0, acos -> pi/2 exactly, pi/2*180/pi = 90.0), so with an interior edge
    AT 90 the 3 pairs belong to the upper bin, and with 90 as the LAST edge they are in range."""
    v = xyz_of([[0, 0], [90, 0], [0, 90]])
    c = oracle.count_auto(v, np.array([0.0, 90.0, 135.0, 180.0]))
    np.testing.assert_array_equal(c.hist, np.array([0, 3, 0], dtype=np.uint64))
    c = oracle.count_auto(v, np.array([10.0, 90.0]))
    assert (c.under, int(c.hist[0]), c.over) == (0, 3, 0)
    c = oracle.count_auto(v, np.array([90.0, 100.0]))
    assert (c.under, int(c.hist[0]), c.over) == (0, 3, 0)


def test_p1_general_pair_two_formulas():
    g = GOLD["general_pair"]
    (ra1, d1), (ra2, d2) = np.radians(g["radec"])
    law_of_cos = math.sin(d1) * math.sin(d2) + math.cos(d1) * math.cos(d2) * math.cos(ra1 - ra2)
    hav = math.sin((d2 - d1) / 2) ** 2 + math.cos(d1) * math.cos(d2) * math.sin((ra2 - ra1) / 2) ** 2
    assert abs(law_of_cos - g["cos_theta"]) < 1e-14
    assert abs(math.degrees(2 * math.asin(math.sqrt(hav))) - g["theta"]) < 1e-11
    v = xyz_of(g["radec"])
    assert abs(float(v[0] @ v[1]) - g["cos_theta"]) < 1e-14
    th = g["theta"]
    c = oracle.count_auto(v, np.array([th - 1e-9, th + 1e-9]))
    assert c.hist[0] == 1
    c = oracle.count_auto(v, np.array([th + 1e-9, th + 1.0]))
    assert (c.under, int(c.hist[0]), c.over) == (1, 0, 0)


@pytest.mark.parametrize("name", ["small_ra", "small_dec"])
def test_p1_small_angle_conditioning(name):
    g = GOLD[name]
    th = g["theta"]
    c = oracle.count_auto(xyz_of(g["radec"]), np.array([th * (1 - 1e-6), th * (1 + 1e-6)]), validate=True)
    assert c.hist[0] == 1 and c.mismatch == 0


def test_p1_cross_counts_on_hand_points():
    a = xyz_of(GOLD["equator"]["radec"][:2])        # RA 0, 1 on the equator
    b = xyz_of([[3, 0], [7, 0], [15, 0]])
    e = unit_bins(0, 20)
    e[0] = 0.0
    c = oracle.count_cross(a, b, e)
    want = np.zeros(21, dtype=np.uint64)
    for s in (3, 7, 15, 2, 6, 14):
        want[s] += 1
    np.testing.assert_array_equal(c.hist, want)
    assert c.total == 6


def test_p1_unit_vectors_convention():
    v = xyz_of([[0, 0], [90, 0], [0, 90], [180, 0], [45, 0], [0, -90]])
    want = np.array([[1, 0, 0], [0, 1, 0], [0, 0, 1], [-1, 0, 0], [math.sqrt(0.5), math.sqrt(0.5), 0], [0, 0, -1]])
    np.testing.assert_allclose(v, want, atol=1.3e-16)
    np.testing.assert_allclose(np.linalg.norm(xyz_of(synth.uniform_sphere(1000, synth.SplitMix(5))), axis=1), 1.0,
                               atol=3e-16)


def test_p1_float32_rows_widen_exactly():
    rd32 = np.array([[10.1, 20.2], [33.3, -44.4]], dtype=np.float32)
    np.testing.assert_array_equal(oracle.radec_to_xyz(rd32), oracle.radec_to_xyz(rd32.astype(np.float64)))


# ------------------------------------------------------------------ P2 totals identity
def test_p2_totals_auto_cross_rows():
    D, R, e, _ = synth.make_config(1, n_d=700, n_r=500)
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    full = np.array([0.0, 1.0, 50.0, 180.0])
    assert oracle.count_auto(d, full).total == 700 * 699 // 2
    assert oracle.count_auto(d, full).under == 0 and oracle.count_auto(d, full).over == 0
    assert oracle.count_cross(d, r, e).total == 700 * 500
    rows = synth.subset_rows(700, 50)
    assert oracle.count_rows(d, rows, d, True, e).total == 50 * 699
    assert oracle.count_rows(d, rows, r, False, e).total == 50 * 500


# ------------------------------------------------------------------ P3 library routine on tiny inputs
@pytest.mark.parametrize("idx,n", [(1, 900), (5, 700)])
def test_p3_numpy_histogram_of_arccos_gram(idx, n):
    D, R, e, _ = synth.make_config(idx, n_d=n, n_r=n // 2)
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    th = np.degrees(np.arccos(np.clip(d @ d.T, -1.0, 1.0)))[np.triu_indices(n, 1)]
    ref, _ = np.histogram(th, bins=e)
    c = oracle.count_auto(d, e)
    # the Gram matrix comes from BLAS (different summation order): allow the few ulp-tie pairs
    assert np.abs(c.hist.astype(np.int64) - ref).sum() <= 2
    assert c.under == int((th < e[0]).sum()) and c.over == int((th > e[-1]).sum())
    thx = np.degrees(np.arccos(np.clip(d @ r.T, -1.0, 1.0))).ravel()
    refx, _ = np.histogram(thx, bins=e)
    assert np.abs(oracle.count_cross(d, r, e).hist.astype(np.int64) - refx).sum() <= 2


def test_p3_explicit_python_loop_tiny():
    """Brute force in pure Python with math.acos on 40 points, exact equality."""
    D, _, e, _ = synth.make_config(1, n_d=40, n_r=8)
    d = oracle.radec_to_xyz(D)
    want = np.zeros(len(e) + 1, dtype=np.uint64)
    for i in range(40):
        for j in range(i + 1, 40):
            s = d[i, 0] * d[j, 0] + d[i, 1] * d[j, 1] + d[i, 2] * d[j, 2]
            th = math.acos(max(-1.0, min(1.0, s))) * 180.0 / math.pi
            if th < e[0]:
                want[0] += 1
            elif th > e[-1]:
                want[-1] += 1
            else:
                want[min(int(np.searchsorted(e, th, side="right")) - 1, len(e) - 2) + 1] += 1
    c = oracle.count_auto(d, e)
    np.testing.assert_array_equal(np.concatenate([[c.under], c.hist, [c.over]]).astype(np.uint64), want)


# ------------------------------------------------------------------ P4 ring closed form
@pytest.mark.parametrize("n", [360, 1000])
def test_p4_ring_auto(n):
    delta = 360.0 / n
    v = xyz_of(synth.great_circle_ring(n))
    e = (np.arange(0, n // 2 + 1) + 0.5) * delta      # bin m-1 = ((m-.5)d, (m+.5)d) holds separation m*d
    e[-1] = 180.0
    c = oracle.count_auto(v, e, validate=True)
    want = np.full(n // 2, n, dtype=np.uint64)
    want[-1] = n // 2                                  # antipodal pairs
    np.testing.assert_array_equal(c.hist, want)
    assert c.under == 0 and c.over == 0 and c.total == n * (n - 1) // 2 and c.mismatch == 0


def test_p4_ring_cross_shifted():
    n = 360
    a = xyz_of(synth.great_circle_ring(n))
    b = xyz_of(synth.great_circle_ring(n, phase_deg=0.5))
    c = oracle.count_cross(a, b, np.arange(0.0, 181.0, 1.0))   # separations (m+1/2) deg, 2n each
    np.testing.assert_array_equal(c.hist, np.full(180, 2 * n, dtype=np.uint64))
    assert c.total == n * n


# ------------------------------------------------------------------ P5 exact integer identities
def test_p5_identities():
    D, R, e, _ = synth.make_config(2, n_d=900, n_r=600)
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    a, b = d[:400], d[400:]
    H = lambda c: np.concatenate([[c.under], c.hist.astype(np.int64), [c.over]])
    dd = H(oracle.count_auto(d, e))
    # permutation invariance
    perm = np.argsort(synth.SplitMix(9).u64(900))
    np.testing.assert_array_equal(H(oracle.count_auto(d[perm], e)), dd)
    # additivity DD(A u B) = DD(A) + DD(B) + DR(A, B)
    np.testing.assert_array_equal(H(oracle.count_auto(a, e)) + H(oracle.count_auto(b, e)) + H(oracle.count_cross(a, b, e)), dd)
    # DR(D, R1 u R2) = DR(D, R1) + DR(D, R2); DR(a,b) = DR(b,a)
    dr = H(oracle.count_cross(d, r, e))
    np.testing.assert_array_equal(H(oracle.count_cross(d, r[:250], e)) + H(oracle.count_cross(d, r[250:], e)), dr)
    np.testing.assert_array_equal(H(oracle.count_cross(r, d, e)), dr)
    # DR(D, D) = 2 DD + N self pairs at theta = 0 (under, because e_0 = 0.01 > 0)
    self_dr = H(oracle.count_cross(d, d, e))
    want = 2 * dd
    want[0] += 900
    np.testing.assert_array_equal(self_dr, want)
    # subset mode over a partition of the rows sums to 2 DD
    rows = np.arange(900)
    parts = [rows[:300], rows[300:301], rows[301:]]
    np.testing.assert_array_equal(sum(H(oracle.count_rows(d, p, d, True, e)) for p in parts), 2 * dd)
    # threads do not change integers
    np.testing.assert_array_equal(H(oracle.count_auto(d, e, threads=3)), dd)
    np.testing.assert_array_equal(H(oracle.count_cross(d, r, e, threads=3)), dr)
    # nested edges: merging adjacent bins = counting with the coarser edges
    coarse = oracle.count_auto(d, e[::2])
    np.testing.assert_array_equal(coarse.hist.astype(np.int64), dd[1:-1].reshape(-1, 2).sum(1))


# ------------------------------------------------------------------ P6 uniform full sphere
def test_p6_uniform_sphere_closed_form():
    n = 6000
    v = xyz_of(synth.uniform_sphere(n, synth.SplitMix(11)))
    e = synth.edges(25, 0.5, 180.0, "log")
    c = oracle.count_auto(v, e, threads=oracle.host_threads())
    npairs = n * (n - 1) / 2
    exp = npairs * (np.cos(np.radians(e[:-1])) - np.cos(np.radians(e[1:]))) / 2.0
    assert np.all(np.abs(c.hist - exp) <= 5.0 * np.sqrt(exp) + 1.0)
    assert abs(c.under - npairs * (1 - math.cos(math.radians(0.5))) / 2) <= 5 * math.sqrt(c.under + 1) + 1
    assert c.over == 0
    # same closed form for a linear binning and for the cross count
    w = xyz_of(synth.uniform_sphere(3000, synth.SplitMix(12)))
    el = synth.edges(18, 0.0, 180.0, "linear")
    cx = oracle.count_cross(v, w, el, threads=oracle.host_threads())
    expx = n * 3000 * (np.cos(np.radians(el[:-1])) - np.cos(np.radians(el[1:]))) / 2.0
    assert np.all(np.abs(cx.hist - expx) <= 5.0 * np.sqrt(expx) + 1.0)


# ------------------------------------------------------------------ P7 null test, P8 Eq. 1 algebra
def test_p7_null_test_w_consistent_with_zero():
    patch = (0.0, 20.0, -10.0, 10.0)
    d = xyz_of(synth.uniform_patch(5000, patch, synth.SplitMix(21)))
    r = xyz_of(synth.uniform_patch(7000, patch, synth.SplitMix(22)))
    e = synth.edges(10, 0.3, 10.0, "log")
    t = oracle.host_threads()
    dd, dr, rr = oracle.count_auto(d, e, threads=t), oracle.count_cross(d, r, e, threads=t), oracle.count_auto(r, e, threads=t)
    w = oracle.estimate(dd.hist, dr.hist, rr.hist, 5000, 7000)
    assert np.all(np.abs(w) <= 5.0 / np.sqrt(np.minimum(dd.hist, rr.hist)))


def test_p8_eq1_hand_case_and_same_catalog():
    g = GOLD["landy_szalay_hand"]
    w = oracle.estimate(g["dd"], g["dr"], g["rr"], g["n_d"], g["n_r"])
    assert abs(w[0] - g["w"][0]) < 1e-15
    assert math.isnan(oracle.estimate([1], [1], [0], 5, 5)[0])
    # D = R (same N rows): DD_k = RR_k, DR_k = 2 DD_k in bins that exclude theta = 0  =>  w_k = 2/N exactly
    D, _, e, _ = synth.make_config(1, n_d=500, n_r=8)
    d = oracle.radec_to_xyz(D)
    dd, dr = oracle.count_auto(d, e), oracle.count_cross(d, d, e)
    w = oracle.estimate(dd.hist, dr.hist, dd.hist, 500, 500)
    ok = dd.hist > 0
    np.testing.assert_allclose(w[ok], 2.0 / 500, rtol=0, atol=1e-12)


def test_p8x_cross_estimator_hand_case_identity_and_null():
    """orc_estimate_cross (the form of PAPER.md:20-25 Eq. 1 with the data term split over two catalogs).
    Hand case: N_1 = 3, N_2 = 2, N_R = 4, one bin, D1D2 = 4, D1R = 5, D2R = 3, RR = 3 -> n12 = 6, n1r = 12, n2r = 8, nrr = 6:
    (4/6 - 5/12 - 3/8 + 3/6) / (3/6) = (3/8) / (1/2) = 3/4.  Each term moved on its own changes w by a hand-computed step,
    so a swapped or mis-signed term fails."""
    w = oracle.estimate_cross([4], [5], [3], [3], 3, 2, 4)
    assert abs(w[0] - 0.75) < 1e-15
    assert abs(oracle.estimate_cross([5], [5], [3], [3], 3, 2, 4)[0] - (0.75 + (1 / 6) / 0.5)) < 1e-15      # +1 pair in D1D2
    assert abs(oracle.estimate_cross([4], [6], [3], [3], 3, 2, 4)[0] - (0.75 - (1 / 12) / 0.5)) < 1e-15     # +1 pair in D1R
    assert abs(oracle.estimate_cross([4], [5], [4], [3], 3, 2, 4)[0] - (0.75 - (1 / 8) / 0.5)) < 1e-15      # +1 pair in D2R
    assert math.isnan(oracle.estimate_cross([1], [1], [1], [0], 5, 5, 5)[0])
    # the same N rows as D1, D2 and R: the three cross counts are 2 DD_k and RR_k = DD_k in bins without theta = 0
    #   => w12_k = 1 - 2 nrr / N^2 = 1/N exactly
    D, _, e, _ = synth.make_config(1, n_d=400, n_r=8)
    d = oracle.radec_to_xyz(D)
    dd, x = oracle.count_auto(d, e), oracle.count_cross(d, d, e)
    w = oracle.estimate_cross(x.hist, x.hist, x.hist, dd.hist, 400, 400, 400)
    np.testing.assert_allclose(w[dd.hist > 0], 1.0 / 400, rtol=0, atol=1e-12)
    # null test: three independent uniform catalogs on one footprint => w12 consistent with 0 (a wrong sign gives +-2, +-1)
    patch = (0.0, 20.0, -10.0, 10.0)
    a, b, r = (xyz_of(synth.uniform_patch(n, patch, synth.SplitMix(s))) for n, s in ((4000, 31), (3000, 32), (6000, 33)))
    e = synth.edges(8, 0.5, 10.0, "log")
    t = oracle.host_threads()
    ab, ar, br, rr = (oracle.count_cross(a, b, e, threads=t), oracle.count_cross(a, r, e, threads=t),
                      oracle.count_cross(b, r, e, threads=t), oracle.count_auto(r, e, threads=t))
    w = oracle.estimate_cross(ab.hist, ar.hist, br.hist, rr.hist, 4000, 3000, 6000)
    assert np.all(np.abs(w) <= 5.0 / np.sqrt(np.minimum(ab.hist, rr.hist)))


# ------------------------------------------------------------------ P9 two independent angle formulas, O6
@pytest.mark.parametrize("idx", [1, 2, 5])
def test_p9_acos_vs_asin_chord(idx):
    D, R, e, _ = synth.make_config(idx, n_d=1200, n_r=800)
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    assert oracle.count_auto(d, e, validate=True).mismatch == 0
    assert oracle.count_cross(d, r, e, validate=True).mismatch == 0


def test_p9_mismatch_counter_does_count():
    """Positive pin of the O8 counter: two points 1e-7 deg apart on the equator.  In fp64 the dot product is
    1 - 1.5e-18 = 1.0, so acos gives theta = 0 (under the first edge) while 2 asin(chord / 2) gives 1e-7 deg
    (inside the bin): the two formulas disagree on exactly this pair and agree on the 1-degree pair."""
    x = xyz_of([[10.0, 0.0], [10.0 + 1e-7, 0.0], [11.0, 0.0]])
    c = oracle.count_auto(x, np.array([5e-8, 2e-7, 0.5, 2.0]), validate=True)
    assert c.mismatch == 1
    assert (c.under, list(c.hist), c.over) == (1, [0, 0, 2], 0)          # the acos path, as the paper computes it
    # far from theta = 0 the same construction does not trip it
    y = xyz_of([[10.0, 0.0], [10.0 + 1e-3, 0.0], [11.0, 0.0]])
    assert oracle.count_auto(y, np.array([5e-4, 2e-3, 0.5, 2.0]), validate=True).mismatch == 0


def test_o6_near_edge_counters_match_numpy():
    D, R, e, _ = synth.make_config(1, n_d=600, n_r=400)
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    s = np.clip(d @ r.T, -1, 1).ravel()
    ce = np.cos(np.radians(e))
    want = np.array([(np.abs(s - c) <= 1e-6).sum() for c in ce])
    got = oracle.count_cross(d, r, e, validate=True).near
    assert np.abs(got.astype(np.int64) - want).sum() <= 2      # BLAS-vs-loop rounding at the 1e-6 boundary
    assert got.sum() > 0                                       # the small log bins do sit within 1e-6 in cos


# ------------------------------------------------------------------ 3-D variant: orc_count_*_xyz
def _lattice_multiplicities(m):
    """Unordered pairs of the m^3 integer lattice by squared distance, from the offset-vector count
    (m - |dx|)(m - |dy|)(m - |dz|) per ordered offset -- no point-by-point loop."""
    out = {}
    rng = range(-(m - 1), m)
    for dx in rng:
        for dy in rng:
            for dz in rng:
                if (dx, dy, dz) == (0, 0, 0):
                    continue
                d2 = dx * dx + dy * dy + dz * dz
                out[d2] = out.get(d2, 0) + (m - abs(dx)) * (m - abs(dy)) * (m - abs(dz))
    return {d2: c // 2 for d2, c in out.items()}


def test_x1_cubic_lattice_multiplicities():
    """X1: 2x2x2 cube: 12 edges, 12 face diagonals, 4 space diagonals; 3x3x3: 54, 72, 32, 27, 72, 48, 18, 24, 4 pairs
    at r^2 = 1, 2, 3, 4, 5, 6, 8, 9, 12 (hand-derived, total 351)."""
    assert _lattice_multiplicities(2) == {1: 12, 2: 12, 3: 4}
    hand3 = {1: 54, 2: 72, 3: 32, 4: 27, 5: 72, 6: 48, 8: 18, 9: 24, 12: 4}
    assert _lattice_multiplicities(3) == hand3 and sum(hand3.values()) == 27 * 26 // 2
    for m, want in ((2, {1: 12, 2: 12, 3: 4}), (3, hand3)):
        x = synth.cubic_lattice(m) * 2.5 + np.array([7.0, -3.0, 11.0])          # scaled and shifted: r = 2.5 sqrt(d2)
        d2s = sorted(want)
        # one bin per distinct distance, edges half way between consecutive distances
        r = 2.5 * np.sqrt(np.array(d2s, dtype=np.float64))
        e = np.concatenate([[0.5 * r[0]], 0.5 * (r[:-1] + r[1:]), [r[-1] + 1.0]])
        c = oracle.count_auto_xyz(x, e)
        assert list(c.hist) == [want[d] for d in d2s] and c.under == 0 and c.over == 0
        # edges exactly ON the distances 2.5 and 5.0 (exact in fp64): lower-inclusive bins, closed last bin
        c = oracle.count_auto_xyz(x, np.array([2.5, 5.0]))
        assert c.hist[0] == sum(v for d, v in want.items() if 1 <= d <= 4) and c.under == 0
        assert c.over == sum(v for d, v in want.items() if d > 4)


def test_x2_totals_and_identities_xyz():
    a = synth.clustered_box(700, 50.0, 9, 2.0, synth.SplitMix(5, 0))
    b = synth.uniform_box(500, 50.0, synth.SplitMix(5, 1))
    e = synth.edges(12, 0.5, 40.0, "log")
    ca, cb, cx = oracle.count_auto_xyz(a, e), oracle.count_auto_xyz(b, e), oracle.count_cross_xyz(a, b, e)
    assert ca.total == 700 * 699 // 2 and cb.total == 500 * 499 // 2 and cx.total == 700 * 500
    cu = oracle.count_auto_xyz(np.concatenate([a, b]), e)                          # DD(A u B) = DD(A) + DD(B) + DR(A, B)
    assert np.array_equal(cu.hist, ca.hist + cb.hist + cx.hist) and cu.under == ca.under + cb.under + cx.under
    rows = synth.subset_rows(700, 700, 3)                                          # a permutation: subset mode sums to 2 DD
    cr = oracle.count_rows_xyz(a, rows, a, True, e)
    assert np.array_equal(cr.hist, 2 * ca.hist) and cr.total == 700 * 699
    assert np.array_equal(oracle.count_auto_xyz(a[::-1].copy(), e).hist, ca.hist)   # order invariance
    assert np.array_equal(oracle.count_cross_xyz(a, b, e, threads=3).hist, cx.hist)


def test_x3_unit_cube_distance_distribution():
    """X3: two uniform points in the unit cube: P(r <= t) = 4 pi t^3/3 - 3 pi t^4/2 + 8 t^5/5 - t^6/6 for t <= 1
    (the classical cube line-picking law); counts within 5 sigma per bin."""
    n = 3000
    x = synth.uniform_box(n, 1.0, synth.SplitMix(77, 0))
    e = np.linspace(0.0, 1.0, 11)
    F = lambda t: 4 * np.pi * t ** 3 / 3 - 1.5 * np.pi * t ** 4 + 1.6 * t ** 5 - t ** 6 / 6
    c = oracle.count_auto_xyz(x, e, threads=oracle.host_threads())
    npairs = n * (n - 1) // 2
    exp = npairs * (F(e[1:]) - F(e[:-1]))
    assert np.all(np.abs(c.hist - exp) <= 5 * np.sqrt(exp) + 1)
    assert abs(c.over - npairs * (1 - F(1.0))) <= 5 * np.sqrt(npairs * (1 - F(1.0)))
    assert abs(F(1.0) - 0.90966) < 1e-4                                             # the law's own checksum


def test_x4_unit_vectors_with_chord_edges_reproduce_angular_histogram():
    """X4: fed unit vectors and r-edges 2 sin(theta_k / 2), the 3-D counter is the angular counter."""
    D, R, e, _ = synth.make_config(2, n_d=900, n_r=700)
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    re = 2.0 * np.sin(np.radians(e) / 2.0)
    for ang, xyz in ((oracle.count_auto(d, e, validate=True), oracle.count_auto_xyz(d, re)),
                     (oracle.count_cross(d, r, e, validate=True), oracle.count_cross_xyz(d, r, re))):
        diff = np.abs(ang.hist.astype(np.int64) - xyz.hist.astype(np.int64))
        assert ang.total == xyz.total and np.all(diff <= ang.tol()) and diff.sum() <= 2


def test_x_near_counter_xyz():
    x = np.array([[0.0, 0, 0], [3.0, 4.0, 0], [3.0, 4.0, 1e-7]])                   # r = 5, 5 + 1e-15, 1e-7
    c = oracle.count_auto_xyz(x, np.array([1.0, 5.0, 9.0]), near_tol=1e-9)
    assert list(c.near) == [0, 2, 0] and c.under == 1 and list(c.hist) == [0, 2]


# ------------------------------------------------------------------ weighted sums: orc_wsum_*
def test_w1_hand_case_and_unit_weights():
    """W1: three points on the equator at RA 0, 1, 3 deg with weights 2, 3, 5: separations 1, 2, 3 deg carry the products
    6, 15, 10; and with unit weights the weighted sums ARE the pair counts (integers, exact in fp64)."""
    v = xyz_of([[0, 0], [1, 0], [3, 0]])
    c = oracle.wsum_auto(v, [2.0, 3.0, 5.0], np.array([0.5, 1.5, 2.5, 3.5]))
    assert list(c.hist) == [6.0, 15.0, 10.0] and c.under == 0.0 and c.over == 0.0
    x = oracle.wsum_cross(v[:1], [2.0], v[1:], [3.0, -5.0], np.array([0.5, 1.5, 2.5, 3.5]))
    assert list(x.hist) == [6.0, 0.0, -10.0] and list(x.abs_hist) == [0.0, 6.0, 0.0, 10.0, 0.0]
    D, R, e, _ = synth.make_config(1, n_d=700, n_r=500)
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    ca, cx = oracle.count_auto(d, e), oracle.count_cross(d, r, e)
    wa, wx = oracle.wsum_auto(d, np.ones(700), e), oracle.wsum_cross(d, np.ones(700), r, np.ones(500), e)
    assert np.array_equal(wa.hist, ca.hist.astype(np.float64)) and (wa.under, wa.over) == (ca.under, ca.over)
    assert np.array_equal(wx.hist, cx.hist.astype(np.float64)) and (wx.under, wx.over) == (cx.under, cx.over)


def test_w2_masks_bilinearity_and_numpy():
    """W2: 0/1 weights select a sub-catalog (its counts, exactly); scaling the weights of one side by 4 scales every sum
    by 4 exactly; general weights against numpy's weighted histogram of arccos(Gram) within the reordering bound."""
    D, R, e, _ = synth.make_config(1, n_d=600, n_r=400)
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    rng = synth.SplitMix(41)
    mask = (rng.uniform(600) < 0.4).astype(np.float64)
    sub = d[mask > 0]
    assert np.array_equal(oracle.wsum_auto(d, mask, e).hist, oracle.count_auto(sub, e).hist.astype(np.float64))
    wd, wr = 0.5 + rng.uniform(600), rng.normal(400)
    x1, x4 = oracle.wsum_cross(d, wd, r, wr, e), oracle.wsum_cross(d, 4.0 * wd, r, wr, e)
    assert np.array_equal(4.0 * x1.hist, x4.hist) and 4.0 * x1.over == x4.over
    assert np.array_equal(oracle.wsum_cross(d, wd, r, wr, e, threads=3).abs_hist.round(6), x1.abs_hist.round(6))
    th = np.degrees(np.arccos(np.clip(d @ r.T, -1.0, 1.0)))
    ref, _ = np.histogram(th.ravel(), bins=e, weights=np.outer(wd, wr).ravel())
    assert np.all(np.abs(ref - x1.hist) <= 600 * 400 * 2.0 ** -53 * x1.abs_hist[1:-1] + 1e-300)
    a = oracle.wsum_auto(d, wd, e)
    tri = np.triu_indices(600, 1)
    tha = np.degrees(np.arccos(np.clip(d @ d.T, -1.0, 1.0)))[tri]
    refa, _ = np.histogram(tha, bins=e, weights=np.outer(wd, wd)[tri])
    assert np.all(np.abs(refa - a.hist) <= 600 * 600 * 2.0 ** -53 * a.abs_hist[1:-1] + 1e-300)
