"""Pins of the oracle's three-point counts (orc_count_triples) -- CPU only.

The definition: every triple i<j<k is counted once in the cell of the ascending slots of its three
side angles (slot 0 = under, 1..nbins = bins, nbins+1 = over).  Pinned by hand triangles, the exact total C(N,3), row
permutation, the side-marginal identity against the pair oracle (every pair is a side of N-2 triples) and an independent
numpy/pure-Python evaluation on 40 points."""
import itertools
import math

import numpy as np

import oracle
import synth


def xyz_of(radec):
    return oracle.radec_to_xyz(np.asarray(radec, dtype=np.float64))


def cells(h3):
    """{(a, b, c): count} of the non-empty cells."""
    return {tuple(int(x) for x in idx): int(h3[tuple(idx)]) for idx in np.argwhere(h3 > 0)}


def test_t1_octahedron_faces_and_antipodal_triples():
    # 6 vertices: 12 pairs at 90 deg, 3 at 180 deg.  C(6,3) = 20 triples: the 8 faces have sides (90, 90, 90); the other 12
    # hold one antipodal pair and a third vertex: (90, 90, 180).  Bins [0,45) [45,135) [135,180] (last closed): 90 -> slot 2,
    # 180 -> slot 3.
    x = xyz_of([(0, 0), (180, 0), (90, 0), (270, 0), (0, 90), (0, -90)])
    h3 = oracle.count_triples(x, [0.0, 45.0, 135.0, 180.0])
    assert h3.shape == (5, 5, 5)
    assert cells(h3) == {(2, 2, 2): 8, (2, 2, 3): 12}


def test_t2_equator_hand_triples_with_under_and_over():
    # RA 0, 10, 20 on the equator: sides 10, 10, 20; edges 5, 15, 25 -> slots 1, 1, 2
    e = [5.0, 15.0, 25.0]
    assert cells(oracle.count_triples(xyz_of([(0, 0), (10, 0), (20, 0)]), e)) == {(1, 1, 2): 1}
    # RA 0, 1, 30: sides 1 (under, slot 0), 30 and 29 (over, slot 3)
    assert cells(oracle.count_triples(xyz_of([(0, 0), (1, 0), (30, 0)]), e)) == {(0, 3, 3): 1}
    # four points RA 0, 10, 20, 30: sides of the 4 triples: (10,10,20), (10,20,30), (10,20,30), (10,10,20)
    got = cells(oracle.count_triples(xyz_of([(0, 0), (10, 0), (20, 0), (30, 0)]), e))
    assert got == {(1, 1, 2): 2, (1, 2, 3): 2}
    # fewer than three points: no triple
    assert oracle.count_triples(xyz_of([(0, 0), (10, 0)]), e).sum() == 0


def test_t3_total_is_n_choose_3_and_t4_row_order_is_irrelevant():
    D, _, e, _ = synth.make_config(1, n_d=57, n_r=8)
    x = oracle.radec_to_xyz(D)
    h3 = oracle.count_triples(x, e)
    assert int(h3.sum()) == 57 * 56 * 55 // 6
    perm = np.argsort(synth.SplitMix(5).u64(57), kind="stable")
    assert np.array_equal(oracle.count_triples(x[perm], e), h3)
    assert np.array_equal(oracle.count_triples(x, e, threads=4), h3)          # the split over i-spans adds up
    a, b, c = np.nonzero(h3)
    assert np.all(a <= b) and np.all(b <= c)                                   # only ascending cells are used


def test_t5_side_marginals_equal_n_minus_2_times_the_pair_counts():
    D, _, e, _ = synth.make_config(1, n_d=150, n_r=8)
    x = oracle.radec_to_xyz(D)
    h3 = oracle.count_triples(x, e, threads=oracle.host_threads()).astype(np.int64)
    dd = oracle.count_auto(x, e)
    pairs = np.concatenate([[dd.under], dd.hist.astype(np.int64), [dd.over]])
    m = h3.shape[0]
    sides = np.zeros(m, dtype=np.int64)
    for s in range(m):                       # cells are (a, b, c): count how many of the three equal s
        sides[s] = h3[s, :, :].sum() + h3[:, s, :].sum() + h3[:, :, s].sum()
    assert np.array_equal(sides, (150 - 2) * pairs)


def test_t6_independent_evaluation_on_40_points():
    D, _, _, _ = synth.make_config(1, n_d=40, n_r=8)
    e = np.array([0.05, 0.4, 1.0, 2.5, 6.0])
    x = oracle.radec_to_xyz(D)
    theta = np.degrees(np.arccos(np.clip(x @ x.T, -1.0, 1.0)))
    nb = len(e) - 1

    def slot(t):                             # numpy.histogram's convention: [e_k, e_{k+1}), last bin closed
        if t < e[0]:
            return 0
        if t > e[-1]:
            return nb + 1
        return min(int(np.searchsorted(e, t, side="right")) - 1, nb - 1) + 1

    want = {}
    for i, j, k in itertools.combinations(range(40), 3):
        key = tuple(sorted((slot(theta[i, j]), slot(theta[i, k]), slot(theta[j, k]))))
        want[key] = want.get(key, 0) + 1
    assert sum(want.values()) == math.comb(40, 3)
    assert cells(oracle.count_triples(x, e)) == want
