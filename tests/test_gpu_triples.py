"""tpcf_count3 (three-point counts) against the oracle's orc_count_triples, cell by
cell, through the C ABI.  The oracle bins each side by acos(dot), the kernels by the fp64 squared chord: the two can
differ only for a pair within fp64 rounding of an edge (reading A13), and one such pair moves N-2 triples -- the
tolerance below allows STRICT such pairs and in practice the arrays are equal."""
import math

import numpy as np
import pytest

import oracle
import paper_1204_6630_b200 as T
import synth

pytestmark = pytest.mark.gpu
STRICT = 4


def test_octahedron_hand_triples():
    rows = np.array([(0, 0), (180, 0), (90, 0), (270, 0), (0, 90), (0, -90)], dtype=np.float64)
    with T.Context(3, [0.0, 45.0, 135.0, 180.0], "explicit") as c:
        c.load("D", rows)
        h3 = c.count3("D")
    assert h3.shape == (5, 5, 5) and int(h3.sum()) == 20
    assert int(h3[2, 2, 2]) == 8 and int(h3[2, 2, 3]) == 12          # 8 faces (90,90,90); 12 x (90,90,180): hand values


@pytest.mark.parametrize("idx,n,nbins,lo,hi,mode", [(1, 2500, 12, 0.05, 8.0, "log"), (2, 3001, 30, 0.0, 30.0, "linear"),
                                                   (5, 1777, 7, 0.02, 3.0, "log"), (1, 129, 20, 0.01, 10.0, "log")])
def test_triples_match_oracle_cell_by_cell(idx, n, nbins, lo, hi, mode, oracle_threads):
    D, _, _, _ = synth.make_config(idx, n_d=n, n_r=8)
    e = synth.edges(nbins, lo, hi, mode)
    want = oracle.count_triples(oracle.radec_to_xyz(D), e, threads=oracle_threads).astype(np.int64)
    with T.Context(nbins, e, "explicit") as c:
        c.load("R", D)                       # any catalog slot
        got = c.count3("R").astype(np.int64)
        st = c.stats()
        h, u, o = c.count("RR")
        pairs = np.concatenate([[u], h.astype(np.int64), [o]])
    assert int(got.sum()) == math.comb(n, 3) == int(want.sum()) == st["pairs"]
    assert int(np.abs(got - want).sum()) <= 2 * STRICT * (n - 2)
    a, b, cc = np.nonzero(got)
    assert np.all(a <= b) and np.all(b <= cc)
    # side marginals against the library's own pair count: every pair is a side of N-2 triples
    m = nbins + 2
    sides = np.array([got[s, :, :].sum() + got[:, s, :].sum() + got[:, :, s].sum() for s in range(m)])
    assert np.array_equal(sides, (n - 2) * pairs)


def test_count3_limits_and_state():
    with T.Context(4, [0.1, 10.0], "log") as c:
        with pytest.raises(T.TpcfError) as ei:
            c.count3("D")
        assert ei.value.status == T.TPCF_ESTATE
        c.load("D", synth.make_config(1, n_d=2, n_r=8)[0])
        assert int(c.count3("D").sum()) == 0                  # two points: no triple
        c.load("D", synth.make_config(1, n_d=T.TPCF_COUNT3_MAX_ROWS + 1, n_r=8)[0])
        with pytest.raises(T.TpcfError) as ei:
            c.count3("D")
        assert ei.value.status == T.TPCF_EINVAL
    with T.Context(31, [0.1, 10.0], "log") as c:
        c.load("D", synth.make_config(1, n_d=100, n_r=8)[0])
        with pytest.raises(T.TpcfError) as ei:
            c.count3("D")
        assert ei.value.status == T.TPCF_EINVAL
