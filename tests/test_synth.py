"""The seeded input generators: determinism, footprints, recipe properties."""
import numpy as np

import synth


def test_splitmix_is_counter_based_and_seeded():
    a = synth.SplitMix(1).u64(10)
    g = synth.SplitMix(1)
    b = np.concatenate([g.u64(4), g.u64(6)])
    np.testing.assert_array_equal(a, b)
    assert not np.array_equal(a, synth.SplitMix(2).u64(10))
    # first output of SplitMix64 started at state 0 with the published constants
    z = np.array([0x9E3779B97F4A7C15], dtype=np.uint64)
    from synth.catalogs import _mix
    assert int(_mix(z)[0]) == 0xE220A8397B1DCDAF
    u = synth.SplitMix(3).uniform(200000)
    assert 0.0 <= u.min() and u.max() < 1.0 and abs(u.mean() - 0.5) < 5e-3
    n = synth.SplitMix(4).normal(200001)
    assert abs(n.mean()) < 1e-2 and abs(n.std() - 1.0) < 1e-2


def test_configs_shapes_dtypes_footprints():
    foot = {1: (0, 10, -5, 5), 2: (0, 30, -15, 15), 3: (0, 90, 0, 90), 4: (0, 360, -90, 90), 5: (0, 5, -2.5, 2.5)}
    for idx in (1, 2, 3, 4, 5):
        D, R, e, cfg = synth.make_config(idx, n_d=3000, n_r=2000)
        D2, _, _, _ = synth.make_config(idx, n_d=3000, n_r=2000)
        np.testing.assert_array_equal(D, D2)
        assert D.shape == (3000, 2) and R.shape == (2000, 2)
        assert D.dtype == (np.float32 if cfg.dtype == "f32" else np.float64)
        ra0, ra1, d0, d1 = foot[idx]
        for X in (D, R):
            assert X[:, 0].min() >= ra0 and X[:, 0].max() <= ra1 and X[:, 1].min() >= d0 and X[:, 1].max() <= d1
        assert e.shape == (cfg.nbins + 1,) and e[0] == cfg.theta_min and e[-1] == cfg.theta_max
        assert np.all(np.diff(e) > 0)


def test_full_size_of_small_configs():
    D, R, e, cfg = synth.make_config(1)
    assert D.shape == (4096, 2) and R.shape == (4096, 2) and e.shape == (21,)
    assert synth.CONFIGS[3].n_d == 430_000 and synth.CONFIGS[4].n_r == 2_000_000 and synth.CONFIGS[5].nbins == 512


def test_log_edges_have_constant_ratio():
    e = synth.edges(40, 0.01, 60.0, "log")
    r = e[1:] / e[:-1]
    assert np.max(np.abs(r / r[0] - 1)) < 1e-13


def test_clump_major_and_shuffle():
    D, _, _, _ = synth.make_config(5, n_d=2000, n_r=10)
    S, _, _, _ = synth.make_config(5, n_d=2000, n_r=10, shuffle_d=True)
    assert not np.array_equal(D, S)
    np.testing.assert_array_equal(np.sort(D.view(np.complex128).ravel()), np.sort(S.view(np.complex128).ravel()))
    # rows of one clump are adjacent: consecutive rows are far closer than random rows
    step = np.abs(np.diff(D[:, 1])).mean()
    assert step < 0.25 * np.abs(np.diff(S[:, 1])).mean()


def test_subset_rows():
    r = synth.subset_rows(430_000)
    assert r.shape == (2000,) and np.all(np.diff(r) > 0) and r.max() < 430_000
    np.testing.assert_array_equal(r, synth.subset_rows(430_000))
    assert synth.subset_rows(10, 2000).shape == (10,)
