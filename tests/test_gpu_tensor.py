"""GPU parity of the tensor engine (TPCF_ENGINE_TENSOR: the window quantity by 3xTF32 tcgen05.mma into tensor memory,
DESIGN.md section 6): against the fp64 oracle element by element where the oracle finishes in seconds, and -- at the
sizes bench.py times -- against the fast and the fp64 engines, whose histograms it must reproduce bit for bit (the
tensor core only changes how q is formed for pairs outside the guard bands; every pair inside one is rechecked in fp64).
"""
import numpy as np
import pytest

import oracle
import paper_1204_6630_b200 as T
import synth
from test_gpu_parity import KINDS, assert_parity, assert_w, full, gpu_all, oracle_all, totals

pytestmark = pytest.mark.gpu


def tensor_ctx(nbins, e):
    c = T.Context(nbins, e, "explicit")
    c.set_engine("tensor")
    c.set_tensor_share_limit(1.0)       # always pair_tensor_kernel, also where the engine on its own would pick the FFMA2 kernel
    return c


@pytest.mark.parametrize("idx,nd,nr", [(1, None, None), (2, 20_000, 17_777), (3, 9_000, 11_111), (4, 6_000, 12_345),
                                       (5, 20_000, 20_000)])
def test_tensor_engine_matches_oracle(idx, nd, nr, oracle_threads):
    D, R, e, cfg = synth.make_config(idx, n_d=nd, n_r=nr)
    nd, nr = D.shape[0], R.shape[0]
    o = oracle_all(D, R, e, oracle_threads)
    with tensor_ctx(cfg.nbins, e) as c:
        c.load("D", D)
        c.load("R", R)
        g = gpu_all(c)
        wg = c.estimate()
        used = np.asarray(c.stats()["win_blocks"])
        c.set_engine("exact64")
        gx = gpu_all(c)
    for k in KINDS:
        assert_parity(g[k], o[k], totals(nd, nr)[k])
        np.testing.assert_array_equal(g[k], gx[k])            # tensor engine == fp64 engine, bit for bit
    assert_w(wg, oracle.estimate(o["DD"].hist, o["DR"].hist, o["RR"].hist, nd, nr))
    if idx != 5:                                              # fine binnings run the FFMA2 kernel instead
        assert used[:3].sum() > 0, "no block went through the tensor-core window path"


@pytest.mark.parametrize("idx", [2, 3, 4])
def test_tensor_engine_full_size_equals_fast_engine(idx):
    """Configs 2-4 at BASELINE.json's sizes, in the launch configuration bench.py times: every histogram of the tensor
    engine equals the fast engine's (which the other tests tie to the oracle on row subsets and to the fp64 engine)."""
    D, R, e, cfg = synth.make_config(idx)
    nd, nr = D.shape[0], R.shape[0]
    res = {}
    for eng in ("fast", "tensor"):
        with T.Context(cfg.nbins, e, "explicit") as c:
            c.set_engine(eng)
            c.load("D", D)
            c.load("R", R)
            res[eng] = gpu_all(c)
            if eng == "tensor":
                st = c.stats()
                # configs 3 and 4: the tensor kernel really ran (4-warp CTAs); config 2 has 5 % of its blocks nearer than
                # the windows allow, so the engine launches the FFMA2 kernel there (tpcf_stats.lookup_share)
                assert st["block"] == (128 if idx != 2 else 256) and (st["lookup_share"] <= 0.025) == (idx != 2)
    for k in KINDS:
        assert int(res["tensor"][k].sum()) == totals(nd, nr)[k]
        np.testing.assert_array_equal(res["tensor"][k], res["fast"][k])


@pytest.mark.parametrize("idx,nrows", [(3, 2000), (4, 2000)])
def test_tensor_engine_row_subset_against_oracle(idx, nrows, oracle_threads):
    D, R, e, cfg = synth.make_config(idx)
    nd, nr = D.shape[0], R.shape[0]
    rows_d, rows_r = synth.subset_rows(nd, nrows, 12345), synth.subset_rows(nr, nrows, 12346)
    d, r = oracle.radec_to_xyz(D), oracle.radec_to_xyz(R)
    with tensor_ctx(cfg.nbins, e) as c:
        c.load("D", D)
        c.load("R", R)
        g = gpu_all(c, {"DD": rows_d, "DR": rows_d, "RR": rows_r})
    o = {"DD": oracle.count_rows(d, rows_d, d, True, e, validate=True, threads=oracle_threads),
         "DR": oracle.count_rows(d, rows_d, r, False, e, validate=True, threads=oracle_threads),
         "RR": oracle.count_rows(r, rows_r, r, True, e, validate=True, threads=oracle_threads)}
    exp = {"DD": nrows * (nd - 1), "DR": nrows * nr, "RR": nrows * (nr - 1)}
    for k in KINDS:
        assert_parity(g[k], o[k], exp[k])


@pytest.mark.parametrize("nd,nr", [(1, 1), (2, 3), (127, 129), (1023, 1025), (2049, 1), (3000, 5000)])
def test_tensor_engine_ragged_sizes(nd, nr):
    D, R, _, _ = synth.make_config(1, n_d=nd, n_r=nr)
    e = np.array([0.0, 0.05, 0.5, 2.0, 180.0])
    o = oracle_all(D, R, e, 1)
    with tensor_ctx(4, e) as c:
        c.load("D", D)
        c.load("R", R)
        g = gpu_all(c)
    for k in KINDS:
        assert_parity(g[k], o[k], totals(nd, nr)[k])


def test_tensor_engine_sparse_and_duplicate_rows(oracle_threads):
    rng = np.random.default_rng(11)
    def sky(n):
        return np.stack([rng.uniform(0.0, 360.0, n), np.degrees(np.arcsin(rng.uniform(-1.0, 1.0, n)))], 1)
    D, R = sky(700), sky(900)
    e = np.linspace(0.0, 180.0, 37)
    with tensor_ctx(36, e) as c:
        c.load("D", D)
        c.load("R", R)
        g = gpu_all(c)
        o = oracle_all(D, R, c.edges(), oracle_threads)
        for k in KINDS:
            assert_parity(g[k], o[k], totals(700, 900)[k])
    P = np.array([[10.0, 20.0], [10.0, 20.0], [10.0, 20.0], [50.0, -30.0]])
    with tensor_ctx(2, [0.0, 1.0, 180.0]) as c:
        c.load("D", P)
        c.load("R", P)
        assert tuple(full(*c.count("DD"))) == (0, 3, 3, 0)
        assert tuple(full(*c.count("DR"))) == (0, 10, 6, 0)


def test_tensor_engine_guard_scale_and_partition_leave_the_counts_unchanged():
    D, R, e, cfg = synth.make_config(3, n_d=60_000, n_r=50_000)
    with tensor_ctx(cfg.nbins, e) as c:
        c.load("D", D)
        c.load("R", R)
        base = gpu_all(c)
        c.set_guard_scale(8.0)                       # 8x wider guard bands: more fp64 rechecks, same integers
        np.testing.assert_array_equal(full(*c.count("DR")), base["DR"])
        c.set_guard_scale(1.0)
        parts = np.zeros_like(base["DD"])
        for part in range(3):                        # work-item partition of the multi-GPU path
            c.set_partition(part, 3)
            parts += full(*c.count("DD"))
        c.set_partition(0, 1)
        np.testing.assert_array_equal(parts, base["DD"])


def tensor_core_error_sample(ntiles=384, seed=20240607):
    """Random blocks in the geometry of the window path (centre distance D, radii down to D >= 3.5 (r_i + r_j), the limit
    of kFarKappa = 2.5) through tpcf_tensor_probe -- the kernel's own operand split, instruction and read-back -- against the
    fp64 value of the same fp32 inputs.  Returns per tile: max |q_tc - q_fp64|, the band half width, t = D^2."""
    rng = np.random.default_rng(seed)
    s_rows = np.empty((ntiles, 128, 4), dtype=np.float32)
    b_rows = np.empty((ntiles, 128, 4), dtype=np.float32)
    tscale = np.empty(ntiles)
    for t in range(ntiles):
        D = 0.02 * 50.0 ** rng.uniform()                       # centre distance 0.02 .. 1
        rs = D / rng.uniform(3.5, 40.0)                        # r_i + r_j
        ri, rj = rs / 3.0, rs * 2.0 / 3.0
        c = rng.normal(size=3)
        c *= D / np.linalg.norm(c)
        s = (c + ri * rng.uniform(-1, 1, size=(128, 3)) / np.sqrt(3.0)).astype(np.float32)
        b = (rj * rng.uniform(-1, 1, size=(128, 3)) / np.sqrt(3.0)).astype(np.float32)
        mid = np.float32(D * D * (1.0 + rng.uniform(-1, 1) * 2.0 * rs / D))      # an edge inside the window
        sx, sy, sz = s[:, 0], s[:, 1], s[:, 2]
        norm = (sz * sz + (sy * sy + sx * sx).astype(np.float32)).astype(np.float32)     # fp32, like the kernel (up to fma)
        s_rows[t, :, :3] = s
        s_rows[t, :, 3] = norm - mid
        b_rows[t, :, :3] = np.float32(-2.0) * b
        b_rows[t, :, 3] = (b.astype(np.float64) ** 2).sum(axis=1).astype(np.float32)
        tscale[t] = D * D
    with T.Context(4, [0.0, 1.0, 2.0, 3.0, 180.0], "explicit") as c:
        q = T.tpcf_tensor_probe(c.handle, s_rows, b_rows).astype(np.float64)
    S, B = s_rows.astype(np.float64), b_rows.astype(np.float64)
    exact = S[:, :, None, 3] + B[:, None, :, 3] + np.einsum("tik,tjk->tij", S[:, :, :3], B[:, :, :3])
    assert np.all(np.isfinite(q))
    # a dot product at all: relative to the size of q the error is ~1e-6
    assert np.all(np.abs(q - exact).max(axis=(1, 2)) < 2.0e-6 * np.abs(exact).max(axis=(1, 2)) + 1e-12)
    return np.abs(q - exact).max(axis=(1, 2)), 3.0e-6 * tscale + 1.0e-7 * np.sqrt(tscale), tscale


def test_tensor_core_accumulation_error_stays_well_inside_the_guard_band():
    """The one step of the tensor engine that is not IEEE arithmetic is the accumulation inside tcgen05.mma.  Measure it
    on random blocks (6.3e6 values): the counters are only trusted for |q| beyond the band half width (tables.cpp
    guard_width_tensor, 4.0e-6 t + 1e-7 sqrt(t)); the measured error stays below a third of the narrower 3.0e-6 t."""
    err, band, _ = tensor_core_error_sample()
    assert np.all(err < band / 3.0), float((err / band).max())


def test_tensor_core_accumulation_model_is_bit_exact():
    """DESIGN.md section 4 proves the tensor engine's guard band from a MODEL of the tensor core's accumulation
    (tests/tc_model.py: products exact, addends aligned to the largest exponent and truncated below 2^(e_max - 25), exact
    sum truncated to fp32).  The hardware has to return exactly the model's bits: 1.05e7 values through tpcf_tensor_probe
    (the kernel's own operand split, tcgen05.mma and tcgen05.ld), block geometry at and away from the kappa = 2.5 limit
    and adversarial operand rows (exponent spreads, cancelling large terms, ties of the truncations)."""
    import tc_model as M
    rng = np.random.default_rng(20261105)
    a_s, a_b, _ = M.block_tiles(rng, 160, at_limit=True)
    r_s, r_b, _ = M.block_tiles(rng, 160)
    x_s, x_b = M.adversarial_tiles(rng, 320)
    s_rows, b_rows = np.concatenate([a_s, r_s, x_s]), np.concatenate([a_b, r_b, x_b])
    with T.Context(4, [0.0, 1.0, 2.0, 3.0, 180.0], "explicit") as c:
        q = T.tpcf_tensor_probe(c.handle, s_rows, b_rows)
    assert q.size >= 10_000_000
    bad = 0
    for t in range(s_rows.shape[0]):
        m = M.emulate(s_rows[t], b_rows[t])
        bad += int(((m.view(np.uint32) != q[t].view(np.uint32)) & ~((m == 0) & (q[t] == 0))).sum())
        assert np.all(np.abs(q[t].astype(np.float64) - M.exact(s_rows[t], b_rows[t])) <= M.bound(s_rows[t], b_rows[t]))
    assert bad == 0, f"{bad} of {q.size} accumulators differ from the model"


@pytest.mark.parametrize("case", ["window_off", "guard_half", "guard_16", "one_bin", "one_narrow_bin", "far_bins",
                                  "linear_64_whole_range", "linear_300_fine", "tiny"])
def test_tensor_engine_equals_fp64_engine_on_unusual_binnings_and_settings(case):
    """Bit-identical to the plain fp64 kernel whatever the binning and the tuning knobs (window loops off: every row takes
    the cell lookup; narrower and wider guard bands; one bin; bins far from 0; linear bins; fewer rows than one tile)."""
    D, R, e, cfg = synth.make_config(3, n_d=30_000, n_r=20_000)
    nb, mode, kw = cfg.nbins, "explicit", {}
    if case == "window_off":
        kw["window"] = False
    elif case == "guard_half":
        kw["gs"] = 0.5
    elif case == "guard_16":
        kw["gs"] = 16.0
    elif case == "one_bin":
        nb, e = 1, [0.0, 180.0]
    elif case == "one_narrow_bin":
        nb, e = 1, [1.0, 1.001]
    elif case == "far_bins":
        nb, e = 3, [30.0, 31.0, 32.0, 33.0]
    elif case == "linear_64_whole_range":
        D, R, _, _ = synth.make_config(4, n_d=40_000, n_r=30_000)
        nb, e, mode = 64, [0.0, 180.0], "linear"
    elif case == "linear_300_fine":
        nb, e, mode = 300, [0.0, 10.0], "linear"
    elif case == "tiny":
        D, R, e, cfg = synth.make_config(1, n_d=100, n_r=130)
        nb = cfg.nbins
    out = {}
    for eng in ("exact64", "tensor"):
        with T.Context(nb, e, mode) as c:
            c.set_engine(eng)
            c.set_tensor_share_limit(1.0)
            if kw.get("window") is False:
                c.set_window(False)
            if "gs" in kw:
                c.set_guard_scale(kw["gs"])
            c.load("D", D)
            c.load("R", R)
            out[eng] = gpu_all(c)
    for k in KINDS:
        np.testing.assert_array_equal(out["tensor"][k], out["exact64"][k])


def test_engine_chooses_its_kernel_from_the_sampled_block_mix():
    """TPCF_ENGINE_TENSOR samples the share of pair-by-pair blocks and launches pair_fast_kernel above the limit
    (tpcf_set_tensor_share_limit); either way the same integers."""
    D, R, e, cfg = synth.make_config(5, n_d=400_000, n_r=30_000)        # fine bins: every block is pair by pair
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.load("D", D)
        c.load("R", R)
        a = full(*c.count("DR"))
        st = c.stats()
        assert st["lookup_share"] > 0.9 and st["block"] == 256
        c.set_tensor_share_limit(1.0)
        b = full(*c.count("DR"))
        assert c.stats()["block"] == 128
        np.testing.assert_array_equal(a, b)
        c.set_tensor_share_limit(0.0)
        np.testing.assert_array_equal(full(*c.count("DR")), a)
        assert c.stats()["block"] == 256
        with pytest.raises(T.TpcfError):
            c.set_tensor_share_limit(1.5)
