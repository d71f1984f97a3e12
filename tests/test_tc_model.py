"""CPU checks of the tensor engine's error bound ("tensor engine") against the accumulation model
of tests/tc_model.py -- the model itself is compared with the hardware bit for bit in tests/test_gpu_tensor.py."""
import numpy as np

import tc_model as M

U = M.U


def test_tf32_split_is_exact_and_small():
    rng = np.random.default_rng(1)
    x = (rng.normal(size=200_000) * np.exp2(rng.integers(-20, 3, 200_000))).astype(np.float32)
    hi, lo = M.split2(x)
    assert np.all((hi.view(np.uint32) & 0x1FFF) == 0) and np.all((lo.view(np.uint32) & 0x1FFF) == 0)
    assert np.all(np.abs(x.astype(np.float64) - hi) <= 2.0 ** -11 * np.abs(x))
    assert np.all(np.abs(x.astype(np.float64) - hi - lo) <= 2.0 ** -22 * np.abs(x))
    h3, m3, l3 = M.split3(x)
    assert np.all(np.abs(x.astype(np.float64) - h3 - m3 - l3) <= 2.0 ** -33 * np.abs(x))


def test_model_hand_cases():
    """The rows of the measurement the model was read from (profiles/r2_tensor_model.md): 1 + small terms."""
    def one(sr, br):
        return float(M.emulate(np.array([sr], np.float32), np.array([br], np.float32))[0, 0])
    p = lambda k: 2.0 ** -k
    assert one((1, p(24), p(24), 0), (1, 1, 1, 0)) == 1 + p(23)        # bits below the fp32 grid take part in the sum ...
    assert one((1, p(23), p(24), 0), (1, 1, 1, 0)) == 1 + p(23)        # ... and the sum is truncated, not rounded
    assert one((1, p(25), p(25), 0), (1, 1, 1, 0)) == 1.0
    assert one((1, -p(25), 0, 0), (1, 1, 1, 0)) == 1 - p(24)           # 1 - 2^-25 chopped toward zero
    assert one((1, -p(26), 0, 0), (1, 1, 1, 0)) == 1.0                 # 2^-26 falls below 2^(e_max - 25): dropped
    assert one((1, 0, 0, p(24)), (1, 1, 1, p(23))) == 1 + p(23)        # second step: accumulator + nsm + w, same rule


def test_lemma_T_holds_for_the_model():
    """|q_model - exact| <= bound(): block geometry at the kappa = 2.5 limit, random blocks, and adversarial operand rows."""
    rng = np.random.default_rng(2)
    worst = 0.0
    for s_rows, b_rows in (M.block_tiles(rng, 60, at_limit=True)[:2], M.block_tiles(rng, 60)[:2], M.adversarial_tiles(rng, 80)):
        for s, b in zip(s_rows, b_rows):
            err = np.abs(M.emulate(s, b).astype(np.float64) - M.exact(s, b))
            bd = M.bound(s, b)
            assert np.all(err <= bd + 1e-300)
            worst = max(worst, float((err / np.maximum(bd, 1e-300)).max()))
    assert worst > 0.15, "the bound is not absurdly loose"


def test_whole_chain_stays_inside_the_tensor_guard_band():
    """fp64 rows -> stored fp32 offsets -> s, |s|^2 - mid, (-2 b', |b'|^2) as the kernels form them -> 3xTF32 MMA (model)
    against the fp64 value d^2 - mid: <= 43.7 u max(d^2, mid), the constant behind tables.cpp guard_width_tensor."""
    rng = np.random.default_rng(3)
    worst = 0.0
    for t in range(120):
        D = 10.0 ** rng.uniform(-3.3, -0.05)
        r = D / (3.5 if t % 2 else rng.uniform(3.5, 50.0))             # D - r = 2.5 r at the limit
        f = rng.choice([0.05, 0.3, 0.6, 0.95])
        ri, rj = f * r, (1.0 - f) * r
        def unit(n):
            v = rng.normal(size=(n, 3))
            return v / np.linalg.norm(v, axis=1, keepdims=True)
        cq64 = unit(1)[0]
        perp = np.cross(cq64, unit(1)[0])
        ct64 = cq64 + perp / np.linalg.norm(perp) * D
        cq, ct = cq64.astype(np.float32), ct64.astype(np.float32)       # fp32 centres: exact values from here on
        a = cq.astype(np.float64) + unit(128) * ri * rng.choice([1.0, 0.7], size=(128, 1))
        b = ct.astype(np.float64) + unit(128) * rj * rng.choice([1.0, 0.7], size=(128, 1))
        ap, bp = (a - cq).astype(np.float32), (b - ct).astype(np.float32)                 # stored offsets, rounded once
        tt = (cq - ct).astype(np.float32)
        s = (ap + tt).astype(np.float32)
        d2 = ((a[:, None, :] - b[None, :, :]) ** 2).sum(-1)
        lo2, hi2 = d2.min(), d2.max()
        mid = np.float32(rng.choice([lo2, 0.5 * (lo2 + hi2), hi2, 1.5 * hi2]))             # an edge in or above the window
        f32 = lambda x: np.asarray(x, dtype=np.float32)
        fma = lambda x, y, z: f32(x.astype(np.float64) * y.astype(np.float64) + z.astype(np.float64))
        n2 = fma(s[:, 2], s[:, 2], fma(s[:, 1], s[:, 1], f32(s[:, 0] * s[:, 0])))
        s_rows = np.concatenate([s, f32(n2 - mid)[:, None]], 1)
        b_rows = np.concatenate([f32(-2.0 * bp), f32((bp.astype(np.float64) ** 2).sum(1))[:, None]], 1)
        q = M.emulate(s_rows, b_rows).astype(np.float64)
        err = np.abs(q - (d2 - float(mid)))
        scale = U * np.maximum(d2, float(mid))
        assert np.all(err <= 41.7 * scale), float((err / scale).max())     # 43.7 u less the 2 u of the further edges
        worst = max(worst, float((err / scale).max()))
    assert 4.0e-6 / (43.7 * U) > 1.5                                    # the margin of guard_width_tensor
    assert worst > 3.0
