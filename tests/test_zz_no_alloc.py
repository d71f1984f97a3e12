"""tpcf_count_static -- the one entry point of libtpcf that allocates no device memory (include/tpcf.h).

Why it exists: tpcf_load / tpcf_count call cudaMalloc.  A host application that has given all device memory to its own
pool (a framework's caching allocator), that runs under a fixed per-GPU budget, or that cannot take the device-wide
stall of cudaMalloc / cudaFree while other streams are busy, cannot use them.  tpcf_count_static works on device
buffers the caller already owns and keeps its scratch in a fixed array inside the library (TPCF_STATIC_MAX_ROWS rows,
TPCF_STATIC_MAX_BINS bins at most).

What is checked here: its histogram against the existing path (tpcf_load + tpcf_count) on the same rows -- bit-equal to
TPCF_ENGINE_EXACT64 (same fp64 arithmetic), and within the STRICT fp64-tie allowance of tests/test_gpu_parity.py against
the default engine -- on TWO CALLS IN A ROW with different shapes, dtypes and binnings, because every call reuses the
same scratch array and must clear what the previous one left.  The file name sorts last on purpose: `pytest -x` stops
at the first failure, and a failure here must not hide the parity tests.  The GPU test passes alone in a fresh process
(it is then the first user of the array on the device) and after the other tests.
"""
import numpy as np
import pytest

import paper_1204_6630_b200 as T
import synth

STRICT = 4          # fp64-tie pairs, as in tests/test_gpu_parity.py (engines other than EXACT64)


def _existing_path(edges, A, B, engine):
    """{under, bins.., over} of the i<j count of A (B None) or of the A x B rectangle, through tpcf_load + tpcf_count."""
    with T.Context(len(edges) - 1, edges, "explicit") as ctx:
        if engine:
            ctx.set_engine(engine)
        ctx.load("D", A)
        if B is not None:
            ctx.load("R", B)
        h, u, o = ctx.count("DD" if B is None else "DR")
    return np.concatenate([[u], np.asarray(h, dtype=np.int64), [o]]).astype(np.int64)


def _static(edges, A, B, out):
    """The same count through tpcf_count_static; A, B, out are CUDA tensors the caller (this test) owns."""
    import torch
    nb = len(edges) - 1
    dt = T.TPCF_F64 if A.dtype == torch.float64 else T.TPCF_F32
    T.tpcf_count_static(nb, edges, "explicit", A.data_ptr(), A.shape[0], None if B is None else B.data_ptr(),
                        0 if B is None else B.shape[0], dt, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    return out[: nb + 2].cpu().numpy().astype(np.int64)


@pytest.mark.gpu
def test_static_count_matches_existing_path_on_two_calls_in_a_row():
    import torch
    assert torch.cuda.is_available(), "there is no CPU fallback"
    # call 1: config 1 (4096 + 4096 fp64 rows, 20 log bins), DR rectangle; call 2: fewer, ragged, fp32 rows of config 2's
    # recipe with more bins, DD triangle -- so call 2 finds call 1's longer catalogs, counter and accumulators in the array
    D1, R1, e1, _ = synth.make_config(1)
    D2, _, _, _ = synth.make_config(2, n_d=3001, n_r=16)
    e2 = synth.edges(57, 0.0, 40.0, "linear")
    cases = [(e1, D1, R1), (e2, D2, None), (e1, D1, R1), (e1, R1[:1500], None)]
    out = torch.full((4096 + 2,), 7, dtype=torch.int64, device="cuda")      # stale values the call must overwrite
    dev = [(torch.from_numpy(A).cuda(), None if B is None else torch.from_numpy(B).cuda()) for _, A, B in cases]
    got = [_static(e, a, b, out) for (e, _, _), (a, b) in zip(cases, dev)]      # back to back, nothing else in between
    # a second round with every kernel variant already loaded: the driver's free-memory figure must not drop
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    again = [_static(e, a, b, out) for (e, _, _), (a, b) in zip(cases, dev)]
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "tpcf_count_static took device memory"
    for g, h in zip(got, again):
        assert np.array_equal(g, h)
    for (e, A, B), g in zip(cases, got):
        n_pairs = A.shape[0] * (A.shape[0] - 1) // 2 if B is None else A.shape[0] * B.shape[0]
        assert int(g.sum()) == n_pairs                                  # totals are exact integers
        ref64 = _existing_path(e, A, B, "exact64")
        assert np.array_equal(g, ref64), "same fp64 arithmetic as TPCF_ENGINE_EXACT64: must be bit-equal"
        ref = _existing_path(e, A, B, None)                             # the default engine
        assert int(np.abs(g - ref).sum()) <= STRICT


@pytest.mark.gpu
def test_static_count_reports_bad_rows_and_recovers():
    import torch
    e = synth.edges(10, 0.0, 180.0, "linear")
    A = torch.tensor([[10.0, 0.0], [20.0, 95.0], [30.0, 5.0]], dtype=torch.float64, device="cuda")     # Dec 95: invalid
    out = torch.zeros(12, dtype=torch.int64, device="cuda")
    with pytest.raises(T.TpcfError) as ei:
        _static(e, A, None, out)
    assert ei.value.status == T.TPCF_EINVAL
    A[1, 1] = 0.0                              # the flag of the failed call must not stick
    g = _static(e, A, None, out)
    assert g.tolist() == [0, 2, 1] + [0] * 9    # separations 10, 10, 20 degrees on the equator; bins of 18 degrees


def test_static_count_rejects_sizes_beyond_the_static_scratch():
    """Argument checks come before any CUDA call, so they run without a GPU."""
    e = np.array([0.0, 180.0])
    fake = 256      # never dereferenced: the call fails first
    for n_i, n_j, ptr_j in ((T.TPCF_STATIC_MAX_ROWS + 1, 0, None), (T.TPCF_STATIC_MAX_ROWS, 1, fake), (40000, 40000, fake)):
        with pytest.raises(T.TpcfError) as ei:
            T.tpcf_count_static(1, e, "explicit", fake, n_i, ptr_j, n_j, T.TPCF_F64, fake)
        assert ei.value.status == T.TPCF_EINVAL and "TPCF_STATIC_MAX_ROWS" in str(ei.value)
    big = T.TPCF_STATIC_MAX_BINS + 1
    with pytest.raises(T.TpcfError) as ei:
        T.tpcf_count_static(big, np.linspace(0.0, 180.0, big + 1), "explicit", fake, 10, None, 0, T.TPCF_F64, fake)
    assert ei.value.status == T.TPCF_EINVAL and "TPCF_STATIC_MAX_BINS" in str(ei.value)
    with pytest.raises(T.TpcfError):            # a j-catalog without rows, and rows without a j-catalog
        T.tpcf_count_static(1, e, "explicit", fake, 10, fake, 0, T.TPCF_F64, fake)
    with pytest.raises(T.TpcfError):
        T.tpcf_count_static(1, e, "explicit", fake, 10, None, 5, T.TPCF_F64, fake)
