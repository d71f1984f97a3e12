"""NEXT-1 ("multi-GPU solution", "full-blown multi-GPU implementation") with the
real kernels in real processes: two ranks (both on cuda:0 -- this pool has one GPU per box; their kernels never wait on
one another), each loading both catalogs, taking its share of the tile work plan (tpcf_set_partition), counting DD, DR
and RR with the CUDA kernels, one all-reduce of the integer histograms (gloo here, NCCL in bench.py --gpus N), then the
estimator on the summed counts.  The sum must equal the single-process histograms bit for bit and match the oracle."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

import oracle
import paper_1204_6630_b200 as T
import synth
from test_gpu_parity import KINDS, assert_parity, assert_w, full, oracle_all, totals

pytestmark = pytest.mark.gpu
ND, NR = 20_000, 17_777


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, engine, q):
    import torch
    import torch.distributed as dist

    import paper_1204_6630_b200 as TT
    from paper_1204_6630_b200 import dist as tdist

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        D, R, e, cfg = synth.make_config(2, n_d=ND, n_r=NR)
        with TT.Context(cfg.nbins, e, "explicit") as c:
            c.set_engine(engine)
            c.set_tensor_share_limit(1.0)          # "tensor" means pair_tensor_kernel here, whatever the block mix
            c.load("D", D)
            c.load("R", R)
            assert tdist.apply_partition(c) == (rank, world)
            mine, pairs = [], []
            for k in KINDS:
                h, u, o = c.count(k)
                mine.append(np.concatenate([[u], h.astype(np.int64), [o]]))
                pairs.append(c.stats()["pairs"])
            mine = np.stack(mine)
            summed = tdist.allreduce_counts(mine.copy())
            w = TT.tpcf_estimate_from(summed[0][1:-1], summed[1][1:-1], summed[2][1:-1], ND, NR)
            q.put((rank, mine.tolist(), pairs, summed.tolist(), w.tolist(), c.stats()["block"]))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("engine", ["tensor", "fast"])
def test_two_processes_count_their_partitions_and_allreduce(engine, oracle_threads):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, engine, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=600) for _ in procs)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    D, R, e, cfg = synth.make_config(2, n_d=ND, n_r=NR)
    with T.Context(cfg.nbins, e, "explicit") as c:
        c.set_engine(engine)
        c.set_tensor_share_limit(1.0)
        c.load("D", D)
        c.load("R", R)
        single = np.stack([full(*c.count(k)) for k in KINDS])
        w1 = c.estimate()
    part0, part1 = np.asarray(got[0][1]), np.asarray(got[1][1])
    want = totals(ND, NR)
    for i, k in enumerate(KINDS):
        assert got[0][2][i] + got[1][2][i] == want[k]                      # the partition covers every pair once
        assert int(part0[i].sum()) == got[0][2][i] and int(part1[i].sum()) == got[1][2][i]
        assert min(got[0][2][i], got[1][2][i]) > 0.3 * want[k]             # and both ranks really worked
    for rank in range(2):
        np.testing.assert_array_equal(np.asarray(got[rank][3]), single)    # all-reduced sum == single process, on both ranks
        np.testing.assert_array_equal(np.asarray(got[rank][4]), w1)
    np.testing.assert_array_equal(part0 + part1, single)
    o = oracle_all(D, R, e, oracle_threads)
    for i, k in enumerate(KINDS):
        assert_parity(single[i], o[k], want[k])
    assert_w(w1, oracle.estimate(o["DD"].hist, o["DR"].hist, o["RR"].hist, ND, NR))


def _run_bench(*flags):
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    return subprocess.run([sys.executable, os.path.join(root, "bench.py"), *flags], cwd=root, env=env, capture_output=True,
                          text=True, timeout=900)


def test_bench_gpus_2_starts_two_ranks_by_itself():
    """`python bench.py --gpus 2` with no launcher around it must start the two ranks itself (it used to
    count on one GPU and print n_gpus 1).  gloo, because this box has one GPU; the totals check inside bench.py runs on the
    all-reduced histograms, so a rank that did not take its share of the plan fails the run."""
    import json
    r = _run_bench("--gpus", "2", "--backend", "gloo", "--config", "2", "--steps", "3", "--no-cpu-baseline")
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, "exactly one JSON line, from rank 0"
    line = json.loads(lines[0])
    assert line["n_gpus"] == 2 and line["config"]["comm_nranks"] == 2
    assert "communicator of 2 ranks" in r.stderr
    assert line["e2e"]["value"] > 0 and "all-reduce of the device histograms" in line["e2e"]["path"]


def test_bench_refuses_nccl_with_more_ranks_than_gpus():
    """NCCL needs one device per rank: with fewer visible GPUs the run must stop with a clear message, not stack the ranks
    on one device and still print n_gpus = world."""
    import torch
    n = torch.cuda.device_count() + 1
    r = _run_bench("--gpus", str(n), "--backend", "nccl", "--config", "1", "--steps", "1", "--no-cpu-baseline")
    assert r.returncode != 0
    assert "needs one GPU per rank" in r.stderr
    assert not [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
