"""World-size-2 gloo run of the multi-process host logic (no GPU): each rank takes its slice of the tile work
plan (the arithmetic tpcf_set_partition uses), builds a stand-in histogram from the number of pairs in its
items, and the all-reduce must reproduce the single-process result exactly."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist

    import paper_1204_6630_b200 as T
    from paper_1204_6630_b200 import dist as tdist

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        nb, n_d, n_r = 12, 23_456, 31_000
        with T.Context(nb, [0.01, 10.0], "log") as c:
            r, w = tdist.apply_partition(c)          # validates and stores (rank, world) in the context
            assert (r, w) == (rank, world)
            out = {}
            for kind in ("DD", "DR", "RR"):
                n_items = c.plan(kind, n_d, n_r)
                mine = np.zeros(nb + 2, dtype=np.uint64)
                for item in range(rank, n_items, world):
                    mine[item % (nb + 2)] += np.uint64(c.plan_item_pairs(kind, n_d, n_r, item))
                out[kind] = tdist.allreduce_counts(mine)
            if rank == 0:
                full = {}
                for kind in ("DD", "DR", "RR"):
                    n_items = c.plan(kind, n_d, n_r)
                    f = np.zeros(nb + 2, dtype=np.uint64)
                    for item in range(n_items):
                        f[item % (nb + 2)] += np.uint64(c.plan_item_pairs(kind, n_d, n_r, item))
                    full[kind] = f
                q.put({k: (out[k].tolist(), full[k].tolist()) for k in out})
    finally:
        dist.destroy_process_group()


def test_two_rank_partition_and_allreduce_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = q.get(timeout=300)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    n_d, n_r = 23_456, 31_000
    want = {"DD": n_d * (n_d - 1) // 2, "DR": n_d * n_r, "RR": n_r * (n_r - 1) // 2}
    for kind, (got, full) in res.items():
        assert got == full
        assert sum(got) == want[kind]
