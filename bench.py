#!/usr/bin/env python
"""bench.py -- one JSON line for the DD+DR+RR pair-count hot path (BASELINE.json metric) on N GPUs of one node.

A "step" is one full pass of the hot path over one synthetic catalog pair: the three histograms DD, DR, RR of
the workload (default: BASELINE.json configs[2], the paper-scale 430k + 430k octant catalogs of Table 2 row 1,
PAPER.md:61) with the catalogs already resident in HBM; `e2e` repeats it through the synchronous C-ABI calls
with pinned HOST buffers (tpcf_load x2 + tpcf_count x3 + tpcf_estimate, host<->device copies inside the timed
region).  `--impl reference` times the fp64 oracle (oracle/, test infrastructure) on the host cores instead.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl ours|reference]
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import synth  # noqa: E402

KINDS = ("DD", "DR", "RR")
METRIC = "pair evals/sec (DD+DR+RR)"
UNIT = "Gpairs/s"
LANES_PER_CLK_PER_SM = 128      # 4 schedulers x 1 warp instruction x 32 lanes
PAPER_CONTEXT = {"table2_row1_0.43e6_lines_seconds": {"cpu_2xE5520": 3.60e4, "gtx295": 3.01e2, "c1060": 2.91e2,
                                                      "c2050": 2.19e2}, "source": "PAPER.md:61 (other hardware; context, not target)"}


def total_pairs(nd: int, nr: int) -> int:
    return nd * (nd - 1) // 2 + nd * nr + nr * (nr - 1) // 2


def workload_name(idx: int, cfg, nd: int, nr: int) -> str:
    return (f"BASELINE.json configs[{idx - 1}] {cfg.name}: N_D={nd}, N_R={nr}, {cfg.nbins} {cfg.mode} bins "
            f"{cfg.theta_min}-{cfg.theta_max} deg, {total_pairs(nd, nr):.4g} pairs per step")


class Workload:
    """The catalogs, edges and names of one bench workload: BASELINE.json configs 1-5 (angular), or 6 = the 3-D variant of
    the paper-scale case: 430k clustered + 430k uniform rows in a 1000-box, 40 log bins
    in r from 1 to 200."""

    def __init__(self, idx: int, shuffle_d: bool = False):
        self.idx, self.spatial = idx, idx == 6
        if self.spatial:
            self.D, self.R, self.e = synth.make_box_config()
            self.nbins, self.max_abs = len(self.e) - 1, 1000.0
            self.name = (f"3-D variant (PAPER.md:18) of the paper-scale case: N_D={len(self.D)} clustered, N_R={len(self.R)} uniform rows "
                         f"(x, y, z) in a 1000-box, 40 log bins in r 1-200, {total_pairs(len(self.D), len(self.R)):.4g} pairs per step")
        else:
            self.D, self.R, self.e, cfg = synth.make_config(idx, shuffle_d=shuffle_d)
            self.nbins, self.max_abs = cfg.nbins, None
            self.name = workload_name(idx, cfg, len(self.D), len(self.R)) + (" (rows of D in a seeded random order, SURVEY.md A16)" if shuffle_d else "")

    def context(self, T):
        return T.Context(self.nbins, self.e, "explicit", max_abs_coord=self.max_abs)

    def oracle_rows(self, oracle, rows_per_hist: int, threads: int):
        """(pairs, seconds) of the oracle on a seeded row subset of each of DD, DR, RR"""
        if self.spatial:
            d, r = self.D, self.R
            cnt = lambda a, rows, b, ex: oracle.count_rows_xyz(a, rows, b, ex, self.e, threads=threads)
        else:
            d, r = oracle.radec_to_xyz(self.D), oracle.radec_to_xyz(self.R)
            cnt = lambda a, rows, b, ex: oracle.count_rows(a, rows, b, ex, self.e, threads=threads)
        rd, rr = synth.subset_rows(len(d), rows_per_hist, 777), synth.subset_rows(len(r), rows_per_hist, 778)
        t0 = time.perf_counter()
        tot = cnt(d, rd, d, True).total + cnt(d, rd, r, False).total + cnt(r, rr, r, True).total
        return tot, time.perf_counter() - t0


class ClockSampler:
    """nvidia-smi SM clock / throttle reasons every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True)
            self.th.start()
        except OSError:
            self.proc = None
        return self

    def __exit__(self, *exc):
        if self.proc:
            time.sleep(0.25)
            self.proc.terminate()
            self.th.join(timeout=2)

    def summary(self):
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "reasons": sorted(reasons), "samples": len(sm)}


# Algorithmic work of one pair: the dot product of PAPER.md:37 in expanded form, 4 FP32
# lane-operations on the FMA pipes (1 add + 3 fused multiply-adds), and its bin decision against one edge, 1.5
# lane-operations on the ALU pipe (sign-bit add + half of a 3-input minimum for the guard band).
OPS_PER_PAIR = 5.5


def profile_summary(cfg_idx: int, engine: str = "fast"):
    """Executed-instruction figures of the pair kernel from the committed ncu capture (profiles/inst_per_pair.json)."""
    path = os.path.join(ROOT, "profiles", "inst_per_pair.json")
    try:
        d = json.load(open(path))
        return d.get(f"cfg{cfg_idx}_{engine}") or {}        # no capture of this (config, kernel): the line prints null
    except Exception:
        return {}


# ------------------------------------------------------------------------------------------------ oracle legs
def oracle_sample_rate(wl, rows_per_hist: int, threads: int):
    """Time the oracle (as it stands) on a seeded row subset of each of DD, DR, RR; returns (pairs, seconds)."""
    import oracle
    return wl.oracle_rows(oracle, rows_per_hist, threads)


def run_reference(args):
    """--impl reference: the oracle on the host cores, each step a bounded sample of the workload."""
    import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = Workload(args.config, args.shuffle_d)
    nd, nr = wl.D.shape[0], wl.R.shape[0]
    threads = oracle.host_threads()
    pairs, dt = oracle_sample_rate(wl, 16, threads)          # probe to size the sample
    rate = pairs / dt
    budget = 150.0 / (args.steps + args.warmup)                   # whole run within a few minutes
    rows = int(max(16, min(2000, rate * min(budget, 20.0) / (nd + nr + nr))))
    for _ in range(args.warmup):
        oracle_sample_rate(wl, rows, threads)
    t_tot, p_tot = 0.0, 0
    for _ in range(args.steps):
        p, t = oracle_sample_rate(wl, rows, threads)
        p_tot += p
        t_tot += t
    val = p_tot / t_tot / 1e9
    sample = f"{rows} seeded rows of each of DD, DR, RR against all j ({p_tot // args.steps:.4g} pairs per step)"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t_tot / args.steps, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "full_workload_seconds_extrapolated": total_pairs(nd, nr) / (val * 1e9)}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_1204_6630_b200 as T
    from paper_1204_6630_b200 import dist as tdist

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: libtpcf has no CPU fallback")
    ndev = torch.cuda.device_count()
    if world > ndev:
        if args.backend == "nccl":      # one rank per GPU, no exceptions: NCCL cannot put two ranks on one device
            print(f"[bench] {world} ranks but only {ndev} CUDA device(s) visible: --backend nccl needs one GPU per rank "
                  f"(use --backend gloo to smoke-test the N > 1 path on fewer GPUs)", file=sys.stderr, flush=True)
            return 2
        local = local % ndev            # gloo smoke test on a box with fewer GPUs than ranks: ranks share devices
    torch.cuda.set_device(local)
    if world > 1:
        if args.backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group(args.backend)
        print(f"[bench] rank {rank}/{world}: communicator of {dist.get_world_size()} ranks, backend {dist.get_backend()}, "
              f"device cuda:{local}", file=sys.stderr, flush=True)
    wl = Workload(args.config, args.shuffle_d)
    D, R, e = wl.D, wl.R, wl.e
    nd, nr = D.shape[0], R.shape[0]
    pairs_step = total_pairs(nd, nr)
    nb = wl.nbins

    st = torch.cuda.Stream()
    ctx = wl.context(T)
    ctx.set_stream(st.cuda_stream)
    if args.engine != "default":
        ctx.set_engine(args.engine)
    if args.pruning:
        ctx.set_pruning(True)
    ctx.load("D", D, stream=st.cuda_stream)
    ctx.load("R", R, stream=st.cuda_stream)
    tdist.apply_partition(ctx)
    out = torch.zeros(3, nb + 2, dtype=torch.int64, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")      # > 126 MB L2

    def step():
        with torch.cuda.stream(st):
            flush.zero_()                                   # L2 flush between steps (inside the timed region)
            ctx.count_all_async(out)                        # DD, DR, RR in flight together (tpcf_count_all_async)
            if world > 1:
                tdist.allreduce_counts(out)                 # 3 x (nbins+2) int64 over NCCL: the only exchange

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    ctx.set_kernel_timing(True)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    kernel_ms = []
    with ClockSampler(local) as clk:
        barrier()
        ev0.record(st)
        for _ in range(args.steps):
            step()
        ev1.record(st)
        barrier()
    ms_total = ev0.elapsed_time(ev1)
    kernel_ms = [float(x) for x in ctx.kernel_times_ms()]                # per pair-kernel launch, CUDA events on the launching stream
    ctx.set_kernel_timing(False)
    t = torch.tensor([ms_total], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_total = float(t.item())
    ms_step = ms_total / args.steps
    value = pairs_step / (ms_step * 1e-3) / 1e9
    stats = ctx.stats()

    # check the result the timed steps produced (totals identity; full parity lives in tests/)
    res = out.cpu().numpy()
    want = (nd * (nd - 1) // 2, nd * nr, nr * (nr - 1) // 2)
    for i in range(3):
        assert int(res[i].sum()) == want[i], (KINDS[i], int(res[i].sum()), want[i])

    # the other engine on the same resident catalogs, a few steps, for the record (its histograms must be the same integers)
    other = None
    if world == 1 and args.engine in ("default", "tensor") and not args.pruning:
        ctx.set_engine("fast")
        out2 = torch.zeros_like(out)
        def step2():
            with torch.cuda.stream(st):
                flush.zero_()
                ctx.count_all_async(out2)
        step2()
        barrier()
        ev2, ev3 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev2.record(st)
        for _ in range(3):
            step2()
        ev3.record(st)
        barrier()
        ms2 = ev2.elapsed_time(ev3) / 3
        assert torch.equal(out2, out), "fast and tensor engines disagree"
        other = {"engine": "fast (FFMA2 window loops)", "value": pairs_step / (ms2 * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": ms2, "steps": 3,
                 "histograms_identical_to_the_timed_engine": True}
        ctx.set_engine("tensor")

    # ---- end to end through the synchronous C ABI with pinned host buffers --------------------------------
    Dp, Rp = torch.from_numpy(D).pin_memory(), torch.from_numpy(R).pin_memory()
    e2e_steps = max(1, min(args.steps, 5))

    e2e_out = torch.zeros_like(out)

    def e2e_step():
        ctx.load("D", Dp, stream=st.cuda_stream)            # H2D copy + on-device conversion
        ctx.load("R", Rp, stream=st.cuda_stream)
        tdist.apply_partition(ctx)
        if world > 1:
            # the partial histograms stay on the device for the all-reduce; one D2H of the summed counts, then Eq. 1
            with torch.cuda.stream(st):
                ctx.count_all_async(e2e_out)
                tdist.allreduce_counts(e2e_out)
                arr = e2e_out.cpu().numpy()
            return T.tpcf_estimate_from(arr[0][1:-1].astype(np.uint64), arr[1][1:-1].astype(np.uint64),
                                        arr[2][1:-1].astype(np.uint64), nd, nr)
        ctx.count_all()                                     # D2H of the three histograms inside
        return ctx.estimate()

    e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        w = e2e_step()
    barrier()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    e2e_s = float(t.item())
    h2d = D.nbytes + R.nbytes
    d2h = 3 * (nb + 2) * 8 + 2 * 4              # the three histograms of tpcf_count_all + the two load flags

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (pair_fast_kernel): plain ALU issue --------------------------------
    clocks = clk.summary()
    tensor_ran = stats["block"] == 128          # fine binnings (config 5) run the FFMA2 kernel under either engine
    prof = profile_summary(args.config, "tensor" if tensor_ran else "fast")
    peak_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        sm_max = float(json.load(open(peak_path))["sm_max_mhz"])
        peak_src = "MEASURED_PEAKS.json sm_max_mhz"
    except Exception:
        sm_max, peak_src = 1965.0, "fallback 1965 MHz (B200_PROFILING.md nominal clocks.max.sm)"
    SM_COUNT = torch.cuda.get_device_properties(local).multi_processor_count
    peak = SM_COUNT * LANES_PER_CLK_PER_SM * sm_max * 1e6 / 1e12          # T lane-operations/s
    # per launch: pairs of that histogram (this rank's share) / its own duration; the three launches repeat DD, DR, RR
    share = [w_ / world for w_ in want]
    # one CUDA-event pair per step around the three overlapping pair kernels (tpcf_count_all_async)
    pairs_per_s_kernel = (sum(share) * len(kernel_ms) / (sum(kernel_ms) * 1e-3)) if kernel_ms else pairs_step / world / (ms_step * 1e-3)
    achieved = pairs_per_s_kernel * OPS_PER_PAIR / 1e12
    ppcs = pairs_per_s_kernel / (SM_COUNT * sm_max * 1e6)          # pairs per clock per SM at the maximum SM clock
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "T lane-operations/s (FP32 FMA-pipe + ALU-pipe operations)",
                "frac": achieved / peak, "traffic": prof.get("dram_bytes_per_launch"),
                "kernel": "pair_tensor_kernel" if tensor_ran else "pair_fast_kernel", "ops_per_pair": OPS_PER_PAIR,
                "ops_per_pair_source": "DESIGN.md section 7: 4 FMA-pipe + 1.5 ALU-pipe lane-operations per pair (1-edge window loop)" +
                                       ("; in the tensor engine the 4 dot-product operations run as a 3xTF32 tcgen05.mma, the 1.5 bin-decision "
                                        "operations on the ALU pipe (bound 42.7 pairs/clk/SM)" if tensor_ran else ""),
                "executed_inst_per_pair": prof.get("inst_per_pair"), "issue_active_pct": prof.get("issue_active_pct"),
                "executed_source": prof.get("source"),
                "kernel_pairs_per_s": pairs_per_s_kernel, "kernel_ms_avg": (sum(kernel_ms) / len(kernel_ms)) if kernel_ms else None,
                "kernel_ms_note": "per step: from the start of the first to the end of the last of the three overlapping pair kernels",
                "kernel_launches_timed": len(kernel_ms),
                "kernel_share_of_step": (sum(kernel_ms) / ms_total) if kernel_ms else None,
                "pairs_per_clk_per_sm_at_max_clock": ppcs,
                # BASELINE.json north_star's own figure: N_SM x 128 x f / (executed instructions per pair), the count taken
                # from the committed ncu capture of THIS (config, kernel variant) -- null when there is none
                "frac_counted_instruction": (ppcs * prof["inst_per_pair"] / LANES_PER_CLK_PER_SM) if prof.get("inst_per_pair") else None,
                # the pipe that binds the tensor kernel: 1.5 ALU-pipe instructions per pair at 64 lanes/clk/SM = 42.7 pairs/clk/SM
                "frac_of_alu_pipe_bound": (ppcs / (64.0 / 1.5)) if tensor_ran else None,
                "fma_pipe_bound_pairs_per_clk_per_sm": LANES_PER_CLK_PER_SM / 4.0,
                "peak_source": f"{SM_COUNT} SMs x {LANES_PER_CLK_PER_SM} FP32 lanes/clk x {sm_max:.0f} MHz ({peak_src}); DESIGN.md section 7",
                "frac_at_sampled_clock": (achieved / (SM_COUNT * LANES_PER_CLK_PER_SM * clocks["sm_mhz"] * 1e6 / 1e12)) if clocks.get("sm_mhz") else None}

    if args.pruning:        # blocks are added wholesale: pairs per second is not work per second, no roofline applies
        roofline.update({"achieved": None, "frac": None, "frac_at_sampled_clock": None,
                         "note": "pruning mode: unevaluated blocks make pairs/s incomparable with the brute-force roofline"})

    # ---- the oracle timed beside it (rank 0, N = 1 only) --------------------------------------------------------
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        threads = oracle.host_threads()
        p0, t0_ = oracle_sample_rate(wl, 16, threads)
        rows = int(max(16, min(2000, (p0 / t0_) * 15.0 / (nd + nr + nr))))
        p1, t1_ = oracle_sample_rate(wl, rows, threads)
        cpu = {"value": p1 / t1_ / 1e9, "unit": UNIT, "cores": threads, "kind": "oracle",
               "sample": f"{rows} seeded rows of each of DD, DR, RR against all j = {p1:.4g} pairs in {t1_:.1f} s",
               "full_workload_seconds_extrapolated": pairs_step / (p1 / t1_)}

    metric = METRIC if not args.pruning else \
        "pairs COUNTED/sec (DD+DR+RR) in pruning mode: blocks without a bin edge in reach are added wholesale, NOT evaluated (SURVEY.md NEXT-3); not BASELINE.json's metric"
    line = {"metric": metric, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": wl.name,
                       "l2": "256 MiB write between steps (inside the timed region); catalogs (28 MB each) are L2-resident by design",
                       "engine": ("tensor (window quantity by 3xTF32 tcgen05.mma into TMEM + tcgen05.ld read-back; guard bands, cell lookup and "
                                  "fp64 recheck as in the fast engine)" if tensor_ran else
                                  "fast (fp32 squared chord by FFMA2 + fp64 recheck of guard-band pairs)"),
                       "parallelism": f"tile work items w % {world} == rank, one all-reduce of 3x{nb + 2} int64" if world > 1 else "1 GPU",
                       "comm_nranks": world, "grid": stats["grid"], "block": stats["block"], "smem_bytes": stats["smem_bytes"], "cells": stats["cells"]},
            "seconds_per_w_theta": ms_step * 1e-3,
            "e2e": {"value": pairs_step / e2e_s / 1e9, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "seconds_per_step": e2e_s, "steps": e2e_steps,
                    "path": ("tpcf_load_xyz" if wl.spatial else "tpcf_load") + "(D), (R) from pinned host rows + " +
                            ("tpcf_count_all + tpcf_estimate" if world == 1 else
                             "tpcf_count_all_async + all-reduce of the device histograms + one D2H + tpcf_estimate_from")},
            "gpu_launches": args.steps * 6,
            "gpu_launches_note": f"per step: 3 x ({'pair_tensor_kernel' if tensor_ran else 'pair_fast_kernel'} + finalize_kernel), the three pair kernels in flight together on three streams (tpcf_count_all_async); memsets are driver memset nodes; the e2e leg adds 2 x 29 load kernels per step",
            "other_engine": other,
            "clocks": clocks, "roofline": roofline, "cpu_baseline": cpu, "paper_context": PAPER_CONTEXT}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def spawn_ranks(n: int) -> int:
    """`python bench.py --gpus N` without a launcher: re-run this command line as N ranks (one per GPU) under
    torch.distributed.run on this node, exactly as the driver launches the N > 1 line; rank 0 prints the JSON line."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5, 6],
                    help="BASELINE.json configs 1-5; 6 = the 3-D variant (Cartesian rows, bins in r) of the paper-scale case")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="torch.distributed backend of the N > 1 run (gloo: smoke test of that path on a box with one GPU)")
    ap.add_argument("--shuffle-d", action="store_true", help="configs 1-5: rows of D in a seeded random order instead of generation order (SURVEY.md A16)")
    ap.add_argument("--pruning", action="store_true",
                    help="time the separately named pruning mode (tpcf_set_pruning; not the brute-force count, not the headline)")
    ap.add_argument("--engine", default="default", choices=["default", "tensor", "fast"],
                    help="pair kernel family (include/tpcf.h tpcf_engine); default = the library's default (tensor); both give the same histograms")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.steps < 1:
        ap.error("--steps must be >= 1")
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args.gpus)
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
