#!/usr/bin/env python
"""bench.py -- headline benchmark of the batched semi-global alignment path (libsdp) on B200.

One "step" is one pass of the whole hot path (validate, bucket, forward score, reverse pass,
traceback + CIGAR, similarity filter, compaction) over one batch of synthetic pairs. The default
workload is BASELINE.json configs[1]: 1,000,000 pairs of 100 bp reads against 500 bp windows cut
from a seeded 100 Mbp reference (mate-rescue shape). Prints ONE JSON line.

    python bench.py --gpus 1 --steps 5 --warmup 3
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...
    python bench.py --impl reference      # the CPU oracle, as it stands, on the host cores
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "gcups"
UNIT = "GCUPS"
SM_COUNT_NOMINAL = 148
SM_MAX_MHZ_FALLBACK = 1965.0
DPX_RATE = 64.0            # int16x2 DPX thread-instructions / clk / SM (measured)
INSTR_PER_2_CELLS = 4.0    # algorithmic work: 4 int16x2 instructions per 2 cells


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, device: int):
        self.device, self.rows, self.proc, self.th = device, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.device), "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.th = threading.Thread(target=self._pump, daemon=True)
        self.th.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        mhz, mx, reasons, power = [], None, set(), []
        for ts, line in self.rows:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 8 or not (t0 - 0.05 <= ts <= t1 + 0.15):
                continue
            try:
                mhz.append(float(f[1])); mx = float(f[2]); power.append(float(f[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(mhz) if mhz else None, "sm_max_mhz": mx,
                "power_w_max": max(power) if power else None, "samples": len(mhz), "reasons": sorted(reasons)}


def dist_setup(n_gpus: int):
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(local)
        dist.init_process_group(backend="nccl" if torch.cuda.is_available() else "gloo",
                                device_id=torch.device("cuda", local) if torch.cuda.is_available() else None)
    return rank, world, local


def oracle_timed(batch, n_pairs: int, threads: int):
    """Time the oracle, as it stands, on the first n_pairs pairs. Returns (seconds, cells, threads used)."""
    import oracle
    sub = batch.subset(np.arange(min(n_pairs, batch.n_pairs)))
    t0 = time.perf_counter()
    r = oracle.align_batch(sub.reads_packed, sub.read_off, sub.read_len, sub.wins_packed, sub.win_off, sub.win_len,
                           sub.pairs, oracle.OracleScoring(), read_nmask=sub.read_nmask, win_nmask=sub.win_nmask,
                           threads=threads)
    return time.perf_counter() - t0, sub.cells, r.threads, sub.n_pairs


def cpu_baseline(batch, budget_s: float = 15.0):
    threads = os.cpu_count() or 1
    dt, cells, used, n = oracle_timed(batch, 4 * threads * 8, threads)          # calibration
    rate = n / max(dt, 1e-6)
    want = int(max(n, min(batch.n_pairs, rate * budget_s)))
    dt, cells, used, n = oracle_timed(batch, want, threads)
    # one thread on the first 20,000 pairs -> per-core figure (bounded to a few seconds)
    n1 = int(min(20_000, batch.n_pairs, max(200, rate / max(used, 1) * 4.0)))
    dt1, cells1, used1, n1 = oracle_timed(batch, n1, 1)
    return {"value": cells / dt / 1e9, "unit": UNIT, "cores": used, "kind": "oracle",
            "pairs_per_s": n / dt, "seconds": dt,
            "sample": f"first {n} pairs of the workload, {used} OpenMP threads over disjoint pair ranges",
            "single_thread": {"value": cells1 / dt1 / 1e9, "unit": UNIT, "cores": used1, "pairs_per_s": n1 / dt1,
                              "seconds": dt1, "sample": f"first {n1} pairs of the workload, one thread"}}


def run_reference(args, rank):
    """--impl reference: the CPU oracle on the host cores (tier rule: the oracle is the reference arm)."""
    if rank != 0:
        return
    from paper_1302_5507_b200 import workloads as W
    import oracle
    oracle.build()
    threads = os.cpu_count() or 1
    n_sample = args.ref_pairs
    batch = W.make_config(args.config, n_pairs=max(n_sample, 1), ref_bases=args.ref_bases if args.config != 1 else 1_000_000)
    for _ in range(args.warmup):
        oracle_timed(batch, min(n_sample, 2000), threads)
    times, cells, used = [], 0, threads
    for _ in range(args.steps):
        dt, cells, used, n = oracle_timed(batch, n_sample, threads)
        times.append(dt)
    tot = sum(times)
    value = cells * args.steps / tot / 1e9
    sample = f"{n_sample} pairs of {W_NAME[args.config]} per step, {used} OpenMP threads"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32",
        "data": "synthetic", "pairs_per_s": n_sample * args.steps / tot,
        "config": {"workload": W_NAME[args.config], "pairs_per_step": n_sample,
                   "note": "bounded sample of the same seeded workload; CPU oracle (three int32 tables + traceback)"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": used, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


W_NAME = {
    1: "cfg1: 1,000 pairs 100bp x 300bp (PR1 ref)",
    2: "cfg2: 1,000,000 pairs 100bp x 500bp mate-rescue shape (BASELINE.json configs[1])",
    3: "cfg3: 2,000,000 pairs 150bp x 600bp, 3' quality decay, tandem repeats",
    4: "cfg4: 500,000 pairs 250bp x 750bp low-similarity stress",
    5: "cfg5: 4,000,000 pairs 50-300bp mixed length, 10% N reference",
}


def time_config(S, W, torch, dev, local, cfg, n_pairs, ref_bases, seed, steps, warmup, flush, peak):
    """One BASELINE.json config at full size on this GPU: device-resident timing of the whole sdp_align_batch call
    (CUDA events on the launching stream, L2 flushed between steps), its own clocks sample, stage split."""
    batch = W.make_config(cfg, n_pairs=n_pairs, ref_bases=ref_bases if cfg != 1 else 1_000_000, seed=seed)
    return time_batch(S, torch, dev, local, batch, W_NAME[cfg], steps, warmup, flush, peak)


def time_batch(S, torch, dev, local, batch, workload, steps, warmup, flush, peak, local_mode=False):
    """The same timing for any batch; local_mode = SDP_MODE_LOCAL (every pair then runs on the int32 lane)."""
    ctx = S.Context(device=local)
    try:
        ctx.set_mode(local=local_mode)
        dbatch = ctx.upload(batch)
        stream = torch.cuda.current_stream(dev)
        ctx.set_timing(True)
        for _ in range(warmup):
            ctx.align_batch(dbatch, stream)
        sampler = ClockSampler(local)
        sampler.start()
        torch.cuda.synchronize(dev)
        t0 = time.time()
        ms, fwd, stats = [], [], {}
        for _ in range(steps):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            ctx.align_batch(dbatch, stream)
            e1.record(stream)
            e1.synchronize()
            ms.append(e0.elapsed_time(e1))
            stats = ctx.stats()
            fwd.append(stats["ms_forward"])
        torch.cuda.synchronize(dev)
        clocks = sampler.stop(t0, time.time())
        mean = statistics.mean(ms)
        fwd_gcups = batch.cells / (statistics.mean(fwd) * 1e-3) / 1e9
        return {"workload": workload, "mode": "local" if local_mode else "semi-global",
                "pairs": batch.n_pairs, "cells": batch.cells, "steps": steps, "warmup": warmup,
                "ms_per_step": mean, "ms_best": min(ms), "ms_median": statistics.median(ms),
                "gcups": batch.cells / (mean * 1e-3) / 1e9, "pairs_per_s": batch.n_pairs / (mean * 1e-3),
                "stages_ms": {k: stats.get(k) for k in ("ms_total", "ms_bucket", "ms_forward", "ms_reverse", "ms_traceback",
                                                        "ms_compact")},
                "kernel_launches_per_step": stats.get("kernel_launches"),
                "pairs_on_int32_lane": bool(stats.get("n_slow_words")),
                "forward_gcups": fwd_gcups, "forward_frac": fwd_gcups / peak,
                "whole_path_frac": batch.cells / (mean * 1e-3) / 1e9 / peak, "clocks": clocks}
    finally:
        ctx.destroy()
        del batch


def time_step3(S, W, torch, dev, local, ref_bases, flush, peak, n_reads=65_000, steps=3, warmup=2):
    """Step-3 shape: every read against U{1..30} candidate windows. Times the
    screening flow -- forward score of every candidate (sdp_set_score_only), the per-read choice (sdp_best_per_read),
    full alignment of the winners only -- beside the full alignment of every candidate, and the screening pass on the
    same pairs in shuffled order (does keeping a read's candidates adjacent in the pair list buy anything?)."""
    b = W.make_step3(n_reads, max_candidates=30, ref_bases=ref_bases)
    ctx = S.Context(device=local)
    stream = torch.cuda.current_stream(dev)

    def timed(fn, reps=steps, warm=warmup):
        for _ in range(warm):
            fn()
        ms = []
        for _ in range(reps):
            flush.fill_(1)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            r = fn()
            e1.record(stream)
            e1.synchronize()
            ms.append(e0.elapsed_time(e1))
        return statistics.mean(ms), min(ms), r

    try:
        db = ctx.upload(b)
        ctx.set_timing(True)
        full_ms, full_best, _ = timed(lambda: ctx.align_batch(db, stream))
        ctx.set_score_only(True)
        scr_ms, scr_best, res = timed(lambda: ctx.align_batch(db, stream))
        scr_fwd = ctx.stats()["ms_forward"]
        best_ms, best_best, best = timed(lambda: ctx.best_per_read(db, res, stream))
        perm = np.random.default_rng(7).permutation(b.n_pairs)
        dsh = ctx.upload(b.subset(perm))
        shuf_ms, shuf_best, _ = timed(lambda: ctx.align_batch(dsh, stream))
        shuf_fwd = ctx.stats()["ms_forward"]
        ctx.set_score_only(False)
        winners = b.subset(best["best_pair"].astype(np.int64))
        dw = ctx.upload(winners)
        win_ms, win_best, _ = timed(lambda: ctx.align_batch(dw, stream))
        return {"workload": f"step-3 shape: {n_reads} reads x U{{1..30}} candidate windows of 500 bp = {b.n_pairs} pairs "
                            "(true window, up to two shifted copies, decoys)",
                "pairs": b.n_pairs, "reads": n_reads, "cells": b.cells,
                "align_every_candidate_ms": full_ms,
                "screen_score_only_ms": scr_ms, "screen_forward_kernel_ms": scr_fwd,
                "screen_gcups": b.cells / (scr_ms * 1e-3) / 1e9, "screen_forward_frac": b.cells / (scr_fwd * 1e-3) / 1e9 / peak,
                "best_per_read_ms": best_ms, "align_winners_ms": win_ms,
                "screening_flow_ms": scr_ms + best_ms + win_ms,
                "screen_shuffled_pair_order_ms": shuf_ms, "screen_shuffled_forward_kernel_ms": shuf_fwd,
                "note": "best_per_read_ms includes its D2H of the per-read arrays (binding); pair list grouped by read vs the "
                        "same pairs in random order: the forward kernel's read fetches hit L1/L2 either way"}
    finally:
        ctx.destroy()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config number (1-5); 2 is the headline")
    ap.add_argument("--pairs", type=int, default=None, help="override the pair count (debugging only)")
    ap.add_argument("--ref-bases", type=int, default=100_000_000)
    ap.add_argument("--ref-pairs", type=int, default=20_000, help="--impl reference: pairs per step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config block (configs 1, 3, 4, 5 at full size)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--chunks", type=int, default=0, help="sdp_set_chunks: lanes per call (0 = the library's choice)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)

    rank, world, local = dist_setup(args.gpus)
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import paper_1302_5507_b200 as S
    from paper_1302_5507_b200 import workloads as W

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)

    # ---- workload: each rank aligns its own shard (pairs are independent: no collective on the data path)
    cfg = args.config
    n_pairs = args.pairs if args.pairs is not None else None
    ref_bases = args.ref_bases if cfg != 1 else 1_000_000
    batch = W.make_config(cfg, n_pairs=n_pairs, ref_bases=ref_bases,
                          seed=W.SEED_BASE + cfg + 1000 * rank)
    cells = batch.cells
    ctx = S.Context(device=local)
    ctx.set_chunks(args.chunks)
    dbatch = ctx.upload(batch)
    stream = torch.cuda.current_stream(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > 126 MB L2

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            torch.distributed.barrier()

    # ---- device-resident timing: K steps, CUDA events on the launching stream, L2 flushed between steps
    ctx.set_timing(True)
    for _ in range(max(args.warmup, 3) if args.warmup else 0):
        ctx.align_batch(dbatch, stream)
    sampler = ClockSampler(local)
    sampler.start()
    barrier()
    t_wall0 = time.time()
    step_ms, fwd_ms, launches, stats = [], [], 0, {}
    for _ in range(args.steps):
        flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        ctx.align_batch(dbatch, stream)
        e1.record(stream)
        e1.synchronize()
        step_ms.append(e0.elapsed_time(e1))
        stats = ctx.stats()
        fwd_ms.append(stats["ms_forward"])
        launches += stats["kernel_launches"]
    barrier()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1)
    # ---- the same steps with the optional ungapped pre-pass on (sdp_set_prefilter; NOT the headline: pairs it
    # settles skip the DP, so "GCUPS" here counts cells that were never updated)
    ctx.set_prefilter(True)
    pf_ms = []
    for it in range(2 + args.steps):
        flush.fill_(1)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        ctx.align_batch(dbatch, stream)
        e1.record(stream)
        e1.synchronize()
        if it >= 2:
            pf_ms.append(e0.elapsed_time(e1))
    pf_stats = ctx.stats()
    ctx.set_prefilter(False)
    ctx.set_timing(False)
    total_ms = sum(step_ms)
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        torch.distributed.all_reduce(t, op=torch.distributed.ReduceOp.MAX)
        total_ms = float(t.item())
        c = torch.tensor([cells], dtype=torch.float64, device=dev)
        torch.distributed.all_reduce(c, op=torch.distributed.ReduceOp.SUM)
        cells_all = float(c.item())
        pairs_all = batch.n_pairs * world
    else:
        cells_all, pairs_all = float(cells), batch.n_pairs
    value = cells_all * args.steps / (total_ms * 1e-3) / 1e9
    ms_per_step = total_ms / max(args.steps, 1)

    # ---- end to end through the host-buffer ABI call: pinned host inputs, H2D + D2H inside the timed region
    e2e = None
    if not args.no_e2e:
        pinned = {}
        for name in ("reads_packed", "read_off", "read_len", "read_nmask", "wins_packed", "win_off", "win_len",
                     "win_nmask"):
            a = getattr(batch, name)
            if a is not None:
                tsr = torch.from_numpy(np.ascontiguousarray(a).view(np.int64 if a.dtype == np.uint64 else np.int32))
                pinned[name] = tsr.pin_memory()
        pinned["pairs"] = torch.from_numpy(batch.pairs.reshape(-1).view(np.int32)).pin_memory()
        ptrs = {k: (pinned[k].data_ptr() if k in pinned else None)
                for k in ("reads_packed", "read_off", "read_len", "read_nmask", "wins_packed", "win_off", "win_len",
                          "win_nmask", "pairs")}
        cb = ctx._c_batch(ptrs, batch)
        h2d = sum(t.numel() * t.element_size() for t in pinned.values())
        for _ in range(2):
            res = ctx.align_batch_host_raw(cb)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            res = ctx.align_batch_host_raw(cb)
        torch.cuda.synchronize(dev)
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device=dev)
            torch.distributed.all_reduce(t, op=torch.distributed.ReduceOp.MAX)
            dt = float(t.item())
        P = batch.n_pairs
        d2h = P * (4 * 7 + 1 + 8 + 4) + int(res.n_cigar_ops) * 4
        single_ms = dt / args.steps * 1e3
        # Same call, two contexts driven by two host threads (separate contexts are independent, sdp.h):
        # the H2D/D2H copies of one batch overlap the kernels of the other, as a caller streaming batches would.
        pipe_ms = None
        if args.steps >= 2:
            ctx2 = S.Context(device=local)
            ctx2.align_batch_host_raw(cb)
            ctx2.align_batch_host_raw(cb)
            ctxs, errs = (ctx, ctx2), []

            def worker(j):
                try:
                    for _ in range(j, args.steps, 2):
                        ctxs[j].align_batch_host_raw(cb)
                except Exception as ex:  # noqa: BLE001
                    errs.append(ex)

            barrier()
            ths = [threading.Thread(target=worker, args=(j,)) for j in range(2)]
            t0 = time.perf_counter()
            for th in ths:
                th.start()
            for th in ths:
                th.join()
            torch.cuda.synchronize(dev)
            dtp = time.perf_counter() - t0
            ctx2.destroy()
            if errs:
                raise errs[0]
            if world > 1:
                t = torch.tensor([dtp], dtype=torch.float64, device=dev)
                torch.distributed.all_reduce(t, op=torch.distributed.ReduceOp.MAX)
                dtp = float(t.item())
            pipe_ms = dtp / args.steps * 1e3
        e2e = {"value": cells_all / (single_ms * 1e-3) / 1e9, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": single_ms, "ms_per_step_one_context": single_ms,
               "ms_per_step_two_contexts": pipe_ms,
               "value_two_contexts": (cells_all / (pipe_ms * 1e-3) / 1e9) if pipe_ms else None,
               "timer": "host wall clock around K calls of sdp_align_batch_host (pinned host inputs, every result array "
                        "copied back to pinned host memory inside the call); value = ONE context called back to back; "
                        "value_two_contexts = the same calls issued by two host threads on two contexts, so that the copies "
                        "of one batch overlap the kernels of the other (how a caller streaming batches would drive it)"}

    if rank != 0:
        return

    # ---- roofline of the dominant kernel (forward score pass): ALU/DPX bound
    peaks = measured_peaks()
    sm_max = float(peaks.get("sm_max_mhz", SM_MAX_MHZ_FALLBACK))
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    peak = sms * sm_max * 1e6 * DPX_RATE * 2.0 / INSTR_PER_2_CELLS / 1e9
    try:        # issue-rate microbenchmark of this very GPU, reported beside the constant the peak uses
        dpx_live = S.sdp_measure_dpx_rate(local)
    except Exception as ex:  # noqa: BLE001
        dpx_live = {"error": str(ex)}
    fwd = cells / (statistics.mean(fwd_ms) * 1e-3) / 1e9 if fwd_ms and statistics.mean(fwd_ms) > 0 else None
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "forward_traffic.json")) as f:
            traffic = json.load(f).get("dram_bytes_per_launch")
    except Exception:
        pass
    roofline = {"bound": "alu", "kernel": "sdp_score_k<K>_f* (forward score pass, score_kernel.cuh)",
                "achieved": fwd, "peak": peak, "unit": UNIT, "frac": (fwd / peak) if fwd else None,
                "traffic": traffic,
                "peak_how": f"{sms} SMs x {sm_max:.0f} MHz (MEASURED_PEAKS.json sm_max_mhz) x {DPX_RATE:.0f} int16x2 DPX "
                            f"instr/clk/SM (measured, profiles/) x 2 cells / {INSTR_PER_2_CELLS:.0f} instr",
                "traffic_how": "dram__bytes_read.sum + dram__bytes_write.sum of one ncu --set full capture of this kernel on "
                               "this workload, stored in profiles/forward_traffic.json (a profiled constant, not re-measured "
                               "by this run)",
                "achieved_how": "sum n*m of the batch / mean CUDA-event time of the forward-kernel launches per step, "
                                "events recorded by libsdp on the launching stream inside the timed steps",
                "whole_path_frac": value / world / peak, "dpx_rate_measured_now": dpx_live}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int16", "data": "synthetic",
        "pairs_per_s": pairs_all * args.steps / (total_ms * 1e-3),
        "config": {"workload": W_NAME[cfg], "pairs_per_gpu": batch.n_pairs, "cells_per_gpu": cells,
                   "scoring": "match +1 mismatch -3 gap 5+2k min_similarity 0.6",
                   "parallelism": f"independent pair shards x{world} (no collective)",
                   "l2": "256 MiB buffer written between timed steps (L2 flush)",
                   "outputs": "score, ref_start, ref_end, read span, CIGAR, n_match, n_cols, pass for every pair"},
        "ms_best": min(step_ms) if step_ms else None, "ms_median": statistics.median(step_ms) if step_ms else None,
        "stages_ms": {k: stats.get(k) for k in ("ms_total", "ms_bucket", "ms_forward", "ms_reverse", "ms_traceback",
                                                "ms_compact")},
        "roofline": roofline, "clocks": clocks, "gpu_launches": launches, "e2e": e2e,
        "with_ungapped_prepass": {
            "ms_per_step": statistics.mean(pf_ms) if pf_ms else None,
            "effective_gcups": (cells / (statistics.mean(pf_ms) * 1e-3) / 1e9) if pf_ms else None,
            "cells_settled_without_dp_frac": pf_stats.get("cells_prefiltered", 0) / max(1, cells),
            "note": "optional sdp_set_prefilter(1), off in every other number of this line: near-exact pairs get score and "
                    "ref_end from a Hamming scan and skip the forward DP; outputs are bit-identical; rank 0 only"},
    }
    if not args.no_cpu_baseline and world == 1:
        import oracle
        oracle.build()
        out["cpu_baseline"] = cpu_baseline(batch)
    if not args.no_per_config and world == 1 and cfg == 2 and args.pairs is None:
        # the other BASELINE.json configs at full size, AFTER every headline number was taken (they cannot disturb it)
        ctx.destroy()
        del dbatch, batch
        per = {}
        for c in (1, 3, 4, 5):
            try:
                per[f"cfg{c}"] = time_config(S, W, torch, dev, local, c, None, args.ref_bases, W.SEED_BASE + c,
                                             steps=3, warmup=2, flush=flush, peak=peak)
            except Exception as ex:  # noqa: BLE001
                per[f"cfg{c}"] = {"error": repr(ex)}
        out["per_config"] = per
        # the lanes beside the int16 hot path, device-resident, same timing rules. `local`:
        # SDP_MODE_LOCAL on config 2's shape and on long reads; `int32_lane`: the default mode on
        # pairs outside the int16 kernels' domain (reads beyond SDP_MAX_READ_LEN), and for scale the
        # int16 path on the 600 bp x 2,000 bp shape. forward_frac / whole_path_frac stay relative to the int16x2 DPX
        # roofline of the headline, so that the distance of these lanes from the hot path is one number.
        def lane_block(name, make, **kw):
            try:
                return time_batch(S, torch, dev, local, make(), name, steps=3, warmup=2, flush=flush, peak=peak, **kw)
            except Exception as ex:  # noqa: BLE001
                return {"error": repr(ex)}

        out["local"] = {
            "cfg2_shape": lane_block(W_NAME[2] + ", SDP_MODE_LOCAL",
                                     lambda: W.make_config(2, ref_bases=args.ref_bases), local_mode=True),
            "long_reads": lane_block("50,000 pairs 600bp x 2,000bp (config 2's recipe at long-read lengths), SDP_MODE_LOCAL",
                                     lambda: W.make_long_reads(50_000, 600, 2000, ref_bases=args.ref_bases), local_mode=True)}
        out["int32_lane"] = {
            "reads_over_1024": lane_block("20,000 pairs 1,500bp x 3,000bp: reads beyond SDP_MAX_READ_LEN, one thread per "
                                          "pair with row arrays in global memory (k_forward_i32)",
                                          lambda: W.make_long_reads(20_000, 1500, 3000, ref_bases=args.ref_bases)),
            "int16_path_600x2000_for_scale": lane_block("50,000 pairs 600bp x 2,000bp on the int16 path (inside the range rule)",
                                                        lambda: W.make_long_reads(50_000, 600, 2000, ref_bases=args.ref_bases))}
        try:
            out["step3"] = time_step3(S, W, torch, dev, local, args.ref_bases, flush, peak)
        except Exception as ex:  # noqa: BLE001
            out["step3"] = {"error": repr(ex)}
    print(json.dumps(out))


if __name__ == "__main__":
    main()
