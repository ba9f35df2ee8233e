#!/usr/bin/env python
"""bench.py -- PairHMM forward throughput (GCUPS) of libpairhmm_b200.so on B200, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload short|long|mixed|verylong|tiny]
                    [--precision fp32|fp64] [--scale F] [--impl b200|reference]

A "step" is one pass of the whole hot path (host batcher, row-constant
prologue, short / long kernels, fp64 rescue, final log10) over one seeded synthetic batch, i.e. one
phmm_forward_batch call.  Default workload = BASELINE.json configs[1], the short-read region batch
the metric is quoted on (2,000 regions x 128 reads x 8 haplotypes = 2.05 M pairs, ~1.14e11 cells).

value      GCUPS = cells / time / 1e9 (TCUPS x 1000), payload resident in HBM, timed
           with CUDA events on the launching stream around exactly K calls, max over ranks.
e2e        same metric through the host entries: all buffers in pinned HOST memory, the host->device copies of the
           payload and the device->host copy of the results of every step inside the timed region (PAPER.md:346
           "with transfers").  value = the streaming entry (phmm_forward_batch_host_async, two calls in flight);
           sync_value = phmm_forward_batch_host, one synchronous call after the other.
roofline   dominant kernel (short: k_short_f32, long: k_long_f32, fp64: k_rescue_f64t / k_long_f64) against the FP32 (FP64)
           non-tensor peak; flops = 10 per cell; duration from the library's CUDA events.
cpu_baseline  the oracle (oracle/, as it stands) on the host cores on a bounded sample of the same batch.

Multi-GPU: the path does not shard (BASELINE.json north_star: one GPU).  --gpus N under torchrun
runs N independent replicas (rank r uses seed base+r), no data-path collective; value = total
cells / max-over-ranks time ("scaling": "weak").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

WORKLOADS = {  # name -> (BASELINE.json config index, description)
    "tiny": (0, "configs[0] tiny: 64 reads x 4 haplotypes, 256 pairs"),
    "short": (1, "configs[1] short-read region batch: 2000 regions x 128 reads x 8 haplotypes, all pairs"),
    "mixed": (2, "configs[2] mixed-length stream: 10M unsorted pairs, 5% unrelated reads"),
    "long": (3, "configs[3] long-read batch: 2000 pairs, reads 5-15 kbp"),
    "verylong": (4, "configs[4] very-long stress: 16 pairs of 100 kbp x 105 kbp"),
    "equal": (5, "paper's scalability-sweep shape (PAPER.md:366): read length = haplotype length = --len, noisy copies"),
}
L2_NOTE = ("no flush: the inputs of a step exceed L2 (payload plus the row-constant table, which is rewritten and re-read "
           "every step; 2.9 GB on the short-read batch, 1.3 GB on the long-read batch, 126 MB of L2)")
FLOPS_PER_CELL = 10.0  # SURVEY 8(d)'s algorithmic count (4 FMA + 2 MUL per cell); DESIGN.md section 7
FLOPS_PER_CELL_EXECUTED = {"fp32": 9.0, "fp64": 9.0}  # what the engines issue: 4 FMA + 1 MUL (the T/J form, in both precisions)


def _measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return {}


def _profiled_traffic(name, workload, scale):
    """DRAM bytes per launch of the dominant kernel from the committed `ncu --set full` capture of THIS kernel on THIS
    workload at THIS scale (profiles/traffic.json; DRAM counters cannot be read outside a profiler); None when the
    committed capture is of another workload or size -- nothing is scaled."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            e = json.load(f).get(name)
        if not e or e.get("workload") != workload or abs(float(e["scale"]) - float(scale)) > 1e-9:
            return None
        return float(e["dram_bytes_per_launch"])
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def make_batch(workload, scale, seed_offset, length=512):
    from paper_2606_25738_b200 import workloads
    cfg = WORKLOADS[workload][0]
    if cfg == 5:  # about 4e10 cells per launch, between 16 and 4M pairs
        n = int(min(4_000_000, max(16, round(4e10 * min(scale, 1.0) / float(length) ** 2))))
        return workloads.generate(5, seed=6 + seed_offset, n=n, len_lo=length), cfg
    full = {0: 0, 1: 2000, 2: 10_000_000, 3: 2000, 4: 16}[cfg]
    n = 0 if (scale >= 1.0 or cfg == 0) else max(1, int(round(full * scale)))
    return workloads.generate(cfg, seed=1 + cfg + seed_offset, n=n), cfg


def oracle_sample(batch, budget_s, rng_seed=12345):
    """Time the oracle on a bounded uniform sample of the batch's pairs (about budget_s of wall time)."""
    import oracle
    rng = np.random.default_rng(rng_seed)
    order = rng.permutation(batch.n_pairs)
    rl, hl = batch.read_len(), batch.hap_len()
    pc = rl[batch.pair_read].astype(np.int64) * hl[batch.pair_hap].astype(np.int64)
    cores = oracle.num_threads()
    # probe: enough pairs to give every thread work, at most ~2e8 cells
    n0 = int(min(batch.n_pairs, max(cores, np.searchsorted(np.cumsum(pc[order]), 2e8) + 1)))
    t = time.perf_counter(); oracle.forward_batch(batch, pairs=order[:n0]); dt0 = time.perf_counter() - t
    rate = pc[order[:n0]].sum() / max(dt0, 1e-6)
    want = rate * budget_s
    n1 = int(min(batch.n_pairs, max(n0, np.searchsorted(np.cumsum(pc[order]), want) + 1)))
    t = time.perf_counter(); oracle.forward_batch(batch, pairs=order[:n1]); dt = time.perf_counter() - t
    cells = int(pc[order[:n1]].sum())
    return {"cells": cells, "pairs": n1, "seconds": dt, "gcups": cells / dt / 1e9, "cores": cores}


def run_reference(args, rank, world):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    batch, cfg = make_batch(args.workload, args.scale, 0, args.len)
    budget = 6.0  # seconds of oracle work per step
    res = None
    for _ in range(args.warmup):
        oracle_sample(batch, 0.5)
    tot_cells, tot_s, tot_pairs = 0, 0.0, 0
    for s in range(args.steps):
        res = oracle_sample(batch, budget, rng_seed=1000 + s)
        tot_cells += res["cells"]; tot_s += res["seconds"]; tot_pairs += res["pairs"]
    v = tot_cells / tot_s / 1e9
    sample = "uniform random sample of %d pairs (%.3g cells) of the batch per step" % (tot_pairs // max(1, args.steps),
                                                                                      tot_cells / max(1, args.steps))
    print(json.dumps({
        "impl": "reference", "metric": "PairHMM forward throughput", "value": v, "unit": "GCUPS", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": tot_s / max(1, args.steps) * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.workload][1] + (" (len %d)" % args.len if cfg == 5 else ""),
                   "precision": "fp32 + fp64 rescue" if args.precision == "fp32" else "fp64",
                   "scale": args.scale, "pairs": int(batch.n_pairs), "cells": int(batch.cells()), "parallelism": "replicas x%d" % world,
                   "l2": L2_NOTE},
        "pairs_per_s": tot_pairs / tot_s,
        "cpu_baseline": {"value": v, "unit": "GCUPS", "cores": res["cores"], "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": "GCUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


def measure(args, workload, steps, rank, world, local, with_cpu):
    """One workload: K pipelined calls (the headline number), 5 individually timed calls (median / best), the end-to-end
    leg, the roofline of the dominant kernel and (rank 0, with_cpu) the oracle on a bounded sample."""
    import torch
    import torch.distributed as dist
    from paper_2606_25738_b200 import binding, replicas

    dev = "cuda:%d" % local
    batch, cfg = make_batch(workload, args.scale, replicas.rank_seed(0, rank), args.len)
    cells, n_pairs = batch.cells(), batch.n_pairs
    prec = binding.PHMM_FP32_RESCUE if args.precision == "fp32" else binding.PHMM_FP64
    ctx = binding.Context(local, profile_events=1)
    db = binding.DeviceBatch(batch, dev)
    out = torch.empty(n_pairs, dtype=torch.float64, device=dev)
    flags = torch.zeros(n_pairs, dtype=torch.uint8, device=dev)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        ctx.forward_batch(db, prec, out=out, flags=flags, sync=True)
    st = ctx.stats()

    # ---- timed region: exactly K calls, CUDA events on the launching stream, clocks sampled meanwhile
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
        time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(steps):
        # asynchronous: the host batcher (row a11) of call s+1 runs while the GPU works on call s
        ctx.forward_batch(db, prec, out=out, flags=flags, sync=False)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    s = ctx.stats()  # per-family CUDA-event durations of the last timed call
    fam = {k: s[k] for k in ("ms_table", "ms_short", "ms_rescue", "ms_long")}
    host_ms = s["host_batch_ms"]
    fam_samples = [dict(fam)]
    # ---- SURVEY 8(d) protocol: 5 calls timed one by one (host batcher inside, nothing to overlap with): median and best
    single = []
    for _ in range(5):
        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        t_host = time.perf_counter()
        a0.record()
        ctx.forward_batch(db, prec, out=out, flags=flags, sync=False)
        a1.record()
        torch.cuda.synchronize()
        single.append((a0.elapsed_time(a1), (time.perf_counter() - t_host) * 1e3))
        s1 = ctx.stats()
        fam_samples.append({k: s1[k] for k in fam})
    # kernel durations: CUDA events the library records around each kernel family, averaged over the last call of the timed
    # region and these five launches (same kernels, same inputs)
    fam = {k: sum(f[k] for f in fam_samples) / len(fam_samples) for k in fam}
    clocks = sampler.stop() if sampler else None
    ms, tot_cells, tot_pairs = replicas.aggregate(ms, cells, n_pairs, dist if world > 1 else None, dev)
    ms_step = ms / steps
    gcups = replicas.whole_job_gcups(ms, tot_cells, steps)
    wall = sorted(w for _, w in single)
    per_call = {"n": len(single), "median_ms": wall[len(wall) // 2], "best_ms": wall[0],
                "median_gcups": cells / (wall[len(wall) // 2] * 1e-3) / 1e9, "best_gcups": cells / (wall[0] * 1e-3) / 1e9,
                "timer": "host wall clock around one synchronised call of this rank (host batcher included, no overlap)"}

    # ---- end to end: host (pinned) buffers in, host results out, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        hb = [binding.HostBatch(batch), binding.HostBatch(batch)]  # two sets of pinned buffers: a stream of batches

        def wall_max(dt):
            if world > 1:
                t = torch.tensor([dt], dtype=torch.float64, device=dev)
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                dt = float(t.item())
            return dt

        for _ in range(2):
            ctx.forward_batch_host(hb[0], prec)
        # (1) one synchronous call after the other: nothing of step s+1 starts before the results of step s are on the host
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            ctx.forward_batch_host(hb[0], prec)
        torch.cuda.synchronize()
        dt_sync = wall_max(time.perf_counter() - t0)
        n_slices_sync = ctx.stats()["n_slices"]
        # (2) the streaming entry, two calls in flight: the copies in and the host plan of step s+1 run under the kernels of
        # step s; every step still copies its inputs in and its results out inside the timed region
        for i in range(2):
            ctx.wait_host(ctx.forward_batch_host_async(hb[i], prec))
        barrier()
        t0 = time.perf_counter()
        prev = None
        for i in range(steps):
            t = ctx.forward_batch_host_async(hb[i & 1], prec)
            if prev is not None:
                ctx.wait_host(prev)
            prev = t
        ctx.wait_host(prev)
        dt = wall_max(time.perf_counter() - t0)
        e2e = {"value": tot_cells / (dt / steps) / 1e9, "unit": "GCUPS",
               "h2d_bytes_per_step": int(hb[0].h2d_bytes()), "d2h_bytes_per_step": int(hb[0].d2h_bytes()),
               "ms_per_step": dt / steps * 1e3,
               "mode": "phmm_forward_batch_host_async / phmm_wait_host, two calls in flight, pinned host buffers",
               "timer": "host wall clock from the first submit to the last wait (results of every step on the host)",
               "sync_value": tot_cells / (dt_sync / steps) / 1e9, "sync_ms_per_step": dt_sync / steps * 1e3,
               "sync_slices": n_slices_sync,
               "sync_mode": "phmm_forward_batch_host, one synchronous call after the other"}
        del hb
    if rank != 0:
        return None

    # ---- roofline of the dominant kernel
    peaks = _measured_peaks()
    prop = torch.cuda.get_device_properties(local)
    sm_max = float(peaks.get("sm_max_mhz") or (clocks or {}).get("sm_max_mhz") or 1965.0)
    if args.precision == "fp32":
        lanes = 128  # FP32 FMA lanes per SM
        meas = binding.measure_peak(1, local)
    else:
        lanes = 64   # FP64 FMA lanes per SM (measured: DFMA at half the FFMA rate)
        meas = binding.measure_peak(2, local)
    peak = prop.multi_processor_count * lanes * 2 * sm_max * 1e6 / 1e12
    if st["n_long_pairs"] * 2 > st["n_pairs"]:
        kname = "k_long_f32" if args.precision == "fp32" else "k_long_f64"
        kms, kcells = fam["ms_long"], cells * 1.0
    elif args.precision == "fp64":
        kname, kms, kcells = "k_rescue_f64t<double> (+ chain fallback)", fam["ms_rescue"], cells * 1.0
    else:
        kname, kms, kcells = "k_short_f32", fam["ms_short"], float(st["short_cells"])
    achieved = FLOPS_PER_CELL * kcells / (kms * 1e-3) / 1e12 if kms > 0 else 0.0
    step_tflops = FLOPS_PER_CELL * tot_cells / world / (ms_step * 1e-3) / 1e12
    roofline = {"bound": "alu", "kernel": kname, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                "frac": achieved / peak, "traffic": _profiled_traffic(kname.split(" ")[0].split("<")[0], workload, args.scale),
                "peak_source": "nominal non-tensor %s peak = %d SMs x %d lanes x 2 x %.0f MHz (DESIGN.md); in-run FMA "
                               "microbenchmark measured %.2f TFLOP/s" % (args.precision.upper(), prop.multi_processor_count,
                                                                        lanes, sm_max, meas),
                "flops_per_cell": FLOPS_PER_CELL, "flops_per_cell_executed": FLOPS_PER_CELL_EXECUTED[args.precision],
                "frac_at_executed_flops": achieved / peak * FLOPS_PER_CELL_EXECUTED[args.precision] / FLOPS_PER_CELL,
                "whole_step_frac": step_tflops / peak,
                "whole_step_frac_at_executed_flops": step_tflops / peak * FLOPS_PER_CELL_EXECUTED[args.precision] / FLOPS_PER_CELL,
                "kernel_ms_per_launch": kms, "kernel_gcups": kcells / (kms * 1e-3) / 1e9 if kms > 0 else 0.0,
                "kernel_share_of_step": kms / ms_step if ms_step > 0 else None,
                "kernel_timer": "CUDA events recorded by the library around each kernel family on the launching stream; mean of "
                                "%d launches (the last call of the timed region and the individually timed calls)" % len(fam_samples),
                "hbm_gbs_achieved": None, "family_ms": fam, "host_batch_ms": host_ms}
    if roofline["traffic"] and kms > 0:  # DRAM bytes of the committed ncu capture of this very workload and scale / this run's kernel time
        roofline["hbm_gbs_achieved"] = roofline["traffic"] / (kms * 1e-3) / 1e9
        roofline["hbm_frac_of_measured_peak"] = roofline["hbm_gbs_achieved"] / float(peaks.get("hbm_gbs") or 6471.1)

    cpu = None
    if with_cpu:
        r = oracle_sample(batch, 15.0)
        cpu = {"value": r["gcups"], "unit": "GCUPS", "cores": r["cores"], "kind": "oracle",
               "sample": "uniform random sample of %d pairs (%.3g cells) of the same batch, %.1f s; the --impl reference arm "
                         "times other samples of the same batch (6 s each)" % (r["pairs"], r["cells"], r["seconds"])}
    ctx.close()
    return {
        "value": gcups, "unit": "GCUPS", "steps": steps, "ms_per_step": ms_step,
        "config": {"workload": WORKLOADS[workload][1] + (" (len %d)" % args.len if cfg == 5 else ""),
                   "precision": "fp32 + fp64 rescue" if args.precision == "fp32" else "fp64",
                   "scale": args.scale, "pairs": int(tot_pairs), "cells": int(tot_cells), "parallelism": "replicas x%d" % world,
                   "l2": L2_NOTE},
        "pairs_per_s": tot_pairs / (ms_step * 1e-3), "per_call": per_call,
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(st["n_kernel_launches"]) * steps,
        "roofline": roofline, "cpu_baseline": cpu,
        "stats": {k: st[k] for k in ("n_short_pairs", "n_long_pairs", "n_rescued", "short_cells", "short_padded_cells", "n_short_warps",
                                     "n_slices", "table_bytes")},
    }

def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="short", choices=sorted(WORKLOADS))
    ap.add_argument("--precision", default="fp32", choices=["fp32", "fp64"])
    ap.add_argument("--scale", type=float, default=1.0, help="fraction of the workload's full size")
    ap.add_argument("--len", type=int, default=512, help="--workload equal: read length = haplotype length")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-secondary", action="store_true",
                    help="default run (short-read batch, full size): do not also measure the long-read target batch configs[3]")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda:%d" % local))

    head = measure(args, args.workload, args.steps, rank, world, local, with_cpu=not args.no_cpu_baseline)
    # north_star names two target batches: the short-read batch (the headline, configs[1]) and the 10k-bp long-read
    # batch (configs[3]); the default run measures both, the second one in `secondary` with the same keys
    secondary = []
    if args.workload == "short" and args.scale >= 1.0 and args.precision == "fp32" and not args.no_secondary:
        sec = measure(args, "long", max(3, min(args.steps, 5)), rank, world, local, with_cpu=False)
        if sec is not None:
            secondary.append(sec)
    if rank == 0:
        line = {"metric": "PairHMM forward throughput", "value": head["value"], "unit": "GCUPS", "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": head["ms_per_step"], "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32" if args.precision == "fp32" else "f64",
                "data": "synthetic"}
        for k in ("config", "pairs_per_s", "per_call", "clocks", "e2e", "roofline", "cpu_baseline", "stats"):
            line[k] = head[k]
        line["gpu_launches"] = head["gpu_launches"] + sum(x["gpu_launches"] for x in secondary)
        line["secondary"] = secondary
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
