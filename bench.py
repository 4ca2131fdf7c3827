#!/usr/bin/env python
"""bench.py -- throughput of the ground-state charge search on the headline workload (BASELINE.json configs[3]:
open 4x4 grid of 16 dots, default algorithm, 100x100 pixels, 2^16 candidates per pixel, fp64).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
                    [--workload config4|config5|small|thermal|closed16|sweep] [--no-parity] [--no-secondary]

The default run (config4) prints ONE JSON line: the headline, its roofline, the oracle baseline, the end-to-end number, the
opt-in walk variants, the full-size parity report of all five BASELINE.json configs ("parity") and the other workloads
("secondary": config5, small, closed16, thermal, sweep).  --workload X prints the line of that workload alone.

One "step" = one pass of the whole hot path (prologue -> candidate walk -> finalize) over
one 100x100 diagram.  Prints ONE JSON line (rank 0).  Multi-GPU: one process per GPU (torchrun), every rank runs its own
diagram (pixels are independent: no data-path collective), value = total candidates / max-over-ranks time ("weak").

--impl reference times the ORACLE (oracle/, plain single-threaded C written from the paper) on the host cores, on a
bounded sample of the same workload per step.  It is a deliberately slow program: a reported baseline, not the target.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "candidate configs scored/s (16 dots, default algorithm, open 4x4 grid, 100x100 pixels)"
UNIT = "candidates/s"
FP64_OPS_PER_CANDIDATE = 312.0 / 256.0   # FP64-pipe instructions per candidate of the min-plus walk
WALK_DRAM_BYTES_NCU = 1632768           # dram__bytes_read + dram__bytes_write per launch, from the ncu capture named below
WALK_DRAM_SOURCE = "profiles/r02_headline_ncu_full.md"
THERMAL_FP64_OPS_PER_CANDIDATE = {"qa_thermal_sp_kernel": 3.0}  # 2 DFMA (rows, columns) + 1 DADD (lower bound of the E_min pass)
FP64_LANES_PER_SM = 64         # 148 SMs x 64 FP64 lanes x SM clock


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config4", choices=["config4", "config5", "small", "thermal", "closed16", "sweep"])
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing leg (profiling runs)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--arrays", type=int, default=256, help="config5: arrays of the dataset batch per GPU")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the oracle sample")
    ap.add_argument("--no-parity", action="store_true", help="skip the full-size parity report (profiling runs)")
    ap.add_argument("--no-secondary", action="store_true", help="skip the secondary workloads of the default run")
    ap.add_argument("--parity-members", type=int, default=256, help="config-5 members compared with the oracle")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.rows, self.proc, self.idx = [], None, gpu_index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.idx), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm = [float(r[1]) for r in self.rows if len(r) >= 9 and r[1].replace(".", "").isdigit()]
        mx = [float(r[2]) for r in self.rows if len(r) >= 9 and r[2].replace(".", "").isdigit()]
        reasons = set()
        for r in self.rows:
            if len(r) < 9:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def make_workloads(name, rank):
    from paper_2404_04994_b200 import workloads as wl
    if name == "config4":
        return [wl.config4(100, 100, seed=3 + 100 * rank)]          # rank r > 0: an independently seeded diagram
    return [wl.config5_array(j + 256 * rank) for j in range(8)]     # a slice of the dataset batch (secondary bench)


def candidates_of(wls, alg="default"):
    return sum(w.P * (2 ** w.n_dot) for w in wls)


# ---------------------------------------------------------------------------------------------------------------------
def run_reference(args, rank):
    """The oracle as the reference arm (this tier has no reference implementation): rank 0 only."""
    if rank != 0:
        return
    import oracle
    from paper_2404_04994_b200 import workloads as wl
    w = wl.config4(100, 100)
    m = oracle.Model(w.C_dd, w.C_gd)
    t0 = time.perf_counter()
    m.ground_state(w.Vg[:8])
    per_px = (time.perf_counter() - t0) / 8
    total_budget = 150.0
    px = int(max(4, min(400, total_budget / max(1, args.steps + args.warmup) / per_px)))
    rng = np.random.default_rng(0)
    sel = np.sort(rng.choice(w.P, size=px, replace=False))
    for _ in range(args.warmup):
        m.ground_state(w.Vg[sel])
    t0 = time.perf_counter()
    for _ in range(args.steps):
        m.ground_state(w.Vg[sel])
    dt = (time.perf_counter() - t0) / args.steps
    val = px * 65536 / dt
    sample = f"{px} of 10000 pixels (seeded random subset) of config4 per step, single thread"
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[3]: open 4x4 grid, 16 dots, default, 100x100 (sampled)",
                       "sample": sample},
            "pixels_per_s": px / dt,
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def cpu_baseline(args):
    import oracle
    from paper_2404_04994_b200 import workloads as wl
    w = wl.config4(100, 100)
    m = oracle.Model(w.C_dd, w.C_gd)
    t0 = time.perf_counter()
    m.ground_state(w.Vg[:8])
    per_px = (time.perf_counter() - t0) / 8
    px = int(max(8, min(1000, args.cpu_seconds / per_px)))
    rng = np.random.default_rng(0)
    sel = np.sort(rng.choice(w.P, size=px, replace=False))
    t0 = time.perf_counter()
    m.ground_state(w.Vg[sel])
    dt = time.perf_counter() - t0
    out = {"value": px * 65536 / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": f"{px} of 10000 pixels (seeded random subset) of config4, {dt:.1f} s",
           "pixels_per_s": px / dt, "host_cores": os.cpu_count()}
    if oracle.has_openmp() and (os.cpu_count() or 1) > 1:
        nt = os.cpu_count()
        px2 = int(min(4000, px * max(1, nt // 2)))
        sel2 = np.sort(rng.choice(w.P, size=px2, replace=False))
        t0 = time.perf_counter()
        m.ground_state(w.Vg[sel2], n_threads=nt)
        dt2 = time.perf_counter() - t0
        out["all_cores"] = {"value": px2 * 65536 / dt2, "unit": UNIT, "cores": nt,
                            "sample": f"{px2} pixels, OpenMP over pixels, {dt2:.1f} s"}
    return out


# ---------------------------------------------------------------------------------------------------------------------
def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2404_04994_b200 import api

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    wls = make_workloads(args.workload, rank)
    models = [api.Model(w.C_dd, w.C_gd) for w in wls]
    Vgs = [torch.from_numpy(w.Vg).to(dev) for w in wls]
    outs = [{"N": torch.empty((w.P, w.n_dot), dtype=torch.int32, device=dev),
             "E": torch.empty(w.P, dtype=torch.float64, device=dev)} for w in wls]
    cand_step = candidates_of(wls)
    px_step = sum(w.P for w in wls)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def step():
        for m, v, o in zip(models, Vgs, outs):
            m.ground_state(v, out=o)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        flush.fill_(1)
        step()
    launches_per_step = api.last_launch_plan()[1] * len(models)
    plan = api.last_launch_plan()[0]

    # ---- timed region: K steps, CUDA events around each step on the launching stream, L2 flushed between steps ----
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    for k in range(args.steps):
        flush.fill_(k & 0xff)
        ev[k][0].record()
        step()
        ev[k][1].record()
    barrier()
    clocks = sampler.stop()
    times = np.array([a.elapsed_time(b) for a, b in ev])            # ms
    tot_ms = float(times.sum())
    if world > 1:
        t = torch.tensor([tot_ms], device=dev, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        tot_ms = float(t.item())
    ms_per_step = tot_ms / args.steps
    value = world * cand_step / (ms_per_step * 1e-3)

    if rank != 0:
        return

    # ---- opt-in variants, reported beside the headline, never instead of it: exact pruning (qa_model_set_walk_variant(2):
    # same charge maps, fewer candidates scored explicitly) and the mixed-precision walk (variant 3: every candidate bounded
    # from below in fp32 with directed rounding, the survivors re-scored in fp64: bit-identical N and E)
    def time_variant(variant, note):
        for m_ in models:
            m_.set_walk_variant(variant)
        try:
            for _ in range(3):
                step()
            evp = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
            for k in range(args.steps):
                flush.fill_(k & 0xff)
                evp[k][0].record()
                step()
                evp[k][1].record()
            torch.cuda.synchronize()
            tp = np.array([a.elapsed_time(b) for a, b in evp])
            ktp = api.kernel_times(models[0], Vgs[0], steps=args.steps, flush=flush)
            return {"ms_per_step": float(tp.mean()), "ms_per_step_median": float(np.median(tp)),
                    "candidates_covered_per_s": cand_step / (float(tp.mean()) * 1e-3), "kernel_times_ms": ktp, "note": note}
        finally:
            for m_ in models:
                m_.set_walk_variant(1)

    pruned = mixed = one_kernel = None
    if args.workload == "config4":
        pruned = time_variant(2, "qa_model_set_walk_variant(2): high patterns excluded by a rigorous lower bound are not walked; "
                                 "identical N and E (tests/test_gpu_parity.py)")
        mixed = time_variant(3, "qa_model_set_walk_variant(3): pass 1 bounds every candidate from below in fp32 (directed rounding), "
                                "pass 2 re-scores the survivors in fp64: N and E bit-identical to the fp64 walk")
        one_kernel = time_variant(4, "qa_model_set_walk_variant(4): S1-S7 in one persistent kernel, no workspace traffic (DESIGN.md "
                                     "section 5.4b); N, E and x bit-identical to the three launches")
        kw32 = mixed["kernel_times_ms"].get("qa_minplus_walk32_kernel", 0.0)
        if kw32 > 0:
            sm_count_ = torch.cuda.get_device_properties(dev).multi_processor_count
            peak32 = sm_count_ * 128 * 1965.0e6
            ops32 = 1.5 * wls[0].P * (2 ** wls[0].n_dot)       # 1 FADD + 1/2 VIMNMX3 per candidate
            mixed["roofline"] = {"bound": "alu", "kernel": "qa_minplus_walk32_kernel", "achieved": ops32 / (kw32 * 1e-3) / 1e9,
                                 "peak": peak32 / 1e9, "unit": "FP32/INT32 Ginst/s", "frac": ops32 / (kw32 * 1e-3) / peak32,
                                 "ops_per_candidate": 1.5,
                                 "peak_source": f"derived: {sm_count_} SMs x 128 FP32 lanes x 1965 MHz (DESIGN.md section 6)"}

    # ---- per-kernel share of the step: CUDA events between the kernels (separate pass, same launch configuration) --
    kt = api.kernel_times(models[0], Vgs[0], steps=args.steps, flush=flush)
    hot = "qa_minplus_walk_kernel" if "qa_minplus_walk_kernel" in kt else "qa_walk_kernel"
    ops_per_cand = FP64_OPS_PER_CANDIDATE if hot == "qa_minplus_walk_kernel" else 3.0
    walk_ms = kt.get(hot, 0.0)                                     # pass 1 only; the finish kernel is listed beside it
    sm_count = torch.cuda.get_device_properties(dev).multi_processor_count
    sm_max_mhz = clocks.get("sm_max_mhz") or 1965.0
    peak_nominal = sm_count * FP64_LANES_PER_SM * sm_max_mhz * 1e6           # FP64 thread-inst/s
    peak_measured = api.measure_fp64_rate(1.0)
    alg_ops = ops_per_cand * wls[0].P * (2 ** wls[0].n_dot)
    achieved = alg_ops / (walk_ms * 1e-3) if walk_ms > 0 else 0.0
    roofline = {"bound": "alu", "kernel": hot, "achieved": achieved / 1e9, "peak": peak_nominal / 1e9,
                "unit": "FP64 Ginst/s", "frac": achieved / peak_nominal,
                "traffic": WALK_DRAM_BYTES_NCU if hot == "qa_minplus_walk_kernel" else None,
                "traffic_unit": "bytes/launch (dram__bytes_read.sum + dram__bytes_write.sum)",
                "traffic_source": "ncu --set full capture of this kernel, " + WALK_DRAM_SOURCE + " (not measured by this run)",
                "peak_source": f"derived: {sm_count} SMs x {FP64_LANES_PER_SM} FP64 lanes x {sm_max_mhz:.0f} MHz "
                               "(DESIGN.md); MEASURED_PEAKS.json has no FP64 figure",
                "peak_measured_dfma_probe": peak_measured / 1e9, "frac_of_measured_probe": achieved / peak_measured,
                "fp64_ops_per_candidate": ops_per_cand, "kernel_ms": walk_ms,
                "kernel_share_of_step": walk_ms / max(1e-9, sum(kt.values())), "kernel_times_ms": kt,
                "gflops_equiv_dadd": achieved / 1e9}

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D + search + D2H inside the timed region --------
    e2e = None
    if not args.no_e2e:
        hv = [torch.from_numpy(w.Vg).pin_memory() for w in wls]
        ho = [{"N": torch.empty((w.P, w.n_dot), dtype=torch.int32).pin_memory(),
               "E": torch.empty(w.P, dtype=torch.float64).pin_memory()} for w in wls]
        for _ in range(3):
            for m, v, o in zip(models, hv, ho):
                m.ground_state_host(v, out=o)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            for m, v, o in zip(models, hv, ho):
                m.ground_state_host(v, out=o)
        torch.cuda.synchronize()
        dt = (time.perf_counter() - t0) / args.steps
        e2e = {"value": cand_step / dt, "unit": UNIT, "ms_per_step": dt * 1e3,
               "h2d_bytes_per_step": int(sum(v.numel() * 8 for v in hv)),
               "d2h_bytes_per_step": int(sum(o["N"].numel() * 4 + o["E"].numel() * 8 for o in ho)),
               "api": "qa_ground_state_host (pinned host buffers)", "n_gpus_measured": 1}

    cpu = None
    if not args.no_cpu_baseline:
        try:
            cpu = cpu_baseline(args)
        except Exception as e:
            cpu = {"error": f"{type(e).__name__}: {e}"}
    del flush, Vgs, outs
    # (N > 1: the other ranks are waiting at the final barrier; the report and the secondary workloads are in the N = 1 line)
    parity = None
    if not (args.no_parity or world > 1):
        try:
            parity = parity_report(args)
        except Exception as e:  # the report must never cost the headline line; an error here reads as "no parity claim"
            parity = {"error": f"{type(e).__name__}: {e}"}
    secondary = None if (args.no_secondary or world > 1) else secondary_workloads(args, local_rank)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[3]: open 4x4 grid, 16 dots, default algorithm, 100x100 pixels, "
                                   "2^16 candidates/pixel, seed 3" if args.workload == "config4" else
                                   "BASELINE.json configs[4] slice: 8 open 8-dot arrays, 128x128, default",
                       "pixels_per_step_per_gpu": px_step, "candidates_per_step_per_gpu": cand_step,
                       "l2": "flushed (256 MiB write) between timed steps", "parallelism": f"pixel-range x{world}"},
            "pixels_per_s": world * px_step / (ms_per_step * 1e-3), "diagram_ms": ms_per_step,
            "ms_per_step_min": float(times.min()), "ms_per_step_median": float(np.median(times)),
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches_per_step * args.steps,
            "kernels_per_step": plan, "clocks": clocks, "pruned_variant": pruned, "mixed_precision_variant": mixed, "one_kernel_variant": one_kernel,
            "parity": parity, "secondary": secondary,
            "paper_context": "paper: same diagram shape in < 1 s on a GTX 1080 Ti via JAX (PAPER.md L7, L498)"}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------------------
def run_config5(args, rank, world, local_rank, steps=None, emit=True):
    """Secondary workload (BASELINE.json configs[4]): the dataset batch of independently seeded open 8-dot arrays, each a
    128x128 sweep, with the default algorithm and the thresholded one at t = 0.2 and 0.5.  One step = every array with
    all three algorithms, through qa_ground_state_batch (semantically a loop over the single-model call, one launch of
    the one-kernel path per algorithm).  Reports pixels/s over the whole batch and the agreement rate of thresholded vs
    default (fraction of pixels with identical N)."""
    import torch
    import torch.distributed as dist
    from paper_2404_04994_b200 import api, workloads as wl

    steps = steps or args.steps
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    B = args.arrays
    wls = [wl.config5_array(j + B * rank) for j in range(B)]
    models = [api.Model(w.C_dd, w.C_gd) for w in wls]
    batch = api.Batch(models)                                    # qa_batch_create: one launch per algorithm
    Vg = torch.from_numpy(np.stack([w.Vg for w in wls])).to(dev)  # [B, P, g]
    algs = (("default", dict(algorithm="default")), ("t0.2", dict(algorithm="thresholded", t=0.2)),
            ("t0.5", dict(algorithm="thresholded", t=0.5)))
    P, n = wls[0].P, wls[0].n_dot
    outs = {a: {"N": torch.empty((B, P, n), dtype=torch.int32, device=dev),
                "E": torch.empty((B, P), dtype=torch.float64, device=dev)} for a, _ in algs}
    px_step = B * P * len(algs)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    multi_spec = [("default", None), ("thresholded", 0.2), ("thresholded", 0.5)]
    multi_out = [outs[a] for a, _ in algs]

    def step():
        for a, kw in algs:
            batch.ground_state(Vg, out=outs[a], **kw)

    def step_multi():   # qa_ground_state_batch_multi: the three algorithms in one launch (V_g, N_c and the QP once per pixel)
        batch.ground_state_multi(Vg, multi_spec, out=multi_out)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(3, args.warmup)):
        flush.fill_(1)
        step()
    launches_per_step = api.last_launch_plan()[1] * len(algs)
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for k in range(steps):
        flush.fill_(k & 0xff)
        ev[k][0].record()
        step()
        ev[k][1].record()
    barrier()
    clocks = sampler.stop()
    times = np.array([a.elapsed_time(b) for a, b in ev])
    tot_ms = float(times.sum())
    if world > 1:
        tt = torch.tensor([tot_ms], device=dev, dtype=torch.float64)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        tot_ms = float(tt.item())
    ms_per_step = tot_ms / steps
    # the same work through qa_ground_state_batch_multi (one launch for the three algorithms), for comparison
    for _ in range(3):
        step_multi()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for k in range(steps):
        flush.fill_(k & 0xff)
        evs[k][0].record()
        step_multi()
        evs[k][1].record()
    torch.cuda.synchronize()
    ms_multi = float(np.mean([a.elapsed_time(b) for a, b in evs]))
    if rank != 0:
        return None
    agree = {}
    for a in ("t0.2", "t0.5"):
        same = int((outs[a]["N"] == outs["default"]["N"]).all(dim=2).sum())
        agree[a] = same / (B * P)
    n, g = wls[0].n_dot, wls[0].n_gate
    bytes_px = 8 * g + 4 * n + 8                       # V_g in, N and E out
    hbm = None
    try:
        hbm = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        pass
    peak = hbm or 6516.0
    achieved = px_step * bytes_px / (ms_per_step * 1e-3) / 1e9
    line = {"metric": "pixels/s over the dataset batch (open 8-dot arrays, 128x128, default + thresholded t=0.2, 0.5)",
            "value": world * px_step / (ms_per_step * 1e-3), "unit": "pixels/s", "n_gpus": world, "steps": steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[4]: {B} open 8-dot arrays (seeds 1000+j), 128x128 each, "
                                   "default + thresholded t=0.2 + t=0.5", "arrays_per_gpu": B,
                       "api": "qa_ground_state_batch: one launch per algorithm over all arrays",
                       "pixels_per_step_per_gpu": px_step, "l2": "flushed (256 MiB write) between timed steps",
                       "parallelism": f"array-range x{world}"},
            "agreement_with_default": agree,
            "one_launch": {"ms_per_step": ms_multi, "pixels_per_s": world * px_step / (ms_multi * 1e-3),
                           "api": "qa_ground_state_batch_multi: the three algorithms in ONE launch (V_g, N_c and the QP once per "
                                  "pixel; results bit-identical; measured 5 % slower than three launches on B200: DESIGN.md 5.5)",
                           "algorithmic_bytes_per_step": B * P * (8 * g + len(algs) * (4 * n + 8))},
            "roofline": {"bound": "hbm", "kernel": "qa_fused_open_kernel (whole step: 3 launches)",
                         "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                         "bytes_per_pixel": bytes_px, "algorithmic_bytes_per_step": px_step * bytes_px,
                         "traffic_source": "not measured by this run; ncu figure in profiles/r02_config5_ncu.md",
                         "peak_source": "MEASURED_PEAKS.json hbm_gbs" if hbm else "fallback 6516 GB/s (SURVEY.md)"},
            "cpu_baseline": None, "e2e": None, "gpu_launches": launches_per_step * steps, "clocks": clocks}
    line["ms_per_step_median"] = float(np.median(times))
    del Vg, outs, flush
    if emit:
        print(json.dumps(line), flush=True)
    return line


# ---------------------------------------------------------------------------------------------------------------------
def run_small(args, rank, steps=None, emit=True):
    """BASELINE.json configs[0..2] (launch-latency-bound diagrams: 10^4 - 4*10^4 pixels, <= 7776 candidates per pixel):
    device time of one diagram per (config, algorithm), CUDA events, L2 flushed between repetitions.  One JSON line."""
    if rank != 0:
        return None
    steps = steps or args.steps
    import torch
    from paper_2404_04994_b200 import api, workloads as wl
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    cases = [("config1 open double dot 100x100", wl.config1(100, 100), [dict(algorithm="default"), dict(algorithm="brute", n_max=5)]),
             ("config2 closed 5-chain N=5 100x100", wl.config2(100, 100), [dict(algorithm="default"), dict(algorithm="brute", n_max=5)]),
             ("config3 open 2x2 + sensor 200x200", wl.config3(200, 200), [dict(algorithm="default")])]
    rows = []
    for name, w, kws in cases:
        m = api.Model(w.C_dd, w.C_gd, sensor_dots=w.sensor_dots)
        Vg = torch.from_numpy(w.Vg).to(dev)
        for kw in kws:
            for _ in range(max(3, args.warmup)):
                m.ground_state(Vg, regime=w.regime, N_hat=w.N_hat, **kw)
            ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
            for k in range(steps):
                flush.fill_(k & 0xff)
                ev[k][0].record()
                r = m.ground_state(Vg, regime=w.regime, N_hat=w.N_hat, want_stats=(k == 0), **kw)
                ev[k][1].record()
                if k == 0:
                    st = r["stats"]
            torch.cuda.synchronize()
            t = np.array([a.elapsed_time(b) for a, b in ev[1:]])
            sd = api.stats_dict(st)
            rows.append({"config": name, "algorithm": kw["algorithm"], "pixels": w.P, "ms_median": float(np.median(t)),
                         "ms_min": float(t.min()), "pixels_per_s": w.P / (float(np.median(t)) * 1e-3),
                         "candidates_enumerated": sd["n_candidates_enumerated"], "candidates_scored": sd["n_candidates_scored"],
                         "qp_pixels": sd["n_qp_pixels"], "kernels": api.last_launch_plan()[0]})
    line = {"metric": "device time per diagram, BASELINE.json configs[0..2]", "unit": "ms", "n_gpus": 1,
            "steps": steps, "warmup": args.warmup, "dtype": "f64", "data": "synthetic",
            "l2": "flushed (256 MiB write) between repetitions", "rows": rows}
    if emit:
        print(json.dumps(line), flush=True)
    return line


# ---------------------------------------------------------------------------------------------------------------------
def _time_calls(torch, fn, steps, warmup, flush):
    """Median / min / mean device time (ms) of fn() over `steps` repetitions, CUDA events, L2 flushed in between."""
    for _ in range(max(3, warmup)):
        fn()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for k in range(steps):
        flush.fill_(k & 0xff)
        ev[k][0].record()
        fn()
        ev[k][1].record()
    torch.cuda.synchronize()
    t = np.array([a.elapsed_time(b) for a, b in ev])
    return float(np.median(t)), float(t.min()), float(t.mean())


def _fp64_peak(torch, dev=0):
    return torch.cuda.get_device_properties(dev).multi_processor_count * FP64_LANES_PER_SM * 1965.0e6


def run_thermal(args, rank, steps=None, emit=True):
    """thermal broadening (Eq. (10)) on the config-4 diagram (16 dots, 100x100, default set: 2^16
    Boltzmann weights per pixel), kT = 0.05 E_C.  Device time per diagram (CUDA events, L2 flushed) and the oracle on one
    host core on a bounded sample.  One JSON line."""
    if rank != 0:
        return None
    steps = steps or args.steps
    import torch
    import oracle
    from paper_2404_04994_b200 import api, workloads as wl
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    w = wl.config4(100, 100)
    m = api.Model(w.C_dd, w.C_gd)
    _, EC = m.inverse()
    kT = 0.05 * EC
    Vg = torch.from_numpy(w.Vg).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ms, ms_min, _ = _time_calls(torch, lambda: m.thermal(Vg, kT), steps, args.warmup, flush)
    r = m.thermal(Vg, kT)
    plan = api.last_launch_plan()[0]
    kt = api.kernel_times(m, Vg, steps=min(steps, 5), flush=flush, call="thermal", kT=kT)
    torch.cuda.synchronize()
    om = oracle.Model(w.C_dd, w.C_gd)
    sel = np.sort(np.random.default_rng(0).choice(w.P, size=40, replace=False))
    t0 = time.perf_counter()
    o = om.thermal(w.Vg[sel], kT)
    dt = time.perf_counter() - t0
    err = float(np.abs(r["Nmean"].cpu().numpy()[sel] - o["Nmean"]).max())
    hot = max(kt, key=kt.get) if kt else None
    ops = THERMAL_FP64_OPS_PER_CANDIDATE.get(hot.split("<")[0], None) if hot else None
    roof = None
    if ops:
        ach = ops * w.P * 65536 / (kt[hot] * 1e-3)
        roof = {"bound": "alu", "kernel": hot, "achieved": ach / 1e9, "peak": _fp64_peak(torch) / 1e9, "unit": "FP64 Ginst/s",
                "frac": ach / _fp64_peak(torch), "fp64_ops_per_candidate": ops, "kernel_ms": kt[hot], "kernel_times_ms": kt,
                "traffic": None, "peak_source": "derived: SMs x 64 FP64 lanes x 1965 MHz (DESIGN.md section 6)"}
    line = {"metric": "Boltzmann-weighted candidate configs/s (thermal broadening, 16 dots, default set, 100x100)",
            "value": w.P * 65536 / (ms * 1e-3), "unit": "candidates/s", "n_gpus": 1, "steps": steps,
            "warmup": args.warmup, "ms_per_step": ms, "ms_per_step_min": ms_min, "higher_is_better": True,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[3] with Eq. (10), kT = 0.05 E_C", "kT": kT,
                       "l2": "flushed (256 MiB write) between timed steps"},
            "kernels_per_step": plan, "roofline": roof, "max_abs_err_vs_oracle_sample": err,
            "cpu_baseline": {"value": len(sel) * 65536 / dt, "unit": "candidates/s", "cores": 1, "kind": "oracle",
                             "sample": f"{len(sel)} of 10000 pixels (seeded random subset), {dt:.1f} s"}}
    if emit:
        print(json.dumps(line), flush=True)
    return line


# ---------------------------------------------------------------------------------------------------------------------
def run_closed16(args, rank, steps=None, emit=True):
    """SURVEY 8(f) NEXT-3, the paper's second headline shape (Fig. 4(b)): CLOSED array of 16 dots with
    N_hat = n_dot = 16, default algorithm, 100x100 pixels, on the config-4 model and sweep.  Only the C(16, k) floor/ceil
    states with the right total are scored (k = N_hat - sum floor(x) per pixel).  Reports candidates SCORED/s, the time
    per diagram, and every pixel against the oracle (OpenMP)."""
    if rank != 0:
        return None
    steps = steps or args.steps
    import torch
    import oracle
    from paper_2404_04994_b200 import api, workloads as wl
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from parity import compare
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    w = wl.config4(100, 100)
    n = w.n_dot
    m = api.Model(w.C_dd, w.C_gd)
    Vg = torch.from_numpy(w.Vg).to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    kw = dict(regime="closed", N_hat=n)
    ms, ms_min, _ = _time_calls(torch, lambda: m.ground_state(Vg, **kw), steps, args.warmup, flush)
    r = m.ground_state(Vg, want_xcont=True, want_stats=True, **kw)
    plan = api.last_launch_plan()[0]
    kt = api.kernel_times(m, Vg, steps=min(steps, 10), flush=flush, **kw)
    torch.cuda.synchronize()
    st = api.stats_dict(r["stats"])
    om = oracle.Model(w.C_dd, w.C_gd)
    t0 = time.perf_counter()
    o = om.ground_state(w.Vg, n_threads=os.cpu_count(), **kw)
    dt = time.perf_counter() - t0
    rep = compare(r["N"].cpu().numpy(), r["E"].cpu().numpy(), o, om.EC, gpu_x=r["xcont"].cpu().numpy(), strict=False)
    # the generic odometer (all 2^16 states visited, filtered on the total) on the same diagram, for reference
    m0 = api.Model(w.C_dd, w.C_gd, walk_variant=0)
    ms0, _, _ = _time_calls(torch, lambda: m0.ground_state(Vg, **kw), max(3, steps // 4), 3, flush)
    hot = max(kt, key=kt.get) if kt else None
    line = {"metric": "candidate configs scored/s (closed array, 16 dots, N_hat = 16, default algorithm, 100x100 pixels)",
            "value": st["n_candidates_scored"] / (ms * 1e-3), "unit": "candidates/s", "n_gpus": 1, "steps": steps,
            "warmup": args.warmup, "ms_per_step": ms, "ms_per_step_min": ms_min, "higher_is_better": True, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[3] model and sweep, closed with N_hat = 16 (PAPER.md L496)",
                       "l2": "flushed (256 MiB write) between timed steps"},
            "pixels_per_s": w.P / (ms * 1e-3), "candidates_scored_per_step": st["n_candidates_scored"],
            "candidates_enumerated_per_step": st["n_candidates_enumerated"], "qp_pixels": st["n_qp_pixels"],
            "kernels_per_step": plan, "kernel_times_ms": kt, "hot_kernel": hot,
            "generic_odometer_ms_per_step": ms0, "speedup_over_generic_odometer": ms0 / ms,
            "parity": rep,
            "cpu_baseline": {"value": int(o["n_scored"].sum()) / dt, "unit": "candidates/s", "cores": os.cpu_count(),
                             "kind": "oracle", "sample": f"the whole diagram, OpenMP over pixels, {dt:.1f} s"},
            "paper_context": "paper: closed 16-dot 100x100 diagram in < 1 s (PAPER.md L7, L498)"}
    if emit:
        print(json.dumps(line), flush=True)
    return line


# ---------------------------------------------------------------------------------------------------------------------
def run_sweep(args, rank, steps=None, emit=True):
    """the SHAPE of the paper's Fig. 4(a)/(b): device time of a 100x100 diagram
    of a random Maxwell array for n_dot = 2..16, default algorithm, open and closed (N_hat = n_dot), random C and V_g as
    L490, with the oracle's time per pixel (one core, bounded sample) beside it."""
    if rank != 0:
        return None
    steps = steps or args.steps
    import torch
    import oracle
    from paper_2404_04994_b200 import api, workloads as wl
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    rows = []
    for n in range(2, 17):
        w = wl.random_open(n, n, 10000, seed=4000 + n, lo=-0.3, hi=2.5)
        m = api.Model(w.C_dd, w.C_gd)
        Vg = torch.from_numpy(w.Vg).to(dev)
        om = oracle.Model(w.C_dd, w.C_gd)
        px = max(4, min(2000, int(2.0e6 / (2 ** n))))
        row = {"n_dot": n}
        for regime, kw in (("open", dict()), ("closed", dict(regime="closed", N_hat=n))):
            med, mn, _ = _time_calls(torch, lambda: m.ground_state(Vg, **kw), steps, 3, flush)
            plan = api.last_launch_plan()[0]
            t0 = time.perf_counter()
            om.ground_state(w.Vg[:px], **kw)
            dt = (time.perf_counter() - t0) / px
            row[regime] = {"ms_per_diagram": med, "ms_min": mn, "kernels": plan,
                           "oracle_ms_per_diagram_1core_extrapolated": dt * 1e4 * 1e3, "oracle_sample_pixels": px}
        rows.append(row)
    line = {"metric": "device time of a 100x100 diagram vs n_dot (default algorithm; shape of PAPER.md Fig. 4)",
            "unit": "ms", "n_gpus": 1, "steps": steps, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "random dense Maxwell arrays (workloads.random_open, seeds 4000+n), 10^4 random gate "
                                   "vectors, open and closed with N_hat = n_dot (PAPER.md L490, L496)",
                       "l2": "flushed (256 MiB write) between repetitions"},
            "rows": rows}
    if emit:
        print(json.dumps(line), flush=True)
    return line


# ---------------------------------------------------------------------------------------------------------------------
def parity_report(args):
    """Every pixel of the five BASELINE.json configs at full size, CUDA path through the binding vs the oracle (OpenMP
    over the host cores); run AFTER the timed region.  tests/parity.py holds the rule (north_star: bit-exact except
    near-ties of the oracle below 1e-9 E_C, counted)."""
    import torch
    import oracle
    from paper_2404_04994_b200 import api, workloads as wl
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    from parity import full_size_report
    t0 = time.perf_counter()
    rep = full_size_report(api, oracle, wl, torch, strict=False, config5_members=args.parity_members)
    rep["wall_s"] = round(time.perf_counter() - t0, 1)
    rep["oracle_threads"] = os.cpu_count()
    rep["unexcused_total"] = int(sum(v.get("unexcused", 0) + v.get("sensor_unexcused", 0) + v.get("unexcused_all_variants", 0)
                                     for v in rep.values() if isinstance(v, dict)))
    rep["rule"] = ("N bit-exact except pixels whose oracle best/second-best energies differ by < 1e-9 E_C (counted as "
                   "excused_near_tie); |dE| <= 1e-9 max(|E|, E_C); |dx| <= 1e-9 max(1, |x|), bit-identical without QP")
    return rep


def secondary_workloads(args, local_rank):
    """The other workloads, measured in the same (default) run so that the driver observes them: the dataset batch
    (config 5), the small configs 1-3, the closed 16-dot diagram, thermal broadening and the n_dot sweep."""
    out = {}
    for name, fn in (("config5", lambda: run_config5(args, 0, 1, local_rank, steps=10, emit=False)),
                     ("small", lambda: run_small(args, 0, steps=12, emit=False)),
                     ("closed16", lambda: run_closed16(args, 0, steps=12, emit=False)),
                     ("thermal", lambda: run_thermal(args, 0, steps=5, emit=False)),
                     ("sweep", lambda: run_sweep(args, 0, steps=5, emit=False))):
        try:
            out[name] = fn()
        except Exception as e:  # a secondary workload must never cost the headline line
            out[name] = {"error": f"{type(e).__name__}: {e}"}
    return out


def main():
    args = parse()
    if args.gpus > 1 and "RANK" not in os.environ:
        # `python bench.py --gpus N` launched plainly: start one rank per GPU ourselves (the driver's torchrun command line)
        port = 29500 + (os.getpid() % 2000)
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *sys.argv[1:]]
        env = dict(os.environ)
        env.setdefault("NCCL_DEBUG", "INFO")          # the communicator log shows the ranks
        env.setdefault("NCCL_DEBUG_SUBSYS", "INIT")
        raise SystemExit(subprocess.call(cmd, env=env))
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    import __graft_entry__ as ge
    if rank == 0:
        ge.build()
    if world > 1:
        import torch
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl")
        dist.barrier()
    if args.workload == "thermal":
        run_thermal(args, rank)
    elif args.workload == "small":
        run_small(args, rank)
    elif args.workload == "closed16":
        run_closed16(args, rank)
    elif args.workload == "sweep":
        run_sweep(args, rank)
    elif args.workload == "config5":
        run_config5(args, rank, world, local_rank)
    else:
        run_ours(args, rank, world, local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
