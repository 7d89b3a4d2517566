#!/usr/bin/env python
"""bench.py -- one JSON line for the ARC hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config config4] [--impl reference]

A "step" is one pass of the whole hot path over the workload: arc_trace (zero accumulators + opacity
table, persistent ray tracer over all sources, finalize) followed by arc_update_chemistry.  The physics
advances from step to step, so later steps trace more segments (the box ionises).
metric = ray-cell segments per second (BASELINE.json), whole job; roofline = the tracer kernel's
algorithmic bytes / its CUDA-event time against the measured HBM copy bandwidth.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC, UNIT = "ray_cell_segments_per_s", "segments/s"
FALLBACK_HBM_GBS = 6650.0          # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def make_workload(name: str):
    from paper_1807_07094_b200 import workloads as wl
    if name.startswith("config5"):
        # config5[_N<grid>][_S<sources>][_T] ; _T = transparent state (B)
        N, S, state = 512, 1024, "neutral"
        for tok in name.split("_")[1:]:
            if tok.startswith("N"): N = int(tok[1:])
            elif tok.startswith("S"): S = int(tok[1:])
            elif tok == "T": state = "transparent"
        return wl.config5(N=N, nsrc=S, state=state)
    if name == "config4_T":
        return wl.config4(state="transparent")
    return wl.by_name(name)


def describe(w) -> dict:
    return {"workload": w.name, "grid": f"{w.N}^3", "sources": w.nsrc, "freq_bins": w.nb, "field_dtype": w.dtype,
            "accumulators": "f64", "l0": int(w.params["l0"]), "Phi": float(w.params["Phi"]),
            "tau_term": float(w.params["tau_term"]) if np.isfinite(w.params["tau_term"]) else "inf",
            "isothermal": int(w.params["isothermal"]), "Yp": float(w.params["Yp"])}


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_capture(config: str) -> dict:
    """What the committed `ncu --set full` capture of the tracer on this workload measured (profiles/ncu_traffic.json
    names the capture): DRAM bytes and warp instructions per launch.  {} if this workload has none."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            return json.load(f).get(config, {})
    except OSError:
        return {}


def ncu_traffic(config: str):
    """dram__bytes_read.sum + dram__bytes_write.sum of one tracer launch on this workload, or None."""
    return ncu_capture(config).get("dram_bytes_per_launch")


def algorithmic_bytes_per_segment(w) -> int:
    """gather nb opacities at the field dtype + read-modify-write nb fp64 accumulators."""
    return (4 if w.dtype == "f32" else 8) * w.nb + 16 * w.nb


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "200",
                                       "-i", str(index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self) -> dict:
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            t = [x.strip() for x in line.split(",")]
            if len(t) < 7:
                continue
            try:
                sm.append(float(t[0])); mx.append(float(t[1]))
            except ValueError:
                continue
            for n, v in zip(names, t[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------ reference arm
def oracle_sample(w, budget_s=12.0):
    """The oracle, as it stands, on a bounded sample of the workload: the step-0 fields, the first S
    sources (S grown until the trace takes about `budget_s`).  -> (segments, seconds, S, threads)"""
    from oracle import oracle as orc
    kappa = orc.opacity(w)
    S, segs, secs = 1, 0, 0.0
    while True:
        S = min(S, w.nsrc)
        t0 = time.perf_counter()
        _, st, _ = orc.trace(w, kappa=kappa, sources=np.arange(S))
        secs = time.perf_counter() - t0
        segs = st["segments"]
        if secs >= budget_s / 3.0 or S >= w.nsrc:
            break
        S = int(min(w.nsrc, max(S + 1, S * min(8.0, budget_s / max(secs, 1e-3)) * 0.8)))
    return segs, secs, S, 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args.config)
    per = []
    tot_seg, tot_s, S = 0, 0.0, 0
    for i in range(args.warmup + args.steps):
        seg, s, S, cores = oracle_sample(w, budget_s=6.0)
        if i >= args.warmup:
            tot_seg += seg; tot_s += s; per.append(s)
    v = tot_seg / tot_s
    sample = f"step-0 fields, first {S} of {w.nsrc} sources, opacity table + ray trace, single thread, {tot_seg // max(1, args.steps)} segments per step"
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded, paper_1807_07094_b200/workloads.py)",
            "config": describe(w),
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------ ranks
def reduce_over_ranks(times_ms, counts, device, world):
    """Replicas only: every rank runs the whole workload on its own GPU and nothing of the data path
    crosses ranks.  The job's time is the MAX over ranks of each device-timed interval, its work the SUM over ranks
    of the units processed.  -> (list of max times, list of summed counts)"""
    import torch
    t = torch.tensor([float(x) for x in times_ms], dtype=torch.float64, device=device)
    s = torch.tensor([float(x) for x in counts], dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(s, op=dist.ReduceOp.SUM)
    return t.tolist(), s.tolist()


def job_throughput(units_all_ranks, ms_max_over_ranks):
    return units_all_ranks / (ms_max_over_ranks * 1e-3) if ms_max_over_ranks > 0 else 0.0


# ------------------------------------------------------------------------------------------------ CUDA arm
def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_1807_07094_b200 import arc, sharded

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the CUDA path is the product and there is no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = make_workload(args.config)
    if args.sources:                      # profiling aid: the first K sources of the workload (named so in config.workload)
        import dataclasses
        K = min(args.sources, w.nsrc)
        w = dataclasses.replace(w, name=f"{w.name}[first {K} sources]", src_pos_cm=w.src_pos_cm[:K], src_Ndot=w.src_Ndot[:K],
                                src_binfrac=w.src_binfrac[:K])
    fdt = np.float32 if w.dtype == "f32" else np.float64
    tdt = torch.float32 if w.dtype == "f32" else torch.float64
    stream = torch.cuda.Stream()
    nc, nb = w.ncell, w.nb
    bytes_seg = algorithmic_bytes_per_segment(w)
    peak, peak_src = hbm_peak()

    # ---- arm 1: inputs resident in HBM (device tensors handed over once, before the timed region)
    dev_fields = [torch.from_numpy(np.ascontiguousarray(np.asarray(a, dtype=fdt))).cuda() for a in w.fields()]
    extra = {"deposit": args.deposit} if args.deposit else {}
    if args.geom_corr:
        extra["geom_corr"] = args.geom_corr
    if args.thin_tau:
        extra["thin_tau"] = args.thin_tau
    cx = arc.Context(w, fields=dev_fields, stream=stream.cuda_stream, **extra)
    shard = args.shard == "sources"
    my_sources = sharded.partition_sources(w.nsrc, world)[rank] if shard else None
    if shard:
        cx.set_sources(my_sources)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    seg_steps, kern_ms, chem_ms, trace_ms, sub_steps, rec_steps = [], [], [], [], [], []

    def one_step(i, record):
        if shard:
            sharded.trace_sharded(cx, None, i)    # this rank's sources, all-reduce of the accumulators, finalize
        else:
            cx.trace(i)
        cx.update_chemistry()
        if record:
            st = cx.stats()                       # synchronises the stream; reads the per-kernel event times
            seg_steps.append(st["segments"]); kern_ms.append(st["trace_kernel_ms"]); chem_ms.append(st["chem_ms"])
            trace_ms.append(st["trace_ms"]); sub_steps.append(st["subcycles"]); rec_steps.append(st["deposit_records"])

    with torch.cuda.stream(stream):               # (the all-reduce of --shard sources goes to torch's current stream)
        for i in range(args.warmup):
            one_step(i, False)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    t_host0 = time.perf_counter()
    with torch.cuda.stream(stream):
        ev[0].record(stream)
        for i in range(args.steps):
            one_step(args.warmup + i, True)
        ev[1].record(stream)
    barrier()
    wall = time.perf_counter() - t_host0
    clocks = sampler.stop() if sampler else None
    dev_ms = ev[0].elapsed_time(ev[1])
    cons = cx.stats()
    if shard:
        with torch.cuda.stream(stream):
            cons = sharded.reduce_stats(cons)
        cons = {k: (np.asarray(v) if isinstance(v, list) else v) for k, v in cons.items()}
    conservation = float(np.max(np.abs((cons["absorbed"] + cons["escaped"]) / cons["emitted"] - 1.0)))
    trace_grid = cons["trace_grid"]
    cx.close()
    del dev_fields

    # deposit records per segment: a statistic the production kernel does not count (digest builds do): one untimed trace
    seg_per_record = None
    if rank == 0:
        with arc.Context(w, digest=1, stream=stream.cuda_stream, **extra) as cxd:
            if shard:
                cxd.set_sources(my_sources)
            cxd.trace(0)
            sd = cxd.stats()
            seg_per_record = sd["segments"] / max(1, sd["deposit_records"])

    # ---- arm 2: end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    pin = [torch.from_numpy(np.ascontiguousarray(np.asarray(a, dtype=fdt))).pin_memory() for a in w.fields()]
    rates_host = [torch.empty(nc, dtype=torch.float64).pin_memory() for _ in range(4)]   # Gamma_HI, Gamma_HeI, Gamma_HeII, heat_total
    cx2 = arc.Context(w, fields=[p.numpy() for p in pin], stream=stream.cuda_stream, **extra)
    if shard:
        cx2.set_sources(my_sources)
    h2d = 5 * nc * pin[0].element_size()
    d2h = 4 * nc * pin[0].element_size() + 4 * nc * 8
    e2e_seg = 0

    def e2e_step(i):
        hp = [p.numpy() for p in pin]
        arc.arc_set_fields(cx2.ctx, *hp)                                   # H2D: the five fields
        if shard:
            with torch.cuda.stream(stream):
                sharded.trace_sharded(cx2, None, i)
        else:
            arc.arc_trace(cx2.ctx, i)
        arc.arc_update_chemistry(cx2.ctx, w.dt_s)
        arc.arc_get_fields(cx2.ctx, None, hp[1], hp[2], hp[3], hp[4])      # D2H: the four updated fields
        rh = [r.numpy() for r in rates_host]
        arc.arc_get_rates(cx2.ctx, rh[0], rh[1], rh[2], None, None, None, rh[3])   # D2H: the step's rates
        return arc.arc_get_stats(cx2.ctx).segments

    for i in range(args.warmup):
        e2e_step(i)
    barrier()
    ev2 = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    ev2[0].record(stream)
    t0 = time.perf_counter()
    for i in range(args.steps):
        e2e_seg += e2e_step(args.warmup + i)
    ev2[1].record(stream)
    barrier()
    e2e_wall = time.perf_counter() - t0
    e2e_ms = max(ev2[0].elapsed_time(ev2[1]), 1e3 * e2e_wall)     # host-blocking copies: the wall clock is the honest one
    cx2.close()

    # ---- reduce over ranks (replicas: every rank ran the same workload on its own GPU)
    tot_seg = float(sum(seg_steps))
    (dev_ms_max, e2e_ms_max), (seg_all, e2e_seg_all) = reduce_over_ranks([dev_ms, e2e_ms], [tot_seg, float(e2e_seg)], "cuda", world)

    if rank == 0:
        kms = float(sum(kern_ms))
        achieved = bytes_seg * tot_seg / (kms * 1e-3) / 1e9 if kms > 0 else 0.0
        line = {
            "metric": METRIC, "value": job_throughput(seg_all, dev_ms_max), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dev_ms_max / args.steps, "higher_is_better": True, "scaling": "strong" if shard else "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded, paper_1807_07094_b200/workloads.py)",
            "config": dict(describe(w), parallelism=(f"sources sharded over {world} rank(s), one all-reduce of the accumulators per step" if shard
                                                     else ("replicas" if world > 1 else "single-gpu")),
                           l2_policy="inputs larger than L2" if (nc * nb * (bytes_seg // nb)) > 126e6 else "working set fits L2 (small config)",
                           trace_grid_blocks=trace_grid, deposit=args.deposit, geom_corr=args.geom_corr, thin_tau=args.thin_tau),
            "e2e": {"value": job_throughput(e2e_seg_all, e2e_ms_max), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": 5 * args.steps,
            "clocks": clocks,
            "roofline": {"bound": "hbm", "kernel": "arc_trace_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "traffic": ncu_traffic(args.config), "peak_source": peak_src,
                         "algorithmic_bytes_per_segment": bytes_seg, "segments_per_launch": tot_seg / args.steps,
                         "kernel_ms_per_launch": kms / args.steps},
            "segments_per_step": [int(x) for x in seg_steps],
            "trace_kernel_ms": [round(x, 3) for x in kern_ms], "chem_ms": [round(x, 3) for x in chem_ms],
            "trace_kernel_segments_per_s": tot_seg / (kms * 1e-3) if kms > 0 else 0.0,
            "cell_updates_per_s": nc * args.steps / (sum(chem_ms) * 1e-3) if sum(chem_ms) > 0 else 0.0,
            "chem_subcycles_per_step": [int(x) for x in sub_steps],
            "photon_conservation_max_rel_err": conservation,
            "segments_per_deposit_record": seg_per_record,
            "host_wall_s": wall,
        }
        cap = ncu_capture(args.config)
        if cap.get("warp_instructions_per_segment") and clocks and clocks.get("sm_mhz") and kms > 0:
            # the limit that binds: issue slots.  4 schedulers x SMs x SM clock under load
            import torch as _t
            n_sm = _t.cuda.get_device_properties(local).multi_processor_count
            ach = cap["warp_instructions_per_segment"] * tot_seg / (kms * 1e-3) / 1e9
            pk = 4 * n_sm * clocks["sm_mhz"] * 1e6 / 1e9
            line["issue"] = {"bound": "issue", "achieved": ach, "peak": pk, "unit": "G warp-instructions/s", "frac": ach / pk,
                             "warp_instructions_per_segment": cap["warp_instructions_per_segment"],
                             "peak_source": f"4 schedulers x {n_sm} SMs x {clocks['sm_mhz']:.0f} MHz (SM clock sampled under load)"}
        if world == 1 and not args.no_cpu_baseline:
            seg, secs, S, cores = oracle_sample(w, budget_s=12.0)
            line["cpu_baseline"] = {"value": seg / secs, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": f"step-0 fields, first {S} of {w.nsrc} sources, ray trace only, {seg} segments in {secs:.1f} s, "
                                              f"host has {os.cpu_count()} cores"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="config4")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--geom-corr", type=int, default=0, help="arc_params.geom_corr (PAPER.md:100-114): 0 none (the north_star path), 1 f_c, 2 f_c + secondary, 3 f_c^2")
    ap.add_argument("--thin-tau", type=float, default=0.0, help="arc_params.thin_tau (PAPER.md:116-130): 0 off (the north_star path), 0.1 in the paper")
    ap.add_argument("--shard", default="none", choices=["none", "sources"],
                    help="N > 1: 'none' = independent replicas (the north_star path, weak scaling); 'sources' = the sources divided among the "
                         "ranks, one all-reduce of the accumulators per step (paper_1807_07094_b200/sharded.py; strong scaling)")
    ap.add_argument("--sources", type=int, default=0, help="profiling aid: keep only the first K sources of the workload")
    ap.add_argument("--deposit", type=int, default=0, help="arc_params.deposit: 0 auto, 1 per-lane REDs, 2 warp-aggregated")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
