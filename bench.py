#!/usr/bin/env python
"""bench.py -- one JSON line for the ARC hot path on B200 (DESIGN.md section 9 "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config NAME] [--impl reference] [--no-per-config]

A "step" is one pass of the whole hot path over the workload: arc_trace (zero accumulators + opacity table,
persistent ray tracer over all sources, finalize) followed by arc_update_chemistry.  The physics advances from step
to step.  Default workload: config5_N512_S1024 - 512^3 cells, 1024 sources, 4 bins, fp32 fields: the largest
single-GPU configuration of BASELINE.json (its metric names no configuration).  The same line carries `per_config`:
the five BASELINE.json configs and the grid / source sweep points, a few timed steps each.

metric = ray-cell segments per second (BASELINE.json), whole job, inputs resident in HBM; `e2e` = the same through the
C ABI with pinned host buffers.  `roofline` = the tracer kernel's ALGORITHMIC bytes over its CUDA-event
time against the measured HBM copy bandwidth - the figure BASELINE.json asks for; it exceeds 1 because L2 and the
in-quad merge of deposits keep most of those bytes off DRAM, so the line also carries what binds the kernel:
`issue` (warp instructions per second against 4 schedulers x SMs x SM clock) and `roofline.dram_frac` (ncu DRAM bytes
over the same time) - both from the committed ncu capture profiles/ncu_traffic.json, used only if that capture is of
this workload, these flags and this build of the tracer's sources (else null).

With --gpus N > 1 and no torchrun environment the script starts its own N ranks (torch.distributed.run, 127.0.0.1).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import socket
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
DEFAULT_CONFIG = "config5_N512_S1024"
# (workload, warm-up steps, timed steps) of the per-config report; the default workload's own numbers are the line's
PER_CONFIG = [("config1", 3, 10), ("config2", 3, 20), ("config3", 3, 5), ("config4", 2, 3),
              ("config5_N128_S1024", 3, 3), ("config5_N256_S1024", 2, 3), ("config5_N512_S256", 1, 2)]


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


TRACER_SOURCES = ("arc_trace_kernel.cuh", "arc_healpix.cuh", "arc_divide.cuh", "arc_internal.cuh", "arc_trace.cu",
                  "arc_trace_inst_f32_lo.cu", "arc_trace_inst_f32_hi.cu", "arc_trace_inst_f64_lo.cu", "arc_trace_inst_f64_hi.cu")


def csrc_sha16() -> str:
    """identifies the build of the TRACER's sources an ncu capture of the tracer belongs to"""
    h = hashlib.sha256()
    for f in TRACER_SOURCES:
        h.update(f.encode()); h.update(open(os.path.join(ROOT, "paper_1807_07094_b200", "csrc", f), "rb").read())
    return h.hexdigest()[:16]


def ncu_capture(workload: str, segments_per_launch: float, flags: dict):
    """-> (capture dict or None, reason).  profiles/ncu_traffic.json holds, per workload, what one committed
    `ncu --set full` capture of the tracer measured (DRAM bytes, warp instructions per launch).  It is used only when it
    is a capture of THIS workload (same segments per launch), THESE flags and THIS build of the tracer's sources."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            cap = json.load(f).get(workload)
    except OSError:
        return None, "profiles/ncu_traffic.json missing"
    if not cap:
        return None, f"no committed ncu capture of {workload}"
    if any(flags.values()):
        return None, "non-default flags: the committed capture is of the default path"
    if int(cap.get("segments_per_launch", -1)) != int(round(segments_per_launch)):
        return None, "the committed capture traced a different number of segments"
    if cap.get("csrc_sha16") != csrc_sha16():
        return None, f"the committed capture ({cap.get('capture')}) is of another build of the tracer's sources"
    return cap, f"{cap.get('capture')} (ncu --set full, one launch, same workload / flags / tracer sources {cap.get('csrc_sha16')})"


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
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f.read().splitlines():
            t = [x.strip() for x in line.split(",")]
            if len(t) < 7:
                continue
            try:
                sm.append(float(t[0])); mx.append(float(t[1])); pw.append(float(t[2]))
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
                "power_w_median": float(np.median(pw)) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------ the oracle, timed as it stands
def oracle_trace_sample(w, budget_s=12.0, units=None):
    """The oracle's tracer, single thread, on a bounded sample of the workload: the step-0 fields and the first `units`
    (source, root pixel) pairs - whole sources first, the last one through an emission mask that leaves only its first
    root rays open (orc_trace_masked).  units = None: grown until one trace takes about `budget_s`.
    -> (segments, seconds, units, A of that trace)"""
    from oracle import oracle as orc
    kappa = orc.opacity(w)
    npix0 = 12 << (2 * int(w.params["l0"]))
    total = w.nsrc * npix0

    def run(u):
        S = -(-u // npix0)
        mask = np.ones((w.nsrc, npix0), dtype=np.uint8)
        mask.reshape(-1)[:u] = 0
        t0 = time.perf_counter()
        A, st, _ = orc.trace(w, kappa=kappa, sources=np.arange(S), blocked=mask)
        return st["segments"], time.perf_counter() - t0, A

    if units is not None:
        seg, secs, A = run(units)
        return seg, secs, units, A
    u = 1
    while True:
        seg, secs, A = run(u)
        if secs >= budget_s / 2.0 or u >= total:
            return seg, secs, u, A
        u = int(min(total, max(u + 1, u * min(4.0, 0.6 * budget_s / max(secs, 1e-3)))))


def sample_text(w, units):
    npix0 = 12 << (2 * int(w.params["l0"]))
    S, rest = divmod(units, npix0)
    return (f"the first {S} of {w.nsrc} sources" if S else "") + (" + " if S and rest else "") + \
           (f"{rest} of the {npix0} root rays of source {S}" if rest else "")


def oracle_chem_sample(w, A, n_cells):
    """The oracle's finalize + chemistry, single thread, on a strided sample of `n_cells` cells of the step-0 fields
    (the update is per cell) with the rates the sample trace `A` gives them.
    -> (cells, seconds, sub-cycles)"""
    import dataclasses
    from oracle import oracle as orc
    side = max(4, int(round(n_cells ** (1.0 / 3.0))))
    n = side ** 3                                               # (the C routine takes a cubic cell count)
    idx = (np.arange(n, dtype=np.int64) * (w.ncell // n)) % w.ncell
    ws = dataclasses.replace(w, N=side, box_cm=w.box_cm * side / w.N)       # (same cell size)
    f = tuple(np.ascontiguousarray(np.asarray(a, dtype=np.float64)[idx]) for a in w.fields())
    G, H, _ = orc.finalize(ws, np.ascontiguousarray(A[idx]), f)
    t0 = time.perf_counter()
    _, sub = orc.chemistry(ws, f, G, H, w.dt_s)
    return n, time.perf_counter() - t0, int(sub.sum())


def cpu_baseline(w, budget_s=12.0):
    seg, secs, units, A = oracle_trace_sample(w, budget_s)
    # chemistry: as many cells as take a comparable time (about 1 us per sub-cycle), at most the grid
    cells, csecs, sub = oracle_chem_sample(w, A, min(w.ncell, 2_000_000))
    return {"value": seg / secs, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"step-0 fields, {sample_text(w, units)}, opacity table + ray trace, {seg} segments in {secs:.1f} s, "
                      f"single thread; host has {os.cpu_count()} cores",
            "chemistry": {"value": cells / csecs, "unit": "cells/s", "subcycles_per_s": sub / csecs,
                          "sample": f"finalize + sub-cycled update of {cells} cells strided through the grid, rates of the sample "
                                    f"trace, {sub} sub-cycles in {csecs:.1f} s, single thread"}}


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores.  Each step = the same fraction f of both halves of a
    step: the trace of the first f n_src 12 4^l0 root rays and the finalize + chemistry of f n_cell cells; f is set so
    that the whole run (warm-up + timed steps) takes about three minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        sys.stderr.write(f"bench.py: rank {rank} of {os.environ.get('WORLD_SIZE', '1')}: the reference arm runs on rank 0 alone\n")
        return
    w = make_workload(args.config)
    npix0 = 12 << (2 * int(w.params["l0"]))
    budget = min(12.0, max(1.0, 180.0 / (args.warmup + args.steps + 1)))
    _, _, units, _ = oracle_trace_sample(w, budget_s=budget)               # (calibration, untimed)
    tot_seg, tot_s, cells = 0, 0.0, 0
    for i in range(args.warmup + args.steps):
        seg, s, _, A = oracle_trace_sample(w, units=units)
        cells, cs, sub = oracle_chem_sample(w, A, max(64, w.ncell * units // (w.nsrc * npix0)))
        if i >= args.warmup:
            tot_seg += seg; tot_s += s + cs
    v = tot_seg / tot_s
    sample = (f"step-0 fields; per step: trace of {sample_text(w, units)} ({tot_seg // max(1, args.steps)} segments) + finalize and "
              f"chemistry of {cells} of {w.ncell} cells; single thread; host has {os.cpu_count()} cores")
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


def free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def self_launch(argv, n: int) -> int:
    """`python bench.py --gpus N` without a torchrun environment: start the N ranks ourselves (one process per GPU,
    rendezvous on 127.0.0.1) and pass their output through; rank 0 prints the one JSON line."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(n), "--master-addr", "127.0.0.1",
           "--master-port", str(free_port()), os.path.abspath(__file__)] + list(argv)
    return subprocess.call(cmd)


# ------------------------------------------------------------------------------------------------ CUDA arm
def timed_run(w, steps, warmup, extra, stream, shard_sources=None, barrier=None, sampler_index=None, graph_steps=0):
    """`warmup` untimed + `steps` timed steps with the fields resident in HBM; device times from CUDA events on the
    library's stream.  -> dict of raw measurements of THIS rank."""
    import torch
    from paper_1807_07094_b200 import arc, sharded
    fdt = np.float32 if w.dtype == "f32" else np.float64
    dev_fields = [torch.from_numpy(np.ascontiguousarray(np.asarray(a, dtype=fdt))).cuda() for a in w.fields()]
    cx = arc.Context(w, fields=dev_fields, stream=stream.cuda_stream, **extra)
    if shard_sources is not None:
        cx.set_sources(shard_sources)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    out = dict(seg=[], kern_ms=[], chem_ms=[], trace_ms=[], sub=[], opacity_ms=[], finalize_ms=[])

    def one_step(i, record):
        if shard_sources is not None:
            sharded.trace_sharded(cx, None, i)    # this rank's sources, all-reduce of the accumulators, finalize
        else:
            cx.trace(i)
        cx.update_chemistry()
        if record:
            st = cx.stats()                       # synchronises the stream; reads the per-kernel event times
            out["seg"].append(st["segments"]); out["kern_ms"].append(st["trace_kernel_ms"]); out["chem_ms"].append(st["chem_ms"])
            out["trace_ms"].append(st["trace_ms"]); out["sub"].append(st["subcycles"])
            out["opacity_ms"].append(st["opacity_ms"]); out["finalize_ms"].append(st["finalize_ms"])

    for i in range(warmup):
        one_step(i, False)
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    sampler = ClockSampler(sampler_index) if sampler_index is not None else None
    launches0 = cx.stats()["kernel_launches"]
    t0 = time.perf_counter()
    ev[0].record(stream)
    for i in range(steps):
        one_step(warmup + i, True)
    ev[1].record(stream)
    if barrier:
        barrier()
    else:
        torch.cuda.synchronize()
    out["wall_s"] = time.perf_counter() - t0
    out["clocks"] = sampler.stop() if sampler else None
    out["dev_ms"] = ev[0].elapsed_time(ev[1])
    cons = cx.stats()
    out["launches"] = cons["kernel_launches"] - launches0
    out["stats"] = cons
    out["trace_grid"] = cons["trace_grid"]
    if graph_steps:
        # the same loop through arc_run_steps: one captured CUDA graph per step, replayed, one synchronisation at the end
        cx.set_fields(dev_fields)                 # (from the initial fields again)
        cx.run_steps(max(3, warmup))
        s0 = cx.stats()
        cx.run_steps(graph_steps)
        s1 = cx.stats()
        seg = s1["segments_total"] - s0["segments_total"]
        out["graph"] = {"steps": graph_steps, "ms_per_step": s1["steps_ms"] / graph_steps,
                        "segments_per_s": seg / (s1["steps_ms"] * 1e-3) if s1["steps_ms"] > 0 else 0.0,
                        "launches_per_step": (s1["kernel_launches"] - s0["kernel_launches"]) / graph_steps}
    cx.close()
    del dev_fields
    return out


def summarise(w, r, steps, peak):
    """per-workload figures from one rank's timed_run (per_config entries and the pieces of the headline)"""
    nc = w.ncell
    tot_seg, kms, cms = float(sum(r["seg"])), float(sum(r["kern_ms"])), float(sum(r["chem_ms"]))
    bps = algorithmic_bytes_per_segment(w)
    ach = bps * tot_seg / (kms * 1e-3) / 1e9 if kms > 0 else 0.0
    st = r["stats"]
    return {"segments_per_s": job_throughput(tot_seg, r["dev_ms"]), "ms_per_step": r["dev_ms"] / steps,
            "trace_kernel_segments_per_s": tot_seg / (kms * 1e-3) if kms > 0 else 0.0, "trace_kernel_ms": kms / steps,
            "cell_updates_per_s": nc * steps / (cms * 1e-3) if cms > 0 else 0.0, "chem_ms": cms / steps,
            "chem_subcycles_per_step": float(sum(r["sub"])) / steps,
            "segments_per_step": tot_seg / steps, "hbm_algorithmic_gbs": ach, "hbm_algorithmic_frac": ach / peak,
            "algorithmic_bytes_per_segment": bps,
            "photon_conservation_max_rel_err": float(np.max(np.abs((st["absorbed"] + st["escaped"]) / st["emitted"] - 1.0)))}


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
    shard = args.shard == "sources"
    if world > 1:
        if shard:
            os.environ.setdefault("NCCL_DEBUG", "INFO")          # the communicator log (algorithm, NVLS) goes to stderr
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = make_workload(args.config)
    fdt = np.float32 if w.dtype == "f32" else np.float64
    stream = torch.cuda.Stream()
    nc, nb = w.ncell, w.nb
    bytes_seg = algorithmic_bytes_per_segment(w)
    peak, peak_src = hbm_peak()
    extra = {}
    if args.geom_corr:
        extra["geom_corr"] = args.geom_corr
    if args.thin_tau:
        extra["thin_tau"] = args.thin_tau
    my_sources = sharded.partition_sources(w.nsrc, world)[rank] if shard else None

    # ---- arm 1: inputs resident in HBM (device tensors handed over once, before the timed region)
    with torch.cuda.stream(stream):               # (the library enqueues on `stream` itself; torch's helpers follow)
        r = timed_run(w, args.steps, args.warmup, extra, stream, my_sources, barrier, local if rank == 0 else None)
    cons = r["stats"]
    if shard:
        with torch.cuda.stream(stream):
            cons = sharded.reduce_stats(cons)
        cons = {k: (np.asarray(v) if isinstance(v, list) else v) for k, v in cons.items()}
        r["stats"] = cons
    head = summarise(w, r, args.steps, peak)

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
            sharded.trace_sharded(cx2, None, i)
        else:
            arc.arc_trace(cx2.ctx, i)
        arc.arc_update_chemistry(cx2.ctx, w.dt_s)
        arc.arc_get_fields(cx2.ctx, None, hp[1], hp[2], hp[3], hp[4])      # D2H: the four updated fields
        rh = [x.numpy() for x in rates_host]
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
    del pin, rates_host

    # ---- reduce over ranks (replicas: every rank ran the same workload on its own GPU)
    tot_seg = float(sum(r["seg"]))
    (dev_ms_max, e2e_ms_max), (seg_all, e2e_seg_all) = reduce_over_ranks([r["dev_ms"], e2e_ms], [tot_seg, float(e2e_seg)], "cuda", world)

    if rank == 0:
        kms = float(sum(r["kern_ms"]))
        clocks = r["clocks"]
        flags = {"geom_corr": args.geom_corr, "thin_tau": args.thin_tau, "shard": shard}
        cap, cap_src = ncu_capture(w.name, tot_seg / args.steps, flags)
        achieved = head["hbm_algorithmic_gbs"]
        traffic = cap["dram_bytes_per_launch"] if cap else None
        line = {
            "metric": METRIC, "value": job_throughput(seg_all, dev_ms_max), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dev_ms_max / args.steps, "higher_is_better": True, "scaling": "strong" if shard else "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded, paper_1807_07094_b200/workloads.py)",
            "config": dict(describe(w), parallelism=(f"sources sharded over {world} rank(s), one all-reduce of the accumulators per step" if shard
                                                     else ("replicas" if world > 1 else "single-gpu")),
                           l2_policy="inputs larger than L2" if (nc * nb * (bytes_seg // nb)) > 126e6 else "working set fits L2 (small config)",
                           trace_grid_blocks=r["trace_grid"], geom_corr=args.geom_corr, thin_tau=args.thin_tau),
            "e2e": {"value": job_throughput(e2e_seg_all, e2e_ms_max), "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h},
            "gpu_launches": int(r["launches"]),
            "clocks": clocks,
            "roofline": {"bound": "hbm", "kernel": "arc_trace_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                         "algorithmic_bytes_per_segment": bytes_seg, "segments_per_launch": tot_seg / args.steps,
                         "kernel_ms_per_launch": kms / args.steps,
                         "dram_frac": (traffic / (kms / args.steps * 1e-3) / 1e9 / peak) if traffic and kms > 0 else None,
                         "traffic_source": cap_src,
                         "binding_limit": "issue slots (see `issue`): `frac` counts algorithmic bytes, most of which L2 and the "
                                          "in-quad merge of deposits keep off DRAM; `dram_frac` is the DRAM traffic ncu measured"},
            "segments_per_step": [int(x) for x in r["seg"]],
            "trace_kernel_ms": [round(x, 3) for x in r["kern_ms"]], "chem_ms": [round(x, 3) for x in r["chem_ms"]],
            "opacity_ms": [round(x, 3) for x in r["opacity_ms"]], "finalize_ms": [round(x, 3) for x in r["finalize_ms"]],
            "trace_kernel_segments_per_s": head["trace_kernel_segments_per_s"],
            "cell_updates_per_s": head["cell_updates_per_s"],
            "chem_subcycles_per_step": [int(x) for x in r["sub"]],
            "photon_conservation_max_rel_err": head["photon_conservation_max_rel_err"],
            "host_wall_s": r["wall_s"],
        }
        if cap and cap.get("warp_instructions_per_launch") and clocks and clocks.get("sm_mhz") and kms > 0:
            # the limit that binds: issue slots.  4 schedulers x SMs x SM clock under load
            n_sm = torch.cuda.get_device_properties(local).multi_processor_count
            ach = cap["warp_instructions_per_launch"] / (kms / args.steps * 1e-3) / 1e9
            pk = 4 * n_sm * clocks["sm_mhz"] * 1e6 / 1e9
            line["issue"] = {"bound": "issue", "achieved": ach, "peak": pk, "unit": "G warp-instructions/s", "frac": ach / pk,
                             "warp_instructions_per_segment": cap["warp_instructions_per_launch"] / cap["segments_per_launch"],
                             "source": cap_src,
                             "peak_source": f"4 schedulers x {n_sm} SMs x {clocks['sm_mhz']:.0f} MHz (SM clock sampled under load)"}
        else:
            line["issue"] = None
        if world == 1 and not args.no_per_config and not any(flags.values()):
            per = {w.name: dict(head, warmup=args.warmup, steps=args.steps, **{k: describe(w)[k] for k in ("grid", "sources", "freq_bins", "field_dtype")})}
            for name, wu, k in PER_CONFIG:
                if name == w.name:
                    continue
                wc = make_workload(name)
                with torch.cuda.stream(stream):
                    rc = timed_run(wc, k, wu, {}, stream, graph_steps=(10 * k if wc.nsrc <= 16 else 0))
                per[wc.name] = dict(summarise(wc, rc, k, peak), warmup=wu, steps=k,
                                    **{kk: describe(wc)[kk] for kk in ("grid", "sources", "freq_bins", "field_dtype")})
                if "graph" in rc:
                    per[wc.name]["arc_run_steps"] = rc["graph"]
                del wc, rc
            line["per_config"] = per
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(w, budget_s=12.0)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main(argv=None):
    argv = sys.argv[1:] if argv is None else argv
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default=DEFAULT_CONFIG,
                    help="config1..config4, config4_T, config5[_N<grid>][_S<sources>][_T] (default: the largest single-GPU configuration)")
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per-config report (the other BASELINE.json configs, a few steps each)")
    ap.add_argument("--geom-corr", type=int, default=0, help="arc_params.geom_corr (PAPER.md:100-114): 0 none (the north_star path), 1 f_c, 2 f_c + secondary, 3 f_c^2")
    ap.add_argument("--thin-tau", type=float, default=0.0, help="arc_params.thin_tau (PAPER.md:116-130): 0 off (the north_star path), 0.1 in the paper")
    ap.add_argument("--shard", default="none", choices=["none", "sources"],
                    help="N > 1: 'none' = independent replicas (the north_star path, weak scaling); 'sources' = the sources divided among the "
                         "ranks, one all-reduce of the accumulators per step (paper_1807_07094_b200/sharded.py; strong scaling)")
    args = ap.parse_args(argv)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        raise SystemExit(self_launch(argv, args.gpus))
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
