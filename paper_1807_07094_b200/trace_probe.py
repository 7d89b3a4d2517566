"""Tracer time of small and few-source traces (the regime where the scheduler, not the segment loop, sets the time).

    python -m paper_1807_07094_b200.trace_probe [--trace-blocks B]

For each workload: 3 warm-up traces, then the minimum and mean `arc_stats.trace_kernel_ms` of 7 traces on the same
fields (no chemistry in between, so every trace does the same work).  Workloads: configs 1 and 2 at their first step,
config 2 with x_HI = 1e-3 everywhere (every ray crosses the box), config 2 with all root rays but one blocked (a lone
ray tree: the critical path), config 3's grid with its first 1 / 4 / 16 sources, config 4 with its first 64 sources.
This is what `profiles/r01j_small_traces.txt` tabulates.  Needs a CUDA device (there is no CPU fallback).
"""
from __future__ import annotations

import argparse
import dataclasses

import numpy as np

from . import arc, workloads as wl


def probe(name, w, fields=None, blocked=None, **params):
    with arc.Context(w, fields=fields, **params) as cx:
        if blocked is not None:
            cx.set_emission_mask(blocked)
        for i in range(3):
            cx.trace(i)
        ms = []
        for i in range(7):
            cx.trace(i)
            st = cx.stats()
            ms.append(st["trace_kernel_ms"])
        print(f"{name}: segments {st['segments']:.3e} rays {st['rays']} grid {st['trace_grid']} blocks | kernel ms min {min(ms):.4f} "
              f"mean {np.mean(ms):.4f} | {st['segments'] / min(ms) / 1e6:.2f} G segments/s | queue high-water {st['queue_high_water']}", flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--trace-blocks", type=int, default=0, help="arc_params.trace_blocks: persistent grid size (0 = all co-resident blocks)")
    a = ap.parse_args()
    kw = {"trace_blocks": a.trace_blocks} if a.trace_blocks else {}
    probe("config1 neutral", wl.config1(), **kw)
    w = wl.config2()
    probe("config2 neutral", w, **kw)
    f = list(w.fields())
    f[1] = np.full_like(f[1], 1e-3)
    probe("config2 x_HI = 1e-3", w, fields=f, **kw)
    bl = np.ones((1, 12 << (2 * int(w.params["l0"]))), np.uint8)
    bl[0, 17] = 0
    probe("config2 lone tree (one open root ray)", w, blocked=bl, **kw)
    for ns in (1, 4, 16):
        probe(f"config3 grid, {ns} source(s)", wl.config3(nsrc=ns), **kw)
    w = wl.config4()
    K = 64
    probe("config4, first 64 sources", dataclasses.replace(w, src_pos_cm=w.src_pos_cm[:K], src_Ndot=w.src_Ndot[:K],
                                                          src_binfrac=w.src_binfrac[:K]), **kw)


if __name__ == "__main__":
    main()
