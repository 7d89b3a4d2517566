"""Source-sharded tracing over several GPUs.

Rays of different sources are independent and the absorbed-photon accumulators add, so the sources are divided among
the ranks (one process per GPU, every rank holds the whole grid: 512^3 with all arrays is 17 GB of 180 GB), each rank
traces its share with `arc_trace_partial`, ONE all-reduce (sum) of the `N^3 x nbins` fp64 accumulators follows, and
every rank forms the rates (`arc_finalize`) and updates the chemistry redundantly - the fields stay identical on all
ranks without a second exchange, as in the paper's replicated-grid mode (:158-164).

Host logic only: the arithmetic is the library's kernels; the sum is torch.distributed's (NCCL on GPUs).  Nothing here
imports `oracle/`.
"""
from __future__ import annotations

import numpy as np


def partition_sources(nsrc: int, world_size: int, weights=None) -> list[np.ndarray]:
    """Deterministic, balanced division of source indices 0..nsrc-1 among `world_size` ranks.

    `weights` = expected work per source (default: equal - without depletion every source crosses the same
    ~10.3 N^3 segments).  Longest-processing-time greedy: sources by decreasing weight (ties by index),
    each to the currently lightest rank (ties to the lowest rank).  Every rank gets its indices in increasing order;
    the shards are disjoint and cover all sources; with equal weights the sizes differ by at most one.
    """
    if world_size < 1 or nsrc < 0:
        raise ValueError("world_size >= 1 and nsrc >= 0 required")
    w = np.ones(nsrc) if weights is None else np.asarray(weights, dtype=np.float64)
    if w.shape != (nsrc,) or not np.all(np.isfinite(w)) or np.any(w < 0):
        raise ValueError("weights must be nsrc finite non-negative numbers")
    order = sorted(range(nsrc), key=lambda i: (-w[i], i))
    load = [0.0] * world_size
    count = [0] * world_size
    shards: list[list[int]] = [[] for _ in range(world_size)]
    for i in order:
        r = min(range(world_size), key=lambda k: (load[k], count[k], k))
        shards[r].append(i)
        load[r] += float(w[i])
        count[r] += 1
    return [np.array(sorted(s), dtype=np.int64) for s in shards]


def trace_sharded(tracer, group=None, step: int = 0):
    """One radiative-transfer pass with the sources sharded over the ranks of `group`.

    `tracer` holds THIS rank's share of the sources and offers `trace_partial(step)`, `accum_tensor()` (a tensor that
    aliases its accumulators) and `finalize()` - `arc.Context` does.  The three steps must run in stream order: the
    all-reduce is issued ON THE CONTEXT'S OWN STREAM (`tracer.stream`, a cudaStream_t handle; 0 / None = the legacy
    default stream), whatever torch's current stream is, so that it follows the tracer's REDs and precedes finalize
    also when the context runs with `async = 1`.
    """
    import contextlib
    import torch.distributed as dist
    tracer.trace_partial(step)
    A = tracer.accum_tensor()
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        on_stream = contextlib.nullcontext()
        handle = getattr(tracer, "stream", None)
        if getattr(A, "is_cuda", False):
            import torch
            on_stream = torch.cuda.stream(torch.cuda.ExternalStream(int(handle)) if handle else torch.cuda.default_stream())
        with on_stream:
            dist.all_reduce(A, op=dist.ReduceOp.SUM, group=group)
    return tracer.finalize()


def reduce_stats(stats: dict, group=None) -> dict:
    """Whole-job tallies from the per-rank `Context.stats()`: counters and emitted / escaped photons add over the
    shards; `absorbed` is already global (it is summed from the reduced accumulators at finalize)."""
    import torch
    import torch.distributed as dist
    out = dict(stats)
    if not (dist.is_initialized() and dist.get_world_size(group) > 1):
        return out
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    for key in ("segments", "rays"):
        t = torch.tensor([int(stats[key])], dtype=torch.int64, device=dev)
        dist.all_reduce(t, group=group)
        out[key] = int(t.item())
    for key in ("splits", "rays_level", "ends"):
        t = torch.tensor([int(v) for v in stats[key]], dtype=torch.int64, device=dev)
        dist.all_reduce(t, group=group)
        out[key] = [int(v) for v in t.tolist()]
    for key in ("emitted", "escaped"):
        t = torch.tensor([float(v) for v in stats[key]], dtype=torch.float64, device=dev)
        dist.all_reduce(t, group=group)
        out[key] = [float(v) for v in t.tolist()]
    return out
