"""Helpers for the `-m gpu` parity tests: run the CUDA path (through the C ABI binding) and the CPU
oracle on the same Workload and compare.  The two sides share only the Workload object."""
from __future__ import annotations

import numpy as np

from oracle import oracle as orc
from paper_1807_07094_b200 import arc

RTOL = {"f64": 1e-5, "f32": 1e-3}      # BASELINE.json north_star: fp64 fields / fp32 fields with fp64 accumulation


def assert_close(a, b, rtol, what, atol_frac=1e-12):
    """|a-b| <= rtol*max(|a|,|b|) + atol_frac*max|b|  (SURVEY 8(c) parity protocol)."""
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    assert a.shape == b.shape, f"{what}: shape {a.shape} vs {b.shape}"
    if a.size == 0:
        return
    scale = float(np.max(np.abs(b))) if b.size else 0.0
    tol = rtol * np.maximum(np.abs(a), np.abs(b)) + atol_frac * scale
    bad = np.abs(a - b) > tol
    if bad.any():
        i = int(np.argmax(np.abs(a - b) - tol))
        raise AssertionError(f"{what}: {int(bad.sum())} of {a.size} values differ; worst at flat index {i}: "
                             f"gpu={a.ravel()[i]!r} oracle={b.ravel()[i]!r}")


def gpu_raylog_to_dict(key, seq, cell):
    """(key, seq, cell) entries -> {(src, level, pix): (tuple(cells), end)}"""
    out = {}
    if len(key) == 0:                      # (every root ray blocked: no ray at all)
        return out
    order = np.lexsort((seq, key))
    key, seq, cell = key[order], seq[order], cell[order]
    bounds = np.flatnonzero(np.diff(key)) + 1
    starts = np.concatenate([[0], bounds]); stops = np.concatenate([bounds, [len(key)]])
    for a, b in zip(starts, stops):
        k = int(key[a])
        assert np.array_equal(seq[a:b], np.arange(b - a, dtype=seq.dtype)), "ray log: missing or duplicated entries"
        assert cell[b - 1] < 0, "ray log: last entry of a ray must be its end marker"
        out[(k >> 40, (k >> 32) & 0xFF, k & 0xFFFFFFFF)] = (tuple(cell[a:b - 1].tolist()), int(-1 - cell[b - 1]))
    return out


def compare_trace_stats(gs, os_, nb, rtol, check_digest=True):
    assert gs["segments"] == os_["segments"], f"segments {gs['segments']} vs {os_['segments']}"
    assert gs["rays"] == os_["rays"], f"rays {gs['rays']} vs {os_['rays']}"
    assert np.array_equal(gs["splits"], os_["splits"]), f"splits {gs['splits']} vs {os_['splits']}"
    assert np.array_equal(gs["rays_level"], os_["rays_level"])
    assert np.array_equal(gs["ends"], os_["ends"]), f"ends {gs['ends']} vs {os_['ends']}"
    if check_digest:
        assert gs["digest"] == os_["digest"], f"traversal digest {gs['digest']:#x} vs {os_['digest']:#x}"
    assert_close(gs["emitted"], os_["emitted"], 1e-14, "emitted")
    assert_close(gs["absorbed"], os_["absorbed"], max(rtol * 1e-2, 1e-9), "absorbed")
    assert_close(gs["escaped"], os_["escaped"], rtol, "escaped", atol_frac=0.0 if False else 1e-12)


def run_gpu_trace(w, fields=None, **override):
    """-> (A, stats, (Gamma, heat, heat_total)) from the CUDA path with the digest on."""
    override.setdefault("digest", 1)
    with arc.Context(w, fields=fields, **override) as cx:
        cx.trace()
        return cx.accum(), cx.stats(), cx.rates()


def oracle_override(override):
    return {k: v for k, v in override.items() if k not in ("digest", "async", "trace_blocks", "deposit")}
