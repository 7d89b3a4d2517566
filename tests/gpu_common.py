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
    # escaped: the protocol's absolute floor is 1e-12 of the array's scale - for the photon tallies that scale is what
    # the sources emit (an opaque box lets e^-hundreds of it out: 1e-68 against 0 is not a difference)
    scale = float(np.max(np.abs(os_["emitted"]))) if len(os_["emitted"]) else 0.0
    e_g, e_o = np.asarray(gs["escaped"], dtype=np.float64), np.asarray(os_["escaped"], dtype=np.float64)
    bad = np.abs(e_g - e_o) > rtol * np.maximum(np.abs(e_g), np.abs(e_o)) + 1e-12 * scale
    assert not bad.any(), f"escaped: gpu={e_g} oracle={e_o} (emitted {os_['emitted']})"


def run_gpu_trace(w, fields=None, **override):
    """-> (A, stats, (Gamma, heat, heat_total)) from the CUDA path with the digest on."""
    override.setdefault("digest", 1)
    with arc.Context(w, fields=fields, **override) as cx:
        cx.trace()
        return cx.accum(), cx.stats(), cx.rates()


def oracle_override(override):
    return {k: v for k, v in override.items() if k not in ("digest", "async", "trace_blocks", "deposit")}


# ---- the oracle on all host cores (tests only; bench.py times it as it stands, single-threaded) -------------------------
def oracle_trace_parallel(w, fields=None, sources=None, threads=None, **override):
    """orc.trace of `sources` (default: all), spread over host threads by (source, root pixel): every job traces ALL the
    listed sources with an emission mask (orc_trace_masked) that leaves open only its share of the root rays,
    so source ids - and with them the per-ray digests - are those of the one-call trace.  Rays are independent and the
    accumulators add: A and the float tallies are summed, integer tallies added, digests added mod 2^64.
    The C oracle itself is untouched and single-threaded; ctypes releases the GIL.  -> (A, stats)"""
    import os
    from concurrent.futures import ThreadPoolExecutor
    threads = threads or min(16, os.cpu_count() or 1)
    src = np.arange(w.nsrc) if sources is None else np.asarray(sources)
    l0 = int(override.get("l0", w.params["l0"]))
    npix0 = 12 << (2 * l0)
    units = [(s, p) for s in range(len(src)) for p in range(npix0)]
    njobs = min(threads, len(units))
    kappa = orc.opacity(w, fields, **{k: v for k, v in override.items() if k in ("Yp",)})
    masks = []
    for j in range(njobs):
        m = np.ones((w.nsrc, npix0), dtype=np.uint8)          # (orc.trace picks the rows of `sources` itself)
        for (s, p) in units[j::njobs]:
            m[src[s], p] = 0
        masks.append(m)

    def job(m):
        return orc.trace(w, kappa=kappa, sources=src, blocked=m, **override)[:2]

    with ThreadPoolExecutor(max_workers=njobs) as ex:
        parts = list(ex.map(job, masks))
    A = parts[0][0]
    st = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in parts[0][1].items()}
    for Ap, sp in parts[1:]:
        A += Ap
        for k in ("segments", "rays"):
            st[k] += sp[k]
        st["digest"] = (st["digest"] + sp["digest"]) & 0xFFFFFFFFFFFFFFFF
        for k in ("splits", "rays_level", "ends", "emitted", "absorbed", "escaped"):
            st[k] = st[k] + sp[k]
    return A, st


def oracle_chemistry_parallel(w, fields, Gamma, heat, dt, threads=None, chunk=64 ** 3, **override):
    """orc.chemistry over a flat range of cells (the whole grid, or a slab of it) on all host cores: the update is per cell
    (PAPER.md:156), so the arrays are cut into chunks of `chunk` = 64^3 cells, each handed to the unchanged C routine
    as a 64^3 'grid'.  -> (new fields tuple, subcycles[cells])"""
    import os
    import dataclasses
    from concurrent.futures import ThreadPoolExecutor
    threads = threads or min(16, os.cpu_count() or 1)
    nc = len(fields[0])
    assert nc % chunk == 0 and round(chunk ** (1 / 3)) ** 3 == chunk
    wc = dataclasses.replace(w, N=round(chunk ** (1 / 3)))
    f = [np.ascontiguousarray(np.asarray(a, dtype=np.float64)) for a in fields]
    G = np.asarray(Gamma, dtype=np.float64); H = np.asarray(heat, dtype=np.float64)
    out = [a.copy() for a in f]
    sub = np.zeros(nc, dtype=np.int32)

    def job(i):
        sl = slice(i * chunk, (i + 1) * chunk)
        nf, sb = orc.chemistry(wc, [a[sl] for a in f], np.ascontiguousarray(G[:, sl]), np.ascontiguousarray(H[:, sl]), dt, **override)
        for k in range(1, 5):
            out[k][sl] = nf[k]
        sub[sl] = sb

    with ThreadPoolExecutor(max_workers=threads) as ex:
        list(ex.map(job, range(nc // chunk)))
    return tuple(out), sub
