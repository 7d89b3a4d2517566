"""Parity at BASELINE.json's full sizes, in the launch configuration bench.py times (default persistent grid,
default deposit route, digest off for the timed variant and on for the compared one).

Configs 2 and 3 are within the oracle's reach and are compared in full (every cell, every counter).  Configs 4
and 5 are not (1e11-1e12 segments per step at ~2e7 segments/s on one core): there the oracle traces a sampled
subset of the sources on the same fields - rates are linear in the sources - and the full
run is checked by what holds at any size: photon conservation, integer repeatability, exact additivity of the
integer statistics over a partition of the sources, and additivity of the accumulators within the float
tolerance.  Tolerances: traversal integers bit-exact; floats 1e-5 (fp64 fields) / 1e-3 (fp32 fields).
"""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_1807_07094_b200 import arc, workloads as wl
from gpu_common import RTOL, assert_close, compare_trace_stats, oracle_trace_parallel

pytestmark = pytest.mark.gpu

INT_KEYS = ("segments", "rays", "digest")
ARR_KEYS = ("splits", "rays_level", "ends")


def _one_step_both(w, cx, fields, step, rtol):
    """oracle step and CUDA step from the same fields; compares everything; -> the oracle's new fields"""
    ref = orc.step(w, fields)
    cx.set_fields(fields)
    cx.trace(step)
    st = cx.stats()
    compare_trace_stats(st, ref["stats"], w.nb, rtol)
    assert_close(cx.accum(), ref["A"], rtol, f"step {step}: A")
    G, H, Ht = cx.rates()
    assert_close(G, ref["Gamma"], rtol, f"step {step}: Gamma")
    assert_close(H, ref["heat"], rtol, f"step {step}: heat per absorber")
    assert_close(Ht, ref["heat_total"], rtol, f"step {step}: heat_total")
    cx.update_chemistry()
    got = cx.get_fields()
    for name, a, b in zip(("x_HI", "x_HeI", "x_HeII", "T"), got[1:], ref["fields"][1:]):
        assert_close(a, b, rtol, f"step {step}: {name}")
    return ref["fields"]


def test_config2_full_grid_three_steps():
    """128^3 Stromgren workload (1 source, 1 bin, fp64): every ray, every cell, 3 of the 100 steps with the oracle's
    fields injected each step (traversal depends on the fields through depletion)."""
    w = wl.config2()
    fields = tuple(np.array(a, dtype=np.float64) for a in w.fields())
    with arc.Context(w, digest=1) as cx:
        for step in range(3):
            fields = _one_step_both(w, cx, fields, step, RTOL["f64"])


def test_config2_full_run_100_steps_against_the_analytic_front():
    """BASELINE.json config 2 in full on the device: 100 steps over 5 recombination times, ionised volume against
    r_S (1 - e^{-t/t_rec})^{1/3} (Eq. 9, reading G1).  With this fixed coarse step the front lags early
     and ends within the 5 % the paper reports."""
    w = wl.config2()
    t_rec = 1.0 / (wl.ALPHA_B_1E4 * 1e-3)
    r_S = (3.0 * 5e48 / (4.0 * np.pi * wl.ALPHA_B_1E4 * 1e-6)) ** (1.0 / 3.0)
    dx = w.box_cm / w.N
    radii, ratios = [], []
    with arc.Context(w) as cx:
        for step in range(w.n_steps):
            cx.trace(step)
            cx.update_chemistry()
            if step % 10 == 9:
                st = cx.stats()
                assert_close(st["absorbed"] + st["escaped"], st["emitted"], 1e-10, "conservation")
                xe = (1.0 - cx.get_fields()[1].astype(np.float64) - 1.2e-3).clip(0)   # above the initial ionised floor
                r = (3.0 * float(xe.sum()) * dx ** 3 / (4.0 * np.pi)) ** (1.0 / 3.0)
                t = (step + 1) * w.dt_s
                radii.append(r); ratios.append(r / (r_S * (1.0 - np.exp(-t / t_rec)) ** (1.0 / 3.0)))
    assert np.all(np.diff(radii) > 0) and np.all(np.diff(ratios) > 0), ratios
    assert ratios[0] < 0.7, ratios                               # "low at early times"
    assert abs(ratios[-1] - 1.0) < 0.05, ratios                  # within 5 % ...
    assert sum(abs(q - 1.0) < 0.05 for q in ratios) >= len(ratios) // 2, ratios     # ... for the majority of the run


def test_config3_full_grid_one_step():
    """128^3 lognormal + clump, 16 sources, 3 bins, H+He, evolving T (fp64): all sources, all cells, one full step."""
    w = wl.config3()
    fields = tuple(np.array(a, dtype=np.float64) for a in w.fields())
    with arc.Context(w, digest=1) as cx:
        _one_step_both(w, cx, fields, 0, RTOL["f64"])


def _stats_ints(st):
    return {k: int(st[k]) for k in INT_KEYS} | {k: st[k].copy() for k in ARR_KEYS}


def _sampled_source_parity(w, sample, rtol, fields=None):
    """the oracle and the CUDA path each trace the sources `sample` alone on the same fields"""
    fields = fields if fields is not None else w.fields()
    Ao, so = oracle_trace_parallel(w, fields=fields, sources=sample, threads=8)      # (the unchanged oracle, on disjoint shares of the root rays)
    with arc.Context(w, fields=fields, digest=1) as cx:
        cx.set_sources(sample)
        cx.trace()
        st = cx.stats()
        compare_trace_stats(st, so, w.nb, rtol)
        assert_close(cx.accum(), Ao, rtol, "A (sampled sources)")
        G, H, Ht = cx.rates()
    Go, Ho, Hto = orc.finalize(w, Ao, fields)
    assert_close(G, Go, rtol, "Gamma (sampled sources)")
    assert_close(Ht, Hto, rtol, "heat_total (sampled sources)")


def test_config4_sampled_sources_against_the_oracle():
    """256^3, fp32 fields: 2 of the 1024 sources (the brightest and a seeded one), traced alone by both sides"""
    w = wl.config4()
    rng = np.random.default_rng(wl.SEED0 + 40)
    _sampled_source_parity(w, np.array([0, int(rng.integers(1, w.nsrc))]), RTOL["f32"])


def test_config4_full_run_properties_in_the_benched_launch_configuration():
    """all 1024 sources, default parameters (exactly what bench.py launches): conservation, repeatable integers,
    and additivity over a partition of the sources into two halves"""
    w = wl.config4()
    import torch
    dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in w.fields()]
    with arc.Context(w, fields=dev) as cx:                      # digest off: the timed kernel variant
        cx.trace()
        full = cx.stats()
        A_full = torch.empty((w.ncell, w.nb), dtype=torch.float64, device="cuda")
        arc.arc_get_accum(cx.ctx, A_full)
        assert_close(full["absorbed"] + full["escaped"], full["emitted"], 1e-10, "conservation (1024 sources)")
        cx.trace()
        again = cx.stats()
        for k in ("segments", "rays"):
            assert int(full[k]) == int(again[k]), k
        for k in ARR_KEYS:
            assert np.array_equal(full[k], again[k]), k
        bench_segments = int(full["segments"])
    with arc.Context(w, fields=dev, digest=1) as cx:
        cx.trace()
        whole = _stats_ints(cx.stats())
        assert whole["segments"] == bench_segments              # the digest variant walks the same segments
        parts, A_sum = [], torch.zeros_like(A_full)
        half = w.nsrc // 2
        for idx in (np.arange(0, half), np.arange(half, w.nsrc)):
            cx.set_sources(idx)
            cx.trace()
            parts.append(_stats_ints(cx.stats()))
            A_part = torch.empty_like(A_full)
            arc.arc_get_accum(cx.ctx, A_part)
            A_sum += A_part
        for k in ("segments", "rays"):
            assert parts[0][k] + parts[1][k] == whole[k], k
        # source ids restart at 0 in each half, so the digests (keyed by source id) differ; the first half's do not
        for k in ARR_KEYS:
            assert np.array_equal(parts[0][k] + parts[1][k], whole[k]), k
        scale = float(A_full.max())
        err = (A_sum - A_full).abs() - (RTOL["f32"] * torch.maximum(A_sum.abs(), A_full.abs()) + 1e-12 * scale)
        assert float(err.max()) <= 0.0, "accumulators are not additive over a partition of the sources"


def test_config5_512_sampled_source_against_the_oracle():
    """512^3, fp32 fields, 1024 peaks: the source nearest a box corner (most of its rays leave quickly, so the oracle
    finishes in seconds) traced alone by both sides on the full grid"""
    w = wl.config5(N=512, nsrc=1024)
    g = w.src_pos_cm / (w.box_cm / w.N)
    d = np.minimum(g, w.N - g)                                   # distance to the nearest face, per axis
    s = int(np.argmin(np.sort(d, axis=1)[:, :2].sum(axis=1)))   # close to two faces at once: near an edge/corner
    _sampled_source_parity(w, np.array([s]), RTOL["f32"])


def test_config5_transparent_state_geometry_bound_counts():
    """state (B) of config 5 at 256^3: tau_term = inf, every ray crosses the box; both sides, 1 sampled source"""
    w = wl.config5(N=256, nsrc=1024, state="transparent")
    _sampled_source_parity(w, np.array([7]), RTOL["f32"])
