"""GPU-vs-oracle parity of the geometric correction (Eq. 2-3), through the C ABI.
The nearest-face choice decides which cell receives photons, so the accumulators must agree cell by cell to the
floating-point tolerance - a differing choice would show up as an O(1) error in two cells."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_1807_07094_b200 import arc, workloads as wl
from gpu_common import RTOL, assert_close, compare_trace_stats, run_gpu_trace

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("N,nsrc,nb,dtype,l0,seed", [
    (8, 2, 1, "f64", 0, 31), (12, 3, 2, "f32", 1, 32), (16, 2, 3, "f64", 1, 33), (16, 4, 4, "f32", 0, 34),
    (11, 2, 5, "f64", 1, 35), (9, 3, 8, "f32", 1, 36), (24, 2, 4, "f32", 2, 37),
])
@pytest.mark.parametrize("mode", [arc.ARC_GEOM_FC, arc.ARC_GEOM_FC_SECONDARY, arc.ARC_GEOM_FC2])
def test_tiny_workloads_accumulators_and_rates(N, nsrc, nb, dtype, l0, seed, mode):
    w = wl.tiny(N=N, nsrc=nsrc, nb=nb, seed=seed, dtype=dtype, l0=l0, kappa_scale=15.0)
    A, st, (G, H, Ht) = run_gpu_trace(w, geom_corr=mode)
    Ao, so, _ = orc.trace(w, geom_corr=mode)
    compare_trace_stats(st, so, nb, RTOL[dtype])              # traversal untouched; absorbed/escaped totals
    assert_close(A, Ao, RTOL[dtype], "A")
    Go, Ho, Hto = orc.finalize(w, Ao)
    assert_close(G, Go, RTOL[dtype], "Gamma")
    assert_close(Ht, Hto, RTOL[dtype], "heat_total")
    lost = 1 - (st["absorbed"] + st["escaped"])[:nb] / st["emitted"][:nb]
    if mode == arc.ARC_GEOM_FC_SECONDARY:
        assert np.all(np.abs(lost) < 1e-10)                   # Eq. 3 conserves photons
    else:
        assert np.all(lost > 0)


def test_axis_ray_closed_form_on_the_gpu():
    """the hand-worked case of tests/test_oracle_geom.py (source at a cell centre, +x ray through cell centres)"""
    import math
    N, kc = 16, 0.37
    w = wl.config1(N)
    c = N // 2
    w.src_pos_cm[:] = (np.array([c, c, c]) + 0.5) * (w.box_cm / N)
    w.sig_HI[:] = kc / (1e-3 * (w.box_cm / N))
    w.params.update(l0=0, Lmax=0, tau_term=math.inf)
    A, _, _ = run_gpu_trace(w, geom_corr=arc.ARC_GEOM_FC_SECONDARY)
    A = A.reshape(N, N, N)
    S, w0 = float(w.src_Ndot[0]) / 12.0, math.sqrt(4 * math.pi / 12)
    a = lambda k: S * (math.exp(-kc * (k - 0.5)) - math.exp(-kc * (k + 0.5)))
    f = lambda k: 1.0 if 1.0 >= k * w0 else 0.5 + 0.5 / (k * w0)
    for k in range(2, N - c - 1):
        expect = f(k) * a(k) + (1 - f(k + 1)) * a(k + 1)
        assert abs(A[c, c, c + k] - expect) <= 1e-9 * expect, k


def test_config1_steps_with_the_papers_correction():
    """config 1 stepped with the paper's chosen mode (f_c + secondary), the oracle's fields injected each step"""
    w = wl.config1()
    fields = tuple(np.array(a, dtype=np.float64) for a in w.fields())
    with arc.Context(w, digest=1, geom_corr=arc.ARC_GEOM_FC_SECONDARY) as cx:
        for step in range(4):
            ref = orc.step(w, fields, geom_corr=2)
            cx.set_fields(fields)
            cx.trace(step)
            st = cx.stats()
            assert st["digest"] == ref["stats"]["digest"] and st["segments"] == ref["stats"]["segments"]
            assert_close(cx.accum(), ref["A"], RTOL["f64"], f"A step {step}")
            G, H, Ht = cx.rates()
            assert_close(G, ref["Gamma"], RTOL["f64"], f"Gamma step {step}")
            cx.update_chemistry()
            assert_close(cx.get_fields()[1], ref["fields"][1], RTOL["f64"], f"x_HI step {step}")
            fields = ref["fields"]


def test_config4_subset_fp32_with_correction():
    """full-size grid (256^3, fp32 fields, 4 bins), 2 of the 1024 sources, the configuration bench.py launches"""
    w = wl.config4()
    idx = np.array([0, 517])
    kap = orc.opacity(w)
    Ao, so, _ = orc.trace(w, kappa=kap, sources=idx, geom_corr=2)
    with arc.Context(w, digest=1, geom_corr=arc.ARC_GEOM_FC_SECONDARY) as cx:
        cx.set_sources(idx)
        cx.trace()
        st = cx.stats()
        A = cx.accum()
    compare_trace_stats(st, so, w.nb, RTOL["f32"])
    assert_close(A, Ao, RTOL["f32"], "A")


def test_geom_needs_auto_deposit():
    w = wl.tiny(N=8, nsrc=1, nb=2, seed=1, dtype="f64")
    with pytest.raises(arc.ArcError):
        arc.Context(w, geom_corr=arc.ARC_GEOM_FC, deposit=arc.ARC_DEPOSIT_RED)
