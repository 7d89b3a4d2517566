"""GPU-vs-oracle parity of the optically thin inner region (arc_params.thin_tau).
Radii are minima of contract-arithmetic radii: bit-exact.  With the radii injected, traversal (digest, counts) is
bit-exact and the accumulators agree to the floating-point tolerance."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_1807_07094_b200 import arc, workloads as wl
from gpu_common import RTOL, assert_close, compare_trace_stats

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("N,nsrc,nb,dtype,l0,seed,ks", [
    (12, 3, 2, "f64", 1, 61, 0.004), (16, 4, 4, "f32", 1, 62, 0.002), (20, 2, 3, "f64", 0, 63, 0.001), (10, 2, 1, "f32", 2, 64, 0.0005),
])
def test_two_traces_radii_bit_exact_and_accumulators(N, nsrc, nb, dtype, l0, seed, ks):
    w = wl.tiny(N=N, nsrc=nsrc, nb=nb, seed=seed, dtype=dtype, l0=l0, kappa_scale=ks)
    kap = orc.opacity(w)
    with arc.Context(w, digest=1, thin_tau=0.1) as cx:
        R = np.zeros(nsrc)
        for it in range(3):                                     # trace 0 finds radii; traces 1, 2 use them
            Ao, so, _ = orc.trace(w, kappa=kap, thin_tau=0.1, Rstart=R)
            assert np.array_equal(cx.thin_radii(), R)
            cx.trace(it)
            st = cx.stats()
            compare_trace_stats(st, so, nb, RTOL[dtype])
            assert_close(cx.accum(), Ao, RTOL[dtype], f"A trace {it}")
            Rn = cx.thin_radii()
            assert np.array_equal(Rn.view(np.uint64), so["R_thin"].view(np.uint64)), (it, Rn, so["R_thin"])
            R = so["R_thin"]
        assert np.any(R > 0)


def test_injected_radii_and_mask_together():
    w = wl.tiny(N=16, nsrc=3, nb=3, seed=71, dtype="f64", l0=1, kappa_scale=0.002)
    rng = np.random.default_rng(5)
    blocked = (rng.random((3, 48)) < 0.4).astype(np.uint8)
    R = np.array([0.0, 2.7, 5.1])
    Ao, so, _ = orc.trace(w, thin_tau=0.1, Rstart=R, blocked=blocked)
    with arc.Context(w, digest=1, thin_tau=0.1) as cx:
        cx.set_emission_mask(blocked)
        cx.set_thin_radii(R)
        cx.trace()
        compare_trace_stats(cx.stats(), so, 3, RTOL["f64"])
        assert_close(cx.accum(), Ao, RTOL["f64"], "A")
        assert np.array_equal(cx.thin_radii().view(np.uint64), so["R_thin"].view(np.uint64))


def test_config3_step_sequence_free_running():
    """config 3 (128^3, 16 sources, 3 bins) for three steps, fields of the oracle injected: radii grow and stay equal"""
    w = wl.config3()
    fields = tuple(np.array(a, dtype=np.float64) for a in w.fields())
    R = np.zeros(w.nsrc)
    with arc.Context(w, digest=1, thin_tau=0.1) as cx:
        for step in range(3):
            kap = orc.opacity(w, fields)
            Ao, so, _ = orc.trace(w, kappa=kap, thin_tau=0.1, Rstart=R)
            Go, Ho, _ = orc.finalize(w, Ao, fields)
            cx.set_fields(fields)
            cx.trace(step)
            st = cx.stats()
            assert st["digest"] == so["digest"] and st["segments"] == so["segments"]
            assert_close(cx.accum(), Ao, RTOL["f64"], f"A step {step}")
            assert np.array_equal(cx.thin_radii().view(np.uint64), so["R_thin"].view(np.uint64))
            R = so["R_thin"]
            fields, _ = orc.chemistry(w, fields, Go, Ho, w.dt_s)


def test_thin_needs_auto_deposit_and_no_geom():
    w = wl.tiny(N=8, nsrc=1, nb=2, seed=1, dtype="f64")
    with pytest.raises(arc.ArcError):
        arc.Context(w, thin_tau=0.1, geom_corr=arc.ARC_GEOM_FC)
    with pytest.raises(arc.ArcError):
        arc.Context(w, thin_tau=0.1, deposit=arc.ARC_DEPOSIT_RED)
