"""GPU-vs-oracle parity of anisotropic emission (arc_set_emission_mask)."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_1807_07094_b200 import arc, workloads as wl
from gpu_common import RTOL, assert_close, compare_trace_stats, gpu_raylog_to_dict

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("N,nsrc,nb,dtype,l0,seed,frac", [
    (10, 3, 2, "f64", 0, 51, 0.5), (16, 4, 4, "f32", 1, 52, 0.3), (12, 2, 3, "f64", 2, 53, 0.9), (8, 2, 1, "f32", 1, 54, 1.0),
])
def test_masked_sources_per_ray(N, nsrc, nb, dtype, l0, seed, frac):
    w = wl.tiny(N=N, nsrc=nsrc, nb=nb, seed=seed, dtype=dtype, l0=l0, kappa_scale=20.0)
    rng = np.random.default_rng(seed)
    blocked = (rng.random((nsrc, 12 << (2 * l0))) < frac).astype(np.uint8)
    Ao, so, rl = orc.trace(w, log=True, blocked=blocked)
    want = orc.raylog_to_dict(rl)
    with arc.Context(w, digest=1) as cx:
        cx.set_emission_mask(blocked)
        key, seq, cell = cx.trace_debug(cap=int(so["segments"] + so["rays"]) + 16)
        st = cx.stats()
        A = cx.accum()
        assert gpu_raylog_to_dict(key, seq, cell) == want
        compare_trace_stats(st, so, nb, RTOL[dtype])
        assert_close(A, Ao, RTOL[dtype], "A")
        # clearing the mask gives the isotropic source back
        cx.set_emission_mask(None)
        cx.trace()
        A0o, s0o, _ = orc.trace(w)
        compare_trace_stats(cx.stats(), s0o, nb, RTOL[dtype])
        assert_close(cx.accum(), A0o, RTOL[dtype], "A isotropic")


def test_mask_level_must_match_l0():
    w = wl.tiny(N=8, nsrc=1, nb=1, seed=2, dtype="f64", l0=1)
    with arc.Context(w) as cx:
        with pytest.raises(arc.ArcError):
            cx.set_emission_mask(np.zeros((1, 12), np.uint8), level=0)


def test_config4_subset_with_chimneys():
    """full-size grid, 2 sources, 75 % of the root rays blocked"""
    w = wl.config4()
    idx = np.array([1, 900])
    rng = np.random.default_rng(9)
    blocked = np.zeros((w.nsrc, 48), np.uint8)
    blocked[idx] = (rng.random((2, 48)) < 0.75)
    Ao, so, _ = orc.trace(w, sources=idx, blocked=blocked)
    with arc.Context(w, digest=1) as cx:
        cx.set_sources(idx)
        cx.set_emission_mask(blocked[idx])
        cx.trace()
        compare_trace_stats(cx.stats(), so, w.nb, RTOL["f32"])
        assert_close(cx.accum(), Ao, RTOL["f32"], "A")
