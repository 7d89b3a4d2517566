"""GPU-vs-oracle parity of arc_suggest_dt, through the C ABI."""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from paper_1807_07094_b200 import arc, workloads as wl
from gpu_common import RTOL

pytestmark = pytest.mark.gpu


def _both(w, steps=1, sources=None):
    fields = tuple(np.array(a, dtype=np.float64) for a in w.fields())
    out = []
    with arc.Context(w) as cx:
        if sources is not None:
            cx.set_sources(sources)
        for s in range(steps):
            kap = orc.opacity(w, fields)
            Ao, _, _ = orc.trace(w, kappa=kap, sources=sources)
            Go, Ho, _ = orc.finalize(w, Ao, fields)
            cx.set_fields(fields)
            cx.trace(s)
            for scheme in (arc.ARC_DT_NEUTRAL, arc.ARC_DT_INTENSITY):
                for eps in (0.1, 0.03):
                    out.append((cx.suggest_dt(scheme, eps), orc.suggest_dt(w, fields, Go[0], scheme=scheme, eps=eps)))
            fields, _ = orc.chemistry(w, fields, Go, Ho, w.dt_s)
    return out


@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_tiny_workload_both_schemes(dtype):
    w = wl.tiny(N=16, nsrc=3, nb=3, seed=41, dtype=dtype, kappa_scale=40.0)
    for (dt, used), (dto, usedo) in _both(w, steps=3):
        assert used == usedo
        assert (math.isinf(dt) and math.isinf(dto)) or abs(dt / dto - 1) < RTOL[dtype]


def test_config1_front():
    w = wl.config1()
    res = _both(w, steps=3)
    assert any(u > 0 and math.isfinite(d) for (d, u), _ in res)
    for (dt, used), (dto, usedo) in res:
        assert used == usedo
        assert (math.isinf(dt) and math.isinf(dto)) or abs(dt / dto - 1) < RTOL["f64"]


def test_config4_full_grid_subset_of_sources():
    w = wl.config4()
    for (dt, used), (dto, usedo) in _both(w, steps=1, sources=np.array([3, 700])):
        assert used == usedo and used > 0
        assert abs(dt / dto - 1) < RTOL["f32"]


def test_errors():
    w = wl.tiny(N=8, nsrc=1, nb=1, seed=2, dtype="f64")
    with arc.Context(w) as cx:
        with pytest.raises(arc.ArcError):
            cx.suggest_dt()                       # no trace yet
        cx.trace()
        with pytest.raises(arc.ArcError):
            cx.suggest_dt(scheme=7)
        with pytest.raises(arc.ArcError):
            cx.suggest_dt(eps=-1.0)
