"""arc_params.async = 1 (include/arc.h, conventions): calls only enqueue; a trace that failed on the device leaves a sticky
error, every later kernel of the context skips its work, and the first synchronising call reports (and clears) it.
The failure is injected with arc_params.debug_fault - the tracer has no other way to be made to fail on demand."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_1807_07094_b200 import arc, workloads as wl
from gpu_common import RTOL, assert_close, compare_trace_stats

pytestmark = pytest.mark.gpu


def _workload():
    w = wl.tiny(N=16, nsrc=4, nb=3, seed=71, dtype="f64", kappa_scale=10.0)
    w.src_Ndot = w.src_Ndot * 1e3
    return w


def test_async_step_equals_the_synchronous_step_and_the_oracle():
    """trace + chemistry + read-backs enqueued without a host synchronisation in between: same integers as the
    synchronous path, rates and fields within the bar of the oracle"""
    import torch
    w = _workload()
    ref = orc.step(w, w.fields())
    s = torch.cuda.Stream()
    with arc.Context(w, stream=s.cuda_stream, digest=1, **{"async": 1}) as cx:
        cx.trace()                                     # returns at once
        G = [torch.empty(w.ncell, dtype=torch.float64, device="cuda") for _ in range(3)]
        H = [torch.empty(w.ncell, dtype=torch.float64, device="cuda") for _ in range(3)]
        Ht = torch.empty(w.ncell, dtype=torch.float64, device="cuda")
        arc.arc_get_rates(cx.ctx, G[0], G[1], G[2], H[0], H[1], H[2], Ht)      # device copies, all seven arrays, stream ordered
        cx.update_chemistry()
        arc.arc_synchronize(cx.ctx)                    # reports deferred errors: none
        st = cx.stats()
        got = cx.get_fields()
    compare_trace_stats(st, ref["stats"], w.nb, RTOL["f64"])
    assert_close(torch.stack(G).cpu().numpy(), ref["Gamma"], RTOL["f64"], "Gamma (async, device copy)")
    assert_close(torch.stack(H).cpu().numpy(), ref["heat"], RTOL["f64"], "heat per absorber (async, device copy)")
    assert_close(Ht.cpu().numpy(), ref["heat_total"], RTOL["f64"], "heat_total (async, device copy)")
    same, _ = orc.chemistry(w, w.fields(), torch.stack(G).cpu().numpy(), torch.stack(H).cpu().numpy(), w.dt_s)
    for n, a, b in zip(("x_HI", "x_HeI", "x_HeII", "T"), got[1:], same[1:]):
        assert_close(a, b, RTOL["f64"], f"async step: {n}")


@pytest.mark.parametrize("fault,code", [(1, arc.ARC_EOVERFLOW), (3, arc.ARC_ECUDA), (4, arc.ARC_ECUDA)])
def test_async_trace_failure_never_reaches_the_fields(fault, code):
    """an aborted trace in async mode: arc_trace and arc_update_chemistry still return OK (they only enqueue), but the
    chemistry kernel sees the device error and leaves the fields alone; the first synchronising call reports the error
    once; afterwards the context is usable again"""
    w = _workload()
    before = [np.array(a, dtype=np.float64) for a in w.fields()]
    with arc.Context(w, **{"async": 1, "debug_fault": fault}) as cx:
        cx.trace()
        cx.update_chemistry()
        with pytest.raises(arc.ArcError) as e:
            cx.get_fields()                            # host read-back synchronises and reports
        assert e.value.code == code, e.value
        after = cx.get_fields()                        # reported once; the fields are readable ...
        for a, b in zip(after, before):
            assert np.array_equal(a, b)                # ... and untouched
        with pytest.raises(arc.ArcError) as e:
            cx.rates()                                 # the rates of the aborted trace are invalid
        assert e.value.code == arc.ARC_ESTATE
        # same again, reported by arc_synchronize this time; a second trace enqueued behind a failed one does not run
        cx.trace(); cx.trace(); cx.update_chemistry()
        with pytest.raises(arc.ArcError) as e:
            arc.arc_synchronize(cx.ctx)
        assert e.value.code == code
        assert all(np.array_equal(a, b) for a, b in zip(cx.get_fields(), before))
        # fault off: the context works
        arc.arc_set_params(cx.ctx, arc.params_from_dict(w.params, **{"async": 1}))
        cx.trace(); cx.update_chemistry()
        arc.arc_synchronize(cx.ctx)
        ref = orc.step(w, w.fields())
        assert cx.stats()["segments"] == ref["stats"]["segments"]
        assert_close(cx.rates()[0], ref["Gamma"], RTOL["f64"], "Gamma after the recovered step")


def test_synchronous_trace_reports_the_injected_failure_itself():
    w = _workload()
    with arc.Context(w, debug_fault=1) as cx:
        with pytest.raises(arc.ArcError) as e:
            cx.trace()
        assert e.value.code == arc.ARC_EOVERFLOW
        with pytest.raises(arc.ArcError) as e:
            cx.update_chemistry()
        assert e.value.code == arc.ARC_ESTATE
