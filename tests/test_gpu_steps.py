"""arc_run_steps (include/arc.h): the time-step loop of PAPER.md:47-59 enqueued without a host round trip per step (one
captured CUDA graph, replayed) must compute exactly what the call-by-call loop computes."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_1807_07094_b200 import arc, workloads as wl
from gpu_common import RTOL, assert_close

pytestmark = pytest.mark.gpu


def _call_by_call(w, n, **kw):
    seg, sub = 0, 0
    with arc.Context(w, **kw) as cx:
        for i in range(n):
            cx.trace(i); cx.update_chemistry()
            st = cx.stats(); seg += st["segments"]; sub += st["subcycles"]
        return cx.get_fields(), cx.rates(), seg, sub, st


@pytest.mark.parametrize("name,n,use_stream", [("config1", 10, True), ("config1", 4, False), ("config3_64", 3, True)])
def test_run_steps_equals_the_call_by_call_loop(name, n, use_stream):
    import torch
    w = wl.config1() if name == "config1" else wl.config3(N=64)
    want_f, want_r, seg, sub, last = _call_by_call(w, n)
    s = torch.cuda.Stream() if use_stream else None             # (no stream: legacy default stream, steps enqueued one by one)
    with arc.Context(w, stream=s.cuda_stream if s else None) as cx:
        cx.run_steps(n)
        st = cx.stats()
        got_f, got_r = cx.get_fields(), cx.rates()
        # a second batch continues from where the first ended (same graph, replayed)
        cx.run_steps(2)
        st2 = cx.stats()
    assert st["segments_total"] == seg and st["subcycles_total"] == sub
    assert st["segments"] == last["segments"] and np.array_equal(st["splits"], last["splits"]) and np.array_equal(st["ends"], last["ends"])
    assert st["kernel_launches"] == 4 * n + 1                  # queue reset once; opacity + reset, tracer, finalize, chemistry per step
    assert st["steps_ms"] > 0.0 and st["trace_kernel_ms"] == 0.0
    assert st2["kernel_launches"] == 4 * (n + 2) + 1 and st2["segments_total"] > seg
    # same kernels on the same inputs: only the order of the atomic sums differs
    for a, b, what in zip(got_f[1:], want_f[1:], ("x_HI", "x_HeI", "x_HeII", "T")):
        assert_close(a, b, 1e-7, f"{name}: {what} after {n} steps", atol_frac=1e-12)
    assert_close(got_r[0], want_r[0], 1e-7, f"{name}: Gamma of the last step")


def test_run_steps_follows_the_oracle_free_running():
    w = wl.config1()
    fields = tuple(np.array(a, dtype=np.float64) for a in w.fields())
    for _ in range(w.n_steps):
        fields = orc.step(w, fields)["fields"]
    import torch
    s = torch.cuda.Stream()
    with arc.Context(w, stream=s.cuda_stream) as cx:
        cx.run_steps(w.n_steps)
        got = cx.get_fields()
    vol_o = float((1.0 - fields[1]).sum()); vol_g = float((1.0 - got[1]).sum())
    assert abs(vol_g - vol_o) <= 1e-6 * vol_o
    assert_close(got[1], fields[1], 1e-4, "x_HI after 10 graph-replayed steps", atol_frac=1e-9)


def test_run_steps_reports_a_device_error_and_leaves_the_fields_alone():
    import torch
    w = wl.config1()
    before = [np.array(a, dtype=np.float64) for a in w.fields()]
    s = torch.cuda.Stream()
    with arc.Context(w, stream=s.cuda_stream, debug_fault=1) as cx:
        with pytest.raises(arc.ArcError) as e:
            cx.run_steps(5)
        assert e.value.code == arc.ARC_EOVERFLOW
        assert all(np.array_equal(a, b) for a, b in zip(cx.get_fields(), before))
        arc.arc_set_params(cx.ctx, arc.params_from_dict(w.params))          # fault off: new graph, works
        cx.run_steps(2)
        assert cx.stats()["segments"] > 0
    with arc.Context(w, thin_tau=0.1) as cx:
        with pytest.raises(arc.ArcError) as e:
            cx.run_steps(2)
        assert e.value.code == arc.ARC_EINVAL
