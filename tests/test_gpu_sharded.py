"""Source-sharded tracing on the CUDA path (arc_trace_partial / arc_accum_device / arc_finalize; SURVEY 8(e), 8(f)-4;
PAPER.md:56, 134).  One GPU is all there is here, so the two shards of a world-size-2 job run one after the other in
two contexts and their accumulators are added in place where the all-reduce would add them; `sharded.trace_sharded`
itself runs with a one-rank NCCL group.  Compared with the oracle's trace of ALL sources."""
import os
import socket

import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_1807_07094_b200 import arc, sharded, workloads as wl
from gpu_common import RTOL, assert_close

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dtype,nb,nsrc", [("f64", 3, 5), ("f32", 4, 6), ("f64", 1, 3)])
def test_two_shards_add_up_to_the_whole_trace(dtype, nb, nsrc):
    w = wl.tiny(N=16, nsrc=nsrc, nb=nb, seed=21, dtype=dtype)
    A_o, st_o, _ = orc.trace(w)
    G_o, H_o, Ht_o = orc.finalize(w, A_o)
    shards = sharded.partition_sources(w.nsrc, 2, w.src_Ndot)
    with arc.Context(w) as c0, arc.Context(w) as c1:
        c0.set_sources(shards[0]); c1.set_sources(shards[1])
        c0.trace_partial(); c1.trace_partial()
        with pytest.raises(arc.ArcError):                      # no rates before arc_finalize
            c0.rates()
        t0, t1 = c0.accum_tensor(), c1.accum_tensor()
        ptr, n = arc.arc_accum_device(c0.ctx)
        assert t0.data_ptr() == ptr and t0.numel() == n and t0.dtype == torch.float64      # an alias, not a copy
        s0, s1 = c0.stats(), c1.stats()
        t0 += t1                                               # what the all-reduce does on rank 0
        c0.finalize()
        A = c0.accum(); G, H, Ht = c0.rates()
        absorbed = c0.stats()["absorbed"]
        with pytest.raises(arc.ArcError):                      # nothing pending any more
            c0.finalize()
    rtol = RTOL[dtype]
    assert s0["segments"] + s1["segments"] == st_o["segments"] and s0["rays"] + s1["rays"] == st_o["rays"]
    assert np.array_equal(s0["splits"] + s1["splits"], st_o["splits"]) and np.array_equal(s0["ends"] + s1["ends"], st_o["ends"])
    assert_close(s0["emitted"] + s1["emitted"], st_o["emitted"], 1e-14, "emitted")
    assert_close(s0["escaped"] + s1["escaped"], st_o["escaped"], rtol, "escaped")
    assert_close(absorbed, st_o["absorbed"], rtol, "absorbed (from the summed accumulators)")
    assert_close(A, A_o, rtol, "accumulators")
    assert_close(G, G_o, rtol, "Gamma"); assert_close(H, H_o, rtol, "heat"); assert_close(Ht, Ht_o, rtol, "heat_total")


def test_partial_plus_finalize_equals_trace_and_state_checks():
    w = wl.tiny(N=12, nsrc=3, nb=2, seed=4)
    with arc.Context(w) as cx:
        with pytest.raises(arc.ArcError):
            cx.finalize()                                      # ARC_ESTATE: no partial trace
        cx.trace()
        G1 = cx.rates()[0]; A1 = cx.accum()
        cx.trace_partial()
        cx.set_fields(w.fields())                              # new fields discard the pending accumulators
        with pytest.raises(arc.ArcError):
            cx.finalize()
        cx.trace_partial(); cx.finalize()
        G2 = cx.rates()[0]; A2 = cx.accum()
        st = cx.stats()
        cx.update_chemistry()                                  # rates are valid again
    assert_close(A2, A1, 1e-12, "accumulators"); assert_close(G2, G1, 1e-12, "Gamma")
    assert st["finalize_ms"] > 0 and st["trace_ms"] >= st["trace_kernel_ms"]


def test_trace_sharded_with_a_one_rank_nccl_group():
    import torch.distributed as dist
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK="0", WORLD_SIZE="1")
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        w = wl.tiny(N=12, nsrc=4, nb=3, seed=9, dtype="f32")
        A_o, st_o, _ = orc.trace(w)
        with arc.Context(w, stream=torch.cuda.current_stream().cuda_stream) as cx:
            cx.set_sources(sharded.partition_sources(w.nsrc, 1)[0])
            sharded.trace_sharded(cx)
            A = cx.accum()
            st = sharded.reduce_stats(cx.stats())
            # the collective really runs on the aliased accumulators: all-reduce of a one-rank group leaves them as they are
            t = cx.accum_tensor(); before = t.clone(); dist.all_reduce(t); torch.cuda.synchronize()
            assert torch.equal(t, before)
        assert st["segments"] == st_o["segments"]
        assert_close(A, A_o, RTOL["f32"], "accumulators")
    finally:
        dist.destroy_process_group()
