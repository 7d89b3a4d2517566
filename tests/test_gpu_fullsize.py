"""Parity at the sizes bench.py runs, by the protocol of SURVEY 8(d) "Oracle timing".

Configs 4 and 5 are out of the oracle's reach in full (1e11-1e12 segments per step), so
  * the TRACER is compared on a seeded 16-source subset (rates are linear in the sources), on the
    fields a free-running device run has reached at steps 0, 10 and 19 - injected into both sides;
  * the CHEMISTRY is compared on the whole 256^3 fp32 grid (every cell, strict) with the device's own rates of those
    steps handed to the oracle - the first comparison of arc_chem_kernel<float> at the size the bench runs;
  * one full-size fp32 case ends rays DEPLETED (tau_term = 0.5), which config 4 as specified never does;
  * config 5: the source nearest the centre of the 512^3 grid, and the chemistry on a 512 x 512 x 32 slab.
The oracle runs on all host cores here (gpu_common.oracle_*_parallel: the unchanged single-threaded C routine, called on
disjoint shares of the rays / cells); bench.py times it as it stands.
Tolerances: integers bit-exact; floats 1e-3 relative (fp32 fields, fp64 accumulation) + 1e-12 of the array maximum.
"""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_1807_07094_b200 import arc, workloads as wl
from gpu_common import RTOL, assert_close, compare_trace_stats, oracle_chemistry_parallel, oracle_trace_parallel

pytestmark = pytest.mark.gpu
R32 = RTOL["f32"]


def _subset_parity(w, fields, sample, what, **override):
    """both sides trace the sources `sample` alone on `fields`; -> the device's statistics"""
    Ao, so = oracle_trace_parallel(w, fields=fields, sources=sample, **override)
    with arc.Context(w, fields=fields, digest=1, **override) as cx:
        cx.set_sources(sample)
        cx.trace()
        st = cx.stats()
        compare_trace_stats(st, so, w.nb, R32)
        assert_close(cx.accum(), Ao, R32, f"{what}: A")
        G, H, Ht = cx.rates()
    Go, Ho, Hto = orc.finalize(w, Ao, fields, **{k: v for k, v in override.items() if k == "Yp"})
    assert_close(G, Go, R32, f"{what}: Gamma")
    assert_close(H, Ho, R32, f"{what}: heat per absorber")
    assert_close(Ht, Hto, R32, f"{what}: heat_total")
    return st


def _chemistry_parity(w, before, G, H, got, what):
    """the oracle's update of `before` with the DEVICE's rates against the device's updated fields `got`, every cell"""
    want, sub = oracle_chemistry_parallel(w, before, G, H, w.dt_s)
    for name, a, b in zip(("x_HI", "x_HeI", "x_HeII", "T"), got[1:], want[1:]):
        assert_close(a, b, R32, f"{what}: {name}")
    return sub


def test_config4_sixteen_sources_and_the_whole_grid_chemistry_at_steps_0_10_19():
    w = wl.config4()
    rng = np.random.default_rng(wl.SEED0 + 416)
    sample = np.sort(rng.choice(w.nsrc, size=16, replace=False))
    checked = 0
    with arc.Context(w) as cx:                                   # the benched launch configuration, free running
        for step in range(20):
            if step in (0, 10, 19):
                before = cx.get_fields()                         # fp32 arrays: what both sides start this step from
                cx.trace(step)
                st = cx.stats()
                assert_close(st["absorbed"] + st["escaped"], st["emitted"], 1e-10, f"step {step}: conservation")
                G, H, _ = cx.rates()
                cx.update_chemistry()
                got = cx.get_fields()
                st2 = cx.stats()
                sub = _chemistry_parity(w, before, G, H, got, f"step {step}, 256^3 chemistry with the device's rates")
                tot = int(sub.sum())
                assert abs(st2["subcycles"] - tot) <= max(16, tot // 10000), (st2["subcycles"], tot)
                assert st2["max_subcycles_cell"] == int(sub.max())
                del G, H, got
                _subset_parity(w, before, sample, f"step {step}, 16 sources")
                checked += 1
            else:
                cx.trace(step); cx.update_chemistry()
        xe = 1.0 - float(np.mean(cx.get_fields()[1].astype(np.float64)))
    assert checked == 3 and xe > 0.05                            # the box really ionised over the run


def test_config4_sixteen_sources_with_rays_that_deplete():
    """tau_term = 0.5 on the neutral step-0 fields: a third of the rays end DEPLETED on their way through the box (config 4
    as specified never gets there: the optical depth of its hardest bin across the box stays below 2, far from
    tau_term = 30) - the depleted branch of arc_trace_kernel<4, float> at full size"""
    w = wl.config4()
    rng = np.random.default_rng(wl.SEED0 + 417)
    sample = np.sort(rng.choice(w.nsrc, size=16, replace=False))
    st = _subset_parity(w, w.fields(), sample, "tau_term = 0.5", tau_term=0.5)
    assert st["ends"][arc.ARC_END_DEPLETED] > 0.25 * (st["ends"][1] + st["ends"][2])
    assert_close(st["absorbed"] + st["escaped"], st["emitted"], 1e-10, "conservation with depletion")


def test_config5_512_central_source_and_slab_chemistry():
    w = wl.config5(N=512, nsrc=1024)
    N = w.N
    g = w.src_pos_cm / (w.box_cm / N)
    s = int(np.argmin(np.sum((g - 0.5 * N) ** 2, axis=1)))       # the source nearest the centre: its rays cross half the box
    assert np.all(np.abs(g[s] - 0.5 * N) < 0.2 * N)
    Ao, so = oracle_trace_parallel(w, sources=np.array([s]), threads=8)
    import torch
    with arc.Context(w, digest=1) as cx:
        cx.set_sources(np.array([s]))
        cx.trace()
        compare_trace_stats(cx.stats(), so, w.nb, R32)
        A = torch.empty((w.ncell, w.nb), dtype=torch.float64, device="cuda")
        arc.arc_get_accum(cx.ctx, A)
        assert_close(A.cpu().numpy(), Ao, R32, "512^3 central source: A")
        del A, Ao
    # chemistry: all 1024 sources on the device, then the update of the slab iz in [240, 272) against the oracle
    lo, hi = 240 * N * N, 272 * N * N
    with arc.Context(w) as cx:
        cx.trace()
        rates = [torch.empty(w.ncell, dtype=torch.float64, device="cuda") for _ in range(6)]
        arc.arc_get_rates(cx.ctx, *rates)
        G = np.stack([r[lo:hi].cpu().numpy() for r in rates[:3]]); H = np.stack([r[lo:hi].cpu().numpy() for r in rates[3:]])
        del rates
        cx.update_chemistry()
        got = [a[lo:hi] for a in cx.get_fields()]
    before = [np.asarray(a)[lo:hi] for a in w.fields()]
    want, sub = oracle_chemistry_parallel(w, before, G, H, w.dt_s)      # 2^23 cells, in chunks of 64^3
    for name, a, b in zip(("x_HI", "x_HeI", "x_HeII", "T"), got[1:], want[1:]):
        assert_close(a, b, R32, f"512^3 slab chemistry: {name}")
    assert sub.max() > 1



def test_largest_grid_1024_cubed_per_ray_sequences():
    """N = 1024 is the largest grid the library takes (10 bits per cell coordinate in the tracer, cell indices up to
    2^30 - 1; the paper's production size): 12 root rays that never split (l0 = Lmax = 0) from a source next to
    the far corner, so that rays run the whole length of the box through coordinates 0 and 1023 and through the highest cell
    indices - per-ray cell sequences bit-exact against the oracle, accumulators and rates within the fp32 bar.  One bin,
    fp32 fields: 96 GB of the 180 GB on the device."""
    import dataclasses
    import torch
    from gpu_common import gpu_raylog_to_dict
    N = 1024
    n = N ** 3
    w0 = wl.config2(8, dtype="f32")
    box = w0.box_cm
    pos = (np.array([[1000, 1010, 1021]]) + 0.5) * (box / N)
    w = dataclasses.replace(w0, name="grid1024", N=N, n_H=np.full(n, 1e-3, np.float32), x_HI=np.full(n, 2e-2, np.float32),
                            x_HeI=np.ones(n, np.float32), x_HeII=np.zeros(n, np.float32), T=np.full(n, 1e4, np.float32),
                            src_pos_cm=pos, params=dict(w0.params, l0=0, Lmax=0, tau_term=float("inf")))
    w.x_HI[:: 7] = 0.5                                             # (not uniform: every 7th cell is 25 times as opaque)
    Ao, so, rl = orc.trace(w, log=True, cap_rays=64, cap_cells=100_000)
    want = orc.raylog_to_dict(rl)
    assert so["rays"] == 12 and so["segments"] > 3000 and max(len(c) for c, _ in want.values()) > 2000
    cells = np.concatenate([np.array(c) for c, _ in want.values()])
    assert cells.max() > 2 ** 30 - 2 ** 21 and cells.min() < 2 ** 27     # both ends of the index range are visited
    with arc.Context(w, digest=1) as cx:
        key, seq, cell = cx.trace_debug(cap=int(so["segments"] + so["rays"]) + 16)
        st = cx.stats()
        A = torch.empty((n, 1), dtype=torch.float64, device="cuda")
        arc.arc_get_accum(cx.ctx, A)
        G = torch.empty(n, dtype=torch.float64, device="cuda")
        arc.arc_get_rates(cx.ctx, Gamma_HI=G)
    assert gpu_raylog_to_dict(key, seq, cell) == want
    compare_trace_stats(st, so, 1, R32)
    hit = np.unique(cells)
    A_h = A[:, 0].cpu().numpy()
    assert_close(A_h[hit], Ao[hit, 0], R32, "1024^3: A in the visited cells")
    # nothing outside the visited cells (a visited cell may hold exactly 0: the tied diagonal rays cross it in a zero-length segment)
    assert np.count_nonzero(A_h) == np.count_nonzero(Ao[:, 0]) <= len(hit) and np.count_nonzero(A_h[hit]) == np.count_nonzero(A_h)
    V = (box / N) ** 3
    G_want = Ao[hit, 0] / (V * (w.n_H[hit].astype(np.float64) * w.x_HI[hit].astype(np.float64)))     # Eq. 1, one absorber, one bin
    assert_close(G.cpu().numpy()[hit], G_want, R32, "1024^3: Gamma_HI in the visited cells")
    for bad in (1025, 2048):
        with pytest.raises(arc.ArcError) as e:
            arc.arc_create_grid(bad, box, arc.ARC_F32)
        assert e.value.code == arc.ARC_EINVAL
