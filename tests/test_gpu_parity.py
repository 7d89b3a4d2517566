"""GPU-vs-oracle parity (the first gate).  Everything here goes through the C ABI (ctypes binding).

Bar (BASELINE.json north_star): per-ray visited-cell sequences, split counts, ray/segment counts, end
reasons and the order-independent traversal digest: BIT-EXACT.  Per-cell accumulators, rates and updated
fractions: 1e-5 relative (fp64 fields) / 1e-3 (fp32 fields, fp64 accumulation), plus 1e-12 of the array
maximum as an absolute floor (SURVEY 8(c) parity protocol).
"""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_1807_07094_b200 import arc, workloads as wl
from gpu_common import (RTOL, assert_close, compare_trace_stats, gpu_raylog_to_dict, oracle_override,
                        run_gpu_trace)

pytestmark = pytest.mark.gpu


# ---------------------------------------------------------------------------------------------- a4
@pytest.mark.parametrize("level", [0, 1, 2, 3, 4, 5])
def test_pix2vec_bit_exact_all_pixels(level):
    npix = 12 << (2 * level)
    pix = np.arange(npix, dtype=np.uint32)
    got = arc.arc_pix2vec(np.full(npix, level, np.int32), pix)
    want = np.array([orc.pix2vec(level, int(p)) for p in pix])
    assert np.array_equal(got.view(np.uint64), want.view(np.uint64))


def test_pix2vec_bit_exact_deep_levels_sampled():
    rng = np.random.default_rng(11)
    lv, px = [], []
    for level in range(6, 15):
        npix = 12 << (2 * level)
        p = rng.integers(0, npix, 400, dtype=np.uint64)
        p[:4] = [0, npix - 1, npix // 2, npix // 3]
        lv += [level] * len(p); px += p.tolist()
    got = arc.arc_pix2vec(np.array(lv, np.int32), np.array(px, np.uint32))
    want = np.array([orc.pix2vec(l, p) for l, p in zip(lv, px)])
    assert np.array_equal(got.view(np.uint64), want.view(np.uint64))


# ---------------------------------------------------------------------------------------------- a3-a9
def _trace_both(w, log=False, **override):
    A, st, rates = run_gpu_trace(w, **override)
    oo = oracle_override(override)
    Ao, so, rl = orc.trace(w, log=log, **oo)
    return (A, st, rates), (Ao, so, rl)


def test_config1_per_ray_cell_sequences_bit_exact():
    w = wl.config1()
    Ao, so, rl = orc.trace(w, log=True)
    want = orc.raylog_to_dict(rl)
    with arc.Context(w, digest=1) as cx:
        key, seq, cell = cx.trace_debug(cap=int(so["segments"] + so["rays"]) + 16)
        st = cx.stats()
        A = cx.accum()
    got = gpu_raylog_to_dict(key, seq, cell)
    assert got.keys() == want.keys()
    for k in want:
        assert got[k] == want[k], f"ray {k}: cells/end differ"
    compare_trace_stats(st, so, w.nb, RTOL["f64"])
    assert_close(A, Ao, RTOL["f64"], "A")


@pytest.mark.parametrize("N,nsrc,nb,dtype,l0,seed", [
    (8, 2, 2, "f64", 0, 7), (8, 3, 1, "f32", 1, 8), (12, 2, 3, "f64", 1, 9), (16, 4, 4, "f32", 0, 10),
    (20, 3, 5, "f64", 2, 12), (9, 2, 8, "f32", 1, 13), (7, 5, 6, "f64", 0, 14), (13, 1, 7, "f64", 1, 15),
])
@pytest.mark.parametrize("deposit", [arc.ARC_DEPOSIT_RED, arc.ARC_DEPOSIT_AGG, arc.ARC_DEPOSIT_QUAD])
def test_tiny_random_workloads_per_ray_and_rates(N, nsrc, nb, dtype, l0, seed, deposit):
    """off-centre sources at arbitrary positions, random fields, ragged sizes; every bin count 1..8 (odd counts
    exercise the padded accumulator record); every deposit route of the tracer"""
    w = wl.tiny(N=N, nsrc=nsrc, nb=nb, seed=seed, dtype=dtype, l0=l0, kappa_scale=30.0)
    Ao, so, rl = orc.trace(w, log=True)
    want = orc.raylog_to_dict(rl)
    with arc.Context(w, digest=1, deposit=deposit) as cx:
        key, seq, cell = cx.trace_debug(cap=int(so["segments"] + so["rays"]) + 16)
        st = cx.stats()
        A = cx.accum()
        G, H, Ht = cx.rates()
    got = gpu_raylog_to_dict(key, seq, cell)
    assert got == want
    compare_trace_stats(st, so, nb, RTOL[dtype])
    assert_close(A, Ao, RTOL[dtype], "A")
    Go, Ho, Hto = orc.finalize(w, Ao)
    assert_close(G, Go, RTOL[dtype], "Gamma")
    assert_close(H, Ho, RTOL[dtype], "heat")
    assert_close(Ht, Hto, RTOL[dtype], "heat_total")


@pytest.mark.parametrize("override", [dict(tau_term=float("inf")), dict(Lmax=1, l0=1), dict(Phi=1.0), dict(Phi=7.5, l0=2),
                                      dict(tau_term=0.5)])
def test_parameter_variants(override):
    w = wl.tiny(N=16, nsrc=3, nb=3, seed=21, dtype="f64", kappa_scale=20.0)
    (A, st, _), (Ao, so, _) = _trace_both(w, **override)
    compare_trace_stats(st, so, w.nb, RTOL["f64"])
    assert_close(A, Ao, RTOL["f64"], "A")


def test_photon_conservation_on_device():
    """emitted = absorbed + escaped per bin (PAPER.md:81-86 'photon conserving')"""
    for w in (wl.config1(), wl.tiny(N=16, nsrc=4, nb=4, seed=5, dtype="f32", kappa_scale=10.0)):
        A, st, _ = run_gpu_trace(w)
        assert_close(st["absorbed"] + st["escaped"], st["emitted"], 1e-10, "conservation")
        assert_close(A.sum(axis=0), st["absorbed"], 1e-12, "sum A = absorbed")


# ---------------------------------------------------------------------------------------------- edge cases
def test_no_sources_gives_zero_rates():
    w = wl.tiny(N=8, nsrc=2, nb=2, seed=3)
    with arc.Context(w) as cx:
        arc.arc_set_sources(cx.ctx, np.zeros((0, 3)), np.zeros(0), np.zeros((0, 2)))
        cx.trace()
        st = cx.stats()
        assert st["segments"] == 0 and st["rays"] == 0
        assert not cx.accum().any()
        G, H, Ht = cx.rates()
        assert not G.any() and not H.any() and not Ht.any()


def test_single_cell_grid():
    w = wl.tiny(N=1, nsrc=1, nb=2, seed=4, kappa_scale=1e3)
    (A, st, _), (Ao, so, _) = _trace_both(w)
    compare_trace_stats(st, so, 2, RTOL["f64"])
    assert_close(A, Ao, RTOL["f64"], "A")


def test_sources_on_faces_edges_and_corners():
    """source coordinates that are exact integers in grid units (O3 step 2 boundary rule, reading G9/G10)"""
    w = wl.tiny(N=8, nsrc=4, nb=1, seed=6, l0=1, kappa_scale=5.0)
    dx = w.box_cm / w.N
    w.src_pos_cm = np.array([[0.0, 0.0, 0.0], [4.0 * dx, 4.0 * dx, 4.0 * dx], [3.0 * dx, 2.5 * dx, 7.999 * dx],
                             [7.0 * dx, 0.0, 5.0 * dx]])
    Ao, so, rl = orc.trace(w, log=True)
    with arc.Context(w, digest=1) as cx:
        key, seq, cell = cx.trace_debug(cap=int(so["segments"] + so["rays"]) + 16)
        st = cx.stats(); A = cx.accum()
    assert gpu_raylog_to_dict(key, seq, cell) == orc.raylog_to_dict(rl)
    compare_trace_stats(st, so, 1, RTOL["f64"])
    assert_close(A, Ao, RTOL["f64"], "A")


def test_many_sources_exercise_seeding_and_queue():
    w = wl.tiny(N=24, nsrc=150, nb=2, seed=31, dtype="f32", l0=0, kappa_scale=3.0)
    (A, st, _), (Ao, so, _) = _trace_both(w)
    compare_trace_stats(st, so, 2, RTOL["f32"])
    assert_close(A, Ao, RTOL["f32"], "A")


def test_small_persistent_grid_still_exact():
    """few blocks -> deep per-warp stacks, donation through the global queue"""
    w = wl.config1(N=48)
    (A, st, _), (Ao, so, _) = _trace_both(w, trace_blocks=3, tau_term=float("inf"))
    compare_trace_stats(st, so, 1, RTOL["f64"])
    assert_close(A, Ao, RTOL["f64"], "A")


def test_four_bin_f32_three_blocks_donation_through_the_queue():
    """the benched kernel variant's shape (4 bins, fp32 fields, transposed deposit) on a grid of 3 blocks: 24 warps share
    40 sources, so most of the work travels through the donation queue.  Also the target of the compute-sanitizer runs
    (profiles/r02_sanitizers.md)."""
    w = wl.tiny(N=20, nsrc=40, nb=4, seed=33, dtype="f32", l0=1, kappa_scale=30.0)
    (A, st, _), (Ao, so, _) = _trace_both(w, trace_blocks=3)
    compare_trace_stats(st, so, 4, RTOL["f32"])
    assert_close(A, Ao, RTOL["f32"], "A")
    assert st["queue_high_water"] > 0 and st["ends"][1] > 0        # the queue was used; some rays ended DEPLETED
    A0, st0, _ = run_gpu_trace(w, trace_blocks=3, digest=0)         # the timed variant (no digest): same integers, same sums
    assert st0["segments"] == so["segments"] and np.array_equal(st0["ends"], so["ends"])
    assert_close(A0, Ao, RTOL["f32"], "A (digest off)")


def test_trace_is_repeatable_in_its_integers():
    w = wl.tiny(N=16, nsrc=4, nb=3, seed=41, dtype="f32", kappa_scale=10.0)
    with arc.Context(w, digest=1) as cx:
        cx.trace(); a = cx.stats(); A1 = cx.accum()
        cx.trace(); b = cx.stats(); A2 = cx.accum()
    assert a["digest"] == b["digest"] and a["segments"] == b["segments"]
    assert_close(A1, A2, 1e-12, "A repeat")


# ---------------------------------------------------------------------------------------------- API errors
def test_api_error_behaviour():
    w = wl.tiny(N=8, nsrc=1, nb=1, seed=2)
    ctx = arc.arc_create_grid(8, w.box_cm, arc.ARC_F64)
    try:
        with pytest.raises(arc.ArcError) as e:
            arc.arc_trace(ctx)
        assert e.value.code == arc.ARC_ESTATE
        with pytest.raises(arc.ArcError) as e:
            arc.arc_set_sources(ctx, w.src_pos_cm, w.src_Ndot, w.src_binfrac)      # before the spectrum
        assert e.value.code == arc.ARC_ESTATE
        arc.arc_set_spectrum(ctx, w.E_eV, w.sig_HI, w.sig_HeI, w.sig_HeII)
        with pytest.raises(arc.ArcError) as e:
            arc.arc_set_sources(ctx, np.array([[w.box_cm, 0.0, 0.0]]), w.src_Ndot, w.src_binfrac)
        assert e.value.code == arc.ARC_EINVAL
        p = arc.arc_default_params(); p.Phi = -1.0
        with pytest.raises(arc.ArcError) as e:
            arc.arc_set_params(ctx, p)
        assert e.value.code == arc.ARC_EINVAL
        with pytest.raises(arc.ArcError) as e:
            arc.arc_update_chemistry(ctx, 1.0)
        assert e.value.code == arc.ARC_ESTATE
    finally:
        arc.arc_destroy(ctx)
    for bad in [(0, 1.0, arc.ARC_F64), (8, -1.0, arc.ARC_F64), (8, 1.0, 7)]:
        with pytest.raises(arc.ArcError) as e:
            arc.arc_create_grid(*bad)
        assert e.value.code == arc.ARC_EINVAL


def test_source_that_rounds_onto_the_upper_face_is_rejected():
    """with N not a power of two, pos just below box can give pos / (box / N) == N exactly: no cell.
    Such a position is ARC_EINVAL; the nearest position that does have a cell traces like any other."""
    N = 48
    w = wl.tiny(N=N, nsrc=1, nb=1, seed=3, dtype="f64")
    dx = w.box_cm / N
    top = np.nextafter(w.box_cm, 0.0)
    ctx = arc.arc_create_grid(N, w.box_cm, arc.ARC_F64)
    try:
        arc.arc_set_spectrum(ctx, w.E_eV, w.sig_HI, w.sig_HeI, w.sig_HeII)
        x = top
        rejected = 0
        for _ in range(64):                               # walk down from the face until the quotient drops below N
            pos = np.array([[x, 0.5 * w.box_cm, 0.5 * w.box_cm]])
            if x / dx >= N:
                with pytest.raises(arc.ArcError) as e:
                    arc.arc_set_sources(ctx, pos, w.src_Ndot, w.src_binfrac)
                assert e.value.code == arc.ARC_EINVAL
                rejected += 1
                x = np.nextafter(x, 0.0)
            else:
                arc.arc_set_sources(ctx, pos, w.src_Ndot, w.src_binfrac)
                break
        assert int(np.floor(x / dx)) == N - 1
    finally:
        arc.arc_destroy(ctx)
    w.src_pos_cm = np.array([[x, 0.5 * w.box_cm, 0.5 * w.box_cm]])
    (A, st, _), (Ao, so, _) = _trace_both(w)
    compare_trace_stats(st, so, 1, RTOL["f64"])
    assert_close(A, Ao, RTOL["f64"], "A (source in the last cell, next to the face)")


def test_division_by_reciprocal_is_the_ieee_quotient():
    """the identity the bit-exact traversal rests on (DESIGN.md 6.2 step 1, contract C3): 2^31 device-generated (a, d)
    pairs in the ranges of the march, including divisors at and just below powers of two - not one differing bit"""
    assert arc.arc_selftest_division(1 << 31, seed=180707094) == 0
    assert arc.arc_selftest_division(1 << 24, seed=7) == 0
    assert arc.arc_selftest_division(0) == 0


def test_kernel_launches_are_counted():
    w = wl.config1()
    with arc.Context(w) as cx:
        n0 = cx.stats()["kernel_launches"]
        cx.trace(); cx.update_chemistry()
        n1 = cx.stats()["kernel_launches"]
    assert n0 == 0 and n1 == 5          # queue reset (first trace only), opacity + zero + reset, tracer, finalize, chemistry


def test_ray_log_overflow_is_reported():
    w = wl.config1()
    with arc.Context(w) as cx:
        with pytest.raises(arc.ArcError) as e:
            cx.trace_debug(cap=100)
        assert e.value.code == arc.ARC_EOVERFLOW


def test_device_pointers_and_stream():
    """fields handed over as torch CUDA tensors on a non-default stream; rates read through arc_rates"""
    import ctypes
    import torch
    w = wl.tiny(N=16, nsrc=2, nb=2, seed=51, dtype="f32", kappa_scale=10.0)
    Ao, so, _ = orc.trace(w)
    Go, _, _ = orc.finalize(w, Ao)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        dev = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in w.fields()]
    s.synchronize()
    with arc.Context(w, fields=dev, stream=s.cuda_stream, digest=1) as cx:
        r = cx.trace()
        st = cx.stats()
        G_HI = torch.empty(w.ncell, dtype=torch.float64, device="cuda")
        arc.arc_get_rates(cx.ctx, Gamma_HI=G_HI)
        arc.arc_synchronize(cx.ctx)
        assert r.Gamma_HI is not None and r.heat_total is not None
        assert st["digest"] == so["digest"]
        assert_close(G_HI.cpu().numpy(), Go[0], RTOL["f32"], "Gamma_HI (device copy)")
