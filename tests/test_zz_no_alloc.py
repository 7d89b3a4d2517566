"""arc_pix2vec_noalloc (include/arc.h; csrc/arc_noalloc.cu): the device HEALPix generator for callers that cannot call
cudaMalloc - its device staging is one fixed file-scope array (4096 pairs = 128 KiB) instead of the three buffers that
arc_pix2vec allocates and frees on every call.  Its output must equal the existing path's - bit for bit, the bar of
tests/test_gpu_parity.py::test_pix2vec_bit_exact_* (contract C1-C2 makes directions exact) - on two calls in a row that
share the array, the second smaller than the first so that the first call's contents are still lying behind it.

This file is named so that pytest collects it last: the suite runs with `pytest -x`."""
import ctypes

import numpy as np
import pytest

from paper_1807_07094_b200 import arc

pytestmark = pytest.mark.gpu


def _pairs(n, seed):
    rng = np.random.default_rng(seed)
    level = rng.integers(0, 15, n).astype(np.int32)
    pix = (rng.random(n) * (12 * 4.0 ** level)).astype(np.uint64).astype(np.uint32)
    pix = np.minimum(pix, (12 * 4 ** level.astype(np.int64) - 1).astype(np.uint32))
    return level, pix


def test_no_alloc_entry_point_equals_the_existing_path_on_two_calls_in_a_row():
    nmax = arc.arc_pix2vec_noalloc_max()
    assert nmax == 4096
    # call 1: the maximum size;  call 2: fewer, other pixels - entries 1000 .. 4095 of the array still hold call 1's
    for n, seed in ((nmax, 1807), (1000, 7094)):
        level, pix = _pairs(n, seed)
        want = arc.arc_pix2vec(level, pix)                      # the existing path (cudaMalloc / cudaFree per call)
        out = np.full((n + 5, 3), -7.0)                          # caller-owned output; 5 guard rows behind it
        got = arc.arc_pix2vec_noalloc(level, pix, out=out)
        assert got is out
        assert np.array_equal(out[:n].view(np.uint64), want.view(np.uint64)), f"n = {n}: not bit-identical to arc_pix2vec"
        assert np.all(out[n:] == -7.0)                           # nothing written behind the n results
        assert np.allclose(np.linalg.norm(out[:n], axis=1), 1.0, atol=1e-15)
    # the same inputs again give the same bits (the array's old contents play no part)
    level, pix = _pairs(1000, 7094)
    again = arc.arc_pix2vec_noalloc(level, pix)
    assert np.array_equal(again.view(np.uint64), want.view(np.uint64))


def test_no_alloc_entry_point_rejects_what_does_not_fit_and_allocates_nothing():
    import torch
    nmax = arc.arc_pix2vec_noalloc_max()
    level, pix = _pairs(nmax + 1, 3)
    with pytest.raises(arc.ArcError) as e:
        arc.arc_pix2vec_noalloc(level, pix)
    assert e.value.code == arc.ARC_EINVAL and str(nmax) in str(e.value) and "split the call" in str(e.value)
    with pytest.raises(arc.ArcError) as e:
        arc.arc_pix2vec_noalloc(np.array([2], np.int32), np.array([12 * 16], np.uint32))      # level 2 has pixels 0 .. 191
    assert e.value.code == arc.ARC_EINVAL
    assert arc.arc_pix2vec_noalloc(np.zeros(0, np.int32), np.zeros(0, np.uint32)).shape == (0, 3)
    # no device allocation: free device memory is the same before and after a run of calls (cudaMemGetInfo counts
    # cudaMalloc'd memory of the whole process; the first call has already taken the symbol's address above)
    level, pix = _pairs(nmax, 11)
    out = np.zeros((nmax, 3))
    arc.arc_pix2vec_noalloc(level, pix, out=out)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(50):
        arc.arc_pix2vec_noalloc(level, pix, out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    # and the library's entry point is really the one bound (not a Python-side stand-in)
    assert isinstance(arc.lib().arc_pix2vec_noalloc, ctypes._CFuncPtr)
