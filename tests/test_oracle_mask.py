"""Pins for anisotropic emission in the oracle: blocked root rays do not exist, the
open ones carry the mean rate per ray."""
import math

import numpy as np

from oracle import oracle as orc
from paper_1807_07094_b200 import workloads as wl


def test_single_open_ray_is_the_exact_axis_attenuation():
    N, kc = 16, 0.37
    w = wl.config1(N)
    c = N // 2
    w.src_pos_cm[:] = (np.array([c, c, c]) + 0.5) * (w.box_cm / N)
    w.sig_HI[:] = kc / (1e-3 * (w.box_cm / N))
    w.params.update(l0=0, Lmax=0, tau_term=math.inf)
    blocked = np.ones((1, 12), np.uint8)
    blocked[0, 4] = 0                                        # pixel 4 = +x
    A, st, _ = orc.trace(w, blocked=blocked)
    S = float(w.src_Ndot[0]) / 12.0
    assert abs(st["emitted"][0] / S - 1) < 1e-15 and st["rays"] == 1
    A3 = A.reshape(N, N, N)
    on_axis = np.zeros_like(A3, dtype=bool)
    on_axis[c, c, c:] = True
    assert np.all(A3[~on_axis] == 0.0)
    for k in range(1, N - c):
        expect = S * (math.exp(-kc * (k - 0.5)) - math.exp(-kc * (k + 0.5)))
        assert abs(A3[c, c, c + k] - expect) <= 1e-13 * expect
    assert abs((st["absorbed"][0] + st["escaped"][0]) / st["emitted"][0] - 1) < 1e-12


def test_mask_and_complement_add_up_to_the_isotropic_source():
    w = wl.tiny(N=12, nsrc=3, nb=2, seed=17, dtype="f64", l0=1, kappa_scale=10.0)
    rng = np.random.default_rng(1)
    blocked = (rng.random((3, 48)) < 0.4).astype(np.uint8)
    A, st, _ = orc.trace(w)
    A1, s1, _ = orc.trace(w, blocked=blocked)
    A2, s2, _ = orc.trace(w, blocked=1 - blocked)
    assert np.allclose(A1 + A2, A, rtol=1e-12, atol=1e-12 * A.max())
    assert s1["rays"] + s2["rays"] == st["rays"] and s1["segments"] + s2["segments"] == st["segments"]
    assert (s1["digest"] + s2["digest"]) % 2 ** 64 == st["digest"]
    # escape fraction: emitted = (open rays / all rays) x Ndot, per source summed
    open_frac = 1 - blocked.mean(axis=1)
    want = (w.src_Ndot * open_frac) @ w.src_binfrac
    assert np.allclose(s1["emitted"], want, rtol=1e-14)
    for s in (s1, s2):
        assert np.allclose((s["absorbed"] + s["escaped"]) / s["emitted"], 1, rtol=0, atol=1e-10)
