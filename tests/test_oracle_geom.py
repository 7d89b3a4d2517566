"""Pins for the geometric correction of the oracle (Eq. 2-3, study at :338-354; readings G25-G29):
an exact special case worked by hand (axis-aligned ray), photon conservation with the secondary correction, Eq. 3's
absorber-density ratio in the rates, and the paper's own statement of what the corrections do to the Stromgren radius
(Fig. 11)."""
import math

import numpy as np

from oracle import oracle as orc
from paper_1807_07094_b200 import workloads as wl

GOLD = dict(l.split()[:2] for l in open(__file__.rsplit("/", 1)[0] + "/golden/paper_values.txt")
            if l.strip() and not l.startswith("#"))


def _uniform(N=16, kappa_cell=0.3, l0=0, Lmax=13, tau_term=math.inf, Phi=3.0, Ndot=1e48):
    w = wl.config1(N)
    c = N // 2
    w.src_pos_cm[:] = (np.array([c, c, c]) + 0.5) * (w.box_cm / N)
    w.src_Ndot[:] = Ndot
    w.sig_HI[:] = kappa_cell / (1e-3 * (w.box_cm / N))
    w.params.update(l0=l0, Lmax=Lmax, tau_term=tau_term, Phi=Phi)
    return w


def test_axis_aligned_ray_closed_form():
    """l0 = Lmax = 0: pixel 4 runs exactly along +x through cell centres.  Segment k (k = 0 the source cell, length 1/2;
    k >= 1 length 1) has its midpoint at the cell centre for k >= 1, so D_edge = 1/2 with the x- face first in the order
    x-, x+, y-, ...; L_pix = r_mid sqrt(4 pi / 12) with r_mid = k.  Hence f_k = 1 while 1 >= L_pix, else 1/2 + 1/(2 L_pix),
    and with the secondary correction cell k receives f_k a_k + (1 - f_{k+1}) a_{k+1} (the part removed from segment k+1
    goes to its x- neighbour, cell k).  Segment 0: midpoint 1/4 from the x+ face, L_pix = 0.256: f_0 = 1."""
    N, kc = 16, 0.37
    c = N // 2
    S = 1e48 / 12.0
    w0 = math.sqrt(4 * math.pi / 12)                      # sqrt(Omega_0)
    nseg = N - c

    def a(k):                                             # absorbed in segment k, uncorrected (exact attenuation)
        lo = 0.0 if k == 0 else kc * (k - 0.5)
        return S * (math.exp(-lo) - math.exp(-kc * (k + 0.5)))

    def f(k, mode):
        if k == 0:
            return 1.0
        L = k * w0
        fk = 1.0 if 1.0 >= L else 0.5 + 0.5 / L
        return fk * fk if mode == 3 else fk

    assert f(1, 1) < 1.0 and f(1, 1) > 0.98               # the correction bites from the first full cell on
    for mode in (1, 2, 3):
        w = _uniform(N, kc, l0=0, Lmax=0)
        A, st, _ = orc.trace(w, geom_corr=mode)
        A = A.reshape(N, N, N)
        for k in range(2, nseg):                          # cells k >= 2 on the axis are touched by this ray only
            expect = f(k, mode) * a(k)
            if mode == 2 and k + 1 < nseg:
                expect += (1 - f(k + 1, 2)) * a(k + 1)
            got = A[c, c, c + k]
            assert abs(got - expect) <= 1e-12 * expect, (mode, k, got, expect)
    # the same along -y (pixel 7): the y- face comes third in the order, but x- (D = 1/2 as well) is first: the removed
    # part goes to the x- NEIGHBOUR column, not back along the ray
    w = _uniform(N, kc, l0=0, Lmax=0)
    A2 = orc.trace(w, geom_corr=2)[0].reshape(N, N, N)
    A1 = orc.trace(w, geom_corr=1)[0].reshape(N, N, N)
    for k in range(3, c):
        assert abs(A1[c, c - k, c] - f(k, 1) * a(k)) <= 1e-12 * a(k)
        assert abs(A2[c, c - k, c] - f(k, 1) * a(k)) <= 1e-12 * a(k)                 # nothing comes back to the axis
        assert abs(A2[c, c - k, c - 1] - A1[c, c - k, c - 1] - (1 - f(k, 1)) * a(k)) <= 1e-9 * a(k)


def test_secondary_correction_conserves_photons_and_primary_does_not():
    for w in (wl.tiny(N=12, nsrc=3, nb=3, seed=5, dtype="f64", kappa_scale=20.0), _uniform(16, 0.4, l0=1, tau_term=30.0)):
        em = None
        lost = {}
        for mode in (0, 1, 2, 3):
            A, st, _ = orc.trace(w, geom_corr=mode)
            em = st["emitted"][:w.nb]
            tot = (st["absorbed"] + st["escaped"])[:w.nb]
            assert np.allclose(A.sum(axis=0), st["absorbed"][:w.nb], rtol=1e-12)
            lost[mode] = 1 - tot / em
            if mode in (0, 2):
                assert np.all(np.abs(lost[mode]) < 1e-10), (mode, lost[mode])      # Eq. 3 restores conservation
        assert np.all(lost[1] > 1e-3) and np.all(lost[3] > lost[1])               # f_c only removes; f_c^2 removes more


def test_correction_does_not_change_the_traversal():
    w = wl.tiny(N=10, nsrc=2, nb=2, seed=3, dtype="f64", kappa_scale=10.0)
    ref = orc.trace(w, geom_corr=0)[1]
    for mode in (1, 2, 3):
        st = orc.trace(w, geom_corr=mode)[1]
        assert st["digest"] == ref["digest"] and st["segments"] == ref["segments"]
        assert np.array_equal(st["escaped"], ref["escaped"])                     # the ray itself is attenuated as before


def test_eq3_absorber_density_ratio_in_the_rates():
    """Eq. 3: the rate added to the neighbour is (1 - f_c) x_abs / x'_abs times the cell's rate.  Uniform n_H, pure
    hydrogen, the neighbour column (x- of the -y axis ray, previous test) given half the neutral fraction: the photons
    moved are the same, so the neighbour's Gamma doubles (absorbed photons per absorber)."""
    N, kc = 16, 0.05
    c = N // 2
    w = _uniform(N, kc, l0=0, Lmax=0)
    f0 = [np.array(x, dtype=np.float64) for x in w.fields()]
    kap = orc.opacity(w, f0)
    A1 = orc.trace(w, kappa=kap, geom_corr=1)[0]
    A2 = orc.trace(w, kappa=kap, geom_corr=2)[0]
    moved = (A2 - A1).reshape(N, N, N)[c, c - 5, c - 1]                         # photons/s the secondary term put there
    assert moved > 0
    for xn in (1.0, 0.5):
        f = [x.copy() for x in f0]
        x3 = f[1].reshape(N, N, N)
        x3[c, c - 5, c - 1] = xn
        G = orc.finalize(w, (A2 - A1), f)[0]                                    # rates of the moved photons alone
        V = (w.box_cm / N) ** 3
        assert abs(G[0].reshape(N, N, N)[c, c - 5, c - 1] - moved / (1e-3 * xn * V)) <= 1e-12 * moved / (1e-3 * xn * V)


def _stromgren_ratio(mode, N=32, nsteps=100, dtfrac=0.05):
    w = wl.config2(N)
    aB = orc.rate_coeffs(1e4)[0]
    t_rec = 1.0 / (aB * 1e-3)
    R_S = (3 * 5e48 / (4 * math.pi * aB * 1e-6)) ** (1 / 3)
    dx = w.box_cm / N
    f = tuple(np.asarray(a, dtype=np.float64) for a in w.fields())
    for _ in range(nsteps):
        f = orc.step(w, f, dt=dtfrac * t_rec, geom_corr=mode)["fields"]
    xe = (1.0 - f[1] - 1.2e-3).clip(0)
    rV = (3 * xe.sum() * dx ** 3 / (4 * math.pi)) ** (1 / 3)
    return rV / (R_S * (1 - math.exp(-nsteps * dtfrac)) ** (1 / 3))


def test_stromgren_radius_under_the_corrections_matches_fig11():
    """PAPER.md:340 (Fig. 11, Phi = 3): f_c alone shrinks the ionised region by roughly 5 %, f_c^2 by roughly 10 %, and the
    secondary correction brings it back to the uncorrected size."""
    r = {m: _stromgren_ratio(m) for m in (0, 1, 2, 3)}
    s1, s3 = 1 - r[1] / r[0], 1 - r[3] / r[0]
    assert abs(s1 - float(GOLD["geom_fc_radius_shrink"])) < 0.02, s1
    assert abs(s3 - float(GOLD["geom_fc2_radius_shrink"])) < 0.03, s3
    assert abs(r[2] / r[0] - 1) < 0.005, r
    assert abs(r[2] - 1) < float(GOLD["stromgren_accuracy"])
