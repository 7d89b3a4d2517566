"""Pins for the oracle's HEALPix direction generator and split radii (O1, O2).

Nothing here re-types the oracle's formula: the ring-scheme closed form, libm, brute force and the
worked values (z, phi) derived in SURVEY.md 8(c) O1 are independent statements.
"""
import math
from fractions import Fraction

import numpy as np
import pytest

from oracle import oracle as orc


def _ring_closed_form(level):
    """Multiset of (z, phi/pi) as exact fractions from the RING scheme (Gorski et al. 2005)."""
    ns = 1 << level
    out = []
    for i in range(1, ns):                       # polar caps
        z = 1 - Fraction(i * i, 3 * ns * ns)
        for j in range(1, 4 * i + 1):
            ph = Fraction(2 * j - 1, 4 * i)
            out.append((z, ph))
            out.append((-z, ph))
    for i in range(ns, 3 * ns + 1):              # belt
        z = Fraction(4, 3) - Fraction(2 * i, 3 * ns)
        s = (i - ns + 1) % 2
        for j in range(1, 4 * ns + 1):
            out.append((z, Fraction(2 * j - s, 4 * ns) % 2))     # phi = 2 pi is phi = 0
    return sorted(out)


@pytest.mark.parametrize("level", [0, 1, 2, 3, 4, 5])
def test_nested_pixels_equal_ring_closed_form(level):
    npix = 12 * 4 ** level
    got = []
    for p in range(npix):
        zn, zd, m, nr = orc.pix2ring(level, p)
        got.append((Fraction(zn, zd), Fraction(m, 4 * nr)))
    assert sorted(got) == _ring_closed_form(level)
    assert len({g[0] for g in got}) == 4 * (1 << level) - 1       # distinct z rings


def test_level1_is_48_packets_golden():
    vals = dict(l.split()[:2] for l in open(__file__.rsplit("/", 1)[0] + "/golden/paper_values.txt")
                if l.strip() and not l.startswith("#"))
    assert 12 * 4 ** 1 == int(vals["healpix_level1_packets"])


def test_worked_values():
    # SURVEY.md 8(c) O1 worked values: (level, pix) -> (z, phi/pi)
    cases = {(0, 0): (Fraction(2, 3), Fraction(1, 4)), (0, 1): (Fraction(2, 3), Fraction(3, 4)),
             (0, 4): (0, 0), (0, 5): (0, Fraction(1, 2)), (0, 6): (0, 1), (0, 7): (0, Fraction(3, 2)),
             (0, 8): (Fraction(-2, 3), Fraction(1, 4)), (0, 11): (Fraction(-2, 3), Fraction(7, 4)),
             (1, 0): (Fraction(1, 3), Fraction(1, 4)), (1, 1): (Fraction(2, 3), Fraction(3, 8)),
             (1, 3): (Fraction(11, 12), Fraction(1, 4)), (1, 16): (Fraction(-1, 3), 0),
             (1, 17): (0, Fraction(1, 8)), (1, 18): (0, Fraction(15, 8))}
    for (l, p), (z, ph) in cases.items():
        zn, zd, m, nr = orc.pix2ring(l, p)
        assert Fraction(zn, zd) == z and Fraction(m, 4 * nr) == ph, (l, p)


def test_axis_directions_exact():
    # level-0 pixels 4..7 are exactly +x, +y, -x, -y
    assert orc.pix2vec(0, 4).tolist() == [1.0, 0.0, 0.0]
    assert orc.pix2vec(0, 5).tolist() == [0.0, 1.0, 0.0]
    assert orc.pix2vec(0, 6).tolist() == [-1.0, 0.0, 0.0]
    d = orc.pix2vec(0, 7)
    assert d[0] == 0.0 and d[1] == -1.0 and d[2] == 0.0


@pytest.mark.parametrize("level", [0, 1, 2, 3, 6, 10, 13])
def test_vectors_match_libm_and_are_unit(level):
    rng = np.random.default_rng(level)
    npix = 12 * 4 ** level
    pix = range(npix) if npix <= 768 else rng.integers(0, npix, 600).tolist()
    acc = np.zeros(3)
    for p in pix:
        zn, zd, m, nr = orc.pix2ring(level, p)
        z = zn / zd
        phi = math.pi * m / (4 * nr)
        s = math.sqrt((1 - z) * (1 + z))
        ref = np.array([s * math.cos(phi), s * math.sin(phi), z])
        d = orc.pix2vec(level, p)
        assert np.all(np.abs(d - ref) <= 1e-15), (level, p, d - ref)   # libm phi itself is rounded
        assert abs(np.dot(d, d) - 1.0) < 5e-16
        acc += d
    if npix <= 768:
        assert np.linalg.norm(acc) <= 1e-15 * npix


def test_own_sincos_within_2ulp_of_libm():
    rng = np.random.default_rng(3)
    worst = 0.0
    for _ in range(4000):
        nr = int(rng.integers(1, 9000))
        m = int(rng.integers(0, 8 * nr))
        s, c = orc.sincos_frac(m, nr)
        # reference in extended precision via exact reduction to the first octant
        from mpmath import mp, mpf, sin, cos, pi
        mp.prec = 120
        a = pi * mpf(m) / (4 * nr)
        for got, ref in ((s, sin(a)), (c, cos(a))):
            ref_f = float(ref)
            ulp = math.ulp(abs(ref_f)) if ref_f != 0 else 5e-324
            if m % (2 * nr) == 0 and abs(ref_f) < 1e-30:      # exactly on an axis: the true value is 0
                assert got == 0.0
            else:
                worst = max(worst, abs(got - ref_f) / ulp)
    assert worst <= 2.0, worst


def test_sincos_exact_on_axes():
    for nr in (1, 2, 7, 64):
        assert orc.sincos_frac(0, nr) == (0.0, 1.0)
        assert orc.sincos_frac(2 * nr, nr) == (1.0, 0.0)
        s, c = orc.sincos_frac(4 * nr, nr)
        assert s == 0.0 and c == -1.0
        s, c = orc.sincos_frac(6 * nr, nr)
        assert s == -1.0 and c == 0.0


@pytest.mark.parametrize("level", [0, 1, 2])
def test_children_are_nearest_to_their_parent(level):
    npar = 12 * 4 ** level
    par = np.array([orc.pix2vec(level, p) for p in range(npar)])
    for p in range(npar):
        for j in range(4):
            c = orc.pix2vec(level + 1, 4 * p + j)
            assert int(np.argmax(par @ c)) == p


def test_split_radius_closed_form():
    for Phi in (1.0, 3.0, 5.5):
        for l in range(0, 12):
            r = orc.rsplit(Phi, l)
            # Omega_l r^2 = 1/Phi (cell units), Omega_l = 4pi/(12 4^l)
            omega = 4 * math.pi / (12 * 4 ** l)
            assert abs(omega * r * r * Phi - 1.0) < 1e-14
            assert orc.rsplit(Phi, l + 1) == 2.0 * r            # exact power-of-two scaling
    assert abs(orc.rsplit(3.0, 0) - 0.56419) < 1e-5 and abs(orc.rsplit(1.0, 0) - 0.97721) < 1e-5
    assert orc.rsplit(3.0, 13, 13) == math.inf


def test_rays_per_cell_area_stays_between_phi_and_4phi():
    Phi = 3.0
    for l in range(1, 10):
        # level-l rays live on r in [rsplit(l-1), rsplit(l)]: rays per unit cell area = Npix/(4 pi r^2)
        for r in (orc.rsplit(Phi, l - 1), orc.rsplit(Phi, l)):
            dens = 12 * 4 ** l / (4 * math.pi * r * r)
            assert Phi * (1 - 1e-12) <= dens <= 4 * Phi * (1 + 1e-12)
