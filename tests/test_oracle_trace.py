"""Pins for the oracle's ray tracer, opacity table and finalisation (O3-O5)."""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from paper_1807_07094_b200 import workloads as wl


def _uniform(N=16, kappa_cell=0.3, l0=0, Lmax=13, tau_term=math.inf, Phi=3.0, src_cell=None, Ndot=1e48):
    w = wl.config1(N)
    c = N // 2 if src_cell is None else src_cell
    w.src_pos_cm[:] = (np.array([c, c, c]) + 0.5) * (w.box_cm / N)
    w.src_Ndot[:] = Ndot
    dx = w.box_cm / N
    w.sig_HI[:] = kappa_cell / (1e-3 * dx)         # tau per cell length = kappa_cell
    w.params.update(l0=l0, Lmax=Lmax, tau_term=tau_term, Phi=Phi)
    return w


def test_exact_attenuation_on_axis_aligned_rays():
    # level 0 only (l0 = Lmax = 0): pixels 4..7 are exactly +-x, +-y.  Along +x the k-th cell from the
    # source cell receives (Ndot/12)(e^-tau_{k-1} - e^-tau_k), tau_k = kappa dx (k + 1/2).
    N, kc = 16, 0.37
    w = _uniform(N, kc, l0=0, Lmax=0)
    A, st, _ = orc.trace(w)
    A = A.reshape(N, N, N)                       # [z, y, x]
    c = N // 2
    S = 1e48 / 12.0
    for sgn, axis in ((+1, "x"), (-1, "x"), (+1, "y"), (-1, "y")):
        for k in range(1, N - c if sgn > 0 else c + 1):
            expect = S * (math.exp(-kc * (k - 0.5)) - math.exp(-kc * (k + 0.5)))
            got = A[c, c, c + sgn * k] if axis == "x" else A[c, c + sgn * k, c]
            assert abs(got - expect) <= 1e-13 * expect, (sgn, axis, k)
    # what leaves the box along +x
    n_cells = N - c                              # source cell + (N-c-1) more
    esc_x = S * math.exp(-kc * (n_cells - 0.5))
    assert st["escaped"][0] > 4 * esc_x * 0.999   # 4 axis rays at least (the -x ones travel further)


def test_axis_ray_cell_sequence_and_segment_lengths():
    N = 12
    w = _uniform(N, 0.1, l0=0, Lmax=0)
    _, _, log = orc.trace(w, log=True)
    rays = orc.raylog_to_dict(log)
    c = N // 2
    cells, end = rays[(0, 0, 4)]                                   # +x
    assert end == orc.END_ESCAPED
    assert list(cells) == [(c * N + c) * N + i for i in range(c, N)]
    i = list(log["pix"]).index(4)
    f, n = log["first"][i], log["count"][i]
    # the source position pos_cm/dx is itself rounded (6.5 dx / dx), hence 1e-14 and not equality
    assert np.allclose(log["ds"][f:f + n], [0.5] + [1.0] * (n - 1), rtol=0, atol=1e-14)
    assert abs(log["r_end"][i] - (N - c - 0.5)) < 1e-14


def _brute_cells(g, d, r0, r1, N, h=2e-4):
    """Cells entered by the line g + t d, t in [r0, r1], sampled every h (in cell units)."""
    n = max(2, int((r1 - r0) / h))
    t = r0 + (np.arange(n) + 0.5) * ((r1 - r0) / n)
    xyz = g[None, :] + t[:, None] * d[None, :]
    ijk = np.floor(xyz).astype(np.int64)
    ok = np.all((ijk >= 0) & (ijk < N), axis=1)
    ijk = ijk[ok]
    lin = (ijk[:, 2] * N + ijk[:, 1]) * N + ijk[:, 0]
    keep = np.ones(len(lin), bool)
    keep[1:] = lin[1:] != lin[:-1]
    return lin[keep].tolist(), h


def _is_subsequence(a, b):
    it = iter(b)
    return all(any(x == y for y in it) for x in a)


@pytest.mark.parametrize("N,seed,l0", [(4, 1, 0), (6, 2, 1), (8, 3, 0)])
def test_cell_sequences_against_brute_force_line_sampling(N, seed, l0):
    w = wl.tiny(N=N, nsrc=2, nb=1, seed=seed, l0=l0, tau_term=math.inf)
    _, st, log = orc.trace(w, log=True)
    dx = w.box_cm / N
    Phi = w.params["Phi"]
    checked = 0
    for i in range(len(log["src"])):
        s, l, p = int(log["src"][i]), int(log["level"][i]), int(log["pix"][i])
        g = w.src_pos_cm[s] / dx
        d = orc.pix2vec(l, p)
        r0 = 0.0 if l == l0 else orc.rsplit(Phi, l - 1)
        r1 = float(log["r_end"][i])
        f, n = int(log["first"][i]), int(log["count"][i])
        dda = log["cells"][f:f + n].tolist()
        ds = log["ds"][f:f + n]
        if n == 0:
            continue
        assert abs(ds.sum() - (r1 - r0)) < 1e-12                   # sum of ds = path length
        brute, h = _brute_cells(g, d, r0, r1, N)
        long_cells = [c for c, s_ in zip(dda, ds) if s_ > 3 * h]
        assert _is_subsequence(brute, dda), (s, l, p)                # every sampled cell is visited, in order
        assert _is_subsequence(long_cells, brute), (s, l, p)         # every non-tiny segment is a real crossing
        # cells are face-connected steps of exactly one axis
        ijk = np.array([[c % N, (c // N) % N, c // (N * N)] for c in dda])
        if len(ijk) > 1:
            assert np.all(np.abs(np.diff(ijk, axis=0)).sum(axis=1) == 1)
        checked += 1
    assert checked > 100


def test_geometry_only_ray_counts():
    # transparent medium: every level-l ray whose start point is inside the box is traced and, unless it
    # leaves the box first, splits at rsplit(l); rays = sum_l (number of rays created at level l)
    N = 16
    w = _uniform(N, 0.0, l0=1)
    _, st, log = orc.trace(w, log=True)
    g = w.src_pos_cm[0] / (w.box_cm / N)
    lv = log["level"]
    assert st["rays_level"][1] == 48
    for l in range(1, 8):
        created = int((lv == l).sum())
        if l > 1:
            assert created == 4 * int(st["splits"][l - 1])
        # rays of level l that split = those still inside the box at rsplit(l) (brute force geometry)
        rs = orc.rsplit(3.0, l)
        n_inside = 0
        for p in log["pix"][lv == l]:
            x = g + rs * orc.pix2vec(l, int(p))
            n_inside += bool(np.all((x >= 0) & (x < N)))
        # a ray can leave through a corner region and re-enter is impossible (convex box): equality
        assert int(st["splits"][l]) == n_inside, l
    assert st["segments"] == len(log["cells"])
    assert st["ends"].sum() == st["rays"]


@pytest.mark.parametrize("maker", [
    lambda: wl.config1(),
    lambda: wl.tiny(N=8, nsrc=3, nb=3, seed=11),
    lambda: wl.tiny(N=12, nsrc=2, nb=4, seed=12, dtype="f32", kappa_scale=30.0),
    lambda: wl.config3(N=32, nsrc=4),
    lambda: wl.config4(N=32, nsrc=8),
])
def test_photon_conservation(maker):
    w = maker()
    A, st, _ = orc.trace(w)
    em, ab, es = st["emitted"], st["absorbed"], st["escaped"]
    assert np.all(np.abs(ab + es - em) <= 1e-10 * em)              # north_star: 1e-10 relative
    assert np.all(np.abs(A.sum(axis=0) - ab) <= 1e-10 * em)
    assert np.allclose(em, (w.src_Ndot[:, None] * w.src_binfrac).sum(axis=0), rtol=1e-14)
    assert st["segments"] > 0 and A.min() >= 0.0


def test_depletion_terminates_rays_and_conserves():
    w = _uniform(16, 5.0, l0=0, tau_term=30.0)                    # tau 5 per cell: everything dies in ~6 cells
    A, st, _ = orc.trace(w)
    assert st["ends"][orc.END_ESCAPED] == 0 and st["ends"][orc.END_DEPLETED] > 0
    assert abs(st["absorbed"][0] / st["emitted"][0] - 1) < 1e-12
    A3 = A.reshape(16, 16, 16)
    assert A3[0, 0, 0] == 0.0 and A3[8, 8, 8] > 0


def test_opacity_table_rounding_and_values():
    w = wl.tiny(N=6, nsrc=1, nb=3, seed=5, dtype="f32")
    k = orc.opacity(w)
    nH = w.n_H.astype(np.float64)
    nHe = nH * 0.24 / (4 * 0.76)
    ref = (w.sig_HI[None, :] * (nH * w.x_HI)[:, None] + w.sig_HeI[None, :] * (nHe * w.x_HeI)[:, None]
           + w.sig_HeII[None, :] * (nHe * w.x_HeII)[:, None])
    assert np.all(k == k.astype(np.float32).astype(np.float64))   # representable in f32
    assert np.allclose(k, ref, rtol=1e-7)
    k64 = orc.opacity(w, field_dtype=1)
    assert np.allclose(k64, ref, rtol=1e-15)


def test_finalize_partition_of_unity_and_single_species():
    w = wl.tiny(N=8, nsrc=2, nb=4, seed=21)
    A, st, _ = orc.trace(w)
    G, H, Ht = orc.finalize(w, A)
    dx = w.box_cm / w.N
    V = dx ** 3
    nH = w.n_H.astype(np.float64)
    nHe = nH * 0.24 / (4 * 0.76)
    n = np.stack([nH * w.x_HI, nHe * w.x_HeI, nHe * w.x_HeII])
    lhs = (G * n).sum(axis=0) * V
    rhs = A.sum(axis=1)
    assert np.allclose(lhs, rhs, rtol=1e-12, atol=1e-12 * rhs.max())
    assert np.allclose(Ht, (H * n).sum(axis=0), rtol=1e-13)
    assert np.all(H >= 0)
    # single species, single bin: Gamma = A/(V n_HI)  (Eq. 1), heating = Gamma (E - 13.598 eV)
    w1 = wl.config1(16)
    w1.E_eV[:] = 20.0
    A1, _, _ = orc.trace(w1)
    G1, H1, _ = orc.finalize(w1, A1)
    V1 = (w1.box_cm / 16) ** 3
    assert np.allclose(G1[0], A1[:, 0] / (V1 * 1e-3), rtol=1e-14)
    assert np.allclose(H1[0], G1[0] * (20.0 - 13.598) * 1.602176634e-12, rtol=1e-14)
    assert np.all(G1[1:] == 0)


def test_finalize_of_a_hand_worked_three_species_cell():
    """orc_finalize with all three absorbers and three bins, numbers worked by hand (Eq. 1 with n_abs = n_SI, PAPER.md:83;
    heating h(nu - nu_S) s_nu n_SI; the species' share of a bin is its share of the opacity, reading G8).
    Y_p = 0.2: n_He = n_H/16.  Cell: n_H = 1.6e-2, x = (0.5, 0.25, 0.5) -> n_HI = 8e-3, n_HeI = 2.5e-4, n_HeII = 5e-4;
    kappa = (4.8e-20, 1.7e-20, 9e-21) cm^-1 (tests/test_oracle_chem_pins.py works those out)."""
    w = wl.tiny(N=2, nb=3, dtype="f64")
    w.E_eV = np.array([20.0, 40.0, 80.0])
    w.sig_HI = np.array([6e-18, 2e-18, 1e-18]); w.sig_HeI = np.array([0.0, 4e-18, 2e-18]); w.sig_HeII = np.array([0.0, 0.0, 1e-18])
    f = (np.full(8, 1.6e-2), np.full(8, 0.5), np.full(8, 0.25), np.full(8, 0.5), np.full(8, 1e4))
    A = np.zeros((8, 3)); A[0] = (3e40, 2e40, 1e40)
    G, H, Ht = orc.finalize(w, A, f, Yp=0.2)
    V = (w.box_cm / 2) ** 3
    eV = 1.602176634e-12
    per_bin_HI = np.array([3e40 * 6e-18 / 4.8e-20, 2e40 * 2e-18 / 1.7e-20, 1e40 * 1e-18 / 9e-21])       # 3.75e42, 2.3529e42, 1.1111e42
    per_bin_HeI = np.array([0.0, 2e40 * 4e-18 / 1.7e-20, 1e40 * 2e-18 / 9e-21])
    per_bin_HeII = np.array([0.0, 0.0, 1e40 * 1e-18 / 9e-21])
    assert abs(G[0, 0] * V / 7.214052e42 - 1) < 1e-6 and abs(G[0, 0] * V / per_bin_HI.sum() - 1) < 1e-13
    assert abs(G[1, 0] * V / per_bin_HeI.sum() - 1) < 1e-13 and abs(G[2, 0] * V / per_bin_HeII.sum() - 1) < 1e-13
    # every absorbed photon ionises exactly one atom: sum_S Gamma_S n_S V = sum_nu A_nu = 6e40
    assert abs((G[0, 0] * 8e-3 + G[1, 0] * 2.5e-4 + G[2, 0] * 5e-4) * V / 6e40 - 1) < 1e-13
    # heating per absorber: photon energy above each species' OWN threshold (13.598, 24.587, 54.418 eV)
    want_H = [(per_bin_HI * (w.E_eV - 13.598)).sum(), (per_bin_HeI * (w.E_eV - 24.587)).sum(), (per_bin_HeII * (w.E_eV - 54.418)).sum()]
    assert abs(want_H[0] / 1.599099e44 - 1) < 1e-6 and abs(want_H[1] / 1.956718e44 - 1) < 1e-6 and abs(want_H[2] / 2.842444e43 - 1) < 1e-6
    for S in range(3):
        assert abs(H[S, 0] * V / (want_H[S] * eV) - 1) < 1e-13, S
    assert abs(Ht[0] / (H[0, 0] * 8e-3 + H[1, 0] * 2.5e-4 + H[2, 0] * 5e-4) - 1) < 1e-13
    assert np.all(G[:, 1:] == 0) and np.all(Ht[1:] == 0)
    # a bin below a species' threshold ionises nothing of it by construction (sigma = 0); if a caller gives it a
    # cross-section anyway, the photons are counted but heat nothing (no negative heating)
    w.sig_HeI = np.array([1e-18, 4e-18, 2e-18])
    G2, H2, _ = orc.finalize(w, A, f, Yp=0.2)
    k0 = 6e-18 * 8e-3 + 1e-18 * 2.5e-4
    assert abs(G2[1, 0] * V / (3e40 * 1e-18 / k0 + per_bin_HeI[1:].sum()) - 1) < 1e-13
    assert abs(H2[1, 0] / H[1, 0] - 1) < 1e-13


def test_flux_unit_arithmetic_from_the_paper():
    # the paper's own worked numbers pin the unit constants of the input module
    vals = dict(l.split()[:2] for l in open(__file__.rsplit("/", 1)[0] + "/golden/paper_values.txt")
                if l.strip() and not l.startswith("#"))
    kpc = wl.KPC_CM
    f0 = float(vals["test0_luminosity"]) / (4 * math.pi * (float(vals["test0_box_kpc"]) * kpc) ** 2)
    assert abs(f0 / float(vals["test0_flux"]) - 1) < 0.01
    r3 = float(vals["test3_distance_cells"]) * 6.6 / 128 * kpc
    f3 = float(vals["test3_luminosity"]) / (4 * math.pi * r3 ** 2)
    assert abs(f3 / float(vals["test3_flux"]) - 1) < 0.01


def test_inverse_square_in_optically_thin_limit():
    # thin uniform medium: sum of A over a shell ~ Ndot * kappa * dr, i.e. rate per cell ~ 1/(4 pi r^2)
    N = 32
    w = _uniform(N, 1e-6, l0=1)
    A, _, _ = orc.trace(w)
    A3 = A.reshape(N, N, N)
    c = N // 2
    zz, yy, xx = np.meshgrid(*(np.arange(N) - c,) * 3, indexing="ij")
    r = np.sqrt(xx ** 2 + yy ** 2 + zz ** 2)
    for r0 in (4, 8, 12):
        m = (r >= r0) & (r < r0 + 1)
        shell = A3[m].sum()
        vol_shell = m.sum()
        # photons absorbed per unit volume at r: Ndot kappa /(4 pi r^2): integrate over the voxelised shell
        expect = (1e48 * 1e-6 / (4 * math.pi * r[m] ** 2)).sum()
        assert abs(shell / expect - 1) < 0.03, (r0, shell / expect, vol_shell)
