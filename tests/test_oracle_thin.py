"""Pins for the optically thin inner region of the oracle (readings G33-G37)."""
import math

import numpy as np

from oracle import oracle as orc
from paper_1807_07094_b200 import workloads as wl


def _uniform(N=16, kappa_cell=0.02, l0=1, Phi=3.0, tau_term=math.inf):
    w = wl.config1(N)
    c = N // 2
    w.src_pos_cm[:] = (np.array([c, c, c]) + 0.5) * (w.box_cm / N)
    w.sig_HI[:] = kappa_cell / (1e-3 * (w.box_cm / N))
    w.params.update(l0=l0, tau_term=tau_term, Phi=Phi)
    return w


def _radius_from_logs(w, kap_cell, log, thin_tau):
    """brute force over the ray tree: tau (bin 0) along every path from the logged cells and segment lengths"""
    rays = {}
    for i in range(len(log["pix"])):
        f, n = int(log["first"][i]), int(log["count"][i])
        rays[(int(log["src"][i]), int(log["level"][i]), int(log["pix"][i]))] = (log["cells"][f:f + n], log["ds"][f:f + n],
                                                                                int(log["end"][i]), float(log["r_end"][i]))
    R = {}
    tau_end = {}
    for key in sorted(rays, key=lambda k: k[1]):                     # parents before children
        s, l, p = key
        cells, ds, end, r_end = rays[key]
        par = (s, l - 1, p >> 2)
        tau = tau_end.get(par, 0.0)
        r = r_end - float(np.sum(ds))                                 # start radius
        for c, d in zip(cells, ds):
            dt = kap_cell[c] * d
            if tau < thin_tau <= tau + dt:
                R[s] = min(R.get(s, math.inf), r)
            tau += dt
            r += d
        tau_end[key] = tau
        if end != orc.END_SPLIT and tau < thin_tau:
            R[s] = min(R.get(s, math.inf), r_end)
    return R


def test_radius_is_the_brute_force_minimum_over_the_ray_tree():
    w = wl.tiny(N=12, nsrc=3, nb=2, seed=23, dtype="f64", l0=1, kappa_scale=0.004)
    kap = orc.opacity(w)
    _, st, log = orc.trace(w, kappa=kap, log=True, thin_tau=0.1)
    dx = w.box_cm / w.N
    want = _radius_from_logs(w, kap[:, 0] * dx, log, 0.1)
    assert all(st["R_thin"] > 0.3)                                    # (random opacities: a fraction of a cell to a few cells)
    for s in range(3):
        assert abs(st["R_thin"][s] - want[s]) < 1e-11, (s, st["R_thin"][s], want[s])
    # off: no radii
    assert np.all(orc.trace(w, kappa=kap)[1]["R_thin"] == 0)


def test_uniform_medium_radius_is_where_tau_reaches_the_threshold():
    """tau = kappa r along every ray: the radius lies within one segment (< sqrt(3) cells) below thin_tau / kappa"""
    w = _uniform(24, kappa_cell=0.02)
    st = orc.trace(w, thin_tau=0.1)[1]
    R = st["R_thin"][0]
    assert 0.1 / 0.02 - math.sqrt(3) <= R <= 0.1 / 0.02


def test_inner_cells_get_the_papers_thin_limit_rate_and_rays_start_at_R():
    N, kc, R0 = 24, 1e-3, 4.3
    w = _uniform(N, kc)
    kap = orc.opacity(w)
    A, st, log = orc.trace(w, kappa=kap, log=True, thin_tau=0.1, Rstart=np.array([R0]))
    A0 = orc.trace(w, kappa=kap, log=False)[0]
    c = N // 2
    S = float(w.src_Ndot[0])
    idx = np.indices((N, N, N))                                       # [z, y, x]
    d2 = sum((idx[k] - c).astype(float) ** 2 for k in range(3))
    inner = (d2 <= R0 * R0).ravel()
    # (iii) S x sigma / (4 pi R^2) per absorber = S kappa V / (4 pi r^2) photons/s per cell
    far = inner & (d2.ravel() > 0) & (np.sqrt(d2.ravel()) + 1.0 <= R0)          # cells no ray segment reaches
    want = S * kc / (4 * math.pi * d2.ravel()[far])
    assert np.allclose(A[far, 0], want, rtol=1e-12)
    assert abs(A[(c * N + c) * N + c, 0] - S * kc / (4 * math.pi * 0.25)) < 1e-12 * S     # source cell: r^2 floor (d/2)^2
    # the closed form is what ray tracing gives in the thin limit, shell by shell
    r = np.sqrt(d2.ravel())
    for lo, hi, tol in ((1.5, 2.3, 0.06), (2.3, 3.31, 0.03)):         # (1/r^2 at the cell centre vs its cell average: coarser near the source)
        sh = (r >= lo) & (r < hi) & far
        assert sh.sum() > 20
        assert abs(A0[sh, 0].sum() / A[sh, 0].sum() - 1) < tol, lo
    # (iv) rays start at R0, at the level they would have there, with tau = 0
    lv = 1
    while orc.rsplit(3.0, lv) <= R0:
        lv += 1
    roots = [i for i in range(len(log["pix"])) if log["level"][i] == lv]
    assert len(roots) == 12 * 4 ** lv and min(log["level"]) == lv
    g = np.array([c + 0.5] * 3)
    for i in roots[::37]:
        d = orc.pix2vec(lv, int(log["pix"][i]))
        first = log["cells"][log["first"][i]]
        ijk = np.floor(g + R0 * d).astype(int)
        assert first == (ijk[2] * N + ijk[1]) * N + ijk[0]


def test_outside_the_region_rates_differ_by_the_neglected_inner_attenuation_only():
    """beyond R the same rays cross the same cells; they were not attenuated inside: ratio in [1, e^thin_tau]"""
    N, kc = 24, 0.02
    w = _uniform(N, kc)
    kap = orc.opacity(w)
    A0, s0, _ = orc.trace(w, kappa=kap, thin_tau=0.1)
    R = s0["R_thin"]
    A1, s1, _ = orc.trace(w, kappa=kap, thin_tau=0.1, Rstart=R)
    c = N // 2
    idx = np.indices((N, N, N))
    r = np.sqrt(sum((idx[k] - c).astype(float) ** 2 for k in range(3))).ravel()
    out = r > R[0] + 2.0
    ratio = A1[out, 0] / A0[out, 0]
    assert ratio.min() >= 1.0 - 1e-12 and ratio.max() <= math.exp(0.1) + 1e-12
    assert abs(ratio.mean() - math.exp(kc * R[0])) < 0.01
    assert s1["R_thin"][0] >= R[0]                                     # the region can only grow from where rays start
    assert s1["segments"] < s0["segments"]                             # the point of it: fewer segments
