"""Pins for the oracle's radiative-transfer time step: relations the paper's own
derivation fixes, the tau > 0.5 restriction, photo-ionisation equilibrium, and consistency with the (separately pinned)
backward-difference update."""
import math

import numpy as np

from oracle import oracle as orc
from paper_1807_07094_b200 import workloads as wl


def _cells(N=4, seed=0):
    w = wl.config2(N)                         # pure hydrogen, isothermal 1e4 K, case B, no collisional ionisation
    rng = np.random.default_rng(seed)
    n = w.ncell
    f = [np.asarray(a, dtype=np.float64).copy() for a in w.fields()]
    f[0][:] = 1e-3 * 10 ** rng.uniform(-0.5, 0.5, n)
    f[1][:] = 10 ** rng.uniform(-3, -0.01, n)
    G = 10 ** rng.uniform(-16, -12, n)
    return w, f, G


def test_dt_I_is_dt_n_over_tau_cell_by_cell():
    """dt_I = eps / (sigma d |dn/dt|) = dt_n / (n_HI sigma d): one cell at a time"""
    w, f, G = _cells()
    d = w.box_cm / w.N
    for c in range(0, w.ncell, 7):
        one = wl.config2(1)
        one.box_cm = d                           # a one-cell grid of the same cell width
        fc = [a[c:c + 1] for a in f]
        tau = fc[0][0] * fc[1][0] * w.sig_HI[0] * d
        dtI, usedI = orc.suggest_dt(one, fc, G[c:c + 1], scheme=2)
        dtn, usedn = orc.suggest_dt(one, fc, G[c:c + 1], scheme=1)
        assert usedI == 1 and math.isfinite(dtI)
        if tau > 0.5:
            assert usedn == 1 and abs(dtI * tau / dtn - 1) < 1e-14
        else:
            assert usedn == 0 and dtn == math.inf       # only cells with tau > 0.5 count


def test_minimum_over_cells_and_linear_in_eps():
    w, f, G = _cells(seed=3)
    d = w.box_cm / w.N
    per = []
    for c in range(w.ncell):
        one = wl.config2(1); one.box_cm = d
        per.append(orc.suggest_dt(one, [a[c:c + 1] for a in f], G[c:c + 1], scheme=2)[0])
    dt, used = orc.suggest_dt(w, f, G, scheme=2)
    assert used == w.ncell and dt == min(per)
    assert abs(orc.suggest_dt(w, f, G, scheme=2, eps=0.05)[0] / dt - 0.5) < 1e-15


def test_equilibrium_cell_does_not_limit_the_step():
    """Gamma x_HI = alpha_B n_H (1 - x_HI)^2 (no collisional ionisation): dn_HI/dt = 0 there"""
    w = wl.config2(1)
    aB = orc.rate_coeffs(1e4)[0]
    nH, x = 1e-3, 0.3
    G = aB * nH * (1 - x) ** 2 / x
    f = [np.array([v]) for v in (nH, x, 1.0, 0.0, 1e4)]
    dt_eq, _ = orc.suggest_dt(w, f, np.array([G]), scheme=2)
    dt_off, _ = orc.suggest_dt(w, f, np.array([2 * G]), scheme=2)
    assert dt_eq > 1e12 * dt_off                 # (the root is hit to rounding, not exactly)


def test_consistent_with_the_backward_difference_update():
    """a step of 1e-3 dt_n changes n_HI by 1e-3 eps (first order), with the chemistry pinned in test_oracle_chem.py"""
    w = wl.config2(1)
    w.box_cm = 1e22                              # tau > 0.5 in this cell
    nH, x, G = 1e-3, 0.6, 3e-13
    f = [np.array([v]) for v in (nH, x, 1.0, 0.0, 1e4)]
    dtn, used = orc.suggest_dt(w, f, np.array([G]), scheme=1, eps=0.1)
    assert used == 1
    xn, _, _ = orc.chem_cell(w, nH, [x, 1.0, 0.0], 1e4, [G, 0, 0], [0, 0, 0], 1e-3 * dtn)
    assert abs(abs(xn[0] - x) / x / 1e-4 - 1) < 2e-3
