"""Pins for the parts of the oracle's chemistry / thermal update that tests/test_oracle_chem.py left open
("parity unpinned"): the helium branches of Eq. 4-5, the electron density
(PAPER.md:73), the energy update and T(E) (readings G16, G17), the collisional-excitation,
dielectronic and free-free fits (reading G11) and the opacity table.

Every expected value here is typed from the paper's equations (in the paper's variables: n_b, A_H, A_He, n_SI, n_SII),
from a conservation law, from a closed-form solution, from an independent integrator (scipy) or from textbook numbers
kept in tests/golden/textbook_rates.txt - never from the oracle's own expressions.  Each test names, in its docstring,
the line of oracle/arc_oracle.c whose plausible mistakes it catches.
"""
import math
import os

import numpy as np
import pytest

from oracle import oracle as orc
from paper_1807_07094_b200 import workloads as wl

KB = 1.380649e-16            # erg / K
EV = 1.602176634e-12         # erg
KB_EV = 8.617333262e-5       # eV / K
A_H, A_HE = 1.0, 4.0


def _p(**kw):
    """oracle parameters of a small H + He workload; keyword overrides"""
    w = wl.tiny(N=4, nb=3)
    d = dict(isothermal=1, caseB=1, coll_ion=0, max_subcycles=1, Yp=0.24, eps_sub=0.1, x_floor=1e-12)
    d.update(kw)
    return orc.make_params(w, **d)


def _ne_paper(nH, Yp, xHII, xHeII, xHeIII):
    """PAPER.md:73, in the paper's variables: n_e = n_b [ (1 - Y_p)/A_H x_HII + Y_p/A_He (x_HeII + 2 x_HeIII) ],
    with the hydrogen number density n_H = n_b (1 - Y_p) / A_H."""
    n_b = nH * A_H / (1.0 - Yp)
    return n_b * ((1.0 - Yp) / A_H * xHII + Yp / A_HE * (xHeII + 2.0 * xHeIII))


def _golden(prefix):
    rows = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "textbook_rates.txt")) as f:
        for line in f:
            t = line.split("#")[0].split()
            if t and t[0].startswith(prefix):
                rows[t[0][len(prefix):]] = [float(x) for x in t[1:]]
    return rows


# ------------------------------------------------------------------------------------------------ electron density
@pytest.mark.parametrize("Yp,x", [(0.24, (0.3, 0.5, 0.2)), (0.24, (0.9, 0.1, 0.9)), (0.1, (0.05, 0.0, 0.4)), (0.0, (0.5, 1.0, 0.0))])
def test_electron_density_is_the_papers_formula_in_baryon_units(Yp, x):
    """arc_oracle.c n_e line (`ne = nH*xHII + nHe*(x[2] + 2*xHeIII)`) and `n_He_of`.  Probe: with Gamma = 0 and no
    collisional ionisation one backward-difference step of hydrogen is x' = x + alpha n_e x_HII dt exactly, so
    n_e = (x' - x) / (alpha x_HII dt) is read off the oracle and compared with PAPER.md:73 typed with n_b, A_H, A_He.
    A wrong helium abundance (Yp/4 vs Yp/(4(1-Yp))), a missing factor 2 for He III or a dropped He II term fails."""
    p = _p(Yp=Yp)
    T, nH = 1.5e4, 3e-3
    alpha = orc.rate_coeffs(T, caseB=1, coll_ion=0)[0]
    x0, x1, x2 = x
    xHeIII = 1.0 - x1 - x2
    ne_want = _ne_paper(nH, Yp, 1.0 - x0, x2, xHeIII)
    dt = 0.05 / (alpha * ne_want)                      # x_HI changes by ~ 0.05 x_HII: no cancellation, no clamp
    xn, Tn, k = orc.chem_cell(p, nH, [x0, x1, x2], T, [0.0, 0.0, 0.0], [0, 0, 0], dt)
    assert k == 1 and Tn == T
    ne_got = (xn[0] - x0) / (alpha * (1.0 - x0) * dt)
    assert abs(ne_got / ne_want - 1.0) < 1e-12, (ne_got, ne_want)


# ------------------------------------------------------------------------------------------------ helium, Eq. 4-5
HELIUM_CASES = [
    # T [K], (x_HI, x_HeI, x_HeII): all three helium stages populated.  At 3e4 K the photo-, collisional (He I) and
    # recombination terms are of one order; at 1.5e5 K the collisional ionisation of He II carries weight.
    (3e4, (0.2, 0.35, 0.45)),
    (1.5e5, (0.2, 1e-3, 0.6)),
]


def _helium_case(T, x, nH=2e-3, Yp=0.24):
    """-> ne, table, photo-rates (set to the order of the collisional + recombination rates of their stage), dt"""
    co = orc.rate_coeffs(T, caseB=1, coll_ion=1)
    ne = _ne_paper(nH, Yp, 1.0 - x[0], x[2], 1.0 - x[1] - x[2])
    G = [1.5 * (co[0] + co[3]) * ne, 0.8 * (co[1] + co[4]) * ne, 0.5 * (co[2] + co[5]) * ne]
    return nH, Yp, ne, co, G


def _helium_terms(x, ne, co, G):
    """Eq. 4 per helium stage, as named (sink / source) rates per unit fraction:
       S = He I :  d x_HeI /dt = - x_HeI (Gamma_HeI + C_HeI n_e) + alpha_HeII n_e x_HeII
       S = He II:  d x_HeII/dt = - x_HeII (Gamma_HeII + C_HeII n_e) + alpha_HeIII n_e x_HeIII      (to / from He III)
                                 + x_HeI (Gamma_HeI + C_HeI n_e)    - alpha_HeII n_e x_HeII          (from / to He I)"""
    a_HeII, a_HeIII, c_HeI, c_HeII = co[1], co[2], co[4], co[5]
    x_HeIII = 1.0 - x[1] - x[2]
    sink1 = {"Gamma_HeI": G[1], "C_HeI": c_HeI * ne}
    src1 = {"alpha_HeII": a_HeII * ne * x[2]}
    sink2 = {"Gamma_HeII": G[2], "C_HeII": c_HeII * ne, "alpha_HeII": a_HeII * ne}
    src2 = {"Gamma_HeI": G[1] * x[1], "C_HeI": c_HeI * ne * x[1], "alpha_HeIII": a_HeIII * ne * x_HeIII}
    return sink1, src1, sink2, src2


def test_one_bdf_step_of_helium_is_the_backward_difference_of_eq4():
    """arc_oracle.c `C1, D1, C2, D2` and the three `y = (x + D dts)/(1 + C dts)` lines.  Eq. 4 for
    S = He I and S = He II, written as Eq. 5 (D - C n): He I loses by photo- and collisional ionisation and gains the
    recombinations of He II; He II loses by its own ionisation and by recombining to He I, and gains the ionisations
    of He I and the recombinations of He III.  One step with max_subcycles = 1 takes the whole dt (no limiter), so
    the result must be (n + D dt)/(1 + C dt) with these D, C - typed here from Eq. 4, rates from the (pinned)
    coefficient table.  Every one of the nine terms moves a result by > 1e-3 in at least one of the two states, so
    dropping the alpha_HeIII source, double counting alpha_HeII in the He II sink, swapping alpha_HeII / alpha_HeIII
    or forgetting a collisional term cannot pass the 1e-13 comparison."""
    weight = {}
    for T, x in HELIUM_CASES:
        nH, Yp, ne, co, G = _helium_case(T, x)
        p = _p(Yp=Yp, coll_ion=1)
        sink1, src1, sink2, src2 = _helium_terms(x, ne, co, G)
        C1, D1, C2, D2 = sum(sink1.values()), sum(src1.values()), sum(sink2.values()), sum(src2.values())
        C0, D0 = G[0] + co[3] * ne, co[0] * ne * (1.0 - x[0])
        dt = 0.5 / max(C1, C2)
        want = [(x[0] + D0 * dt) / (1.0 + C0 * dt), (x[1] + D1 * dt) / (1.0 + C1 * dt), (x[2] + D2 * dt) / (1.0 + C2 * dt)]
        assert want[1] + want[2] < 1.0                   # (no re-closure in these states)
        xn, _, k = orc.chem_cell(p, nH, list(x), T, G, [0, 0, 0], dt)
        assert k == 1
        for i in range(3):
            assert abs(xn[i] / want[i] - 1.0) < 1e-13, (T, i, xn[i], want[i])
        # what each term is worth in this state
        for name, v in sink1.items():
            weight[("sink1", name)] = max(weight.get(("sink1", name), 0), abs((x[1] + D1 * dt) / (1 + (C1 - v) * dt) / want[1] - 1))
        for name, v in src1.items():
            weight[("src1", name)] = max(weight.get(("src1", name), 0), abs((x[1] + (D1 - v) * dt) / (1 + C1 * dt) / want[1] - 1))
        for name, v in sink2.items():
            weight[("sink2", name)] = max(weight.get(("sink2", name), 0), abs((x[2] + D2 * dt) / (1 + (C2 - v) * dt) / want[2] - 1))
        for name, v in src2.items():
            weight[("src2", name)] = max(weight.get(("src2", name), 0), abs((x[2] + (D2 - v) * dt) / (1 + C2 * dt) / want[2] - 1))
    assert len(weight) == 9 and all(v > 1e-3 for v in weight.values()), weight


def test_helium_nuclei_are_conserved_to_first_order_by_the_three_equations():
    """The same lines, pinned by a conservation law instead of typed terms: for dt -> 0 the oracle's rates of change of
    x_HeI and x_HeII, with x_HeIII by closure, must add up so that d x_HeIII / dt is exactly Eq. 4's He III balance
    (ionisations of He II minus recombinations of He III) - what leaves one stage arrives in the next.  A sink
    without its matching source (or a doubled one) breaks it."""
    for T, x in HELIUM_CASES:
        nH, Yp, ne, co, G = _helium_case(T, x)
        p = _p(Yp=Yp, coll_ion=1)
        x_HeIII = 1.0 - x[1] - x[2]
        dt = 1e-7 / (max(co[1:6]) * ne + max(G))
        xn, _, _ = orc.chem_cell(p, nH, list(x), T, G, [0, 0, 0], dt)
        rate3 = ((1.0 - xn[1] - xn[2]) - x_HeIII) / dt
        want3 = (G[2] + co[5] * ne) * x[2] - co[2] * ne * x_HeIII
        assert abs(rate3 / want3 - 1.0) < 1e-4, (T, rate3, want3)
        rate1 = (xn[1] - x[1]) / dt
        assert abs(rate1 / (co[1] * ne * x[2] - (G[1] + co[4] * ne) * x[1]) - 1.0) < 1e-4


def test_helium_reclosure_when_the_jacobi_step_overshoots():
    """arc_oracle.c `if (x[1] + x[2] > 1.0) { ... / sum }` (reading G24).  Pure recombination over a long step: He I
    grows to above 1 and is clamped to 1, He II relaxes to alpha_HeIII x_HeIII / alpha_HeII of its own: the sum exceeds
    1 and both are divided by it - hand-worked below."""
    nH, Yp, T = 1e-2, 0.24, 1e4
    p = _p(Yp=Yp)
    co = orc.rate_coeffs(T, caseB=1, coll_ion=0)
    x = [1e-12, 0.2, 0.7]                                # H ionised, x_HeIII = 0.1
    ne = _ne_paper(nH, Yp, 1.0 - x[0], x[2], 1.0 - 0.2 - 0.7)
    dt = 50.0 / (co[1] * ne)
    y1 = min(1.0, x[1] + co[1] * ne * x[2] * dt)         # no sink: C = 0
    y2 = (x[2] + co[2] * ne * (1.0 - 0.2 - 0.7) * dt) / (1.0 + co[1] * ne * dt)
    assert y1 == 1.0 and 0.0 < y2 < 1.0
    xn, _, _ = orc.chem_cell(p, nH, x, T, [0, 0, 0], [0, 0, 0], dt)
    assert abs(xn[1] - y1 / (y1 + y2)) < 1e-15 and abs(xn[2] - y2 / (y1 + y2)) < 1e-15
    assert abs(xn[1] + xn[2] - 1.0) < 2e-16


def test_helium_photoionisation_equilibrium_is_the_two_level_root():
    """C1/D1 against a closed form.  Neutral hydrogen that nothing ionises (Gamma_HI = 0, no collisions), helium with
    Gamma_HeI only: He III never appears, n_e = n_He x_HeII, and the steady state of Eq. 4 is
    Gamma_HeI x_HeI = alpha_HeII n_e x_HeII with x_HeI + x_HeII = 1, i.e. the positive root of
    alpha n_He x^2 + Gamma x - Gamma = 0."""
    nH, Yp, T, G1 = 1e-2, 0.24, 1e4, 4e-14
    p = _p(Yp=Yp)
    a = orc.rate_coeffs(T, caseB=1, coll_ion=0)[1]
    n_He = nH * A_H / (1.0 - Yp) * Yp / A_HE
    k = a * n_He
    root = (-G1 + math.sqrt(G1 * G1 + 4.0 * k * G1)) / (2.0 * k)
    x = [1.0, 1.0 - 1e-3, 1e-3]
    for _ in range(4000):
        x, _, _ = orc.chem_cell(p, nH, list(x), T, [0.0, G1, 0.0], [0, 0, 0], 0.02 / G1)
    assert x[0] == 1.0
    assert abs(x[2] / root - 1.0) < 1e-6 and abs(x[1] + x[2] - 1.0) < 1e-6, (x, root)


def test_helium_recombination_cascade_matches_the_analytic_two_level_solution():
    """D1, C2, D2 in time: Gamma = 0 for helium, hydrogen held ionised by a strong Gamma_HI and a trace helium abundance
    (Y_p = 0.004: n_e = n_H to 0.1 %), so He III -> He II -> He I is the linear chain
    x3 = x3(0) e^{-k3 t},  x2 = x2(0) e^{-k2 t} + x3(0) k3/(k2 - k3) (e^{-k3 t} - e^{-k2 t}),  x1 = 1 - x2 - x3,
    k3 = alpha_HeIII n_e, k2 = alpha_HeII n_e.  Backward differences converge to it at first order in the step."""
    nH, Yp, T = 1e-2, 0.004, 2e4
    p = _p(Yp=Yp)
    co = orc.rate_coeffs(T, caseB=1, coll_ion=0)
    ne = nH                                              # to 1e-3: helium adds n_He (x2 + 2 x3) <= 2e-3 n_H
    k2, k3 = co[1] * ne, co[2] * ne
    t = 1.5 / k3
    x30, x20 = 0.8, 0.2
    x3 = x30 * math.exp(-k3 * t)
    x2 = x20 * math.exp(-k2 * t) + x30 * k3 / (k2 - k3) * (math.exp(-k3 * t) - math.exp(-k2 * t))
    errs = []
    for n in (50, 500, 5000):
        x = [1e-12, 1e-12, x20]
        for _ in range(n):
            x, _, _ = orc.chem_cell(p, nH, list(x), T, [1e-6, 0.0, 0.0], [0, 0, 0], t / n)
        errs.append(max(abs(x[2] - x2), abs((1.0 - x[1] - x[2]) - x3)))
    assert errs[0] > errs[1] > errs[2] and errs[2] < 3e-3, errs        # first order, down to the 1e-3 n_e approximation
    assert 0.05 < errs[1] / errs[0] < 0.3


# ------------------------------------------------------------------------------------------------ energy
def _cooling_paper(co, ne, nHI, nHII, nHeI, nHeII, nHeIII):
    """recombination, collisional ionisation, collisional excitation, bremsstrahlung - each process is
    n_e times the density of the particle that recombines / is ionised / is excited / scatters, times its coefficient
    from the table (indices as documented above orc_rate_coeffs); free-free per n_e Z^2 n_ion."""
    rec = co[6] * nHII + co[7] * nHeII + co[8] * nHeIII
    cion = co[9] * nHI + co[10] * nHeI + co[11] * nHeII
    cexc = co[12] * nHI + co[13] * nHeII
    ff = co[14] * (1.0 * nHII + 1.0 * nHeII + 4.0 * nHeIII)
    return ne * (rec + cion + cexc + ff)


ENERGY_STATES = [
    # name: the processes of PAPER.md:172 that carry the cooling there; Yp, T, x = (x_HI, x_HeI, x_HeII), heating per absorber (erg/s)
    ("ionised pure hydrogen: H II recombination + free-free", 0.0, 2e4, (1e-9, 1.0, 0.0), (0, 0, 0)),
    ("mostly neutral hydrogen at 2e4 K: Ly-alpha excitation + collisional ionisation of H I", 0.0, 2e4, (0.98, 1.0, 0.0), (0, 0, 0)),
    ("helium-rich, doubly ionised: He III recombination and Z^2 = 4 free-free", 0.9, 2e5, (1e-9, 1e-9, 1e-9), (0, 0, 0)),
    ("helium-rich, singly ionised at 1e5 K: He II excitation", 0.9, 1e5, (1e-9, 1e-3, 0.997), (0, 0, 0)),
    ("helium-rich, singly ionised at 2e4 K: He II recombination", 0.9, 2e4, (1e-9, 1e-3, 0.997), (0, 0, 0)),
    ("helium-rich, mostly neutral at 5e4 K: collisional ionisation of He I", 0.9, 5e4, (1e-9, 0.9, 0.1), (0, 0, 0)),
    ("helium-rich, singly ionised at 4e5 K: collisional ionisation of He II", 0.9, 4e5, (1e-9, 1e-6, 0.9), (0, 0, 0)),
    ("cold neutral gas, photo-heated: heating of all three absorbers", 0.24, 300.0, (0.9, 0.8, 0.15), (4e-24, 7e-24, 9e-24)),
]


@pytest.mark.parametrize("name,Yp,T,x,H", ENERGY_STATES, ids=[s[0].split(":")[0] for s in ENERGY_STATES])
def test_one_step_of_the_energy_equation(name, Yp, T, x, H):
    """arc_oracle.c `heat`, `cool`, `E`, `En = (E + heat dts)/(1 + (cool/E) dts)` and `Tn = En/(1.5 k_B n_tot)`
    (readings G16, G17).  One step (max_subcycles = 1: no limiter) from states chosen so that one or two processes of
    PAPER.md:172 carry the cooling; expected values typed from the paper's process list, E = 3/2 k_B T n_tot with
    n_tot = n_H + n_He + n_e.  A missing process, the wrong partner density, Z^2 missing in the free-free term,
    5/2 for 3/2, or T from the OLD electron density each fail."""
    nH = 5e-2
    p = _p(Yp=Yp, isothermal=0, coll_ion=1)
    co = orc.rate_coeffs(T, caseB=1, coll_ion=1)
    n_b = nH * A_H / (1.0 - Yp)
    nHe = n_b * Yp / A_HE
    x3 = 1.0 - x[1] - x[2]
    ne = _ne_paper(nH, Yp, 1.0 - x[0], x[2], x3)
    nHI, nHII, nHeI, nHeII, nHeIII = nH * x[0], nH * (1.0 - x[0]), nHe * x[1], nHe * x[2], nHe * x3
    cool = _cooling_paper(co, ne, nHI, nHII, nHeI, nHeII, nHeIII)
    heat = H[0] * nHI + H[1] * nHeI + H[2] * nHeII
    E = 1.5 * KB * T * (nH + nHe + ne)
    dt = 0.5 * E / max(cool, heat)                                # a step that changes E by tens of per cent
    G = [1e-14, 1e-14, 1e-15] if any(H) else [0.0, 0.0, 0.0]
    xn, Tn, k = orc.chem_cell(p, nH, list(x), T, G, list(H), dt)
    assert k == 1
    En = (E + heat * dt) / (1.0 + (cool / E) * dt)
    x3n = max(0.0, 1.0 - xn[1] - xn[2])
    ne_new = _ne_paper(nH, Yp, 1.0 - xn[0], xn[2], x3n)           # T from E with the NEW electron density
    T_want = En / (1.5 * KB * (nH + nHe + ne_new))
    assert abs(Tn / T_want - 1.0) < 1e-12, (name, Tn, T_want)
    assert abs(T_want / T - 1.0) > 0.05                           # the step did something


def test_cooling_terms_each_matter_in_the_state_that_isolates_them():
    """guards the table above: every one of the nine cooling coefficients (table entries 6..14) carries > 5 % of the
    cooling in at least one of the states, so a mistake in that term cannot hide inside the 1e-12 agreement"""
    nH = 5e-2
    best = {i: 0.0 for i in range(6, 15)}
    for name, Yp, T, x, H in ENERGY_STATES[:7]:
        co = orc.rate_coeffs(T, caseB=1, coll_ion=1)
        nHe = nH / (1.0 - Yp) * Yp / 4.0
        x3 = 1.0 - x[1] - x[2]
        ne = _ne_paper(nH, Yp, 1.0 - x[0], x[2], x3)
        dens = dict(nHI=nH * x[0], nHII=nH * (1.0 - x[0]), nHeI=nHe * x[1], nHeII=nHe * x[2], nHeIII=nHe * x3)
        tot = _cooling_paper(co, ne, **dens)
        for i in range(6, 15):
            z = np.array(co); z[i] = 0.0
            best[i] = max(best[i], 1.0 - _cooling_paper(z, ne, **dens) / tot)
    assert all(v > 0.05 for v in best.values()), best


def test_temperature_follows_the_particle_count_at_fixed_energy():
    """`Tn = En / (1.5 k_B (nH + nHe + ne_n))`, by hand: a tenuous cell (cooling negligible, no heating) whose hydrogen
    and He II are ionised within one step keeps its energy while the particle number grows from
    n_H + n_He + n_He (H I, He II + its electron) to 2 n_H + 3 n_He.  Y_p = 0.24: n_He/n_H = 0.24/(4 x 0.76) = 3/38,
    so T'/T = (1 + 6/38)/(2 + 9/38) = 44/85 = 0.517647 - i.e. mu goes from 1.136 to the textbook 0.588 of fully
    ionised primordial gas."""
    p = _p(Yp=0.24, isothermal=0, coll_ion=0)
    xn, Tn, k = orc.chem_cell(p, 1e-12, [1.0, 0.0, 1.0], 1e4, [1e-3, 0.0, 1e-3], [0, 0, 0], 1e12)
    assert k == 1 and xn[0] < 1e-8 and xn[2] < 1e-8
    assert abs(Tn / 1e4 - 44.0 / 85.0) < 1e-7, Tn
    mu_ionised = (1.0 + 4.0 * 3.0 / 38.0) / (2.0 + 9.0 / 38.0)
    assert abs(mu_ionised - 0.588) < 1e-3


def test_cooling_only_cell_follows_the_backward_difference_of_dE_dt():
    """`(cool / E) dts` in the denominator (Eq. 5 form with C = Lambda/E, reading G16): with the ionisation frozen
    (hot hydrogen held ionised by a strong Gamma_HI that carries no heat) and n steps of dt, E_n = E_0 prod 1/(1 + c_i dt)
    with c_i = Lambda(T_i)/E_i evaluated at the start of each step; for dt -> 0 this converges to the solution of
    dE/dt = -Lambda(T): checked against scipy's integration of that ODE."""
    from scipy.integrate import solve_ivp
    nH, T0 = 1e-1, 3e5
    p = _p(Yp=0.0, isothermal=0, coll_ion=0)
    ntot = 2.0 * nH

    def lam(T):
        co = orc.rate_coeffs(T, caseB=1, coll_ion=0)
        return nH * nH * (co[6] + co[14])                 # fully ionised pure H: recombination + free-free

    t_end = 0.5 * 1.5 * KB * T0 * ntot / lam(T0)
    sol = solve_ivp(lambda t, y: [-lam(y[0]) / (1.5 * KB * ntot)], (0.0, t_end), [T0], rtol=1e-10, atol=1e-3)
    T_ref = sol.y[0, -1]
    assert T_ref < 0.75 * T0
    errs = []
    for n in (20, 200, 2000):
        x, T = [1e-12, 1.0, 0.0], T0
        for _ in range(n):
            x, T, _ = orc.chem_cell(p, nH, [1e-12, 1.0, 0.0], T, [1e-3, 0, 0], [0, 0, 0], t_end / n)
        errs.append(abs(T / T_ref - 1.0))
    assert errs[0] > errs[1] > errs[2] and errs[2] < 2e-4 and 0.05 < errs[1] / errs[0] < 0.2, errs


def test_subcycled_update_converges_to_an_independent_integration_of_eq4_and_the_energy_equation():
    """The whole of orc_chem_cell (H + He, evolving T, sub-cycling with PAPER.md:152's limiter) against scipy's
    implicit integrator on the ODE system typed here from Eq. 4 and section 2.8: as eps -> 0 the sub-cycled backward
    differences must converge (first order) to the solution.  Catches a wrong coupling term, limiter, mu or cooling
    partner anywhere in the loop."""
    from scipy.integrate import solve_ivp
    nH, Yp, T0 = 1e-2, 0.24, 8e3
    G = [2e-12, 1.5e-12, 2e-13]
    Hh = [g * e * EV for g, e in zip(G, (4.0, 6.0, 10.0))]       # a few eV per ionisation
    n_b = nH / (1.0 - Yp)
    nHe = n_b * Yp / 4.0
    x_init = [0.99, 0.99, 0.01]
    t_end = 3e12

    def rhs(t, y):
        x0, x1, x2, E = y
        x3 = 1.0 - x1 - x2
        ne = _ne_paper(nH, Yp, 1.0 - x0, x2, x3)
        T = E / (1.5 * KB * (nH + nHe + ne))
        co = orc.rate_coeffs(T, caseB=1, coll_ion=1)
        d0 = -x0 * (G[0] + co[3] * ne) + co[0] * ne * (1.0 - x0)
        d1 = -x1 * (G[1] + co[4] * ne) + co[1] * ne * x2
        d3 = x2 * (G[2] + co[5] * ne) - co[2] * ne * x3
        d2 = -d1 - d3
        heat = Hh[0] * nH * x0 + Hh[1] * nHe * x1 + Hh[2] * nHe * x2
        cool = _cooling_paper(co, ne, nH * x0, nH * (1.0 - x0), nHe * x1, nHe * x2, nHe * x3)
        return [d0, d1, d2, heat - cool]

    ne0 = _ne_paper(nH, Yp, 1.0 - x_init[0], x_init[2], 0.0)
    E0 = 1.5 * KB * T0 * (nH + nHe + ne0)
    sol = solve_ivp(rhs, (0.0, t_end), x_init + [E0], method="Radau", rtol=1e-10, atol=[1e-14, 1e-14, 1e-14, 1e-30])
    x_ref = sol.y[:3, -1]
    x3r = 1.0 - x_ref[1] - x_ref[2]
    T_ref = sol.y[3, -1] / (1.5 * KB * (nH + nHe + _ne_paper(nH, Yp, 1.0 - x_ref[0], x_ref[2], x3r)))
    assert 8e3 < T_ref < 4e4 and x_ref[0] < 0.2                  # the cell really was heated and ionised
    errs = []
    for eps in (0.1, 0.01, 0.001):
        p = _p(Yp=Yp, isothermal=0, coll_ion=1, eps_sub=eps, max_subcycles=10 ** 7)
        xn, Tn, k = orc.chem_cell(p, nH, list(x_init), T0, G, Hh, t_end)
        errs.append(max(abs(Tn / T_ref - 1.0), *[abs(xn[i] - x_ref[i]) for i in range(3)]))
    assert errs[0] > errs[1] > errs[2] and errs[2] < 5e-4 and errs[1] / errs[0] < 0.3, errs


def test_thermal_equilibrium_temperature_is_the_root_of_heating_equals_cooling():
    """replaces the loose 5e3..4e4 K bound of test_thermal_equilibrium_is_around_1e4_K: a photo-heated pure-hydrogen cell
    run to its steady state must sit where Gamma x_HI = alpha n_e x_HII AND H x_HI n_H = Lambda(T) - the two roots are
    found here with brentq from the coefficient table."""
    from scipy.optimize import brentq
    nH, G, eps_heat = 1e-3, 1e-12, 5.0e-12
    p = _p(Yp=0.0, isothermal=0, coll_ion=1, max_subcycles=4096)

    def state(T):
        co = orc.rate_coeffs(T, caseB=1, coll_ion=1)
        # (Gamma + c n_H (1-x)) x = alpha n_H (1-x)^2
        x = brentq(lambda x: (G + co[3] * nH * (1 - x)) * x - co[0] * nH * (1 - x) ** 2, 0.0, 1.0, xtol=1e-16)
        ne = nH * (1 - x)
        return x, G * eps_heat * x * nH - _cooling_paper(co, ne, nH * x, ne, 0.0, 0.0, 0.0)

    T_eq = brentq(lambda T: state(T)[1], 3e3, 1e5, xtol=1e-6)
    x, T = [1.0 - 1.2e-3, 1.0, 0.0], 100.0
    for _ in range(400):
        x, T, _ = orc.chem_cell(p, nH, list(x), T, [G, 0, 0], [G * eps_heat, 0, 0], 3e14)
    assert abs(T / T_eq - 1.0) < 1e-5 and abs(x[0] / state(T_eq)[0] - 1.0) < 1e-5, (T, T_eq)
    assert 8e3 < T_eq < 3e4                                     # PAPER.md:172 "temperatures above 2e4 K is rare"


def test_subcycle_limiter_is_eps_times_E_over_Edot_and_n_over_ndot():
    """dt = min(eps E/|dE/dt|, eps n_HI/|dn_HI/dt|).  With max_subcycles = 2 the first sub-step is the
    limiter's and the second takes the rest; the state after the FIRST is reconstructed by hand for a cell where the
    energy term is the smaller one, and for one where the hydrogen term is."""
    for T, H0, which in ((200.0, 3e-22, "energy"), (2e4, 0.0, "hydrogen")):
        nH, x0, G0 = 1e-2, 0.6, 1e-12
        p1 = _p(Yp=0.0, isothermal=0, coll_ion=0, max_subcycles=2)
        co = orc.rate_coeffs(T, caseB=1, coll_ion=0)
        ne = nH * (1 - x0)
        xdot = co[0] * ne * (1 - x0) - G0 * x0
        heat = H0 * nH * x0
        cool = _cooling_paper(co, ne, nH * x0, ne, 0, 0, 0)
        E = 1.5 * KB * T * (nH + ne)
        lim_E, lim_n = 0.1 * E / abs(heat - cool), 0.1 * x0 / abs(xdot)
        assert (lim_E < lim_n) == (which == "energy")
        d1 = min(lim_E, lim_n)
        dt = 5.0 * d1
        # first sub-step by hand
        xa = (x0 + co[0] * ne * (1 - x0) * d1) / (1 + G0 * d1)
        Ea = (E + heat * d1) / (1 + cool / E * d1)
        Ta = Ea / (1.5 * KB * (nH + nH * (1 - xa)))
        # second (last allowed) sub-step takes all the time left (reading G15)
        xb, Tb, kb = orc.chem_cell(_p(Yp=0.0, isothermal=0, coll_ion=0, max_subcycles=1), nH, [xa, 1.0, 0.0], Ta, [G0, 0, 0], [H0, 0, 0], dt - d1)
        xg, Tg, kg = orc.chem_cell(p1, nH, [x0, 1.0, 0.0], T, [G0, 0, 0], [H0, 0, 0], dt)
        assert kg == 2 and kb == 1
        assert abs(xg[0] / xb[0] - 1) < 1e-12 and abs(Tg / Tb - 1) < 1e-12, which


# ------------------------------------------------------------------------------------------------ rate table
def test_collisional_excitation_cooling_has_the_lyman_alpha_thresholds_and_magnitude():
    """out[12], out[13] of orc_rate_coeffs.  (i) the Boltzmann factors: the excitation energy of n = 1 -> 2 is 3/4 of the
    ionisation energy, 118 348 K for H I and 473 638 K for He II; read off the oracle as the slope of
    ln[coefficient x (1 + sqrt(T/1e5)) (x T^0.397 for He II)] against 1/T.  (ii) the magnitude: collisional excitation
    cooling = E_12 x 8.629e-6 / (g_1 sqrt(T)) x Omega(T) e^{-E_12/kT} with the effective collision strengths of the
    1s -> 2s, 2p transitions (textbook table, tests/golden/textbook_rates.txt; hydrogenic scaling Omega/Z^2 at T/Z^2
    for He II).  The classic fit sits within 25 % of that for H I around 1e4 K and within a factor two for He II."""
    def slope(i, extra):
        T1, T2 = 1.2e4, 6e4
        f = lambda T: math.log(orc.rate_coeffs(T)[i] * (1.0 + math.sqrt(T / 1e5)) * extra(T))
        return -(f(T1) - f(T2)) / (1.0 / T1 - 1.0 / T2)
    th_H = slope(12, lambda T: 1.0)
    th_He = slope(13, lambda T: T ** 0.397)
    assert abs(th_H / (0.75 * 13.598 / KB_EV) - 1.0) < 2e-4, th_H
    assert abs(th_He / (0.75 * 54.418 / KB_EV) - 1.0) < 2e-4, th_He
    om = _golden("omega_H_n2_")                               # key = temperature, value = Omega(1s-2s) + Omega(1s-2p)
    assert len(om) == 3
    for Tk, (omega, tol) in om.items():
        T = float(Tk)
        E12 = 0.75 * 13.598 * EV
        want = E12 * 8.629e-6 / (2.0 * math.sqrt(T)) * omega * math.exp(-E12 / (KB * T))
        got = orc.rate_coeffs(T)[12]
        assert abs(got / want - 1.0) < tol, (T, got, want)
        # He II at 4 T: Omega_H(T)/4, E_12 x 4
        TZ = 4.0 * T
        wantZ = 4.0 * E12 * 8.629e-6 / (2.0 * math.sqrt(TZ)) * (omega / 4.0) * math.exp(-4.0 * E12 / (KB * TZ))
        gotZ = orc.rate_coeffs(TZ)[13]
        assert 0.5 < gotZ / wantZ < 2.0, (TZ, gotZ, wantZ)


def test_free_free_cooling_is_the_textbook_emissivity():
    """out[14]: 1.42e-27 g_ff sqrt(T) erg cm^3/s per n_e n_ion Z^2 (thermal bremsstrahlung, frequency-integrated), with
    a Gaunt factor inside the textbook range 1.1-1.5 that peaks near 10^5.5 K."""
    g = {T: orc.rate_coeffs(T)[14] / (1.42e-27 * math.sqrt(T)) for T in (1e3, 1e4, 10 ** 5.5, 1e7, 1e8)}
    assert all(1.1 <= v <= 1.5 for v in g.values()), g
    assert g[10 ** 5.5] == max(g.values()) and abs(g[10 ** 5.5] - 1.44) < 1e-12
    assert abs(g[1e4] - 1.26) < 0.01 and abs(g[1e8] - 1.1) < 0.05


def test_dielectronic_recombination_of_helium():
    """`ad` in orc_rate_coeffs and its cooling.  (i) the published parameters of Aldrovandi & Pequignot (1973) for He+
    (tests/golden/textbook_rates.txt), evaluated here in their general form A T^-3/2 e^{-T0/T} (1 + B e^{-T1/T});
    (ii) physics the numbers must obey: the capture goes through the 1s -> 2p excitation of the core, so T0 is 3/4 of
    the He II ionisation energy (40.8 eV) within 1 % and each capture radiates that energy (6.54e-11 erg);
    dielectronic recombination is negligible below 3e4 K and exceeds the radiative rate tenfold at 1e5-2e5 K."""
    (A, T0, B, T1), = [v for v in _golden("dielectronic_HeII").values()]
    assert abs(T0 * KB_EV / (0.75 * 54.418) - 1.0) < 0.01
    for T in (5e4, 1e5, 2e5, 1e6):
        rad = 1.26e-14 * (2.0 * 285335.0 / T) ** 0.75          # case-B radiative part: pinned at 1e4 K by the textbook table
        co = orc.rate_coeffs(T, caseB=1)
        ad = A * T ** -1.5 * math.exp(-T0 / T) * (1.0 + B * math.exp(-T1 / T))
        assert abs((co[1] - rad) / ad - 1.0) < 1e-9, (T, co[1] - rad, ad)
        # cooling: k_B T per radiative recombination + the 2p -> 1s photon per dielectronic capture
        e_capture = (co[7] - KB * T * rad) / ad
        assert abs(e_capture / (0.75 * 54.418 * EV) - 1.0) < 2e-3, e_capture
    lo = orc.rate_coeffs(3e4, caseB=1)
    assert (lo[1] - 1.26e-14 * (2.0 * 285335.0 / 3e4) ** 0.75) / lo[1] < 1e-2
    for T in (1e5, 2e5):
        co = orc.rate_coeffs(T, caseB=1)
        assert co[1] > 10.0 * 1.26e-14 * (2.0 * 285335.0 / T) ** 0.75


# ------------------------------------------------------------------------------------------------ opacity table
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_opacity_of_three_hand_worked_cells(dtype):
    """orc_opacity (PAPER.md:67 "total optical depth due to all atomic species ... for each frequency bin", :81):
    kappa_nu = sum_S sigma_S,nu n_S.  Y_p = 0.2 makes n_He = n_H 0.2/(4 x 0.8) = n_H/16; the numbers below are worked
    by hand, not with the oracle's expression."""
    w = wl.tiny(N=2, nb=3, dtype=dtype)
    w.sig_HI = np.array([6e-18, 2e-18, 1e-18]); w.sig_HeI = np.array([0.0, 4e-18, 2e-18]); w.sig_HeII = np.array([0.0, 0.0, 1e-18])
    nH = np.array([1.6e-2, 1.0, 4e-3] + [1.0] * 5)
    xHI = np.array([0.5, 1.0, 0.0] + [0.0] * 5)
    xHeI = np.array([0.25, 1.0, 0.0] + [0.0] * 5)
    xHeII = np.array([0.5, 0.0, 1.0] + [0.0] * 5)
    dt = np.float32 if dtype == "f32" else np.float64
    fields = tuple(a.astype(dt) for a in (nH, xHI, xHeI, xHeII, np.full(8, 1e4)))
    k = orc.opacity(w, fields, Yp=0.2)
    want = np.array([[4.8e-20, 1.7e-20, 9.0e-21],            # n_HI 8e-3, n_HeI 2.5e-4, n_HeII 5e-4
                     [6.0e-18, 2.25e-18, 1.125e-18],         # neutral: n_HI 1, n_HeI 1/16
                     [0.0, 0.0, 2.5e-22]])                   # H II + He II only: n_HeII 2.5e-4
    if dtype == "f64":
        assert np.allclose(k[:3], want, rtol=1e-14, atol=0.0)
    else:
        # fp32 fields: the inputs are the fp32-rounded values, the table is rounded to fp32 (contract C5)
        assert np.allclose(k[:3], want, rtol=3e-7, atol=0.0)
        assert np.array_equal(k, k.astype(np.float32).astype(np.float64))
    assert np.all(k[3:] == 0.0)                              # fully ionised to He III: transparent
