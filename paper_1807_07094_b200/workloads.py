"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves BOTH the CPU oracle (tests, bench cpu_baseline) and the CUDA
path.  It holds none of the method's arithmetic: no ray geometry, no optical
depths, no rate coefficients - only what a user would hand to the library
(grid fields, source list, frequency bins with their cross-sections, and the
run parameters).  Everything is numpy on the host, seeded with
``default_rng(180707094 + config number)``.

Where the paper measured on the RT06 comparison-project density field and halo
list - files that are not available here - the seeded lognormal
fields below stand in for that workload's shape (DESIGN.md says so too).
"""
from __future__ import annotations

import functools
from dataclasses import dataclass, field
import numpy as np

KPC_CM = 3.0856775814913673e21
MYR_S = 3.15576e13
SEED0 = 180707094

# ionization thresholds [eV] and threshold cross-sections [cm^2]: INPUTS to the
# library (arc_set_spectrum), not library constants.
E_HI, E_HEI, E_HEII = 13.598, 24.587, 54.418
SIG0_HI, SIG0_HEI, SIG0_HEII = 6.30e-18, 7.4e-18, 1.58e-18

# the one coefficient the paper pins: t_rec = 122.4 Myr at n_H = 1e-3
ALPHA_B_1E4 = 2.59e-13


@dataclass
class Workload:
    name: str
    N: int
    box_cm: float
    dtype: str                      # "f32" | "f64" : dtype of the five gas fields
    n_H: np.ndarray                 # [N^3] x-fastest, index (iz*N+iy)*N+ix
    x_HI: np.ndarray
    x_HeI: np.ndarray
    x_HeII: np.ndarray
    T: np.ndarray
    E_eV: np.ndarray                # [nb]
    sig_HI: np.ndarray              # [nb] cm^2
    sig_HeI: np.ndarray
    sig_HeII: np.ndarray
    src_pos_cm: np.ndarray          # [nsrc,3]
    src_Ndot: np.ndarray            # [nsrc] photons/s
    src_binfrac: np.ndarray         # [nsrc,nb], rows sum to 1
    dt_s: float
    n_steps: int
    params: dict = field(default_factory=dict)   # l0, Phi, Lmax, tau_term, Yp, isothermal, caseB, coll_ion...

    @property
    def nb(self) -> int:
        return int(self.E_eV.shape[0])

    @property
    def nsrc(self) -> int:
        return int(self.src_Ndot.shape[0])

    @property
    def ncell(self) -> int:
        return self.N ** 3

    def fields(self):
        return self.n_H, self.x_HI, self.x_HeI, self.x_HeII, self.T


DEFAULT_PARAMS = dict(l0=1, Phi=3.0, Lmax=13, tau_term=30.0, Yp=0.0, isothermal=1,
                      caseB=1, coll_ion=0, eps_sub=0.1, max_subcycles=4096, x_floor=1e-12)


def _np_dtype(dtype: str):
    return np.float32 if dtype == "f32" else np.float64


def _cell_centre_cm(ijk, N, box_cm):
    return (np.asarray(ijk, dtype=np.float64) + 0.5) * (box_cm / N)


def mono_spectrum(E=13.6, sig=SIG0_HI):
    return (np.array([E]), np.array([sig]), np.array([0.0]), np.array([0.0]))


def powerlaw_spectrum(edges_eV, alpha=-1.5):
    """Bins between `edges_eV`; photon-number spectrum dN/dE ~ E^(alpha-1) so that the photon
    fraction of a bin is ~ E_lo^alpha - E_hi^alpha (alpha = -1.5: SURVEY 8(d) config 3).
    Bin energy = photon-weighted mean energy; cross-sections sigma_S0 (E/E_S)^-3 above
    threshold, evaluated at the bin energy."""
    e = np.asarray(edges_eV, dtype=np.float64)
    lo, hi = e[:-1], e[1:]
    w = lo ** alpha - hi ** alpha
    frac = w / w.sum()
    # <E> = int E * E^(alpha-1) dE / int E^(alpha-1) dE
    a1 = alpha + 1.0
    num = (hi ** a1 - lo ** a1) / a1
    den = (hi ** alpha - lo ** alpha) / alpha
    E = num / den

    def sig(E0, s0):
        return np.where(E >= E0, s0 * (E / E0) ** -3.0, 0.0)

    return E, sig(E_HI, SIG0_HI), sig(E_HEI, SIG0_HEI), sig(E_HEII, SIG0_HEII), frac


def gaussian_field(N, rng, kmax=None):
    """Unit-variance Gaussian random field: white noise filtered in Fourier space with
    amplitude ~ 1/k for k >= 1 (k in fundamental units), optionally band-limited to k <= kmax."""
    wn = rng.standard_normal((N, N, N))
    fk = np.fft.rfftn(wn)
    kx = np.fft.fftfreq(N, d=1.0 / N)
    kz = np.fft.rfftfreq(N, d=1.0 / N)
    k = np.sqrt(kx[:, None, None] ** 2 + kx[None, :, None] ** 2 + kz[None, None, :] ** 2)
    amp = np.zeros_like(k)
    m = k >= 1.0
    amp[m] = 1.0 / k[m]
    if kmax is not None:
        amp[k > kmax] = 0.0
    g = np.fft.irfftn(fk * amp, s=(N, N, N), axes=(0, 1, 2))
    g -= g.mean()
    g /= g.std()
    return g


def lognormal_density(N, rng, sigma_ln, mean=1e-3, kmax=None):
    g = gaussian_field(N, rng, kmax=kmax)
    return mean * np.exp(sigma_ln * g - 0.5 * sigma_ln ** 2)


def density_peaks(n3, count):
    """Cells (ix,iy,iz) and values of the `count` highest 26-neighbour local maxima of n3[z,y,x], highest first."""
    from scipy.ndimage import maximum_filter
    mx = maximum_filter(n3, size=3, mode="nearest")
    cand = np.flatnonzero((n3 == mx).ravel())
    vals = n3.ravel()[cand]
    order = np.argsort(-vals, kind="stable")[:count]          # (count = None: all of them)
    idx = cand[order]
    if count is not None and idx.size < count:
        raise ValueError(f"only {idx.size} local maxima, need {count}")
    iz, iy, ix = np.unravel_index(idx, n3.shape)
    return np.stack([ix, iy, iz], axis=1), vals[order]


# ----------------------------------------------------------------------------------------------
def config1(N=32):
    """32^3 uniform, box 6 kpc, fp64, x_HI = 1, T = 1e4 K fixed, 1 central source 1e48 s^-1,
    13.6 eV, l0 = 0, Phi = 3, 10 steps of 0.1 t_rec."""
    box = 6.0 * KPC_CM
    n = N ** 3
    E, s1, s2, s3 = mono_spectrum()
    t_rec = 1.0 / (ALPHA_B_1E4 * 1e-3)
    p = dict(DEFAULT_PARAMS, l0=0)
    c = N // 2
    return Workload("config1", N, box, "f64",
                    np.full(n, 1e-3), np.full(n, 1.0), np.full(n, 1.0), np.zeros(n), np.full(n, 1e4),
                    E, s1, s2, s3,
                    _cell_centre_cm([[c, c, c]], N, box), np.array([1e48]), np.array([[1.0]]),
                    0.1 * t_rec, 10, p)


def config2(N=128, dtype="f64"):
    """128^3 uniform pure-H Stromgren test, box 15 kpc (reading G20), x_HII,0 = 1.2e-3, T = 1e4 K
    isothermal, centred source 5e48 s^-1, 13.6 eV, l0 = 1, Phi = 3, 100 steps of 0.05 t_rec."""
    box = 15.0 * KPC_CM
    n = N ** 3
    dt = _np_dtype(dtype)
    E, s1, s2, s3 = mono_spectrum()
    t_rec = 1.0 / (ALPHA_B_1E4 * 1e-3)
    c = N // 2
    return Workload("config2", N, box, dtype,
                    np.full(n, 1e-3, dt), np.full(n, 1.0 - 1.2e-3, dt), np.full(n, 1.0, dt),
                    np.zeros(n, dt), np.full(n, 1e4, dt),
                    E, s1, s2, s3,
                    _cell_centre_cm([[c, c, c]], N, box), np.array([5e48]), np.array([[1.0]]),
                    0.05 * t_rec, 100, dict(DEFAULT_PARAMS))


def _clumpy(N, rng, sigma_ln, kmax=None):
    n3 = lognormal_density(N, rng, sigma_ln, kmax=kmax)     # [z,y,x]
    return n3


def config3(N=128, nsrc=16, dtype="f64"):
    """128^3 lognormal (sigma_ln = 1) + one dense clump (200x mean, radius 8 cells), 16 sources at
    seeded uniform cell centres, Ndot log-uniform 1e47..1e49, 3 bins (H, HeI, HeII edges),
    H+He Yp = 0.24, T evolving from 100 K; 10 steps of dt = 0.05 N_atoms/sum(Ndot)."""
    rng = np.random.default_rng(SEED0 + 3)
    box = 15.0 * KPC_CM
    n3 = _clumpy(N, rng, 1.0)
    rad = 8.0 * N / 128.0
    cc = rng.integers(int(rad) + 2, N - int(rad) - 2, size=3)          # clump centre (ix,iy,iz)
    zz, yy, xx = np.meshgrid(np.arange(N), np.arange(N), np.arange(N), indexing="ij")
    d2 = (xx - cc[0]) ** 2 + (yy - cc[1]) ** 2 + (zz - cc[2]) ** 2
    n3[d2 <= rad * rad] = 200.0 * 1e-3
    # sources: uniform cell centres at least 12 cells (scaled) from the clump centre
    src = []
    while len(src) < nsrc:
        c = rng.integers(0, N, size=3)
        if np.sum((c - cc) ** 2) >= (12.0 * N / 128.0) ** 2 and not any((c == s).all() for s in src):
            src.append(c)
    src = np.array(src)
    Ndot = 10.0 ** rng.uniform(47.0, 49.0, size=nsrc)
    E, s1, s2, s3, frac = powerlaw_spectrum([E_HI, E_HEI, E_HEII, 200.0])
    dtp = _np_dtype(dtype)
    n = N ** 3
    nH = n3.ravel().astype(dtp)
    dx = box / N
    n_atoms = float(n3.sum()) * dx ** 3
    p = dict(DEFAULT_PARAMS, Yp=0.24, isothermal=0, caseB=1, coll_ion=1)
    w = Workload("config3", N, box, dtype,
                 nH, np.full(n, 1.0 - 1.2e-3, dtp), np.full(n, 1.0 - 1.2e-3, dtp),
                 np.full(n, 1.2e-3, dtp), np.full(n, 100.0, dtp),
                 E, s1, s2, s3,
                 _cell_centre_cm(src, N, box), Ndot, np.tile(frac, (nsrc, 1)),
                 0.05 * n_atoms / Ndot.sum(), 10, p)
    w.params["_clump_centre"] = cc.tolist()
    return w


@functools.lru_cache(maxsize=2)
def _peaks_field(N, sigma_ln, seed, kmax):
    """the density field of configs 4 / 5 and its local maxima in decreasing order (cached: a source-count sweep on one
    grid shares them; the 512^3 field takes half a minute to make)"""
    rng = np.random.default_rng(seed)
    n3 = _clumpy(N, rng, sigma_ln, kmax=kmax)
    pk, vals = density_peaks(n3, None)
    for a in (n3, pk, vals):
        a.setflags(write=False)
    return n3, pk, vals


def _peaks_workload(name, N, nsrc, sigma_ln, seed, n_steps, kmax=None, state="neutral"):
    box = 15.0 * KPC_CM
    n3, pk, vals = _peaks_field(N, sigma_ln, seed, kmax)
    if len(vals) < nsrc:
        raise ValueError(f"only {len(vals)} local maxima, need {nsrc}")
    pk, vals = pk[:nsrc].copy(), vals[:nsrc].copy()
    Ndot = 1e48 * vals / vals.mean()
    E, s1, s2, s3, frac = powerlaw_spectrum([E_HI, E_HEI, E_HEII, 100.0, 200.0])
    n = N ** 3
    dtp = np.float32
    dx = box / N
    n_atoms = float(n3.sum()) * dx ** 3
    p = dict(DEFAULT_PARAMS, Yp=0.24, isothermal=0, caseB=1, coll_ion=1)
    if state == "transparent":           # config 5 state (B): every ray crosses the box
        xn, xe = 1e-6, 1e-6
        p["tau_term"] = float("inf")
        x_HI = np.full(n, xn, dtp); x_HeI = np.full(n, xn, dtp); x_HeII = np.full(n, 1.0 - 2e-6, dtp)
        T = np.full(n, 1e4, dtp)
    else:
        x_HI = np.full(n, 1.0 - 1.2e-3, dtp); x_HeI = np.full(n, 1.0 - 1.2e-3, dtp)
        x_HeII = np.full(n, 1.2e-3, dtp); T = np.full(n, 100.0, dtp)
    return Workload(name + ("_T" if state == "transparent" else ""), N, box, "f32", n3.ravel().astype(dtp), x_HI, x_HeI, x_HeII, T,
                    E, s1, s2, s3, _cell_centre_cm(pk, N, box), Ndot, np.tile(frac, (nsrc, 1)),
                    0.05 * n_atoms / Ndot.sum(), n_steps, p)


def config4(N=256, nsrc=1024, state="neutral"):
    """256^3 lognormal sigma_ln = 1.5, 1024 sources at the highest density peaks, Ndot ~ peak
    density, 4 bins power-law alpha = -1.5, fp32 fields / fp64 accumulation, 20 steps."""
    return _peaks_workload("config4", N, nsrc, 1.5, SEED0 + 4, 20, state=state)


def config5(N=512, nsrc=1024, state="neutral"):
    """512^3 (and the 128..512 grid sweep): same realisation band-limited to the 128^3 modes
    (k <= 64) so that refining the grid keeps the physical field."""
    return _peaks_workload(f"config5_N{N}_S{nsrc}", N, nsrc, 1.5, SEED0 + 5, 1, kmax=64.0, state=state)


def by_name(name: str, **kw) -> Workload:
    return {"config1": config1, "config2": config2, "config3": config3,
            "config4": config4, "config5": config5}[name](**kw)


def tiny(N=8, nsrc=2, nb=2, seed=7, dtype="f64", Yp=0.24, l0=0, Phi=3.0, tau_term=30.0,
         kappa_scale=1.0, off_centre=True):
    """Small random workload for brute-force / parity unit tests: lognormal-ish density, sources at
    random (optionally off-centre, non cell-centre) positions, nb bins."""
    rng = np.random.default_rng(seed)
    box = 1.0 * KPC_CM * N / 8.0
    n = N ** 3
    dtp = _np_dtype(dtype)
    nH = (1e-2 * kappa_scale * np.exp(rng.normal(0, 1.0, n))).astype(dtp)
    x_HI = rng.uniform(0.05, 1.0, n).astype(dtp)
    x_HeI = rng.uniform(0.05, 0.9, n)
    x_HeII = ((1.0 - x_HeI) * rng.uniform(0.0, 1.0, n)).astype(dtp)
    x_HeI = x_HeI.astype(dtp)
    T = (10.0 ** rng.uniform(2.0, 4.5, n)).astype(dtp)
    edges = [E_HI, E_HEI, E_HEII, 100.0, 200.0, 400.0, 800.0, 1600.0, 3200.0][: nb + 1]
    if nb == 1:
        E, s1, s2, s3 = mono_spectrum(); frac = np.array([1.0])
    else:
        E, s1, s2, s3, frac = powerlaw_spectrum(edges)
    if off_centre:
        pos = rng.uniform(0.05, 0.95, (nsrc, 3)) * box
    else:
        pos = _cell_centre_cm(rng.integers(0, N, (nsrc, 3)), N, box)
    Ndot = 10.0 ** rng.uniform(46.0, 48.0, nsrc)
    p = dict(DEFAULT_PARAMS, l0=l0, Phi=Phi, tau_term=tau_term, Yp=Yp, isothermal=0, coll_ion=1)
    dx = box / N
    n_atoms = float(nH.astype(np.float64).sum()) * dx ** 3
    return Workload(f"tiny{N}", N, box, dtype, nH, x_HI, x_HeI, x_HeII, T, E, s1, s2, s3,
                    pos, Ndot, np.tile(frac, (nsrc, 1)), 0.05 * n_atoms / Ndot.sum(), 2, p)
