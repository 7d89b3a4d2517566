"""ctypes wrapper around oracle/arc_oracle.c -- CPU ORACLE, TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may import
this.  It never imports the CUDA package's binding and shares no code with it; the only thing both
sides consume is a `Workload` object (plain numpy arrays) from the seeded input generators.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "arc_oracle.c")
# ARC_ORACLE_SANITIZE=1: the same source built with -fsanitize=address,undefined into a library of its own (run the
# oracle's pin tests under it with LD_PRELOAD=$(gcc -print-file-name=libasan.so); profiles/r02_sanitizers.md)
_SAN = os.environ.get("ARC_ORACLE_SANITIZE", "") not in ("", "0")
_LIB = os.path.join(_HERE, "libarc_oracle_san.so" if _SAN else "libarc_oracle.so")

MAXNB, MAXLEVEL = 8, 16
END_SPLIT, END_DEPLETED, END_ESCAPED = 0, 1, 2


def build(force: bool = False) -> str:
    """gcc -O2, no FMA contraction, no fast-math (arithmetic contract C0)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        san = ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if _SAN else []
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fno-fast-math", "-shared",
                               "-fPIC"] + san + ["-o", _LIB, _SRC, "-lm"])
    return _LIB


class Params(C.Structure):
    _fields_ = [("N", C.c_int32), ("field_dtype", C.c_int32), ("box_cm", C.c_double),
                ("l0", C.c_int32), ("Lmax", C.c_int32), ("Phi", C.c_double), ("tau_term", C.c_double),
                ("Yp", C.c_double), ("isothermal", C.c_int32), ("caseB", C.c_int32),
                ("coll_ion", C.c_int32), ("max_subcycles", C.c_int32), ("eps_sub", C.c_double),
                ("x_floor", C.c_double), ("geom_corr", C.c_int32), ("pad_", C.c_int32), ("thin_tau", C.c_double)]


class Stats(C.Structure):
    _fields_ = [("segments", C.c_uint64), ("rays", C.c_uint64), ("digest", C.c_uint64),
                ("max_stack", C.c_uint64), ("splits", C.c_uint64 * MAXLEVEL),
                ("rays_level", C.c_uint64 * MAXLEVEL), ("ends", C.c_uint64 * 3),
                ("emitted", C.c_double * MAXNB), ("absorbed", C.c_double * MAXNB),
                ("escaped", C.c_double * MAXNB)]


class RayLog(C.Structure):
    _fields_ = [("cap_rays", C.c_int64), ("cap_cells", C.c_int64), ("n_rays", C.c_int64),
                ("n_cells", C.c_int64), ("src", C.c_void_p), ("level", C.c_void_p), ("pix", C.c_void_p),
                ("end", C.c_void_p), ("first", C.c_void_p), ("count", C.c_void_p), ("r_end", C.c_void_p),
                ("cells", C.c_void_p), ("ds", C.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        assert _lib.orc_sizeof_params() == C.sizeof(Params)
        assert _lib.orc_sizeof_stats() == C.sizeof(Stats)
        _lib.orc_rsplit.restype = C.c_double
        _lib.orc_rsplit.argtypes = [C.c_double, C.c_int, C.c_int]
        _lib.orc_chemistry.restype = C.c_int64
        _lib.orc_pix2vec.argtypes = [C.c_int, C.c_uint64, C.c_void_p]
        _lib.orc_pix2ring.argtypes = [C.c_int, C.c_uint64] + [C.c_void_p] * 4
        _lib.orc_sincos_frac.argtypes = [C.c_int64, C.c_int64, C.c_void_p, C.c_void_p]
        _lib.orc_rate_coeffs.argtypes = [C.c_double, C.c_int, C.c_int, C.c_void_p]
    return _lib


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def make_params(w, **override) -> Params:
    d = dict(w.params)
    d.update(override)
    return Params(N=w.N, field_dtype=0 if w.dtype == "f32" else 1, box_cm=w.box_cm, l0=int(d["l0"]),
                  Lmax=int(d["Lmax"]), Phi=float(d["Phi"]), tau_term=float(d["tau_term"]),
                  Yp=float(d["Yp"]), isothermal=int(d["isothermal"]), caseB=int(d["caseB"]),
                  coll_ion=int(d["coll_ion"]), max_subcycles=int(d["max_subcycles"]),
                  eps_sub=float(d["eps_sub"]), x_floor=float(d["x_floor"]), geom_corr=int(d.get("geom_corr", 0)), thin_tau=float(d.get("thin_tau", 0.0)))


# ---- O1/O2 -------------------------------------------------------------------------------
def pix2vec(level: int, pix: int) -> np.ndarray:
    d = np.zeros(3)
    lib().orc_pix2vec(level, pix, _p(d))
    return d


def pix2ring(level: int, pix: int):
    """-> (zn, zd, m, nr): z = zn/zd exactly, phi = m*pi/(4*nr)."""
    o = np.zeros(4, dtype=np.int64)
    b = o.ctypes.data
    lib().orc_pix2ring(level, pix, C.c_void_p(b), C.c_void_p(b + 8), C.c_void_p(b + 16), C.c_void_p(b + 24))
    return tuple(int(v) for v in o)


def sincos_frac(m: int, nr: int):
    o = np.zeros(2)
    lib().orc_sincos_frac(m, nr, C.c_void_p(o.ctypes.data), C.c_void_p(o.ctypes.data + 8))
    return float(o[0]), float(o[1])


def rsplit(Phi: float, level: int, Lmax: int = 13) -> float:
    return float(lib().orc_rsplit(Phi, level, Lmax))


def rate_coeffs(T: float, caseB: int = 1, coll_ion: int = 1) -> np.ndarray:
    o = np.zeros(15)
    lib().orc_rate_coeffs(float(T), int(caseB), int(coll_ion), _p(o))
    return o


# ---- O3-O6 -------------------------------------------------------------------------------
def opacity(w, fields=None, **override) -> np.ndarray:
    """kappa[cell, v] (fp64 array holding values rounded to the field dtype)."""
    p = make_params(w, **override)
    nH, xHI, xHeI, xHeII, _ = [_f64(a) for a in (fields or w.fields())]
    k = np.zeros((w.ncell, w.nb))
    lib().orc_opacity(C.byref(p), w.nb, _p(nH), _p(xHI), _p(xHeI), _p(xHeII), _p(_f64(w.sig_HI)),
                      _p(_f64(w.sig_HeI)), _p(_f64(w.sig_HeII)), _p(k))
    return k


def trace(w, kappa=None, fields=None, log=False, cap_rays=2_000_000, cap_cells=60_000_000,
          sources=None, blocked=None, Rstart=None, **override):
    """-> (A[cell, v] absorbed photons/s, stats dict, raylog dict or None).
    blocked: None or uint8 [nsrc, 12 4^l0], non-zero = root ray blocked (anisotropic emission).
    With thin_tau > 0 (optically thin inner region): Rstart = per-source radii [cells] found by the
    previous trace (None = 0), and stats["R_thin"] = the radii this trace found."""
    p = make_params(w, **override)
    if kappa is None:
        kappa = opacity(w, fields, **override)
    kappa = _f64(kappa)
    pos, Nd, bf = _f64(w.src_pos_cm), _f64(w.src_Ndot), _f64(w.src_binfrac)
    if sources is not None:
        sources = np.asarray(sources)
        pos, Nd, bf = _f64(pos[sources]), _f64(Nd[sources]), _f64(bf[sources])
    A = np.zeros((w.ncell, w.nb))
    st = Stats()
    rl = None
    keep = []
    if log:
        rl = RayLog(cap_rays=cap_rays, cap_cells=cap_cells)
        arrs = dict(src=np.zeros(cap_rays, np.int32), level=np.zeros(cap_rays, np.int32),
                    pix=np.zeros(cap_rays, np.int64), end=np.zeros(cap_rays, np.int32),
                    first=np.zeros(cap_rays, np.int64), count=np.zeros(cap_rays, np.int32),
                    r_end=np.zeros(cap_rays), cells=np.zeros(cap_cells, np.int32), ds=np.zeros(cap_cells))
        for k, v in arrs.items():
            setattr(rl, k, v.ctypes.data)
        keep = arrs
    bl = None
    if blocked is not None:
        bl = np.ascontiguousarray(blocked, dtype=np.uint8)
        if sources is not None:
            bl = np.ascontiguousarray(bl[sources])
        assert bl.shape == (len(Nd), 12 << (2 * p.l0))
    Rs = None
    if Rstart is not None:
        Rs = _f64(np.asarray(Rstart, dtype=np.float64))
        if sources is not None and len(Rs) != len(Nd):
            Rs = _f64(Rs[sources])
        assert Rs.shape == (len(Nd),)
    Rn = np.zeros(len(Nd))
    rc = lib().orc_trace_thin(C.byref(p), w.nb, _p(kappa), len(Nd), _p(pos), _p(Nd), _p(bf),
                              _p(bl) if bl is not None else None, _p(Rs) if Rs is not None else None, _p(Rn), _p(A),
                              C.byref(st), C.byref(rl) if rl is not None else None)
    if rc != 0:
        raise RuntimeError(f"orc_trace failed: {rc}")
    nb = w.nb
    stats = dict(segments=int(st.segments), rays=int(st.rays), digest=int(st.digest),
                 max_stack=int(st.max_stack), splits=np.array(st.splits[:], dtype=np.uint64),
                 rays_level=np.array(st.rays_level[:], dtype=np.uint64), ends=np.array(st.ends[:], dtype=np.uint64),
                 emitted=np.array(st.emitted[:nb]), absorbed=np.array(st.absorbed[:nb]),
                 escaped=np.array(st.escaped[:nb]), R_thin=Rn)
    raylog = None
    if log:
        nr, ncs = int(rl.n_rays), int(rl.n_cells)
        raylog = {k: (v[:ncs] if k in ("cells", "ds") else v[:nr]) for k, v in keep.items()}
    return A, stats, raylog


def raylog_to_dict(raylog):
    """{(src, level, pix): (tuple(cells), end)}"""
    out = {}
    cells = raylog["cells"]
    for i in range(len(raylog["src"])):
        f, n = int(raylog["first"][i]), int(raylog["count"][i])
        out[(int(raylog["src"][i]), int(raylog["level"][i]), int(raylog["pix"][i]))] = (
            tuple(cells[f:f + n].tolist()), int(raylog["end"][i]))
    return out


def finalize(w, A, fields=None, **override):
    """-> Gamma[3, nc] (1/s per absorber), heat[3, nc] (erg/s per absorber), heat_total[nc] (erg/s/cm^3)."""
    p = make_params(w, **override)
    nH, xHI, xHeI, xHeII, _ = [_f64(a) for a in (fields or w.fields())]
    G = np.zeros((3, w.ncell)); H = np.zeros((3, w.ncell)); Ht = np.zeros(w.ncell)
    lib().orc_finalize(C.byref(p), w.nb, _p(_f64(A)), _p(nH), _p(xHI), _p(xHeI), _p(xHeII), _p(_f64(w.E_eV)),
                       _p(_f64(w.sig_HI)), _p(_f64(w.sig_HeI)), _p(_f64(w.sig_HeII)), _p(G), _p(H), _p(Ht))
    return G, H, Ht


def chemistry(w, fields, Gamma, heat, dt, **override):
    """-> (new fields tuple (fp64 arrays holding field-dtype values), subcycles[nc])."""
    p = make_params(w, **override)
    nH = _f64(fields[0])
    xHI, xHeI, xHeII, T = [_f64(a).copy() for a in fields[1:]]
    sub = np.zeros(w.ncell, dtype=np.int32)
    lib().orc_chemistry(C.byref(p), _p(nH), _p(xHI), _p(xHeI), _p(xHeII), _p(T), _p(_f64(Gamma)),
                        _p(_f64(heat)), C.c_double(dt), _p(sub))
    return (nH, xHI, xHeI, xHeII, T), sub


def chem_cell(w_or_params, nH, x, T, G, H, dt):
    p = w_or_params if isinstance(w_or_params, Params) else make_params(w_or_params)
    xx = _f64(np.array(x, dtype=np.float64)).copy()
    TT = np.array([T], dtype=np.float64)
    l = lib()
    l.orc_chem_cell.argtypes = [C.c_void_p, C.c_double, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double]
    k = l.orc_chem_cell(C.byref(p), float(nH), _p(xx), _p(TT), _p(_f64(np.array(G, dtype=np.float64))),
                        _p(_f64(np.array(H, dtype=np.float64))), float(dt))
    return xx, float(TT[0]), int(k)


def suggest_dt(w, fields, GammaHI, scheme=1, eps=0.1, **override):
    """Radiative-transfer time step: scheme 1 = neutral-fraction change in cells with tau > 0.5,
    scheme 2 = intensity change.  -> (dt_s, cells that entered the minimum)."""
    p = make_params(w, **override)
    nH, xHI, xHeI, xHeII, T = [_f64(a) for a in fields]
    used = C.c_int64(0)
    l = lib()
    l.orc_suggest_dt.restype = C.c_double
    l.orc_suggest_dt.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double] + [C.c_void_p] * 7
    dt = l.orc_suggest_dt(C.byref(p), int(scheme), float(eps), float(w.sig_HI[0]), _p(nH), _p(xHI), _p(xHeI), _p(xHeII),
                          _p(T), _p(_f64(GammaHI)), C.byref(used))
    return float(dt), int(used.value)


def step(w, fields, dt=None, **override):
    """One full hot-path pass: opacity -> trace -> finalize -> chemistry.  -> dict."""
    kappa = opacity(w, fields, **override)
    A, st, _ = trace(w, kappa=kappa, **override)
    G, H, Ht = finalize(w, A, fields, **override)
    newf, sub = chemistry(w, fields, G, H, w.dt_s if dt is None else dt, **override)
    return dict(A=A, stats=st, Gamma=G, heat=H, heat_total=Ht, fields=newf, subcycles=sub)
