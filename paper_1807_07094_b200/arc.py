"""Thin ctypes binding of include/arc.h (libarc_b200.so).  Argument marshalling only.

Every step of the path runs in the library's CUDA kernels; nothing here computes.  Functions carry the
names of the C entry points.  Array arguments may be

  * numpy arrays            -> passed as ARC_HOST pointers,
  * torch CUDA tensors      -> passed as ARC_DEVICE pointers (torch is used for device memory and
                               streams only; it is imported lazily and is optional for host callers).

If the shared library is missing this module raises: there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

ARC_F32, ARC_F64 = 0, 1
ARC_HOST, ARC_DEVICE = 0, 1
ARC_OK, ARC_EINVAL, ARC_ENOMEM, ARC_ECUDA, ARC_ESTATE, ARC_EOVERFLOW = 0, -1, -2, -3, -4, -5
ARC_END_SPLIT, ARC_END_DEPLETED, ARC_END_ESCAPED = 0, 1, 2
ARC_DEPOSIT_AUTO, ARC_DEPOSIT_RED, ARC_DEPOSIT_AGG, ARC_DEPOSIT_QUAD = 0, 1, 2, 3
ARC_GEOM_NONE, ARC_GEOM_FC, ARC_GEOM_FC_SECONDARY, ARC_GEOM_FC2 = 0, 1, 2, 3
ARC_MAX_BINS, ARC_MAX_LEVEL = 8, 16

_HERE = os.path.dirname(os.path.abspath(__file__))
# ARC_B200_LIB: another build of the same library, e.g. libarc_b200_checked.so (device-side bounds checks)
LIB_PATH = os.environ.get("ARC_B200_LIB") or os.path.join(_HERE, "libarc_b200.so")

EXPORTS = ["arc_create_grid", "arc_destroy", "arc_default_params", "arc_set_params", "arc_set_stream",
           "arc_set_fields", "arc_get_fields", "arc_set_spectrum", "arc_set_sources", "arc_set_emission_mask", "arc_get_thin_radii", "arc_set_thin_radii", "arc_trace",
           "arc_trace_partial", "arc_accum_device", "arc_finalize",
           "arc_get_rates", "arc_get_accum", "arc_update_chemistry", "arc_run_steps", "arc_suggest_dt", "arc_synchronize", "arc_get_stats",
           "arc_trace_debug", "arc_pix2vec", "arc_selftest_division", "arc_pix2vec_noalloc", "arc_pix2vec_noalloc_max",
           "arc_noalloc_last_error", "arc_last_error", "arc_version"]


class ArcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"arc error {code}: {msg}")
        self.code = code


class arc_params(C.Structure):
    _fields_ = [("l0", C.c_int32), ("Lmax", C.c_int32), ("Phi", C.c_double), ("tau_term", C.c_double),
                ("Yp", C.c_double), ("isothermal", C.c_int32), ("caseB", C.c_int32), ("coll_ion", C.c_int32),
                ("max_subcycles", C.c_int32), ("eps_sub", C.c_double), ("x_floor", C.c_double),
                ("digest", C.c_int32), ("async_", C.c_int32), ("trace_blocks", C.c_int32), ("deposit", C.c_int32),
                ("geom_corr", C.c_int32), ("debug_fault", C.c_int32), ("thin_tau", C.c_double)]


class arc_rates(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("Gamma_HI", "Gamma_HeI", "Gamma_HeII", "heat_HI", "heat_HeI",
                                         "heat_HeII", "heat_total")]


class arc_stats(C.Structure):
    _fields_ = [("segments", C.c_uint64), ("rays", C.c_uint64), ("digest", C.c_uint64),
                ("queue_high_water", C.c_uint64), ("splits", C.c_uint64 * ARC_MAX_LEVEL),
                ("rays_level", C.c_uint64 * ARC_MAX_LEVEL), ("ends", C.c_uint64 * 3),
                ("emitted", C.c_double * ARC_MAX_BINS), ("absorbed", C.c_double * ARC_MAX_BINS),
                ("escaped", C.c_double * ARC_MAX_BINS), ("subcycles", C.c_uint64),
                ("max_subcycles_cell", C.c_uint32), ("pad", C.c_uint32), ("trace_ms", C.c_float),
                ("chem_ms", C.c_float), ("trace_kernel_ms", C.c_float), ("opacity_ms", C.c_float),
                ("finalize_ms", C.c_float), ("trace_grid", C.c_int32), ("pad2", C.c_int32),
                ("deposit_records", C.c_uint64), ("kernel_launches", C.c_uint64), ("segments_total", C.c_uint64),
                ("subcycles_total", C.c_uint64), ("steps_ms", C.c_float), ("pad3", C.c_int32)]


class arc_raylog(C.Structure):
    _fields_ = [("cap", C.c_int64), ("n", C.c_int64), ("key", C.c_void_p), ("seq", C.c_void_p), ("cell", C.c_void_p)]


_lib = None


def lib():
    """Load libarc_b200.so (building it is `python -m paper_1807_07094_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_1807_07094_b200.build` "
                              "(the CUDA extension is the product; there is no CPU fallback)")
        l = C.CDLL(LIB_PATH)
        vp, dbl, i32 = C.c_void_p, C.c_double, C.c_int
        l.arc_create_grid.argtypes = [C.POINTER(vp), i32, dbl, i32]
        l.arc_destroy.argtypes = [vp]
        l.arc_default_params.argtypes = [C.POINTER(arc_params)]
        l.arc_default_params.restype = None
        l.arc_set_params.argtypes = [vp, C.POINTER(arc_params)]
        l.arc_set_stream.argtypes = [vp, vp]
        l.arc_set_fields.argtypes = [vp] + [vp] * 5 + [i32]
        l.arc_get_fields.argtypes = [vp] + [vp] * 5 + [i32]
        l.arc_set_spectrum.argtypes = [vp, i32] + [vp] * 4
        l.arc_set_sources.argtypes = [vp, i32] + [vp] * 3
        l.arc_trace.argtypes = [vp, i32, C.POINTER(arc_rates)]
        l.arc_get_rates.argtypes = [vp] + [vp] * 7 + [i32]
        l.arc_trace_partial.argtypes = [vp, i32]
        l.arc_accum_device.argtypes = [vp, C.POINTER(vp), C.POINTER(C.c_int64)]
        l.arc_finalize.argtypes = [vp, C.POINTER(arc_rates)]
        l.arc_get_accum.argtypes = [vp, vp, i32]
        l.arc_update_chemistry.argtypes = [vp, dbl]
        l.arc_run_steps.argtypes = [vp, i32, dbl]
        l.arc_suggest_dt.argtypes = [vp, i32, dbl, vp, vp]
        l.arc_set_emission_mask.argtypes = [vp, vp, i32]
        l.arc_get_thin_radii.argtypes = [vp, vp]
        l.arc_set_thin_radii.argtypes = [vp, vp]
        l.arc_synchronize.argtypes = [vp]
        l.arc_get_stats.argtypes = [vp, C.POINTER(arc_stats)]
        l.arc_trace_debug.argtypes = [vp, i32, C.POINTER(arc_raylog)]
        l.arc_pix2vec.argtypes = [vp, vp, i32, vp]
        l.arc_selftest_division.argtypes = [C.c_uint64, C.c_uint64, C.POINTER(C.c_uint64)]
        l.arc_pix2vec_noalloc.argtypes = [vp, vp, i32, vp]
        l.arc_pix2vec_noalloc_max.restype = i32
        l.arc_noalloc_last_error.restype = C.c_char_p
        l.arc_last_error.argtypes = [vp]
        l.arc_last_error.restype = C.c_char_p
        l.arc_version.restype = C.c_char_p
        _lib = l
    return _lib


# ---- marshalling ----------------------------------------------------------------------------------
def _is_torch(a):
    return type(a).__module__.startswith("torch")


def _ptr(a):
    """-> (pointer, where) for a numpy array or a torch tensor; None -> (None, None)."""
    if a is None:
        return None, None
    if _is_torch(a):
        if not a.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return C.c_void_p(a.data_ptr()), (ARC_DEVICE if a.is_cuda else ARC_HOST)
    if not isinstance(a, np.ndarray) or not a.flags["C_CONTIGUOUS"]:
        raise ValueError("array must be a C-contiguous numpy array or a torch tensor")
    return C.c_void_p(a.ctypes.data), ARC_HOST


def _same_where(arrs):
    ws = {w for _, w in arrs if w is not None}
    if len(ws) > 1:
        raise ValueError("all arrays of one call must live in the same place (host or device)")
    return ws.pop() if ws else ARC_HOST


def _check(ctx, rc):
    if rc != ARC_OK:
        raise ArcError(rc, (lib().arc_last_error(ctx) or b"").decode())
    return rc


def _host_f64(a):
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


# ---- the entry points (same names as the C ABI) ---------------------------------------------------
def arc_version() -> str:
    return lib().arc_version().decode()


def arc_last_error(ctx=None) -> str:
    """Text of the last failure of `ctx` (None: of the last failed arc_create_grid on this thread)."""
    return (lib().arc_last_error(ctx) or b"").decode()


def arc_create_grid(N: int, box_cm: float, dtype: int):
    ctx = C.c_void_p()
    rc = lib().arc_create_grid(C.byref(ctx), int(N), float(box_cm), int(dtype))
    if rc != ARC_OK:
        raise ArcError(rc, (lib().arc_last_error(None) or b"").decode())
    return ctx


def arc_destroy(ctx):
    return lib().arc_destroy(ctx)


def arc_default_params() -> arc_params:
    p = arc_params()
    lib().arc_default_params(C.byref(p))
    return p


def arc_set_params(ctx, p: arc_params):
    return _check(ctx, lib().arc_set_params(ctx, C.byref(p)))


def arc_set_stream(ctx, cuda_stream: int):
    return _check(ctx, lib().arc_set_stream(ctx, C.c_void_p(int(cuda_stream) or None)))


def arc_set_fields(ctx, n_H, x_HI, x_HeI, x_HeII, T):
    ps = [_ptr(a) for a in (n_H, x_HI, x_HeI, x_HeII, T)]
    return _check(ctx, lib().arc_set_fields(ctx, *[p for p, _ in ps], _same_where(ps)))


def arc_get_fields(ctx, n_H=None, x_HI=None, x_HeI=None, x_HeII=None, T=None):
    ps = [_ptr(a) for a in (n_H, x_HI, x_HeI, x_HeII, T)]
    return _check(ctx, lib().arc_get_fields(ctx, *[p for p, _ in ps], _same_where(ps)))


def arc_set_spectrum(ctx, E_eV, sig_HI, sig_HeI, sig_HeII):
    a = [_host_f64(x) for x in (E_eV, sig_HI, sig_HeI, sig_HeII)]
    return _check(ctx, lib().arc_set_spectrum(ctx, len(a[0]), *[C.c_void_p(x.ctypes.data) for x in a]))


def arc_set_sources(ctx, pos_cm, Ndot, binfrac):
    pos, nd, bf = _host_f64(pos_cm), _host_f64(Ndot), _host_f64(binfrac)
    return _check(ctx, lib().arc_set_sources(ctx, len(nd), C.c_void_p(pos.ctypes.data), C.c_void_p(nd.ctypes.data),
                                             C.c_void_p(bf.ctypes.data)))


def arc_trace(ctx, step: int = 0) -> arc_rates:
    """-> arc_rates: library-owned DEVICE pointers, valid until the next arc_trace / arc_destroy."""
    out = arc_rates()
    _check(ctx, lib().arc_trace(ctx, int(step), C.byref(out)))
    return out


def arc_trace_partial(ctx, step: int = 0):
    """rows a1-a9 for this context's sources only (source-sharded tracing); rates after arc_finalize"""
    return _check(ctx, lib().arc_trace_partial(ctx, int(step)))


def arc_accum_device(ctx):
    """-> (device pointer, number of doubles) of the library-owned accumulators"""
    p = C.c_void_p()
    n = C.c_int64()
    _check(ctx, lib().arc_accum_device(ctx, C.byref(p), C.byref(n)))
    return int(p.value or 0), int(n.value)


def arc_finalize(ctx) -> arc_rates:
    """row a10 from whatever the accumulators hold (after the caller's sum over shards)"""
    out = arc_rates()
    _check(ctx, lib().arc_finalize(ctx, C.byref(out)))
    return out


def arc_get_rates(ctx, Gamma_HI=None, Gamma_HeI=None, Gamma_HeII=None, heat_HI=None, heat_HeI=None,
                  heat_HeII=None, heat_total=None):
    ps = [_ptr(a) for a in (Gamma_HI, Gamma_HeI, Gamma_HeII, heat_HI, heat_HeI, heat_HeII, heat_total)]
    return _check(ctx, lib().arc_get_rates(ctx, *[p for p, _ in ps], _same_where(ps)))


def arc_get_accum(ctx, A):
    p, w = _ptr(A)
    return _check(ctx, lib().arc_get_accum(ctx, p, w))


def arc_update_chemistry(ctx, dt_s: float):
    return _check(ctx, lib().arc_update_chemistry(ctx, float(dt_s)))


def arc_run_steps(ctx, n_steps: int, dt_s: float):
    """n_steps x (arc_trace + arc_update_chemistry(dt_s)) without a host round trip per step (one CUDA graph, replayed)"""
    return _check(ctx, lib().arc_run_steps(ctx, int(n_steps), float(dt_s)))


ARC_DT_NEUTRAL, ARC_DT_INTENSITY = 1, 2


def arc_get_thin_radii(ctx, nsrc: int) -> np.ndarray:
    """radii [cells] the next arc_trace will use (optically thin inner region)."""
    R = np.zeros(int(nsrc))
    _check(ctx, lib().arc_get_thin_radii(ctx, R.ctypes.data_as(C.c_void_p)))
    return R


def arc_set_thin_radii(ctx, R):
    R = np.ascontiguousarray(R, dtype=np.float64)
    return _check(ctx, lib().arc_set_thin_radii(ctx, R.ctypes.data_as(C.c_void_p)))


def arc_set_emission_mask(ctx, blocked, level: int):
    """blocked: None (clear) or uint8 [nsrc, 12 4^level], non-zero = root ray blocked."""
    if blocked is None:
        return _check(ctx, lib().arc_set_emission_mask(ctx, None, int(level)))
    b = np.ascontiguousarray(blocked, dtype=np.uint8)
    return _check(ctx, lib().arc_set_emission_mask(ctx, b.ctypes.data_as(C.c_void_p), int(level)))


def arc_suggest_dt(ctx, scheme: int = ARC_DT_NEUTRAL, eps: float = 0.1):
    """-> (dt_s, cells that entered the minimum)."""
    dt = C.c_double(0.0)
    used = C.c_int64(0)
    _check(ctx, lib().arc_suggest_dt(ctx, int(scheme), float(eps), C.byref(dt), C.byref(used)))
    return float(dt.value), int(used.value)


def arc_synchronize(ctx):
    return _check(ctx, lib().arc_synchronize(ctx))


def arc_get_stats(ctx) -> arc_stats:
    s = arc_stats()
    _check(ctx, lib().arc_get_stats(ctx, C.byref(s)))
    return s


def arc_trace_debug(ctx, cap: int, step: int = 0):
    """-> (key[u64], seq[u32], cell[i32]) host arrays with one entry per segment plus one closing entry
    per ray (cell = -1 - end reason), in arbitrary order."""
    key = np.zeros(cap, np.uint64); seq = np.zeros(cap, np.uint32); cell = np.zeros(cap, np.int32)
    log = arc_raylog(cap=cap, n=0, key=key.ctypes.data, seq=seq.ctypes.data, cell=cell.ctypes.data)
    _check(ctx, lib().arc_trace_debug(ctx, int(step), C.byref(log)))
    n = int(log.n)
    return key[:n], seq[:n], cell[:n]


def arc_pix2vec(level, pix) -> np.ndarray:
    lv = np.ascontiguousarray(np.asarray(level, dtype=np.int32))
    px = np.ascontiguousarray(np.asarray(pix, dtype=np.uint32))
    out = np.zeros((len(lv), 3))
    rc = lib().arc_pix2vec(C.c_void_p(lv.ctypes.data), C.c_void_p(px.ctypes.data), len(lv), C.c_void_p(out.ctypes.data))
    if rc != ARC_OK:
        raise ArcError(rc, "arc_pix2vec failed")
    return out


def arc_pix2vec_noalloc_max() -> int:
    return int(lib().arc_pix2vec_noalloc_max())


def arc_noalloc_last_error() -> str:
    return (lib().arc_noalloc_last_error() or b"").decode()


def arc_pix2vec_noalloc(level, pix, out=None) -> np.ndarray:
    """arc_pix2vec without any device allocation (fixed 128 KiB device scratch; at most arc_pix2vec_noalloc_max() pairs
    per call).  `out` (float64 [n, 3], C order) may be passed in so that the host side allocates nothing either."""
    lv = np.ascontiguousarray(np.asarray(level, dtype=np.int32))
    px = np.ascontiguousarray(np.asarray(pix, dtype=np.uint32))
    if out is None:
        out = np.zeros((len(lv), 3))
    if out.dtype != np.float64 or not out.flags["C_CONTIGUOUS"] or out.size < 3 * len(lv):
        raise ValueError("out must be a C-contiguous float64 array of at least 3 n values")
    rc = lib().arc_pix2vec_noalloc(C.c_void_p(lv.ctypes.data), C.c_void_p(px.ctypes.data), len(lv), C.c_void_p(out.ctypes.data))
    if rc != ARC_OK:
        raise ArcError(rc, arc_noalloc_last_error())
    return out


def arc_selftest_division(n_pairs: int, seed: int = 1) -> int:
    """-> number of (a, d) pairs for which the tracer's division differs from IEEE division (must be 0)"""
    bad = C.c_uint64(0)
    rc = lib().arc_selftest_division(int(n_pairs), int(seed), C.byref(bad))
    if rc != ARC_OK:
        raise ArcError(rc, "arc_selftest_division failed")
    return int(bad.value)


# ---- helpers that only move data (no arithmetic) ---------------------------------------------------
def stats_dict(s: arc_stats, nb: int) -> dict:
    return dict(segments=int(s.segments), rays=int(s.rays), digest=int(s.digest),
                queue_high_water=int(s.queue_high_water),
                splits=np.array(s.splits[:], dtype=np.uint64), rays_level=np.array(s.rays_level[:], dtype=np.uint64),
                ends=np.array(s.ends[:], dtype=np.uint64), emitted=np.array(s.emitted[:nb]),
                absorbed=np.array(s.absorbed[:nb]), escaped=np.array(s.escaped[:nb]),
                subcycles=int(s.subcycles), max_subcycles_cell=int(s.max_subcycles_cell),
                trace_ms=float(s.trace_ms), chem_ms=float(s.chem_ms), trace_kernel_ms=float(s.trace_kernel_ms),
                opacity_ms=float(s.opacity_ms), finalize_ms=float(s.finalize_ms), trace_grid=int(s.trace_grid),
                deposit_records=int(s.deposit_records), kernel_launches=int(s.kernel_launches),
                segments_total=int(s.segments_total), subcycles_total=int(s.subcycles_total), steps_ms=float(s.steps_ms))


def params_from_dict(d: dict, **override) -> arc_params:
    p = arc_default_params()
    dd = dict(d)
    dd.update(override)
    for k, v in dd.items():
        if k.startswith("_"):
            continue
        name = "async_" if k == "async" else k
        if not hasattr(p, name):
            raise KeyError(f"unknown arc_params field {k}")
        setattr(p, name, type(getattr(p, name))(v))
    return p


class Context:
    """Owns one arc_ctx; convenience around the flat calls for a workloads.Workload."""

    def __init__(self, w, fields=None, where="host", stream=None, **param_override):
        self.w = w
        self.nb = w.nb
        self.np_dtype = np.float32 if w.dtype == "f32" else np.float64
        self.ctx = arc_create_grid(w.N, w.box_cm, ARC_F32 if w.dtype == "f32" else ARC_F64)
        self.stream = stream                        # cudaStream_t handle the library enqueues on (None: legacy default stream)
        try:
            arc_set_params(self.ctx, params_from_dict(w.params, **param_override))
            if stream is not None:
                arc_set_stream(self.ctx, stream)
            arc_set_spectrum(self.ctx, w.E_eV, w.sig_HI, w.sig_HeI, w.sig_HeII)
            arc_set_sources(self.ctx, w.src_pos_cm, w.src_Ndot, w.src_binfrac)
            self._nsrc = w.nsrc
            self.set_fields(fields if fields is not None else w.fields())
        except Exception:
            self.close()
            raise

    def set_fields(self, fields):
        arrs = []
        for a in fields:
            if _is_torch(a):
                arrs.append(a)
            else:
                arrs.append(np.ascontiguousarray(np.asarray(a, dtype=self.np_dtype)))
        arc_set_fields(self.ctx, *arrs)

    def set_sources(self, idx):
        w = self.w
        self._nsrc = len(idx)
        arc_set_sources(self.ctx, w.src_pos_cm[idx], w.src_Ndot[idx], w.src_binfrac[idx])

    def get_fields(self):
        out = [np.zeros(self.w.ncell, self.np_dtype) for _ in range(5)]
        arc_get_fields(self.ctx, *out)
        return tuple(out)

    def trace(self, step=0):
        return arc_trace(self.ctx, step)

    def trace_partial(self, step=0):
        return arc_trace_partial(self.ctx, step)

    def finalize(self):
        return arc_finalize(self.ctx)

    def accum_tensor(self):
        """the library's accumulators as a torch CUDA tensor that ALIASES them (no copy), for an in-place reduction"""
        import torch
        ptr, n = arc_accum_device(self.ctx)

        class _Alias:                               # __cuda_array_interface__ v2: 1-d float64, C order
            __cuda_array_interface__ = {"shape": (n,), "typestr": "<f8", "data": (ptr, False), "version": 2, "strides": None}

        return torch.as_tensor(_Alias(), device="cuda")

    def rates(self):
        """-> Gamma[3, nc], heat[3, nc], heat_total[nc] as host arrays."""
        nc = self.w.ncell
        G = np.zeros((3, nc)); H = np.zeros((3, nc)); Ht = np.zeros(nc)
        arc_get_rates(self.ctx, G[0], G[1], G[2], H[0], H[1], H[2], Ht)
        return G, H, Ht

    def accum(self):
        A = np.zeros((self.w.ncell, self.nb))
        arc_get_accum(self.ctx, A)
        return A

    def thin_radii(self):
        """radii [cells] the next trace will use (optically thin inner region)"""
        return arc_get_thin_radii(self.ctx, self._nsrc)

    def set_thin_radii(self, R):
        R = np.ascontiguousarray(R, dtype=np.float64)
        assert R.shape == (self._nsrc,)
        return arc_set_thin_radii(self.ctx, R)

    def set_emission_mask(self, blocked, level=None):
        return arc_set_emission_mask(self.ctx, blocked, int(self.w.params["l0"]) if level is None else int(level))

    def suggest_dt(self, scheme=ARC_DT_NEUTRAL, eps=0.1):
        return arc_suggest_dt(self.ctx, scheme, eps)

    def update_chemistry(self, dt=None):
        return arc_update_chemistry(self.ctx, self.w.dt_s if dt is None else dt)

    def run_steps(self, n_steps, dt=None):
        return arc_run_steps(self.ctx, n_steps, self.w.dt_s if dt is None else dt)

    def stats(self):
        return stats_dict(arc_get_stats(self.ctx), self.nb)

    def trace_debug(self, cap=1 << 22):
        return arc_trace_debug(self.ctx, cap)

    def close(self):
        if self.ctx is not None:
            arc_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
