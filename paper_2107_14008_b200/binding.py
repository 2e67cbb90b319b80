"""ctypes binding of libphotons.so — argument marshalling only; every step of the path runs in the CUDA
library (include/photons.h).  PyTorch appears here only as the owner of device memory and streams: tensors
are passed by ``data_ptr()`` and ``torch.cuda.current_stream().cuda_stream``.

There is no fallback: if the shared library is missing, or there is no CUDA device, calls raise.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libphotons.so")

OK, EINVAL, ESTATE, ENOMEM, ECUDA, ENODEVICE, EBOX, ENONFINITE = range(8)
FP64, FP32, MIXED = 0, 1, 2
G_DIRECT, G_TABLE, G_POLY, G_FUSED = 0, 1, 2, 3
TABLE_PAPER, TABLE_COEF = 0, 1
MEM_HOST, MEM_DEVICE = 0, 1
DTYPE_F64, DTYPE_F32 = 0, 1

PRECISIONS = {"fp64": FP64, "fp32": FP32, "mixed": MIXED}
G_MODES = {"direct": G_DIRECT, "table": G_TABLE, "poly": G_POLY, "fused": G_FUSED}
TABLE_QUAD = 2
TABLE_LAYOUTS = {"paper": TABLE_PAPER, "coef": TABLE_COEF, "quad": TABLE_QUAD}
ERROR_NAMES = ["OK", "EINVAL", "ESTATE", "ENOMEM", "ECUDA", "ENODEVICE", "EBOX", "ENONFINITE"]

EXPORTS = [
    "photons_default_params", "photons_create", "photons_set_stream", "photons_set_particles", "photons_build_leaves",
    "photons_short_range_acc", "photons_get_leaf_order", "photons_get_interaction_list", "photons_get_stats",
    "photons_peak_probe", "photons_poly_fit", "photons_fused_fit", "photons_m2l", "photons_m2l_noalloc", "photons_last_error", "photons_destroy",
]


class Params(ctypes.Structure):
    _fields_ = [
        ("boxsize", ctypes.c_double), ("n_pm", ctypes.c_int), ("rs_over_cell", ctypes.c_double),
        ("rcut_over_rs", ctypes.c_double), ("G", ctypes.c_double), ("maxleaf", ctypes.c_int),
        ("precision", ctypes.c_int), ("g_mode", ctypes.c_int), ("table_nodes", ctypes.c_int),
        ("table_level", ctypes.c_int), ("n_streams", ctypes.c_int), ("device", ctypes.c_int),
        ("close_pair_radius", ctypes.c_double), ("chunk_max", ctypes.c_int), ("warps_per_leaf", ctypes.c_int),
        ("targets_per_lane", ctypes.c_int), ("poly_degree", ctypes.c_int), ("periodic", ctypes.c_int),
        ("softening", ctypes.c_double), ("table_layout", ctypes.c_int), ("leaf_order", ctypes.c_int), ("orb_method", ctypes.c_int),
        ("mass_path", ctypes.c_int),
    ]


class Stats(ctypes.Structure):
    _fields_ = [
        ("n_particles", ctypes.c_longlong), ("n_leaves", ctypes.c_longlong), ("n_chunks", ctypes.c_longlong),
        ("n_leaf_pairs", ctypes.c_longlong), ("pairs_evaluated", ctypes.c_longlong),
        ("max_leaves_per_target", ctypes.c_longlong), ("build_ms", ctypes.c_double),
        ("kernel_ms", ctypes.c_double), ("total_ms", ctypes.c_double), ("kernel_launches", ctypes.c_longlong),
    ]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class PhotonsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"photons: {ERROR_NAMES[code] if 0 <= code < len(ERROR_NAMES) else code}: {msg}")
        self.code = code


_lib = None


def load():
    """Load libphotons.so (built by ``python -m paper_2107_14008_b200.build``); raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2107_14008_b200.build` "
                          "(there is no CPU fallback for the CUDA path)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, ll, ci = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int
    lib.photons_default_params.restype = None
    lib.photons_default_params.argtypes = [ctypes.POINTER(Params)]
    lib.photons_create.restype = ci
    lib.photons_create.argtypes = [ctypes.POINTER(Params), ctypes.POINTER(vp), ctypes.c_char_p, ci]
    lib.photons_set_stream.restype = ci
    lib.photons_set_stream.argtypes = [vp, vp]
    lib.photons_set_particles.restype = ci
    lib.photons_set_particles.argtypes = [vp, ll, vp, vp, ci, ci, vp]
    lib.photons_build_leaves.restype = ci
    lib.photons_build_leaves.argtypes = [vp]
    lib.photons_short_range_acc.restype = ci
    lib.photons_short_range_acc.argtypes = [vp, vp, ci, ci, ctypes.POINTER(Stats)]
    lib.photons_get_leaf_order.restype = ci
    lib.photons_get_leaf_order.argtypes = [vp, vp, vp]
    lib.photons_get_interaction_list.restype = ci
    lib.photons_get_interaction_list.argtypes = [vp, vp, vp, vp, vp]
    lib.photons_get_stats.restype = ci
    lib.photons_get_stats.argtypes = [vp, ctypes.POINTER(Stats)]
    lib.photons_peak_probe.restype = ci
    lib.photons_peak_probe.argtypes = [ci, ci, ctypes.POINTER(ctypes.c_double)]
    lib.photons_poly_fit.restype = ci
    lib.photons_poly_fit.argtypes = [ci, ctypes.c_double, vp, ctypes.POINTER(ctypes.c_double)]
    lib.photons_fused_fit.restype = ci
    lib.photons_fused_fit.argtypes = [ci, ctypes.c_double, vp, ctypes.POINTER(ctypes.c_double)]
    lib.photons_m2l.restype = ci
    lib.photons_m2l.argtypes = [ci, ci, ctypes.c_double, ctypes.c_double, ll, vp, vp, vp, vp, vp, vp, ci, vp,
                                ctypes.POINTER(ctypes.c_double)]
    lib.photons_m2l_noalloc.restype = ci
    lib.photons_m2l_noalloc.argtypes = [ci, ci, ctypes.c_double, ctypes.c_double, ll, vp, vp, vp, vp, vp, vp, vp, ctypes.c_char_p, ci]
    lib.photons_last_error.restype = ctypes.c_char_p
    lib.photons_last_error.argtypes = [vp]
    lib.photons_destroy.restype = None
    lib.photons_destroy.argtypes = [vp]
    _lib = lib
    return lib


def default_params(**overrides) -> Params:
    p = Params()
    load().photons_default_params(ctypes.byref(p))
    for k, v in overrides.items():
        if k == "precision" and isinstance(v, str):
            v = PRECISIONS[v]
        if k == "g_mode" and isinstance(v, str):
            v = G_MODES[v]
        if k == "table_layout" and isinstance(v, str):
            v = TABLE_LAYOUTS[v]
        if not hasattr(p, k):
            raise TypeError(f"unknown parameter {k!r}")
        setattr(p, k, v)
    return p


def _is_tensor(x):
    return type(x).__module__.startswith("torch")


def _marshal(x, name):
    """(pointer, dtype code, mem kind, keep-alive object) of a numpy array or a torch tensor."""
    if _is_tensor(x):
        import torch
        if x.dtype == torch.float64:
            dt = DTYPE_F64
        elif x.dtype == torch.float32:
            dt = DTYPE_F32
        else:
            raise TypeError(f"{name}: float32 or float64 expected")
        if not x.is_contiguous():
            raise ValueError(f"{name}: tensor must be contiguous")
        return x.data_ptr(), dt, (MEM_DEVICE if x.is_cuda else MEM_HOST), x
    a = np.asarray(x)
    if a.dtype == np.float64:
        dt = DTYPE_F64
    elif a.dtype == np.float32:
        dt = DTYPE_F32
    else:
        raise TypeError(f"{name}: float32 or float64 expected")
    if not a.flags.c_contiguous:
        raise ValueError(f"{name}: array must be C-contiguous")
    return a.ctypes.data, dt, MEM_HOST, a


class Photons:
    """Thin object wrapper over the C ABI: same calls, same names."""

    def __init__(self, **params):
        self._lib = load()
        self._ctx = ctypes.c_void_p()
        self.params = default_params(**params)
        buf = ctypes.create_string_buffer(512)
        rc = self._lib.photons_create(ctypes.byref(self.params), ctypes.byref(self._ctx), buf, len(buf))
        if rc != OK:
            self._ctx = ctypes.c_void_p()
            raise PhotonsError(rc, buf.value.decode(errors="replace"))
        self.n = 0

    def set_stream(self, stream):
        """Make a CUDA stream (torch.cuda.Stream, raw handle or None) the context's main stream."""
        handle = getattr(stream, "cuda_stream", stream)
        self._check(self._lib.photons_set_stream(self._ctx, ctypes.c_void_p(handle or 0)))

    def _check(self, rc):
        if rc != OK:
            raise PhotonsError(rc, (self._lib.photons_last_error(self._ctx) or b"").decode(errors="replace"))

    def set_particles(self, pos, mass=None, stream=None):
        ptr, dt, kind, _keep = _marshal(pos, "pos")
        n = int(pos.shape[0])
        if tuple(pos.shape) != (n, 3):
            raise ValueError("pos must be n x 3")
        mptr = None
        if mass is not None:
            mptr, mdt, mkind, _keepm = _marshal(mass, "mass")
            if mdt != dt or mkind != kind or tuple(mass.shape) != (n,):
                raise ValueError("mass must match pos in dtype, memory kind and length")
        if stream is None and kind == MEM_DEVICE:
            import torch
            stream = torch.cuda.current_stream().cuda_stream
        self._check(self._lib.photons_set_particles(self._ctx, n, ptr, mptr, dt, kind, ctypes.c_void_p(stream or 0)))
        self.n = n

    def build_leaves(self):
        self._check(self._lib.photons_build_leaves(self._ctx))

    def short_range_acc(self, out):
        """Fill ``out`` (n x 3 numpy array or torch tensor, fp32/fp64, host or device) and return the stats."""
        ptr, dt, kind, _keep = _marshal(out, "acc")
        if tuple(out.shape) != (self.n, 3):
            raise ValueError("acc must be n x 3")
        if kind == MEM_DEVICE:
            import torch
            torch.cuda.current_stream().synchronize()   # unless set_stream was used the library has its own streams
        st = Stats()
        self._check(self._lib.photons_short_range_acc(self._ctx, ptr, dt, kind, ctypes.byref(st)))
        return st.as_dict()

    def stats(self):
        st = Stats()
        self._check(self._lib.photons_get_stats(self._ctx, ctypes.byref(st)))
        return st.as_dict()

    def leaf_order(self):
        st = self.stats()
        perm = np.empty(st["n_particles"], dtype=np.int64)
        leaf_start = np.empty(st["n_leaves"] + 1, dtype=np.int64)
        self._check(self._lib.photons_get_leaf_order(self._ctx, perm.ctypes.data, leaf_start.ctypes.data))
        return perm, leaf_start

    def interaction_list(self):
        st = self.stats()
        ptr = np.empty(st["n_leaves"] + 1, dtype=np.int64)
        first = np.empty(st["n_chunks"], dtype=np.int32)
        nleaf = np.empty(st["n_chunks"], dtype=np.int32)
        code = np.empty(st["n_chunks"], dtype=np.int32)
        self._check(self._lib.photons_get_interaction_list(self._ctx, ptr.ctypes.data, first.ctypes.data,
                                                           nleaf.ctypes.data, code.ctypes.data))
        return ptr, first, nleaf, code

    def close(self):
        if self._ctx:
            self._lib.photons_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def peak_probe(kind: int, device: int = 0) -> float:
    out = ctypes.c_double()
    rc = load().photons_peak_probe(device, kind, ctypes.byref(out))
    if rc != OK:
        raise PhotonsError(rc, "peak_probe failed")
    return out.value


def poly_fit(degree: int, rcut_over_rs: float = 6.0):
    """(coeffs[degree+1] lowest power first, max |g_poly - g|) of the PHOTONS_G_POLY polynomial; host only."""
    coeffs = np.empty(degree + 1, dtype=np.float64)
    err = ctypes.c_double()
    rc = load().photons_poly_fit(degree, float(rcut_over_rs), coeffs.ctypes.data, ctypes.byref(err))
    if rc != OK:
        raise PhotonsError(rc, "poly_fit: bad argument")
    return coeffs, err.value


def fused_fit(degree: int, rcut_over_rs: float = 6.0):
    """(coeffs[degree+1] lowest power first, max |g_fused - g|) of the PHOTONS_G_FUSED polynomial; host only."""
    coeffs = np.empty(degree + 1, dtype=np.float64)
    err = ctypes.c_double()
    rc = load().photons_fused_fit(degree, float(rcut_over_rs), coeffs.ctypes.data, ctypes.byref(err))
    if rc != OK:
        raise PhotonsError(rc, "fused_fit: bad argument")
    return coeffs, err.value


def m2l_n_coeffs(p: int) -> int:
    return (p + 1) * (p + 2) * (p + 3) // 6


def m2l(centres, multipoles, pair_ptr, pair_src, pair_shift=None, *, p, r_s, boxsize=0.0, out=None, device=0, stream=None):
    """photons_m2l: numpy arrays (host) or torch CUDA tensors (device), all of one kind.  Returns (locals, kernel_ms)."""
    def ptr(x, dtype_np, dtype_name):
        if x is None:
            return None, MEM_HOST, None
        if _is_tensor(x):
            if str(x.dtype) != "torch." + dtype_name or not x.is_contiguous():
                raise TypeError(f"contiguous {dtype_name} tensor expected")
            return x.data_ptr(), (MEM_DEVICE if x.is_cuda else MEM_HOST), x
        a = np.ascontiguousarray(x, dtype=dtype_np)
        return a.ctypes.data, MEM_HOST, a
    n_cells = int(centres.shape[0])
    nc = m2l_n_coeffs(p)
    if tuple(multipoles.shape) != (n_cells, nc):
        raise ValueError("multipoles must be n_cells x NC(p)")
    c_ptr, kind, k0 = ptr(centres, np.float64, "float64")
    m_ptr, kind_m, k1 = ptr(multipoles, np.float64, "float64")
    pp_ptr, kind_p, k2 = ptr(pair_ptr, np.int64, "int64")
    ps_ptr, kind_s, k3 = ptr(pair_src, np.int32, "int32")
    sh_ptr, _, k4 = ptr(pair_shift, np.int8, "int8")
    if len({kind, kind_m, kind_p, kind_s}) != 1:
        raise ValueError("all arrays must be of one memory kind")
    if out is None:
        if kind == MEM_DEVICE:
            import torch
            out = torch.empty((n_cells, nc), dtype=torch.float64, device=centres.device)
        else:
            out = np.empty((n_cells, nc), dtype=np.float64)
    o_ptr, kind_o, k5 = ptr(out, np.float64, "float64")
    if kind_o != kind:
        raise ValueError("out must be of the inputs' memory kind")
    ms = ctypes.c_double()
    handle = getattr(stream, "cuda_stream", stream)
    rc = load().photons_m2l(device, int(p), float(r_s), float(boxsize), n_cells, c_ptr, m_ptr, pp_ptr, ps_ptr, sh_ptr, o_ptr,
                            kind, ctypes.c_void_p(handle or 0), ctypes.byref(ms))
    if rc != OK:
        raise PhotonsError(rc, "photons_m2l failed")
    return out, ms.value


M2L_NOALLOC_SCRATCH_BYTES = 8 << 20      # PHOTONS_M2L_NOALLOC_SCRATCH_BYTES


def m2l_noalloc(centres, multipoles, pair_ptr, pair_src, pair_shift=None, *, out, p, r_s, boxsize=0.0, stream=None):
    """photons_m2l_noalloc: torch CUDA tensors only, `out` (n_cells x NC float64) supplied by the caller; enqueues on
    `stream` (default: torch's current stream) and returns without synchronising."""
    import torch

    def ptr(x, dtype, name):
        if x is None:
            return None
        if not (_is_tensor(x) and x.is_cuda and x.dtype == dtype and x.is_contiguous()):
            raise TypeError(f"{name}: contiguous CUDA tensor of {dtype} expected")
        return x.data_ptr()
    n_cells = int(centres.shape[0])
    if tuple(multipoles.shape) != (n_cells, m2l_n_coeffs(p)) or tuple(out.shape) != tuple(multipoles.shape):
        raise ValueError("multipoles and out must be n_cells x NC(p)")
    if stream is None:
        stream = torch.cuda.current_stream(centres.device)
    handle = getattr(stream, "cuda_stream", stream)
    err = ctypes.create_string_buffer(512)
    rc = load().photons_m2l_noalloc(centres.device.index or 0, int(p), float(r_s), float(boxsize), n_cells,
                                    ptr(centres, torch.float64, "centres"), ptr(multipoles, torch.float64, "multipoles"),
                                    ptr(pair_ptr, torch.int64, "pair_ptr"), ptr(pair_src, torch.int32, "pair_src"),
                                    ptr(pair_shift, torch.int8, "pair_shift"), ptr(out, torch.float64, "out"),
                                    ctypes.c_void_p(handle or 0), err, len(err))
    if rc != OK:
        raise PhotonsError(rc, err.value.decode(errors="replace"))
    return out


def short_range_acc(pos, mass=None, *, out=None, **params):
    """One-shot convenience: create -> set_particles -> build_leaves -> short_range_acc -> destroy."""
    with Photons(**params) as ph:
        ph.set_particles(pos, mass)
        ph.build_leaves()
        if out is None:
            out = np.empty((pos.shape[0], 3), dtype=np.float64)
        st = ph.short_range_acc(out)
    return out, st
