"""ctypes binding of oracle/p2p_oracle.c (ORACLE — test infrastructure, not the product).

Argument marshalling only; every number comes out of the C file.  The shared object is built
with gcc into ``oracle/build/`` (git-ignored) on first use or by ``__graft_entry__.build()``.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "p2p_oracle.c")
_OUT_DIR = os.path.join(_HERE, "build")
_OUT = os.path.join(_OUT_DIR, "libp2p_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile p2p_oracle.c -> oracle/build/libp2p_oracle.so (gcc -O2 -fopenmp)."""
    if not force and os.path.exists(_OUT) and os.path.getmtime(_OUT) >= os.path.getmtime(_SRC):
        return _OUT
    os.makedirs(_OUT_DIR, exist_ok=True)
    tmp = _OUT + f".tmp{os.getpid()}"
    # -O2 without -ffast-math: libm erfc/exp/sqrt/nearbyint keep their IEEE meaning
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, _OUT)
    return _OUT


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        lib.oracle_T.restype = ctypes.c_double
        lib.oracle_T.argtypes = [ctypes.c_double]
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_p2p.restype = None
        lib.oracle_p2p.argtypes = [
            ctypes.c_longlong, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_longlong, ctypes.c_void_p,
            ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_double,
            ctypes.c_void_p, ctypes.c_void_p]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def oracle_T(x):
    """Eq. 1 in x = r/2r_s, evaluated by the C oracle (scalar or array)."""
    lib = _load()
    xs = np.atleast_1d(np.asarray(x, dtype=np.float64))
    out = np.array([lib.oracle_T(float(v)) for v in xs.ravel()]).reshape(xs.shape)
    return out if np.ndim(x) else float(out[0])


def _call(pos, mass, tgt, boxsize, r_s, r_cut, G, eps=0.0):
    lib = _load()
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    n = pos.shape[0]
    assert pos.shape == (n, 3)
    mass = np.ascontiguousarray(mass, dtype=np.float64)
    assert mass.shape == (n,)
    if tgt is None:
        nt, tptr = n, None
    else:
        tgt = np.ascontiguousarray(tgt, dtype=np.int64)
        nt, tptr = tgt.shape[0], tgt.ctypes.data
    acc = np.zeros((nt, 3), dtype=np.float64)
    counts = np.zeros(2, dtype=np.int64)
    if nt:
        lib.oracle_p2p(n, pos.ctypes.data, mass.ctypes.data, nt, tptr,
                       float(boxsize), float(r_s), float(r_cut), float(G), float(eps),
                       acc.ctypes.data, counts.ctypes.data)
    return acc, {"pair_tests": int(counts[0]), "pairs_in_cut": int(counts[1])}


def p2p(pos, mass, *, boxsize, r_s, r_cut, G=1.0, eps=0.0):
    """Full O(N^2) sum: acc[n,3] and counters.  boxsize <= 0 means isolated boundaries (no images);
    eps > 0 = Plummer softening length (A23)."""
    return _call(pos, mass, None, boxsize, r_s, r_cut, G, eps)


def p2p_sampled(pos, mass, targets, *, boxsize, r_s, r_cut, G=1.0, eps=0.0):
    """Accelerations of the listed targets against all N sources."""
    return _call(pos, mass, targets, boxsize, r_s, r_cut, G, eps)
