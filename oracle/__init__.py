"""Python loader for the CPU oracle (oracle/coarse_oracle.cpp).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  The product package
(paper_2212_12559_b200) never imports this module, and this module never imports it.

`build()` compiles the C++ source with g++ (-O3 -fopenmp, no fast-math, no FMA
contraction, baseline x86-64 so the .so also runs on the GPU box's host CPU).
The wrappers take numpy arrays (or anything `np.asarray` accepts) in the C-ABI
layouts described in the source header and return numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_DIR = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_DIR, "coarse_oracle.cpp")
_LIB = os.path.join(_DIR, "liboracle.so")
_lib: Optional[ctypes.CDLL] = None

LINK_C64 = 0
LINK_I16 = 1


def build(force: bool = False) -> str:
    """Compile liboracle.so if missing or older than its source; return its path."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
        return _LIB
    cmd = ["g++", "-std=c++17", "-O3", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", _LIB, _SRC]
    subprocess.run(cmd, check=True, cwd=_DIR)
    return _LIB


def _load() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i4 = ctypes.POINTER(ctypes.c_int)
        vp, ci, ci64 = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64
        lib.oracle_max_threads.restype = ci
        lib.oracle_coarse_apply.restype = ci
        lib.oracle_coarse_apply.argtypes = [i4, ci, ci, vp, vp, vp, vp, ci, ci, ci]
        lib.oracle_coarse_apply_sites.restype = ci
        lib.oracle_coarse_apply_sites.argtypes = [i4, ci, ci, vp, vp, vp, vp, ci, ci, vp, ci64, ci]
        lib.oracle_neighbours.restype = ci
        lib.oracle_neighbours.argtypes = [i4, ci64, vp]
        lib.oracle_quantize_i16.restype = ci
        lib.oracle_quantize_i16.argtypes = [vp, ci64, ci, vp, vp]
        lib.oracle_dequantize_i16.restype = ci
        lib.oracle_dequantize_i16.argtypes = [vp, vp, ci64, ci, vp]
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def _dims(dims: Sequence[int]):
    return (ctypes.c_int * 4)(*[int(d) for d in dims])


def _as_links(links, link_precision: int, V: int, Nc: int) -> np.ndarray:
    if link_precision == LINK_C64:
        a = np.ascontiguousarray(np.asarray(links))
        if a.dtype == np.complex64:
            a = a.view(np.float32)
        if a.dtype != np.float32 or a.size != V * 9 * Nc * Nc * 2:
            raise ValueError("c64 links must be complex64/float32 of V*9*Nc*Nc entries")
        return a
    a = np.ascontiguousarray(np.asarray(links))
    if a.dtype != np.int16 or a.size != V * 9 * Nc * Nc * 2:
        raise ValueError("i16 links must be int16 [V][9][Nc][Nc][2]")
    return a


def _as_vec(v, V: int, Nc: int, nrhs: int) -> np.ndarray:
    a = np.ascontiguousarray(np.asarray(v))
    if a.dtype == np.complex64:
        a = a.view(np.float32)
    if a.dtype != np.float32 or a.size != V * Nc * nrhs * 2:
        raise ValueError("vectors must be complex64 [V][Nc][nrhs]")
    return a


def coarse_apply(dims, Nc: int, links, vec, nrhs: int = 1, dagger: int = 0,
                 link_precision: int = LINK_C64, scales=None, nthreads: int = 0) -> np.ndarray:
    """Full-lattice oracle apply; returns complex128 [V][Nc][nrhs]."""
    V = int(np.prod([int(d) for d in dims]))
    L = _as_links(links, link_precision, V, Nc)
    x = _as_vec(vec, V, Nc, nrhs)
    sc = None
    if link_precision == LINK_I16:
        sc = np.ascontiguousarray(np.asarray(scales, dtype=np.float32))
        if sc.size != V * 9:
            raise ValueError("scales must be float32 [V][9]")
    out = np.empty((V, Nc, nrhs), dtype=np.complex128)
    rc = _load().oracle_coarse_apply(_dims(dims), Nc, link_precision, L.ctypes.data,
                                     sc.ctypes.data if sc is not None else None,
                                     x.ctypes.data, out.ctypes.data, nrhs, dagger, nthreads)
    if rc != 0:
        raise ValueError(f"oracle_coarse_apply rejected its arguments (rc={rc})")
    return out


def coarse_apply_sites(dims, Nc: int, links, vec, sites, nrhs: int = 1, dagger: int = 0,
                       link_precision: int = LINK_C64, scales=None, nthreads: int = 0) -> np.ndarray:
    """Oracle apply evaluated only at `sites`; returns complex128 [len(sites)][Nc][nrhs]."""
    V = int(np.prod([int(d) for d in dims]))
    L = _as_links(links, link_precision, V, Nc)
    x = _as_vec(vec, V, Nc, nrhs)
    sc = None
    if link_precision == LINK_I16:
        sc = np.ascontiguousarray(np.asarray(scales, dtype=np.float32))
    st = np.ascontiguousarray(np.asarray(sites, dtype=np.int64))
    out = np.empty((st.size, Nc, nrhs), dtype=np.complex128)
    rc = _load().oracle_coarse_apply_sites(_dims(dims), Nc, link_precision, L.ctypes.data,
                                           sc.ctypes.data if sc is not None else None,
                                           x.ctypes.data, out.ctypes.data, nrhs, dagger,
                                           st.ctypes.data, st.size, nthreads)
    if rc != 0:
        raise ValueError(f"oracle_coarse_apply_sites rejected its arguments (rc={rc})")
    return out


def neighbours(dims, s: int) -> np.ndarray:
    """[s, s(x+0^),..,s(x+3^), s(x-0^),..,s(x-3^)] as int64[9]."""
    nbr = np.empty(9, dtype=np.int64)
    rc = _load().oracle_neighbours(_dims(dims), int(s), nbr.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_neighbours rejected its arguments")
    return nbr


def quantize_i16(links, Nc: int):
    """O5 quantiser. links: complex64 [...][Nc][Nc]; returns (int16 [...][Nc][Nc][2], float32 [...])."""
    a = np.ascontiguousarray(np.asarray(links))
    if a.dtype == np.complex64:
        a = a.view(np.float32)
    if a.dtype != np.float32 or a.size % (2 * Nc * Nc) != 0:
        raise ValueError("links must be complex64/float32 matrices of Nc*Nc entries")
    n = a.size // (2 * Nc * Nc)
    q = np.empty(a.size, dtype=np.int16)
    scales = np.empty(n, dtype=np.float32)
    rc = _load().oracle_quantize_i16(a.ctypes.data, n, Nc, q.ctypes.data, scales.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_quantize_i16 rejected its arguments")
    return q.reshape(n, Nc, Nc, 2), scales


def dequantize_i16(q, scales, Nc: int) -> np.ndarray:
    """(int16, float32 scales) -> complex128 [n][Nc][Nc], entry = q*scale in double."""
    qa = np.ascontiguousarray(np.asarray(q, dtype=np.int16))
    sc = np.ascontiguousarray(np.asarray(scales, dtype=np.float32))
    n = sc.size
    out = np.empty((n, Nc, Nc), dtype=np.complex128)
    rc = _load().oracle_dequantize_i16(qa.ctypes.data, sc.ctypes.data, n, Nc, out.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_dequantize_i16 rejected its arguments")
    return out
