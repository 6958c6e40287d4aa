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
        lib.oracle_coarse_apply_parts.restype = ci
        lib.oracle_coarse_apply_parts.argtypes = [i4, ci, ci, vp, vp, vp, vp, vp, ci, ci, ci, ci,
                                                  ctypes.c_double, ctypes.c_double, ci]
        lib.oracle_coarse_apply_hvec.restype = ci
        lib.oracle_coarse_apply_hvec.argtypes = [i4, ci, ci, vp, vp, vp, vp, vp, ci, ci, ci]
        lib.oracle_coarse_apply_hvec_sites.restype = ci
        lib.oracle_coarse_apply_hvec_sites.argtypes = [i4, ci, ci, vp, vp, vp, vp, vp, ci, ci, vp, ci64, ci]
        lib.oracle_quantize_vec_i16.restype = ci
        lib.oracle_quantize_vec_i16.argtypes = [vp, ci64, ci, ci, vp, vp]
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


# ----------------------------------------------------------------------------- even/odd (row f1)
PARITY_EVEN, PARITY_ODD, PARITY_ALL = 0, 1, 2
LOCAL_NONE, LOCAL_X, LOCAL_IDENTITY = 0, 1, 2


def site_parities(dims) -> np.ndarray:
    """pi(x) = (x0+x1+x2+x3) mod 2 for every site index s(x) (x0 fastest)."""
    L0, L1, L2, L3 = (int(d) for d in dims)
    x3, x2, x1, x0 = np.meshgrid(np.arange(L3), np.arange(L2), np.arange(L1), np.arange(L0), indexing="ij")
    return ((x0 + x1 + x2 + x3) & 1).reshape(-1)


def coarse_apply_parts(dims, Nc: int, links, u, w, nrhs: int = 1, dagger: int = 0, parity: int = PARITY_ALL,
                       local: int = LOCAL_X, alpha: float = 1.0, beta: float = 1.0,
                       link_precision: int = LINK_C64, scales=None, nthreads: int = 0) -> np.ndarray:
    """O7: out(x) = alpha*Loc(x) + beta*Hop(x) on the sites of `parity` (zero elsewhere);
    Loc = X.u | u | 0, Hop = the eight hopping terms applied to w.  complex128 [V][Nc][nrhs]."""
    V = int(np.prod([int(d) for d in dims]))
    L = _as_links(links, link_precision, V, Nc)
    ww = _as_vec(w, V, Nc, nrhs)
    uu = None if u is None else _as_vec(u, V, Nc, nrhs)
    sc = None
    if link_precision == LINK_I16:
        sc = np.ascontiguousarray(np.asarray(scales, dtype=np.float32))
    out = np.empty((V, Nc, nrhs), dtype=np.complex128)
    rc = _load().oracle_coarse_apply_parts(_dims(dims), Nc, link_precision, L.ctypes.data,
                                           sc.ctypes.data if sc is not None else None,
                                           uu.ctypes.data if uu is not None else None,
                                           ww.ctypes.data, out.ctypes.data, nrhs, dagger, parity, local,
                                           float(alpha), float(beta), nthreads)
    if rc != 0:
        raise ValueError(f"oracle_coarse_apply_parts rejected its arguments (rc={rc})")
    return out


def _even_dims(dims):
    if any(int(d) % 2 for d in dims):
        raise ValueError("the even/odd decomposition needs every extent to be even")


def schur_apply(dims, Nc: int, links, v, parity: int, nrhs: int = 1) -> np.ndarray:
    """Textbook Schur complement of the coarse operator on the sites of parity p (q = 1-p):
        S_p v = X_p v - D_pq X_q^{-1} D_qp v          ("Schur-preconditioned")
    with D the hopping part.  v lives on parity p (its other-parity entries are ignored).  Steps:
    O7 hop to parity q, numpy dense solve with X(x) per site of q, O7 X - hop back to p.  The
    intermediate vectors are rounded to complex64 exactly where the CUDA path stores them."""
    _even_dims(dims)
    links = np.asarray(links)
    V = links.shape[0]
    q = 1 - parity
    par = site_parities(dims)
    vp = np.where((par == parity)[:, None, None], np.asarray(v).reshape(V, Nc, nrhs), 0).astype(np.complex64)
    t = coarse_apply_parts(dims, Nc, links, None, vp, nrhs, 0, q, LOCAL_NONE, 0.0, 1.0)
    t2 = np.zeros_like(t)
    for s in np.nonzero(par == q)[0]:
        t2[s] = np.linalg.solve(links[s, 0].astype(np.complex128), t[s])
    return coarse_apply_parts(dims, Nc, links, vp, t2.astype(np.complex64), nrhs, 0, parity, LOCAL_X, 1.0, -1.0)


def hat_links(links, slot0_inverse: bool = False) -> np.ndarray:
    """Block-preconditioned links: Yhat_m(x) = X(x)^{-1} Y_m(x), m = 1..8; slot 0
    holds the identity, or X(x)^{-1} when slot0_inverse.  complex128 [V][9][Nc][Nc] (cast to complex64
    before use as an input)."""
    links = np.asarray(links).astype(np.complex128)
    out = np.empty_like(links)
    Nc = links.shape[-1]
    for s in range(links.shape[0]):
        out[s, 0] = np.linalg.solve(links[s, 0], np.eye(Nc)) if slot0_inverse else np.eye(Nc)
        out[s, 1:] = np.linalg.solve(links[s, 0][None, :, :], links[s, 1:])
    return out


def schur_hat_apply(dims, Nc: int, hat, v, parity: int, nrhs: int = 1, dagger: int = 0) -> np.ndarray:
    """Left-preconditioned Schur operator from block-preconditioned links, two O7 hops:
        Shat_p v = v - Dhat_pq Dhat_qp v        ( = X_p^{-1} S_p v when hat = hat_links(links) )
    dagger = 1 gives its adjoint, v - (Dhat^H)_pq (Dhat^H)_qp v."""
    _even_dims(dims)
    V = int(np.prod([int(d) for d in dims]))
    q = 1 - parity
    par = site_parities(dims)
    vp = np.where((par == parity)[:, None, None], np.asarray(v).reshape(V, Nc, nrhs), 0).astype(np.complex64)
    t = coarse_apply_parts(dims, Nc, hat, None, vp, nrhs, dagger, q, LOCAL_NONE, 0.0, 1.0)
    return coarse_apply_parts(dims, Nc, hat, vp, t.astype(np.complex64), nrhs, dagger, parity,
                              LOCAL_IDENTITY, 1.0, -1.0)


# ----------------------------------------------------------------------------- half vectors (row f2)
def quantize_vec_i16(v, Nc: int, nrhs: int = 1):
    """O8 quantiser. v: complex64 [V][Nc][nrhs]; returns (int16 [V][Nc][nrhs][2], float32 [V][nrhs])."""
    a = _as_vec(v, np.asarray(v).size // (Nc * nrhs), Nc, nrhs)
    V = a.size // (2 * Nc * nrhs)
    q = np.empty((V, Nc, nrhs, 2), dtype=np.int16)
    norms = np.empty((V, nrhs), dtype=np.float32)
    rc = _load().oracle_quantize_vec_i16(a.ctypes.data, V, Nc, nrhs, q.ctypes.data, norms.ctypes.data)
    if rc != 0:
        raise ValueError("oracle_quantize_vec_i16 rejected its arguments")
    return q, norms


def coarse_apply_hvec(dims, Nc: int, links, vec_q, vec_norms, nrhs: int = 1, dagger: int = 0,
                      link_precision: int = LINK_C64, scales=None, nthreads: int = 0) -> np.ndarray:
    """O8: full apply on half-precision input vectors (int16 + per-(site,rhs) norm); complex128 out."""
    V = int(np.prod([int(d) for d in dims]))
    L = _as_links(links, link_precision, V, Nc)
    q = np.ascontiguousarray(np.asarray(vec_q, dtype=np.int16))
    nm = np.ascontiguousarray(np.asarray(vec_norms, dtype=np.float32))
    if q.size != V * Nc * nrhs * 2 or nm.size != V * nrhs:
        raise ValueError("half vectors must be int16 [V][Nc][nrhs][2] with float32 norms [V][nrhs]")
    sc = None
    if link_precision == LINK_I16:
        sc = np.ascontiguousarray(np.asarray(scales, dtype=np.float32))
    out = np.empty((V, Nc, nrhs), dtype=np.complex128)
    rc = _load().oracle_coarse_apply_hvec(_dims(dims), Nc, link_precision, L.ctypes.data,
                                          sc.ctypes.data if sc is not None else None, q.ctypes.data,
                                          nm.ctypes.data, out.ctypes.data, nrhs, dagger, nthreads)
    if rc != 0:
        raise ValueError(f"oracle_coarse_apply_hvec rejected its arguments (rc={rc})")
    return out


def coarse_apply_hvec_sites(dims, Nc: int, links, vec_q, vec_norms, sites, nrhs: int = 1, dagger: int = 0,
                            link_precision: int = LINK_C64, scales=None, nthreads: int = 0) -> np.ndarray:
    """O8 evaluated only at `sites`; returns complex128 [len(sites)][Nc][nrhs]."""
    V = int(np.prod([int(d) for d in dims]))
    L = _as_links(links, link_precision, V, Nc)
    q = np.ascontiguousarray(np.asarray(vec_q, dtype=np.int16))
    nm = np.ascontiguousarray(np.asarray(vec_norms, dtype=np.float32))
    if q.size != V * Nc * nrhs * 2 or nm.size != V * nrhs:
        raise ValueError("half vectors must be int16 [V][Nc][nrhs][2] with float32 norms [V][nrhs]")
    sc = None
    if link_precision == LINK_I16:
        sc = np.ascontiguousarray(np.asarray(scales, dtype=np.float32))
    st = np.ascontiguousarray(np.asarray(sites, dtype=np.int64))
    out = np.empty((st.size, Nc, nrhs), dtype=np.complex128)
    rc = _load().oracle_coarse_apply_hvec_sites(_dims(dims), Nc, link_precision, L.ctypes.data,
                                                sc.ctypes.data if sc is not None else None, q.ctypes.data,
                                                nm.ctypes.data, out.ctypes.data, nrhs, dagger,
                                                st.ctypes.data, st.size, nthreads)
    if rc != 0:
        raise ValueError(f"oracle_coarse_apply_hvec_sites rejected its arguments (rc={rc})")
    return out


# ----------------------------------------------------------------------------- CA-GCR(s) (row f3)
def _apply_fp64(apply_fn, v):
    """A v for a complex128 v through an operator that takes complex64 input: A is linear, so
    A v = A hi + A lo with hi = complex64(v), lo = complex64(v - hi) (error ~1e-15 |v|)."""
    hi = v.astype(np.complex64)
    lo = (v - hi.astype(np.complex128)).astype(np.complex64)
    return apply_fn(hi) + apply_fn(lo)


def cagcr(apply_fn, b, x0, s: int, cycles: int = 1):
    """Communication-avoiding GCR(s), the paper's smoother / coarsest-level solver ("CA-GCR(8)",
    Table 1 L116/L122/L130, "Chebyshev-basis CA-GCR(16)" L134; reading R23).  One cycle, by its
    definition, minimises the residual over the Krylov space:
        r0 = b - A x0;    x = x0 + argmin_{z in K_s(A, r0)} || r0 - A z ||_2,   K_s = span{r0, A r0, .., A^(s-1) r0}
    The definition names no basis (power, Chebyshev, ... span the same space), so the oracle evaluates it the
    numerically safest way, entirely in fp64: an orthonormal basis of K_s by Arnoldi with re-orthogonalisation,
    then a dense least-squares problem for the coefficients (numpy.linalg.lstsq, no cut-off).  A CUDA path
    is free to build the space however it likes; how close it gets to this minimum is what is tested.
    apply_fn(v complex64 [n]) -> complex128 [n].  Returns (x complex128, [||r||_2 before each cycle and
    after the last])."""
    b = np.asarray(b).reshape(-1).astype(np.complex128)
    x = np.asarray(x0).reshape(-1).astype(np.complex128)
    norms = []
    r = b - _apply_fp64(apply_fn, x) if np.any(x != 0) else b.copy()
    for _ in range(cycles):
        beta = float(np.linalg.norm(r))
        norms.append(beta)
        if beta == 0.0:
            continue
        V = [r / beta]                       # orthonormal basis of K_s
        AV = []                              # A V_k
        for k in range(s):
            w = _apply_fp64(apply_fn, V[k])
            AV.append(w)
            if k + 1 < s:
                u = w.copy()
                for _pass in range(2):       # modified Gram-Schmidt, twice
                    for q in V:
                        u -= np.vdot(q, u) * q
                nu = float(np.linalg.norm(u))
                if nu <= 1e-14 * float(np.linalg.norm(w)):
                    break                    # the Krylov space is exhausted (invariant subspace)
                V.append(u / nu)
        Vm = np.stack(V, axis=1)
        Qm = np.stack(AV[:Vm.shape[1]], axis=1)
        y = np.linalg.lstsq(Qm, r, rcond=1e-300)[0]
        x = x + Vm @ y
        r = r - Qm @ y
    norms.append(float(np.linalg.norm(r)))
    return x, norms
