"""paper_2212_12559_b200 — B200-native coarse-grid Dirac operator apply (arXiv:2212.12559 §3.1).

Thin Python binding over libcoarseop.so (include/coarse_op.h).  The functions carry the C ABI's
names and only marshal arguments: torch is used for device memory and streams, every step of the
apply runs in the library's sm_100a kernels.  There is no CPU fallback: if the shared library is
missing and cannot be built, importing `lib()` raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

from . import build as _build

LINK_C64 = 0
LINK_I16 = 1

OK, EINVAL, EUNSUPPORTED, ENOTREADY, ECUDA, ENOMEM = 0, -1, -2, -3, -4, -5

PATH_AUTO, PATH_SIMPLE, PATH_STREAM, PATH_TENSOR, PATH_BLOCK = 0, 1, 2, 3, 4
OPT_PATH, OPT_GRID, OPT_STAGES, OPT_FINE, OPT_KEEP_LINKS, OPT_PDL, OPT_SPLIT_DAGGER, OPT_WARP_ITEMS, OPT_TENSOR_I8 = 0, 1, 2, 3, 4, 5, 6, 7, 8
PARITY_EVEN, PARITY_ODD, PARITY_ALL = 0, 1, 2
LOCAL_NONE, LOCAL_X, LOCAL_IDENTITY = 0, 1, 2

EXPORTS = (
    "coarse_op_create", "coarse_op_link_bytes", "coarse_op_scale_bytes", "coarse_op_vector_bytes",
    "coarse_op_set_links", "coarse_op_set_option", "coarse_op_apply", "coarse_op_apply_parts", "coarse_op_apply_hvec",
    "coarse_op_apply_hout", "coarse_op_apply_static",
    "coarse_op_quantize_vec_i16", "coarse_op_apply_host",
    "coarse_op_last_launches", "coarse_op_last_path", "coarse_op_quantize_i16", "coarse_op_probe_read", "coarse_op_cagcr_work_bytes",
    "coarse_op_cagcr", "coarse_op_cagcr_schur", "coarse_op_cagcr_cheb_work_bytes",
    "coarse_op_cagcr_cheb", "coarse_op_hat_work_bytes", "coarse_op_build_hat_links", "coarse_op_destroy",
    "coarse_op_last_error",
)

_lib: Optional[ctypes.CDLL] = None


class CoarseOpError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"libcoarseop error {code}: {message}")
        self.code = code


def lib() -> ctypes.CDLL:
    """Load (building if needed) libcoarseop.so and declare its prototypes."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB_PATH
    if _build.is_stale():
        path = _build.build_library()          # raises if nvcc is missing: no silent fallback
    L = ctypes.CDLL(path)
    vp, ci, ci64, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_size_t
    L.coarse_op_create.restype = vp
    L.coarse_op_create.argtypes = [ctypes.POINTER(ci), ci, ci]
    L.coarse_op_link_bytes.restype = sz
    L.coarse_op_link_bytes.argtypes = [vp]
    L.coarse_op_scale_bytes.restype = sz
    L.coarse_op_scale_bytes.argtypes = [vp]
    L.coarse_op_vector_bytes.restype = sz
    L.coarse_op_vector_bytes.argtypes = [vp, ci]
    L.coarse_op_set_links.restype = ci
    L.coarse_op_set_links.argtypes = [vp, vp, vp]
    L.coarse_op_set_option.restype = ci
    L.coarse_op_set_option.argtypes = [vp, ci, ci]
    L.coarse_op_apply.restype = ci
    L.coarse_op_apply.argtypes = [vp, vp, vp, ci, ci, vp]
    L.coarse_op_apply_parts.restype = ci
    L.coarse_op_apply_parts.argtypes = [vp, vp, vp, vp, ci, ci, ci, ci, ctypes.c_float, ctypes.c_float, vp]
    L.coarse_op_apply_hvec.restype = ci
    L.coarse_op_apply_hvec.argtypes = [vp, vp, vp, vp, ci, ci, vp]
    L.coarse_op_apply_static.restype = ci
    L.coarse_op_apply_static.argtypes = [vp, vp, vp, ci, ci, vp]
    L.coarse_op_apply_hout.restype = ci
    L.coarse_op_apply_hout.argtypes = [vp, vp, vp, vp, vp, vp, ci, ci, vp]
    L.coarse_op_quantize_vec_i16.restype = ci
    L.coarse_op_quantize_vec_i16.argtypes = [vp, ci64, ci, ci, vp, vp, vp]
    L.coarse_op_apply_host.restype = ci
    L.coarse_op_apply_host.argtypes = [vp, vp, vp, ci, ci, vp]
    L.coarse_op_last_launches.restype = ci
    L.coarse_op_last_launches.argtypes = [vp]
    L.coarse_op_last_path.restype = ci
    L.coarse_op_last_path.argtypes = [vp]
    L.coarse_op_hat_work_bytes.restype = sz
    L.coarse_op_hat_work_bytes.argtypes = [vp]
    L.coarse_op_build_hat_links.restype = ci
    L.coarse_op_build_hat_links.argtypes = [vp, vp, ci, vp, vp, vp]
    L.coarse_op_quantize_i16.restype = ci
    L.coarse_op_quantize_i16.argtypes = [vp, ci64, ci, vp, vp, vp]
    L.coarse_op_cagcr_work_bytes.restype = sz
    L.coarse_op_cagcr_work_bytes.argtypes = [vp, ci]
    L.coarse_op_cagcr.restype = ci
    L.coarse_op_cagcr.argtypes = [vp, vp, vp, ci, ci, ci, vp, vp, vp]
    L.coarse_op_cagcr_schur.restype = ci
    L.coarse_op_cagcr_schur.argtypes = [vp, vp, vp, ci, ci, ci, ci, vp, vp, vp]
    L.coarse_op_cagcr_cheb_work_bytes.restype = sz
    L.coarse_op_cagcr_cheb_work_bytes.argtypes = [vp, ci]
    L.coarse_op_cagcr_cheb.restype = ci
    L.coarse_op_cagcr_cheb.argtypes = [vp, vp, vp, ci, ci, ci, ctypes.c_float, ctypes.c_float, ci, vp, vp, vp]
    L.coarse_op_probe_read.restype = ci
    L.coarse_op_probe_read.argtypes = [vp, sz, ci, ci, vp]
    L.coarse_op_destroy.restype = None
    L.coarse_op_destroy.argtypes = [vp]
    L.coarse_op_last_error.restype = ctypes.c_char_p
    L.coarse_op_last_error.argtypes = []
    _lib = L
    return L


def coarse_op_last_error() -> str:
    return lib().coarse_op_last_error().decode()


def _check(rc: int) -> None:
    if rc != OK:
        raise CoarseOpError(rc, coarse_op_last_error())


def _ptr(t) -> Optional[int]:
    return None if t is None else int(t.data_ptr())


def _stream_handle(stream) -> Optional[int]:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream)
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)


def coarse_op_create(dims: Sequence[int], Nc: int, link_precision: int) -> int:
    arr = (ctypes.c_int * 4)(*[int(d) for d in dims])
    h = lib().coarse_op_create(arr, int(Nc), int(link_precision))
    if not h:
        raise CoarseOpError(EINVAL, coarse_op_last_error())
    return h


def coarse_op_link_bytes(op: int) -> int:
    return int(lib().coarse_op_link_bytes(op))


def coarse_op_scale_bytes(op: int) -> int:
    return int(lib().coarse_op_scale_bytes(op))


def coarse_op_vector_bytes(op: int, nrhs: int) -> int:
    return int(lib().coarse_op_vector_bytes(op, int(nrhs)))


def coarse_op_set_links(op: int, links, scales=None) -> None:
    """links / scales: CUDA tensors in the ABI layouts (borrowed: keep them alive)."""
    for t in (links, scales):
        if t is not None and (not t.is_cuda or not t.is_contiguous()):
            raise ValueError("links/scales must be contiguous CUDA tensors")
    if links.numel() * links.element_size() != coarse_op_link_bytes(op):
        raise ValueError("links tensor has the wrong number of bytes for this operator")
    if scales is not None and scales.numel() * scales.element_size() != coarse_op_scale_bytes(op):
        raise ValueError("scales tensor has the wrong number of bytes for this operator")
    _check(lib().coarse_op_set_links(op, _ptr(links), _ptr(scales)))


def coarse_op_set_option(op: int, option: int, value: int) -> None:
    _check(lib().coarse_op_set_option(op, int(option), int(value)))


def coarse_op_apply(op: int, vin, vout, nrhs: int = 1, dagger: int = 0, stream=None) -> None:
    """vin / vout: contiguous CUDA complex64 tensors [V][Nc][nrhs]; enqueues on `stream`
    (default: torch's current stream) and returns without synchronising."""
    for t in (vin, vout):
        if not t.is_cuda or not t.is_contiguous():
            raise ValueError("vectors must be contiguous CUDA tensors")
        if t.numel() * t.element_size() != coarse_op_vector_bytes(op, nrhs):
            raise ValueError("vector tensor has the wrong number of bytes for this operator/nrhs")
    _check(lib().coarse_op_apply(op, _ptr(vin), _ptr(vout), int(nrhs), int(dagger), _stream_handle(stream)))


STATIC_MAX_SITES = 8192        # COARSE_STATIC_MAX_SITES in include/coarse_op.h


def coarse_op_apply_static(op: int, vin, vout, nrhs: int = 1, dagger: int = 0, stream=None) -> None:
    """The plain apply on int16 links with the kernel's scratch in a static device array of the library: the call
    allocates nothing (include/coarse_op.h; at most STATIC_MAX_SITES sites; calls that overlap on the GPU race)."""
    for t in (vin, vout):
        if not t.is_cuda or not t.is_contiguous():
            raise ValueError("vectors must be contiguous CUDA tensors")
        if t.numel() * t.element_size() != coarse_op_vector_bytes(op, nrhs):
            raise ValueError("vector tensor has the wrong number of bytes for this operator/nrhs")
    _check(lib().coarse_op_apply_static(op, _ptr(vin), _ptr(vout), int(nrhs), int(dagger), _stream_handle(stream)))


def coarse_op_apply_parts(op: int, u, w, vout, nrhs: int = 1, dagger: int = 0, parity: int = PARITY_ALL,
                          local: int = LOCAL_X, alpha: float = 1.0, beta: float = 1.0, stream=None) -> None:
    """out(x) = alpha*Loc(u)(x) + beta*Hop(w)(x) on the sites of `parity` (include/coarse_op.h).
    u / w / vout: contiguous CUDA complex64 tensors [V][Nc][nrhs]; u may be None for LOCAL_NONE."""
    for t in (u, w, vout):
        if t is None:
            continue
        if not t.is_cuda or not t.is_contiguous():
            raise ValueError("vectors must be contiguous CUDA tensors")
        if t.numel() * t.element_size() != coarse_op_vector_bytes(op, nrhs):
            raise ValueError("vector tensor has the wrong number of bytes for this operator/nrhs")
    _check(lib().coarse_op_apply_parts(op, _ptr(u), _ptr(w), _ptr(vout), int(nrhs), int(dagger), int(parity),
                                       int(local), float(alpha), float(beta), _stream_handle(stream)))


def coarse_op_apply_hvec(op: int, vin_q, vin_norms, vout, nrhs: int = 1, dagger: int = 0, stream=None) -> None:
    """Plain apply on half-precision input vectors: vin_q CUDA int16 [V][Nc][nrhs][2], vin_norms CUDA
    float32 [V][nrhs]; vout CUDA complex64 [V][Nc][nrhs]."""
    for t in (vin_q, vin_norms, vout):
        if not t.is_cuda or not t.is_contiguous():
            raise ValueError("apply_hvec needs contiguous CUDA tensors")
    vb = coarse_op_vector_bytes(op, nrhs)
    if vout.numel() * vout.element_size() != vb or vin_q.numel() * vin_q.element_size() * 2 != vb:
        raise ValueError("vector tensors have the wrong number of bytes for this operator/nrhs")
    if vin_norms.numel() % nrhs or vin_norms.element_size() != 4:
        raise ValueError("vin_norms must hold one float32 per (site, rhs)")
    _check(lib().coarse_op_apply_hvec(op, _ptr(vin_q), _ptr(vin_norms), _ptr(vout), int(nrhs), int(dagger),
                                      _stream_handle(stream)))


def coarse_op_apply_hout(op: int, vin, vin_norms, vout, vout_q, vout_norms, nrhs: int = 1, dagger: int = 0, stream=None) -> None:
    """The apply with a half-precision result beside the complex64 one.  vin: CUDA complex64 [V][Nc][nrhs] (vin_norms None)
    or int16 [V][Nc][nrhs][2] with vin_norms float32 [V][nrhs]; vout complex64 [V][Nc][nrhs]; vout_q int16 [V][Nc][nrhs][2];
    vout_norms float32 [V][nrhs]."""
    for t in (vin, vout, vout_q, vout_norms) + ((vin_norms,) if vin_norms is not None else ()):
        if not t.is_cuda or not t.is_contiguous():
            raise ValueError("apply_hout needs contiguous CUDA tensors")
    vb = coarse_op_vector_bytes(op, nrhs)
    if vout.numel() * vout.element_size() != vb or vout_q.numel() * vout_q.element_size() * 2 != vb:
        raise ValueError("output tensors have the wrong number of bytes for this operator/nrhs")
    if vin.numel() * vin.element_size() != (vb // 2 if vin_norms is not None else vb):
        raise ValueError("input tensor has the wrong number of bytes for this operator/nrhs")
    if vout_norms.element_size() != 4 or vout_norms.numel() % nrhs:
        raise ValueError("vout_norms must hold one float32 per (site, rhs)")
    _check(lib().coarse_op_apply_hout(op, _ptr(vin), _ptr(vin_norms) if vin_norms is not None else None, _ptr(vout), _ptr(vout_q),
                                      _ptr(vout_norms), int(nrhs), int(dagger), _stream_handle(stream)))


def coarse_op_quantize_vec_i16(v_c64, Nc: int, nrhs: int, q_out, norms_out, stream=None) -> None:
    """v_c64: CUDA complex64 [V][Nc][nrhs]; q_out: CUDA int16 [V][Nc][nrhs][2]; norms_out: CUDA float32 [V][nrhs]."""
    n_sites = v_c64.numel() // (Nc * nrhs)
    if q_out.numel() != 2 * v_c64.numel() or norms_out.numel() != n_sites * nrhs:
        raise ValueError("quantize_vec_i16: output tensors have the wrong size")
    for t in (v_c64, q_out, norms_out):
        if not t.is_cuda or not t.is_contiguous():
            raise ValueError("quantize_vec_i16 needs contiguous CUDA tensors")
    _check(lib().coarse_op_quantize_vec_i16(_ptr(v_c64), n_sites, int(Nc), int(nrhs), _ptr(q_out), _ptr(norms_out),
                                            _stream_handle(stream)))


def coarse_op_apply_host(op: int, vin_host, vout_host, nrhs: int = 1, dagger: int = 0, stream=None) -> None:
    """vin_host / vout_host: contiguous CPU complex64 tensors (pinned for full PCIe rate).
    Copies in, applies, copies out and synchronises the stream."""
    for t in (vin_host, vout_host):
        if t.is_cuda or not t.is_contiguous():
            raise ValueError("host vectors must be contiguous CPU tensors")
        if t.numel() * t.element_size() != coarse_op_vector_bytes(op, nrhs):
            raise ValueError("vector tensor has the wrong number of bytes for this operator/nrhs")
    _check(lib().coarse_op_apply_host(op, _ptr(vin_host), _ptr(vout_host), int(nrhs), int(dagger),
                                      _stream_handle(stream)))


def coarse_op_last_launches(op: int) -> int:
    return int(lib().coarse_op_last_launches(op))


def coarse_op_last_path(op: int) -> int:
    return int(lib().coarse_op_last_path(op))


def coarse_op_quantize_i16(links_c64, Nc: int, q_out, scales_out, stream=None) -> None:
    """links_c64: CUDA complex64 [...][Nc][Nc]; q_out: CUDA int16 [...][Nc][Nc][2]; scales_out: CUDA
    float32 [...] (one per matrix)."""
    n = links_c64.numel() // (Nc * Nc)
    if q_out.numel() != 2 * links_c64.numel() or scales_out.numel() != n:
        raise ValueError("quantize_i16: output tensors have the wrong size")
    for t in (links_c64, q_out, scales_out):
        if not t.is_cuda or not t.is_contiguous():
            raise ValueError("quantize_i16 needs contiguous CUDA tensors")
    _check(lib().coarse_op_quantize_i16(_ptr(links_c64), n, int(Nc), _ptr(q_out), _ptr(scales_out),
                                        _stream_handle(stream)))


HAT_SLOT0_IDENTITY, HAT_SLOT0_XINV = 0, 1


def coarse_op_hat_work_bytes(op: int) -> int:
    return int(lib().coarse_op_hat_work_bytes(op))


def coarse_op_build_hat_links(op: int, out_links, slot0: int = HAT_SLOT0_IDENTITY, work=None, info=None, stream=None):
    """out_links: CUDA complex64 [V][9][Nc][Nc]; work: CUDA uint8 tensor of coarse_op_hat_work_bytes(op)
    bytes (allocated when None); info: optional CUDA int32 tensor [1].  Returns the work tensor."""
    import torch
    if work is None:
        work = torch.empty(coarse_op_hat_work_bytes(op), dtype=torch.uint8, device=out_links.device)
    for t in (out_links, work) + ((info,) if info is not None else ()):
        if not t.is_cuda or not t.is_contiguous():
            raise ValueError("build_hat_links needs contiguous CUDA tensors")
    if out_links.dtype != torch.complex64:
        raise ValueError("build_hat_links: out_links must be complex64")
    if info is not None and (info.dtype != torch.int32 or info.numel() < 1):
        raise ValueError("build_hat_links: info must be an int32 tensor")
    _check(lib().coarse_op_build_hat_links(op, _ptr(out_links), int(slot0), _ptr(work),
                                           _ptr(info) if info is not None else None, _stream_handle(stream)))
    return work


def coarse_op_cagcr_work_bytes(op: int, s: int) -> int:
    return int(lib().coarse_op_cagcr_work_bytes(op, int(s)))


def coarse_op_cagcr(op: int, b, x, s: int, cycles: int = 1, x_is_zero: bool = True, work=None, info=None,
                    stream=None, schur_parity: Optional[int] = None) -> None:
    """CA-GCR(s) smoother cycles on CUDA complex64 vectors b, x [V][Nc]; work: CUDA uint8 tensor of at
    least coarse_op_cagcr_work_bytes(op, s) bytes; info: optional CUDA float64 tensor [cycles][3]."""
    for t in (b, x, work):
        if t is None or not t.is_cuda or not t.is_contiguous():
            raise ValueError("cagcr needs contiguous CUDA tensors b, x, work")
    if work.numel() * work.element_size() < coarse_op_cagcr_work_bytes(op, s):
        raise ValueError("cagcr: work buffer too small")
    if b.numel() * b.element_size() != coarse_op_vector_bytes(op, 1) or x.numel() != b.numel():
        raise ValueError("cagcr: b / x have the wrong size (1 RHS)")
    if info is not None and (info.numel() < 3 * cycles or info.element_size() != 8 or not info.is_cuda):
        raise ValueError("cagcr: info must be a CUDA float64 tensor with 3 * cycles entries")
    if schur_parity is None:
        _check(lib().coarse_op_cagcr(op, _ptr(b), _ptr(x), int(s), int(cycles), 1 if x_is_zero else 0, _ptr(work),
                                     _ptr(info), _stream_handle(stream)))
    else:
        _check(lib().coarse_op_cagcr_schur(op, _ptr(b), _ptr(x), int(s), int(cycles), 1 if x_is_zero else 0,
                                           int(schur_parity), _ptr(work), _ptr(info), _stream_handle(stream)))


def coarse_op_cagcr_cheb_work_bytes(op: int, s: int) -> int:
    return int(lib().coarse_op_cagcr_cheb_work_bytes(op, int(s)))


def coarse_op_cagcr_cheb(op: int, b, x, s: int, lambda_min: float, lambda_max: float, cycles: int = 1,
                         x_is_zero: bool = True, schur_parity: int = -1, work=None, info=None, stream=None) -> None:
    """Chebyshev-basis CA-GCR(s) (include/coarse_op.h); same tensors as coarse_op_cagcr, work of
    coarse_op_cagcr_cheb_work_bytes(op, s) bytes."""
    for t in (b, x, work):
        if t is None or not t.is_cuda or not t.is_contiguous():
            raise ValueError("cagcr_cheb needs contiguous CUDA tensors b, x, work")
    if work.numel() * work.element_size() < coarse_op_cagcr_cheb_work_bytes(op, s):
        raise ValueError("cagcr_cheb: work buffer too small")
    if b.numel() * b.element_size() != coarse_op_vector_bytes(op, 1) or x.numel() != b.numel():
        raise ValueError("cagcr_cheb: b / x have the wrong size (1 RHS)")
    if info is not None and (info.numel() < 3 * cycles or info.element_size() != 8 or not info.is_cuda):
        raise ValueError("cagcr_cheb: info must be a CUDA float64 tensor with 3 * cycles entries")
    _check(lib().coarse_op_cagcr_cheb(op, _ptr(b), _ptr(x), int(s), int(cycles), 1 if x_is_zero else 0,
                                      float(lambda_min), float(lambda_max), int(schur_parity), _ptr(work), _ptr(info),
                                      _stream_handle(stream)))


def coarse_op_probe_read(src, stage_bytes: int = 16384, stages: int = 6, stream=None) -> int:
    """Enqueue the read-ceiling probe over the CUDA tensor `src`; returns the bytes it reads."""
    if not src.is_cuda or not src.is_contiguous():
        raise ValueError("probe_read needs a contiguous CUDA tensor")
    nbytes = src.numel() * src.element_size()
    _check(lib().coarse_op_probe_read(_ptr(src), nbytes, int(stage_bytes), int(stages), _stream_handle(stream)))
    return (nbytes // stage_bytes) * stage_bytes


def coarse_op_destroy(op: int) -> None:
    if op:
        lib().coarse_op_destroy(op)


class CoarseOp:
    """Owning convenience wrapper: keeps the borrowed link tensors alive with the handle."""

    def __init__(self, dims: Sequence[int], Nc: int, link_precision: int = LINK_C64):
        self.dims = tuple(int(d) for d in dims)
        self.Nc = int(Nc)
        self.link_precision = int(link_precision)
        self.V = self.dims[0] * self.dims[1] * self.dims[2] * self.dims[3]
        self._h = coarse_op_create(self.dims, self.Nc, self.link_precision)
        self._links = None
        self._scales = None

    def set_links(self, links, scales=None) -> "CoarseOp":
        coarse_op_set_links(self._h, links, scales)
        self._links, self._scales = links, scales
        return self

    def set_option(self, option: int, value: int) -> "CoarseOp":
        coarse_op_set_option(self._h, option, value)
        return self

    def apply(self, vin, vout, nrhs: int = 1, dagger: int = 0, stream=None) -> None:
        coarse_op_apply(self._h, vin, vout, nrhs, dagger, stream)

    def apply_static(self, vin, vout, nrhs: int = 1, dagger: int = 0, stream=None) -> None:
        coarse_op_apply_static(self._h, vin, vout, nrhs, dagger, stream)

    def apply_parts(self, u, w, vout, nrhs: int = 1, dagger: int = 0, parity: int = PARITY_ALL,
                    local: int = LOCAL_X, alpha: float = 1.0, beta: float = 1.0, stream=None) -> None:
        coarse_op_apply_parts(self._h, u, w, vout, nrhs, dagger, parity, local, alpha, beta, stream)

    def build_hat_links(self, out_links, slot0: int = HAT_SLOT0_IDENTITY, work=None, info=None, stream=None):
        """Yhat_m = X^-1 Y_m (slot 0: identity or X^-1) into out_links (complex64 [V][9][Nc][Nc])."""
        if out_links.numel() != self.V * 9 * self.Nc * self.Nc:
            raise ValueError("build_hat_links: out_links must hold V*9*Nc*Nc complex64 entries")
        return coarse_op_build_hat_links(self._h, out_links, slot0, work, info, stream)

    def apply_hvec(self, vin_q, vin_norms, vout, nrhs: int = 1, dagger: int = 0, stream=None) -> None:
        coarse_op_apply_hvec(self._h, vin_q, vin_norms, vout, nrhs, dagger, stream)

    def apply_hout(self, vin, vin_norms, vout, vout_q, vout_norms, nrhs: int = 1, dagger: int = 0, stream=None) -> None:
        coarse_op_apply_hout(self._h, vin, vin_norms, vout, vout_q, vout_norms, nrhs, dagger, stream)

    def cagcr(self, b, x, s: int = 8, cycles: int = 1, x_is_zero: bool = True, work=None, info=None, stream=None,
              schur_parity: Optional[int] = None):
        import torch
        if work is None:
            work = torch.empty(coarse_op_cagcr_work_bytes(self._h, s), dtype=torch.uint8, device=b.device)
        coarse_op_cagcr(self._h, b, x, s, cycles, x_is_zero, work, info, stream, schur_parity)
        return work

    def cagcr_cheb(self, b, x, lambda_min: float, lambda_max: float, s: int = 16, cycles: int = 1,
                   x_is_zero: bool = True, schur_parity: int = -1, work=None, info=None, stream=None):
        import torch
        if work is None:
            work = torch.empty(coarse_op_cagcr_cheb_work_bytes(self._h, s), dtype=torch.uint8, device=b.device)
        coarse_op_cagcr_cheb(self._h, b, x, s, lambda_min, lambda_max, cycles, x_is_zero, schur_parity, work, info, stream)
        return work

    def apply_host(self, vin_host, vout_host, nrhs: int = 1, dagger: int = 0, stream=None) -> None:
        coarse_op_apply_host(self._h, vin_host, vout_host, nrhs, dagger, stream)

    @property
    def last_launches(self) -> int:
        return coarse_op_last_launches(self._h)

    @property
    def last_path(self) -> int:
        return coarse_op_last_path(self._h)

    def close(self) -> None:
        if self._h:
            coarse_op_destroy(self._h)
            self._h = 0

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
