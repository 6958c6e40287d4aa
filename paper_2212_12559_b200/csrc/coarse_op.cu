// coarse_op.cu — C ABI of libcoarseop (include/coarse_op.h): argument checking, kernel selection
// and launches.  All arithmetic of the coarse-op apply lives in the kernels included below.
#include "internal.h"

#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>

#include "common.cuh"
#include "quantize_kernel.cuh"
#include "simple_kernel.cuh"
#include "stream_kernel.cuh"
#include "block_kernel.cuh"
#include "tensor_kernel.cuh"
#include "probe_kernel.cuh"
#include "cagcr_kernel.cuh"
#include "hat_kernel.cuh"

using namespace coarse;

namespace {
thread_local std::string g_last_error = "";
}

namespace coarse {

int fail(int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof(buf), fmt, ap);
    va_end(ap);
    g_last_error = buf;
    return code;
}

int cuda_fail(cudaError_t e, const char* what) {
    return fail(COARSE_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}

}  // namespace coarse

namespace {

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

bool overlaps(const void* a, size_t na, const void* b, size_t nb) {
    const uintptr_t x = reinterpret_cast<uintptr_t>(a), y = reinterpret_cast<uintptr_t>(b);
    return x < y + nb && y < x + na;
}

// The handle belongs to the device that was current in coarse_op_create: launches and allocations made
// with another device current would go to the wrong GPU with this one's pointers.
int check_device(const coarse_op* op, const char* who) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (dev != op->device)
        return fail(COARSE_EINVAL, "%s: the handle was created on device %d but device %d is current", who, op->device, dev);
    return COARSE_OK;
}

}  // namespace

namespace {

const PartsSpec kPlain = {false, nullptr, 2, 1, 1.f, 1.f, nullptr, 0, 0};

bool stream_supports(int Nc, int nrhs) {
    if (nrhs != 1) return false;
    switch (Nc) {
        case 32: case 48: case 64: case 96: case 128: case 192: return true;
        default: return false;
    }
}

bool stream_mr_supports(int Nc, int nrhs) { return stream_supports(Nc, 1) && nrhs >= 2 && nrhs <= 4; }

int launch_stream_mr(const coarse_op* op, const void* in, void* out, int nrhs, int dagger, const PartsSpec& ps, cudaStream_t stream) {
    StreamParams p = {};
    p.lat = op->lat;
    p.links = static_cast<const unsigned char*>(op->links);
    p.scales = op->scales;
    p.in = static_cast<const float2*>(in);
    p.out = static_cast<float2*>(out);
    p.keep_links = op->keep_opt == 2 || (op->keep_opt == 0 && coarse_op_link_bytes(op) <= (size_t)op->l2_bytes / 2);
    p.parity = ps.parity;
    p.n_sites = ps.parity == 2 ? op->lat.V : op->lat.V / 2;
    p.n_items = ps.site_end > 0 ? ps.site_end : 0;
    p.item_begin = ps.site_end > 0 ? ps.site_begin : 0;
    p.gen = ps.gen ? 1 : 0;                                    // parts apply: runtime flags of the multi-RHS kernel
    p.in_local = static_cast<const float2*>(ps.gen && ps.local != 0 ? ps.u : in);
    p.alpha = ps.alpha;
    p.beta = ps.beta;
    p.m_begin = ps.local == 1 ? 0 : 1;
    p.identity = ps.local == 2 ? 1 : 0;
    switch (op->Nc) {
#define COARSE_CASE_NC(NC) case NC: return COARSE_CAT(launch_stream_mr_nc, NC)(op, p, nrhs, dagger, stream);
        COARSE_FOR_EACH_NC(COARSE_CASE_NC)
#undef COARSE_CASE_NC
        default: return fail(COARSE_EUNSUPPORTED, "STREAM path is not compiled for Nc=%d", op->Nc);
    }
}

int launch_stream(const coarse_op* op, const void* in, void* out, int dagger, const PartsSpec& ps, cudaStream_t stream) {
    StreamParams p;
    p.lat = op->lat;
    p.links = static_cast<const unsigned char*>(op->links);
    p.scales = op->scales;
    p.in = static_cast<const float2*>(in);
    p.out = static_cast<float2*>(out);
    p.n_items = ps.site_end > 0 ? ps.site_end : 0;
    p.item_begin = ps.site_end > 0 ? ps.site_begin : 0;
    p.stages = 0;
    // links that fit L2 (with room for the vectors) are re-read from L2 by the next apply: keep them
    p.keep_links = op->keep_opt == 2 || (op->keep_opt == 0 && coarse_op_link_bytes(op) <= (size_t)op->l2_bytes / 2);
    p.in_local = static_cast<const float2*>(ps.gen ? ps.u : in);
    p.alpha = ps.alpha;
    p.beta = ps.beta;
    p.m_begin = ps.local == 1 ? 0 : 1;
    p.identity = ps.local == 2 ? 1 : 0;
    p.parity = ps.parity;
    p.n_sites = ps.parity == 2 ? op->lat.V : op->lat.V / 2;
    p.vnorms = ps.vnorms;
    p.hout_q = static_cast<short2*>(ps.hout_q);
    p.hout_norms = ps.hout_norms;
    // Programmatic dependent launch: always (1), never (2), or auto (0): in the latency-limited regime (links
    // resident in L2), for every launch but the first after coarse_op_set_links - work that PRODUCED the links
    // may still be in flight on the stream in front of that one, and the link stages are read before the
    // kernel orders itself against its predecessor.  Site-range launches (apply_host) never use it.
    p.pdl = (op->pdl_opt == 1 || (op->pdl_opt == 0 && !op->links_fresh && ps.site_end == 0 &&
                                  coarse_op_link_bytes(op) <= (size_t)op->l2_bytes)) ? 1 : 0;
    switch (op->Nc) {
#define COARSE_CASE_NC(NC) case NC: return COARSE_CAT(launch_stream_nc, NC)(op, p, dagger, ps.gen, stream);
        COARSE_FOR_EACH_NC(COARSE_CASE_NC)
#undef COARSE_CASE_NC
        default: return fail(COARSE_EUNSUPPORTED, "STREAM path is not compiled for Nc=%d", op->Nc);
    }
}

bool block_supports_nc(int Nc) { return stream_supports(Nc, 1); }
bool block_supports(int Nc, int nrhs) { return block_supports_nc(Nc) && nrhs >= 1 && nrhs <= 16; }

int launch_block(const coarse_op* op, const void* in, void* out, int nrhs, int dagger, cudaStream_t stream) {
    BlockParams p;
    p.lat = op->lat;
    p.links = static_cast<const unsigned char*>(op->links);
    p.scales = op->scales;
    p.in = static_cast<const float2*>(in);
    p.out = static_cast<float2*>(out);
    p.n_items = 0;
    p.stages = 0;
    p.nrhs = nrhs;
    p.keep_links = op->keep_opt == 2 || (op->keep_opt == 0 && coarse_op_link_bytes(op) <= (size_t)op->l2_bytes / 2);
    switch (op->Nc) {
#define COARSE_CASE_NC(NC) case NC: return COARSE_CAT(launch_block_nc, NC)(op, p, dagger, stream);
        COARSE_FOR_EACH_NC(COARSE_CASE_NC)
#undef COARSE_CASE_NC
        default: return fail(COARSE_EUNSUPPORTED, "BLOCK path is not compiled for Nc=%d", op->Nc);
    }
}

// TENSOR: any nrhs (groups of 16 / 8 columns, zero padded), both link formats, the parts apply included.
// Returns the number of launches beyond the first, or a negative error code.
int launch_tensor(const coarse_op* op, const void* in, void* out, int nrhs, int dagger, const PartsSpec& ps, cudaStream_t stream) {
    if (!op->link_map_ok) return fail(COARSE_EUNSUPPORTED, "TENSOR path: no tensor map for these links");
    TensorParams p = {};
    p.lat = op->lat;
    p.scales = op->scales;
    p.in = static_cast<const float2*>(in);
    p.in_local = static_cast<const float2*>(ps.gen && ps.local != 0 ? ps.u : in);
    p.out = static_cast<float2*>(out);
    p.parity = ps.parity;
    p.n_sites = ps.parity == 2 ? op->lat.V : op->lat.V / 2;
    p.site_begin = 0;
    if (ps.site_end > 0) {
        p.site_begin = ps.site_begin;
        p.n_sites = ps.site_end - ps.site_begin;
    }
    p.m_begin = ps.local == 1 ? 0 : 1;
    p.identity = ps.local == 2 ? 1 : 0;
    p.alpha = ps.alpha;
    p.beta = ps.beta;
    p.nrhs = nrhs;
    // int16 links: the integer tensor-core kernel (exact link operand, 4x fewer and 4x deeper MMAs), unless a
    // site range is launched (coarse_op_apply_host: its input arrives slice by slice, the per-site scales of
    // the fixed-point B operand need whole neighbour vectors) or the scale buffer is too small and cannot grow
    if (op->prec == COARSE_LINK_I16 && op->link_map_i8_ok && op->tensor_i8_opt != 1 && ps.site_end == 0 && op->vscale) {
        const void* u_other = (ps.gen && ps.local == 1 && ps.u != in) ? ps.u : nullptr;   // X.u needs u's scales; the identity term does not
        switch (op->Nc) {
#define COARSE_CASE_NC(NC) case NC: return COARSE_CAT(launch_tensor_i8_nc, NC)(op, p, u_other, op->vscale, dagger, stream);
            COARSE_FOR_EACH_NC(COARSE_CASE_NC)
#undef COARSE_CASE_NC
            default: return fail(COARSE_EUNSUPPORTED, "TENSOR path is not compiled for Nc=%d", op->Nc);
        }
    }
    switch (op->Nc) {
#define COARSE_CASE_NC(NC) case NC: return COARSE_CAT(launch_tensor_nc, NC)(op, p, dagger, stream);
        COARSE_FOR_EACH_NC(COARSE_CASE_NC)
#undef COARSE_CASE_NC
        default: return fail(COARSE_EUNSUPPORTED, "TENSOR path is not compiled for Nc=%d", op->Nc);
    }
}

// TENSOR on int16 links with HALF-PRECISION vectors (int16 pairs + fp32 norm per (site, rhs)): the plain apply only.
// Returns the number of launches beyond the first, or a negative error code.
bool tensor_hvec_supports(const coarse_op* op, int nrhs) {
    return op->prec == COARSE_LINK_I16 && op->link_map_i8_ok && tensor_supports(op->Nc, op->prec, nrhs);
}

int launch_tensor_hvec(const coarse_op* op, const void* in_q, const float* in_norms, void* out, int nrhs, int dagger, cudaStream_t stream) {
    TensorParams p = {};
    p.lat = op->lat;
    p.scales = op->scales;
    p.in = static_cast<const float2*>(in_q);        // int16 (re, im) pairs; the HV kernels re-type the pointer
    p.in_local = p.in;
    p.out = static_cast<float2*>(out);
    p.parity = 2;
    p.n_sites = op->lat.V;
    p.site_begin = 0;
    p.m_begin = 0;
    p.identity = 0;
    p.alpha = 1.f;
    p.beta = 1.f;
    p.nrhs = nrhs;
    switch (op->Nc) {
#define COARSE_CASE_NC(NC) case NC: return COARSE_CAT(launch_tensor_i8h_nc, NC)(op, p, in_norms, dagger, stream);
        COARSE_FOR_EACH_NC(COARSE_CASE_NC)
#undef COARSE_CASE_NC
        default: return fail(COARSE_EUNSUPPORTED, "TENSOR path is not compiled for Nc=%d", op->Nc);
    }
}

int launch_simple(const coarse_op* op, const void* in, void* out, int nrhs, int dagger, const PartsSpec& ps, cudaStream_t stream) {
    SimpleParams p;
    p.lat = op->lat;
    p.Nc = op->Nc;
    p.nrhs = nrhs;
    p.dagger = dagger;
    p.links = op->links;
    p.scales = op->scales;
    p.in = static_cast<const float2*>(in);
    p.out = static_cast<float2*>(out);
    p.in_local = static_cast<const float2*>(ps.gen ? ps.u : in);
    p.alpha = ps.alpha;
    p.beta = ps.beta;
    p.local = ps.local;
    p.parity = ps.parity;
    p.vnorms = ps.vnorms;
    const int64_t total = (int64_t)op->lat.V * op->Nc * nrhs;
    const int64_t blocks = (total + 255) / 256;
    if (blocks > 0x7fffffffLL) return fail(COARSE_EUNSUPPORTED, "SIMPLE path: problem too large");
    if (op->prec == COARSE_LINK_I16)
        coarse_apply_simple<true><<<(unsigned)blocks, 256, 0, stream>>>(p);
    else
        coarse_apply_simple<false><<<(unsigned)blocks, 256, 0, stream>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "simple kernel launch");
    return COARSE_OK;
}

// COARSE_PATH_AUTO.  1 RHS: STREAM.  2-4 RHS: STREAM-MR, except int16 links, where the integer tensor-core kernel
// (4-wide column tile, two sites per MMA tile for Nc <= 64) is faster from 2 RHS on - Nc = 48 only at 4 (measured ms,
// dagger 0 / 1, HBM-sized lattices, STREAM-MR against TENSOR: Nc = 128, 3 RHS 0.74 / 0.65 against 0.58 / 0.55; Nc = 64,
// 2 RHS 3.07 / 2.68 against 2.59 / 2.61, 3 RHS 3.26 / 3.20 against 2.66 / 2.67, 4 RHS 4.46 / 4.17 against 2.67 / 2.68;
// Nc = 48, 2 RHS 2.20 / 2.45 against 2.77 / 2.90, 3 RHS 2.57 / 2.63 against 2.79 / 2.92, 4 RHS 3.60 / 4.61 against 2.80 / 2.93;
// Nc = 32, 2 RHS 4.28 / 2.95 against 2.32 / 2.41).  5 and more: TENSOR (BLOCK only on request, or when no tensor map
// could be made), outside the compiled Nc: SIMPLE.
// Complex64 links with exactly 4 RHS in dagger = 0 also go to TENSOR for Nc >= 48: there every warp of STREAM-MR reads
// the whole 4-wide vector block of a stage with 4-way bank conflicts (stream_mr_kernel.cuh) and the kernel is bound by
// shared-memory bandwidth at twice the time of 3 RHS (measured ms, STREAM-MR against TENSOR: Nc = 192 1.10 / 0.59,
// Nc = 128 2.15 / 1.06, Nc = 96 4.33 / 2.82, Nc = 64 6.35 / 5.00, Nc = 48 4.46 / 3.86, Nc = 32 4.76 / 4.71); its
// dagger = 1 (1.03 ms at Nc = 128) stays.
int tensor_i8_min_nrhs(int Nc) { return Nc == 48 ? 4 : 2; }

int auto_path(const coarse_op* op, int nrhs, int dagger) {
    const bool tensor_ok = tensor_supports(op->Nc, op->prec, nrhs) && op->link_map_ok;
    if (stream_supports(op->Nc, nrhs)) return COARSE_PATH_STREAM;
    if (stream_mr_supports(op->Nc, nrhs)) {
        const bool i8 = op->prec == COARSE_LINK_I16 && op->link_map_i8_ok && op->vscale && op->tensor_i8_opt != 1;
        // ... on lattices that give the tensor kernel at least two work items per SM.  Below that its long per-item chain
        // (9 matrices x Nc / 32 stages) sets a floor of 15-30 us, and 2-3 right-hand sides are faster on STREAM-MR (measured
        // us, dagger 0 / 1, STREAM-MR against TENSOR, 3 RHS: the paper's level-3 volume, 32 sites Nc = 192, 16 / 36 against
        // 29 / 30; 32 sites Nc = 128 7 / 17 against 21 / 22; 256 sites Nc = 64 12 / 11 against 15 / 15; 1024 sites Nc = 64
        // 37 / 34 against 35 / 36).  4 right-hand sides stay on TENSOR (some STREAM-MR int16 instantiations spill at 4).
        const int64_t t_items = op->Nc <= 64 ? ((int64_t)op->lat.V + 1) / 2 : (int64_t)op->lat.V * (op->Nc > 128 ? 2 : 1);
        const bool tiny = nrhs <= 3 && t_items < 2 * (int64_t)op->num_sms;
        if (tensor_ok && i8 && !tiny && nrhs >= tensor_i8_min_nrhs(op->Nc)) return COARSE_PATH_TENSOR;
        if (tensor_ok && op->prec == COARSE_LINK_C64 && nrhs == 4 && dagger == 0 && op->Nc >= 48) return COARSE_PATH_TENSOR;
        return COARSE_PATH_STREAM;
    }
    if (tensor_ok) return COARSE_PATH_TENSOR;
    if (block_supports(op->Nc, nrhs)) return COARSE_PATH_BLOCK;
    return COARSE_PATH_SIMPLE;
}

int check_apply_args(const coarse_op* op, const void* in, const void* out, int nrhs, int dagger) {
    if (!op) return fail(COARSE_EINVAL, "apply: op is NULL");
    if (!op->links) return fail(COARSE_ENOTREADY, "apply: coarse_op_set_links has not been called");
    if (!in || !out) return fail(COARSE_EINVAL, "apply: in/out is NULL");
    if (nrhs < 1) return fail(COARSE_EINVAL, "apply: nrhs must be >= 1 (got %d)", nrhs);
    if (dagger != 0 && dagger != 1) return fail(COARSE_EINVAL, "apply: dagger must be 0 or 1 (got %d)", dagger);
    return check_device(op, "apply");
}

}  // namespace

extern "C" {

coarse_op_t* coarse_op_create(const int dims[4], int Nc, int link_precision) {
    if (!dims) { fail(COARSE_EINVAL, "create: dims is NULL"); return nullptr; }
    int64_t V = 1;
    for (int mu = 0; mu < 4; ++mu) {
        if (dims[mu] < 1) { fail(COARSE_EINVAL, "create: dims[%d] = %d must be >= 1", mu, dims[mu]); return nullptr; }
        V *= dims[mu];
        if (V > 0x7fffffffLL) { fail(COARSE_EINVAL, "create: lattice volume exceeds 2^31-1 sites"); return nullptr; }
    }
    if (Nc < 2 || (Nc & 1)) { fail(COARSE_EINVAL, "create: Nc = %d must be even and >= 2", Nc); return nullptr; }
    if (link_precision != COARSE_LINK_C64 && link_precision != COARSE_LINK_I16) {
        fail(COARSE_EINVAL, "create: unknown link_precision %d", link_precision);
        return nullptr;
    }
    int dev = 0, count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess || count < 1) {
        cudaGetLastError();
        fail(COARSE_ECUDA, "create: no CUDA device (libcoarseop has no CPU fallback)");
        return nullptr;
    }
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) { cuda_fail(e, "cudaGetDevice"); return nullptr; }
    int major = 0, sms = 0, smem = 0;
    cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (major != 10) {
        fail(COARSE_ECUDA, "create: device %d has compute capability %d.x; this library is built for sm_100a only", dev, major);
        return nullptr;
    }
    coarse_op* op = new (std::nothrow) coarse_op();
    if (!op) { fail(COARSE_ENOMEM, "create: out of host memory"); return nullptr; }
    for (int mu = 0; mu < 4; ++mu) op->lat.L[mu] = dims[mu];
    op->lat.V = (int)V;
    op->Nc = Nc;
    op->prec = link_precision;
    op->links = nullptr;
    op->scales = nullptr;
    op->path_opt = COARSE_PATH_AUTO;
    op->grid_opt = 0;
    op->stages_opt = 0;
    op->fine_opt = 0;
    op->keep_opt = 0;
    op->pdl_opt = 0;
    op->links_fresh = true;
    op->split_opt = 0;
    op->warp_items_opt = 0;
    op->split_ws = nullptr;
    op->split_count = nullptr;
    op->split_ws_bytes = 0;
    { int l2 = 0; cudaDeviceGetAttribute(&l2, cudaDevAttrL2CacheSize, dev); op->l2_bytes = l2; }
    op->last_launches = 0;
    op->last_path = 0;
    op->device = dev;
    op->num_sms = sms;
    op->max_smem = smem;
    op->stage_in = op->stage_out = nullptr;
    op->stage_bytes = 0;
    op->s_h2d = op->s_d2h = nullptr;
    op->host_pipe_ok = false;
    op->link_map_ok = false;
    op->link_map_i8_ok = false;
    op->vscale = nullptr;
    op->tensor_i8_opt = 0;
    g_last_error = "";
    return op;
}

size_t coarse_op_link_bytes(const coarse_op_t* op) {
    if (!op) return 0;
    return (size_t)op->lat.V * 9 * op->Nc * op->Nc * (op->prec == COARSE_LINK_I16 ? 4 : 8);
}

size_t coarse_op_scale_bytes(const coarse_op_t* op) {
    if (!op || op->prec != COARSE_LINK_I16) return 0;
    return (size_t)op->lat.V * 9 * 4;
}

size_t coarse_op_vector_bytes(const coarse_op_t* op, int nrhs) {
    if (!op || nrhs < 1) return 0;
    return (size_t)op->lat.V * op->Nc * nrhs * 8;
}

int coarse_op_set_links(coarse_op_t* op, const void* links_dev, const float* scales_dev) {
    if (!op) return fail(COARSE_EINVAL, "set_links: op is NULL");
    if (!links_dev) return fail(COARSE_EINVAL, "set_links: links_dev is NULL");
    if (!aligned16(links_dev)) return fail(COARSE_EINVAL, "set_links: links_dev must be 16-byte aligned");
    { int rc = check_device(op, "set_links"); if (rc != COARSE_OK) return rc; }
    if (op->prec == COARSE_LINK_I16) {
        if (!scales_dev) return fail(COARSE_EINVAL, "set_links: I16 links need scales_dev");
        if ((reinterpret_cast<uintptr_t>(scales_dev) & 3u) != 0)
            return fail(COARSE_EINVAL, "set_links: scales_dev must be 4-byte aligned");
    } else if (scales_dev) {
        return fail(COARSE_EINVAL, "set_links: scales_dev must be NULL for C64 links");
    }
    op->links = links_dev;
    op->scales = scales_dev;
    op->links_fresh = true;
    // tiny lattices (fewer sites than SMs): workspace for the split dagger apply, V * (Nc/8) chunks * Nc
    // complex numbers at most (a few MB); the only allocation the library makes besides apply_host's staging
    if (!op->split_ws && op->lat.V < op->num_sms && stream_supports(op->Nc, 1)) {
        const size_t bytes = (size_t)op->lat.V * (op->Nc / 8) * op->Nc * 8;
        const size_t cbytes = (size_t)op->lat.V * sizeof(unsigned int);
        if (cudaMalloc(reinterpret_cast<void**>(&op->split_ws), bytes + cbytes) == cudaSuccess) {
            op->split_count = reinterpret_cast<unsigned int*>(reinterpret_cast<unsigned char*>(op->split_ws) + bytes);
            // the counters start at zero and every launch leaves them at zero; the clear is complete before any
            // stream can use them (one synchronisation per handle, at set-up time)
            if (cudaMemset(op->split_count, 0, cbytes) == cudaSuccess && cudaDeviceSynchronize() == cudaSuccess) {
                op->split_ws_bytes = bytes;
            } else {
                cudaGetLastError();
                cudaFree(op->split_ws);
                op->split_ws = nullptr;
                op->split_count = nullptr;
            }
        } else {
            cudaGetLastError();
            op->split_ws = nullptr;
            op->split_ws_bytes = 0;
        }
    }
    {
        const int rc = make_link_maps(op);
        if (rc != COARSE_OK) return rc;
    }
    // int16 links: scale buffer of the integer tensor-core kernel, (g, 1/g) per (site, column) for two operands and
    // the 16 columns of one launch (V x 256 bytes); without it multi-RHS applies run on the 3xTF32 kernel
    if (op->prec == COARSE_LINK_I16 && op->link_map_i8_ok && !op->vscale) {
        if (cudaMalloc(reinterpret_cast<void**>(&op->vscale), (size_t)2 * 2 * op->lat.V * 16 * sizeof(float)) != cudaSuccess) {
            cudaGetLastError();
            op->vscale = nullptr;
        }
    }
    return COARSE_OK;
}

int coarse_op_set_option(coarse_op_t* op, int option, int value) {
    if (!op) return fail(COARSE_EINVAL, "set_option: op is NULL");
    switch (option) {
        case COARSE_OPT_PATH:
            if (value == COARSE_PATH_AUTO || value == COARSE_PATH_SIMPLE) { op->path_opt = value; return COARSE_OK; }
            if (value == COARSE_PATH_STREAM) {
                if (!stream_supports(op->Nc, 1))
                    return fail(COARSE_EUNSUPPORTED, "set_option: STREAM path is not compiled for Nc=%d", op->Nc);
                op->path_opt = value;
                return COARSE_OK;
            }
            if (value == COARSE_PATH_BLOCK) {
                if (!block_supports_nc(op->Nc))
                    return fail(COARSE_EUNSUPPORTED, "set_option: BLOCK path is not compiled for Nc=%d", op->Nc);
                op->path_opt = value;
                return COARSE_OK;
            }
            if (value == COARSE_PATH_TENSOR) {
                if (!tensor_supports_nc(op->Nc, op->prec))
                    return fail(COARSE_EUNSUPPORTED, "set_option: TENSOR path is compiled for Nc in {32,48,64,96,128,192} (got Nc=%d)", op->Nc);
                op->path_opt = value;
                return COARSE_OK;
            }
            return fail(COARSE_EINVAL, "set_option: unknown path %d", value);
        case COARSE_OPT_GRID:
            if (value < 0) return fail(COARSE_EINVAL, "set_option: grid must be >= 0");
            op->grid_opt = value;
            return COARSE_OK;
        case COARSE_OPT_FINE:
            if (value < 0 || value > 2) return fail(COARSE_EINVAL, "set_option: fine must be 0 (auto), 1 (never) or 2 (always)");
            op->fine_opt = value;
            return COARSE_OK;
        case COARSE_OPT_KEEP_LINKS:
            if (value < 0 || value > 2) return fail(COARSE_EINVAL, "set_option: keep_links must be 0 (auto), 1 (never) or 2 (always)");
            op->keep_opt = value;
            return COARSE_OK;
        case COARSE_OPT_SPLIT_DAGGER:
            if (value < 0 || value > 3) return fail(COARSE_EINVAL, "set_option: split_dagger must be 0 (auto), 1 (never), 2 (always) or 3 (always, workspace scheme)");
            op->split_opt = value;
            return COARSE_OK;
        case COARSE_OPT_TENSOR_I8:
            if (value < 0 || value > 2) return fail(COARSE_EINVAL, "set_option: tensor_i8 must be 0 (auto), 1 (never) or 2 (always)");
            op->tensor_i8_opt = value;
            return COARSE_OK;
        case COARSE_OPT_WARP_ITEMS:
            if (!(value >= 0 && value <= 2) && value != 12 && value != 14)
                return fail(COARSE_EINVAL, "set_option: warp_items must be 0 (auto), 1 (never), 2 (always) or 12 / 14 (always, 2 / 4 warps per team)");
            op->warp_items_opt = value;
            return COARSE_OK;
        case COARSE_OPT_PDL:
            if (value < 0 || value > 2) return fail(COARSE_EINVAL, "set_option: pdl must be 0 (auto), 1 (always) or 2 (never)");
            op->pdl_opt = value;
            return COARSE_OK;
        case COARSE_OPT_STAGES:
            if (value < 0 || value == 1) return fail(COARSE_EINVAL, "set_option: stages must be 0 (default) or >= 2");
            op->stages_opt = value;
            return COARSE_OK;
        default:
            return fail(COARSE_EINVAL, "set_option: unknown option %d", option);
    }
}

int coarse_op_apply(coarse_op_t* op, const void* in_dev, void* out_dev, int nrhs, int dagger, void* stream) {
    int rc = check_apply_args(op, in_dev, out_dev, nrhs, dagger);
    if (rc != COARSE_OK) return rc;
    if (!aligned16(in_dev) || !aligned16(out_dev))
        return fail(COARSE_EINVAL, "apply: in_dev/out_dev must be 16-byte aligned");
    const size_t vb = coarse_op_vector_bytes(op, nrhs);
    const uintptr_t a = reinterpret_cast<uintptr_t>(in_dev), b = reinterpret_cast<uintptr_t>(out_dev);
    if (a < b + vb && b < a + vb) return fail(COARSE_EINVAL, "apply: in and out overlap (the stencil reads neighbours)");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    int path = op->path_opt;
    if (path == COARSE_PATH_AUTO) path = auto_path(op, nrhs, dagger);
    op->last_launches = 0;
    if (path == COARSE_PATH_TENSOR) {
        if (!tensor_supports(op->Nc, op->prec, nrhs))
            return fail(COARSE_EUNSUPPORTED, "apply: TENSOR path is not compiled for Nc=%d", op->Nc);
        rc = launch_tensor(op, in_dev, out_dev, nrhs, dagger, kPlain, st);
    } else if (path == COARSE_PATH_BLOCK) {
        if (!block_supports(op->Nc, nrhs))
            return fail(COARSE_EUNSUPPORTED, "apply: BLOCK path covers nrhs <= 16 (got Nc=%d nrhs=%d)", op->Nc, nrhs);
        rc = launch_block(op, in_dev, out_dev, nrhs, dagger, st);
    } else if (path == COARSE_PATH_STREAM) {
        if (stream_mr_supports(op->Nc, nrhs))
            rc = launch_stream_mr(op, in_dev, out_dev, nrhs, dagger, kPlain, st);
        else if (!stream_supports(op->Nc, nrhs))
            return fail(COARSE_EUNSUPPORTED, "apply: STREAM path covers nrhs <= 4 (got Nc=%d nrhs=%d)", op->Nc, nrhs);
        else
            rc = launch_stream(op, in_dev, out_dev, dagger, kPlain, st);
    } else {
        rc = launch_simple(op, in_dev, out_dev, nrhs, dagger, kPlain, st);
    }
    if (rc < 0) return rc;
    op->last_launches = 1 + rc;      // the split dagger apply reports its second (reduce) launch as rc = 1
    op->last_path = path;
    op->links_fresh = false;
    return COARSE_OK;
}

int coarse_op_apply_parts(coarse_op_t* op, const void* u_dev, const void* w_dev, void* out_dev, int nrhs,
                          int dagger, int parity, int local, float alpha, float beta, void* stream) {
    int rc = check_apply_args(op, w_dev, out_dev, nrhs, dagger);
    if (rc != COARSE_OK) return rc;
    if (parity < 0 || parity > 2) return fail(COARSE_EINVAL, "apply_parts: parity must be 0 (even), 1 (odd) or 2 (all), got %d", parity);
    if (local < 0 || local > 2) return fail(COARSE_EINVAL, "apply_parts: local must be 0 (none), 1 (X) or 2 (identity), got %d", local);
    if (local != 0 && !u_dev) return fail(COARSE_EINVAL, "apply_parts: u_dev is NULL but a local term was requested");
    if (parity != 2)
        for (int mu = 0; mu < 4; ++mu)
            if (op->lat.L[mu] & 1)
                return fail(COARSE_EINVAL, "apply_parts: the even/odd decomposition needs even extents (dims[%d] = %d)", mu, op->lat.L[mu]);
    if (!aligned16(w_dev) || !aligned16(out_dev) || (u_dev && !aligned16(u_dev)))
        return fail(COARSE_EINVAL, "apply_parts: device vectors must be 16-byte aligned");
    const size_t vb = coarse_op_vector_bytes(op, nrhs);
    const uintptr_t b = reinterpret_cast<uintptr_t>(out_dev);
    const uintptr_t a = reinterpret_cast<uintptr_t>(w_dev);
    // w is read at neighbours: it may share a buffer with out only when the two parities are disjoint,
    // which the caller cannot express here, so overlap is always refused.
    if (a < b + vb && b < a + vb) return fail(COARSE_EINVAL, "apply_parts: w and out overlap (the stencil reads neighbours)");
    // u: with the identity local term every output element reads exactly its own u element first, so
    // u == out (in place) is safe; a shifted overlap is not.  With LOCAL_X the whole vector u(x) is read by
    // work items that run concurrently with the writers of out(x): any overlap is refused.
    if (local != COARSE_LOCAL_NONE && overlaps(u_dev, vb, out_dev, vb)) {
        if (local == COARSE_LOCAL_X)
            return fail(COARSE_EINVAL, "apply_parts: u and out overlap with COARSE_LOCAL_X (X.u reads all of u(x) while out(x) is written)");
        if (u_dev != out_dev)
            return fail(COARSE_EINVAL, "apply_parts: u and out overlap partially (only u == out is allowed, with COARSE_LOCAL_IDENTITY)");
    }
    PartsSpec ps = {true, local != 0 ? u_dev : w_dev, parity, local, alpha, beta, nullptr, 0, 0};
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // 1 RHS: STREAM (GEN instantiations); 2-4: STREAM-MR (runtime flags), except int16 links with Nc >= 96; more: the
    // TENSOR kernels (parity list, alpha / beta folded into the B operand, identity term in the epilogue); shapes none of
    // them covers: SIMPLE.
    int path = op->path_opt;
    const bool tensor_ok = tensor_supports(op->Nc, op->prec, nrhs) && op->link_map_ok;
    const bool stream_ok = stream_supports(op->Nc, nrhs) || stream_mr_supports(op->Nc, nrhs);
    if (path == COARSE_PATH_AUTO || path == COARSE_PATH_BLOCK) {
        path = auto_path(op, nrhs, dagger);                                     // the plain apply's rule; BLOCK has no parts variant
        if (path == COARSE_PATH_BLOCK) path = COARSE_PATH_SIMPLE;
    } else if ((path == COARSE_PATH_STREAM && !stream_ok) || (path == COARSE_PATH_TENSOR && !tensor_ok)) {
        path = stream_ok ? COARSE_PATH_STREAM : tensor_ok ? COARSE_PATH_TENSOR : COARSE_PATH_SIMPLE;
    }
    op->last_launches = 0;
    if (path == COARSE_PATH_STREAM) {
        rc = nrhs == 1 ? launch_stream(op, w_dev, out_dev, dagger, ps, st) : launch_stream_mr(op, w_dev, out_dev, nrhs, dagger, ps, st);
    } else if (path == COARSE_PATH_TENSOR) {
        rc = launch_tensor(op, w_dev, out_dev, nrhs, dagger, ps, st);
    } else {
        rc = launch_simple(op, w_dev, out_dev, nrhs, dagger, ps, st);
    }
    if (rc < 0) return rc;
    op->last_launches = 1 + rc;
    op->last_path = path;
    op->links_fresh = false;
    return COARSE_OK;
}

int coarse_op_apply_hvec(coarse_op_t* op, const void* in_q_dev, const float* in_norms_dev, void* out_dev, int nrhs,
                         int dagger, void* stream) {
    int rc = check_apply_args(op, in_q_dev, out_dev, nrhs, dagger);
    if (rc != COARSE_OK) return rc;
    if (!in_norms_dev) return fail(COARSE_EINVAL, "apply_hvec: in_norms_dev is NULL");
    if (!aligned16(in_q_dev) || !aligned16(out_dev) || (reinterpret_cast<uintptr_t>(in_norms_dev) & 3u))
        return fail(COARSE_EINVAL, "apply_hvec: in_q_dev/out_dev must be 16-byte aligned, in_norms_dev 4-byte aligned");
    if (op->Nc % 4) return fail(COARSE_EUNSUPPORTED, "apply_hvec: Nc must be a multiple of 4 (got %d)", op->Nc);
    const size_t vb = coarse_op_vector_bytes(op, nrhs);
    const uintptr_t a = reinterpret_cast<uintptr_t>(in_q_dev), b = reinterpret_cast<uintptr_t>(out_dev);
    if (a < b + vb && b < a + vb / 2) return fail(COARSE_EINVAL, "apply_hvec: in and out overlap");
    PartsSpec ps = kPlain;
    ps.vnorms = in_norms_dev;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    // 1 RHS: STREAM (the norm folded into the vector operand); several right-hand sides on int16 links: the integer
    // tensor-core kernel, both operands exact int8 planes (tensor_i8_kernel.cuh, HV); otherwise SIMPLE
    int path = op->path_opt;
    if (path == COARSE_PATH_TENSOR && !tensor_hvec_supports(op, nrhs)) path = COARSE_PATH_AUTO;
    if (path == COARSE_PATH_AUTO || path == COARSE_PATH_BLOCK)
        path = stream_supports(op->Nc, nrhs) ? COARSE_PATH_STREAM : tensor_hvec_supports(op, nrhs) ? COARSE_PATH_TENSOR : COARSE_PATH_SIMPLE;
    op->last_launches = 0;
    if (path == COARSE_PATH_TENSOR) {
        rc = launch_tensor_hvec(op, in_q_dev, in_norms_dev, out_dev, nrhs, dagger, st);
        if (rc < 0) return rc;
        op->last_launches = 1 + rc;
        op->last_path = path;
        op->links_fresh = false;
        return COARSE_OK;
    }
    if (path == COARSE_PATH_STREAM) {
        if (!stream_supports(op->Nc, nrhs))
            return fail(COARSE_EUNSUPPORTED, "apply_hvec: STREAM path does not cover Nc=%d nrhs=%d", op->Nc, nrhs);
        rc = launch_stream(op, in_q_dev, out_dev, dagger, ps, st);
    } else {
        rc = launch_simple(op, in_q_dev, out_dev, nrhs, dagger, ps, st);
    }
    if (rc != COARSE_OK) return rc;
    op->last_launches = 1;
    op->last_path = path;
    op->links_fresh = false;
    return COARSE_OK;
}

int coarse_op_apply_hout(coarse_op_t* op, const void* in_dev, const float* in_norms_dev, void* out_c64_dev, void* out_q_dev,
                         float* out_norms_dev, int nrhs, int dagger, void* stream) {
    int rc = check_apply_args(op, in_dev, out_c64_dev, nrhs, dagger);
    if (rc != COARSE_OK) return rc;
    if (!out_q_dev || !out_norms_dev) return fail(COARSE_EINVAL, "apply_hout: out_q_dev / out_norms_dev is NULL");
    if (!aligned16(in_dev) || !aligned16(out_c64_dev) || !aligned16(out_q_dev) || (reinterpret_cast<uintptr_t>(out_norms_dev) & 3u) ||
        (in_norms_dev && (reinterpret_cast<uintptr_t>(in_norms_dev) & 3u)))
        return fail(COARSE_EINVAL, "apply_hout: vectors must be 16-byte aligned, norm arrays 4-byte aligned");
    const size_t vb = coarse_op_vector_bytes(op, nrhs);
    const size_t in_b = in_norms_dev ? vb / 2 : vb;
    if (overlaps(in_dev, in_b, out_c64_dev, vb) || overlaps(in_dev, in_b, out_q_dev, vb / 2) || overlaps(out_c64_dev, vb, out_q_dev, vb / 2))
        return fail(COARSE_EINVAL, "apply_hout: in, out_c64 and out_q must not overlap");
    if (in_norms_dev && op->Nc % 4) return fail(COARSE_EUNSUPPORTED, "apply_hout: half-precision input needs Nc % 4 == 0 (got %d)", op->Nc);
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const bool fused = nrhs == 1 && stream_supports(op->Nc, 1) &&
                       (op->path_opt == COARSE_PATH_AUTO || op->path_opt == COARSE_PATH_STREAM);
    if (fused) {
        PartsSpec ps = kPlain;
        ps.vnorms = in_norms_dev;
        ps.hout_q = out_q_dev;
        ps.hout_norms = out_norms_dev;
        op->last_launches = 0;
        rc = launch_stream(op, in_dev, out_c64_dev, dagger, ps, st);
        if (rc < 0) return rc;
        op->last_launches = 1 + rc;
        op->last_path = COARSE_PATH_STREAM;
        op->links_fresh = false;
        return COARSE_OK;
    }
    // several right-hand sides, or a shape outside the STREAM kernels: the apply, then the vector quantiser
    rc = in_norms_dev ? coarse_op_apply_hvec(op, in_dev, in_norms_dev, out_c64_dev, nrhs, dagger, stream)
                      : coarse_op_apply(op, in_dev, out_c64_dev, nrhs, dagger, stream);
    if (rc != COARSE_OK) return rc;
    const int launches = op->last_launches;
    rc = coarse_op_quantize_vec_i16(out_c64_dev, op->lat.V, op->Nc, nrhs, out_q_dev, out_norms_dev, stream);
    if (rc != COARSE_OK) return rc;
    op->last_launches = launches + 1;
    return COARSE_OK;
}

int coarse_op_quantize_vec_i16(const void* v_c64_dev, int64_t n_sites, int Nc, int nrhs, void* q_dev,
                               float* norms_dev, void* stream) {
    if (!v_c64_dev || !q_dev || !norms_dev) return fail(COARSE_EINVAL, "quantize_vec_i16: NULL pointer");
    if (n_sites < 0 || Nc < 1 || nrhs < 1) return fail(COARSE_EINVAL, "quantize_vec_i16: bad sizes");
    if (n_sites == 0) return COARSE_OK;
    const int64_t total = n_sites * nrhs;
    const int64_t blocks = (total + 127) / 128;
    if (blocks > 0x7fffffffLL) return fail(COARSE_EINVAL, "quantize_vec_i16: too many vectors");
    quantize_vec_i16_kernel<<<(unsigned)blocks, 128, 0, static_cast<cudaStream_t>(stream)>>>(
        static_cast<const float2*>(v_c64_dev), (long long)n_sites, Nc, nrhs, static_cast<short2*>(q_dev), norms_dev);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "vector quantize kernel launch");
    return COARSE_OK;
}

int coarse_op_apply_host(coarse_op_t* op, const void* in_host, void* out_host, int nrhs, int dagger, void* stream) {
    int rc = check_apply_args(op, in_host, out_host, nrhs, dagger);
    if (rc != COARSE_OK) return rc;
    const size_t vb = coarse_op_vector_bytes(op, nrhs);
    if (op->stage_bytes < vb) {
        if (op->stage_in) cudaFree(op->stage_in);
        if (op->stage_out) cudaFree(op->stage_out);
        op->stage_in = op->stage_out = nullptr;
        op->stage_bytes = 0;
        cudaError_t e = cudaMalloc(&op->stage_in, vb);
        if (e == cudaSuccess) e = cudaMalloc(&op->stage_out, vb);
        if (e != cudaSuccess) {
            cudaGetLastError();
            if (op->stage_in) cudaFree(op->stage_in);
            op->stage_in = nullptr;
            return fail(COARSE_ENOMEM, "apply_host: cannot allocate %zu-byte staging buffers", vb);
        }
        op->stage_bytes = vb;
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    cudaError_t e;
    // Pipelined path (STREAM kernels for 1-4 RHS, TENSOR kernel beyond; at least 8 time slices): the lattice is cut into 4 (or 8) ranges
    // of x3-slices; range c is launched as soon as the slices it reads (its own and one on either side)
    // are on the device, and its result goes back to the host while the next range computes.  H2D, the
    // kernels and D2H run on three streams; nothing is reordered inside a range, so the result is
    // bit-identical to the plain path.
    const int T = op->lat.L[3];
    // the family coarse_op_apply would pick; STREAM (1-4 RHS) and TENSOR launch site ranges
    int hpath = op->path_opt;
    if (hpath == COARSE_PATH_AUTO) hpath = auto_path(op, nrhs, dagger);
    const bool ranged = (hpath == COARSE_PATH_STREAM && (stream_supports(op->Nc, nrhs) || stream_mr_supports(op->Nc, nrhs))) ||
                        (hpath == COARSE_PATH_TENSOR && tensor_supports(op->Nc, op->prec, nrhs) && op->link_map_ok);
    if (ranged && T >= 8 && vb >= ((size_t)1 << 22)) {
        if (!op->host_pipe_ok) {
            // create the two copy streams and nine events; on a partial failure destroy what exists
            cudaStream_t ss[2] = {nullptr, nullptr};
            cudaEvent_t ev[17] = {};
            bool ok = true;
            for (int i = 0; ok && i < 2; ++i) ok = cudaStreamCreateWithFlags(&ss[i], cudaStreamNonBlocking) == cudaSuccess;
            for (int i = 0; ok && i < 17; ++i) ok = cudaEventCreateWithFlags(&ev[i], cudaEventDisableTiming) == cudaSuccess;
            if (!ok) {
                cudaGetLastError();
                for (int i = 0; i < 17; ++i) if (ev[i]) cudaEventDestroy(ev[i]);
                for (int i = 0; i < 2; ++i) if (ss[i]) cudaStreamDestroy(ss[i]);
                return fail(COARSE_ECUDA, "apply_host: cannot create copy streams/events");
            }
            op->s_h2d = ss[0];
            op->s_d2h = ss[1];
            for (int i = 0; i < 8; ++i) { op->ev_up[i] = ev[i]; op->ev_k[i] = ev[8 + i]; }
            op->ev_done = ev[16];
            op->host_pipe_ok = true;
        }
        const size_t plane = (size_t)(op->lat.V / T);               // sites per x3-slice
        const size_t pb = plane * op->Nc * nrhs * 8;                 // bytes per slice
        const unsigned char* hin = static_cast<const unsigned char*>(in_host);
        unsigned char* hout = static_cast<unsigned char*>(out_host);
        unsigned char* din = static_cast<unsigned char*>(op->stage_in);
        unsigned char* dout = static_cast<unsigned char*>(op->stage_out);
        // Once a copy is queued the host buffers are in use by the device: every exit, error or not,
        // first drains the three streams (the header promises the call has synchronised when it returns).
        auto drain = [&]() {
            cudaStreamSynchronize(op->s_h2d);
            cudaStreamSynchronize(st);
            cudaStreamSynchronize(op->s_d2h);
        };
        auto bail_cuda = [&](cudaError_t err, const char* what) { drain(); cudaGetLastError(); return cuda_fail(err, what); };
        // the copy streams start after whatever the caller's stream has queued
        if ((e = cudaEventRecord(op->ev_done, st)) != cudaSuccess) return cuda_fail(e, "apply_host: event record");
        if ((e = cudaStreamWaitEvent(op->s_h2d, op->ev_done, 0)) != cudaSuccess) return cuda_fail(e, "apply_host: stream wait");
        if ((e = cudaStreamWaitEvent(op->s_d2h, op->ev_done, 0)) != cudaSuccess) return cuda_fail(e, "apply_host: stream wait");
        // slice T-1 first (range 0 reads it through the periodic wrap), then slices in order
        if ((e = cudaMemcpyAsync(din + (size_t)(T - 1) * pb, hin + (size_t)(T - 1) * pb, pb, cudaMemcpyHostToDevice, op->s_h2d)) != cudaSuccess)
            return bail_cuda(e, "apply_host: H2D copy");
        int uploaded = 0;                                            // slices [0, uploaded) are queued
        PartsSpec ps = kPlain;
        op->last_launches = 0;
        // 4 ranges; 8 when the copies dominate (vectors of 32 MiB and more: several right-hand sides), so that less of the
        // first upload and the last download is exposed
        const int NR = (vb >= ((size_t)1 << 25) && T >= 8) ? 8 : 4;
        for (int c = 0; c < NR; ++c) {
            const int t0 = (int)((long long)T * c / NR), t1 = (int)((long long)T * (c + 1) / NR);
            int need = t1 + 1 < T - 1 ? t1 + 1 : T - 1;              // slices [0, need) plus slice T-1
            if (need > uploaded) {
                e = cudaMemcpyAsync(din + (size_t)uploaded * pb, hin + (size_t)uploaded * pb, (size_t)(need - uploaded) * pb,
                                    cudaMemcpyHostToDevice, op->s_h2d);
                if (e != cudaSuccess) return bail_cuda(e, "apply_host: H2D copy");
                uploaded = need;
            }
            if ((e = cudaEventRecord(op->ev_up[c], op->s_h2d)) != cudaSuccess) return bail_cuda(e, "apply_host: event record");
            if ((e = cudaStreamWaitEvent(st, op->ev_up[c], 0)) != cudaSuccess) return bail_cuda(e, "apply_host: stream wait");
            ps.site_begin = (int)(plane * t0);
            ps.site_end = (int)(plane * t1);
            if (hpath == COARSE_PATH_TENSOR) rc = launch_tensor(op, op->stage_in, op->stage_out, nrhs, dagger, ps, st);
            else if (nrhs == 1) rc = launch_stream(op, op->stage_in, op->stage_out, dagger, ps, st);
            else rc = launch_stream_mr(op, op->stage_in, op->stage_out, nrhs, dagger, ps, st);
            if (rc < 0) { drain(); return rc; }
            op->last_launches += 1 + rc;
            if ((e = cudaEventRecord(op->ev_k[c], st)) != cudaSuccess) return bail_cuda(e, "apply_host: event record");
            if ((e = cudaStreamWaitEvent(op->s_d2h, op->ev_k[c], 0)) != cudaSuccess) return bail_cuda(e, "apply_host: stream wait");
            e = cudaMemcpyAsync(hout + (size_t)t0 * pb, dout + (size_t)t0 * pb, (size_t)(t1 - t0) * pb, cudaMemcpyDeviceToHost, op->s_d2h);
            if (e != cudaSuccess) return bail_cuda(e, "apply_host: D2H copy");
        }
        op->last_path = hpath;
        op->links_fresh = false;
        if ((e = cudaEventRecord(op->ev_done, op->s_d2h)) != cudaSuccess) return bail_cuda(e, "apply_host: event record");
        if ((e = cudaStreamWaitEvent(st, op->ev_done, 0)) != cudaSuccess) return bail_cuda(e, "apply_host: stream wait");
        e = cudaStreamSynchronize(st);
        if (e != cudaSuccess) return cuda_fail(e, "apply_host: stream synchronize");
        return COARSE_OK;
    }
    e = cudaMemcpyAsync(op->stage_in, in_host, vb, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e, "apply_host: H2D copy");
    rc = coarse_op_apply(op, op->stage_in, op->stage_out, nrhs, dagger, stream);
    if (rc != COARSE_OK) { cudaStreamSynchronize(st); return rc; }      // the H2D copy reads in_host until then
    e = cudaMemcpyAsync(out_host, op->stage_out, vb, cudaMemcpyDeviceToHost, st);
    if (e != cudaSuccess) { cudaStreamSynchronize(st); cudaGetLastError(); return cuda_fail(e, "apply_host: D2H copy"); }
    e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(e, "apply_host: stream synchronize");
    return COARSE_OK;
}

int coarse_op_last_launches(const coarse_op_t* op) { return op ? op->last_launches : 0; }
int coarse_op_last_path(const coarse_op_t* op) { return op ? op->last_path : 0; }

int coarse_op_quantize_i16(const void* links_c64_dev, int64_t n_matrices, int Nc, void* q_dev, float* scales_dev,
                           void* stream) {
    if (!links_c64_dev || !q_dev || !scales_dev) return fail(COARSE_EINVAL, "quantize_i16: NULL pointer");
    if (n_matrices < 0 || Nc < 1) return fail(COARSE_EINVAL, "quantize_i16: bad sizes");
    if (n_matrices == 0) return COARSE_OK;
    if ((int64_t)2 * Nc * Nc > 0x7fffffffLL) return fail(COARSE_EINVAL, "quantize_i16: Nc too large");
    const unsigned grid = (unsigned)(n_matrices < 148 * 16 ? n_matrices : 148 * 16);
    quantize_i16_kernel<<<grid, 256, 0, static_cast<cudaStream_t>(stream)>>>(
        static_cast<const float*>(links_c64_dev), n_matrices, Nc, static_cast<short*>(q_dev), scales_dev);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "quantize kernel launch");
    return COARSE_OK;
}

size_t coarse_op_cagcr_work_bytes(const coarse_op_t* op, int s) { return coarse_op_cagcr_cheb_work_bytes(op, s); }

// CA-GCR(s) on the Chebyshev basis (cagcr_kernel.cuh): P_k = T_k((A - c)/d) r0, T_k = A P_k kept as separate
// vectors.  Slots: P_0..P_{s-1} | T_0..T_{s-1} | R (the update's output, swapped with P_0 every cycle).
// lambda_min = lambda_max = 0: the interval is estimated on the device in the first cycle.
// schur_parity < 0: the operator is A (coarse_op_apply).  schur_parity = 0 | 1: the operator is the
// left-preconditioned Schur operator on that parity, Shat_p v = v - Dhat_pq Dhat_qp v, two
// parity-restricted launches on this handle's (block-preconditioned) links.
static int cagcr_cheb_impl(coarse_op_t* op, const void* b_dev, void* x_dev, int s, int cycles, int x_is_zero,
                           float lambda_min, float lambda_max, int schur_parity, void* work_dev, double* info_dev,
                           void* stream) {
    if (!op) return fail(COARSE_EINVAL, "cagcr_cheb: op is NULL");
    if (!op->links) return fail(COARSE_ENOTREADY, "cagcr_cheb: coarse_op_set_links has not been called");
    if (!b_dev || !x_dev || !work_dev) return fail(COARSE_EINVAL, "cagcr_cheb: NULL pointer");
    if (s < 1 || s > CAGCR_MAX_S) return fail(COARSE_EINVAL, "cagcr_cheb: 1 <= s <= %d (got %d)", CAGCR_MAX_S, s);
    if (cycles < 1) return fail(COARSE_EINVAL, "cagcr_cheb: cycles must be >= 1");
    const bool auto_interval = lambda_min == 0.f && lambda_max == 0.f;
    if (!auto_interval && !(lambda_max > lambda_min))
        return fail(COARSE_EINVAL, "cagcr_cheb: need lambda_max > lambda_min (or both 0: estimate the interval)");
    if (!aligned16(b_dev) || !aligned16(x_dev) || !aligned16(work_dev)) return fail(COARSE_EINVAL, "cagcr_cheb: pointers must be 16-byte aligned");
    { int rc0 = check_device(op, "cagcr_cheb"); if (rc0 != COARSE_OK) return rc0; }
    if (op->path_opt == COARSE_PATH_TENSOR || op->path_opt == COARSE_PATH_BLOCK)
        return fail(COARSE_EUNSUPPORTED, "cagcr_cheb: the handle is pinned to a block-apply path; the smoother applies 1 RHS");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    const size_t vec = coarse_op_vector_bytes(op, 1);
    {
        const size_t wb = coarse_op_cagcr_cheb_work_bytes(op, s);
        if (overlaps(b_dev, vec, x_dev, vec) || overlaps(b_dev, vec, work_dev, wb) || overlaps(x_dev, vec, work_dev, wb))
            return fail(COARSE_EINVAL, "cagcr_cheb: b, x and work must not overlap");
    }
    op->last_launches = 0;
    const long long n = (long long)op->lat.V * op->Nc;
    const int S1 = s + 1, NSLOT = 2 * s + 1;
    unsigned char* w = static_cast<unsigned char*>(work_dev);
    float2* slot[2 * CAGCR_MAX_S + 1];
    for (int k = 0; k < NSLOT; ++k) slot[k] = reinterpret_cast<float2*>(w + (size_t)k * vec);
    float2* tmp = reinterpret_cast<float2*>(w + (size_t)NSLOT * vec);
    double2* partial = reinterpret_cast<double2*>(w + (size_t)(NSLOT + 1) * vec);
    double2* alpha = partial + (size_t)CAGCR_GRAM_BLOCKS * S1 * S1;
    double* cd = reinterpret_cast<double*>(alpha + CAGCR_MAX_S);          // {c, d} of the Chebyshev interval
    const int vgrid = op->num_sms * 4;
    int launches = 0, rc;
    if (!auto_interval) {
        cagcr_set_interval_kernel<<<1, 1, 0, st>>>(0.5 * ((double)lambda_max + (double)lambda_min),
                                                   0.5 * ((double)lambda_max - (double)lambda_min), cd);
        ++launches;
    }
    if (schur_parity >= 0) {
        for (int mu = 0; mu < 4; ++mu)
            if (op->lat.L[mu] & 1) return fail(COARSE_EINVAL, "cagcr_cheb: the even/odd decomposition needs even extents");
        cudaError_t e = cudaMemsetAsync(work_dev, 0, (size_t)NSLOT * vec, st);
        if (e != cudaSuccess) return cuda_fail(e, "cagcr_cheb: memset work");
    }
    auto apply_op = [&](const void* in, void* out) -> int {
        if (schur_parity < 0) {
            ++launches;
            return coarse_op_apply(op, in, out, 1, 0, stream);
        }
        launches += 2;
        int r = coarse_op_apply_parts(op, nullptr, in, tmp, 1, 0, 1 - schur_parity, COARSE_LOCAL_NONE, 0.f, 1.f, stream);
        if (r != COARSE_OK) return r;
        return coarse_op_apply_parts(op, in, tmp, out, 1, 0, schur_parity, COARSE_LOCAL_IDENTITY, 1.f, -1.f, stream);
    };
    int p0 = 0, rslot = 2 * s;          // slot of P_0 and of the update's output; swapped after every cycle
    bool p0_is_b = false;
    if (x_is_zero) {
        cudaError_t e = cudaMemsetAsync(x_dev, 0, vec, st);
        if (e != cudaSuccess) return cuda_fail(e, "cagcr_cheb: memset x");
        p0_is_b = true;
    } else {
        rc = apply_op(x_dev, slot[s]);
        if (rc != COARSE_OK) return rc;
        cagcr_residual_kernel<<<vgrid, 256, 0, st>>>(static_cast<const float2*>(b_dev), slot[s], n, slot[p0]);
        ++launches;
    }
    for (int cyc = 0; cyc < cycles; ++cyc) {
        CagcrVecs P, T, Gv;
        for (int k = 0; k <= CAGCR_MAX_S; ++k) { P.p[k] = nullptr; T.p[k] = nullptr; Gv.p[k] = nullptr; }
        for (int k = 0; k < s; ++k) {
            P.p[k] = k == 0 ? (p0_is_b ? static_cast<const float2*>(b_dev) : slot[p0]) : slot[k];
            T.p[k] = slot[s + k];
        }
        for (int k = 0; k < s; ++k) {
            rc = apply_op(P.p[k], const_cast<float2*>(T.p[k]));
            if (rc != COARSE_OK) { op->last_launches = launches; return rc; }
            if (k == 0 && cyc == 0 && auto_interval) {
                // moments of the first residual -> interval, on the device (no host round trip)
                CagcrVecs Mv;
                for (int q = 0; q <= CAGCR_MAX_S; ++q) Mv.p[q] = nullptr;
                Mv.p[0] = P.p[0];
                Mv.p[1] = T.p[0];
                cagcr_gram_kernel<<<CAGCR_GRAM_BLOCKS, 256, 0, st>>>(Mv, n, 1, partial);
                cagcr_interval_kernel<<<1, 32, 0, st>>>(partial, CAGCR_GRAM_BLOCKS, cd);
                launches += 2;
            }
            if (k + 1 < s) {
                cagcr_cheb_step_kernel<<<vgrid, 256, 0, st>>>(T.p[k], P.p[k], k == 0 ? P.p[k] : P.p[k - 1], cd, k == 0 ? 1 : 0, n,
                                                              const_cast<float2*>(P.p[k + 1]));
                ++launches;
            }
        }
        Gv.p[0] = P.p[0];
        for (int k = 0; k < s; ++k) Gv.p[k + 1] = T.p[k];
        cagcr_gram_kernel<<<CAGCR_GRAM_BLOCKS, 256, 0, st>>>(Gv, n, s, partial);
        cagcr_solve_kernel<<<1, 320, 0, st>>>(partial, CAGCR_GRAM_BLOCKS, s, alpha, info_dev ? info_dev + 3 * cyc : nullptr);
        cagcr_update2_kernel<<<vgrid, 256, 0, st>>>(P, T, P.p[0], n, s, alpha, static_cast<float2*>(x_dev), slot[rslot]);
        launches += 3;
        {
            cudaError_t ec = cudaGetLastError();
            if (ec != cudaSuccess) { op->last_launches = launches; return cuda_fail(ec, "cagcr_cheb kernel launch"); }
        }
        if (p0_is_b) { p0 = rslot; rslot = 0; p0_is_b = false; }   // slot 0 was unused while P_0 = b
        else { const int t2 = p0; p0 = rslot; rslot = t2; }
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "cagcr_cheb kernel launch");
    op->last_launches = launches;
    return COARSE_OK;
}

size_t coarse_op_cagcr_cheb_work_bytes(const coarse_op_t* op, int s) {
    if (!op || s < 1 || s > CAGCR_MAX_S) return 0;
    const size_t vec = coarse_op_vector_bytes(op, 1);
    const size_t S1 = (size_t)s + 1;
    return (2 * (size_t)s + 2) * vec + (size_t)CAGCR_GRAM_BLOCKS * S1 * S1 * sizeof(double2) + (size_t)CAGCR_MAX_S * sizeof(double2) + 256;
}

int coarse_op_cagcr_cheb(coarse_op_t* op, const void* b_dev, void* x_dev, int s, int cycles, int x_is_zero,
                         float lambda_min, float lambda_max, int schur_parity, void* work_dev, double* info_dev,
                         void* stream) {
    if (schur_parity < -1 || schur_parity > 1) return fail(COARSE_EINVAL, "cagcr_cheb: schur_parity must be -1 (full operator), 0 or 1");
    return cagcr_cheb_impl(op, b_dev, x_dev, s, cycles, x_is_zero, lambda_min, lambda_max, schur_parity, work_dev, info_dev, stream);
}

int coarse_op_cagcr(coarse_op_t* op, const void* b_dev, void* x_dev, int s, int cycles, int x_is_zero,
                    void* work_dev, double* info_dev, void* stream) {
    return cagcr_cheb_impl(op, b_dev, x_dev, s, cycles, x_is_zero, 0.f, 0.f, -1, work_dev, info_dev, stream);
}

int coarse_op_cagcr_schur(coarse_op_t* op_hat, const void* b_dev, void* x_dev, int s, int cycles, int x_is_zero,
                          int parity, void* work_dev, double* info_dev, void* stream) {
    if (parity != 0 && parity != 1) return fail(COARSE_EINVAL, "cagcr_schur: parity must be 0 (even) or 1 (odd)");
    return cagcr_cheb_impl(op_hat, b_dev, x_dev, s, cycles, x_is_zero, 0.f, 0.f, parity, work_dev, info_dev, stream);
}

static int hat_grid(const coarse_op* op) {
    const int g = 2 * op->num_sms;
    return op->lat.V < g ? op->lat.V : g;
}

size_t coarse_op_hat_work_bytes(const coarse_op_t* op) {
    if (!op) return 0;
    return (size_t)hat_grid(op) * op->Nc * op->Nc * sizeof(double2);
}

int coarse_op_build_hat_links(coarse_op_t* op, void* out_links_c64_dev, int slot0, void* work_dev, int* info_dev,
                              void* stream) {
    if (!op) return fail(COARSE_EINVAL, "build_hat_links: op is NULL");
    if (!op->links) return fail(COARSE_ENOTREADY, "build_hat_links: coarse_op_set_links has not been called");
    if (!out_links_c64_dev || !work_dev) return fail(COARSE_EINVAL, "build_hat_links: NULL pointer");
    if (slot0 != COARSE_HAT_SLOT0_IDENTITY && slot0 != COARSE_HAT_SLOT0_XINV)
        return fail(COARSE_EINVAL, "build_hat_links: slot0 must be COARSE_HAT_SLOT0_IDENTITY or COARSE_HAT_SLOT0_XINV");
    if (!aligned16(out_links_c64_dev) || !aligned16(work_dev)) return fail(COARSE_EINVAL, "build_hat_links: pointers must be 16-byte aligned");
    int rc = check_device(op, "build_hat_links");
    if (rc != COARSE_OK) return rc;
    const size_t out_bytes = (size_t)op->lat.V * 9 * op->Nc * op->Nc * 8;
    if (overlaps(out_links_c64_dev, out_bytes, op->links, coarse_op_link_bytes(op)))
        return fail(COARSE_EINVAL, "build_hat_links: out_links overlaps the operator's own links (not an in-place operation)");
    if (overlaps(work_dev, coarse_op_hat_work_bytes(op), out_links_c64_dev, out_bytes) ||
        overlaps(work_dev, coarse_op_hat_work_bytes(op), op->links, coarse_op_link_bytes(op)))
        return fail(COARSE_EINVAL, "build_hat_links: work overlaps the links");
    if (op->lat.V == 0) return COARSE_OK;
    HatParams p;
    p.lat = op->lat;
    p.Nc = op->Nc;
    p.i16 = op->prec == COARSE_LINK_I16;
    p.links = op->links;
    p.scales = op->scales;
    p.out = static_cast<float2*>(out_links_c64_dev);
    p.work = static_cast<double2*>(work_dev);
    p.slot0_inverse = slot0 == COARSE_HAT_SLOT0_XINV;
    p.info = info_dev;
    const size_t smem = hat_smem_bytes(op->Nc);
    if (smem > (size_t)op->max_smem) return fail(COARSE_EUNSUPPORTED, "build_hat_links: Nc=%d needs %zu bytes of shared memory", op->Nc, smem);
    static SmemAttrCache attr_cache;
    cudaError_t e = ensure_dynamic_smem(hat_links_kernel, op->device, (int)smem, attr_cache);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(hat kernel)");
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (info_dev && (e = cudaMemsetAsync(info_dev, 0, sizeof(int), st)) != cudaSuccess) return cuda_fail(e, "build_hat_links: memset info");
    hat_links_kernel<<<hat_grid(op), HAT_THREADS, smem, st>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "hat kernel launch");
    op->last_launches = 1;
    return COARSE_OK;
}

int coarse_op_probe_read(const void* src_dev, size_t bytes, int stage_bytes, int stages, void* stream) {
    if (!src_dev || !aligned16(src_dev)) return fail(COARSE_EINVAL, "probe_read: src_dev must be a 16-byte aligned device pointer");
    if (stage_bytes < 1024 || (stage_bytes & 15) || stages < 2 || stages > 32)
        return fail(COARSE_EINVAL, "probe_read: stage_bytes must be a multiple of 16 >= 1024 and 2 <= stages <= 32");
    int dev = 0, sms = 0, max_smem = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "probe_read: cudaGetDevice");
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    const int smem = stages * (stage_bytes + 16) + 64;
    if (smem > max_smem) return fail(COARSE_EINVAL, "probe_read: %d stages of %d bytes do not fit shared memory", stages, stage_bytes);
    const unsigned long long n_stages = bytes / (size_t)stage_bytes;
    if (n_stages < 1) return fail(COARSE_EINVAL, "probe_read: fewer bytes than one stage");
    static SmemAttrCache attr_cache;
    e = ensure_dynamic_smem(probe_read_kernel, dev, smem, attr_cache);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(probe kernel)");
    const int grid = n_stages < (unsigned long long)sms ? (int)n_stages : sms;
    probe_read_kernel<<<grid, 64, smem, static_cast<cudaStream_t>(stream)>>>(static_cast<const unsigned char*>(src_dev),
                                                                           n_stages, stage_bytes, stages, nullptr);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "probe kernel launch");
    return COARSE_OK;
}

void coarse_op_destroy(coarse_op_t* op) {
    if (!op) return;
    if (op->stage_in) cudaFree(op->stage_in);
    if (op->stage_out) cudaFree(op->stage_out);
    if (op->split_ws) cudaFree(op->split_ws);
    if (op->vscale) cudaFree(op->vscale);
    if (op->host_pipe_ok) {
        for (int i = 0; i < 8; ++i) { cudaEventDestroy(op->ev_up[i]); cudaEventDestroy(op->ev_k[i]); }
        cudaEventDestroy(op->ev_done);
        cudaStreamDestroy(op->s_h2d);
        cudaStreamDestroy(op->s_d2h);
    }
    delete op;
}

const char* coarse_op_last_error(void) { return g_last_error.c_str(); }

}  // extern "C"
