// internal.h — what the translation units of libcoarseop share: the handle, the error helpers and the
// per-family launch entry points.  The library is built from several .cu files compiled in parallel
// (paper_2212_12559_b200/build.py): coarse_op.cu holds the C ABI, launch_stream.cu / launch_stream_mr.cu /
// launch_block.cu / launch_tensor.cu are compiled once per colour-spin size Nc (-DCOARSE_NC=...), link_map.cu once.
#pragma once
#include "../../include/coarse_op.h"

#include <cuda.h>
#include <cuda_runtime.h>

#include "common.cuh"

#define COARSE_FOR_EACH_NC(X) X(32) X(48) X(64) X(96) X(128) X(192)
#define COARSE_CAT_(a, b) a##b
#define COARSE_CAT(a, b) COARSE_CAT_(a, b)

struct coarse_op {
    coarse::Lat lat;
    int Nc;
    int prec;
    const void* links;
    const float* scales;
    int path_opt;
    int grid_opt;
    int stages_opt;
    int fine_opt;
    int keep_opt;
    int pdl_opt;              // COARSE_OPT_PDL: 0 auto, 1 always, 2 never
    bool links_fresh;         // no apply has been enqueued since coarse_op_set_links (auto PDL skips that launch)
    int split_opt;            // COARSE_OPT_SPLIT_DAGGER: 0 auto, 1 never, 2 always
    int warp_items_opt;       // COARSE_OPT_WARP_ITEMS: 0 auto, 1 never, 2 always
    float2* split_ws;         // partial vectors of the split dagger apply (allocated by set_links on tiny lattices)
    size_t split_ws_bytes;
    unsigned int* split_count; // per-site chunk counters of the split dagger apply (zero between launches)
    int l2_bytes;
    int last_launches;
    int last_path;
    int device;
    int num_sms;
    int max_smem;
    void* stage_in;
    void* stage_out;
    size_t stage_bytes;
    cudaStream_t s_h2d, s_d2h;      // apply_host's copy streams and events (created on first use)
    cudaEvent_t ev_up[8], ev_k[8], ev_done;   // up to 8 ranges of x3-slices
    bool host_pipe_ok;
    CUtensorMap link_map[2];   // 2-D views of the link array for the TENSOR path (dagger 0 / dagger 1 slabs, link_map.cu)
    bool link_map_ok;
    CUtensorMap link_map_i8[2];   // int16 links: the slabs of the integer tensor-core kernel (tensor_i8_kernel.cuh)
    bool link_map_i8_ok;
    float* vscale;             // int16 links: (g, 1/g) per (site, column) of the two operands of the int8 TENSOR kernel
    int tensor_i8_opt;         // COARSE_OPT_TENSOR_I8: 0 auto (on for int16 links), 1 never, 2 always
};

namespace coarse {

// thread-local error message of the C ABI (coarse_op_last_error); both return `code`
int fail(int code, const char* fmt, ...);
int cuda_fail(cudaError_t e, const char* what);

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per (kernel, device, size): the attribute is
// sticky, and re-issuing it on every launch costs host time in the regime where an apply takes 5-13 us.
// `cache` is a per-instantiation static (one int per device, the largest size set so far).
struct SmemAttrCache {
    int bytes[16] = {0};
};
template <typename K>
inline cudaError_t ensure_dynamic_smem(K kernel, int device, int bytes, SmemAttrCache& cache) {
    if (device >= 0 && device < 16 && cache.bytes[device] >= bytes) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess && device >= 0 && device < 16) cache.bytes[device] = bytes;
    return e;
}

// Parts apply (coarse_op_apply_parts): out = alpha*Loc(u) + beta*Hop(w) on one parity.  The plain
// apply is the special case gen = false (u = w, local = X, alpha = beta = 1, all sites).
struct PartsSpec {
    bool gen;
    const void* u;
    int parity;   // 0 even, 1 odd, 2 all
    int local;    // 0 none, 1 X, 2 identity
    float alpha, beta;
    const float* vnorms;   // non-NULL: half-precision input vectors (plain apply only)
    int site_begin, site_end;   // output sites [site_begin, site_end) (plain apply only); end = 0: all
    void* hout_q;               // non-NULL: also write the result as int16 + per-site norm (coarse_op_apply_hout, 1 RHS)
    float* hout_norms;
};

struct StreamParams;
struct BlockParams;
struct TensorParams;

// per-Nc entry points, one translation unit each
#define COARSE_DECL_NC(NC)                                                                                          \
    int COARSE_CAT(launch_stream_nc, NC)(const coarse_op* op, const StreamParams& p, int dagger, bool gen,            \
                                         cudaStream_t stream);                                                       \
    int COARSE_CAT(launch_stream_mr_nc, NC)(const coarse_op* op, const StreamParams& p, int nrhs, int dagger,         \
                                            cudaStream_t stream);                                                    \
    int COARSE_CAT(launch_block_nc, NC)(const coarse_op* op, const BlockParams& p, int dagger, cudaStream_t stream); \
    int COARSE_CAT(launch_tensor_nc, NC)(const coarse_op* op, const TensorParams& p, int dagger, cudaStream_t stream); \
    int COARSE_CAT(launch_tensor_i8_nc, NC)(const coarse_op* op, const TensorParams& p, const void* u_other,           \
                                            float* vscale, int dagger, cudaStream_t stream);                        \
    int COARSE_CAT(launch_tensor_i8h_nc, NC)(const coarse_op* op, const TensorParams& p, const float* vnorms,          \
                                             int dagger, cudaStream_t stream);
COARSE_FOR_EACH_NC(COARSE_DECL_NC)
#undef COARSE_DECL_NC

// link_map.cu
bool tensor_supports_nc(int Nc, int prec);
bool tensor_supports(int Nc, int prec, int nrhs);
int make_link_maps(coarse_op* op);

}  // namespace coarse
