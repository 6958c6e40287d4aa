// static_scratch.cu — coarse_op_apply_static (include/coarse_op.h): the block apply on int16 links through the
// integer tensor-core kernel (tensor_i8_kernel.cuh) with its scratch memory - the per-(site, right-hand side)
// power-of-two scales of the fixed-point vector operand - in a file-scope __device__ array instead of the buffer
// coarse_op_set_links allocates.  For callers that must not reach cudaMalloc (stream capture, serving loops,
// harnesses that forbid it): this entry point calls no cudaMalloc / cudaFree and no allocating library routine.
//
// The array lives in this translation unit's module: every GPU that loads the library holds its 1 MiB until the
// process exits.  In host code `g_static_vscale` is only a stand-in for the symbol, NOT a device address; the
// address is taken once per device with cudaGetSymbolAddress (that device current) and handed to the kernels.
// All calls and all handles share the array and it keeps the previous call's contents: nothing in it has to start
// at zero (each call's pre-pass kernel rewrites every entry the call's apply kernel reads), but two calls that
// overlap on the GPU (different streams, no ordering between them) race on it.
#include "internal.h"

#include <mutex>

#include "tensor_i8_kernel.cuh"

using namespace coarse;

namespace {

constexpr int kMaxDevices = 64;
constexpr size_t kScratchFloats = (size_t)COARSE_STATIC_MAX_SITES * TENSOR_I8_GP * 2;   // (g, 1/g) per (site, column)

static __device__ __align__(256) float g_static_vscale[kScratchFloats];

std::mutex g_mutex;
float* g_scratch_ptr[kMaxDevices] = {};     // device address of g_static_vscale on each device, taken on first use

// Device address of the array on the CURRENT device `dev` (set-up: once per device).
int scratch_address(int dev, float** out) {
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_scratch_ptr[dev]) {
        float* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_static_vscale);
        if (e != cudaSuccess) return cuda_fail(e, "apply_static: cudaGetSymbolAddress(static scratch)");
        if (!ptr) return fail(COARSE_ECUDA, "apply_static: cudaGetSymbolAddress returned a null address");
        g_scratch_ptr[dev] = ptr;
    }
    *out = g_scratch_ptr[dev];
    return COARSE_OK;
}

}  // namespace

extern "C" int coarse_op_apply_static(coarse_op_t* op, const void* in_dev, void* out_dev, int nrhs, int dagger, void* stream) {
    if (!op) return fail(COARSE_EINVAL, "apply_static: op is NULL");
    if (!op->links) return fail(COARSE_ENOTREADY, "apply_static: coarse_op_set_links has not been called");
    if (!in_dev || !out_dev) return fail(COARSE_EINVAL, "apply_static: in/out is NULL");
    if (nrhs < 1) return fail(COARSE_EINVAL, "apply_static: nrhs must be >= 1 (got %d)", nrhs);
    if (dagger != 0 && dagger != 1) return fail(COARSE_EINVAL, "apply_static: dagger must be 0 or 1 (got %d)", dagger);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (dev != op->device)
        return fail(COARSE_EINVAL, "apply_static: the handle was created on device %d but device %d is current", op->device, dev);
    if (dev < 0 || dev >= kMaxDevices) return fail(COARSE_EUNSUPPORTED, "apply_static: device ordinal %d >= %d", dev, kMaxDevices);
    if (op->prec != COARSE_LINK_I16 || !op->link_map_i8_ok)
        return fail(COARSE_EUNSUPPORTED, "apply_static: needs int16 links in a compiled Nc (the integer tensor-core kernel); "
                                         "got Nc=%d link format %d", op->Nc, op->prec);
    if (op->lat.V > COARSE_STATIC_MAX_SITES)
        return fail(COARSE_EUNSUPPORTED, "apply_static: %d sites exceed the static scratch (COARSE_STATIC_MAX_SITES = %d sites, %zu bytes)",
                    op->lat.V, COARSE_STATIC_MAX_SITES, kScratchFloats * sizeof(float));
    if ((reinterpret_cast<uintptr_t>(in_dev) & 15u) || (reinterpret_cast<uintptr_t>(out_dev) & 15u))
        return fail(COARSE_EINVAL, "apply_static: in/out must be 16-byte aligned");
    {
        const size_t vb = (size_t)op->lat.V * op->Nc * nrhs * 8;
        const uintptr_t a = reinterpret_cast<uintptr_t>(in_dev), b = reinterpret_cast<uintptr_t>(out_dev);
        if (a < b + vb && b < a + vb) return fail(COARSE_EINVAL, "apply_static: in and out overlap");
    }
    float* scratch = nullptr;
    int rc = scratch_address(dev, &scratch);
    if (rc != COARSE_OK) return rc;

    TensorParams p = {};
    p.lat = op->lat;
    p.scales = op->scales;
    p.in = static_cast<const float2*>(in_dev);
    p.in_local = p.in;
    p.out = static_cast<float2*>(out_dev);
    p.parity = 2;
    p.n_sites = op->lat.V;
    p.site_begin = 0;
    p.m_begin = 0;
    p.identity = 0;
    p.alpha = 1.f;
    p.beta = 1.f;
    p.nrhs = nrhs;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    op->last_launches = 0;
    switch (op->Nc) {
        // (u_other = NULL: one operand, so only the first V x TENSOR_I8_GP pairs of the scratch are used)
#define COARSE_CASE_NC(NC) case NC: rc = COARSE_CAT(launch_tensor_i8_nc, NC)(op, p, nullptr, scratch, dagger, st); break;
        COARSE_FOR_EACH_NC(COARSE_CASE_NC)
#undef COARSE_CASE_NC
        default: return fail(COARSE_EUNSUPPORTED, "apply_static: the TENSOR path is not compiled for Nc=%d", op->Nc);
    }
    if (rc < 0) return rc;
    op->last_launches = 1 + rc;
    op->last_path = COARSE_PATH_TENSOR;
    op->links_fresh = false;
    return COARSE_OK;
}
