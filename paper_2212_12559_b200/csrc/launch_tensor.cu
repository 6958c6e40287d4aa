// launch_tensor.cu — launch of the tcgen05 TENSOR kernels (block apply) for ONE colour-spin size
// (compiled once per Nc with -DCOARSE_NC=<Nc>; see internal.h).
#include "internal.h"
#include "tensor_kernel.cuh"
#include "tensor_i8_kernel.cuh"

#ifndef COARSE_NC
#error "compile with -DCOARSE_NC=<Nc>"
#endif

namespace coarse {
namespace {

template <int NC, bool I16, int NP, bool DAG>
int launch_tensor_t(const coarse_op* op, const TensorParams& p, cudaStream_t stream) {
    using Gm = TensorGeom<NC, I16, NP>;
    auto kern = coarse_apply_tensor<NC, I16, NP, DAG>;
    static SmemAttrCache attr_cache;
    cudaError_t e = ensure_dynamic_smem(kern, op->device, Gm::SMEM_BYTES, attr_cache);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(tensor kernel)");
    int grid = op->grid_opt > 0 ? op->grid_opt : op->num_sms;
    const int n_items = Gm::NS == 2 ? (p.n_sites + 1) / 2 : p.n_sites * Gm::NT;
    if (grid > n_items) grid = n_items;
    if (grid < 1) return COARSE_OK;
    kern<<<grid, Gm::THREADS, Gm::SMEM_BYTES, stream>>>(op->link_map[DAG ? 1 : 0], p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "tensor kernel launch");
    return COARSE_OK;
}

template <int NC, bool I16, int NP>
int launch_tensor_d(const coarse_op* op, const TensorParams& p, int dagger, cudaStream_t stream) {
    return dagger ? launch_tensor_t<NC, I16, NP, true>(op, p, stream) : launch_tensor_t<NC, I16, NP, false>(op, p, stream);
}

// int16 links on the integer tensor cores (tensor_i8_kernel.cuh)
template <int NC, int NP, bool DAG, bool HV = false>
int launch_tensor_i8_t(const coarse_op* op, const TensorI8Params& p, cudaStream_t stream) {
    using Gm = TensorI8Geom<NC, NP, HV>;
    auto kern = coarse_apply_tensor_i8<NC, NP, DAG, HV>;
    static SmemAttrCache attr_cache;
    cudaError_t e = ensure_dynamic_smem(kern, op->device, Gm::SMEM_BYTES, attr_cache);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(tensor-i8 kernel)");
    int grid = op->grid_opt > 0 ? op->grid_opt : op->num_sms;
    const int n_items = Gm::NS == 2 ? (p.t.n_sites + 1) / 2 : p.t.n_sites * Gm::NT;
    if (grid > n_items) grid = n_items;
    if (grid < 1) return COARSE_OK;
    kern<<<grid, Gm::THREADS, Gm::SMEM_BYTES, stream>>>(op->link_map_i8[DAG ? 1 : 0], p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "tensor-i8 kernel launch");
    return COARSE_OK;
}

}  // namespace

// int16 links: per group of up to 16 right-hand sides one (or, when the local operand u differs from w, two)
// pre-pass launches for the power-of-two scales of the fixed-point B operand, then the kernel.  `vscale`
// holds 2 x V x TENSOR_I8_GP (g, 1/g) pairs.  Returns the number of launches beyond the first.
int COARSE_CAT(launch_tensor_i8_nc, COARSE_NC)(const coarse_op* op, const TensorParams& base, const void* u_other, float* vscale,
                                               int dagger, cudaStream_t stream) {
    int launches = 0;
    float* gw = vscale;
    float* gu = vscale + (size_t)2 * op->lat.V * TENSOR_I8_GP;
    for (int r0 = 0; r0 < base.nrhs; r0 += 16) {
        TensorI8Params p;
        p.t = base;
        p.t.r0 = r0;
        p.t.width = base.nrhs - r0 < 16 ? base.nrhs - r0 : 16;
        p.vscale_w = gw;
        p.vscale_u = u_other ? gu : gw;
        p.vnorms = nullptr;
        const long long total = (long long)op->lat.V * p.t.width;
        const unsigned blocks = (unsigned)((total + 127) / 128);
        vec_pow2_scale_kernel<<<blocks, 128, 0, stream>>>(base.in, op->lat.V, op->Nc, base.nrhs, r0, p.t.width, reinterpret_cast<float2*>(gw));
        ++launches;
        if (u_other) {
            vec_pow2_scale_kernel<<<blocks, 128, 0, stream>>>(static_cast<const float2*>(u_other), op->lat.V, op->Nc, base.nrhs, r0,
                                                              p.t.width, reinterpret_cast<float2*>(gu));
            ++launches;
        }
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "vector scale kernel launch");
        int rc = COARSE_OK;
        bool done = false;
        if constexpr (TensorI8Geom<COARSE_NC, 4>::OK) {      // Nc <= 64: 4-wide tile (two sites per item) for 2-4 right-hand sides
            if (p.t.width <= 4) {
                rc = dagger ? launch_tensor_i8_t<COARSE_NC, 4, true>(op, p, stream) : launch_tensor_i8_t<COARSE_NC, 4, false>(op, p, stream);
                done = true;
            }
        }
        if (done)
            ;
        else if (p.t.width <= 8)
            rc = dagger ? launch_tensor_i8_t<COARSE_NC, 8, true>(op, p, stream) : launch_tensor_i8_t<COARSE_NC, 8, false>(op, p, stream);
        else
            rc = dagger ? launch_tensor_i8_t<COARSE_NC, 16, true>(op, p, stream) : launch_tensor_i8_t<COARSE_NC, 16, false>(op, p, stream);
        if (rc != COARSE_OK) return rc;
        ++launches;
    }
    return launches > 0 ? launches - 1 : 0;
}

// int16 links AND int16 + norm vectors (coarse_op_apply_hvec with several right-hand sides): base.in holds int16 pairs,
// no pre-pass (the components are the fixed-point operand).  One launch per group of up to 16 right-hand sides; returns
// the number of launches beyond the first.
int COARSE_CAT(launch_tensor_i8h_nc, COARSE_NC)(const coarse_op* op, const TensorParams& base, const float* vnorms, int dagger,
                                                cudaStream_t stream) {
    int launches = 0;
    for (int r0 = 0; r0 < base.nrhs; r0 += 16) {
        TensorI8Params p;
        p.t = base;
        p.t.r0 = r0;
        p.t.width = base.nrhs - r0 < 16 ? base.nrhs - r0 : 16;
        p.vscale_w = p.vscale_u = nullptr;
        p.vnorms = vnorms;
        int rc = COARSE_OK;
        bool done = false;
        if constexpr (TensorI8Geom<COARSE_NC, 4, true>::OK) {
            if (p.t.width <= 4) {
                rc = dagger ? launch_tensor_i8_t<COARSE_NC, 4, true, true>(op, p, stream) : launch_tensor_i8_t<COARSE_NC, 4, false, true>(op, p, stream);
                done = true;
            }
        }
        if (done)
            ;
        else if (p.t.width <= 8)
            rc = dagger ? launch_tensor_i8_t<COARSE_NC, 8, true, true>(op, p, stream) : launch_tensor_i8_t<COARSE_NC, 8, false, true>(op, p, stream);
        else
            rc = dagger ? launch_tensor_i8_t<COARSE_NC, 16, true, true>(op, p, stream) : launch_tensor_i8_t<COARSE_NC, 16, false, true>(op, p, stream);
        if (rc != COARSE_OK) return rc;
        ++launches;
    }
    return launches > 0 ? launches - 1 : 0;
}

// One launch per group of up to 16 right-hand sides (8-wide tile when at most 8 are left); returns the
// number of launches beyond the first, or a negative error code.
int COARSE_CAT(launch_tensor_nc, COARSE_NC)(const coarse_op* op, const TensorParams& base, int dagger, cudaStream_t stream) {
    int extra = -1;
    for (int r0 = 0; r0 < base.nrhs; r0 += 16) {
        TensorParams p = base;
        p.r0 = r0;
        p.width = base.nrhs - r0 < 16 ? base.nrhs - r0 : 16;
        int rc;
        if (op->prec == COARSE_LINK_I16)
            rc = p.width <= 8 ? launch_tensor_d<COARSE_NC, true, 8>(op, p, dagger, stream) : launch_tensor_d<COARSE_NC, true, 16>(op, p, dagger, stream);
        else
            rc = p.width <= 8 ? launch_tensor_d<COARSE_NC, false, 8>(op, p, dagger, stream) : launch_tensor_d<COARSE_NC, false, 16>(op, p, dagger, stream);
        if (rc != COARSE_OK) return rc;
        ++extra;
    }
    return extra < 0 ? 0 : extra;
}

}  // namespace coarse
