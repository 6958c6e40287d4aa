// launch_tensor.cu — tensor map set-up and launch of the tcgen05 TENSOR kernels (block apply, nrhs in {8,16}).
#include "internal.h"
#include "tensor_kernel.cuh"

namespace coarse {

// ---------------------------------------------------------------- TENSOR dispatch
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* sym = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &sym, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(sym);
        else
            cudaGetLastError();
    }
    return fn;
}

bool tensor_supports_nc(int Nc, int prec) {
    return prec == COARSE_LINK_C64 && (Nc == 48 || Nc == 64 || Nc == 128);
}
bool tensor_supports(int Nc, int prec, int nrhs) { return tensor_supports_nc(Nc, prec) && (nrhs == 8 || nrhs == 16); }

// links[V*9*Nc rows][2*Nc floats]; box = Nc rows x 32 floats (128 B), SWIZZLE_128B.
int make_link_map(coarse_op* op) {
    op->link_map_ok = false;
    if (!tensor_supports_nc(op->Nc, op->prec)) return COARSE_OK;
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return COARSE_OK;   // TENSOR path stays unavailable; apply reports it if it is requested
    const cuuint64_t gdim[2] = {(cuuint64_t)2 * op->Nc, (cuuint64_t)op->lat.V * 9 * op->Nc};
    const cuuint64_t gstride[1] = {(cuuint64_t)op->Nc * 8};
    const cuuint32_t box[2] = {32, (cuuint32_t)op->Nc};
    const cuuint32_t estr[2] = {1, 1};
    CUresult r = fn(&op->link_map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(op->links), gdim, gstride, box,
                    estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    op->link_map_ok = (r == CUDA_SUCCESS);
    return COARSE_OK;
}

template <int NC, int NRHS, bool DAG>
int launch_tensor_t(const coarse_op* op, const TensorParams& p, cudaStream_t stream) {
    using Gm = TensorGeom<NC, NRHS>;
    auto kern = coarse_apply_tensor<NC, NRHS, DAG>;
    static SmemAttrCache attr_cache;
    cudaError_t e = ensure_dynamic_smem(kern, op->device, Gm::SMEM_BYTES, attr_cache);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(tensor kernel)");
    int grid = op->grid_opt > 0 ? op->grid_opt : op->num_sms;
    if (grid > p.n_sites) grid = p.n_sites;
    kern<<<grid, Gm::THREADS, Gm::SMEM_BYTES, stream>>>(op->link_map, p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "tensor kernel launch");
    return COARSE_OK;
}

template <int NC>
int launch_tensor_nc(const coarse_op* op, const TensorParams& p, int nrhs, int dagger, cudaStream_t stream) {
    if (nrhs == 8)
        return dagger ? launch_tensor_t<NC, 8, true>(op, p, stream) : launch_tensor_t<NC, 8, false>(op, p, stream);
    return dagger ? launch_tensor_t<NC, 16, true>(op, p, stream) : launch_tensor_t<NC, 16, false>(op, p, stream);
}

int launch_tensor(const coarse_op* op, const void* in, void* out, int nrhs, int dagger, cudaStream_t stream) {
    if (!op->link_map_ok) return fail(COARSE_EUNSUPPORTED, "TENSOR path: no tensor map for these links");
    TensorParams p;
    p.lat = op->lat;
    p.links = static_cast<const unsigned char*>(op->links);
    p.in = static_cast<const float2*>(in);
    p.out = static_cast<float2*>(out);
    p.n_sites = op->lat.V;
    switch (op->Nc) {
        case 48: return launch_tensor_nc<48>(op, p, nrhs, dagger, stream);
        case 64: return launch_tensor_nc<64>(op, p, nrhs, dagger, stream);
        case 128: return launch_tensor_nc<128>(op, p, nrhs, dagger, stream);
        default: return fail(COARSE_EUNSUPPORTED, "TENSOR path is not compiled for Nc=%d", op->Nc);
    }
}


}  // namespace coarse
