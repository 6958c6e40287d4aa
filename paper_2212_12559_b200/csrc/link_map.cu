// link_map.cu — TMA tensor maps of the link array for the TENSOR kernels (tensor_kernel.cuh) and the
// shape predicates of that path.  Compiled once; the kernels live in launch_tensor.cu (one unit per Nc).
#include "internal.h"

namespace coarse {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_tiled_fn() {
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
    (void)prec;   // complex64 and int16 links
    switch (Nc) {
        case 32: case 48: case 64: case 96: case 128: case 192: return true;
        default: return false;
    }
}
bool tensor_supports(int Nc, int prec, int nrhs) { return tensor_supports_nc(Nc, prec) && nrhs >= 1; }

// The link array as a 2-D tensor of 32-bit elements: V*9*Nc rows (one per matrix row) of Nc*E elements,
// E = 2 (complex64: re, im floats) or 1 (int16: one (re,im) pair per element).
//   dagger 0 map: box = MT rows x 16 complex columns (128 B | 64 B per row), SWIZZLE_128B | SWIZZLE_64B
//   dagger 1 map: box = 16 rows x MT complex columns, no swizzle
// MT = Nc (Nc <= 128) or Nc / 2 (the output tile of one work item).
int make_link_maps(coarse_op* op) {
    op->link_map_ok = false;
    op->link_map_i8_ok = false;
    if (!tensor_supports_nc(op->Nc, op->prec)) return COARSE_OK;
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return COARSE_OK;   // TENSOR path stays unavailable; apply reports it if it is requested
    const int64_t rows = (int64_t)op->lat.V * 9 * op->Nc;
    if (rows > 0x7fffffffLL) return COARSE_OK;      // TMA coordinates are 32-bit
    const bool i16 = op->prec == COARSE_LINK_I16;
    const int E = i16 ? 1 : 2;
    const int MT = op->Nc > 128 ? op->Nc / 2 : op->Nc;
    const CUtensorMapDataType dt = i16 ? CU_TENSOR_MAP_DATA_TYPE_UINT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    const cuuint64_t gdim[2] = {(cuuint64_t)op->Nc * E, (cuuint64_t)rows};
    const cuuint64_t gstride[1] = {(cuuint64_t)op->Nc * E * 4};
    const cuuint32_t estr[2] = {1, 1};
    const cuuint32_t box0[2] = {(cuuint32_t)(16 * E), (cuuint32_t)MT};
    CUresult r = fn(&op->link_map[0], dt, 2, const_cast<void*>(op->links), gdim, gstride, box0, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, i16 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return COARSE_OK;
    const cuuint32_t box1[2] = {(cuuint32_t)(MT * E), 16};
    r = fn(&op->link_map[1], dt, 2, const_cast<void*>(op->links), gdim, gstride, box1, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    op->link_map_ok = (r == CUDA_SUCCESS);
    if (!op->link_map_ok || !i16) return COARSE_OK;
    // int16 links, integer tensor-core kernel: stages of KC = 32 complex columns (16 when 32 does not divide Nc)
    const int KC = op->Nc % 32 == 0 ? 32 : 16;
    const cuuint32_t box2[2] = {(cuuint32_t)KC, (cuuint32_t)MT};
    r = fn(&op->link_map_i8[0], dt, 2, const_cast<void*>(op->links), gdim, gstride, box2, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
           KC == 32 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return COARSE_OK;
    const cuuint32_t box3[2] = {(cuuint32_t)MT, (cuuint32_t)KC};
    r = fn(&op->link_map_i8[1], dt, 2, const_cast<void*>(op->links), gdim, gstride, box3, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    op->link_map_i8_ok = (r == CUDA_SUCCESS);
    return COARSE_OK;
}

}  // namespace coarse
