// launch_block.cu — launch of the CUDA-core BLOCK kernels for ONE colour-spin size (-DCOARSE_NC=<Nc>).
#include "internal.h"
#include "block_kernel.cuh"

#ifndef COARSE_NC
#error "compile with -DCOARSE_NC=<Nc>"
#endif

namespace coarse {
namespace {

// ---------------------------------------------------------------- BLOCK dispatch
template <int NC, bool I16, bool DAG, int RP>
int launch_block_t(const coarse_op* op, const BlockParams& base, cudaStream_t stream) {
    using Gm = BlockGeom<NC, I16, RP>;
    BlockParams p = base;
    p.n_items = DAG ? op->lat.V : op->lat.V * Gm::NB;
    const int sb = Gm::stage_bytes(DAG, p.nrhs);
    int stages = (op->max_smem - Gm::fixed_bytes(DAG)) / (sb + 16);
    if (stages < 2) return fail(COARSE_EUNSUPPORTED, "BLOCK: shared memory too small for Nc=%d nrhs=%d", NC, p.nrhs);
    int want = (114688 + sb / 2) / sb;
    if (want < 3) want = 3;
    if (op->stages_opt > 0) want = op->stages_opt;
    if (stages > want) stages = want;
    p.stages = stages;
    const int smem = Gm::smem_bytes(DAG, p.nrhs, stages);
    auto kern = coarse_apply_block<NC, I16, DAG, RP>;
    static SmemAttrCache attr_cache;
    cudaError_t e = ensure_dynamic_smem(kern, op->device, smem, attr_cache);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(block kernel)");
    int grid = op->grid_opt > 0 ? op->grid_opt : op->num_sms;
    if (grid > p.n_items) grid = p.n_items;
    kern<<<grid, Gm::THREADS, smem, stream>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "block kernel launch");
    return COARSE_OK;
}

template <int NC>
int launch_block_nc(const coarse_op* op, const BlockParams& p, int dagger, cudaStream_t stream) {
    const bool i16 = op->prec == COARSE_LINK_I16;
    if (p.nrhs <= 8) {
        if (i16) return dagger ? launch_block_t<NC, true, true, 8>(op, p, stream) : launch_block_t<NC, true, false, 8>(op, p, stream);
        return dagger ? launch_block_t<NC, false, true, 8>(op, p, stream) : launch_block_t<NC, false, false, 8>(op, p, stream);
    }
    if (i16) return dagger ? launch_block_t<NC, true, true, 16>(op, p, stream) : launch_block_t<NC, true, false, 16>(op, p, stream);
    return dagger ? launch_block_t<NC, false, true, 16>(op, p, stream) : launch_block_t<NC, false, false, 16>(op, p, stream);
}

}  // namespace

int COARSE_CAT(launch_block_nc, COARSE_NC)(const coarse_op* op, const BlockParams& p, int dagger, cudaStream_t stream) {
    return launch_block_nc<COARSE_NC>(op, p, dagger, stream);
}

}  // namespace coarse
