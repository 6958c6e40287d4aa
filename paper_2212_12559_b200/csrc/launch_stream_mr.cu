// launch_stream_mr.cu — launch of the 2-4 RHS STREAM-MR kernels for ONE colour-spin size (-DCOARSE_NC=<Nc>).
#include "internal.h"
#include "stream_mr_kernel.cuh"

#ifndef COARSE_NC
#error "compile with -DCOARSE_NC=<Nc>"
#endif

namespace coarse {
namespace {

// ---------------------------------------------------------------- STREAM-MR dispatch (2 <= nrhs <= 4)
template <int NC, bool I16, bool DAG, int R>
int launch_stream_mr_t(const coarse_op* op, const StreamParams& base, cudaStream_t stream) {
    using Gm = StreamGeom<NC, I16, false, false, true>;
    using Gr = StreamMrGeom<NC, I16, R>;
    StreamParams p = base;
    p.cluster = 0;
    p.n_items = DAG ? base.n_sites : base.n_sites * Gm::NB;      // n_sites: the parity set of a parts apply, else V
    p.item_begin = 0;
    if (base.n_items > 0) {                       // a site range [item_begin, n_items) was requested (in sites)
        p.item_begin = DAG ? base.item_begin : base.item_begin * Gm::NB;
        p.n_items = DAG ? base.n_items : base.n_items * Gm::NB;
    }
    int stages = (op->max_smem - Gr::fixed_bytes(DAG)) / (Gr::stage_bytes(DAG) + 16);
    if (stages > 12) stages = 12;
    if (stages < 2) return fail(COARSE_EUNSUPPORTED, "STREAM-MR: shared memory too small for Nc=%d nrhs=%d", NC, R);
    int want = (114688 + Gr::stage_bytes(DAG) / 2) / Gr::stage_bytes(DAG);
    if (want < 4) want = 4;
    if (op->stages_opt > 0) want = op->stages_opt;
    if (stages > want) stages = want;
    p.stages = stages;
    const int smem = Gr::smem_bytes(DAG, stages);
    auto kern = coarse_apply_stream_mr<NC, I16, DAG, R>;
    static SmemAttrCache attr_cache;
    cudaError_t e = ensure_dynamic_smem(kern, op->device, smem, attr_cache);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(stream-mr kernel)");
    int grid = op->grid_opt > 0 ? op->grid_opt : op->num_sms;
    if (grid > p.n_items - p.item_begin) grid = p.n_items - p.item_begin;
    if (grid < 1) return COARSE_OK;
    // dagger = 1 on a lattice with fewer sites than SMs: thread-block clusters, one site per cluster, the contraction of a
    // site split over the cluster's CTAs (COARSE_OPT_SPLIT_DAGGER 1 / 3: off); falls back to the plain launch
    if constexpr (DAG) {
        int auto_cluster = 0;                 // every site a cluster of its own at once (launch_stream.cu)
        if (Gm::NB >= STREAM_MAX_CLUSTER && (int64_t)p.n_sites * STREAM_MAX_CLUSTER <= op->num_sms) auto_cluster = STREAM_MAX_CLUSTER;
        else if ((int64_t)p.n_sites * 2 <= op->num_sms) auto_cluster = 2;
        if (base.n_items == 0 && Gm::NB > 1 && op->split_opt != 1 && op->split_opt != 3 && (op->split_opt == 2 || auto_cluster > 0)) {
            p.cluster = op->split_opt == 0 ? auto_cluster : (Gm::NB >= STREAM_MAX_CLUSTER ? STREAM_MAX_CLUSTER : 2);
            int n_cl = (op->grid_opt > 0 ? op->grid_opt : op->num_sms) / p.cluster;
            if (n_cl < 1) n_cl = 1;
            if (n_cl > p.n_sites) n_cl = p.n_sites;
            auto kern_cl = coarse_apply_stream_mr<NC, I16, DAG, R, true>;
            static SmemAttrCache attr_cache_cl;
            e = ensure_dynamic_smem(kern_cl, op->device, smem, attr_cache_cl);
            if (e == cudaSuccess && n_cl >= 1) {
                cudaLaunchConfig_t cfg = {};
                cfg.gridDim = dim3(n_cl * p.cluster);
                cfg.blockDim = dim3(Gm::THREADS);
                cfg.dynamicSmemBytes = smem;
                cfg.stream = stream;
                cudaLaunchAttribute attr[1];
                attr[0].id = cudaLaunchAttributeClusterDimension;
                attr[0].val.clusterDim.x = p.cluster;
                attr[0].val.clusterDim.y = 1;
                attr[0].val.clusterDim.z = 1;
                cfg.attrs = attr;
                cfg.numAttrs = 1;
                e = cudaLaunchKernelEx(&cfg, kern_cl, p);
                if (e == cudaSuccess) return COARSE_OK;
            }
            cudaGetLastError();
            p.cluster = 0;
        }
    }
    kern<<<grid, Gm::THREADS, smem, stream>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e, "stream-mr kernel launch");
    return COARSE_OK;
}

template <int NC, int R>
int launch_stream_mr_r(const coarse_op* op, const StreamParams& p, int dagger, cudaStream_t stream) {
    if (op->prec == COARSE_LINK_I16)
        return dagger ? launch_stream_mr_t<NC, true, true, R>(op, p, stream) : launch_stream_mr_t<NC, true, false, R>(op, p, stream);
    return dagger ? launch_stream_mr_t<NC, false, true, R>(op, p, stream) : launch_stream_mr_t<NC, false, false, R>(op, p, stream);
}

template <int NC>
int launch_stream_mr_nc(const coarse_op* op, const StreamParams& p, int nrhs, int dagger, cudaStream_t stream) {
    switch (nrhs) {
        case 2: return launch_stream_mr_r<NC, 2>(op, p, dagger, stream);
        case 3: return launch_stream_mr_r<NC, 3>(op, p, dagger, stream);
        default: return launch_stream_mr_r<NC, 4>(op, p, dagger, stream);
    }
}

}  // namespace

int COARSE_CAT(launch_stream_mr_nc, COARSE_NC)(const coarse_op* op, const StreamParams& p, int nrhs, int dagger,
                                               cudaStream_t stream) {
    return launch_stream_mr_nc<COARSE_NC>(op, p, nrhs, dagger, stream);
}

}  // namespace coarse
