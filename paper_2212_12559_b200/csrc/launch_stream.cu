// launch_stream.cu — kernel selection and launch of the 1-RHS STREAM kernels for ONE colour-spin size
// (compiled once per Nc with -DCOARSE_NC=<Nc>; see internal.h).
#include "internal.h"
#include "stream_kernel.cuh"
#include "stream2_kernel.cuh"

#ifndef COARSE_NC
#error "compile with -DCOARSE_NC=<Nc>"
#endif

namespace coarse {
namespace {

// ---------------------------------------------------------------- STREAM dispatch
template <int NC, bool I16, bool DAG, bool FINE, bool GEN, bool HV = false>
int launch_stream_t(const coarse_op* op, const StreamParams& base, cudaStream_t stream) {
    using Gm = StreamGeom<NC, I16, FINE, HV>;
    static_assert(Gm::OK, "unsupported STREAM geometry");
    StreamParams p = base;
    p.n_items = DAG ? p.n_sites : p.n_sites * Gm::NB;
    if (base.n_items > 0) {                       // a site range [item_begin, n_items) was requested (in sites)
        p.item_begin = DAG ? base.item_begin : base.item_begin * Gm::NB;
        p.n_items = DAG ? base.n_items : base.n_items * Gm::NB;
    }
    // dagger = 1 has one work item per site; on a lattice with fewer sites than SMs (the paper's level 3:
    // 32 sites per GPU) the contraction of a site is split over its NB row chunks, one item each, and the
    // CTA that finishes a site's last chunk adds the NB partial vectors in order (stream_kernel.cuh).
    // COARSE_OPT_SPLIT_DAGGER: 0 auto (clusters on lattices with fewer sites than SMs), 1 never, 2 always (clusters),
    // 3 always with the global-memory scheme: partial vectors in a workspace, a per-site counter, the CTA that counts a
    // site's last chunk in adds them (a device-scope fence, an atomic round trip and an L2 read at the end of the
    // kernel: measured 3.7 us of a 12.2 us apply on the paper's level-3 volume, against ~1 us for the cluster barrier).
    p.split = 0;
    p.partial = nullptr;
    p.split_count = nullptr;
    p.cluster = 0;
    const bool split_ok = DAG && !FINE && base.n_items == 0 && !base.hout_q && Gm::NB > 1;     // (HV, parts apply: clusters only)
    // auto: only when every site gets a cluster of its own at once - the largest cluster size (4, 2) with n_sites x size <= SMs.
    // Measured on Nc = 192 int16 (us, clusters / workspace scheme / no split): 32 sites 10.1 / 12.6 / 20.7, 64 sites (size 4, two
    // sites per cluster in turn) 19.5 / 18.8 / 21.0, 128 sites 57.7 / 40.7 / 27.0 - several sites per cluster, or chunks of
    // several sites per CTA, lose against one CTA per site.
    int auto_cluster = 0;
    if (Gm::NB >= STREAM_MAX_CLUSTER && (int64_t)p.n_sites * STREAM_MAX_CLUSTER <= op->num_sms) auto_cluster = STREAM_MAX_CLUSTER;
    else if ((int64_t)p.n_sites * 2 <= op->num_sms) auto_cluster = 2;
    const bool split_wanted = op->split_opt >= 2 || (op->split_opt == 0 && auto_cluster > 0);
    if (split_ok && split_wanted && op->split_opt != 3)
        p.cluster = op->split_opt == 0 ? auto_cluster : (Gm::NB >= STREAM_MAX_CLUSTER ? STREAM_MAX_CLUSTER : 2);
    auto use_workspace_split = [&]() {
        p.cluster = 0;
        if (split_ok && !HV && !GEN && split_wanted && op->split_ws && (size_t)p.n_sites * Gm::NB * NC * 8 <= op->split_ws_bytes) {
            p.split = 1;
            p.partial = op->split_ws;
            p.split_count = op->split_count;
            p.n_items = p.n_sites * Gm::NB;
        }
    };
    if (!p.cluster) use_workspace_split();
    int stages = (op->max_smem - Gm::fixed_bytes(DAG)) / (Gm::stage_bytes(DAG) + 16);
    if (stages > 12) stages = 12;
    if (stages < 2) return fail(COARSE_EUNSUPPORTED, "STREAM: shared memory too small for Nc=%d", NC);
    // Default depth: ~112 KB in flight per SM (the measured optimum, see stream_kernel.cuh), at
    // least 4 stages; COARSE_OPT_STAGES overrides.
    int want = (114688 + Gm::stage_bytes(DAG) / 2) / Gm::stage_bytes(DAG);
    if (want < 4) want = 4;
    if (op->stages_opt > 0) want = op->stages_opt;
    if (stages > want) stages = want;
    p.stages = stages;
    int smem = Gm::smem_bytes(DAG, stages);
    // PDL: a kernel whose shared-memory carve-out differs from its predecessor's cannot take over an SM
    // before it has drained completely (measured: an alternating dagger 0 / dagger 1 chain gained nothing
    // until both kernels asked for the same size), so under PDL both modes request the larger of the two.
    if (base.pdl && Gm::smem_bytes(!DAG, stages) > smem && Gm::smem_bytes(!DAG, stages) <= op->max_smem)
        smem = Gm::smem_bytes(!DAG, stages);
    auto kern = coarse_apply_stream<NC, I16, DAG, FINE, GEN, HV>;
    static SmemAttrCache attr_cache;
    cudaError_t e = ensure_dynamic_smem(kern, op->device, smem, attr_cache);
    if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(stream kernel)");
    int grid = op->grid_opt > 0 ? op->grid_opt : op->num_sms;
    p.pdl = base.pdl;
    if (p.cluster) {
        // one site per cluster at a time; as many clusters as the chip holds (or COARSE_OPT_GRID / cluster size)
        int n_cl = grid / p.cluster;
        if (n_cl < 1) n_cl = 1;
        if (n_cl > p.n_sites) n_cl = p.n_sites;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(n_cl * p.cluster);
        cfg.blockDim = dim3(Gm::THREADS);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = stream;
        cudaLaunchAttribute attr[2];
        attr[0].id = cudaLaunchAttributeClusterDimension;
        attr[0].val.clusterDim.x = p.cluster;
        attr[0].val.clusterDim.y = 1;
        attr[0].val.clusterDim.z = 1;
        attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[1].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = p.pdl ? 2 : 1;
        if constexpr (DAG && !FINE) {
            auto kern_cl = coarse_apply_stream<NC, I16, DAG, FINE, GEN, HV, true>;
            static SmemAttrCache attr_cache_cl;
            e = ensure_dynamic_smem(kern_cl, op->device, smem, attr_cache_cl);
            if (e == cudaSuccess) e = cudaLaunchKernelEx(&cfg, kern_cl, p);
            if (e == cudaSuccess) return COARSE_OK;
            cudaGetLastError();              // clusters of this size cannot be scheduled here: the workspace scheme
        }
        use_workspace_split();
    }
    if (grid > p.n_items - p.item_begin) grid = p.n_items - p.item_begin;
    if (grid < 1) return COARSE_OK;
    if (p.pdl) {
        // programmatic dependent launch: this kernel may start while the previous kernel of the stream
        // drains; it orders itself against that kernel's memory with griddepcontrol.wait (stream_kernel.cuh)
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3(grid);
        cfg.blockDim = dim3(Gm::THREADS);
        cfg.dynamicSmemBytes = smem;
        cfg.stream = stream;
        cudaLaunchAttribute attr[1];
        attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[0].val.programmaticStreamSerializationAllowed = 1;
        cfg.attrs = attr;
        cfg.numAttrs = 1;
        e = cudaLaunchKernelEx(&cfg, kern, p);
        if (e != cudaSuccess) return cuda_fail(e, "stream kernel launch (PDL)");
    } else {
        kern<<<grid, Gm::THREADS, smem, stream>>>(p);
        e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "stream kernel launch");
    }
    return COARSE_OK;
}

// Team-owned stages (stream2_kernel.cuh): plain apply on the whole lattice or a site range, no PDL.
template <int NC, bool I16, bool DAG, int TW, bool HV = false>
int launch_stream2_w(const coarse_op* op, const StreamParams& base, cudaStream_t stream) {
    using Gm = Stream2Geom<NC, I16, TW, HV>;
    if constexpr (!Gm::OK) {
        return fail(COARSE_EUNSUPPORTED, "STREAM (warp teams): no geometry for Nc=%d with %d warps per team", NC, TW);
    } else {
        StreamParams p = base;
        p.n_items = DAG ? p.n_sites : p.n_sites * Gm::NB;
        p.item_begin = 0;
        if (base.n_items > 0) {                       // a site range [item_begin, n_items) was requested (in sites)
            p.item_begin = DAG ? base.item_begin : base.item_begin * Gm::NB;
            p.n_items = DAG ? base.n_items : base.n_items * Gm::NB;
        }
        // ring: one slot per team being read + ~104 KB in flight (the measured optimum of the read stream),
        // a multiple of the team count so that every slot has a fixed owner; COARSE_OPT_STAGES overrides
        const int sb = Gm::stage_bytes(DAG);
        int slots = Gm::T + (106496 + sb / 2) / sb;
        if (op->stages_opt > 0) slots = op->stages_opt;
        const int fit = (op->max_smem - Gm::fixed_bytes(DAG)) / (sb + 16);
        if (slots > fit) slots = fit;
        slots = (slots + Gm::T / 2) / Gm::T * Gm::T;
        if (slots > fit) slots -= Gm::T;
        if (slots < 2 * Gm::T) slots = 2 * Gm::T;
        if (slots > fit) return fail(COARSE_EUNSUPPORTED, "STREAM (warp teams): shared memory too small for Nc=%d", NC);
        p.stages = slots;
        const int smem = Gm::smem_bytes(DAG, slots);
        auto kern = coarse_apply_stream2<NC, I16, DAG, TW, HV>;
        static SmemAttrCache attr_cache;
        cudaError_t e = ensure_dynamic_smem(kern, op->device, smem, attr_cache);
        if (e != cudaSuccess) return cuda_fail(e, "cudaFuncSetAttribute(stream2 kernel)");
        int grid = op->grid_opt > 0 ? op->grid_opt : op->num_sms;
        const int need = (p.n_items - p.item_begin + Gm::T - 1) / Gm::T;
        if (grid > need) grid = need;
        if (grid < 1) return COARSE_OK;
        kern<<<grid, Gm::THREADS, smem, stream>>>(p);
        e = cudaGetLastError();
        if (e != cudaSuccess) return cuda_fail(e, "stream2 kernel launch");
        return COARSE_OK;
    }
}

// COARSE_OPT_WARP_ITEMS: 2 = default team width (4 warps: two teams; measured best on C4 and P2, where
// its default ring of 8 slots has the 6 x 16 KB in flight the read stream peaks at), 12 / 14 = 2 / 4 warps
template <int NC, bool I16, bool DAG, bool HV = false>
int launch_stream2_t(const coarse_op* op, const StreamParams& base, cudaStream_t stream) {
    // rows of 24 / 48 quads (Nc = 96 / 192 int16) run best with 2 warps per team (measured: Nc 96 6.6 / 6.8 TB/s
    // against 6.0 / 6.7 with 4 and 5.4 / 5.4 on the cooperative kernel), the others with 4
    constexpr bool has4 = Stream2Geom<NC, I16, 4>::OK, has2 = Stream2Geom<NC, I16, 2>::OK;
    const bool two = !has4 || (has2 && (op->warp_items_opt == 12 || (op->warp_items_opt != 14 && (NC % 3 == 0 || NC == 32))));
    if (two) return launch_stream2_w<NC, I16, DAG, 2, HV>(op, base, stream);
    return launch_stream2_w<NC, I16, DAG, 4, HV>(op, base, stream);
}

template <int NC, bool I16>
bool use_warp_items(const coarse_op* op, const StreamParams& p, int dagger, bool gen) {
    // (site-range launches take the decision the full-lattice apply takes, so that coarse_op_apply_host stays
    // bit-identical to coarse_op_apply)
    if (gen || (p.vnorms && !I16) || p.pdl || op->warp_items_opt == 1) return false;   // (half vectors: int16 links only)
    if (p.hout_q) {
        // half-precision output: int16 links, and in dagger = 0 only when a work item is a whole site (a team then holds
        // all rows of the site; otherwise the cooperative kernel's site-owning CTAs do it)
        constexpr int nb4 = Stream2Geom<NC, I16, 4>::OK ? Stream2Geom<NC, I16, 4>::NB : 1;
        constexpr int nb2 = Stream2Geom<NC, I16, 2>::OK ? Stream2Geom<NC, I16, 2>::NB : 1;
        if (!I16 || (!dagger && (nb4 > 1 || nb2 > 1))) return false;
    }
    if (op->warp_items_opt >= 2) return true;
    // auto: int16 links with Nc >= 48 (issue-bound on the cooperative kernel; Nc = 48: 5.5 / 5.2 -> 6.3 / 6.4 TB/s with
    // 2 warps per team) and the 4-8 KB matrices of Nc = 32 (the cooperative kernel pays its per-stage handshake eight
    // times per 8 KB there: complex64 5.6 / 5.1 -> 7.2 / 7.0 TB/s, int16 2.7 / 2.5 -> 3.7 / 3.7), on lattices with at
    // least 4 items per team of the chip
    using G2 = Stream2Geom<NC, I16, (Stream2Geom<NC, I16, 4>::OK ? 4 : 2)>;
    const int64_t items = dagger ? (int64_t)p.n_sites : (int64_t)p.n_sites * G2::NB;
    return ((I16 && NC >= 48) || NC == 32) && items >= (int64_t)4 * G2::T * op->num_sms;
}

// dagger = 0 on a tiny lattice: switch to the fine row-block geometry when the regular one gives
// fewer work items than SMs (COARSE_OPT_FINE: 0 auto, 1 never, 2 always).  Measured on C1
// (256 sites, Nc = 48: 256 regular items on 148 SMs) the regular geometry is 2.8x faster (5.6 us
// vs 15.4 us warm): 3 KB stages pay the per-stage handshake 6x more often, so the fine split only
// pays when SMs would otherwise sit idle.
template <int NC, bool I16, bool GEN>
int launch_stream_n(const coarse_op* op, const StreamParams& p, cudaStream_t stream) {
    constexpr bool HAS_FINE = StreamGeom<NC, I16, true>::NB > StreamGeom<NC, I16, false>::NB;
    if constexpr (HAS_FINE) {
        const bool few = (int64_t)p.n_sites * StreamGeom<NC, I16, false>::NB < (int64_t)op->num_sms;
        if (op->fine_opt == 2 || (op->fine_opt == 0 && few)) return launch_stream_t<NC, I16, false, true, GEN>(op, p, stream);
    }
    return launch_stream_t<NC, I16, false, false, GEN>(op, p, stream);
}

template <int NC, bool GEN>
int launch_stream_nc(const coarse_op* op, const StreamParams& p, int dagger, cudaStream_t stream) {
    if (op->prec == COARSE_LINK_I16)
        return dagger ? launch_stream_t<NC, true, true, false, GEN>(op, p, stream) : launch_stream_n<NC, true, GEN>(op, p, stream);
    return dagger ? launch_stream_t<NC, false, true, false, GEN>(op, p, stream) : launch_stream_n<NC, false, GEN>(op, p, stream);
}

template <int NC>
int launch_stream_g(const coarse_op* op, const StreamParams& p, int dagger, bool gen, cudaStream_t stream) {
    if (p.vnorms) {   // half-precision input vectors: regular geometry, plain apply
        if (op->prec == COARSE_LINK_I16) {
            // the paper's storage for both operands: warp teams on large lattices, as for complex64 vectors
            if constexpr (Stream2Geom<NC, true, 4>::OK || Stream2Geom<NC, true, 2>::OK)
                if (use_warp_items<NC, true>(op, p, dagger, gen))
                    return dagger ? launch_stream2_t<NC, true, true, true>(op, p, stream) : launch_stream2_t<NC, true, false, true>(op, p, stream);
        }
        if (op->prec == COARSE_LINK_I16)
            return dagger ? launch_stream_t<NC, true, true, false, false, true>(op, p, stream)
                          : launch_stream_t<NC, true, false, false, false, true>(op, p, stream);
        return dagger ? launch_stream_t<NC, false, true, false, false, true>(op, p, stream)
                      : launch_stream_t<NC, false, false, false, false, true>(op, p, stream);
    }
    if (op->prec == COARSE_LINK_I16) {
        if constexpr (Stream2Geom<NC, true, 4>::OK || Stream2Geom<NC, true, 2>::OK)
            if (use_warp_items<NC, true>(op, p, dagger, gen))
                return dagger ? launch_stream2_t<NC, true, true>(op, p, stream) : launch_stream2_t<NC, true, false>(op, p, stream);
    } else {
        if constexpr (Stream2Geom<NC, false, 4>::OK || Stream2Geom<NC, false, 2>::OK)
            if (use_warp_items<NC, false>(op, p, dagger, gen))
                return dagger ? launch_stream2_t<NC, false, true>(op, p, stream) : launch_stream2_t<NC, false, false>(op, p, stream);
    }
    return gen ? launch_stream_nc<NC, true>(op, p, dagger, stream) : launch_stream_nc<NC, false>(op, p, dagger, stream);
}

}  // namespace

int COARSE_CAT(launch_stream_nc, COARSE_NC)(const coarse_op* op, const StreamParams& p, int dagger, bool gen,
                                            cudaStream_t stream) {
    return launch_stream_g<COARSE_NC>(op, p, dagger, gen, stream);
}

}  // namespace coarse
