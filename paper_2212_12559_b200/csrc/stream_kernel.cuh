// stream_kernel.cuh — COARSE_PATH_STREAM: the single-RHS coarse-op apply as an HBM streaming kernel.
//
// 97-99 % of the bytes of one apply are the nine Nc x Nc link matrices per site (SURVEY.md §8(a)
// row a3), each read exactly once, and in the C-ABI layout links[s][m][i][j] every (site, matrix,
// row range) is one contiguous run of bytes.  So the kernel is a persistent producer/consumer
// pipeline per SM:
//
//   producer (1 elected thread)  walks its work items and, per pipeline stage, issues two 1-D TMA
//       bulk copies (cp.async.bulk, SASS UBLKCP) into a ring of S shared-memory slots: the link rows
//       of one (site, matrix, row range) with an L2 evict_first hint, and the neighbour vector
//       entries that those rows multiply with an evict_last hint (the vector field is re-read 9x
//       and stays L2-resident).  Completion is counted in bytes on the slot's `full` mbarrier.
//       The ring depth S is chosen by the host so that ~112 KB per SM (~16 MB chip-wide) is in
//       flight: measured on B200, throughput peaks there (S = 6-7 at 16-19 KB stages, 7.3-7.4 TB/s)
//       and DROPS by 5 % when the ring is deepened to the 227 KB that would fit (12 stages): past
//       the latency x bandwidth product more outstanding requests only lengthen the DRAM queues.
//       No registers are tied up by loads in flight.
//   consumers (W = 8 warps)      wait on `full`, read the slot with conflict-free LDS.128 (lane <->
//       16-byte column quad, warp <-> rows), accumulate in fp32 registers across all nine matrices
//       of the item, release the slot through its `empty` mbarrier, and combine partial sums ONCE
//       per item (not per matrix): warp shuffles over the column slices (dagger = 0) or a
//       shared-memory sum over the row slices (dagger = 1).
//
// dagger = 0: item = (site, row block of RS rows), 9 stages (one per matrix m); lane holds the
//             vector entries of its columns, accumulators are per row.
// dagger = 1: item = site, 9 * Nc/RS stages (matrix m of the dagger-neighbour, row chunk c);
//             rows are the contraction index, lane <-> OUTPUT columns, the vector entry of a row is
//             a shared-memory broadcast.  The same row-major layout serves both (no transposed copy).
// int16 links: a 16-byte quad holds 4 complex entries; decode is in registers, the per-matrix fp32
//             scale is folded into the (short) vector operand once per stage, never per entry.
//
// Summation order is fixed by the static schedule: results are bit-identical run to run.
#pragma once
#include "common.cuh"

namespace coarse {

struct StreamParams {
    Lat lat;
    const unsigned char* links;
    const float* scales;
    const float2* in;
    float2* out;
    int n_items;
    int stages;
    int keep_links;   // 1: the whole link field fits L2 and is re-read every apply -> do not mark it evict_first
    // GEN (parts apply, include/coarse_op.h coarse_op_apply_parts): out = alpha*Loc + beta*Hop on one parity
    const float2* in_local;   // u: operand of the local term (in = w: operand of the hopping term)
    float alpha, beta;
    int m_begin;              // 0: the X stage runs (local = X); 1: it is skipped
    int identity;             // 1: add alpha*u(x) to the result (local = identity)
    int parity;               // 0 even, 1 odd, 2 all sites
    int n_sites;              // sites in the parity set
    int gen;                  // STREAM-MR only (runtime flag there): 1 = parts apply (the 1-RHS kernels use the GEN template)
    int pdl;                  // 1: launched with programmatic stream serialization (COARSE_OPT_PDL)
    int item_begin;           // work items [item_begin, n_items): coarse_op_apply_host launches site ranges
    // dagger = 1 on a tiny lattice: split a site's contraction over its NB row chunks (item = (site, chunk)):
    // partial vectors go to `partial`, and the CTA that finishes a site's LAST chunk (split_count) adds the NB
    // partial vectors in chunk order - one launch, and the sum does not depend on which CTA that is
    int split;
    float2* partial;          // [n_sites * NB][Nc]
    unsigned int* split_count;   // [n_sites], zero between launches (the reducing CTA resets its site's counter)
    // ... or, launched as thread-block CLUSTERS of `cluster` CTAs (one site per cluster, the CTA of rank r takes the
    // chunks r, r + cluster, ..): the partial vectors meet in the shared memory of the rank-0 CTA (distributed shared
    // memory stores, one cluster barrier per site) - no global round trip, no device-scope fence, no atomic
    int cluster;
    // HV (half-precision input vectors, coarse_op_apply_hvec): `in` points at int16 (re,im) entries
    const float* vnorms;      // fp32 norm per site (nrhs = 1)
    // Half-precision OUTPUT (coarse_op_apply_hout): besides the complex64 result in `out`, the CTA takes
    // the site's norm max|component| / 32767 and writes the 16-bit fixed-point vector.  For that a CTA OWNS whole
    // sites: with several row blocks per site (dagger = 0) its work items are walked site-major (all row blocks of a
    // site in a row), the rows are kept in a small shared-memory buffer and the epilogue is CTA-local
    // (two named barriers per site; a first version with a global counter per site cost 1.7 us per item).
    short2* hout_q;           // NULL: off
    float* hout_norms;        // [V]
};

// Split dagger apply in clusters (StreamParams::cluster): ranks 1.. of a cluster store their partial vector into the rank-0
// CTA's buffer [2 site parities][STREAM_MAX_CLUSTER - 1][NC].
constexpr int STREAM_MAX_CLUSTER = 4;

constexpr int stream_pow2ceil(int v) { return v <= 1 ? 1 : v <= 2 ? 2 : v <= 4 ? 4 : v <= 8 ? 8 : v <= 16 ? 16 : 32; }
constexpr int stream_passes(int q) {
    for (int p = 1; p <= 8; ++p)
        if (q % p == 0 && q / p <= 32) return p;
    return 0;
}
// int16 links make the kernel issue-bound, so idle lanes cost time there: prefer a pass count that leaves
// a power-of-two number of quads per pass (rows of 12 / 24 / 48 quads, Nc = 48 / 96 / 192, otherwise run
// with 12 or 24 of every 16 or 32 lanes: measured 4.9-5.7 TB/s against 7.4 TB/s at Nc = 64).
constexpr int stream_passes_full(int q) {
    for (int p = 1; p <= 8; ++p)
        if (q % p == 0 && q / p <= 32 && stream_pow2ceil(q / p) == q / p) return p;
    return stream_passes(q);
}
constexpr int stream_rows_per_stage(int nc, int rowbytes, int unit, int max_bytes) {
    int best = 0;
    for (int d = unit; d <= nc; d += unit)
        if (nc % d == 0 && d * rowbytes <= max_bytes) best = d;
    return best;
}

// FINE = the small-lattice geometry (dagger = 0 only): as few rows per stage as the warp layout
// allows, so that V * NB work items still fill 148 SMs when the local volume is a few hundred
// sites or less ("additional parallelism is exposed in the matrix-vector application
// to compensate for reduction in parallelism possible by the size of the local volume alone").
// consumer warps: 8, or 6 when only a multiple of 6 warp-loads of rows divides Nc (Nc = 48 with 8 rows per load)
constexpr int stream_warps(int nc, int rowbytes, int rpl) {
    return stream_rows_per_stage(nc, rowbytes, 8 * rpl, 24576) > 0 ? 8
           : stream_rows_per_stage(nc, rowbytes, 6 * rpl, 24576) > 0 ? 6 : 8;
}

template <int NC, bool I16, bool FINE = false, bool HV = false, bool FULL = I16>
struct StreamGeom {
    static constexpr int ENTRY_BYTES = I16 ? 4 : 8;            // one complex link entry
    static constexpr int ROWBYTES = NC * ENTRY_BYTES;
    static constexpr int Q = ROWBYTES / 16;                    // 16-byte quads per row
    static constexpr int CPQ = 16 / ENTRY_BYTES;               // complex entries per quad
    static constexpr int PASSES = FULL ? stream_passes_full(Q) : stream_passes(Q);   // FULL: all 32 lanes busy
    static constexpr int QP = Q / PASSES;                      // quads per row per pass (<= 32)
    static constexpr int G = stream_pow2ceil(QP);              // lanes that share one row
    static constexpr int RPL = 32 / G;                         // rows per warp-wide load
    static constexpr int W = stream_warps(NC, ROWBYTES, RPL);  // consumer warps
    static constexpr int RS = stream_rows_per_stage(NC, ROWBYTES, W * RPL, FINE ? (W * RPL * ROWBYTES) : 24576);
    static constexpr int NB = NC / RS;                         // row blocks per matrix
    static constexpr int WL = RS / (W * RPL);                  // warp-wide loads per warp, stage, pass
    static constexpr int LINK_STAGE = RS * ROWBYTES;
    static constexpr int VEC_ENTRY = HV ? 4 : 8;               // complex64, or int16 (re,im) half vectors
    static constexpr int VEC_STAGE_N = NC * VEC_ENTRY;         // dagger = 0: whole neighbour vector
    static constexpr int VEC_STAGE_D = RS * VEC_ENTRY;         // dagger = 1: the RS entries of the chunk
    static constexpr int RED_BYTES = 2 * W * RPL * NC * 8;     // dagger = 1: double-buffered partial sums
    static constexpr bool OK = (ROWBYTES % 16 == 0) && PASSES > 0 && RS > 0 && (QP * PASSES == Q);
    static constexpr int THREADS = (W + 1) * 32;

    static constexpr int stage_bytes(bool dag) { return LINK_STAGE + (dag ? VEC_STAGE_D : VEC_STAGE_N); }
    static constexpr int SITE_BYTES = NC * 8;                  // half-precision output: the site's complex64 rows
    static constexpr int CL_BYTES = 2 * (STREAM_MAX_CLUSTER - 1) * NC * 8;   // split dagger apply in clusters (rank 0's inbox)
    static constexpr int fixed_bytes(bool dag) { return (dag ? RED_BYTES + CL_BYTES : 0) + 128 + SITE_BYTES; }
    static int smem_bytes(bool dag, int stages) { return stages * (stage_bytes(dag) + 16) + fixed_bytes(dag); }
};

// acc += M * v   (conj = false)   |   acc += conj(M) * v   (conj = true)
// Two packed FMAs (fma.rn.f32x2, SASS FFMA2, new on sm_100): acc += mre * (v.x, v.y), then
// acc += mim * (-v.y, v.x) (conj: mim * (v.y, -v.x)).  Each half is an ordinary IEEE fp32 FMA, so the
// result is the one the four scalar FMAs gave, in the same order; the instruction count of the
// kernels' inner loops - which is what bounds the int16 and multi-RHS variants - halves.
template <bool CONJ>
__device__ __forceinline__ void cmac(float2& acc, float mre, float mim, const float2 v) {
    const float2 vs = CONJ ? make_float2(v.y, -v.x) : make_float2(-v.y, v.x);
    acc = ptx::ffma2(make_float2(mre, mre), v, acc);
    acc = ptx::ffma2(make_float2(mim, mim), vs, acc);
}

// The same complex MAC with the MATRIX entry as the packed operand, for the kernels whose issue slots
// are what bounds them (int16 links, several right-hand sides).  cmac<> needs (mre, mre) and (mim, mim)
// as register pairs - two MOVs per link entry (ncu / SASS: 28 IMAD.MOV of 300 instructions per stage and
// lane in the int16 kernel, 40 of 260 with 3 right-hand sides).  Here the decoded entry (re, im) IS the
// packed operand, the duplicated pairs (v.re, v.re), (v.im, v.im) are built once per stage and reused for
// every row, and the accumulator is kept as two packed partial sums
//     a = sum (m.re, m.im) * v.re,    b = sum (m.re, m.im) * v.im
// that are combined once per item: M.v = (a.x - b.y, a.y + b.x), conj(M).v = (a.x + b.y, b.x - a.y).
struct CAcc {
    float2 a, b;
};
struct VDup {
    float2 re, im;
};
__device__ __forceinline__ VDup vdup(const float2 v) {
    VDup d;
    d.re = make_float2(v.x, v.x);
    d.im = make_float2(v.y, v.y);
    return d;
}
__device__ __forceinline__ void cmacp(CAcc& acc, const float2 m, const VDup& v) {
    acc.a = ptx::ffma2(m, v.re, acc.a);
    acc.b = ptx::ffma2(m, v.im, acc.b);
}
template <bool CONJ>
__device__ __forceinline__ float2 cfinal(const CAcc& acc) {
    return CONJ ? make_float2(acc.a.x + acc.b.y, acc.b.x - acc.a.y) : make_float2(acc.a.x - acc.b.y, acc.a.y + acc.b.x);
}

// Per-site half-precision epilogue, called by all consumer threads of the CTA that owns site s once its NC result
// entries are in `sbuf` (shared memory).  scratch: 9 words of shared memory.  The arithmetic is that of
// quantize_vec_i16_kernel (R22): norm = amax / 32767 (fp32 division), q = clamp(rint(component / norm)).
namespace ptx {
__device__ __forceinline__ uint32_t mapa_shared(uint32_t addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster_f2(uint32_t addr, float2 v) {
    asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
}  // namespace ptx

template <int NC, int NTHREADS>
__device__ __forceinline__ void half_out_epilogue(const StreamParams& p, int s, const float2* sbuf, uint32_t* scratch) {
    ptx::named_bar_sync(1, NTHREADS);                    // every row of the site is in sbuf
    float amax = 0.f;
    for (int t = threadIdx.x; t < NC; t += NTHREADS) {
        const float2 x = sbuf[t];
        amax = fmaxf(amax, fmaxf(fabsf(x.x), fabsf(x.y)));
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    if ((threadIdx.x & 31) == 0) scratch[1 + (threadIdx.x >> 5)] = __float_as_uint(amax);
    ptx::named_bar_sync(1, NTHREADS);
    amax = 0.f;
#pragma unroll
    for (int w = 0; w < NTHREADS / 32; ++w) amax = fmaxf(amax, __uint_as_float(scratch[1 + w]));
    const float norm = amax == 0.f ? 0.f : __fdiv_rn(amax, 32767.0f);
    if (threadIdx.x == 0) p.hout_norms[s] = norm;
    for (int t = threadIdx.x; t < NC; t += NTHREADS) {
        short2 o = make_short2(0, 0);
        if (amax != 0.f) {
            const float2 x = sbuf[t];
            o.x = (short)fminf(32767.f, fmaxf(-32767.f, rintf(__fdiv_rn(x.x, norm))));
            o.y = (short)fminf(32767.f, fmaxf(-32767.f, rintf(__fdiv_rn(x.y, norm))));
        }
        p.hout_q[(int64_t)s * NC + t] = o;
    }
    ptx::named_bar_sync(1, NTHREADS);                    // sbuf and scratch are reused by the next site
}

// CL: the instantiation launched as thread-block clusters (split dagger apply).  It is a separate kernel because the mere
// presence of cluster instructions (mapa, barrier.cluster) in a kernel costs ~0.9 us per launch even when they are never
// executed (measured on the 256-site C1 lattice: dagger = 1 6.4 -> 7.3 us warm with one kernel for both).
template <int NC, bool I16, bool DAG, bool FINE = false, bool GEN = false, bool HV = false, bool CL = false>
__global__ void __launch_bounds__(StreamGeom<NC, I16, FINE, HV>::THREADS, 1) coarse_apply_stream(StreamParams p) {
    static_assert(!CL || (DAG && !FINE), "cluster launches: dagger = 1 (plain apply, half-precision input, parts apply)");
    static_assert(!(DAG && FINE), "the fine geometry splits output rows: dagger = 0 only");
    static_assert(!(GEN && HV), "half-precision input vectors are implemented for the plain apply");
    using Gm = StreamGeom<NC, I16, FINE, HV>;
    constexpr int VE = Gm::VEC_ENTRY;
    constexpr int W = Gm::W, RS = Gm::RS, NB = Gm::NB, WL = Gm::WL, QP = Gm::QP, G = Gm::G, RPL = Gm::RPL;
    constexpr int PASSES = Gm::PASSES, CPQ = Gm::CPQ, ROWBYTES = Gm::ROWBYTES;
    constexpr int LINK_STAGE = Gm::LINK_STAGE;
    constexpr int VEC_STAGE = DAG ? Gm::VEC_STAGE_D : Gm::VEC_STAGE_N;

    extern __shared__ __align__(128) unsigned char smem[];
    const int S = p.stages;
    unsigned char* link_smem = smem;
    unsigned char* vec_smem = link_smem + (size_t)S * LINK_STAGE;
    unsigned char* red_smem = vec_smem + (size_t)S * VEC_STAGE;
    uint64_t* bars = reinterpret_cast<uint64_t*>(red_smem + (DAG ? Gm::RED_BYTES : 0));
    const uint32_t full0 = ptx::smem_u32(bars);
    const uint32_t empty0 = full0 + 8u * S;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int i = 0; i < S; ++i) {
            ptx::mbar_init(full0 + 8u * i, 1);
            ptx::mbar_init(empty0 + 8u * i, W);
        }
        ptx::fence_mbar_init();
    }
    __syncthreads();
    if (p.pdl) ptx::pdl_launch_dependents();   // the next kernel's CTAs may take SMs as ours exit

    // The it-th work item of this CTA.  Default: items blockIdx.x, blockIdx.x + gridDim.x, ...  Half-precision output
    // with several row blocks per site: site-major, the NB items of a site in a row (the CTA owns the site).
    const bool site_major = !DAG && NB > 1 && p.hout_q != nullptr;
    // cluster mode (split dagger apply): the CTAs of a cluster share their work items (sites); rank r takes the chunks r, r + CR, ..
    const int CR = CL ? p.cluster : 0;
    const int crank = CR ? (int)blockIdx.x % CR : 0;
    auto item_at = [&](int it) -> int {
        if (site_major) return p.item_begin + ((int)blockIdx.x + (it / NB) * (int)gridDim.x) * NB + it % NB;
        if (CR) return p.item_begin + (int)blockIdx.x / CR + it * ((int)gridDim.x / CR);
        return p.item_begin + (int)blockIdx.x + it * (int)gridDim.x;
    };

    if (warp == W) {
        // ------------------------------------------------------------------ producer
        // The whole warp walks the loop (uniform control flow, so the bulk copies are not wrapped
        // in per-lane replay loops) and one elected lane issues the copies.
        const uint64_t pol_vec = ptx::policy_evict_last();
        const uint64_t pol_links = p.keep_links ? pol_vec : ptx::policy_evict_first();
        const uint32_t link_u32 = ptx::smem_u32(link_smem), vec_u32 = ptx::smem_u32(vec_smem);
        int slot = 0;
        uint32_t phase = 0;
        // PDL: the links do not depend on the previous kernel of the stream, the vectors do.  The first S
        // stages' LINK copies go out at once (they overlap the previous kernel's tail), their vector copies
        // are queued; griddepcontrol.wait then makes the previous kernel's output visible and the queue
        // is flushed.  Every store of this kernel comes after a vector copy, hence after the wait.
        bool cl_pending = false;
        bool deferring = p.pdl != 0;
        int n_def = 0;
        const unsigned char* def_src[12];
        auto flush_deferred = [&]() {
            ptx::pdl_wait();
            if (ptx::elect_one())
                for (int q = 0; q < n_def; ++q)
                    ptx::bulk_g2s(vec_u32 + q * VEC_STAGE, def_src[q], VEC_STAGE, full0 + 8u * q, pol_vec);
            __syncwarp();
            deferring = false;
        };
        for (int it = 0;; ++it) {
            const int item = item_at(it);
            if (item >= p.n_items) break;
            const int sidx = (DAG && !p.split) ? item : item / NB;
            const int s = (GEN && p.parity != 2) ? parity_site(p.lat, sidx, p.parity) : sidx;
            const int rb = DAG ? 0 : item % NB;
            const SiteX cx = site_coords(p.lat, s);
#pragma unroll
            for (int m = 0; m < 9; ++m) {
                if (GEN && m < p.m_begin) continue;
                const int sv = stencil_site_x(p.lat, s, cx, m, DAG ? 1 : 0);
                const int sm = DAG ? sv : s;
                const unsigned char* mat = p.links + ((int64_t)sm * 9 + m) * ((int64_t)NC * ROWBYTES);
                const unsigned char* vec = reinterpret_cast<const unsigned char*>((GEN && m == 0) ? p.in_local : p.in) + (int64_t)sv * NC * VE;
                const int c_begin = (DAG && p.split) ? item % NB : crank;
                const int c_end = DAG ? (p.split ? c_begin + 1 : NB) : 1;
                const int c_step = CR ? CR : 1;
#pragma unroll 1
                for (int c = c_begin; c < c_end; c += c_step) {
                    const int r0 = DAG ? c * RS : rb * RS;
                    if (deferring && n_def == S) flush_deferred();    // the ring is full: the vectors are needed now
                    ptx::mbar_wait(empty0 + 8u * slot, phase ^ 1u);
                    const unsigned char* vsrc = DAG ? (vec + r0 * VE) : vec;
                    if (ptx::elect_one()) {
                        ptx::mbar_arrive_expect_tx(full0 + 8u * slot, LINK_STAGE + VEC_STAGE);
                        ptx::bulk_g2s(link_u32 + slot * LINK_STAGE, mat + (int64_t)r0 * ROWBYTES, LINK_STAGE,
                                      full0 + 8u * slot, pol_links);
                        if (!deferring)
                            ptx::bulk_g2s(vec_u32 + slot * VEC_STAGE, vsrc, VEC_STAGE, full0 + 8u * slot, pol_vec);
                    }
                    if (deferring) def_src[n_def++] = vsrc;            // slot index = position in the queue
                    __syncwarp();
                    if (++slot == S) { slot = 0; phase ^= 1u; }
                }
            }
            if (CR) {
                // the site's cluster barrier counts every thread of the cluster.  The producer ARRIVES once the site's last
                // stage is issued (queued vector copies must be out first, the consumers are waiting for them) and goes on
                // with the next site's stages; it completes the barrier (wait) only before its next arrival, so the ring
                // does not drain at site boundaries
                if (deferring) flush_deferred();
                if (cl_pending) ptx::cluster_wait();
                ptx::cluster_arrive();
                cl_pending = true;
            }
        }
        if (deferring) flush_deferred();
        if (cl_pending) ptx::cluster_wait();
        return;
    }

    // ---------------------------------------------------------------------- consumers
    if ((GEN || HV) && p.pdl) ptx::pdl_wait();      // these variants read the input from global memory themselves
    const int grp = lane / G;          // which of the RPL rows of a warp-wide load
    const int qi = lane % G;           // quad index inside the pass
    const bool active = qi < QP;
    const uint32_t link_u32 = ptx::smem_u32(link_smem), vec_u32 = ptx::smem_u32(vec_smem);
    int slot = 0;
    uint32_t phase = 0;
    int red_parity = 0;

    // int16: lane m (< 9) carries the fp32 scale of matrix m of the current item.  The scales are
    // fetched TWO items ahead: under a saturated HBM a DRAM miss takes about as long as a whole
    // item (~3 us), and with a one-item lead ncu showed 12 % of the dagger = 1 samples waiting on it.
    float cur_scale = 1.f, next_scale = 1.f, next2_scale = 1.f;
    auto site_of = [&](int item) -> int {
        const int sidx = (DAG && !p.split) ? item : item / NB;
        return (GEN && p.parity != 2) ? parity_site(p.lat, sidx, p.parity) : sidx;
    };
    auto fetch_scale = [&](int item) -> float {
        if (!(I16 || HV) || lane >= 9 || item >= p.n_items) return 1.f;
        const int s = site_of(item);
        const int sv = stencil_site(p.lat, s, lane, DAG ? 1 : 0);   // site of stage `lane`'s vector
        const int sm = DAG ? sv : s;                                 // site of its link matrix
        float f = 1.f;
        if constexpr (I16) f = __ldg(p.scales + (int64_t)sm * 9 + lane);
        if constexpr (HV) f *= __ldg(p.vnorms + sv);                 // half vectors: per-site norm folded in
        return f;
    };
    const int M0 = GEN ? p.m_begin : 0;
    next_scale = fetch_scale(item_at(0));
    next2_scale = fetch_scale(item_at(1));
    float2* sbuf = reinterpret_cast<float2*>(reinterpret_cast<unsigned char*>(bars + 2 * S) + 128);     // half-precision output
    uint32_t* hscratch = reinterpret_cast<uint32_t*>(bars + 2 * S);
    // cluster mode: rank 0's inbox [2][STREAM_MAX_CLUSTER - 1][NC] behind the half-output buffer; the other ranks address it
    // through the cluster's shared-memory window
    static_assert(NC <= W * 32, "cluster mode: one output column per consumer thread");
    float2* cl_buf = reinterpret_cast<float2*>(reinterpret_cast<unsigned char*>(bars + 2 * S) + 128 + Gm::SITE_BYTES);
    const uint32_t cl_inbox = CR ? ptx::mapa_shared(ptx::smem_u32(cl_buf), 0u) : 0u;
    float2 cl_keep = make_float2(0.f, 0.f);

    for (int it = 0;; ++it) {
        const int item = item_at(it);
        if (item >= p.n_items) break;
        const int s = site_of(item);
        const int rb = DAG ? 0 : item % NB;
        cur_scale = next_scale;
        next_scale = next2_scale;
        next2_scale = fetch_scale(item_at(it + 2));

        if (!DAG) {
            float2 acc[WL];
#pragma unroll
            for (int k = 0; k < WL; ++k) acc[k] = make_float2(0.f, 0.f);
            // identity local term: fetch u(x) for this lane's rows now, so that the L2 latency hides
            // behind the item's stages instead of stalling the warp in front of the store
            float2 uloc[GEN ? WL : 1];
            if constexpr (GEN) {
#pragma unroll
                for (int k = 0; k < WL; ++k)
                    uloc[k] = p.identity ? __ldg(p.in_local + (int64_t)s * NC + rb * RS + (k * W + warp) * RPL + grp)
                                         : make_float2(0.f, 0.f);
            }
#pragma unroll 1
            for (int m = M0; m < 9; ++m) {
                float sc = (I16 || HV) ? __shfl_sync(0xffffffffu, cur_scale, m) : 1.f;
                if constexpr (GEN) sc *= (m == 0) ? p.alpha : p.beta;
                ptx::mbar_wait(full0 + 8u * slot, phase);
                const uint32_t lbase = link_u32 + slot * LINK_STAGE + qi * 16;
                const uint32_t vbase = vec_u32 + slot * VEC_STAGE;
                float2 v[PASSES][CPQ];
                if (active) {
#pragma unroll
                    for (int ps = 0; ps < PASSES; ++ps) {
                        const int col0 = (ps * QP + qi) * CPQ;
                        if constexpr (HV) {
                            if constexpr (CPQ == 2) {
                                const float2 t = ptx::lds64(vbase + col0 * 4);
                                v[ps][0] = unpack_i16x2(__float_as_uint(t.x));
                                v[ps][1] = unpack_i16x2(__float_as_uint(t.y));
                            } else {
                                const uint4 t = ptx::lds128u(vbase + col0 * 4);
                                v[ps][0] = unpack_i16x2(t.x);
                                v[ps][1] = unpack_i16x2(t.y);
                                v[ps][2] = unpack_i16x2(t.z);
                                v[ps][3] = unpack_i16x2(t.w);
                            }
                        } else {
#pragma unroll
                            for (int h = 0; h < CPQ / 2; ++h) {
                                const float4 t = ptx::lds128(vbase + (col0 + 2 * h) * 8);
                                v[ps][2 * h] = make_float2(t.x, t.y);
                                v[ps][2 * h + 1] = make_float2(t.z, t.w);
                            }
                        }
                        if constexpr (I16 || GEN || HV) {
#pragma unroll
                            for (int e = 0; e < CPQ; ++e) { v[ps][e].x *= sc; v[ps][e].y *= sc; }
                        }
                    }
#pragma unroll
                    for (int k = 0; k < WL; ++k) {
                        const int rl = (k * W + warp) * RPL + grp;
#pragma unroll
                        for (int ps = 0; ps < PASSES; ++ps) {
                            const uint32_t a = lbase + rl * ROWBYTES + ps * QP * 16;
                            if constexpr (I16) {
                                const uint4 t = ptx::lds128u(a);
                                float2 m0, m1, m2, m3;
                                unpack_i16_quad<2>(t, m0, m1, m2, m3);
                                cmac<false>(acc[k], m0.x, m0.y, v[ps][0]);
                                cmac<false>(acc[k], m1.x, m1.y, v[ps][1]);
                                cmac<false>(acc[k], m2.x, m2.y, v[ps][2]);
                                cmac<false>(acc[k], m3.x, m3.y, v[ps][3]);
                            } else {
                                const float4 t = ptx::lds128(a);
                                cmac<false>(acc[k], t.x, t.y, v[ps][0]);
                                cmac<false>(acc[k], t.z, t.w, v[ps][1]);
                            }
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
                if (++slot == S) { slot = 0; phase ^= 1u; }
            }
            // a6: combine the column-slice partial sums, once per item
#pragma unroll
            for (int k = 0; k < WL; ++k) {
#pragma unroll
                for (int o = G / 2; o > 0; o >>= 1) {
                    acc[k].x += __shfl_xor_sync(0xffffffffu, acc[k].x, o);
                    acc[k].y += __shfl_xor_sync(0xffffffffu, acc[k].y, o);
                }
                if (qi == 0) {
                    const int row = rb * RS + (k * W + warp) * RPL + grp;
                    if constexpr (GEN) {
                        acc[k].x = fmaf(p.alpha, uloc[k].x, acc[k].x);
                        acc[k].y = fmaf(p.alpha, uloc[k].y, acc[k].y);
                    }
                    p.out[(int64_t)s * NC + row] = acc[k];
                    if (p.hout_q) sbuf[row] = acc[k];
                }
            }
            if (p.hout_q && rb == NB - 1) half_out_epilogue<NC, W * 32>(p, s, sbuf, hscratch);
        } else {
            constexpr int UL = (NC + W * 32 - 1) / (W * 32);
            float2 uloc[GEN ? UL : 1];
            if constexpr (GEN) {
#pragma unroll
                for (int k = 0; k < UL; ++k) {
                    const int t = threadIdx.x + k * W * 32;
                    uloc[k] = (p.identity && t < NC) ? __ldg(p.in_local + (int64_t)s * NC + t) : make_float2(0.f, 0.f);
                }
            }
            float2 acc[PASSES][CPQ];
#pragma unroll
            for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
                for (int e = 0; e < CPQ; ++e) acc[ps][e] = make_float2(0.f, 0.f);
#pragma unroll 1
            for (int m = M0; m < 9; ++m) {
                float sc = (I16 || HV) ? __shfl_sync(0xffffffffu, cur_scale, m) : 1.f;
                if constexpr (GEN) sc *= (m == 0) ? p.alpha : p.beta;
#pragma unroll 1
                for (int c = p.split ? item % NB : crank; c < (p.split ? item % NB + 1 : NB); c += (CR ? CR : 1)) {
                    ptx::mbar_wait(full0 + 8u * slot, phase);
                    const uint32_t lbase = link_u32 + slot * LINK_STAGE + qi * 16;
                    const uint32_t vbase = vec_u32 + slot * VEC_STAGE;
                    if (active) {
#pragma unroll
                        for (int k = 0; k < WL; ++k) {
                            const int rl = (k * W + warp) * RPL + grp;
                            float2 vj;
                            if constexpr (HV) {
                                uint32_t w;
                                asm volatile("ld.shared.u32 %0, [%1];" : "=r"(w) : "r"(vbase + rl * 4));
                                vj = unpack_i16x2(w);
                            } else {
                                vj = ptx::lds64(vbase + rl * 8);
                            }
                            if constexpr (I16 || GEN || HV) { vj.x *= sc; vj.y *= sc; }
#pragma unroll
                            for (int ps = 0; ps < PASSES; ++ps) {
                                const uint32_t a = lbase + rl * ROWBYTES + ps * QP * 16;
                                if constexpr (I16) {
                                    const uint4 t = ptx::lds128u(a);
                                    float2 m0, m1, m2, m3;
                                    unpack_i16_quad<1>(t, m0, m1, m2, m3);
                                    cmac<true>(acc[ps][0], m0.x, m0.y, vj);
                                    cmac<true>(acc[ps][1], m1.x, m1.y, vj);
                                    cmac<true>(acc[ps][2], m2.x, m2.y, vj);
                                    cmac<true>(acc[ps][3], m3.x, m3.y, vj);
                                } else {
                                    const float4 t = ptx::lds128(a);
                                    cmac<true>(acc[ps][0], t.x, t.y, vj);
                                    cmac<true>(acc[ps][1], t.z, t.w, vj);
                                }
                            }
                        }
                    }
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
                    if (++slot == S) { slot = 0; phase ^= 1u; }
                }
            }
            // a6: combine the row-slice partial sums (W warps x RPL row groups), once per item
            float2* red = reinterpret_cast<float2*>(red_smem) + red_parity * (W * RPL * NC);
            if (active) {
#pragma unroll
                for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
                    for (int e = 0; e < CPQ; ++e)
                        red[(warp * RPL + grp) * NC + (ps * QP + qi) * CPQ + e] = acc[ps][e];
            }
            ptx::named_bar_sync(1, W * 32);
            for (int t = threadIdx.x, ku = 0; t < NC; t += W * 32, ++ku) {
                float2 sum = make_float2(0.f, 0.f);
#pragma unroll
                for (int g = 0; g < W * RPL; ++g) {
                    const float2 x = red[g * NC + t];
                    sum.x += x.x;
                    sum.y += x.y;
                }
                if constexpr (GEN) {
                    if (crank == 0) {                                  // (cluster mode: the identity term once per site)
                        sum.x = fmaf(p.alpha, uloc[(GEN && UL > 1) ? ku : 0].x, sum.x);
                        sum.y = fmaf(p.alpha, uloc[(GEN && UL > 1) ? ku : 0].y, sum.y);
                    }
                }
                if (CR) {
                    // ranks 1.. send their partial sum to the rank-0 CTA's inbox (distributed shared memory); rank 0 keeps its
                    // own in a register and adds the others, in rank order, behind the site's cluster barrier
                    if (crank) ptx::st_cluster_f2(cl_inbox + (uint32_t)(((it & 1) * (STREAM_MAX_CLUSTER - 1) + crank - 1) * NC + t) * 8u, sum);
                    else cl_keep = sum;
                } else if (p.split) p.partial[(int64_t)item * NC + t] = sum;
                else p.out[(int64_t)s * NC + t] = sum;
                if (p.hout_q) sbuf[t] = sum;
            }
            if (CR) {
                ptx::cluster_sync_all();
                if (crank == 0 && threadIdx.x < NC) {
                    float2 sum = cl_keep;
                    for (int r = 1; r < CR; ++r) {
                        const float2 x = cl_buf[((it & 1) * (STREAM_MAX_CLUSTER - 1) + r - 1) * NC + threadIdx.x];
                        sum.x += x.x;
                        sum.y += x.y;
                    }
                    p.out[(int64_t)s * NC + threadIdx.x] = sum;
                }
            }
            if (p.split) {
                // last-arriver reduction: every consumer thread publishes its part of the partial vector, one
                // thread counts the chunk in; the CTA that counted the NB-th chunk of the site sums all of them
                uint32_t* last_flag = reinterpret_cast<uint32_t*>(bars + 2 * S);
                __threadfence();
                ptx::named_bar_sync(1, W * 32);
                if (threadIdx.x == 0) {
                    const unsigned int old = atomicAdd(p.split_count + s, 1u);
                    *last_flag = (old == (unsigned int)(NB - 1)) ? 1u : 0u;
                    if (old == (unsigned int)(NB - 1)) p.split_count[s] = 0u;      // all NB arrivals are in: reset for the next launch
                }
                ptx::named_bar_sync(1, W * 32);
                if (*last_flag) {
                    __threadfence();
                    for (int t = threadIdx.x; t < NC; t += W * 32) {
                        float2 sum = make_float2(0.f, 0.f);
                        for (int c = 0; c < NB; ++c) {
                            const float2 x = __ldcg(p.partial + ((int64_t)s * NB + c) * NC + t);
                            sum.x += x.x;
                            sum.y += x.y;
                        }
                        p.out[(int64_t)s * NC + t] = sum;
                    }
                }
            }
            if (p.hout_q) half_out_epilogue<NC, W * 32>(p, s, sbuf, hscratch);
            red_parity ^= 1;
        }
    }
}

}  // namespace coarse
