// block_kernel.cuh — COARSE_PATH_BLOCK: the multi-RHS (block) coarse-op apply on the CUDA cores
// (the comparison arm north_star (4) asks the tensor path to beat, and the
// path for the shapes the tensor kernel does not cover: int16 links, nrhs not in {8,16},
// Nc in {32,96,192}; a propagator is 3 right-hand sides).
//
// Per site the block apply is out[Nc x R] = sum_m M_m[Nc x Nc] . in_m[Nc x R].  The link stream is
// the same as in stream_kernel.cuh (persistent CTA per SM, one elected producer lane issuing 1-D TMA
// bulk copies into a shared-memory ring, evict_first links / evict_last vectors); what changes is
// the register tile.  With the vectors stored RHS-innermost (v[s][a][r]) the natural mapping is
//
//     lane  <->  (right-hand side r, contraction subset)          RP lanes per subset, RP = 8 | 16
//
// so that a vector load is one contiguous 8 RP-byte row (conflict-free) and a link load is a
// shared-memory BROADCAST (all RP lanes of a subset read the same entries).
//
// dagger = 0: item = (site, block of RS <= 16 rows), 9 stages.  The W.KS subsets split the columns
//   (the contraction index); every thread keeps acc[RS] for its r, reads 2 vector entries and RS
//   broadcast 16-byte link quads per column pair (8 RS FMAs), and the subsets' partial sums are
//   combined ONCE per item through shared memory (row a6).
// dagger = 1: item = site, 9 Nc/RS stages of RS full rows (rows are the contraction index).  The
//   subsets split the OUTPUT columns: acc[KPT] per thread, no cross-thread reduction at all.
// int16 links: decoded in registers, the per-matrix scale folded into the vector entries.
// nrhs < RP: the surplus lanes compute on a clamped r and do not store.
// Summation order is fixed by the static schedule: bit-identical run to run.
#pragma once
#include "common.cuh"
#include "stream_kernel.cuh"   // cmac<>

namespace coarse {

struct BlockParams {
    Lat lat;
    const unsigned char* links;
    const float* scales;
    const float2* in;
    float2* out;
    int n_items;
    int stages;
    int nrhs;
    int keep_links;
};

constexpr int block_rows_per_stage(int nc, int rowbytes) {
    int best = 1;
    for (int d = 1; d <= 16; ++d)
        if (nc % d == 0 && d * rowbytes <= 24576) best = d;
    return best;
}

template <int NC, bool I16, int RP>
struct BlockGeom {
    static constexpr int W = (NC % 3 == 0) ? 6 : 8;           // consumer warps
    static constexpr int KS = 32 / RP;                         // subsets per warp
    static constexpr int NSUB = W * KS;
    static constexpr int KPT = NC / NSUB;                      // columns per subset
    static constexpr int ENTRY_BYTES = I16 ? 4 : 8;
    static constexpr int ROWBYTES = NC * ENTRY_BYTES;
    static constexpr int RS = block_rows_per_stage(NC, ROWBYTES);
    static constexpr int NB = NC / RS;
    static constexpr int LINK_STAGE = RS * ROWBYTES;
    static constexpr int RED_BYTES = NSUB * RS * RP * 8;       // dagger = 0 only
    static constexpr int THREADS = (W + 1) * 32;
    static constexpr bool OK = (RP == 8 || RP == 16) && (NC % NSUB == 0) && KPT >= 1 && (LINK_STAGE % 16 == 0);

    static int vec_stage(bool dag, int nrhs) { return (dag ? RS : NC) * nrhs * 8; }
    static int stage_bytes(bool dag, int nrhs) { return LINK_STAGE + vec_stage(dag, nrhs); }
    static int fixed_bytes(bool dag) { return (dag ? 0 : RED_BYTES) + 128; }
    static int smem_bytes(bool dag, int nrhs, int stages) { return stages * (stage_bytes(dag, nrhs) + 16) + fixed_bytes(dag); }
};

namespace ptx {
__device__ __forceinline__ uint2 lds64u(uint32_t addr) {
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint32_t lds32u(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}
}  // namespace ptx

// Load the link entries of columns [col, col+N) of one shared-memory row (N = 1 or 2) as floats.
template <bool I16, int N>
__device__ __forceinline__ void block_load_entries(uint32_t addr, float2 (&m)[2]) {
    if constexpr (I16) {
        if constexpr (N == 2) {
            const uint2 t = ptx::lds64u(addr);
            m[0] = unpack_i16x2(t.x);
            m[1] = unpack_i16x2(t.y);
        } else {
            m[0] = unpack_i16x2(ptx::lds32u(addr));
        }
    } else {
        if constexpr (N == 2) {
            const float4 t = ptx::lds128(addr);
            m[0] = make_float2(t.x, t.y);
            m[1] = make_float2(t.z, t.w);
        } else {
            m[0] = ptx::lds64(addr);
        }
    }
}

template <int NC, bool I16, bool DAG, int RP>
__global__ void __launch_bounds__(BlockGeom<NC, I16, RP>::THREADS, 1) coarse_apply_block(BlockParams p) {
    using Gm = BlockGeom<NC, I16, RP>;
    static_assert(Gm::OK, "unsupported BLOCK geometry");
    constexpr int W = Gm::W, KS = Gm::KS, KPT = Gm::KPT, RS = Gm::RS, NB = Gm::NB;
    constexpr int ROWBYTES = Gm::ROWBYTES, LINK_STAGE = Gm::LINK_STAGE, EB = Gm::ENTRY_BYTES;
    constexpr int STEP = (KPT % 2 == 0) ? 2 : 1;               // columns per link load

    extern __shared__ __align__(128) unsigned char smem[];
    const int S = p.stages;
    const int R = p.nrhs;
    const int VEC_STAGE = (DAG ? RS : NC) * R * 8;
    unsigned char* link_smem = smem;
    unsigned char* vec_smem = link_smem + (size_t)S * LINK_STAGE;
    unsigned char* red_smem = vec_smem + (size_t)S * VEC_STAGE;
    uint64_t* bars = reinterpret_cast<uint64_t*>(red_smem + (DAG ? 0 : Gm::RED_BYTES));
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

    if (warp == W) {
        // ------------------------------------------------------------------ producer
        const uint64_t pol_vec = ptx::policy_evict_last();
        const uint64_t pol_links = p.keep_links ? pol_vec : ptx::policy_evict_first();
        const uint32_t link_u32 = ptx::smem_u32(link_smem), vec_u32 = ptx::smem_u32(vec_smem);
        int slot = 0;
        uint32_t phase = 0;
        for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
            const int s = DAG ? item : item / NB;
            const int rb = DAG ? 0 : item % NB;
            const SiteX cx = site_coords(p.lat, s);
#pragma unroll
            for (int m = 0; m < 9; ++m) {
                const int sv = stencil_site_x(p.lat, s, cx, m, DAG ? 1 : 0);
                const int sm = DAG ? sv : s;
                const unsigned char* mat = p.links + ((int64_t)sm * 9 + m) * ((int64_t)NC * ROWBYTES);
                const float2* vec = p.in + (int64_t)sv * NC * R;
#pragma unroll 1
                for (int c = 0; c < (DAG ? NB : 1); ++c) {
                    const int r0 = DAG ? c * RS : rb * RS;
                    ptx::mbar_wait(empty0 + 8u * slot, phase ^ 1u);
                    if (ptx::elect_one()) {
                        ptx::mbar_arrive_expect_tx(full0 + 8u * slot, LINK_STAGE + VEC_STAGE);
                        ptx::bulk_g2s(link_u32 + slot * LINK_STAGE, mat + (int64_t)r0 * ROWBYTES, LINK_STAGE,
                                      full0 + 8u * slot, pol_links);
                        ptx::bulk_g2s(vec_u32 + slot * VEC_STAGE, DAG ? (vec + (int64_t)r0 * R) : vec, VEC_STAGE,
                                      full0 + 8u * slot, pol_vec);
                    }
                    __syncwarp();
                    if (++slot == S) { slot = 0; phase ^= 1u; }
                }
            }
        }
        return;
    }

    // ---------------------------------------------------------------------- consumers
    const int r = lane % RP;                      // right-hand side of this lane
    const int rr = r < R ? r : R - 1;             // clamped: surplus lanes recompute the last RHS
    const int sub = warp * KS + lane / RP;        // contraction (dagger 0) / output-column (dagger 1) subset
    const int c0 = sub * KPT;                     // first column of the subset
    const uint32_t link_u32 = ptx::smem_u32(link_smem), vec_u32 = ptx::smem_u32(vec_smem);
    int slot = 0;
    uint32_t phase = 0;

    float cur_scale = 1.f, next_scale = 1.f, next2_scale = 1.f;
    auto fetch_scale = [&](int item) -> float {
        if (!I16 || lane >= 9 || item >= p.n_items) return 1.f;
        const int s = DAG ? item : item / NB;
        const int sm = DAG ? stencil_site(p.lat, s, lane, 1) : s;
        return __ldg(p.scales + (int64_t)sm * 9 + lane);
    };
    next_scale = fetch_scale(blockIdx.x);
    next2_scale = fetch_scale(blockIdx.x + gridDim.x);

    for (int item = blockIdx.x; item < p.n_items; item += gridDim.x) {
        const int s = DAG ? item : item / NB;
        const int rb = DAG ? 0 : item % NB;
        cur_scale = next_scale;
        next_scale = next2_scale;
        next2_scale = fetch_scale(item + 2 * gridDim.x);

        if (!DAG) {
            float2 acc[RS];
#pragma unroll
            for (int t = 0; t < RS; ++t) acc[t] = make_float2(0.f, 0.f);
#pragma unroll 1
            for (int m = 0; m < 9; ++m) {
                const float sc = I16 ? __shfl_sync(0xffffffffu, cur_scale, m) : 1.f;
                ptx::mbar_wait(full0 + 8u * slot, phase);
                const uint32_t lbase = link_u32 + slot * LINK_STAGE + c0 * EB;
                const uint32_t vbase = vec_u32 + slot * VEC_STAGE + (c0 * R + rr) * 8;
#pragma unroll
                for (int k = 0; k < KPT; k += STEP) {
                    float2 v[2];
#pragma unroll
                    for (int e = 0; e < STEP; ++e) {
                        v[e] = ptx::lds64(vbase + (k + e) * R * 8);
                        if constexpr (I16) { v[e].x *= sc; v[e].y *= sc; }
                    }
#pragma unroll
                    for (int t = 0; t < RS; ++t) {
                        float2 mm[2];
                        block_load_entries<I16, STEP>(lbase + t * ROWBYTES + k * EB, mm);
#pragma unroll
                        for (int e = 0; e < STEP; ++e) cmac<false>(acc[t], mm[e].x, mm[e].y, v[e]);
                    }
                }
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
                if (++slot == S) { slot = 0; phase ^= 1u; }
            }
            // a6: combine the column-subset partial sums through shared memory, once per item
            float2* red = reinterpret_cast<float2*>(red_smem);
#pragma unroll
            for (int t = 0; t < RS; ++t) red[(sub * RS + t) * RP + r] = acc[t];
            ptx::named_bar_sync(1, W * 32);
            for (int idx = threadIdx.x; idx < RS * RP; idx += W * 32) {
                const int t = idx / RP, ro = idx % RP;
                float2 sum = make_float2(0.f, 0.f);
#pragma unroll 4
                for (int g = 0; g < Gm::NSUB; ++g) {
                    const float2 x = red[(g * RS + t) * RP + ro];
                    sum.x += x.x;
                    sum.y += x.y;
                }
                if (ro < R) p.out[((int64_t)s * NC + rb * RS + t) * R + ro] = sum;
            }
            ptx::named_bar_sync(1, W * 32);
        } else {
            float2 acc[KPT];
#pragma unroll
            for (int j = 0; j < KPT; ++j) acc[j] = make_float2(0.f, 0.f);
#pragma unroll 1
            for (int m = 0; m < 9; ++m) {
                const float sc = I16 ? __shfl_sync(0xffffffffu, cur_scale, m) : 1.f;
#pragma unroll 1
                for (int c = 0; c < NB; ++c) {
                    ptx::mbar_wait(full0 + 8u * slot, phase);
                    const uint32_t lbase = link_u32 + slot * LINK_STAGE + c0 * EB;
                    const uint32_t vbase = vec_u32 + slot * VEC_STAGE + rr * 8;
#pragma unroll
                    for (int i = 0; i < RS; ++i) {
                        float2 vi = ptx::lds64(vbase + i * R * 8);
                        if constexpr (I16) { vi.x *= sc; vi.y *= sc; }
#pragma unroll
                        for (int j = 0; j < KPT; j += STEP) {
                            float2 mm[2];
                            block_load_entries<I16, STEP>(lbase + i * ROWBYTES + j * EB, mm);
#pragma unroll
                            for (int e = 0; e < STEP; ++e) cmac<true>(acc[j + e], mm[e].x, mm[e].y, vi);
                        }
                    }
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
                    if (++slot == S) { slot = 0; phase ^= 1u; }
                }
            }
            if (r < R) {
#pragma unroll
                for (int j = 0; j < KPT; ++j) p.out[((int64_t)s * NC + c0 + j) * R + r] = acc[j];
            }
        }
    }
}

}  // namespace coarse
