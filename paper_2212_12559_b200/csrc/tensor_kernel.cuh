// tensor_kernel.cuh — COARSE_PATH_TENSOR: the block (multi-RHS) coarse-op apply on the tcgen05
// tensor cores, error-compensated 3xTF32.
//
// Per site the block apply is a complex GEMM  out[Nc x nrhs] = [X Y...][Nc x 9Nc] . in[9Nc x nrhs].
// A row-major interleaved-complex link matrix IS a real M = Nc x K = 2Nc operand as stored:
//   A[i][2j] = Re M_ij, A[i][2j+1] = Im M_ij.  The vectors become a real K x N = 2Nc x 2nrhs
//   operand B = [B1 | B2],   B1[2j][r] = Re v_jr, B1[2j+1][r] = -Im v_jr   (-> Re out)
//                            B2[2j][r] = Im v_jr, B2[2j+1][r] =  Re v_jr   (-> Im out)
// (dagger: A[i][2j] = Re M_ji, A[i][2j+1] = Im M_ji, B1 = (Re v, Im v), B2 = (Im v, -Re v)).
// TF32 keeps 10 mantissa bits, so each fp32 operand is split x = hi + lo (hi = x with the low 13
// mantissa bits cleared, lo = x - hi, exact) and the product is hi.hi + hi.lo + lo.hi in fp32
// accumulators: relative error ~2^-21 per term instead of 2^-11.
//
// Since the split has to touch every link entry with CUDA threads anyway, the kernel is a
// four-role pipeline per SM (persistent, one CTA per SM, items = sites):
//   producer (1 thread)     TMA: per stage one 16-complex-column slab of a link matrix
//                           (dagger 0: 2-D tensor-map box Nc rows x 128 B, SWIZZLE_128B, so that
//                            "lane = row" reads are bank-conflict free; dagger 1: 16 full rows, one
//                            contiguous bulk copy) + the matching 16 x nrhs vector entries.
//   converters (2 x 4 warps) read the slab (lane <-> matrix row for dagger 0, lane <-> matrix
//                           column for dagger 1: TMEM transposes for free), split hi/lo and write
//                           the A operand straight into TENSOR MEMORY (tcgen05.st), so the link
//                           bytes cross shared memory exactly twice (TMA write + one LDS read);
//                           build B hi/lo in shared memory in the canonical K-major UMMA layout.
//   MMA issuer (1 thread)   tcgen05.mma kind::tf32, A from TMEM, B from smem, D (128 x 2nrhs fp32)
//                           in TMEM, 8 MMAs per stage (4 k-steps x {A_hi.[B_hi|B_lo], A_lo.B_hi}), one accumulator
//                           slot per link matrix; tcgen05.commit releases the operand slot / publishes D.
//   epilogue (4 warps)      tcgen05.ld D -> registers, adds the nine per-matrix partial results in
//                           round-to-nearest fp32 -> out[s][i][r]; a ring of 4 accumulator slots lets
//                           the next matrices' MMAs overlap the read-out.
// Summation order is fixed: results are bit-identical run to run.
#pragma once
#include <cuda.h>

#include "common.cuh"

namespace coarse {

struct TensorParams {
    Lat lat;
    const unsigned char* links;
    const float2* in;
    float2* out;
    int n_sites;
};

template <int NC, int NRHS>
struct TensorGeom {
    static constexpr int KSTAGE = 32;                   // real k per stage = 16 complex columns
    static constexpr int CHUNKS = 2 * NC / KSTAGE;      // stages per link matrix
    static constexpr int LINK_STAGE = NC * 128;         // bytes per stage (both dagger modes)
    static constexpr int VEC_STAGE = 16 * NRHS * 8;
    static constexpr int N = 2 * NRHS;                  // MMA N: [Re out | Im out]
    static constexpr int B_HALF = KSTAGE * N * 4;       // B hi (or lo) bytes per stage
    static constexpr int B_SBO = (KSTAGE / 4) * 128;    // byte stride between 8-column groups of n
    static constexpr int LS = 8;                        // link ring depth (TMA -> converters)
    static constexpr int AS = 4;                        // operand ring depth (converters -> MMA)
    static constexpr int A_COLS = 2 * KSTAGE;           // TMEM columns per operand stage: hi | lo
    static constexpr int D_COL0 = AS * A_COLS;
    static constexpr int DS = 4;                        // accumulator ring depth (MMA -> epilogue), one slot per link matrix
    static constexpr int D_COLS = 2 * N;                // per slot: [hi.hi chain | hi.lo + lo.hi chain]
    static constexpr int TMEM_COLS = 512;
    static constexpr int THREADS = 16 * 32;
    static constexpr int NBAR = 2 * LS + 2 * AS + 2 * DS;
    static constexpr int SMEM_BYTES = 1024 + LS * LINK_STAGE + LS * VEC_STAGE + AS * 2 * B_HALF + NBAR * 8 + 16;
    static constexpr bool OK = (NC % 16 == 0) && NC <= 128 && (NRHS % 8 == 0) && NRHS <= 16 &&
                               (D_COL0 + DS * D_COLS <= TMEM_COLS) && SMEM_BYTES <= 232448;
};

namespace ptx {

__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar,
                                            uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4}], [%2], %5;"
        ::"r"(dst), "l"(map), "r"(bar), "r"(c0), "r"(c1), "l"(policy)
        : "memory");
}
__device__ __forceinline__ void tmem_alloc(uint32_t smem_dst, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(cols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[tmem] . B[smem], kind::tf32, fp32 accumulate
__device__ __forceinline__ void mma_tf32_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc,
                                            uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void tmem_st16(uint32_t taddr, const uint32_t* v) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16};"
        ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]),
        "r"(v[8]), "r"(v[9]), "r"(v[10]), "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15])
        : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t* v) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
          "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void fence_cta() { asm volatile("fence.acq_rel.cta;" ::: "memory"); }
__device__ __forceinline__ void sts64(uint32_t addr, float a, float b) {
    asm volatile("st.shared.v2.f32 [%0], {%1,%2};" ::"r"(addr), "f"(a), "f"(b) : "memory");
}

}  // namespace ptx

// x = hi + lo with hi exactly representable in TF32 (low 13 mantissa bits zero); lo = x - hi is exact.
__device__ __forceinline__ void split_tf32(float x, uint32_t& hi, uint32_t& lo) {
    hi = __float_as_uint(x) & 0xffffe000u;
    lo = __float_as_uint(x - __uint_as_float(hi));
}

// K-major, no-swizzle UMMA shared-memory descriptor (SM100 format): 8 x 16-byte core matrices,
// LBO = byte step between the two k-halves of one MMA (128), SBO = byte step between 8-wide n groups.
__device__ __forceinline__ uint64_t umma_desc_kmajor(uint32_t smem_addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr >> 4) & 0x3fffu);
    d |= (uint64_t)((lbo_bytes >> 4) & 0x3fffu) << 16;
    d |= (uint64_t)((sbo_bytes >> 4) & 0x3fffu) << 32;
    d |= (uint64_t)1 << 46;  // descriptor version (Blackwell)
    return d;                // base_offset 0, layout_type 0 = SWIZZLE_NONE
}

template <int NC, int NRHS, bool DAG>
__global__ void __launch_bounds__(TensorGeom<NC, NRHS>::THREADS, 1)
coarse_apply_tensor(const __grid_constant__ CUtensorMap link_map, TensorParams p) {
    using Gm = TensorGeom<NC, NRHS>;
    static_assert(Gm::OK, "unsupported TENSOR geometry");
    constexpr int LS = Gm::LS, AS = Gm::AS, DS = Gm::DS, CHUNKS = Gm::CHUNKS, N = Gm::N;
    constexpr int LINK_STAGE = Gm::LINK_STAGE, VEC_STAGE = Gm::VEC_STAGE, B_HALF = Gm::B_HALF, B_SBO = Gm::B_SBO;
    constexpr int STAGES_PER_SITE = 9 * CHUNKS;
    // instruction descriptor: D fp32, A/B tf32, both K-major, N, M = 128
    constexpr uint32_t IDESC = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((128u >> 4) << 24);
    constexpr uint32_t IDESC2 = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(2 * N >> 3) << 17) | ((128u >> 4) << 24);
    static_assert(B_HALF == (N / 8) * B_SBO, "B lo must continue B hi's n groups");

    extern __shared__ unsigned char smem_raw[];
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t link_u32 = base;
    const uint32_t vec_u32 = link_u32 + LS * LINK_STAGE;
    const uint32_t b_u32 = vec_u32 + LS * VEC_STAGE;
    const uint32_t bar_u32 = b_u32 + AS * 2 * B_HALF;
    const uint32_t full0 = bar_u32, empty0 = full0 + 8u * LS;
    const uint32_t abfull0 = empty0 + 8u * LS, abempty0 = abfull0 + 8u * AS;
    const uint32_t dfull0 = abempty0 + 8u * AS, dempty0 = dfull0 + 8u * DS;
    const uint32_t tmem_slot = dempty0 + 8u * DS;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int i = 0; i < LS; ++i) {
            ptx::mbar_init(full0 + 8u * i, 1);
            ptx::mbar_init(empty0 + 8u * i, 4);
        }
        for (int i = 0; i < AS; ++i) {
            ptx::mbar_init(abfull0 + 8u * i, 4);
            ptx::mbar_init(abempty0 + 8u * i, 1);
        }
        for (int i = 0; i < DS; ++i) {
            ptx::mbar_init(dfull0 + 8u * i, 1);
            ptx::mbar_init(dempty0 + 8u * i, 4);
        }
        ptx::fence_mbar_init();
    }
    if (warp == 1) ptx::tmem_alloc(tmem_slot, Gm::TMEM_COLS);
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

    const int n_my = (p.n_sites > (int)blockIdx.x) ? (p.n_sites - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;

    if (warp == 0) {
        // ---------------------------------------------------------------- TMA producer
        // (whole warp in uniform control flow, one elected lane issues: see the MMA issuer below)
        const uint64_t pol_links = ptx::policy_evict_first();
        const uint64_t pol_vec = ptx::policy_evict_last();
        uint32_t t = 0;
        for (int it = 0; it < n_my; ++it) {
            const int s = blockIdx.x + it * gridDim.x;
            const SiteX cx = site_coords(p.lat, s);
#pragma unroll
            for (int m = 0; m < 9; ++m) {
                const int sv = stencil_site_x(p.lat, s, cx, m, DAG ? 1 : 0);
                const int sm = DAG ? sv : s;
                const int64_t mat_row0 = ((int64_t)sm * 9 + m) * NC;
                const float2* vec = p.in + (int64_t)sv * NC * NRHS;
#pragma unroll 1
                for (int c = 0; c < CHUNKS; ++c, ++t) {
                    const uint32_t slot = t % LS, ph = (t / LS) & 1u;
                    ptx::mbar_wait(empty0 + 8u * slot, ph ^ 1u);
                    if (ptx::elect_one()) {
                        ptx::mbar_arrive_expect_tx(full0 + 8u * slot, LINK_STAGE + VEC_STAGE);
                        if (!DAG) {
                            ptx::tma_load_2d(link_u32 + slot * LINK_STAGE, &link_map, c * 32, (int)mat_row0,
                                             full0 + 8u * slot, pol_links);
                        } else {
                            ptx::bulk_g2s(link_u32 + slot * LINK_STAGE,
                                          p.links + (mat_row0 + 16 * c) * (int64_t)(NC * 8), LINK_STAGE,
                                          full0 + 8u * slot, pol_links);
                        }
                        ptx::bulk_g2s(vec_u32 + slot * VEC_STAGE, vec + (int64_t)16 * c * NRHS, VEC_STAGE,
                                      full0 + 8u * slot, pol_vec);
                    }
                    __syncwarp();
                }
            }
        }
    } else if (warp == 1) {
        // ---------------------------------------------------------------- MMA issuer
        // The whole warp walks the loop (uniform control flow) and ONE elected lane issues the MMAs:
        // tcgen05.mma/commit read uniform registers, and inside a divergent `if (lane == 0)` the
        // compiler wraps every one of them in a per-lane replay loop (~100 issue cycles per MMA,
        // which made this warp the bottleneck of the kernel; profiles/r01_ncu_full_c5_tensor.md).
        //
        // One accumulator slot per link matrix: the tensor core truncates (rounds toward zero) when it
        // adds into the fp32 accumulator, a bias that grows linearly with the chain length, so the
        // chains are kept short (32 MMAs for hi.hi, 64 for the two cross terms, which are 2^-11
        // smaller and live in their own columns) and the nine partial results are added with
        // round-to-nearest fp32 in the epilogue.
        uint32_t t = 0;
        const uint32_t n_mat = (uint32_t)n_my * 9u;
        for (uint32_t tm = 0; tm < n_mat; ++tm) {
            const uint32_t ds = tm % DS, dph = (tm / DS) & 1u;
            ptx::mbar_wait(dempty0 + 8u * ds, dph ^ 1u);
            ptx::tc_fence_after();
            const uint32_t d_main = tmem_base + Gm::D_COL0 + ds * Gm::D_COLS, d_small = d_main + N;
#pragma unroll 1
            for (int c = 0; c < CHUNKS; ++c, ++t) {
                const uint32_t as = t % AS, aph = (t / AS) & 1u;
                ptx::mbar_wait(abfull0 + 8u * as, aph);
                ptx::tc_fence_after();
                if (ptx::elect_one()) {
                    const uint32_t a_hi = tmem_base + as * Gm::A_COLS, a_lo = a_hi + Gm::KSTAGE;
                    // B hi and B lo are adjacent 8-wide n groups of one K-major tile, so
                    // A_hi . [B_hi | B_lo] is ONE N = 2N MMA writing [main | small]
                    const uint64_t dbh0 = umma_desc_kmajor(b_u32 + as * 2 * B_HALF, 128, B_SBO);
#pragma unroll
                    for (int kk = 0; kk < Gm::KSTAGE / 8; ++kk) {
                        const uint64_t dbh = dbh0 + (uint64_t)(kk * 256 >> 4);
                        ptx::mma_tf32_ts(d_main, a_hi + kk * 8, dbh, IDESC2, (c | kk) != 0 ? 1u : 0u);
                        ptx::mma_tf32_ts(d_small, a_lo + kk * 8, dbh, IDESC, 1u);
                    }
                    ptx::tc_commit(abempty0 + 8u * as);
                    if (c == CHUNKS - 1) ptx::tc_commit(dfull0 + 8u * ds);
                }
                __syncwarp();
            }
        }
    } else if (warp >= 4 && warp < 12) {
        // ---------------------------------------------------------------- converters
        const int grp = (warp - 4) >> 2;              // stages t with t % 2 == grp
        const int q = warp & 3;                       // TMEM lane quadrant of this warp
        const int row = q * 32 + lane;                // A-operand row = output index i
        const int gtid = (warp & 3) * 32 + lane;      // 0..127 inside the group
        const uint32_t lane_addr = (uint32_t)(q * 32) << 16;
        const uint32_t total = (uint32_t)n_my * STAGES_PER_SITE;
        for (uint32_t t = grp; t < total; t += 2) {
            const uint32_t slot = t % LS, ph = (t / LS) & 1u;
            const uint32_t as = t % AS, aph = (t / AS) & 1u;
            ptx::mbar_wait(full0 + 8u * slot, ph);
            uint32_t a[32];
            if (row < NC) {
                if (!DAG) {
                    const uint32_t rb = link_u32 + slot * LINK_STAGE + row * 128;
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const uint4 x = ptx::lds128u(rb + (((uint32_t)u ^ ((uint32_t)row & 7u)) << 4));
                        a[4 * u] = x.x; a[4 * u + 1] = x.y; a[4 * u + 2] = x.z; a[4 * u + 3] = x.w;
                    }
                } else {
                    const uint32_t cb = link_u32 + slot * LINK_STAGE + row * 8;
#pragma unroll
                    for (int jj = 0; jj < 16; ++jj) {
                        const float2 x = ptx::lds64(cb + jj * (NC * 8));
                        a[2 * jj] = __float_as_uint(x.x); a[2 * jj + 1] = __float_as_uint(x.y);
                    }
                }
            } else {
#pragma unroll
                for (int u = 0; u < 32; ++u) a[u] = 0u;
            }
            float2 v[NRHS / 8];
#pragma unroll
            for (int x = 0; x < NRHS / 8; ++x) v[x] = ptx::lds64(vec_u32 + slot * VEC_STAGE + (gtid + 128 * x) * 8);
#ifndef COARSE_EXP_LATE_RELEASE
            // The loaded values are not consumed before the release below, and SYNCS.ARRIVE does not wait
            // for in-flight LDS: without this fence the producer's next TMA write into the slot can overtake
            // the reads (seen on B200 as sporadic stale 512-byte runs).  The fence completes the loads.
            ptx::fence_cta();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);      // link slot back to the producer
#endif

            ptx::mbar_wait(abempty0 + 8u * as, aph ^ 1u);            // MMAs that read this operand slot are done
            ptx::tc_fence_after();
            uint32_t hi[16], lo[16];
            const uint32_t a_hi = tmem_base + lane_addr + as * Gm::A_COLS, a_lo = a_hi + Gm::KSTAGE;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
#pragma unroll
                for (int u = 0; u < 16; ++u) split_tf32(__uint_as_float(a[16 * h + u]), hi[u], lo[u]);
                ptx::tmem_st16(a_hi + 16 * h, hi);
                ptx::tmem_st16(a_lo + 16 * h, lo);
            }
            const uint32_t b_hi = b_u32 + as * 2 * B_HALF, b_lo = b_hi + B_HALF;
#pragma unroll
            for (int x = 0; x < NRHS / 8; ++x) {
                const int e = gtid + 128 * x;
                const int j = e / NRHS, r = e % NRHS;
                // k = 2j, 2j+1 -> one 8-byte store; n = r (-> Re out) and n = NRHS + r (-> Im out)
                const uint32_t koff = (uint32_t)(j >> 1) * 128u + (uint32_t)(j & 1) * 8u;
                const uint32_t o1 = koff + (uint32_t)(r >> 3) * B_SBO + (uint32_t)(r & 7) * 16u;
                const uint32_t o2 = koff + (uint32_t)((NRHS + r) >> 3) * B_SBO + (uint32_t)((NRHS + r) & 7) * 16u;
                const float b1x = v[x].x, b1y = DAG ? v[x].y : -v[x].y;
                const float b2x = v[x].y, b2y = DAG ? -v[x].x : v[x].x;
                uint32_t h0, l0, h1, l1;
                split_tf32(b1x, h0, l0);
                split_tf32(b1y, h1, l1);
                ptx::sts64(b_hi + o1, __uint_as_float(h0), __uint_as_float(h1));
                ptx::sts64(b_lo + o1, __uint_as_float(l0), __uint_as_float(l1));
                split_tf32(b2x, h0, l0);
                split_tf32(b2y, h1, l1);
                ptx::sts64(b_hi + o2, __uint_as_float(h0), __uint_as_float(h1));
                ptx::sts64(b_lo + o2, __uint_as_float(l0), __uint_as_float(l1));
            }
            ptx::tc_wait_st();
            ptx::fence_proxy_async();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(abfull0 + 8u * as);
#ifdef COARSE_EXP_LATE_RELEASE
            if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
#endif
        }
    } else if (warp >= 12) {
        // ---------------------------------------------------------------- epilogue
        const int q = warp & 3;
        const int row = q * 32 + lane;
        const uint32_t lane_addr = (uint32_t)(q * 32) << 16;
        uint32_t tm = 0;
        for (int it = 0; it < n_my; ++it) {
            const int s = blockIdx.x + it * gridDim.x;
            float acc[N];
#pragma unroll
            for (int n = 0; n < N; ++n) acc[n] = 0.f;
#pragma unroll 1
            for (int m = 0; m < 9; ++m, ++tm) {
                const uint32_t ds = tm % DS, dph = (tm / DS) & 1u;
                ptx::mbar_wait(dfull0 + 8u * ds, dph);
                ptx::tc_fence_after();
                uint32_t d[2 * N];
                const uint32_t d_tmem = tmem_base + lane_addr + Gm::D_COL0 + ds * Gm::D_COLS;
#pragma unroll
                for (int c = 0; c < 2 * N / 16; ++c) ptx::tmem_ld16(d_tmem + 16 * c, d + 16 * c);
                ptx::tc_wait_ld();
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(dempty0 + 8u * ds);
#pragma unroll
                for (int n = 0; n < N; ++n) acc[n] += __uint_as_float(d[n]) + __uint_as_float(d[N + n]);
            }
            if (row < NC) {
                float4* o = reinterpret_cast<float4*>(p.out + ((int64_t)s * NC + row) * NRHS);
#pragma unroll
                for (int r = 0; r < NRHS; r += 2)
                    o[r >> 1] = make_float4(acc[r], acc[NRHS + r], acc[r + 1], acc[NRHS + r + 1]);
            }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem_base, Gm::TMEM_COLS);
}

}  // namespace coarse
