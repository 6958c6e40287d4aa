// tensor_kernel.cuh — COARSE_PATH_TENSOR: the block (multi-RHS) coarse-op apply on the tcgen05
// tensor cores, error-compensated 3xTF32 (multi-RHS is the paper's stated
// future work, its propagators are 3 right-hand sides at a time, L188, on 16-bit links, L99).
//
// Per site the block apply is a complex GEMM  out[Nc x nrhs] = [X Y...][Nc x 9Nc] . in[9Nc x nrhs].
// A row-major interleaved-complex link matrix IS a real M = Nc x K = 2Nc operand as stored:
//   A[i][2j] = Re M_ij, A[i][2j+1] = Im M_ij.  The vectors become a real K x N = 2Nc x 2NP
//   operand B = [B1 | B2],   B1[2j][r] = Re v_jr, B1[2j+1][r] = -Im v_jr   (-> Re out)
//                            B2[2j][r] = Im v_jr, B2[2j+1][r] =  Re v_jr   (-> Im out)
// (dagger: A[i][2j] = Re M_ji, A[i][2j+1] = Im M_ji, B1 = (Re v, Im v), B2 = (Im v, -Re v)).
// TF32 keeps 11 significant bits, so each fp32 operand is split x = hi + lo (hi = x with the low 13
// mantissa bits cleared, lo = x - hi, exact) and the product is hi.hi + hi.lo + lo.hi in fp32
// accumulators: relative error ~2^-21 per term instead of 2^-11.  int16 links decode
// to 16-bit integers in fp32, for which the same split is EXACT in both halves (11 + 5 bits); the
// per-matrix scale is folded into the B operand like the STREAM kernels fold it into the vector.
//
// Since the split has to touch every link entry with CUDA threads anyway, the kernel is a
// four-role pipeline per SM (persistent, one CTA per SM):
//   producer (1 elected lane) TMA: per stage one slab of a link matrix = the MT output rows of the item x
//                           16 contraction columns (dagger 0: box MT rows x 128 B | 64 B, SWIZZLE_128B |
//                           64B, so that "lane = row" reads are bank-conflict free; dagger 1: box 16 rows x
//                           MT entries, lane = column).
//   converters (3 x 4 warps) read the slab (lane <-> output index: TMEM transposes for free), decode /
//                           split hi/lo and write the A operand straight into TENSOR MEMORY (tcgen05.st),
//                           so the link bytes cross shared memory exactly twice (TMA write + one LDS
//                           read); fetch the 16 x NP vector entries of the stage from global memory (L2
//                           resident, prefetched one stage ahead into registers: any nrhs, any row pitch,
//                           zero padding for free), scale, split and store B hi/lo in shared memory in
//                           the canonical K-major UMMA layout.
//   MMA issuer (1 elected lane) tcgen05.mma kind::tf32, A from TMEM, B from smem, D (128 x 2NP fp32)
//                           in TMEM, 8 MMAs per stage (4 k-steps x {A_hi.[B_hi|B_lo], A_lo.B_hi}), one accumulator
//                           slot per link matrix; tcgen05.commit releases the operand slot / publishes D.
//   epilogue (4 warps)      tcgen05.ld D -> registers, adds the nine per-matrix partial results in
//                           round-to-nearest fp32 -> out[s][i][r]; a ring of 4 accumulator slots lets
//                           the next matrices' MMAs overlap the read-out.
// Work item = (site, tile of MT = Nc / NT output indices); NT = 2 for Nc = 192 (M = 128 per MMA); for Nc <= 64 a work
// item is a PAIR of sites sharing the 128-lane tile (TensorGeom::NS).
// One launch handles NP = 8 or 16 right-hand-side columns [r0, r0 + width) of vectors with `nrhs`
// columns; columns >= width are zero-padded in B and not stored (nrhs = 3 runs as NP = 8, nrhs = 40 as
// three launches).  The parts apply (coarse_op_apply_parts: parity-restricted site list, X stage on/off,
// alpha / beta folded into B, identity term added in the epilogue) is the same kernel with runtime flags.
// Summation order is fixed: results are bit-identical run to run.
#pragma once
#include <cuda.h>

#include "common.cuh"

#ifndef COARSE_TENSOR_RING_BYTES
#define COARSE_TENSOR_RING_BYTES 131072      // link bytes in the TMA ring per SM (slots being converted included)
#endif

namespace coarse {

struct TensorParams {
    Lat lat;
    const float* scales;      // int16 links: fp32 scale per (site, matrix)
    const float2* in;         // w: operand of the hopping terms (plain apply: the input vector)
    const float2* in_local;   // u: operand of the X term and of the identity term (plain apply: = in)
    float2* out;
    int n_sites;              // sites of the parity set (plain apply: V), or of the site range
    int site_begin;           // first site (index in the parity list) of this launch: coarse_op_apply_host launches ranges
    int parity;               // 0 even, 1 odd, 2 all sites
    int m_begin;              // 0: the X stage runs; 1: it is skipped (local = none | identity)
    int identity;             // 1: add alpha * u(x) to the result
    float alpha, beta;        // out = alpha * Loc + beta * Hop (plain apply: 1, 1)
    int nrhs;                 // right-hand sides stored per vector entry (row pitch of in / out)
    int r0, width;            // this launch computes columns [r0, r0 + width), width <= NP
};

constexpr int tensor_clamp(int v, int lo, int hi) { return v < lo ? lo : v > hi ? hi : v; }

template <int NC, bool I16, int NP>
struct TensorGeom {
    static constexpr int NT = NC > 128 ? 2 : 1;         // output tiles per site
    static constexpr int MT = NC / NT;                  // output indices per item (<= 128 TMEM lanes)
    static constexpr int ENTRY = I16 ? 4 : 8;           // bytes per complex link entry
    static constexpr int KSTAGE = 32;                   // real k per stage = 16 complex columns
    static constexpr int CHUNKS = NC / 16;              // stages per link matrix
    static constexpr int SLAB_ROW = 16 * ENTRY;         // dagger 0: bytes per slab row (128 | 64)
    // Matrices of at most 64 rows (Nc <= 64) would leave half of the 128-lane MMA tile idle while the kernel is bound by
    // the NUMBER of MMAs and pipeline stages (a stage costs ~350 ns whatever its size): a work item then holds TWO
    // sites - site 0 in lanes 0.., site 1 in lanes 64.. - whose B operands sit side by side along N; each MMA computes both
    // (the two off-diagonal blocks of its result are never read).  Half the stages and MMAs per site.
    static constexpr int NS = MT <= 64 ? 2 : 1;         // sites per work item
    static constexpr int SLAB_BYTES = MT * 16 * ENTRY;  // one site's slab of a stage (both dagger modes)
    static constexpr int SLAB_PITCH = NS == 2 ? 64 * SLAB_ROW : SLAB_BYTES;   // smem distance between the two sites' slabs
    static constexpr int LINK_STAGE = NS * SLAB_PITCH;  // smem bytes per stage
    static constexpr int N = 2 * NP * NS;               // MMA N: per site [Re out | Im out]
    static constexpr int NE = NS * NP / 8;              // B entries per converter thread and stage
    static constexpr int B_HALF = KSTAGE * N * 4;       // B hi (or lo) bytes per stage
    static constexpr int B_SBO = (KSTAGE / 4) * 128;    // byte stride between 8-column groups of n
    static constexpr int LS = tensor_clamp(COARSE_TENSOR_RING_BYTES / LINK_STAGE, 4, 20);   // link ring depth (TMA -> converters)
    static constexpr int AS = 4;                        // operand ring depth (converters -> MMA)
    static constexpr int A_COLS = 2 * KSTAGE;           // TMEM columns per operand stage: hi | lo
    static constexpr int D_COL0 = AS * A_COLS;
    static constexpr int D_COLS = 2 * N;                // per slot: [hi.hi chain | hi.lo + lo.hi chain]
    static constexpr int DS = tensor_clamp((512 - D_COL0) / D_COLS, 2, 4);   // accumulator ring depth (MMA -> epilogue), one slot per link matrix
    static constexpr int TMEM_COLS = 512;
    static constexpr int NG = 3;                        // converter groups of 4 warps (stage t -> group t mod NG)
    static constexpr int CONV_W0 = 2;                   // warps: 0 producer, 1 MMA issuer, 2 .. 2+4NG-1 converters, then 4 epilogue
    static constexpr int EPI_W0 = CONV_W0 + 4 * NG;
    static constexpr int THREADS = (EPI_W0 + 4) * 32;   // 18 warps; any 4 consecutive warps cover the 4 TMEM lane quadrants
    static constexpr int NBAR = 2 * LS + 2 * AS + 2 * DS;
    static constexpr int SMEM_BYTES = 1024 + LS * LINK_STAGE + AS * 2 * B_HALF + NBAR * 8 + 16;
    static constexpr bool OK = (NC % 16 == 0) && (MT % 8 == 0) && MT <= 128 && CHUNKS >= 2 && (NP == 8 || NP == 16) &&
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
__device__ __forceinline__ uint32_t lds32(uint32_t addr) {
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
    return v;
}

}  // namespace ptx

// x = hi + lo with hi exactly representable in TF32 (low 13 mantissa bits zero); lo = x - hi is exact.
__device__ __forceinline__ void split_tf32(float x, uint32_t& hi, uint32_t& lo) {
    hi = __float_as_uint(x) & 0xffffe000u;
    lo = __float_as_uint(x - __uint_as_float(hi));
}

// The same for a pair: the two low parts come from ONE packed FMA, lo = x - hi = fma(hi, -1, x) (exact).
__device__ __forceinline__ void split_tf32_pair(float x0, float x1, uint32_t& hi0, uint32_t& hi1, uint32_t& lo0, uint32_t& lo1) {
    hi0 = __float_as_uint(x0) & 0xffffe000u;
    hi1 = __float_as_uint(x1) & 0xffffe000u;
    const float2 lo = ptx::ffma2(make_float2(__uint_as_float(hi0), __uint_as_float(hi1)), make_float2(-1.f, -1.f), make_float2(x0, x1));
    lo0 = __float_as_uint(lo.x);
    lo1 = __float_as_uint(lo.y);
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

template <int NC, bool I16, int NP, bool DAG>
__global__ void __launch_bounds__(TensorGeom<NC, I16, NP>::THREADS, 1)
coarse_apply_tensor(const __grid_constant__ CUtensorMap link_map, TensorParams p) {
    using Gm = TensorGeom<NC, I16, NP>;
    static_assert(Gm::OK, "unsupported TENSOR geometry");
    constexpr int LS = Gm::LS, AS = Gm::AS, DS = Gm::DS, CHUNKS = Gm::CHUNKS, N = Gm::N, NT = Gm::NT, MT = Gm::MT, NE = Gm::NE;
    constexpr int NS = Gm::NS, SLAB_BYTES = Gm::SLAB_BYTES, SLAB_PITCH = Gm::SLAB_PITCH;
    constexpr int LINK_STAGE = Gm::LINK_STAGE, B_HALF = Gm::B_HALF, B_SBO = Gm::B_SBO, ENTRY = Gm::ENTRY;
    // instruction descriptor: D fp32, A/B tf32, both K-major, N, M = 128
    constexpr uint32_t IDESC = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((128u >> 4) << 24);
    constexpr uint32_t IDESC2 = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(2 * N >> 3) << 17) | ((128u >> 4) << 24);
    static_assert(B_HALF == (N / 8) * B_SBO, "B lo must continue B hi's n groups");

    extern __shared__ unsigned char smem_raw[];
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t link_u32 = base;
    const uint32_t b_u32 = link_u32 + LS * LINK_STAGE;
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

    const int n_items = NS == 2 ? (p.n_sites + 1) / 2 : p.n_sites * NT;
    const int n_my = (n_items > (int)blockIdx.x) ? (n_items - 1 - (int)blockIdx.x) / (int)gridDim.x + 1 : 0;
    const int M0 = p.m_begin;
    const int n_mat_item = 9 - M0;                                   // link matrices per item
    // site sg (0 | 1) of a work item; an odd site count leaves the last item's second half without a site: it
    // re-computes the first one (valid memory, constant byte counts) and does not store
    auto site_valid = [&](int item, int sg) -> bool { return NS == 1 || 2 * item + sg < p.n_sites; };
    auto site_of_item = [&](int item, int sg = 0) -> int {
        int h = NS == 2 ? 2 * item + (site_valid(item, sg) ? sg : 0) : (NT == 1 ? item : item / NT);
        h += p.site_begin;
        return p.parity != 2 ? parity_site(p.lat, h, p.parity) : h;
    };

    if (warp == 0) {
        // ---------------------------------------------------------------- TMA producer
        // (whole warp in uniform control flow, one elected lane issues: see the MMA issuer below)
        const uint64_t pol_links = ptx::policy_evict_first();
        uint32_t t = 0;
        for (int it = 0; it < n_my; ++it) {
            const int item = blockIdx.x + it * gridDim.x;
            const int i0 = NT == 1 ? 0 : (item % NT) * MT;
            int s[NS];
            SiteX cx[NS];
#pragma unroll
            for (int sg = 0; sg < NS; ++sg) {
                s[sg] = site_of_item(item, sg);
                cx[sg] = site_coords(p.lat, s[sg]);
            }
#pragma unroll
            for (int m = 0; m < 9; ++m) {
                if (m < M0) continue;
                int mat_row0[NS];
#pragma unroll
                for (int sg = 0; sg < NS; ++sg) {
                    const int sv = stencil_site_x(p.lat, s[sg], cx[sg], m, DAG ? 1 : 0);
                    const int sm = DAG ? sv : s[sg];
                    mat_row0[sg] = (sm * 9 + m) * NC;               // < 2^31: checked by the host (make_link_maps)
                }
#pragma unroll 1
                for (int c = 0; c < CHUNKS; ++c, ++t) {
                    const uint32_t slot = t % LS, ph = (t / LS) & 1u;
                    ptx::mbar_wait(empty0 + 8u * slot, ph ^ 1u);
                    if (ptx::elect_one()) {
                        ptx::mbar_arrive_expect_tx(full0 + 8u * slot, NS * SLAB_BYTES);
#pragma unroll
                        for (int sg = 0; sg < NS; ++sg) {
                            const uint32_t dst = link_u32 + slot * LINK_STAGE + sg * SLAB_PITCH;
                            if (!DAG)      // rows [i0, i0 + MT) x complex columns [16c, 16c + 16)
                                ptx::tma_load_2d(dst, &link_map, c * (16 * ENTRY / 4), mat_row0[sg] + i0, full0 + 8u * slot, pol_links);
                            else           // rows [16c, 16c + 16) x complex columns [i0, i0 + MT)
                                ptx::tma_load_2d(dst, &link_map, i0 * (ENTRY / 4), mat_row0[sg] + 16 * c, full0 + 8u * slot, pol_links);
                        }
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
        // chains are kept short (4 CHUNKS MMAs for hi.hi, 8 CHUNKS for the two cross terms, which are
        // 2^-11 smaller and live in their own columns) and the nine partial results are added with
        // round-to-nearest fp32 in the epilogue.
        uint32_t t = 0;
        const uint32_t n_mat = (uint32_t)n_my * (uint32_t)n_mat_item;
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
    } else if (warp >= Gm::CONV_W0 && warp < Gm::EPI_W0) {
        // ---------------------------------------------------------------- converters
        // Three groups in flight: ncu on the two-group version showed the converter warps issuing 22 % of the
        // time (275 instructions per stage in ~1250 cycles: mbarrier round trips, tcgen05.st + wait::st, the
        // proxy fence), i.e. bound by the latency chain of a stage, not by issue slots or HBM.
        constexpr int NG = Gm::NG;
        const int grp = (warp - Gm::CONV_W0) >> 2;    // stages t with t % NG == grp
        const int q = warp & 3;                       // TMEM lane quadrant of this warp (hardware: warp id mod 4)
        const int lane_row = q * 32 + lane;           // TMEM lane
        const int sg_row = NS == 2 ? lane_row >> 6 : 0;               // which site of the item this lane serves
        const int row = NS == 2 ? lane_row & 63 : lane_row;           // A-operand row = output index i of that site
        const int gtid = ((warp - Gm::CONV_W0) & 3) * 32 + lane;      // 0..127 inside the group
        const uint32_t lane_addr = (uint32_t)(q * 32) << 16;
        const uint32_t total = (uint32_t)n_my * (uint32_t)(n_mat_item * CHUNKS);

        // B entries of this thread, the same (contraction row j, column r) in every stage.  A half-warp
        // covers the 16 distinct 8-byte bank slots (k mod 4 pair, n mod 8) of the K-major layout, so its
        // stores are conflict-free (e = gtid + 128 x: r = e & 7 [+ 8], j = 2 (e >> 4 [>> 1]) + ((e >> 3) & 1)).
        int b_off_vec[NE];           // element offset inside the stage's 16 x nrhs block
        int b_sg[NE];                // site of the item the entry belongs to
        uint32_t b_o1[NE], b_o2[NE]; // byte offsets of the (n = r) and (n = NP + r) entries in the B tile
        bool b_valid[NE];
#pragma unroll
        for (int x = 0; x < NE; ++x) {
            const int e = gtid + 128 * x;
            int rest = e >> 4;
            int r = e & 7;
            if (NP == 16) { r += (rest & 1) * 8; rest >>= 1; }
            int sg = 0;
            if (NS == 2) { sg = rest & 1; rest >>= 1; }
            const int j = 2 * rest + ((e >> 3) & 1);
            b_valid[x] = r < p.width;
            b_sg[x] = sg;
            b_off_vec[x] = j * p.nrhs + r;
            const uint32_t koff = (uint32_t)(j >> 1) * 128u + (uint32_t)(j & 1) * 8u;
            const int n1 = sg * 2 * NP + r, n2 = n1 + NP;
            b_o1[x] = koff + (uint32_t)(n1 >> 3) * B_SBO + (uint32_t)(n1 & 7) * 16u;
            b_o2[x] = koff + (uint32_t)(n2 >> 3) * B_SBO + (uint32_t)(n2 & 7) * 16u;
        }

        // cursor of the NEXT stage of this group (its vector entries are prefetched while the current
        // stage is converted): item index, matrix, chunk, and what depends on them
        int n_it = 0, n_m = M0, n_c = grp;              // stage t = grp: chunk grp of the first matrix (normalised below)
        int n_s[NS];
        SiteX n_cx[NS];
        const float2* n_vec[NS];
        float n_sc[NS];
#pragma unroll
        for (int sg = 0; sg < NS; ++sg) { n_s[sg] = 0; n_cx[sg] = SiteX{}; n_vec[sg] = p.in; n_sc[sg] = 1.f; }
        auto load_item = [&]() {
            if (n_it < n_my) {
#pragma unroll
                for (int sg = 0; sg < NS; ++sg) {
                    n_s[sg] = site_of_item(blockIdx.x + n_it * gridDim.x, sg);
                    n_cx[sg] = site_coords(p.lat, n_s[sg]);
                }
            }
        };
        auto load_matrix = [&]() {
            if (n_it < n_my) {
#pragma unroll
                for (int sg = 0; sg < NS; ++sg) {
                    const int sv = stencil_site_x(p.lat, n_s[sg], n_cx[sg], n_m, DAG ? 1 : 0);
                    const int sm = DAG ? sv : n_s[sg];
                    n_vec[sg] = (n_m == 0 ? p.in_local : p.in) + (int64_t)sv * NC * p.nrhs + p.r0;
                    n_sc[sg] = n_m == 0 ? p.alpha : p.beta;
                    if constexpr (I16) n_sc[sg] *= __ldg(p.scales + (int64_t)sm * 9 + n_m);
                }
            }
        };
        float2 vn[NE];
        auto fetch = [&]() {
#pragma unroll
            for (int x = 0; x < NE; ++x)
                vn[x] = (n_it < n_my && b_valid[x]) ? __ldg(n_vec[NS == 2 ? b_sg[x] : 0] + (int64_t)(16 * n_c) * p.nrhs + b_off_vec[x])
                                                    : make_float2(0.f, 0.f);
        };
        auto normalise = [&]() -> bool {               // carry n_c into (n_m, n_it); true if the item changed
            bool item_changed = false;
            while (n_c >= CHUNKS) {
                n_c -= CHUNKS;
                if (++n_m == 9) { n_m = M0; ++n_it; item_changed = true; }
            }
            return item_changed;
        };
        normalise();
        load_item();
        load_matrix();
        fetch();

        for (uint32_t t = grp; t < total; t += NG) {
            const uint32_t slot = t % LS, ph = (t / LS) & 1u;
            const uint32_t as = t % AS, aph = (t / AS) & 1u;
            // this stage's vector entries and scale; then move the cursor two stages on and prefetch
            float2 v[NE];
#pragma unroll
            for (int x = 0; x < NE; ++x) v[x] = vn[x];
            float sc[NS];
#pragma unroll
            for (int sg = 0; sg < NS; ++sg) sc[sg] = n_sc[sg];
            n_c += NG;
            if (n_c >= CHUNKS) {
                if (normalise()) load_item();
                load_matrix();
            }
            fetch();

            ptx::mbar_wait(full0 + 8u * slot, ph);
            float a[32];
            if (row < MT) {
                const uint32_t sb = link_u32 + slot * LINK_STAGE + sg_row * SLAB_PITCH;
                if constexpr (!DAG && !I16) {
                    const uint32_t rb = sb + row * 128;            // SWIZZLE_128B: chunk u of row at u ^ (row & 7)
#pragma unroll
                    for (int u = 0; u < 8; ++u) {
                        const float4 x = ptx::lds128(rb + (((uint32_t)u ^ ((uint32_t)row & 7u)) << 4));
                        a[4 * u] = x.x; a[4 * u + 1] = x.y; a[4 * u + 2] = x.z; a[4 * u + 3] = x.w;
                    }
                } else if constexpr (!DAG && I16) {
                    const uint32_t rb = sb + row * 64;             // SWIZZLE_64B: chunk u of row at u ^ ((row >> 1) & 3)
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const uint4 x = ptx::lds128u(rb + (((uint32_t)u ^ (((uint32_t)row >> 1) & 3u)) << 4));
                        const float2 e0 = unpack_i16x2(x.x), e1 = unpack_i16x2(x.y), e2 = unpack_i16x2(x.z), e3 = unpack_i16x2(x.w);
                        a[8 * u] = e0.x; a[8 * u + 1] = e0.y; a[8 * u + 2] = e1.x; a[8 * u + 3] = e1.y;
                        a[8 * u + 4] = e2.x; a[8 * u + 5] = e2.y; a[8 * u + 6] = e3.x; a[8 * u + 7] = e3.y;
                    }
                } else if constexpr (DAG && !I16) {
                    const uint32_t cb = sb + row * 8;              // [16 rows][MT entries], lane = column
#pragma unroll
                    for (int jj = 0; jj < 16; ++jj) {
                        const float2 x = ptx::lds64(cb + jj * (MT * 8));
                        a[2 * jj] = x.x; a[2 * jj + 1] = x.y;
                    }
                } else {
                    const uint32_t cb = sb + row * 4;
#pragma unroll
                    for (int jj = 0; jj < 16; ++jj) {
                        const float2 x = unpack_i16x2(ptx::lds32(cb + jj * (MT * 4)));
                        a[2 * jj] = x.x; a[2 * jj + 1] = x.y;
                    }
                }
            } else {
#pragma unroll
                for (int u = 0; u < 32; ++u) a[u] = 0.f;
            }

            ptx::mbar_wait(abempty0 + 8u * as, aph ^ 1u);            // MMAs that read this operand slot are done
            ptx::tc_fence_after();
            uint32_t hi[16], lo[16];
            const uint32_t a_hi = tmem_base + lane_addr + as * Gm::A_COLS, a_lo = a_hi + Gm::KSTAGE;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
#pragma unroll
                for (int u = 0; u < 16; u += 2) split_tf32_pair(a[16 * h + u], a[16 * h + u + 1], hi[u], hi[u + 1], lo[u], lo[u + 1]);
                ptx::tmem_st16(a_hi + 16 * h, hi);
                ptx::tmem_st16(a_lo + 16 * h, lo);
            }
            const uint32_t b_hi = b_u32 + as * 2 * B_HALF, b_lo = b_hi + B_HALF;
#pragma unroll
            for (int x = 0; x < NE; ++x) {
                // k = 2j, 2j+1 -> one 8-byte store; n = r (-> Re out) and n = NP + r (-> Im out)
                const float scx = sc[NS == 2 ? b_sg[x] : 0];
                const float vx = v[x].x * scx, vy = v[x].y * scx;
                const float b1x = vx, b1y = DAG ? vy : -vy;
                const float b2x = vy, b2y = DAG ? -vx : vx;
                uint32_t h0, l0, h1, l1;
                split_tf32_pair(b1x, b1y, h0, h1, l0, l1);
                ptx::sts64(b_hi + b_o1[x], __uint_as_float(h0), __uint_as_float(h1));
                ptx::sts64(b_lo + b_o1[x], __uint_as_float(l0), __uint_as_float(l1));
                split_tf32_pair(b2x, b2y, h0, h1, l0, l1);
                ptx::sts64(b_hi + b_o2[x], __uint_as_float(h0), __uint_as_float(h1));
                ptx::sts64(b_lo + b_o2[x], __uint_as_float(l0), __uint_as_float(l1));
            }
            ptx::tc_wait_st();
            ptx::fence_proxy_async();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(abfull0 + 8u * as);
            // Link slot back to the producer - only HERE, after the loaded values have gone through the split into
            // tensor memory (wait::st above): the release must come after a CONSUMER of the loads in program order.
            // Releasing right after the loads behind a fence.acq_rel.cta (rounds 1 and 2 until a stress run) let the
            // producer's next TMA write overtake the reads once in ~600-2000 applies (a few wrong rows at one site).
            if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
        }
    } else if (warp >= Gm::EPI_W0) {
        // ---------------------------------------------------------------- epilogue
        const int q = warp & 3;
        const int lane_row = q * 32 + lane;
        const int sg_row = NS == 2 ? lane_row >> 6 : 0;       // site of the item this lane's row belongs to (warp-uniform)
        const int row = NS == 2 ? lane_row & 63 : lane_row;
        const uint32_t lane_addr = (uint32_t)(q * 32) << 16;
        constexpr int NA = 2 * NP;                             // accumulators of a row: [Re out | Im out] of ITS site
        uint32_t tm = 0;
        for (int it = 0; it < n_my; ++it) {
            const int item = blockIdx.x + it * gridDim.x;
            const int s = site_of_item(item, sg_row);
            const int i0 = NT == 1 ? 0 : (item % NT) * MT;
            float acc[NA];
#pragma unroll
            for (int n = 0; n < NA; ++n) acc[n] = 0.f;
#pragma unroll 1
            for (int m = M0; m < 9; ++m, ++tm) {
                const uint32_t ds = tm % DS, dph = (tm / DS) & 1u;
                ptx::mbar_wait(dfull0 + 8u * ds, dph);
                ptx::tc_fence_after();
                // this row's site: columns [sg NA, sg NA + NA) of the main chain and of the cross-term chain
                const uint32_t d_tmem = tmem_base + lane_addr + Gm::D_COL0 + ds * Gm::D_COLS + sg_row * NA;
                // 16 columns of the main chain and the matching 16 of the cross-term chain at a time
#pragma unroll
                for (int c = 0; c < NA / 16; ++c) {
                    uint32_t dm[16], dx[16];
                    ptx::tmem_ld16(d_tmem + 16 * c, dm);
                    ptx::tmem_ld16(d_tmem + N + 16 * c, dx);
                    ptx::tc_wait_ld();
#pragma unroll
                    for (int n = 0; n < 16; ++n) acc[16 * c + n] += __uint_as_float(dm[n]) + __uint_as_float(dx[n]);
                }
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(dempty0 + 8u * ds);
            }
            if (row < MT && site_valid(item, sg_row)) {
                const int64_t o = ((int64_t)s * NC + i0 + row) * p.nrhs + p.r0;
                if (p.identity) {
#pragma unroll
                    for (int r = 0; r < NP; ++r)
                        if (r < p.width) {
                            const float2 u = __ldg(p.in_local + o + r);
                            acc[r] = fmaf(p.alpha, u.x, acc[r]);
                            acc[NP + r] = fmaf(p.alpha, u.y, acc[NP + r]);
                        }
                }
                if (((p.nrhs | p.r0) & 1) == 0) {
                    float4* o4 = reinterpret_cast<float4*>(p.out + o);
#pragma unroll
                    for (int r = 0; r < NP; r += 2) {
                        if (r + 1 < p.width) o4[r >> 1] = make_float4(acc[r], acc[NP + r], acc[r + 1], acc[NP + r + 1]);
                        else if (r < p.width) p.out[o + r] = make_float2(acc[r], acc[NP + r]);
                    }
                } else {
#pragma unroll
                    for (int r = 0; r < NP; ++r)
                        if (r < p.width) p.out[o + r] = make_float2(acc[r], acc[NP + r]);
                }
            }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 1) ptx::tmem_dealloc(tmem_base, Gm::TMEM_COLS);
}

}  // namespace coarse
