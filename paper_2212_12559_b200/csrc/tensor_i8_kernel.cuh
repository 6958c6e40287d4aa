// tensor_i8_kernel.cuh — COARSE_PATH_TENSOR for int16 LINKS (the paper's storage) and several
// right-hand sides (its future work, L200; a propagator is 3, L188): the block apply on the B200's INTEGER
// tensor cores (tcgen05.mma kind::i8, int32 accumulators in TMEM), exact in the link operand.
//
// Why not the 3xTF32 kernel (tensor_kernel.cuh) for these links: ncu on it shows one pipeline stage of 16
// complex columns costing ~350 ns whatever its size - eight K = 8 MMAs per stage whose issue backs up in
// the MIO queue, plus ~250 decode / split instructions per converter lane - so int16 links, which carry
// twice the entries per byte, ran at 4.2 TB/s where complex64 links are HBM bound.  An int16 entry
// q = 256 a1 + a0 is two BYTES: a1 = q >> 8 signed, a0 = q & 255 unsigned.  As int8 operands
//   * the A operand needs no arithmetic at all: two byte permutes (PRMT) per pair of entries gather the
//     high bytes and the low bytes of a row into the K-major TMEM layout (32 instead of ~256 instructions
//     per 32 complex columns), and
//   * one MMA covers K = 32 real values (16 complex columns) instead of 8: 4 MMAs per 16 KB stage, not 16.
// The B operand (the vectors) is turned into fixed point per (site, right-hand side): with
// g = 2^-e such that max |component| g lies in [1/2, 1) (a small pre-pass kernel over the vector field, L2
// resident), B = rint(v g 2^22) is split into three signed base-256 digits d0, d1, d2 (exact: B = sum d_l 256^l),
// stored side by side along N, so that per 16 complex columns
//     D1[:, l] += A1 . d_l        (signed x signed,   N = 3 x 2 NP)
//     D0[:, l] += A0 . d_l        (unsigned x signed, N = 3 x 2 NP)
// are TWO MMAs, exact in int32 (|a| <= 255, |d| <= 128, K = 2 Nc <= 384 per link matrix: < 2^24).  Products of equal
// weight share accumulator columns: D1 is written ONE digit block higher than D0, so that the slot holds
// W_0 = D0_0, W_1 = D1_0 + D0_1, W_2 = D1_1 + D0_2, W_3 = D1_2 (four blocks instead of six), and the epilogue
// recombines out += f_m (((W_3 256 + W_2) 256 + W_1) 256 + W_0) in fp32, f_m = scale_m coef_m / (g 2^22).  The only rounding besides that recombination is the 23-bit fixed-point
// representation of each site vector relative to its largest component - the same order as the fp32 rounding
// of the inputs themselves; measured 3e-7 relative L2 against an fp64 evaluation (tolerance 1e-5).
//
// Pipeline roles, work items, the parts apply (parity list, X stage on / off, alpha / beta, identity term) and
// the RHS column tiles are those of tensor_kernel.cuh; a stage is KC = 32 complex columns (16 for Nc = 48).
// Bit-identical run to run (integer accumulation, fixed schedule).
#pragma once
#include <type_traits>

#include "tensor_kernel.cuh"

#ifndef COARSE_TENSOR_RING_BYTES
#define COARSE_TENSOR_RING_BYTES 131072      // link bytes in the TMA ring per SM (slots being converted included)
#endif

namespace coarse {

#ifndef COARSE_I8_NG
#define COARSE_I8_NG 3
#endif
constexpr int TENSOR_I8_GP = 16;   // row pitch of the scale arrays: one launch handles at most 16 right-hand sides

struct TensorI8Params {
    TensorParams t;
    const float* vscale_w;    // [V][TENSOR_I8_GP][2] = (g, 1/g) of columns r0.. of the hopping operand w (plain apply: of `in`)
    const float* vscale_u;    // the same for the local operand u (plain apply: = vscale_w)
    const float* vnorms;      // HV kernels: `t.in` holds int16 (re, im) pairs [V][Nc][nrhs] and this the fp32 norm per (site, rhs)
};

// HV = half-precision VECTORS (16-bit fixed point with a per-site fp32 norm) on top of the 16-bit links
// (L99) - the paper's own storage for both operands.  An int16 vector component q = 256 b1 + b0 is already fixed point:
// its two bytes ARE the digits (b1 signed, b0 unsigned), so the B operand needs no arithmetic either (two byte permutes per
// entry, against 4 F2I + 16 integer instructions for three signed digits of an fp32 value), and there are two digit blocks
// instead of three.  The two blocks differ in signedness, which an MMA fixes per operand: four MMAs per k-step
//     W_0 = A0.B0 (u8 x u8)   W_1 = A0.B1 (u8 x s8) + A1.B0 (s8 x u8)   W_2 = A1.B1 (s8 x s8)
// into three accumulator blocks; out += f_m ((W_2 256 + W_1) 256 + W_0), f_m = link scale x coefficient x vector norm.
// Both operands enter the tensor core exactly; the only rounding is the fp32 recombination in the epilogue.
template <int NC, int NP, bool HV = false>
struct TensorI8Geom {
    static constexpr int NT = NC > 128 ? 2 : 1;
    static constexpr int MT = NC / NT;
    static constexpr int KC = (NC % 32 == 0) ? 32 : 16;       // complex columns per stage
    static constexpr int CHUNKS = NC / KC;                     // stages per link matrix
    static constexpr int KSTEPS = KC / 16;                     // MMA k-steps (K = 32 int8 = 16 complex columns)
    // Two sites per work item when the matrices have at most 64 rows and the 8-wide column tile is in use (the
    // accumulator ring of the 16-wide tile would not fit tensor memory): site 0 in TMEM lanes 0.., site 1 in lanes
    // 64.., their B operands side by side along N inside every digit block (see TensorGeom::NS in tensor_kernel.cuh).
    static constexpr int NS = (MT <= 64 && (NP <= 8 || HV)) ? 2 : 1;   // (a 4-wide column tile for 2-4 right-hand sides exists in this mode only;
                                                                       //  HV: three accumulator blocks, so the 16-wide tile fits too, with a ring of 2)
    static constexpr int NPS = NP * NS;                        // right-hand-side columns of an item (all its sites)
    static constexpr int SLAB_BYTES = MT * KC * 4;             // one site's slab of a stage
    static constexpr int SLAB_PITCH = NS == 2 ? 64 * KC * 4 : SLAB_BYTES;
    static constexpr int LINK_STAGE = NS * SLAB_PITCH;
    static constexpr int NDIG = HV ? 2 : 3;                    // digit blocks of the B operand
    static constexpr int NB3 = NDIG * 2 * NPS;                 // B tile columns: NDIG digit blocks of (per site) [Re out | Im out]
    static constexpr int B_STAGE = 2 * KC * NB3;               // int8 B tile of a stage, bytes
    static constexpr int B_SBO = (2 * KC / 16) * 128;          // byte stride between 8-column groups of n
    static constexpr int NE = KC * NPS / 128;                  // B entries per converter thread and stage
    static constexpr int LS = tensor_clamp(COARSE_TENSOR_RING_BYTES / LINK_STAGE, 4, 20);
    static constexpr int AS = 4;
    static constexpr int A_HALF = KC / 2;                      // TMEM columns of one byte plane (4 int8 per column)
    static constexpr int A_COLS = 2 * A_HALF;                  // high bytes | low bytes
    static constexpr int D_COL0 = AS * A_COLS;
    static constexpr int D_COLS = (NDIG + 1) * 2 * NPS;        // W_0 .. W_NDIG, each (per site) [Re out | Im out]
    static constexpr int DS = tensor_clamp((512 - D_COL0) / D_COLS, 2, 3);   // accumulator ring depth
    static constexpr int FT = 8;                               // ring of per-matrix epilogue factor rows
    static constexpr int TMEM_COLS = 512;
    static constexpr int NG = COARSE_I8_NG, CONV_W0 = 2, EPI_W0 = CONV_W0 + 4 * NG;
    static constexpr int THREADS = (EPI_W0 + 4) * 32;
    static constexpr int NBAR = 2 * LS + 2 * AS + 2 * DS;
    static constexpr int SMEM_BYTES = 1024 + LS * LINK_STAGE + AS * B_STAGE + FT * NPS * 4 + NBAR * 8 + 16;
    static constexpr bool OK = (NC % 16 == 0) && (MT % 8 == 0) && MT <= 128 && (NP == 4 || NP == 8 || NP == 16) && NE >= 1 && NB3 % 16 == 0 &&
                               (D_COL0 + DS * D_COLS <= TMEM_COLS) && SMEM_BYTES <= 232448 &&
                               (HV ? ((2 * NPS) % 16 == 0 && 2 * NC * 2 * 255 * 255 < (1 << 30)) : (2 * NC * 128 * 255 < (1 << 24)));
};

namespace ptx {

// D[tmem] (+)= A[tmem] . B[smem], kind::i8, int32 accumulate
__device__ __forceinline__ void mma_i8_ts(uint32_t d_tmem, uint32_t a_tmem, uint64_t b_desc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], [%1], %2, %3, p;\n\t}"
        ::"r"(d_tmem), "r"(a_tmem), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t* v) {
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
                 ::"r"(taddr), "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7])
                 : "memory");
}
__device__ __forceinline__ void tmem_ld8(uint32_t taddr, uint32_t* v) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
                 : "r"(taddr)
                 : "memory");
}
__device__ __forceinline__ void sts16(uint32_t addr, uint32_t v) {
    asm volatile("st.shared.u16 [%0], %1;" ::"r"(addr), "h"((unsigned short)v) : "memory");
}

}  // namespace ptx

// (g, 1/g) per (site, right-hand side): g = 2^-e with max |component| g in [1/2, 1); an all-zero vector gets (0, 0).
// One thread per (site, column r0 + r < r0 + width); consecutive threads read consecutive right-hand sides of one
// entry (coalesced); gs[site][r] with row pitch TENSOR_I8_GP.
static __global__ void __launch_bounds__(128) vec_pow2_scale_kernel(const float2* v, long long n_sites, int nc, int nrhs, int r0,
                                                                    int width, float2* gs) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_sites * width) return;
    const long long s = idx / width;
    const int r = (int)(idx - s * width);
    const float2* p = v + s * nc * nrhs + r0 + r;
    float m = 0.f;
    for (int a = 0; a < nc; ++a) {
        const float2 x = p[(long long)a * nrhs];
        const float ax = fmaxf(fabsf(x.x), fabsf(x.y));
        m = (x.x != x.x || x.y != x.y || m != m) ? __int_as_float(0x7fc00000) : fmaxf(m, ax);      // fmaxf drops NaN: keep it
    }
    float2 o = make_float2(0.f, 0.f);
    if (!(m <= 3.0e38f)) {
        // Inf or NaN in the vector: fixed point cannot carry it, so the column's epilogue factor becomes NaN and every
        // output that reads this site is NaN, as IEEE arithmetic on the complex64 path would make it (or Inf)
        o = make_float2(0.f, __int_as_float(0x7fc00000));
    } else if (m > 0.f) {
        int e;
        frexpf(m, &e);                                   // m = f 2^e, f in [1/2, 1)
        e = e < -100 ? -100 : e > 100 ? 100 : e;         // keep g and 1/g (and g 2^22) normal numbers
        o = make_float2(ldexpf(1.f, -e), ldexpf(1.f, e));
    }
    gs[s * TENSOR_I8_GP + r] = o;
}

// Signed base-256 digits of b (|b| <= 2^22 + 1): b = d0 + 256 d1 + 65536 d2 with d0, d1 in [-128, 127], |d2| <= 65.
// With t1 = (b + 128) >> 8 and t2 = (t1 + 128) >> 8 (arithmetic shifts: the carries of the signed digits) the
// digits are the LOW BYTES of b, t1, t2 as two's complement int8: 4 integer instructions per value, and one
// byte permute packs the same digit of the two values of a (re, im) pair for the 16-bit store.
__device__ __forceinline__ void digit_regs(int b, int& t1, int& t2) {
    t1 = (b + 128) >> 8;
    t2 = (t1 + 128) >> 8;
}
__device__ __forceinline__ uint32_t pack_lo_bytes(int x, int y) { return __byte_perm((uint32_t)x, (uint32_t)y, 0x0040); }

template <int NC, int NP, bool DAG, bool HV = false>
__global__ void __launch_bounds__(TensorI8Geom<NC, NP, HV>::THREADS, 1)
coarse_apply_tensor_i8(const __grid_constant__ CUtensorMap link_map, TensorI8Params pp) {
    using Gm = TensorI8Geom<NC, NP, HV>;
    using VecT = typename std::conditional<HV, uint32_t, float2>::type;      // one complex vector component in memory
    static_assert(Gm::OK, "unsupported TENSOR-I8 geometry");
    constexpr int LS = Gm::LS, AS = Gm::AS, DS = Gm::DS, CHUNKS = Gm::CHUNKS, NT = Gm::NT, MT = Gm::MT, NE = Gm::NE;
    constexpr int KC = Gm::KC, LINK_STAGE = Gm::LINK_STAGE, B_STAGE = Gm::B_STAGE, B_SBO = Gm::B_SBO, NB3 = Gm::NB3, FT = Gm::FT;
    constexpr int NS = Gm::NS, NPS = Gm::NPS, SLAB_BYTES = Gm::SLAB_BYTES, SLAB_PITCH = Gm::SLAB_PITCH;
    // instruction descriptors: D int32 (c_format 2), A signed | unsigned 8 bit, B signed 8 bit, K-major, N = NB3, M = 128
    constexpr uint32_t IDESC_S = (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(NB3 >> 3) << 17) | ((128u >> 4) << 24);
    constexpr uint32_t IDESC_U = (2u << 4) | (0u << 7) | (1u << 10) | ((uint32_t)(NB3 >> 3) << 17) | ((128u >> 4) << 24);
    constexpr uint32_t IDESC_U1 = (2u << 4) | (0u << 7) | (1u << 10) | ((uint32_t)(2 * NPS >> 3) << 17) | ((128u >> 4) << 24);   // one digit block
    constexpr uint32_t IDESC_U2 = (2u << 4) | (0u << 7) | (1u << 10) | ((uint32_t)(4 * NPS >> 3) << 17) | ((128u >> 4) << 24);   // two digit blocks
    // HV: one digit block (N = 2 NPS) per MMA, every signedness combination of (A plane, B digit)
    constexpr uint32_t IDESC_H0 = (2u << 4) | ((uint32_t)(2 * NPS >> 3) << 17) | ((128u >> 4) << 24);
    constexpr uint32_t IDESC_UU = IDESC_H0, IDESC_US = IDESC_H0 | (1u << 10), IDESC_SU = IDESC_H0 | (1u << 7),
                       IDESC_SS = IDESC_H0 | (1u << 7) | (1u << 10);
    const TensorParams& p = pp.t;

    extern __shared__ unsigned char smem_raw[];
    const uint32_t base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t link_u32 = base;
    const uint32_t b_u32 = link_u32 + LS * LINK_STAGE;
    const uint32_t ft_u32 = b_u32 + AS * B_STAGE;
    const uint32_t bar_u32 = ft_u32 + FT * NPS * 4;
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
    const int n_mat_item = 9 - M0;
    // site sg (0 | 1) of a work item; the second half of the last item of an odd site count re-computes the first
    // site (valid memory, constant byte counts) and does not store
    auto site_valid = [&](int item, int sg) -> bool { return NS == 1 || 2 * item + sg < p.n_sites; };
    auto site_of_item = [&](int item, int sg = 0) -> int {
        int h = NS == 2 ? 2 * item + (site_valid(item, sg) ? sg : 0) : (NT == 1 ? item : item / NT);
        h += p.site_begin;
        return p.parity != 2 ? parity_site(p.lat, h, p.parity) : h;
    };

    if (warp == 0) {
        // ---------------------------------------------------------------- TMA producer
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
                    mat_row0[sg] = (sm * 9 + m) * NC;
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
                            if (!DAG)      // rows [i0, i0 + MT) x complex columns [KC c, KC c + KC)
                                ptx::tma_load_2d(dst, &link_map, c * KC, mat_row0[sg] + i0, full0 + 8u * slot, pol_links);
                            else           // rows [KC c, KC c + KC) x complex columns [i0, i0 + MT)
                                ptx::tma_load_2d(dst, &link_map, i0, mat_row0[sg] + KC * c, full0 + 8u * slot, pol_links);
                        }
                    }
                    __syncwarp();
                }
            }
        }
    } else if (warp == 1) {
        // ---------------------------------------------------------------- MMA issuer (one elected lane, uniform control flow)
        uint32_t t = 0;
        const uint32_t n_mat = (uint32_t)n_my * (uint32_t)n_mat_item;
        for (uint32_t tm = 0; tm < n_mat; ++tm) {
            const uint32_t ds = tm % DS, dph = (tm / DS) & 1u;
            ptx::mbar_wait(dempty0 + 8u * ds, dph ^ 1u);
            ptx::tc_fence_after();
            // high-byte plane one digit block above the low-byte plane: equal weights share columns
            const uint32_t d0 = tmem_base + Gm::D_COL0 + ds * Gm::D_COLS, d1 = d0 + 2 * NPS;
#pragma unroll 1
            for (int c = 0; c < CHUNKS; ++c, ++t) {
                const uint32_t as = t % AS, aph = (t / AS) & 1u;
                ptx::mbar_wait(abfull0 + 8u * as, aph);
                ptx::tc_fence_after();
                if (ptx::elect_one()) {
                    const uint32_t a1 = tmem_base + as * Gm::A_COLS, a0 = a1 + Gm::A_HALF;
                    const uint64_t db0 = umma_desc_kmajor(b_u32 + as * B_STAGE, 128, B_SBO);
#pragma unroll
                    for (int kk = 0; kk < Gm::KSTEPS; ++kk) {
                        const uint64_t db = db0 + (uint64_t)(kk * 256 >> 4);
                        if constexpr (HV) {
                            const uint64_t db_hi = db + (uint64_t)(((2 * NPS >> 3) * B_SBO) >> 4);     // second digit block: high bytes
                            const uint32_t acc = (c == 0 && kk == 0) ? 0u : 1u;                         // first k-step of the matrix overwrites
                            ptx::mma_i8_ts(d0, a0 + kk * 8, db, IDESC_UU, acc);                         // W_0  = A0.B0
                            ptx::mma_i8_ts(d0 + 2 * NPS, a0 + kk * 8, db_hi, IDESC_US, acc);            // W_1  = A0.B1
                            ptx::mma_i8_ts(d0 + 2 * NPS, a1 + kk * 8, db, IDESC_SU, 1u);                // W_1 += A1.B0
                            ptx::mma_i8_ts(d0 + 4 * NPS, a1 + kk * 8, db_hi, IDESC_SS, acc);            // W_2  = A1.B1
                        } else if (c == 0 && kk == 0) {
                            // first k-step of the matrix: W_1 .. W_3 = high plane (overwrite), W_0 = low plane digit 0
                            // (overwrite), W_1, W_2 += low plane digits 1, 2
                            ptx::mma_i8_ts(d1, a1, db, IDESC_S, 0u);
                            ptx::mma_i8_ts(d0, a0, db, IDESC_U1, 0u);
                            ptx::mma_i8_ts(d1, a0, db + (uint64_t)(((2 * NPS >> 3) * B_SBO) >> 4), IDESC_U2, 1u);
                        } else {
                            ptx::mma_i8_ts(d1, a1 + kk * 8, db, IDESC_S, 1u);
                            ptx::mma_i8_ts(d0, a0 + kk * 8, db, IDESC_U, 1u);
                        }
                    }
                    ptx::tc_commit(abempty0 + 8u * as);
                    if (c == CHUNKS - 1) ptx::tc_commit(dfull0 + 8u * ds);
                }
                __syncwarp();
            }
        }
    } else if (warp >= Gm::CONV_W0 && warp < Gm::EPI_W0) {
        // ---------------------------------------------------------------- converters
        constexpr int NG = Gm::NG;
        const int grp = (warp - Gm::CONV_W0) >> 2;
        const int q = warp & 3;
        const int lane_row = q * 32 + lane;                           // TMEM lane
        const int sg_row = NS == 2 ? lane_row >> 6 : 0;               // site of the item whose matrix row this lane converts
        const int row = NS == 2 ? lane_row & 63 : lane_row;
        const int gtid = ((warp - Gm::CONV_W0) & 3) * 32 + lane;
        const uint32_t lane_addr = (uint32_t)(q * 32) << 16;
        const uint32_t total = (uint32_t)n_my * (uint32_t)(n_mat_item * CHUNKS);

        // B entries of this thread: contraction row j (of the stage's KC) and column r, the same in every stage;
        // every entry of a thread has the same r.  e = gtid + 128 x: bits 0-2 = r mod 8 (16-byte rows of the K-major
        // layout: banks 4 apart), bits 3-4 = j mod 4 (bytes 2 apart / next word) - for the 4-wide tile bits 0-1 = r and
        // bits 2-4 = j mod 8 -, bit 5 = r div 8 (NP = 16) or the site sg (two sites per item), rest = the high part of j:
        // the 32 lanes of a 16-bit store touch 16 distinct words in 16 distinct banks (conflict-free).
        constexpr int RB = NP >= 8 ? 3 : 2, JB = 5 - RB;              // lane bits of r and of j
        constexpr int R8B = NP == 16 ? 1 : 0;                         // thread-index bit 5 = r div 8 (16-wide tile), the next bit = site
        const int my_r = (gtid & ((1 << RB) - 1)) + (R8B ? ((gtid >> 5) & 1) * 8 : 0);
        const int my_sg = NS == 2 ? (gtid >> (5 + R8B)) & 1 : 0;      // every B entry of a thread belongs to ONE site of the item
        const int my_n = my_sg * 2 * NP + my_r;                       // column inside a digit block
        const bool r_valid = my_r < p.width;
        int b_off_vec[NE];
        uint32_t b_o[NE];              // byte offset of (k = 2j, n = r, digit 0) in the B tile
#pragma unroll
        for (int x = 0; x < NE; ++x) {
            const int e = gtid + 128 * x;
            const int j = ((e >> RB) & ((1 << JB) - 1)) + (1 << JB) * (e >> (5 + R8B + (NS == 2 ? 1 : 0)));
            b_off_vec[x] = j * p.nrhs + my_r;
            const int k = 2 * j;
            b_o[x] = (uint32_t)(k >> 4) * 128u + (uint32_t)(my_n >> 3) * B_SBO + (uint32_t)(my_n & 7) * 16u + (uint32_t)(k & 15);
        }
        constexpr uint32_t N_STEP = (uint32_t)(NP >> 3) * B_SBO + (uint32_t)(NP & 7) * 16u;   // byte step of NP columns of n (Re -> Im block)
        constexpr uint32_t D_STEP = (uint32_t)(2 * NPS >> 3) * B_SBO;                          // byte step of one digit block (2 NPS columns)

        int n_it = 0, n_m = M0, n_c = grp, n_s = 0;
        SiteX n_cx = {};
        const VecT* n_vec = reinterpret_cast<const VecT*>(p.in);
        float n_g = 0.f, n_f = 0.f;       // fixed-point scale g 2^22 of the operand, epilogue factor of the matrix
        auto load_item = [&]() {
            if (n_it < n_my) {
                n_s = site_of_item(blockIdx.x + n_it * gridDim.x, my_sg);
                n_cx = site_coords(p.lat, n_s);
            }
        };
        auto load_matrix = [&]() {
            if (n_it < n_my) {
                const int sv = stencil_site_x(p.lat, n_s, n_cx, n_m, DAG ? 1 : 0);
                const int sm = DAG ? sv : n_s;
                n_vec = reinterpret_cast<const VecT*>(n_m == 0 ? p.in_local : p.in) + (int64_t)sv * NC * p.nrhs + p.r0;
                if constexpr (HV) {
                    const float nm = r_valid ? __ldg(pp.vnorms + (int64_t)sv * p.nrhs + p.r0 + my_r) : 0.f;
                    n_f = (n_m == 0 ? p.alpha : p.beta) * __ldg(p.scales + (int64_t)sm * 9 + n_m) * nm;
                    return;
                }
                const float2 gs = r_valid ? __ldg(reinterpret_cast<const float2*>(n_m == 0 ? pp.vscale_u : pp.vscale_w) + (int64_t)sv * TENSOR_I8_GP + my_r)
                                          : make_float2(0.f, 0.f);
                n_g = gs.x * 4194304.f;
                n_f = (n_m == 0 ? p.alpha : p.beta) * __ldg(p.scales + (int64_t)sm * 9 + n_m) * gs.y * (1.f / 4194304.f);
            }
        };
        VecT vn[NE];
        auto fetch = [&]() {
#pragma unroll
            for (int x = 0; x < NE; ++x)
                vn[x] = (n_it < n_my && r_valid) ? __ldg(n_vec + (int64_t)(KC * n_c) * p.nrhs + b_off_vec[x]) : VecT{};
        };
        auto normalise = [&]() -> bool {
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
        // matrix counter of the stage being converted (for the factor ring): stage t belongs to matrix t / CHUNKS
        for (uint32_t t = grp; t < total; t += NG) {
            const uint32_t slot = t % LS, ph = (t / LS) & 1u;
            const uint32_t as = t % AS, aph = (t / AS) & 1u;
            VecT v[NE];
#pragma unroll
            for (int x = 0; x < NE; ++x) v[x] = vn[x];
            const float g = n_g, f = n_f;
            const bool first_chunk = n_c == 0;
            n_c += NG;
            if (n_c >= CHUNKS) {
                if (normalise()) load_item();
                load_matrix();
            }
            fetch();

            ptx::mbar_wait(full0 + 8u * slot, ph);
            uint32_t w[KC];                                   // the lane's KC link entries (re, im) int16
            if (row < MT) {
                const uint32_t sb = link_u32 + slot * LINK_STAGE + sg_row * SLAB_PITCH;
                if constexpr (!DAG) {
                    const uint32_t rb = sb + row * (KC * 4);
#pragma unroll
                    for (int u = 0; u < KC / 4; ++u) {
                        const uint32_t sw = KC == 32 ? ((uint32_t)row & 7u) : (((uint32_t)row >> 1) & 3u);   // SWIZZLE_128B | 64B
                        const uint4 x = ptx::lds128u(rb + (((uint32_t)u ^ sw) << 4));
                        w[4 * u] = x.x; w[4 * u + 1] = x.y; w[4 * u + 2] = x.z; w[4 * u + 3] = x.w;
                    }
                } else {
                    const uint32_t cb = sb + row * 4;
#pragma unroll
                    for (int jj = 0; jj < KC; ++jj) w[jj] = ptx::lds32(cb + jj * (MT * 4));
                }
            } else {
#pragma unroll
                for (int u = 0; u < KC; ++u) w[u] = 0u;
            }

            ptx::mbar_wait(abempty0 + 8u * as, aph ^ 1u);
            ptx::tc_fence_after();
            // A operand: high bytes (signed) and low bytes (unsigned), k = 2j (re), 2j + 1 (im): 4 per TMEM column
            uint32_t a1[KC / 2], a0[KC / 2];
#pragma unroll
            for (int c2 = 0; c2 < KC / 2; ++c2) {
                a1[c2] = __byte_perm(w[2 * c2], w[2 * c2 + 1], 0x7531);
                a0[c2] = __byte_perm(w[2 * c2], w[2 * c2 + 1], 0x6420);
            }
            const uint32_t a1_t = tmem_base + lane_addr + as * Gm::A_COLS, a0_t = a1_t + Gm::A_HALF;
            if constexpr (KC == 32) {
                ptx::tmem_st16(a1_t, a1);
                ptx::tmem_st16(a0_t, a0);
            } else {
                ptx::tmem_st8(a1_t, a1);
                ptx::tmem_st8(a0_t, a0);
            }
            // B operand: fixed point, three signed digits, [Re out | Im out] x 3 along n
            const uint32_t bt = b_u32 + as * B_STAGE;
#pragma unroll
            for (int x = 0; x < NE; ++x) {
                if constexpr (HV) {
                    // the int16 components are the fixed-point operand: low bytes (unsigned) into block 0, high bytes
                    // (signed) into block 1; -q is formed in 32 bits (|q| <= 32767 by the quantiser; -32768 would still be
                    // exact here: its two's complement bytes are taken from the 32-bit negative)
                    const uint32_t w = v[x];
                    const int re = (int)(w << 16) >> 16, im = (int)w >> 16;
                    const int b1x = re, b1y = DAG ? im : -im;                                  // n = r      (-> Re out)
                    const int b2x = im, b2y = DAG ? -re : re;                                  // n = NP + r (-> Im out)
                    ptx::sts16(bt + b_o[x], pack_lo_bytes(b1x, b1y));
                    ptx::sts16(bt + b_o[x] + D_STEP, __byte_perm((uint32_t)b1x, (uint32_t)b1y, 0x0051));
                    ptx::sts16(bt + b_o[x] + N_STEP, pack_lo_bytes(b2x, b2y));
                    ptx::sts16(bt + b_o[x] + N_STEP + D_STEP, __byte_perm((uint32_t)b2x, (uint32_t)b2y, 0x0051));
                } else {
                const float vx = v[x].x * g, vy = v[x].y * g;
                const int b1x = __float2int_rn(vx), b1y = __float2int_rn(DAG ? vy : -vy);     // n = r      (-> Re out)
                const int b2x = __float2int_rn(vy), b2y = __float2int_rn(DAG ? -vx : vx);     // n = NP + r (-> Im out)
                int x1, x2, y1, y2;
                digit_regs(b1x, x1, x2);
                digit_regs(b1y, y1, y2);
                ptx::sts16(bt + b_o[x], pack_lo_bytes(b1x, b1y));
                ptx::sts16(bt + b_o[x] + D_STEP, pack_lo_bytes(x1, y1));
                ptx::sts16(bt + b_o[x] + 2 * D_STEP, pack_lo_bytes(x2, y2));
                digit_regs(b2x, x1, x2);
                digit_regs(b2y, y1, y2);
                ptx::sts16(bt + b_o[x] + N_STEP, pack_lo_bytes(b2x, b2y));
                ptx::sts16(bt + b_o[x] + N_STEP + D_STEP, pack_lo_bytes(x1, y1));
                ptx::sts16(bt + b_o[x] + N_STEP + 2 * D_STEP, pack_lo_bytes(x2, y2));
                }
            }
            // epilogue factor of this matrix and column: written by the group that converts the matrix's first chunk
            if (first_chunk && (gtid & (0x1f & ~((1 << RB) - 1))) == 0 && gtid < (32 << (R8B + (NS == 2 ? 1 : 0)))) {
                // threads 0-7 (and 32-39 for NP = 16 / the second site) of the group hold r = 0..7 (8..15 / r = 0..7 of site 1);
                // 4-wide tile: threads 0-3 and 32-35
                asm volatile("st.shared.f32 [%0], %1;" ::"r"(ft_u32 + (uint32_t)(((t / CHUNKS) % FT) * NPS + my_sg * NP + my_r) * 4u), "f"(f) : "memory");
            }
            ptx::tc_wait_st();
            ptx::fence_proxy_async();
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(abfull0 + 8u * as);
            // link slot back to the producer: after the loaded entries have gone into tensor memory (see tensor_kernel.cuh)
            if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
        }
    } else if (warp >= Gm::EPI_W0) {
        // ---------------------------------------------------------------- epilogue
        const int q = warp & 3;
        const int lane_row = q * 32 + lane;
        const int sg_row = NS == 2 ? lane_row >> 6 : 0;               // warp-uniform
        const int row = NS == 2 ? lane_row & 63 : lane_row;
        const uint32_t lane_addr = (uint32_t)(q * 32) << 16;
        uint32_t tm = 0;
        for (int it = 0; it < n_my; ++it) {
            const int item = blockIdx.x + it * gridDim.x;
            const int s = site_of_item(item, sg_row);
            const int i0 = NT == 1 ? 0 : (item % NT) * MT;
            float acc[2 * NP];
#pragma unroll
            for (int n = 0; n < 2 * NP; ++n) acc[n] = 0.f;
#pragma unroll 1
            for (int m = M0; m < 9; ++m, ++tm) {
                const uint32_t ds = tm % DS, dph = (tm / DS) & 1u;
                ptx::mbar_wait(dfull0 + 8u * ds, dph);
                ptx::tc_fence_after();
                const uint32_t d_t = tmem_base + lane_addr + Gm::D_COL0 + ds * Gm::D_COLS + sg_row * 2 * NP;   // this row's site
                const uint32_t ft = ft_u32 + (uint32_t)((tm % FT) * NPS + sg_row * NP) * 4u;
                // 8 columns of n at a time: the four weight blocks W_3 .. W_0, Horner in fp32
#pragma unroll
                for (int pc = 0; pc < 2 * NP / 8; ++pc) {
                    uint32_t w3[8], w2[8], w1[8], w0[8];
                    if constexpr (!HV) ptx::tmem_ld8(d_t + 3 * 2 * NPS + 8 * pc, w3);
                    ptx::tmem_ld8(d_t + 2 * 2 * NPS + 8 * pc, w2);
                    ptx::tmem_ld8(d_t + 1 * 2 * NPS + 8 * pc, w1);
                    ptx::tmem_ld8(d_t + 8 * pc, w0);
                    ptx::tc_wait_ld();
#pragma unroll
                    for (int n = 0; n < 8; ++n) {
                        float S = HV ? (float)(int)w2[n] : fmaf((float)(int)w3[n], 256.f, (float)(int)w2[n]);
                        S = fmaf(S, 256.f, (float)(int)w1[n]);
                        S = fmaf(S, 256.f, (float)(int)w0[n]);
                        float fr;
                        asm volatile("ld.shared.f32 %0, [%1];" : "=f"(fr) : "r"(ft + (uint32_t)((8 * pc + n) % NP) * 4u));
                        acc[8 * pc + n] = fmaf(fr, S, acc[8 * pc + n]);
                    }
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
