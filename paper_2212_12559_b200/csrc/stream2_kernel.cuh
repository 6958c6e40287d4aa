// stream2_kernel.cuh — the 1-RHS STREAM apply with stages owned by small warp TEAMS (large lattices).
//
// Why a second mapping.  In stream_kernel.cuh the eight consumer warps of a CTA share every pipeline
// stage (each takes 1/8 of its rows), so everything that is done once per stage - the mbarrier
// wait, the scale shuffle, loading and scaling the vector operand, address arithmetic, the slot
// release - is executed by all eight warps.  ncu on BASELINE config C4 (int16 links, the paper's storage
// format) counts 155 executed instructions per warp and 16 KB stage of which only 84 are
// the decode + FMA work on the link bytes; at the ~1.55 GHz the 1000 W power cap leaves this kernel in
// a sustained loop, the SM side - not HBM - sets the time (profiles/r02_ncu_full_c4_*.md).
//
// Here the eight consumer warps form T = 8 / TW teams of TW warps; a team owns whole work items and
// every T-th stage of the ring, so the per-stage overhead is paid by TW warps instead of 8:
//   dagger = 0: item = (site, block of RS rows); 9 stages (one per matrix m); warp wi of the team takes
//               RS / TW rows, keeps acc[WL] per lane and reduces over its column slices once per item
//               with a transposing butterfly (each shuffle step halves the live values).
//   dagger = 1: item = site; 9 * Nc/RS stages of RS contraction rows; lane <-> output columns; the TW
//               warps' partial sums meet once per item in a small double-buffered shared-memory area
//               behind a team-wide named barrier (no CTA-wide barrier).
// The FEED is unchanged - it is what the memory system likes (measured with coarse_op_probe_read on this
// chip: one sequential stream per SM of >= 8 KB copies with ~100 KB in flight reads 7.4 TB/s; 4 KB
// copies 6.3 TB/s; 190 KB in flight 6.9 TB/s): one producer warp walks ONE ring of S = T * SW slots in a
// fixed global order (round, matrix, chunk, team), stage n going to team n mod T and slot n mod S, so
// every slot has a fixed owner (the parity waits stay sound) and S - T slots are in flight while each
// team works on one.  Versions with fully private rings (one warp per team, 8 KB stages fed by a lane per
// ring, by the warps themselves, or by one producer) were tried first: they cut the instruction count by
// 25 % but starved the consumers or doubled the number of copies the single producer thread must issue,
// and stayed at 5.6-6.6 TB/s.  Measured on C4 (sustained, same box; cooperative kernel 2.28 / 2.50 ms):
// TW = 4 with 8 slots (6 in flight) 2.06 / 2.13 ms = 7.28 / 7.06 TB/s; 6 or 10 slots 2.18-2.26 ms; TW = 2
// with 8 / 12 slots (4 / 8 in flight) 2.20 / 2.17 ms.
// Small lattices keep the cooperative kernel of stream_kernel.cuh: with one item per team a lattice needs
// at least T x 148 items to occupy the chip.
//
// Lane mapping inside a stage, int16 decode, complex MAC and L2 policies are those of stream_kernel.cuh.
// The summation order is fixed by the static schedule: bit-identical run to run.
#pragma once
#include "stream_kernel.cuh"

// Words (of the 4) of every int16 link quad that are decoded through the conversion unit (I2F.S16 on the
// XU pipe: 2 issue slots per word) instead of the magic-number path (LOP3 + 2 PRMT + FADD2: 4 slots on the
// ALU / FMA pipes), see common.cuh.  Measured on C4, 200-step loops under the 1000 W cap (all variants in one
// gpurun call): dagger = 0  2.09 / 2.19 / 2.14 / 2.25 / 2.32 ms for 0 / 1 / 2 / 3 / 4 words,
//               dagger = 1  2.44 / 2.24-2.30 / 2.22-2.30 / - / 2.59 ms for 0 / 1 / 2 / 3 / 4.
#ifndef COARSE_S2_XU_N
#define COARSE_S2_XU_N 0
#endif
#ifndef COARSE_S2_XU_D
#define COARSE_S2_XU_D 1
#endif

// Complex MAC formulation (stream_kernel.cuh): 1 = matrix entry as the packed FFMA2 operand with two packed partial
// sums per accumulator (cmacp: no register-pair duplication MOVs, 300 -> 246 instructions per stage and lane),
// 0 = cmac<> (vector as the packed operand).  A/B in one gpurun call, 100-step loops, two repetitions each, int16
// links: dagger = 0 is SLOWER with the shorter instruction stream (C4 2.19 -> 2.27 ms, Nc = 128 0.513 -> 0.539 ms:
// 16 more live registers for the duplicated vector pairs and no issue-slot shortage left to relieve), dagger = 1 is
// 1 % faster (C4 2.235 -> 2.209 ms, Nc = 128 0.5072 -> 0.5026 ms).  The multi-RHS kernel (stream_mr_kernel.cuh),
// which IS issue-bound, gains 6-19 % from it in both modes.
#ifndef COARSE_S2_PACKED_N
#define COARSE_S2_PACKED_N 0
#endif
#ifndef COARSE_S2_PACKED_D
#define COARSE_S2_PACKED_D 1
#endif

namespace coarse {

constexpr int stream2_rows(int nc, int rowbytes, int unit, int max_bytes, int max_loads) {
    int best = 0;
    for (int d = unit; d <= nc; d += unit)
        if (nc % d == 0 && d * rowbytes <= max_bytes && d / unit <= max_loads) best = d;
    return best;
}

// HV: half-precision input vectors (coarse_op_apply_hvec) - `in` holds int16 (re, im) pairs, the per-site
// norm is folded into the per-matrix operand scale (as in stream_kernel.cuh), a vector stage is half the bytes.
template <int NC, bool I16, int TW, bool HV = false>
struct Stream2Geom {
    using G1 = StreamGeom<NC, I16, false, false, true>;      // all-lanes-busy lane mapping
    static constexpr int W = 8;                               // consumer warps
    static constexpr int T = W / TW;                          // teams
    static constexpr int ROWBYTES = G1::ROWBYTES, Q = G1::Q, CPQ = G1::CPQ, PASSES = G1::PASSES, QP = G1::QP;
    static constexpr int G = G1::G, RPL = G1::RPL;
    static constexpr int RS = stream2_rows(NC, ROWBYTES, TW * RPL, 16384, 16);   // rows per stage
    static constexpr int NB = NC / (RS > 0 ? RS : 1);
    static constexpr int WL = RS / (TW * RPL);                // warp-wide loads per warp, stage and pass
    static constexpr int LINK_STAGE = RS * ROWBYTES;
    static constexpr int VEC_ENTRY = HV ? 4 : 8;
    static constexpr int VEC_STAGE_N = NC * VEC_ENTRY;
    static constexpr int VEC_STAGE_D = RS * VEC_ENTRY;
    static constexpr int RED_BYTES = T * 2 * (TW - 1) * NC * 8;               // dagger = 1 team reduction
    static constexpr bool OK = G1::OK && RS > 0 && QP == G && (TW == 2 || TW == 4);
    static constexpr int THREADS = (W + 1) * 32;
    static constexpr int stage_bytes(bool dag) { return LINK_STAGE + (dag ? VEC_STAGE_D : VEC_STAGE_N); }
    static constexpr int HOUT_BYTES = 2 * W * 4;                              // half-precision output: per-warp maxima, double buffered
    static constexpr int fixed_bytes(bool dag) { return (dag ? RED_BYTES : 0) + 128 + HOUT_BYTES; }
    static int smem_bytes(bool dag, int slots) { return slots * (stage_bytes(dag) + 16) + fixed_bytes(dag); }
};

// Sum acc[0..N) over the lanes at xor distances O, O/2, .., 1 (the G lanes that hold the column slices
// of one row group).  While at least two values are live and their number is even, a step exchanges
// HALF of them (lanes with the step's bit clear keep the lower half), otherwise it is a plain butterfly:
// N + N/2 + ... shuffles instead of N log2(G).  On return acc[0 .. tr_final_n(N, O)) hold the totals of
// the values that were at indices k0 .. k0 + tr_final_n - 1 (k0 is returned); lanes that differ only in
// the bits of tr_plain_mask(N, O) hold the same values.
__host__ __device__ constexpr int tr_final_n(int n, int o) {
    for (; o >= 1; o /= 2)
        if (n >= 2 && n % 2 == 0) n /= 2;
    return n;
}
__host__ __device__ constexpr int tr_plain_mask(int n, int o) {
    int mask = 0;
    for (; o >= 1; o /= 2) {
        if (n >= 2 && n % 2 == 0) n /= 2;
        else mask |= o;
    }
    return mask;
}
template <int N, int O, int NTOT>
__device__ __forceinline__ int transpose_reduce(float2 (&acc)[NTOT], int lane_in_group, int k0) {
    if constexpr (O == 0) {
        return k0;
    } else if constexpr (N >= 2 && N % 2 == 0) {
        const bool hi = (lane_in_group & O) != 0;
#pragma unroll
        for (int k = 0; k < N / 2; ++k) {
            const float2 keep = hi ? acc[k + N / 2] : acc[k];
            const float2 send = hi ? acc[k] : acc[k + N / 2];
            float2 recv;
            recv.x = __shfl_xor_sync(0xffffffffu, send.x, O);
            recv.y = __shfl_xor_sync(0xffffffffu, send.y, O);
            acc[k] = make_float2(keep.x + recv.x, keep.y + recv.y);
        }
        return transpose_reduce<N / 2, O / 2, NTOT>(acc, lane_in_group, k0 + (hi ? N / 2 : 0));
    } else {
#pragma unroll
        for (int k = 0; k < N; ++k) {
            acc[k].x += __shfl_xor_sync(0xffffffffu, acc[k].x, O);
            acc[k].y += __shfl_xor_sync(0xffffffffu, acc[k].y, O);
        }
        return transpose_reduce<N, O / 2, NTOT>(acc, lane_in_group, k0);
    }
}

// Half-precision output (coarse_op_apply_hout): 16-bit component of x for the site norm `norm` (amax = 32767 norm), the
// arithmetic of quantize_vec_i16_kernel (R22).
__device__ __forceinline__ short2 half_out_q(float2 x, float amax, float norm) {
    short2 o = make_short2(0, 0);
    if (amax != 0.f) {
        o.x = (short)fminf(32767.f, fmaxf(-32767.f, rintf(__fdiv_rn(x.x, norm))));
        o.y = (short)fminf(32767.f, fmaxf(-32767.f, rintf(__fdiv_rn(x.y, norm))));
    }
    return o;
}

template <int NC, bool I16, bool DAG, int TW, bool HV = false>
__global__ void __launch_bounds__(Stream2Geom<NC, I16, TW, HV>::THREADS, 1) coarse_apply_stream2(StreamParams p) {
    using Gm = Stream2Geom<NC, I16, TW, HV>;
    constexpr int VE = Gm::VEC_ENTRY;
    constexpr bool SCALED = I16 || HV;                    // the vector operand carries a per-matrix scale
    static_assert(Gm::OK, "unsupported STREAM2 geometry");
    constexpr int W = Gm::W, T = Gm::T, RS = Gm::RS, NB = Gm::NB, WL = Gm::WL, QP = Gm::QP, G = Gm::G, RPL = Gm::RPL;
    constexpr int PASSES = Gm::PASSES, CPQ = Gm::CPQ, ROWBYTES = Gm::ROWBYTES;
    constexpr int LINK_STAGE = Gm::LINK_STAGE;
    constexpr int VEC_STAGE = DAG ? Gm::VEC_STAGE_D : Gm::VEC_STAGE_N;

    extern __shared__ __align__(128) unsigned char smem[];
    const int S = p.stages;                               // ring slots, a multiple of T
    unsigned char* link_smem = smem;
    unsigned char* vec_smem = link_smem + (size_t)S * LINK_STAGE;
    unsigned char* red_smem = vec_smem + (size_t)S * VEC_STAGE;
    uint64_t* bars = reinterpret_cast<uint64_t*>(red_smem + (DAG ? Gm::RED_BYTES : 0));
    const uint32_t full0 = ptx::smem_u32(bars);
    const uint32_t empty0 = full0 + 8u * S;
    float* hmax = reinterpret_cast<float*>(bars + 2 * S);            // [2][W]: half-precision output (dagger = 0)

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (threadIdx.x == 0) {
        for (int i = 0; i < S; ++i) {
            ptx::mbar_init(full0 + 8u * i, 1);
            ptx::mbar_init(empty0 + 8u * i, TW);
        }
        ptx::fence_mbar_init();
    }
    __syncthreads();

    const int item_stride = gridDim.x * T;
    const uint32_t link_u32 = ptx::smem_u32(link_smem), vec_u32 = ptx::smem_u32(vec_smem);

    if (warp == W) {
        // ------------------------------------------------------------------ producer
        // Global stage order: round (one item per team), matrix m, chunk c, team t.  The whole warp walks the
        // loops (uniform control flow), one elected lane issues.  Lane l holds the stencil sites of the item
        // of team (l mod T) for the matrices (l div T) + ML * h of the current round (a1).
        constexpr int ML = 32 / T, NH = (9 + ML - 1) / ML;
        const uint64_t pol_vec = ptx::policy_evict_last();
        const uint64_t pol_links = p.keep_links ? pol_vec : ptx::policy_evict_first();
        int slot = 0;
        uint32_t phase = 0;
        for (int base = p.item_begin + blockIdx.x * T; base < p.n_items; base += item_stride) {
            const int my_item = base + (lane % T);
            int svh[NH];
#pragma unroll
            for (int h = 0; h < NH; ++h) {
                const int mm = lane / T + ML * h;
                svh[h] = (my_item < p.n_items && mm < 9) ? stencil_site(p.lat, DAG ? my_item : my_item / NB, mm, DAG ? 1 : 0) : 0;
            }
#pragma unroll
            for (int m = 0; m < 9; ++m) {
#pragma unroll 1
                for (int c = 0; c < (DAG ? NB : 1); ++c) {
#pragma unroll 1
                    for (int t = 0; t < T; ++t) {
                        const int item = base + t;
                        const int sv = __shfl_sync(0xffffffffu, svh[m / ML], (m % ML) * T + t);
                        ptx::mbar_wait(empty0 + 8u * slot, phase ^ 1u);
                        if (item < p.n_items) {
                            const int s = DAG ? item : item / NB;
                            const int sm = DAG ? sv : s;
                            const int r0 = DAG ? c * RS : (item % NB) * RS;
                            const unsigned char* mat = p.links + ((int64_t)sm * 9 + m) * ((int64_t)NC * ROWBYTES) + (int64_t)r0 * ROWBYTES;
                            const unsigned char* vec = reinterpret_cast<const unsigned char*>(p.in) + ((int64_t)sv * NC + (DAG ? r0 : 0)) * VE;
                            if (ptx::elect_one()) {
                                ptx::mbar_arrive_expect_tx(full0 + 8u * slot, LINK_STAGE + VEC_STAGE);
                                ptx::bulk_g2s(link_u32 + slot * LINK_STAGE, mat, LINK_STAGE, full0 + 8u * slot, pol_links);
                                ptx::bulk_g2s(vec_u32 + slot * VEC_STAGE, vec, VEC_STAGE, full0 + 8u * slot, pol_vec);
                            }
                        } else {
                            // ragged last round: no stage for this team; complete the slot's `full` and `empty`
                            // phases anyway so that the slot's parity sequence stays intact
                            if (ptx::elect_one()) {
                                ptx::mbar_arrive(full0 + 8u * slot);
#pragma unroll
                                for (int a = 0; a < TW; ++a) ptx::mbar_arrive(empty0 + 8u * slot);
                            }
                        }
                        __syncwarp();
                        if (++slot == S) { slot = 0; phase ^= 1u; }
                    }
                }
            }
        }
        return;
    }

    // ---------------------------------------------------------------------- consumers: stage n -> team n mod T
    const int team = warp / TW, wi = warp % TW;
    const int grp = lane / G;          // which of the RPL rows of a warp-wide load
    const int qi = lane % G;           // quad index inside the pass
    const int row0 = wi * (WL * RPL) + grp;     // this lane's first row of a stage; further rows every RPL
    const int item0 = p.item_begin + blockIdx.x * T + team;     // item_begin: site-range launches (coarse_op_apply_host)
    int slot = team;                   // this team's slots: team, team + T, ..
    uint32_t phase = 0;
    auto next_slot = [&]() {
        slot += T;
        if (slot >= S) { slot -= S; phase ^= 1u; }
    };
    int red_buf = 0;

    // int16: lane m (< 9) carries the fp32 scale of matrix m of the current item, fetched two items ahead
    float cur_scale = 1.f, next_scale = 1.f, next2_scale = 1.f;
    auto fetch_scale = [&](int item) -> float {
        if (!SCALED || lane >= 9 || item >= p.n_items) return 1.f;
        const int s = DAG ? item : item / NB;
        const int sv = (DAG || HV) ? stencil_site(p.lat, s, lane, DAG ? 1 : 0) : s;    // site of stage `lane`'s vector
        const int sm = DAG ? sv : s;
        float f = 1.f;
        if constexpr (I16) f = __ldg(p.scales + (int64_t)sm * 9 + lane);
        if constexpr (HV) f *= __ldg(p.vnorms + sv);                                  // half vectors: per-site norm folded in
        return f;
    };
    next_scale = fetch_scale(item0);
    next2_scale = fetch_scale(item0 + item_stride);

    for (int item = item0; item < p.n_items; item += item_stride) {
        const int s = DAG ? item : item / NB;
        const int rb = DAG ? 0 : item % NB;
        cur_scale = next_scale;
        next_scale = next2_scale;
        next2_scale = fetch_scale(item + 2 * item_stride);

        if constexpr (!DAG) {
#if COARSE_S2_PACKED_N
            static_assert(!HV, "half vectors are implemented in the cmac<> formulation of dagger = 0");
            CAcc pacc[WL];
#pragma unroll
            for (int k = 0; k < WL; ++k) pacc[k].a = pacc[k].b = make_float2(0.f, 0.f);
#pragma unroll 1
            for (int m = 0; m < 9; ++m) {
                const float sc = SCALED ? __shfl_sync(0xffffffffu, cur_scale, m) : 1.f;
                ptx::mbar_wait(full0 + 8u * slot, phase);
                const uint32_t lbase = link_u32 + slot * LINK_STAGE + (row0 * ROWBYTES + qi * 16);
                const uint32_t vbase = vec_u32 + slot * VEC_STAGE;
                VDup v[PASSES][CPQ];
#pragma unroll
                for (int ps = 0; ps < PASSES; ++ps) {
                    const int col0 = (ps * QP + qi) * CPQ;
#pragma unroll
                    for (int h = 0; h < CPQ / 2; ++h) {
                        float4 t = ptx::lds128(vbase + (col0 + 2 * h) * 8);
                        if constexpr (I16) { t.x *= sc; t.y *= sc; t.z *= sc; t.w *= sc; }
                        v[ps][2 * h] = vdup(make_float2(t.x, t.y));
                        v[ps][2 * h + 1] = vdup(make_float2(t.z, t.w));
                    }
                }
#pragma unroll
                for (int k = 0; k < WL; ++k) {
#pragma unroll
                    for (int ps = 0; ps < PASSES; ++ps) {
                        const uint32_t a = lbase + k * (RPL * ROWBYTES) + ps * QP * 16;
                        if constexpr (I16) {
                            const uint4 t = ptx::lds128u(a);
                            float2 m0, m1, m2, m3;
                            unpack_i16_quad<COARSE_S2_XU_N>(t, m0, m1, m2, m3);
                            cmacp(pacc[k], m0, v[ps][0]);
                            cmacp(pacc[k], m1, v[ps][1]);
                            cmacp(pacc[k], m2, v[ps][2]);
                            cmacp(pacc[k], m3, v[ps][3]);
                        } else {
                            const float4 t = ptx::lds128(a);
                            cmacp(pacc[k], make_float2(t.x, t.y), v[ps][0]);
                            cmacp(pacc[k], make_float2(t.z, t.w), v[ps][1]);
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
                next_slot();
            }
            float2 acc[WL];
#pragma unroll
            for (int k = 0; k < WL; ++k) acc[k] = cfinal<false>(pacc[k]);
#else
            float2 acc[WL];
#pragma unroll
            for (int k = 0; k < WL; ++k) acc[k] = make_float2(0.f, 0.f);
#pragma unroll 1
            for (int m = 0; m < 9; ++m) {
                const float sc = SCALED ? __shfl_sync(0xffffffffu, cur_scale, m) : 1.f;
                ptx::mbar_wait(full0 + 8u * slot, phase);
                const uint32_t lbase = link_u32 + slot * LINK_STAGE + (row0 * ROWBYTES + qi * 16);
                const uint32_t vbase = vec_u32 + slot * VEC_STAGE;
                float2 v[PASSES][CPQ];
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
                    if constexpr (SCALED) {
#pragma unroll
                        for (int e = 0; e < CPQ; ++e) { v[ps][e].x *= sc; v[ps][e].y *= sc; }
                    }
                }
#pragma unroll
                for (int k = 0; k < WL; ++k) {
#pragma unroll
                    for (int ps = 0; ps < PASSES; ++ps) {
                        const uint32_t a = lbase + k * (RPL * ROWBYTES) + ps * QP * 16;
                        if constexpr (I16) {
                            const uint4 t = ptx::lds128u(a);
                            float2 m0, m1, m2, m3;
                            unpack_i16_quad<COARSE_S2_XU_N>(t, m0, m1, m2, m3);
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
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
                next_slot();
            }
#endif
            // a6: combine the column-slice partial sums, once per item
            const int k0 = transpose_reduce<WL, G / 2, WL>(acc, qi, 0);
            constexpr int NF = tr_final_n(WL, G / 2);
            constexpr int PLAIN = tr_plain_mask(WL, G / 2);
            if ((qi & PLAIN) == 0) {
#pragma unroll
                for (int j = 0; j < NF; ++j) p.out[(int64_t)s * NC + rb * RS + row0 + (k0 + j) * RPL] = acc[j];
            }
            if constexpr (NB == 1) {
                // half-precision result beside it (the launcher sends hout here only when an item is a whole site): the
                // site's rows are spread over the team's lanes, so the team takes the maximum through hmax[buf][warp]
                // behind ONE team-wide named barrier (double buffered: the next item's barrier orders the reuse), then every
                // lane quantises the rows it holds
                if (p.hout_q) {
                    float amax = 0.f;
                    if ((qi & PLAIN) == 0) {
#pragma unroll
                        for (int j = 0; j < NF; ++j) amax = fmaxf(amax, fmaxf(fabsf(acc[j].x), fabsf(acc[j].y)));
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
                    if (lane == 0) hmax[red_buf * W + warp] = amax;
                    ptx::named_bar_sync(1 + team, TW * 32);
                    amax = 0.f;
#pragma unroll
                    for (int w = 0; w < TW; ++w) amax = fmaxf(amax, hmax[red_buf * W + team * TW + w]);
                    red_buf ^= 1;
                    const float norm = amax == 0.f ? 0.f : __fdiv_rn(amax, 32767.0f);
                    if (wi == 0 && lane == 0) p.hout_norms[s] = norm;
                    if ((qi & PLAIN) == 0) {
                        short2* hq = p.hout_q;
#pragma unroll
                        for (int j = 0; j < NF; ++j) hq[(int64_t)s * NC + row0 + (k0 + j) * RPL] = half_out_q(acc[j], amax, norm);
                    }
                }
            }
        } else {
#if COARSE_S2_PACKED_D
            CAcc pacc[PASSES][CPQ];
#pragma unroll
            for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
                for (int e = 0; e < CPQ; ++e) pacc[ps][e].a = pacc[ps][e].b = make_float2(0.f, 0.f);
#pragma unroll 1
            for (int m = 0; m < 9; ++m) {
                const float sc = SCALED ? __shfl_sync(0xffffffffu, cur_scale, m) : 1.f;
#pragma unroll 1
                for (int c = 0; c < NB; ++c) {
                    ptx::mbar_wait(full0 + 8u * slot, phase);
                    const uint32_t lbase = link_u32 + slot * LINK_STAGE + (row0 * ROWBYTES + qi * 16);
                    const uint32_t vbase = vec_u32 + slot * VEC_STAGE + row0 * VE;
#pragma unroll
                    for (int k = 0; k < WL; ++k) {
                        float2 vj;
                        if constexpr (HV) {
                            uint32_t w;
                            asm volatile("ld.shared.u32 %0, [%1];" : "=r"(w) : "r"(vbase + k * (RPL * 4)));
                            vj = unpack_i16x2(w);
                        } else {
                            vj = ptx::lds64(vbase + k * (RPL * 8));
                        }
                        if constexpr (SCALED) { vj.x *= sc; vj.y *= sc; }
                        const VDup vd = vdup(vj);
#pragma unroll
                        for (int ps = 0; ps < PASSES; ++ps) {
                            const uint32_t a = lbase + k * (RPL * ROWBYTES) + ps * QP * 16;
                            if constexpr (I16) {
                                const uint4 t = ptx::lds128u(a);
                                float2 m0, m1, m2, m3;
                                unpack_i16_quad<COARSE_S2_XU_D>(t, m0, m1, m2, m3);
                                cmacp(pacc[ps][0], m0, vd);
                                cmacp(pacc[ps][1], m1, vd);
                                cmacp(pacc[ps][2], m2, vd);
                                cmacp(pacc[ps][3], m3, vd);
                            } else {
                                const float4 t = ptx::lds128(a);
                                cmacp(pacc[ps][0], make_float2(t.x, t.y), vd);
                                cmacp(pacc[ps][1], make_float2(t.z, t.w), vd);
                            }
                        }
                    }
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
                    next_slot();
                }
            }
            float2 acc[PASSES][CPQ];
#pragma unroll
            for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
                for (int e = 0; e < CPQ; ++e) acc[ps][e] = cfinal<true>(pacc[ps][e]);
#else
            static_assert(!HV, "half vectors are implemented in the packed formulation of dagger = 1");
            float2 acc[PASSES][CPQ];
#pragma unroll
            for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
                for (int e = 0; e < CPQ; ++e) acc[ps][e] = make_float2(0.f, 0.f);
#pragma unroll 1
            for (int m = 0; m < 9; ++m) {
                const float sc = SCALED ? __shfl_sync(0xffffffffu, cur_scale, m) : 1.f;
#pragma unroll 1
                for (int c = 0; c < NB; ++c) {
                    ptx::mbar_wait(full0 + 8u * slot, phase);
                    const uint32_t lbase = link_u32 + slot * LINK_STAGE + (row0 * ROWBYTES + qi * 16);
                    const uint32_t vbase = vec_u32 + slot * VEC_STAGE + row0 * 8;
#pragma unroll
                    for (int k = 0; k < WL; ++k) {
                        float2 vj = ptx::lds64(vbase + k * (RPL * 8));
                        if constexpr (I16) { vj.x *= sc; vj.y *= sc; }
#pragma unroll
                        for (int ps = 0; ps < PASSES; ++ps) {
                            const uint32_t a = lbase + k * (RPL * ROWBYTES) + ps * QP * 16;
                            if constexpr (I16) {
                                const uint4 t = ptx::lds128u(a);
                                float2 m0, m1, m2, m3;
                                unpack_i16_quad<COARSE_S2_XU_D>(t, m0, m1, m2, m3);
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
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
                    next_slot();
                }
            }
#endif
            // a6: combine the RPL row-group partial sums of the warp (lanes qi, qi + G, ...), then the TW warps'
#pragma unroll
            for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
                for (int e = 0; e < CPQ; ++e)
#pragma unroll
                    for (int o = 16; o >= G; o >>= 1) {
                        acc[ps][e].x += __shfl_xor_sync(0xffffffffu, acc[ps][e].x, o);
                        acc[ps][e].y += __shfl_xor_sync(0xffffffffu, acc[ps][e].y, o);
                    }
            if constexpr (TW > 1) {
                float4* red = reinterpret_cast<float4*>(red_smem) + (size_t)((team * 2 + red_buf) * (TW - 1)) * (NC / 2);
                if (wi > 0 && grp == 0) {
#pragma unroll
                    for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
                        for (int h = 0; h < CPQ / 2; ++h)
                            red[(wi - 1) * (NC / 2) + ((ps * QP + qi) * CPQ) / 2 + h] =
                                make_float4(acc[ps][2 * h].x, acc[ps][2 * h].y, acc[ps][2 * h + 1].x, acc[ps][2 * h + 1].y);
                }
                ptx::named_bar_sync(1 + team, TW * 32);
                if (wi == 0 && grp == 0) {
#pragma unroll
                    for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
                        for (int h = 0; h < CPQ / 2; ++h)
#pragma unroll
                            for (int o = 0; o < TW - 1; ++o) {
                                const float4 x = red[o * (NC / 2) + ((ps * QP + qi) * CPQ) / 2 + h];
                                acc[ps][2 * h].x += x.x;
                                acc[ps][2 * h].y += x.y;
                                acc[ps][2 * h + 1].x += x.z;
                                acc[ps][2 * h + 1].y += x.w;
                            }
                }
                red_buf ^= 1;
            }
            if (wi == 0 && grp == 0) {
#pragma unroll
                for (int ps = 0; ps < PASSES; ++ps) {
                    float4* dst = reinterpret_cast<float4*>(p.out + (int64_t)s * NC + (ps * QP + qi) * CPQ);
#pragma unroll
                    for (int h = 0; h < CPQ / 2; ++h)
                        dst[h] = make_float4(acc[ps][2 * h].x, acc[ps][2 * h].y, acc[ps][2 * h + 1].x, acc[ps][2 * h + 1].y);
                }
            }
            // half-precision result: the whole site sits in the grp == 0 lanes of the team's first warp - one warp-wide maximum
            if (p.hout_q && wi == 0) {
                float amax = 0.f;
                if (grp == 0) {
#pragma unroll
                    for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
                        for (int e = 0; e < CPQ; ++e) amax = fmaxf(amax, fmaxf(fabsf(acc[ps][e].x), fabsf(acc[ps][e].y)));
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
                const float norm = amax == 0.f ? 0.f : __fdiv_rn(amax, 32767.0f);
                if (lane == 0) p.hout_norms[s] = norm;
                if (grp == 0) {
                    short2* hq = p.hout_q;
#pragma unroll
                    for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
                        for (int e = 0; e < CPQ; ++e) hq[(int64_t)s * NC + (ps * QP + qi) * CPQ + e] = half_out_q(acc[ps][e], amax, norm);
                }
            }
        }
    }
}

}  // namespace coarse
