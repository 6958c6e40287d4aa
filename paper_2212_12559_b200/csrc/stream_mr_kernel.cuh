// stream_mr_kernel.cuh — the STREAM kernel for a FEW right-hand sides (R = 2, 3, 4): the paper's
// propagator workload is 3 RHS at a time on 16-bit links (L99), and multi-RHS is its
// stated future work (L200).  With R this small the apply is still bound by the link stream, so the
// kernel keeps stream_kernel.cuh's pipeline and thread mapping (lane <-> 16-byte column quad of a link
// row, warp <-> rows, one elected producer lane feeding a TMA ring) and only widens the register tile:
// every link entry is decoded ONCE and used for R complex MACs, so 3 right-hand sides cost the bytes
// of one.  (The BLOCK kernel's lane <-> RHS mapping repeats the int16 decode in every lane of a
// subset and leaves 5 of 8 lanes idle at R = 3: measured 5.7 ms / 12.7 ms on the C2 / C4 shapes
// where this kernel is HBM-bound.)
//
// Vectors are RHS-innermost (v[s][a][r]): the lane's CPQ columns x R right-hand sides are one
// contiguous run of CPQ*R complex numbers in the staged vector block.
// dagger = 0: acc[WL rows][R], one shuffle reduction per (row, r) per item.
// dagger = 1: acc[PASSES][CPQ][R] per lane (output columns), partial sums over the row slices combined
//             through shared memory once per item.
#pragma once
#include "stream_kernel.cuh"

// Words (of the 4) of every int16 link quad decoded through the conversion unit (see stream2_kernel.cuh)
#ifndef COARSE_MR_XU_N
#define COARSE_MR_XU_N 2
#endif
#ifndef COARSE_MR_XU_D
#define COARSE_MR_XU_D 1
#endif

namespace coarse {

template <int NC, bool I16, int R>
struct StreamMrGeom {
    using G1 = StreamGeom<NC, I16, false, false, true>;
    static constexpr int VEC_STAGE_N = NC * R * 8;
    static constexpr int VEC_STAGE_D = G1::RS * R * 8;
    static constexpr int RED_BYTES = G1::W * G1::RPL * NC * R * 8;   // dagger = 1, single buffer (two barriers per item)
    // dagger = 0: a lane's vector operand is a block of N16 = CPQ*R/2 16-byte chunks.  When N16 = 8
    // (int16 links, R = 4) the lane stride is 128 bytes and every block load is 8-way bank conflicted
    // (measured: C4 shape 7.7 ms).  Each warp then re-stages the stage's vector block into a private
    // copy with one chunk of padding per lane block (pitch 9 chunks): a few conflict-free LDS/STS.128
    // per stage, after which the block loads are conflict-free (4.5 ms).  At N16 = 4 (4-way) the
    // re-stage costs as much as it saves (measured), so it is not used there: with every warp reading
    // the whole vector block, R = 4 is bound by shared-memory bandwidth rather than HBM in dagger = 0.
    static constexpr int N16 = G1::CPQ * R / 2;
    static constexpr bool PAD = (N16 % 8 == 0);
    static constexpr int PRIV_WARP = PAD ? G1::Q * (N16 + 1) * 16 : 0;
    static constexpr int PRIV_BYTES = G1::W * PRIV_WARP;
    static constexpr bool OK = G1::OK && R >= 2 && R <= 4;
    static constexpr int stage_bytes(bool dag) { return G1::LINK_STAGE + (dag ? VEC_STAGE_D : VEC_STAGE_N); }
    static constexpr int CL_BYTES = 2 * (STREAM_MAX_CLUSTER - 1) * NC * R * 8;   // dagger = 1 in clusters: rank 0's inbox (stream_kernel.cuh)
    static constexpr int fixed_bytes(bool dag) { return (dag ? RED_BYTES + CL_BYTES : PRIV_BYTES) + 128; }
    static int smem_bytes(bool dag, int stages) { return stages * (stage_bytes(dag) + 16) + fixed_bytes(dag); }
};

// CL: launched as thread-block clusters on lattices with fewer sites than SMs (dagger = 1: one site per cluster, the CTA of rank r
// contracts the row chunks r, r + cluster, .., the partial vectors meet in rank 0's shared memory) - its own instantiation, see
// stream_kernel.cuh.
template <int NC, bool I16, bool DAG, int R, bool CL = false>
__global__ void __launch_bounds__(StreamGeom<NC, I16, false, false, true>::THREADS, 1) coarse_apply_stream_mr(StreamParams p) {
    static_assert(!CL || DAG, "cluster launches: dagger = 1");
    using Gm = StreamGeom<NC, I16, false, false, true>;
    using Gr = StreamMrGeom<NC, I16, R>;
    static_assert(Gr::OK, "unsupported STREAM-MR geometry");
    constexpr int W = Gm::W, RS = Gm::RS, NB = Gm::NB, WL = Gm::WL, QP = Gm::QP, G = Gm::G, RPL = Gm::RPL;
    constexpr int PASSES = Gm::PASSES, CPQ = Gm::CPQ, ROWBYTES = Gm::ROWBYTES, LINK_STAGE = Gm::LINK_STAGE;
    constexpr int VEC_STAGE = DAG ? Gr::VEC_STAGE_D : Gr::VEC_STAGE_N;

    extern __shared__ __align__(128) unsigned char smem[];
    const int S = p.stages;
    unsigned char* link_smem = smem;
    unsigned char* vec_smem = link_smem + (size_t)S * LINK_STAGE;
    unsigned char* red_smem = vec_smem + (size_t)S * VEC_STAGE;
    uint64_t* bars = reinterpret_cast<uint64_t*>(red_smem + (DAG ? Gr::RED_BYTES : Gr::PRIV_BYTES));
    const uint32_t full0 = ptx::smem_u32(bars);
    const uint32_t empty0 = full0 + 8u * S;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int CR = CL ? p.cluster : 0;                                  // CTAs per cluster (0: plain launch)
    const int crank = CR ? (int)blockIdx.x % CR : 0;
    const int item0 = p.item_begin + (CR ? (int)blockIdx.x / CR : (int)blockIdx.x);
    const int item_stride = CR ? (int)gridDim.x / CR : (int)gridDim.x;
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
        bool cl_pending = false;
        for (int item = item0; item < p.n_items; item += item_stride) {
            const int sidx = DAG ? item : item / NB;
            const int s = p.parity != 2 ? parity_site(p.lat, sidx, p.parity) : sidx;      // parts apply: one parity
            const int rb = DAG ? 0 : item % NB;
            const SiteX cx = site_coords(p.lat, s);
#pragma unroll
            for (int m = 0; m < 9; ++m) {
                if (m < p.m_begin) continue;                                              // parts apply: no X stage
                const int sv = stencil_site_x(p.lat, s, cx, m, DAG ? 1 : 0);
                const int sm = DAG ? sv : s;
                const unsigned char* mat = p.links + ((int64_t)sm * 9 + m) * ((int64_t)NC * ROWBYTES);
                const float2* vec = (m == 0 ? p.in_local : p.in) + (int64_t)sv * NC * R;
#pragma unroll 1
                for (int c = crank; c < (DAG ? NB : 1); c += (CR ? CR : 1)) {
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
            if (CR) {                             // the site's cluster barrier counts every thread of the cluster: arrive now,
                if (cl_pending) ptx::cluster_wait();  // complete it before the next arrival (no drain at site boundaries)
                ptx::cluster_arrive();
                cl_pending = true;
            }
        }
        if (cl_pending) ptx::cluster_wait();
        return;
    }

    // ---------------------------------------------------------------------- consumers
    const int grp = lane / G;
    const int qi = lane % G;
    const bool active = qi < QP;
    const uint32_t link_u32 = ptx::smem_u32(link_smem), vec_u32 = ptx::smem_u32(vec_smem);
    int slot = 0;
    uint32_t phase = 0;

    float cur_scale = 1.f, next_scale = 1.f, next2_scale = 1.f;
    auto site_of = [&](int item) -> int {
        const int sidx = DAG ? item : item / NB;
        return p.parity != 2 ? parity_site(p.lat, sidx, p.parity) : sidx;
    };
    auto fetch_scale = [&](int item) -> float {
        if (!I16 || lane >= 9 || item >= p.n_items) return 1.f;
        const int s = site_of(item);
        const int sm = DAG ? stencil_site(p.lat, s, lane, 1) : s;
        return __ldg(p.scales + (int64_t)sm * 9 + lane);
    };
    const bool scale_v = I16 || p.gen != 0;        // the vector operand carries the link scale and / or alpha, beta
    next_scale = fetch_scale(item0);
    next2_scale = fetch_scale(item0 + item_stride);

    // cluster mode: rank 0's inbox [2 site parities][STREAM_MAX_CLUSTER - 1][NC R] behind the barriers
    float2* cl_buf = reinterpret_cast<float2*>(reinterpret_cast<unsigned char*>(bars + 2 * S) + 128);
    const uint32_t cl_inbox = CR ? ptx::mapa_shared(ptx::smem_u32(cl_buf), 0u) : 0u;
    constexpr int UL = (NC * R + W * 32 - 1) / (W * 32);
    int it = 0;
    for (int item = item0; item < p.n_items; item += item_stride, ++it) {
        const int s = site_of(item);
        const int rb = DAG ? 0 : item % NB;
        cur_scale = next_scale;
        next_scale = next2_scale;
        next2_scale = fetch_scale(item + 2 * item_stride);

        if (!DAG) {
            CAcc pacc[WL][R];
#pragma unroll
            for (int k = 0; k < WL; ++k)
#pragma unroll
                for (int r = 0; r < R; ++r) pacc[k][r].a = pacc[k][r].b = make_float2(0.f, 0.f);
#pragma unroll 1
            for (int m = p.m_begin; m < 9; ++m) {
                float sc = I16 ? __shfl_sync(0xffffffffu, cur_scale, m) : 1.f;
                if (p.gen) sc *= (m == 0) ? p.alpha : p.beta;
                ptx::mbar_wait(full0 + 8u * slot, phase);
                const uint32_t lbase = link_u32 + slot * LINK_STAGE + qi * 16;
                uint32_t vbase = vec_u32 + slot * VEC_STAGE;
                constexpr int N16 = Gr::N16;
                constexpr int PITCH = Gr::PAD ? (N16 + 1) * 16 : N16 * 16;     // bytes between lane blocks
                if constexpr (Gr::PAD) {
                    const uint32_t priv = ptx::smem_u32(red_smem) + warp * Gr::PRIV_WARP;
                    for (int c = lane; c < Gm::Q * N16; c += 32) {
                        const float4 t = ptx::lds128(vbase + c * 16);
                        const uint32_t d = priv + ((c / N16) * (N16 + 1) + (c % N16)) * 16;
                        asm volatile("st.shared.v4.f32 [%0], {%1,%2,%3,%4};" ::"r"(d), "f"(t.x), "f"(t.y), "f"(t.z), "f"(t.w) : "memory");
                    }
                    __syncwarp();
                    vbase = priv;
                }
                if (active) {
#pragma unroll
                    for (int ps = 0; ps < PASSES; ++ps) {
                        // the lane's CPQ columns x R right-hand sides: CPQ*R contiguous complex numbers
                        VDup v[CPQ * R];
                        const uint32_t va = vbase + (ps * QP + qi) * PITCH;
#pragma unroll
                        for (int h = 0; h < CPQ * R / 2; ++h) {
                            float4 t = ptx::lds128(va + h * 16);
                            if (scale_v) { t.x *= sc; t.y *= sc; t.z *= sc; t.w *= sc; }
                            v[2 * h] = vdup(make_float2(t.x, t.y));
                            v[2 * h + 1] = vdup(make_float2(t.z, t.w));
                        }
#pragma unroll
                        for (int k = 0; k < WL; ++k) {
                            const int rl = (k * W + warp) * RPL + grp;
                            const uint32_t a = lbase + rl * ROWBYTES + ps * QP * 16;
                            float2 mm[CPQ];
                            if constexpr (I16) {
                                const uint4 t = ptx::lds128u(a);
                                unpack_i16_quad<COARSE_MR_XU_N>(t, mm[0], mm[1], mm[CPQ - 2], mm[CPQ - 1]);
                            } else {
                                const float4 t = ptx::lds128(a);
                                mm[0] = make_float2(t.x, t.y);
                                mm[1] = make_float2(t.z, t.w);
                            }
#pragma unroll
                            for (int e = 0; e < CPQ; ++e)
#pragma unroll
                                for (int r = 0; r < R; ++r) cmacp(pacc[k][r], mm[e], v[e * R + r]);
                        }
                    }
                }
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
                if (++slot == S) { slot = 0; phase ^= 1u; }
            }
            // a6: combine the column-slice partial sums, once per item
            float2 acc[WL][R];
#pragma unroll
            for (int k = 0; k < WL; ++k)
#pragma unroll
                for (int r = 0; r < R; ++r) acc[k][r] = cfinal<false>(pacc[k][r]);
#pragma unroll
            for (int k = 0; k < WL; ++k) {
#pragma unroll
                for (int r = 0; r < R; ++r) {
#pragma unroll
                    for (int o = G / 2; o > 0; o >>= 1) {
                        acc[k][r].x += __shfl_xor_sync(0xffffffffu, acc[k][r].x, o);
                        acc[k][r].y += __shfl_xor_sync(0xffffffffu, acc[k][r].y, o);
                    }
                }
                if (qi == 0) {
                    const int row = rb * RS + (k * W + warp) * RPL + grp;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        float2 o = acc[k][r];
                        if (p.identity) {           // parts apply: + alpha u(x); each element reads only its own u element
                            const float2 u = __ldg(p.in_local + ((int64_t)s * NC + row) * R + r);
                            o.x = fmaf(p.alpha, u.x, o.x);
                            o.y = fmaf(p.alpha, u.y, o.y);
                        }
                        p.out[((int64_t)s * NC + row) * R + r] = o;
                    }
                }
            }
        } else {
            CAcc pacc[PASSES][CPQ][R];
#pragma unroll
            for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
                for (int e = 0; e < CPQ; ++e)
#pragma unroll
                    for (int r = 0; r < R; ++r) pacc[ps][e][r].a = pacc[ps][e][r].b = make_float2(0.f, 0.f);
#pragma unroll 1
            for (int m = p.m_begin; m < 9; ++m) {
                float sc = I16 ? __shfl_sync(0xffffffffu, cur_scale, m) : 1.f;
                if (p.gen) sc *= (m == 0) ? p.alpha : p.beta;
#pragma unroll 1
                for (int c = crank; c < NB; c += (CR ? CR : 1)) {
                    ptx::mbar_wait(full0 + 8u * slot, phase);
                    const uint32_t lbase = link_u32 + slot * LINK_STAGE + qi * 16;
                    const uint32_t vbase = vec_u32 + slot * VEC_STAGE;
                    if (active) {
#pragma unroll
                        for (int k = 0; k < WL; ++k) {
                            const int rl = (k * W + warp) * RPL + grp;
                            VDup vj[R];
#pragma unroll
                            for (int r = 0; r < R; ++r) {
                                float2 t = ptx::lds64(vbase + (rl * R + r) * 8);
                                if (scale_v) { t.x *= sc; t.y *= sc; }
                                vj[r] = vdup(t);
                            }
#pragma unroll
                            for (int ps = 0; ps < PASSES; ++ps) {
                                const uint32_t a = lbase + rl * ROWBYTES + ps * QP * 16;
                                float2 mm[CPQ];
                                if constexpr (I16) {
                                    const uint4 t = ptx::lds128u(a);
                                    unpack_i16_quad<COARSE_MR_XU_D>(t, mm[0], mm[1], mm[CPQ - 2], mm[CPQ - 1]);
                                } else {
                                    const float4 t = ptx::lds128(a);
                                    mm[0] = make_float2(t.x, t.y);
                                    mm[1] = make_float2(t.z, t.w);
                                }
#pragma unroll
                                for (int e = 0; e < CPQ; ++e)
#pragma unroll
                                    for (int r = 0; r < R; ++r) cmacp(pacc[ps][e][r], mm[e], vj[r]);
                            }
                        }
                    }
                    __syncwarp();
                    if (lane == 0) ptx::mbar_arrive(empty0 + 8u * slot);
                    if (++slot == S) { slot = 0; phase ^= 1u; }
                }
            }
            // a6: combine the row-slice partial sums (W warps x RPL row groups), once per item
            float2* red = reinterpret_cast<float2*>(red_smem);
            if (active) {
#pragma unroll
                for (int ps = 0; ps < PASSES; ++ps)
#pragma unroll
                    for (int e = 0; e < CPQ; ++e)
#pragma unroll
                        for (int r = 0; r < R; ++r)
                            red[((warp * RPL + grp) * NC + (ps * QP + qi) * CPQ + e) * R + r] = cfinal<true>(pacc[ps][e][r]);
            }
            ptx::named_bar_sync(1, W * 32);
            float2 cl_keep[UL];
#pragma unroll
            for (int ku = 0; ku < UL; ++ku) {
                const int t = (int)threadIdx.x + ku * W * 32;
                cl_keep[ku] = make_float2(0.f, 0.f);
                if (t < NC * R) {
                    float2 sum = make_float2(0.f, 0.f);
#pragma unroll
                    for (int g = 0; g < W * RPL; ++g) {
                        const float2 x = red[g * NC * R + t];
                        sum.x += x.x;
                        sum.y += x.y;
                    }
                    if (p.identity && crank == 0) {
                        const float2 u = __ldg(p.in_local + (int64_t)s * NC * R + t);
                        sum.x = fmaf(p.alpha, u.x, sum.x);
                        sum.y = fmaf(p.alpha, u.y, sum.y);
                    }
                    if (!CR) p.out[(int64_t)s * NC * R + t] = sum;
                    else if (crank) ptx::st_cluster_f2(cl_inbox + (uint32_t)(((it & 1) * (STREAM_MAX_CLUSTER - 1) + crank - 1) * (NC * R) + t) * 8u, sum);
                    else cl_keep[ku] = sum;
                }
            }
            ptx::named_bar_sync(1, W * 32);      // red is reused by the next item
            if (CR) {
                // the ranks' partial vectors are in rank 0's inbox behind the site's cluster barrier; rank 0 adds them in rank order
                ptx::cluster_sync_all();
                if (crank == 0) {
#pragma unroll
                    for (int ku = 0; ku < UL; ++ku) {
                        const int t = (int)threadIdx.x + ku * W * 32;
                        if (t < NC * R) {
                            float2 sum = cl_keep[ku];
                            for (int r = 1; r < CR; ++r) {
                                const float2 x = cl_buf[((it & 1) * (STREAM_MAX_CLUSTER - 1) + r - 1) * (NC * R) + t];
                                sum.x += x.x;
                                sum.y += x.y;
                            }
                            p.out[(int64_t)s * NC * R + t] = sum;
                        }
                    }
                }
            }
        }
    }
}

}  // namespace coarse
