// hat_kernel.cuh — set-up kernel of the even/odd ("Schur-preconditioned", Table 1)
// operators: the block-preconditioned links of PAPER.md:L87,
//
//     Yhat_m(x) = X(x)^-1 . Y_m(x),  m = 1..8,       slot 0 = identity or X(x)^-1,
//
// for every site, from the handle's links (complex64, or int16 + scale dequantised exactly), written as
// complex64 in the canonical layout links[s][m][i][j] (quantise with coarse_op_quantize_i16 afterwards
// for 16-bit storage).  DESIGN.md reading R21.
//
// One CTA per site (persistent loop).  All arithmetic is fp64 - the result is rounded to complex64 once,
// so it agrees with an fp64 LAPACK solve to the last fp32 bit or two whatever the conditioning of X:
//   1. X -> double2 workspace (global memory, Nc x Nc x 16 B per CTA: 262 KB at Nc = 128 does not fit
//      shared memory; the workspace of all CTAs together stays L2-resident);
//   2. in-place Gauss-Jordan inversion with partial (row) pivoting: per step a CTA-wide argmax over the
//      pivot column, a row swap, a scaled pivot row and a rank-1 update of the whole matrix; the row
//      swaps are undone as column swaps at the end;
//   3. eight Nc x Nc x Nc complex products X^-1 . Y_m with 64 x 64 output tiles, K tiles of 16 staged in
//      shared memory, 4 x 4 complex128 accumulators per thread.
// This is a set-up step (once per operator, like the link quantiser): it is bound by fp64 FMA throughput
// (72 Nc^3 flops per site: 67 of them in step 3), not by HBM; bench.py --workload hat reports it so.
// A singular X (zero pivot) leaves non-finite entries at that site and is counted in *info.
#pragma once
#include "common.cuh"

namespace coarse {

struct HatParams {
    Lat lat;
    int Nc;
    int i16;                    // links are int16 + scale
    const void* links;
    const float* scales;
    float2* out;                // [V][9][Nc][Nc] complex64
    double2* work;              // [gridDim.x][Nc][Nc]
    int slot0_inverse;          // 0: out[s][0] = identity, 1: out[s][0] = X^-1
    int* info;                  // may be NULL: += number of sites with a zero pivot
};

__device__ __forceinline__ double2 cmul(const double2 a, const double2 b) {
    return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ void cfma(double2& acc, const double2 a, const double2 b) {
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(a.y, b.x, acc.y);
}

__device__ __forceinline__ double2 hat_link_entry(const HatParams& p, long long s, int m, int i, int j) {
    const long long e = (((s * 9 + m) * p.Nc + i) * p.Nc + j);
    if (p.i16) {
        const short2 q = reinterpret_cast<const short2*>(p.links)[e];
        const double sc = (double)p.scales[s * 9 + m];
        return make_double2((double)q.x * sc, (double)q.y * sc);
    }
    const float2 v = reinterpret_cast<const float2*>(p.links)[e];
    return make_double2((double)v.x, (double)v.y);
}

constexpr int HAT_THREADS = 256;
constexpr int HAT_TILE = 64;       // output tile edge of the products
constexpr int HAT_KT = 16;         // K tile

__global__ void __launch_bounds__(HAT_THREADS) hat_links_kernel(HatParams p) {
    extern __shared__ __align__(16) unsigned char hat_smem[];
    const int Nc = p.Nc;
    double2* rowk = reinterpret_cast<double2*>(hat_smem);                 // [Nc] pivot row
    double2* colk = rowk + Nc;                                            // [Nc] pivot column
    int* piv = reinterpret_cast<int*>(colk + Nc);                         // [Nc] row exchanged with k at step k
    double* red_v = reinterpret_cast<double*>(piv + ((Nc + 1) & ~1));     // [HAT_THREADS / 32]
    int* red_i = reinterpret_cast<int*>(red_v + HAT_THREADS / 32);        // [HAT_THREADS / 32]
    int* flags = red_i + HAT_THREADS / 32;                                // [2]: pivot row, singular
    double2* tA = reinterpret_cast<double2*>((reinterpret_cast<uintptr_t>(flags + 2) + 15) & ~(uintptr_t)15);   // [HAT_TILE][HAT_KT + 1]
    double2* tB = tA + HAT_TILE * (HAT_KT + 1);                           // [HAT_KT][HAT_TILE]
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    double2* A = p.work + (size_t)blockIdx.x * Nc * Nc;

    for (long long s = blockIdx.x; s < p.lat.V; s += gridDim.x) {
        // ---- 1. X -> workspace
        for (int e = tid; e < Nc * Nc; e += HAT_THREADS) A[e] = hat_link_entry(p, s, 0, e / Nc, e % Nc);
        if (tid == 0) flags[1] = 0;
        __syncthreads();
        // ---- 2. in-place Gauss-Jordan with partial pivoting
        for (int k = 0; k < Nc; ++k) {
            double best = -1.0;
            int bi = k;
            for (int i = k + tid; i < Nc; i += HAT_THREADS) {
                const double2 a = A[(size_t)i * Nc + k];
                const double v = a.x * a.x + a.y * a.y;
                if (v > best) { best = v; bi = i; }
            }
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                const double ov = __shfl_xor_sync(0xffffffffu, best, o);
                const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                if (ov > best || (ov == best && oi < bi)) { best = ov; bi = oi; }
            }
            if (lane == 0) { red_v[wid] = best; red_i[wid] = bi; }
            __syncthreads();
            if (tid == 0) {
                double b = red_v[0];
                int r = red_i[0];
                for (int w = 1; w < HAT_THREADS / 32; ++w)
                    if (red_v[w] > b || (red_v[w] == b && red_i[w] < r)) { b = red_v[w]; r = red_i[w]; }
                flags[0] = r;
                piv[k] = r;
                if (!(b > 0.0)) flags[1] = 1;
            }
            __syncthreads();
            const int pr = flags[0];
            // swap rows k and pr, then cache the (new) pivot row and pivot column
            for (int j = tid; j < Nc; j += HAT_THREADS) {
                const double2 a = A[(size_t)pr * Nc + j];
                if (pr != k) {
                    A[(size_t)pr * Nc + j] = A[(size_t)k * Nc + j];
                    A[(size_t)k * Nc + j] = a;
                }
                rowk[j] = a;
            }
            __syncthreads();
            for (int i = tid; i < Nc; i += HAT_THREADS) colk[i] = A[(size_t)i * Nc + k];
            __syncthreads();
            const double2 pv = rowk[k];
            const double d = pv.x * pv.x + pv.y * pv.y;
            const double2 pinv = make_double2(pv.x / d, -pv.y / d);
            // pivot row: a_kj <- a_kj / pivot, with a_kk <- 1 / pivot; other rows: a_ij <- a_ij - a_ik a_kj, a_ik <- -a_ik / pivot
            for (int e = tid; e < Nc * Nc; e += HAT_THREADS) {
                const int i = e / Nc, j = e - i * Nc;
                const double2 rk = (j == k) ? make_double2(1.0, 0.0) : rowk[j];
                const double2 nk = cmul(rk, pinv);                        // the new pivot-row entry of column j
                if (i == k) {
                    A[e] = nk;
                } else {
                    const double2 f = colk[i];
                    double2 a = (j == k) ? make_double2(0.0, 0.0) : A[e];
                    a.x = fma(-f.x, nk.x, a.x);
                    a.x = fma(f.y, nk.y, a.x);
                    a.y = fma(-f.x, nk.y, a.y);
                    a.y = fma(-f.y, nk.x, a.y);
                    A[e] = a;
                }
            }
            __syncthreads();
        }
        // undo the row exchanges as column exchanges, last first
        for (int k = Nc - 1; k >= 0; --k) {
            const int pr = piv[k];
            if (pr != k) {
                for (int i = tid; i < Nc; i += HAT_THREADS) {
                    const double2 a = A[(size_t)i * Nc + k];
                    A[(size_t)i * Nc + k] = A[(size_t)i * Nc + pr];
                    A[(size_t)i * Nc + pr] = a;
                }
                __syncthreads();
            }
        }
        if (tid == 0 && flags[1] && p.info) atomicAdd(p.info, 1);
        // ---- slot 0
        float2* out_s = p.out + (size_t)s * 9 * Nc * Nc;
        for (int e = tid; e < Nc * Nc; e += HAT_THREADS) {
            if (p.slot0_inverse) out_s[e] = make_float2((float)A[e].x, (float)A[e].y);
            else out_s[e] = make_float2((e / Nc == e % Nc) ? 1.f : 0.f, 0.f);
        }
        // ---- 3. Yhat_m = X^-1 . Y_m
        const int ty = tid / 16, tx = tid % 16;                            // 16 x 16 threads, 4 x 4 outputs each
        for (int m = 1; m < 9; ++m) {
            float2* out_m = out_s + (size_t)m * Nc * Nc;
            for (int i0 = 0; i0 < Nc; i0 += HAT_TILE) {
                for (int j0 = 0; j0 < Nc; j0 += HAT_TILE) {
                    double2 acc[4][4];
#pragma unroll
                    for (int a = 0; a < 4; ++a)
#pragma unroll
                        for (int b = 0; b < 4; ++b) acc[a][b] = make_double2(0.0, 0.0);
                    for (int k0 = 0; k0 < Nc; k0 += HAT_KT) {
                        __syncthreads();
                        for (int e = tid; e < HAT_TILE * HAT_KT; e += HAT_THREADS) {
                            const int r = e / HAT_KT, c = e % HAT_KT;       // A tile: rows i0 + r, columns k0 + c
                            tA[r * (HAT_KT + 1) + c] = (i0 + r < Nc && k0 + c < Nc) ? A[(size_t)(i0 + r) * Nc + k0 + c]
                                                                                     : make_double2(0.0, 0.0);
                        }
                        for (int e = tid; e < HAT_KT * HAT_TILE; e += HAT_THREADS) {
                            const int r = e / HAT_TILE, c = e % HAT_TILE;   // B tile: rows k0 + r, columns j0 + c
                            tB[r * HAT_TILE + c] = (k0 + r < Nc && j0 + c < Nc) ? hat_link_entry(p, s, m, k0 + r, j0 + c)
                                                                                 : make_double2(0.0, 0.0);
                        }
                        __syncthreads();
#pragma unroll 4
                        for (int kk = 0; kk < HAT_KT; ++kk) {
                            double2 av[4], bv[4];
#pragma unroll
                            for (int a = 0; a < 4; ++a) av[a] = tA[(ty + 16 * a) * (HAT_KT + 1) + kk];
#pragma unroll
                            for (int b = 0; b < 4; ++b) bv[b] = tB[kk * HAT_TILE + tx + 16 * b];
#pragma unroll
                            for (int a = 0; a < 4; ++a)
#pragma unroll
                                for (int b = 0; b < 4; ++b) cfma(acc[a][b], av[a], bv[b]);
                        }
                    }
#pragma unroll
                    for (int a = 0; a < 4; ++a)
#pragma unroll
                        for (int b = 0; b < 4; ++b) {
                            const int i = i0 + ty + 16 * a, j = j0 + tx + 16 * b;
                            if (i < Nc && j < Nc) out_m[(size_t)i * Nc + j] = make_float2((float)acc[a][b].x, (float)acc[a][b].y);
                        }
                }
            }
        }
        __syncthreads();          // the workspace is rewritten by the next site
    }
}

inline size_t hat_smem_bytes(int Nc) {
    return (size_t)2 * Nc * 16 + (size_t)((Nc + 1) & ~1) * 4 + (HAT_THREADS / 32) * (8 + 4) + 8 +
           (size_t)(HAT_TILE * (HAT_KT + 1) + HAT_KT * HAT_TILE) * 16 + 32;
}

}  // namespace coarse
