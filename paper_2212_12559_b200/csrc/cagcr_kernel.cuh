// cagcr_kernel.cuh — the vector side of CA-GCR(s), the paper's smoother ("CA-GCR(8)",
// Table 1 L116/L122/L130), around s chained coarse-op applies:
//
//   p_k = T_k((A - c)/d) r0, t_k = A p_k (k < s)   s applies (stream_kernel.cuh, 95 % of the time) and s - 1
//                                                 fused three-term recurrence steps: the Chebyshev basis of
//                                                 the Krylov space K_s(A, r0) on [c - d, c + d]
//   G = Gram matrix of (r0, t_0 .. t_{s-1})       ONE fused pass of block inner products (this file);
//                                                 on a partitioned lattice this is the single
//                                                 all-reduce per cycle that makes the method
//                                                 "communication avoiding"
//   (T^H T) alpha = T^H r0                        s x s Hermitian solve, fp64 Cholesky, one thread
//   x += sum_k alpha_k p_k,  r = r0 - sum_k alpha_k t_k      one fused update pass
//
// The interval is either the caller's or estimated on the device, without a host round trip, from the
// moments of the first residual: m1 = <r0, A r0>/<r0, r0>, m2 = <A r0, A r0>/<r0, r0>,
// c = Re m1, d = 2 sqrt(m2 - (Re m1)^2) (twice the spread of the spectrum as r0 sees it).
// The Gram matrix is accumulated in fp64 with a fixed two-level summation order: bit-identical run to run.
#pragma once
#include "common.cuh"

namespace coarse {

constexpr int CAGCR_MAX_S = 16;
constexpr int CAGCR_GRAM_BLOCKS = 296;

struct CagcrVecs {
    const float2* p[CAGCR_MAX_S + 1];   // p_0 .. p_s
};

// Fused block inner products: every CTA walks tiles of CAGCR_TILE lattice elements, stages the s+1
// basis vectors of the tile in shared memory ONCE (each vector is read from global memory exactly once
// per cycle) and its 8 warps share out the (s+1)(s+2)/2 pairs (j <= k), pair index cyclic over warps;
// a lane accumulates conj(p_j[e]) p_k[e] in fp64 over the elements e = lane, lane + 32, ... of the tile.
// partial[block][pair] is written once per CTA; the solve kernel adds the blocks in order.
constexpr int CAGCR_TILE = 256;
constexpr int CAGCR_MAX_PAIRS = (CAGCR_MAX_S + 1) * (CAGCR_MAX_S + 2) / 2;     // 153
constexpr int CAGCR_PAIRS_PER_WARP = (CAGCR_MAX_PAIRS + 7) / 8;                // 20

__host__ __device__ inline int cagcr_pair_index(int j, int k, int S1) { return j * S1 - j * (j - 1) / 2 + (k - j); }

__global__ void __launch_bounds__(256) cagcr_gram_kernel(CagcrVecs v, long long n, int s, double2* partial) {
    __shared__ float2 tile[CAGCR_MAX_S + 1][CAGCR_TILE];
    __shared__ unsigned char pj[CAGCR_MAX_PAIRS], pk[CAGCR_MAX_PAIRS];
    const int S1 = s + 1;
    const int npairs = S1 * (S1 + 1) / 2;
    for (int t = threadIdx.x; t < S1 * S1; t += blockDim.x) {
        const int a = t / S1, b = t % S1;
        if (b >= a) {
            pj[cagcr_pair_index(a, b, S1)] = (unsigned char)a;
            pk[cagcr_pair_index(a, b, S1)] = (unsigned char)b;
        }
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double2 acc[CAGCR_PAIRS_PER_WARP];
#pragma unroll
    for (int q = 0; q < CAGCR_PAIRS_PER_WARP; ++q) acc[q] = make_double2(0.0, 0.0);
    const long long ntiles = (n + CAGCR_TILE - 1) / CAGCR_TILE;
    for (long long t = blockIdx.x; t < ntiles; t += gridDim.x) {
        const long long i = t * CAGCR_TILE + threadIdx.x;
        __syncthreads();                       // previous tile fully consumed (and pj/pk written)
        for (int k = 0; k < S1; ++k) tile[k][threadIdx.x] = i < n ? v.p[k][i] : make_float2(0.f, 0.f);
        __syncthreads();
#pragma unroll
        for (int q = 0; q < CAGCR_PAIRS_PER_WARP; ++q) {
            const int pidx = warp + 8 * q;
            if (pidx < npairs) {
                const float2* a = tile[pj[pidx]];
                const float2* b = tile[pk[pidx]];
                double2 t2 = acc[q];
#pragma unroll
                for (int e = 0; e < CAGCR_TILE / 32; ++e) {
                    const float2 x = a[lane + 32 * e], y = b[lane + 32 * e];
                    t2.x += (double)x.x * (double)y.x + (double)x.y * (double)y.y;
                    t2.y += (double)x.x * (double)y.y - (double)x.y * (double)y.x;
                }
                acc[q] = t2;
            }
        }
    }
#pragma unroll
    for (int q = 0; q < CAGCR_PAIRS_PER_WARP; ++q) {
        const int pidx = warp + 8 * q;
        if (pidx < npairs) {
            double2 t2 = acc[q];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                t2.x += __shfl_xor_sync(0xffffffffu, t2.x, o);
                t2.y += __shfl_xor_sync(0xffffffffu, t2.y, o);
            }
            if (lane == 0) partial[(long long)blockIdx.x * npairs + pidx] = t2;
        }
    }
}

// One CTA: sums the per-block partials in block order, then thread 0 solves the s x s normal equations
// M alpha = c (M_ab = G[a+1][b+1], c_a = G[a+1][0] = <q_a, r0>) by a complex Cholesky factorisation in
// fp64.  A pivot that has lost all its digits truncates the basis there (alpha_k = 0 beyond it).
// info[0] = ||r0||^2, info[1] = predicted ||r||^2 = ||r0||^2 - Re(c^H alpha), info[2] = columns used.
__global__ void __launch_bounds__(320) cagcr_solve_kernel(const double2* partial, int nblocks, int s, double2* alpha,
                                                          double* info) {
    __shared__ double2 G[CAGCR_MAX_S + 1][CAGCR_MAX_S + 1];
    const int S1 = s + 1;
    for (int e = threadIdx.x; e < S1 * S1; e += blockDim.x) {
        const int j = e / S1, k = e % S1;
        if (k >= j) {
            double2 t = make_double2(0.0, 0.0);
            for (int b = 0; b < nblocks; ++b) {
                const double2 x = partial[(long long)b * (S1 * (S1 + 1) / 2) + cagcr_pair_index(j, k, S1)];
                t.x += x.x;
                t.y += x.y;
            }
            G[j][k] = t;
        }
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    double2 L[CAGCR_MAX_S][CAGCR_MAX_S];
    double2 y[CAGCR_MAX_S];
    int used = s;
    // M_ab = G[a+1][b+1] for b >= a, Hermitian: M_ba = conj(M_ab); lower Cholesky M = L L^H
    for (int k = 0; k < s; ++k) {
        double d = G[k + 1][k + 1].x;
        for (int i = 0; i < k; ++i) d -= L[k][i].x * L[k][i].x + L[k][i].y * L[k][i].y;
        if (!(d > 1e-13 * G[k + 1][k + 1].x)) { used = k; break; }
        const double lkk = sqrt(d);
        L[k][k] = make_double2(lkk, 0.0);
        for (int a = k + 1; a < s; ++a) {
            // M_ak = conj(G[k+1][a+1])
            double2 t = make_double2(G[k + 1][a + 1].x, -G[k + 1][a + 1].y);
            for (int i = 0; i < k; ++i) {   // t -= L[a][i] * conj(L[k][i])
                t.x -= L[a][i].x * L[k][i].x + L[a][i].y * L[k][i].y;
                t.y -= L[a][i].y * L[k][i].x - L[a][i].x * L[k][i].y;
            }
            L[a][k] = make_double2(t.x / lkk, t.y / lkk);
        }
    }
    // c_a = <q_a, r0> = conj(G[0][a+1]);  forward solve L y = c
    for (int a = 0; a < used; ++a) {
        double2 t = make_double2(G[0][a + 1].x, -G[0][a + 1].y);
        for (int i = 0; i < a; ++i) {       // t -= L[a][i] * y[i]
            t.x -= L[a][i].x * y[i].x - L[a][i].y * y[i].y;
            t.y -= L[a][i].x * y[i].y + L[a][i].y * y[i].x;
        }
        y[a] = make_double2(t.x / L[a][a].x, t.y / L[a][a].x);
    }
    // backward solve L^H alpha = y
    double gain = 0.0;
    for (int a = used - 1; a >= 0; --a) {
        double2 t = y[a];
        for (int i = a + 1; i < used; ++i) {   // t -= conj(L[i][a]) * alpha[i]
            const double2 al = alpha[i];
            t.x -= L[i][a].x * al.x + L[i][a].y * al.y;
            t.y -= L[i][a].x * al.y - L[i][a].y * al.x;
        }
        alpha[a] = make_double2(t.x / L[a][a].x, t.y / L[a][a].x);
    }
    for (int a = used; a < s; ++a) alpha[a] = make_double2(0.0, 0.0);
    for (int a = 0; a < used; ++a) gain += y[a].x * y[a].x + y[a].y * y[a].y;   // c^H M^-1 c = |y|^2
    if (info) {
        info[0] = G[0][0].x;
        info[1] = G[0][0].x - gain;
        info[2] = (double)used;
    }
}

// r = b - t
__global__ void __launch_bounds__(256) cagcr_residual_kernel(const float2* b, const float2* t, long long n, float2* r) {
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const float2 x = b[i], y = t[i];
        r[i] = make_float2(x.x - y.x, x.y - y.y);
    }
}

// ---- Chebyshev basis (the paper's coarsest-level solver is a "Chebyshev-basis CA-GCR(16)"):
// p_k = T_k((A - c)/d) r0 on the interval [lambda_min, lambda_max] = [c - d, c + d] spans the same Krylov
// space as the power basis A^k r0 but stays well conditioned (the power basis, stored in complex64 with a Gram
// matrix that squares its conditioning, lost the iterate's 5th digit at s = 8 and truncated itself at s = 16).
// With t_k = A p_k:   p_1 = (t_0 - c p_0)/d,   p_{k+1} = (2/d)(t_k - c p_k) - p_{k-1}.
// cd = {c, d} lives in device memory (written by one of the two kernels below).
__global__ void __launch_bounds__(256) cagcr_cheb_step_kernel(const float2* t, const float2* p, const float2* pm,
                                                              const double* cd, int first, long long n, float2* out) {
    const float a = (float)((first ? 1.0 : 2.0) / cd[1]);
    const float b = (float)(-(first ? 1.0 : 2.0) * cd[0] / cd[1]);
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const float2 x = t[i], y = p[i];
        float2 o = make_float2(fmaf(a, x.x, b * y.x), fmaf(a, x.y, b * y.y));
        if (!first) {
            const float2 z = pm[i];
            o.x -= z.x;
            o.y -= z.y;
        }
        out[i] = o;
    }
}

__global__ void cagcr_set_interval_kernel(double c, double d, double* cd) {
    cd[0] = c;
    cd[1] = d;
}

// Interval from the Gram partials of (r0, A r0) (cagcr_gram_kernel with s = 1: pairs (0,0), (0,1), (1,1)).
__global__ void __launch_bounds__(32) cagcr_interval_kernel(const double2* partial, int nblocks, double* cd) {
    if (threadIdx.x != 0) return;
    double g00 = 0.0, g11 = 0.0;
    double2 g01 = make_double2(0.0, 0.0);
    for (int b = 0; b < nblocks; ++b) {
        g00 += partial[(long long)b * 3 + 0].x;
        g01.x += partial[(long long)b * 3 + 1].x;
        g01.y += partial[(long long)b * 3 + 1].y;
        g11 += partial[(long long)b * 3 + 2].x;
    }
    double c = 0.0, d = 1.0;
    if (g00 > 0.0) {
        c = g01.x / g00;
        const double var = g11 / g00 - c * c;                 // includes the imaginary spread of the spectrum
        d = 2.0 * sqrt(var > 0.0 ? var : 0.0);
        const double floor_d = 1e-3 * fabs(c);
        if (!(d > floor_d)) d = floor_d;
        if (!(d > 0.0)) d = 1.0;
    }
    cd[0] = c;
    cd[1] = d;
}

// x += sum_{k<s} alpha_k P_k ;  r_out = r0 - sum_{k<s} alpha_k T_k      (P, T: separate vector lists)
__global__ void __launch_bounds__(256) cagcr_update2_kernel(CagcrVecs P, CagcrVecs T, const float2* r0, long long n, int s,
                                                            const double2* alpha, float2* x, float2* r_out) {
    __shared__ float2 al[CAGCR_MAX_S];
    if (threadIdx.x < s) al[threadIdx.x] = make_float2((float)alpha[threadIdx.x].x, (float)alpha[threadIdx.x].y);
    __syncthreads();
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        float2 xs = x[i];
        float2 rs = r0[i];
#pragma unroll 4
        for (int k = 0; k < s; ++k) {
            const float2 a = al[k];
            const float2 pk = P.p[k][i], tk = T.p[k][i];
            xs.x = fmaf(a.x, pk.x, fmaf(-a.y, pk.y, xs.x));
            xs.y = fmaf(a.x, pk.y, fmaf(a.y, pk.x, xs.y));
            rs.x = fmaf(-a.x, tk.x, fmaf(a.y, tk.y, rs.x));
            rs.y = fmaf(-a.x, tk.y, fmaf(-a.y, tk.x, rs.y));
        }
        x[i] = xs;
        r_out[i] = rs;
    }
}

}  // namespace coarse
