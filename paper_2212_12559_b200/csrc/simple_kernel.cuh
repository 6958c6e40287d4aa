// simple_kernel.cuh — COARSE_PATH_SIMPLE: one thread per output element (s, i, r).
//
// Covers every argument the ABI accepts (any even Nc, any nrhs, both link formats, dagger) with
// no tiling; it is the fall-back for shapes outside the STREAM path's compiled set, not the fast
// path.  fp32 accumulation, fixed summation order (m, then j): deterministic.
#pragma once
#include "common.cuh"

namespace coarse {

struct SimpleParams {
    Lat lat;
    int Nc;
    int nrhs;
    int dagger;
    const void* links;
    const float* scales;
    const float2* in;        // w: operand of the hopping term (and of X in the plain apply)
    float2* out;
    // parts apply (coarse_op_apply_parts): out = alpha*Loc + beta*Hop on one parity; the plain
    // apply is local = 1, alpha = beta = 1, parity = 2, in_local = in
    const float2* in_local;  // u: operand of the local term
    float alpha, beta;
    int local;               // 0 none, 1 X, 2 identity
    int parity;              // 0 even, 1 odd, 2 all
    // half-precision input vectors (coarse_op_apply_hvec): in = int16 (re,im) [V][Nc][nrhs], vnorms[V][nrhs]
    const float* vnorms;     // NULL: complex64 vectors
};

template <bool I16>
__global__ void __launch_bounds__(256) coarse_apply_simple(SimpleParams p) {
    const int64_t total = (int64_t)p.lat.V * p.Nc * p.nrhs;
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= total) return;
    const int r = (int)(idx % p.nrhs);
    const int i = (int)((idx / p.nrhs) % p.Nc);
    const int s = (int)(idx / ((int64_t)p.nrhs * p.Nc));
    const int Nc = p.Nc;

    if (p.parity != 2) {
        int t = s, par = 0;
        par += t % p.lat.L[0]; t /= p.lat.L[0];
        par += t % p.lat.L[1]; t /= p.lat.L[1];
        par += t % p.lat.L[2]; t /= p.lat.L[2];
        par += t;
        if ((par & 1) != p.parity) return;      // sites of the other parity are left untouched
    }

    float acc_re = 0.f, acc_im = 0.f;
    if (p.local == 2) {
        const float2 u = p.in_local[idx];
        acc_re = p.alpha * u.x;
        acc_im = p.alpha * u.y;
    }
    for (int m = (p.local == 1 ? 0 : 1); m < 9; ++m) {
        const int sv = stencil_site(p.lat, s, m, p.dagger);   // site of the input vector
        const int sm = p.dagger ? sv : s;                     // site of the link matrix
        const int64_t mat = ((int64_t)sm * 9 + m) * Nc * Nc;  // entry offset of M(sm, m)
        const float scale = (I16 ? p.scales[(int64_t)sm * 9 + m] : 1.f) * (m == 0 ? p.alpha : p.beta);
        const float2* vin = (m == 0) ? p.in_local : p.in;
        float part_re = 0.f, part_im = 0.f;
        for (int j = 0; j < Nc; ++j) {
            const int64_t e = p.dagger ? mat + (int64_t)j * Nc + i : mat + (int64_t)i * Nc + j;
            float mre, mim;
            if (I16) {
                const float2 q = unpack_i16x2(reinterpret_cast<const uint32_t*>(p.links)[e]);
                mre = q.x;
                mim = q.y;
            } else {
                const float2 q = reinterpret_cast<const float2*>(p.links)[e];
                mre = q.x;
                mim = q.y;
            }
            if (p.dagger) mim = -mim;
            float2 v;
            if (p.vnorms) {
                v = unpack_i16x2(reinterpret_cast<const uint32_t*>(vin)[((int64_t)sv * Nc + j) * p.nrhs + r]);
                const float n = p.vnorms[(int64_t)sv * p.nrhs + r];
                v.x *= n;
                v.y *= n;
            } else {
                v = vin[((int64_t)sv * Nc + j) * p.nrhs + r];
            }
            part_re = fmaf(mre, v.x, part_re);
            part_re = fmaf(-mim, v.y, part_re);
            part_im = fmaf(mre, v.y, part_im);
            part_im = fmaf(mim, v.x, part_im);
        }
        acc_re = fmaf(scale, part_re, acc_re);
        acc_im = fmaf(scale, part_im, acc_im);
    }
    p.out[idx] = make_float2(acc_re, acc_im);
}

}  // namespace coarse
