// quantize_kernel.cuh — the paper's 16-bit fixed-point link storage (§3.1), produced
// on the device: one CTA per Nc x Nc matrix, scale = max|component|/32767 (BASELINE.json config 4),
// q = clamp(rint(component/scale)).  All decisions in IEEE fp32 (no fast-math), so the integers are
// reproducible bit for bit.
#pragma once
#include "common.cuh"

namespace coarse {

__global__ void __launch_bounds__(256) quantize_i16_kernel(const float* __restrict__ links, int64_t n_matrices,
                                                          int Nc, short* __restrict__ q,
                                                          float* __restrict__ scales) {
    __shared__ float warp_max[8];
    __shared__ float s_scale;
    const int per = 2 * Nc * Nc;
    for (int64_t k = blockIdx.x; k < n_matrices; k += gridDim.x) {
        const float* src = links + k * per;
        short* dst = q + k * per;
        float amax = 0.f;
        for (int e = threadIdx.x; e < per; e += blockDim.x) amax = fmaxf(amax, fabsf(src[e]));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
        if ((threadIdx.x & 31) == 0) warp_max[threadIdx.x >> 5] = amax;
        __syncthreads();
        if (threadIdx.x == 0) {
            float a = warp_max[0];
            for (int w = 1; w < (int)(blockDim.x >> 5); ++w) a = fmaxf(a, warp_max[w]);
            const float sc = (a == 0.f) ? 0.f : __fdiv_rn(a, 32767.0f);
            s_scale = sc;
            scales[k] = sc;
        }
        __syncthreads();
        const float sc = s_scale;
        for (int e = threadIdx.x; e < per; e += blockDim.x) {
            float t = 0.f;
            if (sc != 0.f) {
                t = rintf(__fdiv_rn(src[e], sc));
                t = fminf(32767.0f, fmaxf(-32767.0f, t));
            }
            dst[e] = (short)t;
        }
        __syncthreads();
    }
}

// Half-precision vectors (16-bit fixed point with a per-site fp32 norm): one thread per
// (site, right-hand side): norm = max|component| / 32767 (fp32), q = clamp(rint(component / norm)).
// v: float [n_sites][Nc][nrhs][2]; q: int16 same shape; norms: float [n_sites][nrhs].
__global__ void __launch_bounds__(128) quantize_vec_i16_kernel(const float2* v, long long n_sites, int Nc, int nrhs,
                                                               short2* q, float* norms) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= n_sites * nrhs) return;
    const long long s = idx / nrhs;
    const int r = (int)(idx % nrhs);
    float amax = 0.f;
    for (int a = 0; a < Nc; ++a) {
        const float2 x = v[(s * Nc + a) * nrhs + r];
        amax = fmaxf(amax, fmaxf(fabsf(x.x), fabsf(x.y)));
    }
    const float norm = amax == 0.f ? 0.f : __fdiv_rn(amax, 32767.0f);
    norms[idx] = norm;
    for (int a = 0; a < Nc; ++a) {
        const long long e = (s * Nc + a) * nrhs + r;
        short2 o = make_short2(0, 0);
        if (amax != 0.f) {
            const float2 x = v[e];
            o.x = (short)fminf(32767.f, fmaxf(-32767.f, rintf(__fdiv_rn(x.x, norm))));
            o.y = (short)fminf(32767.f, fmaxf(-32767.f, rintf(__fdiv_rn(x.y, norm))));
        }
        q[e] = o;
    }
}

}  // namespace coarse
