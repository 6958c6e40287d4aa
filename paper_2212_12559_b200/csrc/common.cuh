// common.cuh — lattice indexing and PTX helpers shared by the coarse-op kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace coarse {

// Periodic 4-D lattice, site index s(x) = x0 + L0*(x1 + L1*(x2 + L2*x3))  (include/coarse_op.h).
struct Lat {
    int L[4];
    int V;
};

// Site whose data stage m of output site s needs:
//   m = 0           -> s
//   dagger = 0      -> vector from x+mu^ (m = 1+mu) / x-mu^ (m = 5+mu); the link matrix is at s itself
//   dagger = 1      -> link AND vector from x-mu^ (m = 1+mu) / x+mu^ (m = 5+mu)
__device__ __forceinline__ int stencil_site(const Lat& lat, int s, int m, int dagger) {
    if (m == 0) return s;
    const int mu = (m - 1) & 3;
    int sign = (m <= 4) ? 1 : -1;
    if (dagger) sign = -sign;
    int stride = 1;
#pragma unroll
    for (int d = 0; d < 3; ++d)
        if (d < mu) stride *= lat.L[d];
    const int Lmu = mu == 0 ? lat.L[0] : mu == 1 ? lat.L[1] : mu == 2 ? lat.L[2] : lat.L[3];
    const int x = (s / stride) % Lmu;
    int xn = x + sign;
    if (xn == Lmu) xn = 0;
    if (xn < 0) xn = Lmu - 1;
    return s + (xn - x) * stride;
}

// The same neighbour with the site's coordinates already known (one set of divisions per ITEM
// instead of two per pipeline stage: the TMA producer is a single thread and its instruction
// latency, not HBM, was what capped the int16 path).  m is a compile-time constant at every call
// site, so x[mu] and the stride fold into registers.
struct SiteX {
    int x0, x1, x2, x3;
    int st1, st2, st3;   // strides L0, L0*L1, L0*L1*L2
};
__device__ __forceinline__ SiteX site_coords(const Lat& lat, int s) {
    SiteX c;
    c.st1 = lat.L[0];
    c.st2 = lat.L[0] * lat.L[1];
    c.st3 = c.st2 * lat.L[2];
    const unsigned us = (unsigned)s;
    const unsigned q1 = us / (unsigned)lat.L[0];
    c.x0 = (int)(us - q1 * (unsigned)lat.L[0]);
    const unsigned q2 = q1 / (unsigned)lat.L[1];
    c.x1 = (int)(q1 - q2 * (unsigned)lat.L[1]);
    const unsigned q3 = q2 / (unsigned)lat.L[2];
    c.x2 = (int)(q2 - q3 * (unsigned)lat.L[2]);
    c.x3 = (int)q3;
    return c;
}
__device__ __forceinline__ int stencil_site_x(const Lat& lat, int s, const SiteX& c, int m, int dagger) {
    if (m == 0) return s;
    const int mu = (m - 1) & 3;
    bool fwd = (m <= 4);
    if (dagger) fwd = !fwd;
    const int x = mu == 0 ? c.x0 : mu == 1 ? c.x1 : mu == 2 ? c.x2 : c.x3;
    const int Lmu = mu == 0 ? lat.L[0] : mu == 1 ? lat.L[1] : mu == 2 ? lat.L[2] : lat.L[3];
    const int stride = mu == 0 ? 1 : mu == 1 ? c.st1 : mu == 2 ? c.st2 : c.st3;
    if (fwd) return (x + 1 == Lmu) ? s - x * stride : s + stride;
    return (x == 0) ? s + (Lmu - 1) * stride : s - stride;
}

// Site index of the h-th site of a parity (all extents even, checked by the host): consecutive
// h walk along x0 in steps of 2, the offset in x0 alternates with x1+x2+x3.
__device__ __forceinline__ int parity_site(const Lat& lat, int h, int parity) {
    const unsigned half = (unsigned)lat.L[0] >> 1;
    const unsigned q1 = (unsigned)h / half;            // = x1 + L1*(x2 + L2*x3)
    const unsigned x0h = (unsigned)h - q1 * half;
    const unsigned q2 = q1 / (unsigned)lat.L[1];
    const unsigned x1 = q1 - q2 * (unsigned)lat.L[1];
    const unsigned x3 = q2 / (unsigned)lat.L[2];
    const unsigned x2 = q2 - x3 * (unsigned)lat.L[2];
    const unsigned off = (x1 + x2 + x3 + (unsigned)parity) & 1u;
    return (int)(q1 * (unsigned)lat.L[0] + 2u * x0h + off);
}

namespace ptx {

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// 1-D TMA bulk copy global -> shared, completion counted in bytes on an mbarrier.
// dst, src 16-byte aligned; bytes a multiple of 16.
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar,
                                         uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
        ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(policy)
        : "memory");
}
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(pred));
    return pred != 0;
}
// Programmatic dependent launch (PDL): let the next kernel of the stream start its CTAs as ours drain,
// and make a dependent kernel wait for the previous kernel's memory before it reads it.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void named_bar_sync(int id, int threads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(threads) : "memory");
}
__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ uint4 lds128u(uint32_t addr) {
    uint4 v;
    asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(addr));
    return v;
}
// Packed fp32 pairs (sm_100: fma.rn.f32x2 / add.rn.f32x2, SASS FFMA2 / FADD2): one issue slot for two
// independent IEEE fp32 operations on an aligned register pair.
__device__ __forceinline__ float2 ffma2(const float2 a, const float2 b, const float2 c) {
    uint64_t d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;"
        : "=l"(d)
        : "l"(reinterpret_cast<const uint64_t&>(a)), "l"(reinterpret_cast<const uint64_t&>(b)),
          "l"(reinterpret_cast<const uint64_t&>(c)));
    return reinterpret_cast<float2&>(d);
}
__device__ __forceinline__ float2 fadd2(const float2 a, const float2 b) {
    uint64_t d;
    asm("add.rn.f32x2 %0, %1, %2;"
        : "=l"(d)
        : "l"(reinterpret_cast<const uint64_t&>(a)), "l"(reinterpret_cast<const uint64_t&>(b)));
    return reinterpret_cast<float2&>(d);
}
__device__ __forceinline__ float2 lds64(uint32_t addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0,%1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}

}  // namespace ptx

// int16 (re,im) packed in one 32-bit word -> two floats (exact), without the int->float
// conversion instruction: I2F issues on the quarter-rate XU pipe, and at HBM rate the int16 path
// needs ~13 conversions per clock per SM of the 16 that pipe can do (ncu: XU 70 % busy, the
// limiter of config C4).  Instead: q ^ 0x8000 = q + 32768 as an unsigned 16-bit number u; placing
// u in the low mantissa bits of 2^23 gives the float 2^23 + u exactly; subtracting 2^23 + 32768
// (exact: all three are integers below 2^24) leaves q.  One LOP3 per word, one PRMT and one FADD
// per value, all on the full-rate ALU/FMA pipes.
__device__ __forceinline__ float2 unpack_i16x2(uint32_t w) {
    const uint32_t u = w ^ 0x80008000u;
    const uint32_t lo = __byte_perm(u, 0x4B000000u, 0x7610);
    const uint32_t hi = __byte_perm(u, 0x4B000000u, 0x7632);
    return ptx::fadd2(make_float2(__uint_as_float(lo), __uint_as_float(hi)), make_float2(-8421376.0f, -8421376.0f));
}

// The same decode through the conversion unit (I2F on the quarter-rate XU pipe).  The int16 STREAM
// kernels decode XU of the 4 words of a link quad this way: with everything on the ALU/FMA pipes the
// kernel is issue-bound (68 % of the issue slots, ncu) while the XU pipe idles, and with everything on
// the XU pipe that pipe is the limiter (70 % busy).  Measured on C4 (sustained): dagger = 0
// 2.29 / 2.25 / 2.16 / 2.30 ms for XU = 0 / 1 / 2 / 3, dagger = 1 2.42 / 2.31 / 2.39 / 2.40 ms.
__device__ __forceinline__ float2 unpack_i16x2_xu(uint32_t w) {
    return make_float2((float)(short)(w & 0xffffu), (float)(short)(w >> 16));
}
template <int XU>
__device__ __forceinline__ void unpack_i16_quad(const uint4& t, float2& m0, float2& m1, float2& m2, float2& m3) {
    m0 = XU >= 4 ? unpack_i16x2_xu(t.x) : unpack_i16x2(t.x);
    m1 = XU >= 3 ? unpack_i16x2_xu(t.y) : unpack_i16x2(t.y);
    m2 = XU >= 2 ? unpack_i16x2_xu(t.z) : unpack_i16x2(t.z);
    m3 = XU >= 1 ? unpack_i16x2_xu(t.w) : unpack_i16x2(t.w);
}

}  // namespace coarse
