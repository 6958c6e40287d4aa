// probe_kernel.cuh — read-bandwidth ceiling probe: the STREAM kernel's TMA ring
// with an idle consumer.  One elected producer lane per SM streams `bytes` of global memory through
// an S-stage shared-memory ring with the same evict_first bulk copies the apply uses; one consumer
// warp only waits for each stage and hands the slot back.  What it measures is the rate at which
// this chip delivers a pure read stream to the SMs - the practical ceiling of the apply kernels
// (bench.py reports it beside the roofline; MEASURED_PEAKS.json's copy figure is half writes).
#pragma once
#include "common.cuh"

namespace coarse {

__global__ void __launch_bounds__(64, 1) probe_read_kernel(const unsigned char* src, unsigned long long n_stages,
                                                           int stage_bytes, int S, float* sink) {
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + (size_t)S * stage_bytes);
    const uint32_t full0 = ptx::smem_u32(bars), empty0 = full0 + 8u * S;
    if (threadIdx.x == 0) {
        for (int i = 0; i < S; ++i) {
            ptx::mbar_init(full0 + 8u * i, 1);
            ptx::mbar_init(empty0 + 8u * i, 1);
        }
        ptx::fence_mbar_init();
    }
    __syncthreads();
    const int warp = threadIdx.x >> 5;
    int slot = 0;
    uint32_t phase = 0;
    if (warp == 0) {
        const uint64_t pol = ptx::policy_evict_first();
        const uint32_t base = ptx::smem_u32(smem);
        for (unsigned long long st = blockIdx.x; st < n_stages; st += gridDim.x) {
            ptx::mbar_wait(empty0 + 8u * slot, phase ^ 1u);
            if (ptx::elect_one()) {
                ptx::mbar_arrive_expect_tx(full0 + 8u * slot, stage_bytes);
                ptx::bulk_g2s(base + slot * stage_bytes, src + st * (size_t)stage_bytes, stage_bytes, full0 + 8u * slot, pol);
            }
            __syncwarp();
            if (++slot == S) { slot = 0; phase ^= 1u; }
        }
    } else {
        float acc = 0.f;
        for (unsigned long long st = blockIdx.x; st < n_stages; st += gridDim.x) {
            ptx::mbar_wait(full0 + 8u * slot, phase);
            acc += reinterpret_cast<const float*>(smem + (size_t)slot * stage_bytes)[threadIdx.x & 31];
            __syncwarp();
            if ((threadIdx.x & 31) == 0) ptx::mbar_arrive(empty0 + 8u * slot);
            if (++slot == S) { slot = 0; phase ^= 1u; }
        }
        if (sink && acc == 1.2345678f) sink[0] = acc;   // keeps the read alive, never true in practice
    }
}

}  // namespace coarse
