// peak.cuh -- a measured FP32 denominator for the walk's roofline (report against the
// nominal peak AND a measured FMA-chain peak; MEASURED_PEAKS.json has HBM and bf16 tensor figures only).
// Every thread runs 8 independent chains of packed fp32 FMAs (FFMA2, the instruction the walk's
// evaluation uses) or of scalar FMAs; nothing touches memory until the final store.
#pragma once
#include "common.cuh"

namespace bh {

constexpr int kPeakChains = 8;

template <bool PACKED>
__global__ void __launch_bounds__(256)
fp32_fma_chain_kernel(float* __restrict__ out, int iters, float a, float b)
{
    float2 x[kPeakChains];
    #pragma unroll
    for (int k = 0; k < kPeakChains; ++k) x[k] = make_float2(1.0f + 1e-3f * (float)(threadIdx.x + k), 0.5f + 1e-3f * (float)k);
    const float2 aa = make_float2(a, a), bb = make_float2(b, b);
    for (int i = 0; i < iters; ++i) {
        #pragma unroll
        for (int k = 0; k < kPeakChains; ++k) {
            if (PACKED) x[k] = __ffma2_rn(x[k], aa, bb);
            else { x[k].x = __fmaf_rn(x[k].x, a, b); x[k].y = __fmaf_rn(x[k].y, a, b); }
        }
    }
    float s = 0.f;
    #pragma unroll
    for (int k = 0; k < kPeakChains; ++k) s += x[k].x + x[k].y;
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace bh
