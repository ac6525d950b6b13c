// fma_peak.cu -- a MEASUREMENT AID of bench.py, not part of libbh and not in include/bh.h.
// A measured FP32 denominator for the walk's roofline (report against the nominal peak
// AND a measured FMA-chain peak; MEASURED_PEAKS.json has HBM and bf16 tensor figures only).
// Every thread runs 8 independent chains of packed fp32 FMAs (FFMA2, the instruction the walk's
// evaluation issues) or of scalar FMAs from registers; nothing touches memory until the final store.
// Built as its own small library (libbh_fma_peak.so) by paper_1509_07370_b200/build.py.
#include <cuda_runtime.h>

namespace {

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

}  // namespace

// Best of three timed repetitions (after one warm-up) of each chain kernel on `device`, in TFLOP/s
// (2 flops per FMA).  Returns 0, or the cudaError_t that stopped it.  Synchronises the device.
extern "C" int bh_fma_peak_measure(int device, double* tflops_packed, double* tflops_scalar)
{
    if (!tflops_packed || !tflops_scalar) return (int)cudaErrorInvalidValue;
    cudaError_t e;
    if ((e = cudaSetDevice(device)) != cudaSuccess) return (int)e;
    int sms = 0;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device)) != cudaSuccess) return (int)e;
    const int grid = sms * 8, iters = 1 << 15;
    float* out = nullptr;
    if ((e = cudaMalloc(&out, sizeof(float) * (size_t)grid * 256)) != cudaSuccess) return (int)e;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const double flops = (double)grid * 256.0 * iters * kPeakChains * 2.0 * 2.0;   // 2 lanes x (mul + add)
    double* res[2] = {tflops_packed, tflops_scalar};
    for (int v = 0; v < 2 && e == cudaSuccess; ++v) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; ++rep) {          // first repetition warms up
            cudaEventRecord(e0, 0);
            if (v == 0) fp32_fma_chain_kernel<true><<<grid, 256>>>(out, iters, 0.999f, 1e-3f);
            else fp32_fma_chain_kernel<false><<<grid, 256>>>(out, iters, 0.999f, 1e-3f);
            cudaEventRecord(e1, 0);
            if ((e = cudaDeviceSynchronize()) != cudaSuccess) break;
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        *res[v] = flops / (best * 1e-3) / 1e12;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    return (int)e;
}
