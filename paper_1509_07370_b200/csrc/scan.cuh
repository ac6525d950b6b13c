// scan.cuh -- device-wide exclusive prefix sum of u32 arrays (reduce / spine / downsweep).
// Used by the radix sort (tile histograms), the node numbering (a4) and the child-slot numbering.
// HBM-bound: 4 B read (reduce) + 4 B read + 4 B written (downsweep) per element.
#pragma once
#include "common.cuh"

namespace bh {

constexpr int kScanThreads = 256;
constexpr int kScanChunk = kScanThreads * 4 * 4;   // elements per block: 4 iterations of 256 x uint4

__device__ __forceinline__ u32 warp_incl_scan(u32 v)
{
    #pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        u32 t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane_id() >= (u32)o) v += t;
    }
    return v;
}

// exclusive scan of one value per thread over a 256-thread block; returns exclusive prefix, total in `total`
__device__ __forceinline__ u32 block_excl_scan_256(u32 v, u32& total, u32* s_warp /* >= 9 words */)
{
    const u32 incl = warp_incl_scan(v);
    const int w = threadIdx.x >> 5;
    if (lane_id() == 31) s_warp[w] = incl;
    __syncthreads();
    if (threadIdx.x < 32) {
        u32 t = threadIdx.x < 8 ? s_warp[threadIdx.x] : 0u;
        u32 ti = warp_incl_scan(t);
        if (threadIdx.x < 8) s_warp[threadIdx.x] = ti - t;
        if (threadIdx.x == 7) s_warp[8] = ti;
    }
    __syncthreads();
    const u32 r = s_warp[w] + incl - v;
    total = s_warp[8];
    __syncthreads();   // s_warp reusable after return
    return r;
}

__device__ __forceinline__ uint4 load4_guard(const u32* in, i64 e, i64 n)
{
    if (e + 3 < n) return *reinterpret_cast<const uint4*>(in + e);
    uint4 v = make_uint4(0, 0, 0, 0);
    if (e < n) v.x = in[e];
    if (e + 1 < n) v.y = in[e + 1];
    if (e + 2 < n) v.z = in[e + 2];
    return v;
}

__global__ void __launch_bounds__(kScanThreads)
scan_reduce_kernel(const u32* __restrict__ in, i64 n, u32* __restrict__ block_sums)
{
    chain_enter();
    const i64 base = (i64)blockIdx.x * kScanChunk;
    u32 s = 0;
    #pragma unroll
    for (int it = 0; it < 4; ++it) {
        const i64 e = base + ((i64)it * kScanThreads + threadIdx.x) * 4;
        uint4 v = load4_guard(in, e, n);
        s += v.x + v.y + v.z + v.w;
    }
    #pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    __shared__ u32 sw[8];
    if (lane_id() == 0) sw[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        u32 t = 0;
        for (int i = 0; i < 8; ++i) t += sw[i];
        block_sums[blockIdx.x] = t;
    }
}

// one block: exclusive scan of block_sums[nb] in place; total -> *total_out (may be null)
__global__ void __launch_bounds__(kScanThreads)
scan_spine_kernel(u32* __restrict__ block_sums, i64 nb, u32* __restrict__ total_out)
{
    chain_enter();
    __shared__ u32 s_warp[9];
    u32 carry = 0;
    for (i64 base = 0; base < nb; base += kScanThreads) {
        const i64 i = base + threadIdx.x;
        u32 v = i < nb ? block_sums[i] : 0u;
        u32 total;
        u32 ex = block_excl_scan_256(v, total, s_warp);
        if (i < nb) block_sums[i] = carry + ex;
        carry += total;
    }
    if (threadIdx.x == 0 && total_out) *total_out = carry;
}

__global__ void __launch_bounds__(kScanThreads)
scan_down_kernel(const u32* in, u32* out, i64 n, const u32* __restrict__ block_sums)   // in may alias out
{
    chain_enter();
    __shared__ u32 s_warp[9];
    const i64 base = (i64)blockIdx.x * kScanChunk;
    u32 carry = block_sums[blockIdx.x];
    #pragma unroll 1
    for (int it = 0; it < 4; ++it) {
        const i64 e = base + ((i64)it * kScanThreads + threadIdx.x) * 4;
        if (base + (i64)it * kScanThreads * 4 >= n) break;
        uint4 v = load4_guard(in, e, n);
        u32 t = v.x + v.y + v.z + v.w, total;
        u32 ex = carry + block_excl_scan_256(t, total, s_warp);
        uint4 o;
        o.x = ex; o.y = ex + v.x; o.z = o.y + v.y; o.w = o.z + v.z;
        if (e + 3 < n) *reinterpret_cast<uint4*>(out + e) = o;
        else {
            if (e < n) out[e] = o.x;
            if (e + 1 < n) out[e + 1] = o.y;
            if (e + 2 < n) out[e + 2] = o.z;
        }
        carry += total;
    }
}

// host helper: exclusive scan of in[n] into out[n] (may alias); scratch must hold ceil(n/kScanChunk) u32
inline cudaError_t exclusive_scan_u32(const u32* in, u32* out, i64 n, u32* scratch, u32* total_out,
                                      cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    const i64 nb = (n + kScanChunk - 1) / kScanChunk;
    cudaError_t e = launch_chain(scan_reduce_kernel, dim3((unsigned)nb), dim3(kScanThreads), 0, st, in, n, scratch);
    if (e != cudaSuccess) return e;
    e = launch_chain(scan_spine_kernel, dim3(1), dim3(kScanThreads), 0, st, scratch, nb, total_out);
    if (e != cudaSuccess) return e;
    e = launch_chain(scan_down_kernel, dim3((unsigned)nb), dim3(kScanThreads), 0, st, in, out, n, scratch);
    if (e != cudaSuccess) return e;
    return cudaGetLastError();
}
inline size_t scan_scratch_elems(i64 n) { return (size_t)((n + kScanChunk - 1) / kScanChunk) + 1; }

}  // namespace bh
