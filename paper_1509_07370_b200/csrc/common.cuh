// common.cuh -- shared device helpers of libbh (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "libbh is written for sm_100a (B200); compile with -gencode arch=compute_100a,code=sm_100a"
#endif

namespace bh {

typedef unsigned long long u64;
typedef unsigned int u32;
typedef long long i64;

constexpr int kMaxLevel = 21;      // 21 bits per dimension (K1)
constexpr int kWarp = 32;

__device__ __forceinline__ u32 lane_id() { return threadIdx.x & 31u; }
__device__ __forceinline__ u32 lanemask_lt()
{
    u32 m;
    asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
    return m;
}

// Number of whole 3-bit octree levels two 63-bit keys have in common (0..21).
// Keys use bits 0..62, so clz >= 1; identical keys share all 21 levels.
__device__ __forceinline__ int common_levels(u64 a, u64 b)
{
    u64 x = a ^ b;
    return x == 0 ? kMaxLevel : (__clzll((long long)x) - 1) / 3;
}

// streaming (evict-first) global accesses for data touched once per pass
template <typename T> __device__ __forceinline__ T ld_stream(const T* p) { return __ldcs(p); }
template <typename T> __device__ __forceinline__ void st_stream(T* p, T v) { __stcs(p, v); }

}  // namespace bh
