// common.cuh -- shared device helpers of libbh (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "libbh is written for sm_100a (B200); compile with -gencode arch=compute_100a,code=sm_100a"
#endif

// Checked build (`python -m paper_1509_07370_b200.build --checked` -> libbh_checked.so, -DBH_CHECKED): bounds checks
// of our own on every index the kernels compute -- stack and list fills of the walk, slots, node ids, sort positions.
// compute-sanitizer is not available on this GPU pool, so tests/test_gpu_checked.py runs the small parity cases
// through this library in a subprocess; a failed check traps the kernel and the call returns BH_ERR_CUDA.
#ifdef BH_CHECKED
#include <assert.h>
#define BH_DCHECK(cond) assert(cond)
#else
#define BH_DCHECK(cond) ((void)0)
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

// Programmatic dependent launch for the chains of short kernels in bh_build (histogram -> sort passes -> count ->
// scan -> totals; assign -> moments level by level): a kernel launched with launch_chain() may be made resident
// while its predecessor in the stream drains, and starts its work at chain_enter(), which returns once the
// predecessor has completed and its writes are visible -- the launch latency and the ramp-up of every kernel
// overlap the tail of the one before.  chain_enter() must come before the first global access; in a kernel
// launched the ordinary way it returns at once.
__device__ __forceinline__ void chain_enter()
{
#ifndef BH_NO_PDL
    asm volatile("griddepcontrol.launch_dependents;\n\tgriddepcontrol.wait;" ::: "memory");
#endif
}
template <typename... KArgs, typename... Args>
inline cudaError_t launch_chain(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                Args&&... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
#ifndef BH_NO_PDL
    cfg.numAttrs = 1;
#else
    cfg.numAttrs = 0;
#endif
    return cudaLaunchKernelEx(&cfg, kern, static_cast<KArgs>(args)...);
}

// streaming (evict-first) global accesses for data touched once per pass
template <typename T> __device__ __forceinline__ T ld_stream(const T* p) { return __ldcs(p); }
template <typename T> __device__ __forceinline__ void st_stream(T* p, T v) { __stcs(p, v); }

// The cells in sorted order (ascending (key, original index)) as the sort leaves them:
//   packed   : one u64 per cell = (key bits [lo, lo + 64 - ib) << ib) | original index, ib = ceil(log2 n) index
//              bits -- used whenever all varying key bits fit in the 64 - ib bits left (40 at 16.8 M cells: every
//              grid up to 4096^3 and the AMR workloads); cbits holds the key bits outside that window, which are
//              the same for all cells;
//   generic  : keys[] + idx[];
//   identity : all keys equal, nothing was sorted: keys[] as generated, idx(s) = s.
struct SortedView {
    const u64* packed;
    const u64* keys;
    const u32* idx;
    u64 cbits;
    int lo;
    int ib;
};
__device__ __forceinline__ u64 sv_key(const SortedView& v, i64 s)
{
    return v.packed ? (((v.packed[s] >> v.ib) << v.lo) | v.cbits) : v.keys[s];
}
__device__ __forceinline__ u32 sv_idx(const SortedView& v, i64 s)
{
    return v.packed ? (u32)(v.packed[s] & ((1ULL << v.ib) - 1ULL)) : (v.idx ? v.idx[s] : (u32)s);
}

// c(s): octree levels the keys of sorted cells s and s+1 share (s + 1 < n).  In the packed form only the
// key windows differ, so the highest differing key bit is lo + 63 - clz(xor of the windows).
__device__ __forceinline__ int window_common_levels(u64 x, int lo)     // x = xor of two key windows
{
    return x == 0ULL ? kMaxLevel : (__clzll((long long)x) - 1 - lo) / 3;   // (62 - (lo + 63 - clz)) / 3
}
__device__ __forceinline__ int sv_common_levels(const SortedView& v, i64 s)
{
    if (v.packed) return window_common_levels((v.packed[s] ^ v.packed[s + 1]) >> v.ib, v.lo);
    return common_levels(v.keys[s], v.keys[s + 1]);
}

}  // namespace bh
