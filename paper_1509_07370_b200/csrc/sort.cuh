// sort.cuh -- step a2: stable least-significant-digit radix sort of (u64 key, u32 value) pairs,
// 8-bit digits, one pass = tile histograms -> device scan -> ranked scatter.
// Stable, so ties keep ascending original index (DESIGN.md S-rule: ascending (key, index)).
// Only digits that cover varying key bits are sorted (the host picks the passes from the OR/AND of
// all keys).  HBM-bound: per pass 8 B (histogram read) + 12 B read + 12 B written per pair.
#pragma once
#include "common.cuh"
#include "scan.cuh"

namespace bh {

constexpr int kSortThreads = 256;
constexpr int kSortItems = 16;
constexpr int kSortTile = kSortThreads * kSortItems;   // 4096 pairs per CTA
constexpr int kRadix = 256;

// per-tile digit histogram, written digit-major: hist[d * ntiles + tile]
__global__ void __launch_bounds__(kSortThreads)
radix_hist_kernel(const u64* __restrict__ keys, i64 n, int shift, u32 mask, u32* __restrict__ hist, int ntiles)
{
    __shared__ u32 h[kRadix];
    h[threadIdx.x] = 0;
    __syncthreads();
    const i64 base = (i64)blockIdx.x * kSortTile;
    #pragma unroll 4
    for (int i = 0; i < kSortItems; ++i) {
        const i64 e = base + (i64)i * kSortThreads + threadIdx.x;
        if (e < n) atomicAdd(&h[(u32)(ld_stream(keys + e) >> shift) & mask], 1u);
    }
    __syncthreads();
    hist[(size_t)threadIdx.x * ntiles + blockIdx.x] = h[threadIdx.x];
}

struct SortSmem {
    u64 keys[kSortTile];             // 32 KB
    u32 vals[kSortTile];             // 16 KB
    u32 wcnt[kSortThreads / 32][kRadix];   // 8 KB: per-warp digit counts, then per-warp digit offsets
    u32 dstart[kRadix];              // tile-local start of each digit
    u32 gbase[kRadix];               // global position of local slot q of digit d is gbase[d] + q
    u32 s_warp[9];
};

__global__ void __launch_bounds__(kSortThreads)
radix_scatter_kernel(const u64* __restrict__ kin, const u32* __restrict__ vin, u64* __restrict__ kout,
                     u32* __restrict__ vout, const u32* __restrict__ tile_offs, i64 n, int ntiles,
                     int shift, u32 mask)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SortSmem& S = *reinterpret_cast<SortSmem*>(smem_raw);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int tile = blockIdx.x;
    const i64 base = (i64)tile * kSortTile;

    for (int i = tid; i < (kSortThreads / 32) * kRadix; i += kSortThreads) (&S.wcnt[0][0])[i] = 0;
    __syncthreads();

    // warp-striped load: warp w owns the contiguous chunk [w*512, w*512+512) of the tile
    u64 key[kSortItems];
    u32 val[kSortItems];
    u32 rank[kSortItems];
    const i64 wbase = base + (i64)warp * (32 * kSortItems);
    #pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
        const i64 e = wbase + i * 32 + lane;
        const bool ok = e < n;
        key[i] = ok ? ld_stream(kin + e) : ~0ULL;
        val[i] = ok ? ld_stream(vin + e) : 0u;
    }
    // stable rank inside the warp chunk: items are visited in memory order
    const u32 lt = lanemask_lt();
    #pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
        const u32 d = (u32)(key[i] >> shift) & mask;     // padding keys (~0) take the top digit, last
        const u32 peers = __match_any_sync(0xffffffffu, d);
        const u32 cnt = S.wcnt[warp][d];
        __syncwarp();
        const u32 r = __popc(peers & lt);
        if (r == 0) S.wcnt[warp][d] = cnt + __popc(peers);
        __syncwarp();
        rank[i] = cnt + r;
    }
    __syncthreads();
    {   // thread d: exclusive scan of digit d over the warps, then over the digits
        const int d = tid;
        u32 run = 0;
        #pragma unroll
        for (int w = 0; w < kSortThreads / 32; ++w) { u32 c = S.wcnt[w][d]; S.wcnt[w][d] = run; run += c; }
        u32 total;
        const u32 ex = block_excl_scan_256(run, total, S.s_warp);
        S.dstart[d] = ex;
        S.gbase[d] = tile_offs[(size_t)d * ntiles + tile] - ex;
    }
    __syncthreads();
    #pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
        const u32 d = (u32)(key[i] >> shift) & mask;
        const u32 q = S.dstart[d] + S.wcnt[warp][d] + rank[i];
        S.keys[q] = key[i];
        S.vals[q] = val[i];
    }
    __syncthreads();
    const i64 left = n - base;
    const int nvalid = left < kSortTile ? (int)left : kSortTile;
    #pragma unroll 4
    for (int q = tid; q < nvalid; q += kSortThreads) {
        const u64 k = S.keys[q];
        const u32 d = (u32)(k >> shift) & mask;
        const u32 g = S.gbase[d] + (u32)q;
        kout[g] = k;
        vout[g] = S.vals[q];
    }
}

struct SortPlan {
    int npasses;
    int shift[8];
    u32 mask[8];
};

// passes covering exactly the varying bits [lo_bit, hi_bit] in 8-bit digits
inline SortPlan make_sort_plan(u64 varying)
{
    SortPlan p;
    p.npasses = 0;
    if (varying == 0) return p;
    int lo = __builtin_ctzll(varying), hi = 63 - __builtin_clzll(varying);
    for (int b = lo; b <= hi; b += 8) {
        int w = hi - b + 1 < 8 ? hi - b + 1 : 8;
        p.shift[p.npasses] = b;
        p.mask[p.npasses] = (1u << w) - 1u;
        ++p.npasses;
    }
    return p;
}

inline size_t sort_hist_elems(i64 n) { return (size_t)kRadix * (size_t)((n + kSortTile - 1) / kSortTile); }

// one pass (k0,v0) -> (k1,v1); hist holds sort_hist_elems(n) u32, scratch scan_scratch_elems(that)
inline cudaError_t radix_pass(const u64* k0, const u32* v0, u64* k1, u32* v1, i64 n, int shift, u32 mask,
                              u32* hist, u32* scan_scratch, cudaStream_t st)
{
    const int ntiles = (int)((n + kSortTile - 1) / kSortTile);
    radix_hist_kernel<<<ntiles, kSortThreads, 0, st>>>(k0, n, shift, mask, hist, ntiles);
    cudaError_t e = exclusive_scan_u32(hist, hist, (i64)kRadix * ntiles, scan_scratch, nullptr, st);
    if (e != cudaSuccess) return e;
    radix_scatter_kernel<<<ntiles, kSortThreads, sizeof(SortSmem), st>>>(k0, v0, k1, v1, hist, n, ntiles,
                                                                         shift, mask);
    return cudaGetLastError();
}

}  // namespace bh
