// sort.cuh -- step a2: stable least-significant-digit radix sort of (u64 key, u32 value) pairs,
// 8-bit digits.  Stable, so ties keep ascending original index (DESIGN.md S-rule: ascending (key, index)).
// Only digits that cover varying key bits are sorted (the host picks the passes from the OR/AND of
// all keys).  One histogram kernel counts every pass's digits in a single read of the keys; each pass
// is then ONE kernel: a tile ranks its pairs, publishes its digit counts and obtains its global
// offsets by decoupled look-back over the preceding tiles (tiles are handed out by a ticket counter,
// so a tile only ever waits for tiles that are already running).  HBM-bound: 8 B for the
// histograms + 24 B (12 B read, 12 B written) per pass and pair.
#pragma once
#include "common.cuh"
#include "scan.cuh"

namespace bh {

constexpr int kSortThreads = 256;
constexpr int kSortItems = 16;
constexpr int kSortTile = kSortThreads * kSortItems;   // 4096 pairs per CTA
constexpr int kRadix = 256;
constexpr int kMaxPasses = 8;
constexpr u32 kFlagAgg = 1u << 30, kFlagPrefix = 2u << 30, kValMask = (1u << 30) - 1u;   // tile status words

constexpr int kLookWin = 4;                      // tile status words a look-back step fetches at once
__device__ __forceinline__ u32 ld_status(const u32* p)
{
    u32 v;
    asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// lanes of the warp whose 8-bit digit equals this lane's, by ballots over the digit bits in `vary`
// (warp-uniform; must contain every bit on which the warp's digits differ).  Eight ballots when all
// bits vary (match.any slows down with every distinct value instead); cells that are neighbours in
// memory share most key bits, so a warp of grid data in original order needs only 2-3.
// one bit of the match: bit -> predicate, ballot, all-ones mask of the own bit, differ |= ballot ^ mask
// (written out in PTX: the compiler's own forms take five or six instructions per bit)
template <int B>
__device__ __forceinline__ void differ_step(u32& differ, u32 d)
{
    asm volatile("{\n\t.reg .pred p;\n\t.reg .b32 bal, t, s;\n\t"
                 "and.b32 t, %1, %2;\n\tsetp.ne.u32 p, t, 0;\n\t"
                 "vote.sync.ballot.b32 bal, p, 0xffffffff;\n\t"
                 "selp.b32 s, -1, 0, p;\n\t"
                 "lop3.b32 %0, %0, bal, s, 0xf6;\n\t}"
                 : "+r"(differ) : "r"(d), "n"(1 << B));
}

__device__ __forceinline__ u32 digit_peers_on(u32 d, u32 vary)
{
    u32 differ = 0u;                             // lanes whose digit differs from this lane's in some bit
    if (vary == 0xffu) {
        differ_step<0>(differ, d); differ_step<1>(differ, d); differ_step<2>(differ, d); differ_step<3>(differ, d);
        differ_step<4>(differ, d); differ_step<5>(differ, d); differ_step<6>(differ, d); differ_step<7>(differ, d);
    } else {
        while (vary) {
            const u32 m = vary & (0u - vary);                    // lowest bit still to match
            vary ^= m;
            asm volatile("{\n\t.reg .pred p;\n\t.reg .b32 bal, t, s;\n\t"
                         "and.b32 t, %1, %2;\n\tsetp.ne.u32 p, t, 0;\n\t"
                         "vote.sync.ballot.b32 bal, p, 0xffffffff;\n\t"
                         "selp.b32 s, -1, 0, p;\n\t"
                         "lop3.b32 %0, %0, bal, s, 0xf6;\n\t}"
                         : "+r"(differ) : "r"(d), "r"(m));
        }
    }
    return ~differ;
}
__device__ __forceinline__ u32 digit_peers(u32 d)
{
    return digit_peers_on(d, __reduce_or_sync(0xffffffffu, d ^ __shfl_sync(0xffffffffu, d, 0)));
}

// shared-memory add without a return value, 32-bit shared address
__device__ __forceinline__ void red_shared_add_if(u32 saddr, u32 v, bool on)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.u32 p, %2, 0;\n\t@p red.shared.add.u32 [%0], %1;\n\t}"
                 :: "r"(saddr), "r"(v), "r"((u32)on) : "memory");
}

struct SortPlan {
    int npasses;
    int shift[kMaxPasses];           // bit position of each pass's digit in the 63-bit key
    u32 mask[kMaxPasses];
    int lo;                          // lowest varying key bit
    int ib;                          // index bits of the packed word: ceil(log2 n)
    bool packed;                     // all varying bits inside [lo, lo + 64 - ib)
};

// ghist[p * pass_stride + d] = number of keys whose digit of pass p is d
__global__ void __launch_bounds__(kSortThreads)
radix_hist_strided_kernel(const u64* __restrict__ keys, i64 n, const SortPlan plan, u32* __restrict__ ghist,
                          u32 pass_stride)
{
    chain_enter();
    __shared__ u32 h[kMaxPasses * kRadix];
    for (int i = threadIdx.x; i < plan.npasses * kRadix; i += kSortThreads) h[i] = 0;
    __syncthreads();
    constexpr int kRows = 8;                              // rows of 32 keys a warp keeps in flight
    const i64 stride = (i64)gridDim.x * kSortThreads * kRows;
    const u32 lane = threadIdx.x & 31;
    u32 hbase = (u32)__cvta_generic_to_shared(h);
    asm volatile("" : "+r"(hbase));                       // keep the shared base in a register
    for (i64 wb = ((i64)blockIdx.x * kSortThreads + (threadIdx.x & ~31)) * kRows; wb < n; wb += stride) {   // warp-uniform
        u64 k[kRows];
        #pragma unroll
        for (int r = 0; r < kRows; ++r) k[r] = wb + 32 * r + lane < n ? ld_stream(keys + wb + 32 * r + lane) : 0ULL;
        const bool fullblk = wb + 32 * kRows <= n;            // warp-uniform
        #pragma unroll
        for (int p = 0; p < kMaxPasses; ++p) {          // static indices keep the plan in constant memory
            if (p >= plan.npasses) break;
            const int sh = plan.shift[p];
            const u32 mk = plan.mask[p];
            u32 d[kRows];
            bool alleq = true;
            #pragma unroll
            for (int r = 0; r < kRows; ++r) {
                d[r] = (u32)(k[r] >> sh) & mk;
                alleq = alleq && d[r] == d[0];
            }
            // Cells that are neighbours in memory share most key bits: a lane's keys of the 8 rows (32
            // elements apart) usually carry the same digit, and the upper digits are the same for the
            // whole block -- then one shared atomic per lane, or one per warp, counts all 256 keys.
            // (Same-address shared atomics are served one lane at a time, so this matters.)
            if (fullblk && __all_sync(0xffffffffu, alleq)) {
                int uni;
                __match_all_sync(0xffffffffu, d[0], &uni);
                red_shared_add_if(hbase + ((p * kRadix + d[0]) << 2), uni ? 32u * kRows : (u32)kRows, uni ? lane == 0 : true);
            } else {
                #pragma unroll
                for (int r = 0; r < kRows; ++r)
                    red_shared_add_if(hbase + ((p * kRadix + d[r]) << 2), 1u, wb + 32 * r + lane < n);
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < plan.npasses * kRadix; i += kSortThreads)
        if (h[i]) atomicAdd(&ghist[(size_t)(i >> 8) * pass_stride + (i & 255)], h[i]);
}

struct SortSmem {
    u32 klo[kSortTile];              // 16 KB  } the tile in digit order; slot q lives at swz(q), which
    u32 khi[kSortTile];              // 16 KB  } keeps power-of-two strides (digit starts) off one bank
    u32 wcnt[kSortThreads / 32][kRadix];   // 8 KB: per-warp digit counts, then per-warp digit offsets
    u32 dstart[kRadix];              // tile-local start of each digit
    u32 gbase[kRadix];               // global position of local slot q of digit d is gbase[d] + q
    u32 s_warp[9];
    u32 s_tile;
};
struct SortSmemVals { u32 vals[kSortTile]; };    // generic mode only: the values, behind SortSmem

// What one pass reads and writes.
//   kGenericFirst: reads keys, value = element index;  writes (key, value)
//   kGeneric     : reads (key, value);                 writes (key, value)
//   kPackedFirst : reads keys;  writes words (key bits [lo, lo + 64 - ib) << ib | element index)
//   kPacked      : reads words; writes words
enum SortMode { kGenericFirst = 0, kGeneric = 1, kPackedFirst = 2, kPacked = 3 };

// One pass.  status[tile * 256 + d]: flag (bits 31..30) | count (30 bits); ticket: next tile to hand out.
// `shift` addresses the digit inside the element this pass ranks on: the u64 key (generic modes and
// kPackedFirst, which ranks on the raw key) or the packed word (kPacked).
template <int MODE>
__global__ void __launch_bounds__(kSortThreads, (MODE >= kPackedFirst ? 4 : 3))
radix_onesweep_kernel(const u64* __restrict__ kin, const u32* __restrict__ vin, u64* __restrict__ kout,
                      u32* __restrict__ vout, const u32* __restrict__ ghist /* this pass: [256] */,
                      u32* __restrict__ status, u32* __restrict__ ticket, i64 n, int shift, u32 mask, int lo, int ib)
{
    chain_enter();
    constexpr bool kVals = MODE == kGenericFirst || MODE == kGeneric;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    SortSmem& S = *reinterpret_cast<SortSmem*>(smem_raw);
    u32* svals = reinterpret_cast<SortSmemVals*>(smem_raw + sizeof(SortSmem))->vals;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) S.s_tile = atomicAdd(ticket, 1u);
    for (int i = tid; i < (kSortThreads / 32) * kRadix; i += kSortThreads) (&S.wcnt[0][0])[i] = 0;
    __syncthreads();
    const int tile = (int)S.s_tile;
    const i64 base = (i64)tile * kSortTile;

    // warp-striped load: warp w owns the contiguous chunk [w*512, w*512+512) of the tile
    u64 key[kSortItems];
    u32 rank[kSortItems];
    const i64 wbase = base + (i64)warp * (32 * kSortItems);
    const bool full = base + kSortTile <= n;               // every tile but the last: no bounds checks
    if (full) {
        const u64* src = kin + wbase + lane;
        #pragma unroll
        for (int i = 0; i < kSortItems; ++i) key[i] = ld_stream(src + i * 32);
    } else {
        #pragma unroll
        for (int i = 0; i < kSortItems; ++i) {
            const i64 e = wbase + i * 32 + lane;
            key[i] = e < n ? ld_stream(kin + e) : ~0ULL;   // padding takes the top digit, last in the tile
        }
    }
    // stable rank inside the warp chunk: items are visited in memory order
    const u32 lt = (1u << lane) - 1u;
    #pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
        const u32 d = (u32)(key[i] >> shift) & mask;
        // first pass: the input is in memory order, neighbours share most digit bits
        const u32 peers = (MODE == kPackedFirst || MODE == kGenericFirst) ? digit_peers(d) : digit_peers_on(d, 0xffu);
        const u32 cnt = S.wcnt[warp][d];
        __syncwarp();
        const u32 r = __popc(peers & lt);
        if (r == 0) S.wcnt[warp][d] = cnt + __popc(peers);
        __syncwarp();
        rank[i] = cnt + r;
    }
    u32 val[kVals ? kSortItems : 1];
    if (MODE == kGeneric) {
        #pragma unroll
        for (int i = 0; i < kSortItems; ++i) {   // the values arrive while the digit offsets are worked out
            const i64 e = wbase + i * 32 + lane;
            val[i] = (full || e < n) ? ld_stream(vin + e) : 0u;
        }
    }
    __syncthreads();
    // thread d: exclusive scan of digit d over the warps, then over the digits
    const int dg = tid;
    u32 run = 0;
    #pragma unroll
    for (int w = 0; w < kSortThreads / 32; ++w) { u32 c = S.wcnt[w][dg]; S.wcnt[w][dg] = run; run += c; }
    // publish this tile's count of digit d; the look-back for the pairs of digit d in earlier tiles comes AFTER the
    // exchange through shared memory: by then more of the earlier tiles have published their prefixes
    volatile u32* st = status + (size_t)tile * kRadix + dg;
    if (tile == 0) *st = kFlagPrefix | run; else *st = kFlagAgg | run;
    u32 total;
    const u32 ex = block_excl_scan_256(run, total, S.s_warp);          // tile-local start of digit d
    const u32 gstart = block_excl_scan_256(ghist[dg], total, S.s_warp);  // global start of digit d
    S.dstart[dg] = ex;
    __syncthreads();
    #pragma unroll
    for (int i = 0; i < kSortItems; ++i) {
        const u32 d = (u32)(key[i] >> shift) & mask;
        const u32 q = S.dstart[d] + S.wcnt[warp][d] + rank[i];
        BH_DCHECK(q < (u32)kSortTile);
        const u32 qs = q ^ ((q >> 5) & 31u);
        const u32 e32 = (u32)(wbase + i * 32 + lane);
        if (MODE == kPackedFirst) {                         // word = key window | element index
            const u64 word = ((key[i] >> lo) << ib) | (u64)e32;
            S.klo[qs] = (u32)word;
            S.khi[qs] = (u32)(word >> 32);
        } else {
            S.klo[qs] = (u32)key[i];
            S.khi[qs] = (u32)(key[i] >> 32);
        }
        if (MODE == kGenericFirst) svals[qs] = e32;
        if (MODE == kGeneric) svals[qs] = val[i];
    }
    {
        const int d = dg;
        u32 before = 0;
        if (tile > 0) {
            // look-back in windows of kLookWin tiles: the window's status words are fetched together
            // (independent loads, one L2 round trip), then consumed nearest tile first
            bool done = false;
            for (int t0 = tile - 1; !done; t0 -= kLookWin) {
                u32 v[kLookWin];
                #pragma unroll
                for (int j = 0; j < kLookWin; ++j) {
                    const int t = t0 - j > 0 ? t0 - j : 0;
                    v[j] = ld_status(status + (size_t)t * kRadix + d);
                }
                #pragma unroll
                for (int j = 0; j < kLookWin; ++j) {
                    if (done) break;
                    u32 w = v[j];
                    while ((w >> 30) == 0u) w = ld_status(status + (size_t)(t0 - j) * kRadix + d);
                    before += w & kValMask;
                    if (w & kFlagPrefix) done = true;      // tile 0 always publishes a prefix
                }
            }
            *st = kFlagPrefix | (before + run);
        }
        S.gbase[d] = gstart + before - ex;
    }
    __syncthreads();
    const i64 left = n - base;
    const int nvalid = left < kSortTile ? (int)left : kSortTile;
    const int dshift = MODE == kPackedFirst ? shift - lo + ib : shift;   // the digit inside what was stored
    #pragma unroll 4
    for (int q = tid; q < nvalid; q += kSortThreads) {
        const u32 qs = (u32)q ^ (((u32)q >> 5) & 31u);
        const u64 k = ((u64)S.khi[qs] << 32) | S.klo[qs];
        const u32 d = (u32)(k >> dshift) & mask;
        const u32 g = S.gbase[d] + (u32)q;
        BH_DCHECK((i64)g < n);
        kout[g] = k;
        if (kVals) vout[g] = svals[qs];
    }
}

// passes covering exactly the varying bits [lo_bit, hi_bit] in 8-bit digits
inline SortPlan make_sort_plan(u64 varying, i64 n)
{
    SortPlan p;
    p.npasses = 0;
    p.lo = 0;
    p.ib = 1;
    while ((1LL << p.ib) < n) ++p.ib;
    p.packed = false;
    if (varying == 0) return p;
    int lo = __builtin_ctzll(varying), hi = 63 - __builtin_clzll(varying);
    p.lo = lo;
    p.packed = hi - lo + 1 <= 64 - p.ib;
    for (int b = lo; b <= hi; b += 8) {
        int w = hi - b + 1 < 8 ? hi - b + 1 : 8;
        p.shift[p.npasses] = b;
        p.mask[p.npasses] = (1u << w) - 1u;
        ++p.npasses;
    }
    return p;
}

inline i64 sort_tiles(i64 n) { return (n + kSortTile - 1) / kSortTile; }
// u32 words of sort scratch: per pass [256 histogram][ntiles * 256 status][1 ticket]
inline size_t sort_pass_words(i64 n) { return (size_t)kRadix + (size_t)sort_tiles(n) * kRadix + 1; }
inline size_t sort_hist_elems(i64 n) { return (size_t)kMaxPasses * sort_pass_words(n); }
inline size_t sort_smem_bytes(bool packed) { return sizeof(SortSmem) + (packed ? 0 : sizeof(SortSmemVals)); }

// Sorts the n keys in k0 (values = their indices 0..n-1, implicit) in plan.npasses >= 1 passes, ping-ponging
// between (k0, v0) and (k1, v1); pass p writes to buffer 1 if p is even, else to buffer 0, so the result
// is in buffer (npasses & 1).  Packed plans never touch v0 / v1 (may be null).
// scratch holds plan.npasses * sort_pass_words(n) u32, all zero on entry if scratch_is_clear (else cleared here).
// `mark(name, algorithmic bytes)` is called after every launch (bh_build's optional per-pass timing).
template <class Mark>
inline cudaError_t radix_sort_pairs(u64* k0, u32* v0, u64* k1, u32* v1, i64 n, const SortPlan& plan, u32* scratch,
                                    bool scratch_is_clear, int hist_grid, cudaStream_t st, Mark&& mark)
{
    if (plan.npasses == 0) return cudaSuccess;
    const size_t pw = sort_pass_words(n);
    const int ntiles = (int)sort_tiles(n);
    cudaError_t e = cudaSuccess;
    if (!scratch_is_clear) e = cudaMemsetAsync(scratch, 0, sizeof(u32) * pw * plan.npasses, st);
    if (e != cudaSuccess) return e;
    // all histograms in one read; each pass's 256 counters sit at the head of its scratch block
    e = launch_chain(radix_hist_strided_kernel, dim3(hist_grid), dim3(kSortThreads), 0, st, k0, n, plan, scratch, (u32)pw);
    if (e != cudaSuccess) return e;
    mark("sort_hist", 8.0 * (double)n);
    const size_t smem = sort_smem_bytes(plan.packed);
    for (int p = 0; p < plan.npasses; ++p) {
        u32* blk = scratch + pw * p;
        u32* status = blk + kRadix;
        u32* ticket = status + (size_t)ntiles * kRadix;
        if (plan.packed) {
            if (p == 0)
                e = launch_chain(radix_onesweep_kernel<kPackedFirst>, dim3(ntiles), dim3(kSortThreads), smem, st,
                                 k0, nullptr, k1, nullptr, blk, status, ticket, n, plan.shift[p], plan.mask[p], plan.lo, plan.ib);
            else   // the key window sits above the index bits of the word
                e = launch_chain(radix_onesweep_kernel<kPacked>, dim3(ntiles), dim3(kSortThreads), smem, st,
                                 k0, nullptr, k1, nullptr, blk, status, ticket, n, plan.shift[p] - plan.lo + plan.ib, plan.mask[p], plan.lo, plan.ib);
        } else {
            if (p == 0)
                e = launch_chain(radix_onesweep_kernel<kGenericFirst>, dim3(ntiles), dim3(kSortThreads), smem, st,
                                 k0, nullptr, k1, v1, blk, status, ticket, n, plan.shift[p], plan.mask[p], plan.lo, plan.ib);
            else
                e = launch_chain(radix_onesweep_kernel<kGeneric>, dim3(ntiles), dim3(kSortThreads), smem, st,
                                 k0, v0, k1, v1, blk, status, ticket, n, plan.shift[p], plan.mask[p], plan.lo, plan.ib);
        }
        if (e != cudaSuccess) return e;
        mark("sort_pass", 24.0 * (double)n);          // 12 B read + 12 B written per pair and pass
        u64* tk = k0; k0 = k1; k1 = tk;
        u32* tv = v0; v0 = v1; v1 = tv;
    }
    return cudaGetLastError();
}

}  // namespace bh
