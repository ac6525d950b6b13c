// tree.cuh -- steps a3 (permute), a4 (octree topology from sorted keys) and a5 (monopole moments).
//
// The tree is the one PAPER.md:45 (§2) defines -- the cube "is recursively divided into eight sub
// cells ... until only one particle is left for every sub cell" -- under DESIGN.md T1-T5:
// a node is (level l, prefix = key >> 3(21-l)) and owns the contiguous sorted range of cells that
// share the prefix; ranges of >= 2 cells are internal nodes (single-child chains kept), one cell is
// a leaf cell, >= 2 cells with identical keys form a level-21 bucket.
//
// Construction (no locks, no spinning, no searches; the paper inserts cells top-down under locks,
// PAPER.md:146-150):
//   c(s) = number of octree levels the keys of sorted cells s and s+1 share (c(-1) = c(n-1) = -1).
//   Cell s starts an internal node at every level l with c(s-1) < l <= c(s), and it is a leaf
//   child ("leaf entity") at level max(c(s-1), c(s)) + 1 (level 22 = member of a level-21 bucket).
//   A node's children are exactly the level-(l+1) entities inside its range, so:
//     * slot order   = all entities sorted by (level, s): the children of one node are contiguous
//       and in octant order, children of consecutive canonical nodes are consecutive, root = slot 0;
//     * canonical id = internal entities sorted by (level, s) = (level, prefix) order (T5);
//     * the first child of node (l, s) is the entity (l+1, s) of the SAME cell, and the child count
//       is the distance to the first child of the next canonical node.
//   Both orders are stable counting sorts by level with variable fan-out per cell: one counting
//   kernel (per-warp-chunk level histograms), one device scan, one assigning kernel that also
//   gathers the cell data into its slot (a3 is fused into it).
// Moments (Eq. 5; delta PAPER.md:54, 158) are reduced level by level from the
// deepest level up, each node from its children in ascending octant order in fp64 (M-rules).
#pragma once
#include "common.cuh"
#include "keys.cuh"

namespace bh {

constexpr int kNumLevels = kMaxLevel + 1;        // node levels 0..21
constexpr int kSlotLevels = kMaxLevel + 2;       // entity levels 0..22
constexpr int kTopoDigits = kSlotLevels + kNumLevels;   // histogram rows: entities per level, nodes per level
constexpr int kTopoThreads = 256;
constexpr int kTopoItems = 8;
constexpr int kTopoChunk = 32 * kTopoItems;      // cells per warp chunk

struct __align__(16) WalkAux {   // per slot, beside the float4 record (x, y, z, m)
    float size;      // node edge l (fp32 of L/2^level); +inf for a level-21 bucket; 0 for a leaf cell
    float delta;     // |R - geometric centre| (fp32)
    u32 first;       // slot of the first child
    u32 count;       // number of children (0: this slot is a leaf cell)
};

inline i64 topo_chunks(i64 n) { return (n + kTopoChunk - 1) / kTopoChunk; }
inline size_t topo_hist_elems(i64 n) { return (size_t)kTopoDigits * (size_t)topo_chunks(n); }

// entity / internal-node level masks of a cell from c(s-1) = cp and c(s) = cs
__device__ __forceinline__ void entity_masks(int cp, int cs, u32& imask, u32& emask)
{
    imask = cs > cp ? (((1u << (cs + 1)) - 1u) & ~((1u << (cp + 1)) - 1u)) : 0u;
    emask = imask | (1u << ((cp > cs ? cp : cs) + 1));
}

// ---- a4.1: c(s) per cell and the level histograms of every warp chunk -----------------------------
// hist[d * nchunks + chunk]: d < kSlotLevels: entities of level d starting in the chunk;
//                            d >= kSlotLevels: internal nodes of level d - kSlotLevels.
// 8 B read + 1 B written per cell.
__global__ void __launch_bounds__(kTopoThreads)
topo_count_kernel(const SortedView sv, i64 n, signed char* __restrict__ clev, u32* __restrict__ hist,
                  i64 nchunks)
{
    chain_enter();
    const u32 lane = lane_id();
    const int warp = threadIdx.x >> 5;
    const i64 chunk = (i64)blockIdx.x * (kTopoThreads / 32) + warp;
    if (chunk >= nchunks) return;                      // whole warp leaves; only warp-level primitives below
    const i64 wbase = chunk * kTopoChunk;
    // c(s) of the chunk's cells: every load is issued before the first use (indices clamped, results
    // masked), so a warp has its whole chunk in flight at once
    int c[kTopoItems];
    int cprev;                                        // c(wbase - 1)
    const i64 last = n - 1;
    if (sv.packed) {
        const u64* w = sv.packed;
        u64 x[kTopoItems];
        if (wbase + kTopoChunk < n) {                  // interior chunk: no clamping (warp-uniform)
            const u64* wp = w + wbase + lane;
            #pragma unroll
            for (int i = 0; i < kTopoItems; ++i) x[i] = (wp[32 * i] ^ wp[32 * i + 1]) >> sv.ib;
        } else {
            #pragma unroll
            for (int i = 0; i < kTopoItems; ++i) {
                const i64 s = wbase + 32 * i + lane;
                const i64 s0 = s < last ? s : last, s1 = s + 1 < last ? s + 1 : last;
                x[i] = (w[s0] ^ w[s1]) >> sv.ib;
            }
        }
        const u64 xp = wbase > 0 ? ((w[wbase - 1] ^ w[wbase]) >> sv.ib) : 0ULL;
        #pragma unroll
        for (int i = 0; i < kTopoItems; ++i) c[i] = window_common_levels(x[i], sv.lo);
        cprev = window_common_levels(xp, sv.lo);
    } else {
        u64 x[kTopoItems];
        #pragma unroll
        for (int i = 0; i < kTopoItems; ++i) {
            const i64 s = wbase + 32 * i + lane;
            const i64 s0 = s < last ? s : last, s1 = s + 1 < last ? s + 1 : last;
            x[i] = sv.keys[s0] ^ sv.keys[s1];
        }
        const u64 xp = wbase > 0 ? (sv.keys[wbase - 1] ^ sv.keys[wbase]) : 0ULL;
        #pragma unroll
        for (int i = 0; i < kTopoItems; ++i) c[i] = x[i] == 0ULL ? kMaxLevel : (__clzll((long long)x[i]) - 1) / 3;
        cprev = xp == 0ULL ? kMaxLevel : (__clzll((long long)xp) - 1) / 3;
    }
    if (wbase == 0) cprev = -1;
    // level masks of the chunk's cells stay in registers; the histogram rows are then one add-reduction
    // per level that occurs in the chunk (a handful), not atomics per cell
    u32 em[kTopoItems], im[kTopoItems];
    u32 ue = 0u;
    if (wbase + kTopoChunk < n) {                      // interior chunk: every cell and its successor exist
        signed char* cl = clev + wbase + lane;
        #pragma unroll
        for (int i = 0; i < kTopoItems; ++i) {
            const int cs = c[i];
            int cp = __shfl_up_sync(0xffffffffu, cs, 1);
            if (lane == 0) cp = cprev;
            cprev = __shfl_sync(0xffffffffu, cs, 31);
            cl[32 * i] = (signed char)cs;
            entity_masks(cp, cs, im[i], em[i]);
            ue |= em[i];
        }
    } else {
        #pragma unroll
        for (int i = 0; i < kTopoItems; ++i) {
            const i64 s = wbase + 32 * i + lane;
            const bool valid = s < n;
            const int cs = (valid && s + 1 < n) ? c[i] : -1;
            int cp = __shfl_up_sync(0xffffffffu, cs, 1);
            if (lane == 0) cp = cprev;
            cprev = __shfl_sync(0xffffffffu, cs, 31);
            em[i] = 0u; im[i] = 0u;
            if (valid) {
                clev[s] = (signed char)cs;
                entity_masks(cp, cs, im[i], em[i]);
            }
            ue |= em[i];
        }
    }
    u32 U = __reduce_or_sync(0xffffffffu, ue);
    u32 myE = 0u, myI = 0u;                            // lane l: entities / internal nodes of level l
    while (U) {
        const int l = __ffs(U) - 1;
        U &= U - 1u;
        u32 v = 0u;                                    // entities in the low half, nodes in the high half (<= 256 each)
        #pragma unroll
        for (int i = 0; i < kTopoItems; ++i) v += ((em[i] >> l) & 1u) + (((im[i] >> l) & 1u) << 16);
        const u32 tot = __reduce_add_sync(0xffffffffu, v);
        if ((int)lane == l) { myE = tot & 0xffffu; myI = tot >> 16; }
    }
    if (lane < (u32)kSlotLevels) hist[(i64)lane * nchunks + chunk] = myE;
    if (lane < (u32)kNumLevels) hist[(i64)(kSlotLevels + lane) * nchunks + chunk] = myI;
}

// row starts of the scanned histogram (+ the grand total) for the host: out[d] = scanned[d * nchunks].
// A build that speculates the level totals (bh_build: the same mesh as last time) has already been told the totals it
// expects: `*gate` = 1 if the rows and the key reduction just computed equal the expected ones, else 0 -- the
// kernels enqueued behind this one on that assumption (assign, moments) return at once when it is 0.
struct TotalsHint {
    u32 rows[kTopoDigits + 1];
    u64 key_or, key_and;
    int check;                       // 0: nothing was speculated, *gate = 0
};
__global__ void topo_totals_kernel(const u32* __restrict__ scanned, i64 nchunks, const u32* __restrict__ total,
                                   u32* __restrict__ out /* [kTopoDigits + 1], pinned host memory */, const TotalsHint hint,
                                   const KeyReduce* __restrict__ red, KeyReduce* __restrict__ red_out /* host, or null */,
                                   u32* __restrict__ gate)
{
    chain_enter();
    const int d = threadIdx.x;
    u32 v = 0u;
    if (d < kTopoDigits) v = scanned[(i64)d * nchunks];
    else if (d == kTopoDigits) v = *total;
    if (d <= kTopoDigits) out[d] = v;          // straight into the host's pinned mirror: no copy on the stream
    bool same = d > kTopoDigits || v == hint.rows[d];
    if (d == 0) {
        const KeyReduce r = *red;
        if (red_out) *red_out = r;
        same = same && r.key_or == hint.key_or && r.key_and == hint.key_and;
    }
    const int all = __syncthreads_and(same);
    if (d == 0) *gate = (hint.check && all) ? 1u : 0u;
}

// ---- a4.2 + a3: number every entity, link the nodes, move every cell into its slot ------------------
// `scanned` = exclusive scan of the count kernel's histogram (row-major over [digit][chunk]), so
// scanned[l][chunk] is the slot of the chunk's first level-l entity and scanned[23 + l][chunk] - nslots
// the canonical id of its first level-l node.  Per cell: 4 B idx + 1 B c + 32 B gathered; written
// 4 B slot + 32 B fp64 record + 16 B fp32 record; per node 12 B.  The aux record of a leaf slot is
// all zero and is NOT written here: the context keeps aux zero everywhere except on the node slots of
// the last build, which aux_clear_kernel resets before the next one.
__global__ void __launch_bounds__(kTopoThreads)
topo_assign_kernel(const signed char* __restrict__ clev, i64 n, const SortedView sv,
                   const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
                   const double* __restrict__ m, const u32* __restrict__ scanned, i64 nchunks, u32 nslots,
                   u32* __restrict__ leaf_slot, u32* __restrict__ node_slot, u32* __restrict__ nfirst,
                   u32* __restrict__ nlo, double4* __restrict__ rec64, float4* __restrict__ rec,
                   const u32* __restrict__ gate /* null, or: run only if *gate != 0 (speculated level totals) */)
{
    chain_enter();
    if (gate && *gate == 0u) return;
    const u32 lane = lane_id();
    const u32 lt = (1u << lane) - 1u;
    const i64 chunk = (i64)blockIdx.x * (kTopoThreads / 32) + (threadIdx.x >> 5);
    if (chunk >= nchunks) return;
    const i64 wbase = chunk * kTopoChunk;
    // lane l: slot of the next level-l entity / canonical id of the next level-l node
    u32 cntT = lane < (u32)kSlotLevels ? scanned[(i64)lane * nchunks + chunk] : 0u;
    u32 cntI = lane < (u32)kNumLevels ? scanned[(i64)(kSlotLevels + lane) * nchunks + chunk] - nslots : 0u;
    int carry = wbase > 0 ? (int)clev[wbase - 1] : -1;
    u32 oi[kTopoItems];                        // the chunk's permutation entries and c(s), fetched up front so
    int ci[kTopoItems];                        // that a row's gathers do not wait behind them
    #pragma unroll
    for (int i = 0; i < kTopoItems; ++i) {
        const i64 s = wbase + 32 * i + lane;
        oi[i] = s < n ? sv_idx(sv, s) : 0u;
        ci[i] = s < n ? (int)clev[s] : -1;
    }
    #pragma unroll
    for (int i = 0; i < kTopoItems; ++i) {
        if (wbase + 32 * i >= n) break;
        const i64 s = wbase + 32 * i + lane;
        const bool valid = s < n;
        double px = 0.0, py = 0.0, pz = 0.0, pm = 0.0;
        const int cs = ci[i];
        if (valid) {
            const u32 o = oi[i];
            px = __ldg(x + o); py = __ldg(y + o); pz = __ldg(z + o); pm = __ldg(m + o);
        }
        int cp = __shfl_up_sync(0xffffffffu, cs, 1);
        if (lane == 0) cp = carry;
        carry = __shfl_sync(0xffffffffu, cs, 31);
        u32 imask = 0u, emask = 0u;
        if (valid) entity_masks(cp, cs, imask, emask);
        u32 U = __reduce_or_sync(0xffffffffu, emask);
        u32 pend = 0xffffffffu, myslot = 0u;
        while (U) {                                   // ascending levels
            const int l = __ffs(U) - 1;
            U &= U - 1u;
            const bool has = (emask >> l) & 1u, isint = (imask >> l) & 1u;
            const u32 bal = __ballot_sync(0xffffffffu, has);
            const u32 balI = __ballot_sync(0xffffffffu, isint);
            const u32 baseT = __shfl_sync(0xffffffffu, cntT, l);
            const u32 baseI = __shfl_sync(0xffffffffu, cntI, l);
            if ((int)lane == l) { cntT += __popc(bal); cntI += __popc(balI); }
            if (has) {
                const u32 slot = baseT + __popc(bal & lt);
                if (pend != 0xffffffffu) nfirst[pend] = slot;       // entity (l, s) is the first child of (l-1, s)
                if (isint) {
                    const u32 b = baseI + __popc(balI & lt);
                    BH_DCHECK(slot < nslots);
                    node_slot[b] = slot;
                    nlo[b] = (u32)s;
                    pend = b;
                } else {
                    myslot = slot;
                    pend = 0xffffffffu;
                }
            }
        }
        if (valid) {
            BH_DCHECK(myslot < nslots && myslot > 0u);
            st_stream(leaf_slot + s, myslot);          // written once, read much later: keep L2 for the gathers
            double2* o64 = reinterpret_cast<double2*>(rec64 + myslot);
            st_stream(o64, make_double2(px, py));
            st_stream(o64 + 1, make_double2(pz, pm));
            st_stream(rec + myslot, make_float4((float)px, (float)py, (float)pz, (float)pm));
        }
    }
}

// aux[node_slot[b]] = 0 for the nodes of the previous build (16 B per node instead of 16 B per slot)
__global__ void __launch_bounds__(256)
aux_clear_kernel(const u32* __restrict__ node_slot, i64 nn, WalkAux* __restrict__ aux)
{
    chain_enter();
    const i64 b = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (b < nn) reinterpret_cast<uint4*>(aux)[node_slot[b]] = make_uint4(0u, 0u, 0u, 0u);
}

// first index in [a, hi) whose key is >= limit (hi if none); gallops from a
__device__ __forceinline__ i64 gallop_lower_bound(const SortedView& sv, i64 a, i64 hi, u64 limit)
{
    if (a >= hi || sv_key(sv, a) >= limit) return a;
    i64 lo = a;                 // keys[lo] < limit
    i64 step = 1;
    while (lo + step < hi && sv_key(sv, lo + step) < limit) { lo += step; step <<= 1; }
    i64 up = lo + step < hi ? lo + step : hi;   // keys[up] >= limit or up == hi
    while (up - lo > 1) {
        const i64 mid = lo + ((up - lo) >> 1);
        if (sv_key(sv, mid) < limit) lo = mid; else up = mid;
    }
    return up;
}

// ---- a5: moments of the nodes [b0, b1) of one level from their children ---------------------------
__device__ __forceinline__ u32 compact3(u64 v)   // inverse of the key bit-spread: every third bit
{
    v &= 0x1249249249249249ULL;
    v = (v | (v >> 2)) & 0x10c30c30c30c30c3ULL;
    v = (v | (v >> 4)) & 0x100f00f00f00f00fULL;
    v = (v | (v >> 8)) & 0x001f0000ff0000ffULL;
    v = (v | (v >> 16)) & 0x001f00000000ffffULL;
    v = (v | (v >> 32)) & 0x1fffffULL;
    return (u32)v;
}

// Node b of level `level`: children = slots [nfirst[b], nfirst[b+1]) (the last node of the level ends at
// slot_end, the end of the level-(level+1) slots).  Reads 32 B per child, writes 80 B per node.
struct MomentArgs {
    SortedView sv; const u32* nlo; const u32* nfirst; const u32* node_slot;
    double4* rec64; double* delta64; float4* rec; WalkAux* aux; u32* max_bucket;
    double x0, y0, z0, L;
    const u32* gate;                 // null, or: run only if *gate != 0 (speculated level totals)
};

__device__ __forceinline__ void moments_node(i64 b, i64 b1, int level, u32 slot_end, const MomentArgs& A)
{
    const u32* nlo = A.nlo; const u32* nfirst = A.nfirst; const u32* node_slot = A.node_slot;
    double4* rec64 = A.rec64; double* delta64 = A.delta64; float4* rec = A.rec; WalkAux* aux = A.aux;
    u32* max_bucket = A.max_bucket;
    const double x0 = A.x0, y0 = A.y0, z0 = A.z0, L = A.L;
    const u32 first = nfirst[b];
    const u32 cnt = (b + 1 < b1 ? nfirst[b + 1] : slot_end) - first;
    BH_DCHECK(cnt >= 1u && first + cnt <= slot_end && (level == kMaxLevel || cnt <= 8u));
    double M = 0.0, Sx = 0.0, Sy = 0.0, Sz = 0.0;
    for (u32 j = 0; j < cnt; ++j) {       // ascending octant order (M-rule 1); no fma contraction
        const double2* p = reinterpret_cast<const double2*>(rec64 + first + j);
        const double2 xy = p[0], zm = p[1];
        M = __dadd_rn(M, zm.y);
        Sx = __dadd_rn(Sx, __dmul_rn(zm.y, xy.x));
        Sy = __dadd_rn(Sy, __dmul_rn(zm.y, xy.y));
        Sz = __dadd_rn(Sz, __dmul_rn(zm.y, zm.x));
    }
    const double size = ldexp(L, -level);
    const u64 prefix = level == 0 ? 0ULL : sv_key(A.sv, nlo[b]) >> (3 * (kMaxLevel - level));
    const double cx = __dadd_rn(x0, __dmul_rn((double)compact3(prefix) + 0.5, size));
    const double cy = __dadd_rn(y0, __dmul_rn((double)compact3(prefix >> 1) + 0.5, size));
    const double cz = __dadd_rn(z0, __dmul_rn((double)compact3(prefix >> 2) + 0.5, size));
    double Rx, Ry, Rz, del;
    if (M != 0.0) {                        // Eq. 5: R = (1/M) sum m_i r_i
        Rx = Sx / M; Ry = Sy / M; Rz = Sz / M;
        const double ex = Rx - cx, ey = Ry - cy, ez = Rz - cz;
        del = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(ex, ex), __dmul_rn(ey, ey)), __dmul_rn(ez, ez)));
    } else {                               // M-rule 2: zero-mass node sits at its geometric centre
        Rx = cx; Ry = cy; Rz = cz; del = 0.0;
    }
    const u32 slot = node_slot[b];
    double2* o = reinterpret_cast<double2*>(rec64 + slot);
    o[0] = make_double2(Rx, Ry);
    o[1] = make_double2(Rz, M);
    delta64[b] = del;
    rec[slot] = make_float4((float)Rx, (float)Ry, (float)Rz, (float)M);
    WalkAux a;
    a.size = level == kMaxLevel ? __int_as_float(0x7f800000) : (float)size;
    a.delta = (float)del;
    a.first = first;
    a.count = cnt;
    aux[slot] = a;
    if (level == kMaxLevel) atomicMax(max_bucket, cnt);
}

__global__ void __launch_bounds__(128)
moments_kernel(i64 b0, i64 b1, int level, u32 slot_end, const MomentArgs A)
{
    chain_enter();
    if (A.gate && *A.gate == 0u) return;
    const i64 b = b0 + (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (b < b1) moments_node(b, b1, level, slot_end, A);
}

// a run of small levels (deepest first) in ONE block: a level's nodes are complete before the next starts
constexpr int kSmallLevelNodes = 512;
constexpr int kMomSmallThreads = 512;
struct SmallLevels {
    int nlev;
    int level[kNumLevels];
    u32 b0[kNumLevels], b1[kNumLevels], slot_end[kNumLevels];
};

__global__ void __launch_bounds__(kMomSmallThreads)
moments_small_kernel(const SmallLevels sl, const MomentArgs A)
{
    chain_enter();
    if (A.gate && *A.gate == 0u) return;
    for (int k = 0; k < sl.nlev; ++k) {
        for (i64 b = (i64)sl.b0[k] + threadIdx.x; b < (i64)sl.b1[k]; b += kMomSmallThreads)
            moments_node(b, sl.b1[k], sl.level[k], sl.slot_end[k], A);
        __threadfence_block();
        __syncthreads();
    }
}

struct TopoLevels {               // host-computed from the scanned histogram
    u32 node_base[kNumLevels + 1];    // canonical id of the first node of each level; [22] = n_nodes
    u32 slot_base[kSlotLevels + 1];   // first slot of each entity level; [23] = n_slots
};

// ---- export (parity only): the nodes in canonical order ------------------------------------------
__global__ void __launch_bounds__(256)
export_nodes_kernel(i64 nn, i64 n, const TopoLevels lv, const SortedView sv, const u32* __restrict__ nlo,
                    const u32* __restrict__ nfirst, const u32* __restrict__ node_slot,
                    const double4* __restrict__ rec64, const double* __restrict__ delta64,
                    int* level, u64* prefix, i64* lo, i64* hi, int* nch, double* M, double* Rx, double* Ry,
                    double* Rz, double* delta)
{
    const i64 b = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nn) return;
    int l = 0;
    while (l + 1 < kNumLevels && (i64)lv.node_base[l + 1] <= b) ++l;
    const i64 s = nlo[b];
    if (level) level[b] = l;
    if (prefix) prefix[b] = l == 0 ? 0ULL : sv_key(sv, s) >> (3 * (kMaxLevel - l));
    if (lo) lo[b] = s;
    if (hi) {
        if (l == 0) hi[b] = n;
        else {
            const int sh = 3 * (kMaxLevel - l);
            hi[b] = gallop_lower_bound(sv, s + 1, n, ((sv_key(sv, s) >> sh) + 1ULL) << sh);
        }
    }
    if (nch) nch[b] = (int)((b + 1 < (i64)lv.node_base[l + 1] ? nfirst[b + 1] : lv.slot_base[l + 2]) - nfirst[b]);
    const double4 q = rec64[node_slot[b]];
    if (Rx) Rx[b] = q.x;
    if (Ry) Ry[b] = q.y;
    if (Rz) Rz[b] = q.z;
    if (M) M[b] = q.w;
    if (delta) delta[b] = delta64[b];
}

// ---- bh_potential_direct's own copies (built on its first call after a build, not on the hot path) --
__global__ void __launch_bounds__(256)
direct_prepare_kernel(const SortedView sv, const u32* __restrict__ leaf_slot,
                      const double4* __restrict__ rec64, i64 n, double4* __restrict__ leaf64,
                      u32* __restrict__ slot_of)
{
    const i64 s = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    leaf64[s] = rec64[leaf_slot[s]];
    slot_of[sv_idx(sv, s)] = (u32)s;
}

// ---- bh_update_masses: new masses for the cells of the last build (positions, and so the tree, unchanged) ----
// 8 B gathered per cell; the mass fields of its fp64 and fp32 slot records are rewritten.
__global__ void __launch_bounds__(256)
mass_update_kernel(const SortedView sv, const u32* __restrict__ leaf_slot, const double* __restrict__ m, i64 n,
                   double4* __restrict__ rec64, float4* __restrict__ rec)
{
    const i64 s = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const double pm = __ldg(m + sv_idx(sv, s));
    const u32 slot = leaf_slot[s];
    rec64[slot].w = pm;
    rec[slot].w = (float)pm;
}

// sorted keys and permutation as plain arrays (bh_export_tree)
__global__ void __launch_bounds__(256)
export_sorted_kernel(const SortedView sv, i64 n, u64* __restrict__ keys, u32* __restrict__ perm)
{
    const i64 s = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    if (keys) keys[s] = sv_key(sv, s);
    if (perm) perm[s] = sv_idx(sv, s);
}

}  // namespace bh
