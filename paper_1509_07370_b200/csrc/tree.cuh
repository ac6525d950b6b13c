// tree.cuh -- steps a3 (permute), a4 (octree topology from sorted keys) and a5 (monopole moments).
//
// The tree is the one PAPER.md:45 (§2) defines -- the cube "is recursively divided into eight sub
// cells ... until only one particle is left for every sub cell" -- under DESIGN.md T1-T5:
// a node is (level l, prefix = key >> 3(21-l)) and owns the contiguous sorted range of cells that
// share the prefix; ranges of >= 2 cells are internal nodes (single-child chains kept), one cell is
// a leaf cell, >= 2 cells with identical keys form a level-21 bucket.
//
// Construction (no locks, no spinning, unlike the paper's insertion kernel PAPER.md:146-150):
//   c(s) = number of octree levels keys s and s+1 share.  A node of level l starts at sorted slot
//   s iff c(s-1) < l <= c(s); so slot s starts max(0, c(s) - c(s-1)) nodes, and an exclusive scan
//   numbers all nodes in depth-first pre-order.  A stable counting sort by level (one radix pass)
//   turns that into breadth-first = canonical (level, prefix) order.  Per node, the end of its
//   range and its <= 8 child ranges are found by galloping searches in the sorted keys.  Children
//   of consecutive nodes get consecutive "slots" in the walk arrays (root = slot 0), so the <= 8
//   children of a node are one contiguous run of records.
// Moments (Eq. 5; delta PAPER.md:54, 158) are reduced level by level from the
// deepest level up, each node from its children in ascending octant order in fp64 (M-rules).
#pragma once
#include "common.cuh"

namespace bh {

constexpr int kNumLevels = kMaxLevel + 1;   // levels 0..21

struct __align__(16) WalkAux {   // per slot, beside the float4 record (x, y, z, m)
    float size;      // node edge l (fp32 of L/2^level); +inf for a level-21 bucket; 0 for a leaf cell
    float delta;     // |R - geometric centre| (fp32)
    u32 first;       // slot of the first child
    u32 count;       // number of children (0: this slot is a leaf cell)
};

// ---- a3: permute the cells into sorted order ---------------------------------------------------
// leaf64[s] = (x, y, z, m) fp64 of the cell in sorted slot s; leafrec[s] the same rounded to fp32;
// slot_of[i] = sorted slot of original cell i.   84 B algorithmic per cell (+4 B slot_of).
__global__ void __launch_bounds__(256)
permute_kernel(const u32* __restrict__ idx, const double* __restrict__ x, const double* __restrict__ y,
               const double* __restrict__ z, const double* __restrict__ m, i64 n,
               double4* __restrict__ leaf64, float4* __restrict__ leafrec, u32* __restrict__ slot_of)
{
    const i64 s = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const u32 i = ld_stream(idx + s);
    const double px = __ldg(x + i), py = __ldg(y + i), pz = __ldg(z + i), pm = __ldg(m + i);
    double2* o = reinterpret_cast<double2*>(leaf64 + s);
    st_stream(o, make_double2(px, py));
    st_stream(o + 1, make_double2(pz, pm));
    leafrec[s] = make_float4((float)px, (float)py, (float)pz, (float)pm);
    slot_of[i] = (u32)s;
}

// ---- a4.1: nodes starting at each sorted slot + per-level histogram ----------------------------
__global__ void __launch_bounds__(256)
node_count_kernel(const u64* __restrict__ keys, i64 n, u32* __restrict__ cnt, signed char* __restrict__ clev,
                  u32* __restrict__ level_hist /* [kNumLevels] */)
{
    __shared__ u32 h[kNumLevels];
    if (threadIdx.x < kNumLevels) h[threadIdx.x] = 0;
    __syncthreads();
    const i64 stride = (i64)gridDim.x * blockDim.x;
    for (i64 s = (i64)blockIdx.x * blockDim.x + threadIdx.x; s < n; s += stride) {
        const u64 k = keys[s];
        const int cprev = s > 0 ? common_levels(keys[s - 1], k) : -1;
        const int cs = s + 1 < n ? common_levels(k, keys[s + 1]) : -1;
        clev[s] = (signed char)cs;
        const int c = cs > cprev ? cs - cprev : 0;
        cnt[s] = (u32)c;
        for (int l = cprev + 1; l <= cs; ++l) atomicAdd(&h[l], 1u);
    }
    __syncthreads();
    if (threadIdx.x < kNumLevels && h[threadIdx.x]) atomicAdd(&level_hist[threadIdx.x], h[threadIdx.x]);
}

// ---- a4.2: emit the nodes in pre-order: (level as sort key, pre-order id as payload, lo) ---------
__global__ void __launch_bounds__(256)
node_emit_kernel(const signed char* __restrict__ clev, const u32* __restrict__ pre_base, i64 n,
                 u64* __restrict__ nkey, u32* __restrict__ npre, u32* __restrict__ nlo)
{
    const i64 s = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const int cs = clev[s];
    const int cprev = s > 0 ? (int)clev[s - 1] : -1;
    if (cs <= cprev) return;
    u32 p = pre_base[s];
    for (int l = cprev + 1; l <= cs; ++l, ++p) {
        nkey[p] = (u64)l;
        npre[p] = p;
        nlo[p] = (u32)s;
    }
}

// first index in [a, hi) whose key is >= limit (hi if none); gallops from a (ranges are short on average)
__device__ __forceinline__ i64 gallop_lower_bound(const u64* __restrict__ keys, i64 a, i64 hi, u64 limit)
{
    if (a >= hi || keys[a] >= limit) return a;
    i64 lo = a;                 // keys[lo] < limit
    i64 step = 1;
    while (lo + step < hi && keys[lo + step] < limit) { lo += step; step <<= 1; }
    i64 up = lo + step < hi ? lo + step : hi;   // keys[up] >= limit or up == hi
    while (up - lo > 1) {
        const i64 mid = lo + ((up - lo) >> 1);
        if (keys[mid] < limit) lo = mid; else up = mid;
    }
    return up;
}

// ---- a4.3: per node (canonical order b): range end, child boundaries, child count ---------------
__global__ void __launch_bounds__(256)
node_children_kernel(const u64* __restrict__ keys, i64 n, const u64* __restrict__ bkey,
                     const u32* __restrict__ bpre, const u32* __restrict__ nlo, i64 nn,
                     u32* __restrict__ bfs_of, u32* __restrict__ blo, u32* __restrict__ bhi,
                     u32* __restrict__ nchild, u32* __restrict__ cstart /* [8*nn] */,
                     u32* __restrict__ max_bucket)
{
    const i64 b = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nn) return;
    const int level = (int)bkey[b];
    const u32 p = bpre[b];
    const i64 lo = nlo[p];
    bfs_of[p] = (u32)b;
    i64 hi;
    if (level == 0) hi = n;
    else {
        const int sh = 3 * (kMaxLevel - level);
        const u64 limit = ((keys[lo] >> sh) + 1ULL) << sh;
        hi = gallop_lower_bound(keys, lo + 1, n, limit);
    }
    blo[b] = (u32)lo;
    bhi[b] = (u32)hi;
    if (level == kMaxLevel) {             // bucket: its cells are its children
        nchild[b] = (u32)(hi - lo);
        atomicMax(max_bucket, (u32)(hi - lo));
        return;
    }
    const int sh1 = 3 * (kMaxLevel - level - 1);
    int j = 0;
    i64 a = lo;
    while (a < hi) {
        cstart[8 * b + j] = (u32)a;
        ++j;
        const u64 limit = ((keys[a] >> sh1) + 1ULL) << sh1;
        a = gallop_lower_bound(keys, a + 1, hi, limit);
    }
    nchild[b] = (u32)j;
}

// ---- a4.4: fill the slots: leaf-cell records, links to internal children --------------------------
// 8 threads per node.  slot_src[slot] >= 0: sorted cell index;  < 0: ~(canonical id of the internal child)
__global__ void __launch_bounds__(256)
slot_fill_kernel(const u64* __restrict__ bkey, const u32* __restrict__ bpre, const u32* __restrict__ blo,
                 const u32* __restrict__ bhi, const u32* __restrict__ nchild, const u32* __restrict__ cstart,
                 const u32* __restrict__ child_base, const u32* __restrict__ pre_base,
                 const u32* __restrict__ bfs_of, i64 nn, const float4* __restrict__ leafrec,
                 int* __restrict__ slot_src, u32* __restrict__ node_slot, float4* __restrict__ rec,
                 WalkAux* __restrict__ aux)
{
    const i64 t = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    const i64 b = t >> 3;
    const int j0 = (int)(t & 7);
    if (b >= nn) return;
    const int level = (int)bkey[b];
    const u32 cnt = nchild[b];
    const u32 first = 1u + child_base[b];
    const u32 lo = blo[b], hi = bhi[b];
    if (b == 0 && j0 == 0) node_slot[0] = 0u;          // root record lives in slot 0
    WalkAux leaf_aux; leaf_aux.size = 0.f; leaf_aux.delta = 0.f; leaf_aux.first = 0u; leaf_aux.count = 0u;
    if (level == kMaxLevel) {
        for (u32 j = j0; j < cnt; j += 8) {
            const u32 a = lo + j, slot = first + j;
            slot_src[slot] = (int)a;
            rec[slot] = leafrec[a];
            aux[slot] = leaf_aux;
        }
        return;
    }
    if ((u32)j0 >= cnt) return;
    const u32 a = cstart[8 * b + j0];
    const u32 e = (u32)j0 + 1 < cnt ? cstart[8 * b + j0 + 1] : hi;
    const u32 slot = first + j0;
    if (e - a == 1) {
        slot_src[slot] = (int)a;
        rec[slot] = leafrec[a];
        aux[slot] = leaf_aux;
    } else {
        // pre-order id of the child node (level+1, a): this node's id + 1 if it starts at lo, else
        // the first node starting at a (there c(a-1) == level exactly)
        const u32 pre = (a == lo) ? bpre[b] + 1u : pre_base[a];
        const u32 cb = bfs_of[pre];
        slot_src[slot] = ~(int)cb;
        node_slot[cb] = slot;
    }
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

__global__ void __launch_bounds__(128)
moments_kernel(i64 b0, i64 b1, int level, const u64* __restrict__ keys, const u32* __restrict__ blo,
               const u32* __restrict__ nchild, const u32* __restrict__ child_base,
               const int* __restrict__ slot_src, const u32* __restrict__ node_slot,
               const double4* __restrict__ leaf64, double4* __restrict__ mom, double* __restrict__ delta64,
               float4* __restrict__ rec, WalkAux* __restrict__ aux, double x0, double y0, double z0, double L)
{
    const i64 b = b0 + (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= b1) return;
    const u32 cnt = nchild[b];
    const u32 first = 1u + child_base[b];
    double M = 0.0, Sx = 0.0, Sy = 0.0, Sz = 0.0;
    for (u32 j = 0; j < cnt; ++j) {       // ascending octant order (M-rule 1); no fma contraction
        const int src = slot_src[first + j];
        const double2* p = reinterpret_cast<const double2*>(src >= 0 ? leaf64 + src : mom + (~src));
        const double2 xy = p[0], zm = p[1];
        M = __dadd_rn(M, zm.y);
        Sx = __dadd_rn(Sx, __dmul_rn(zm.y, xy.x));
        Sy = __dadd_rn(Sy, __dmul_rn(zm.y, xy.y));
        Sz = __dadd_rn(Sz, __dmul_rn(zm.y, zm.x));
    }
    const double size = ldexp(L, -level);
    const u64 prefix = level == 0 ? 0ULL : keys[blo[b]] >> (3 * (kMaxLevel - level));
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
    double2* o = reinterpret_cast<double2*>(mom + b);
    o[0] = make_double2(Rx, Ry);
    o[1] = make_double2(Rz, M);
    delta64[b] = del;
    const u32 slot = node_slot[b];
    rec[slot] = make_float4((float)Rx, (float)Ry, (float)Rz, (float)M);
    WalkAux a;
    a.size = level == kMaxLevel ? __int_as_float(0x7f800000) : (float)size;
    a.delta = (float)del;
    a.first = first;
    a.count = cnt;
    aux[slot] = a;
}

// ---- export (parity only): prefix of each node in canonical order --------------------------------
__global__ void __launch_bounds__(256)
export_nodes_kernel(i64 nn, const u64* __restrict__ keys, const u64* __restrict__ bkey,
                    const u32* __restrict__ blo, const u32* __restrict__ bhi, const u32* __restrict__ nchild,
                    const double4* __restrict__ mom, const double* __restrict__ delta64,
                    int* level, u64* prefix, i64* lo, i64* hi, int* nch, double* M, double* Rx, double* Ry,
                    double* Rz, double* delta)
{
    const i64 b = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nn) return;
    const int l = (int)bkey[b];
    if (level) level[b] = l;
    if (prefix) prefix[b] = l == 0 ? 0ULL : keys[blo[b]] >> (3 * (kMaxLevel - l));
    if (lo) lo[b] = blo[b];
    if (hi) hi[b] = bhi[b];
    if (nch) nch[b] = (int)nchild[b];
    const double4 q = mom[b];
    if (Rx) Rx[b] = q.x;
    if (Ry) Ry[b] = q.y;
    if (Rz) Rz[b] = q.z;
    if (M) M[b] = q.w;
    if (delta) delta[b] = delta64[b];
}

}  // namespace bh
