// let.cuh -- Find Essential Nodes (§3.2.4, Fig. 7).
// The tree of the last build pruned against a remote domain, the axis-aligned box [blo, bhi]
// (E1-E4): d_c = distance from a node's centre of mass to the nearest point of the box; an
// internal node with d_c > l/theta (+ delta under Eq. 4) is essential and is sent as ONE point mass
// (R, M); otherwise it is opened; a leaf cell under an opened node is essential as it is; a level-21
// bucket is always opened.  Decisions in fp64 on the fp64 moments, products and sums rounded
// separately (the oracle's expression), so the selected set is identical, not merely close.
//
// Like the paper's kernel it runs level by level from the root ("called once for each depth ...
// Neither atomic operations nor direct synchronization calls are used"), one thread per node of the
// level; unlike it, levels of <= 1024 nodes share one single-block launch, and the index list is not
// copied to the host: the records are compacted on the device (flag -> scan -> gather) in ascending
// slot order = ascending (level, first sorted cell), ready to be handed to the exchange.
#pragma once
#include "common.cuh"
#include "tree.cuh"

namespace bh {

struct EssArgs {
    const u32* nfirst; const u32* node_slot; const double4* rec64; const double* delta64; const WalkAux* aux;
    unsigned char* state;     // per slot: 1 = reached internal node (to be tested at its level)
    u32* emit;                // per slot: 1 = essential
    double blo[3], bhi[3];
    double theta, L;
    int mac;
};

__device__ __forceinline__ double ess_axis_dist(double r, double lo, double hi)
{
    return r < lo ? __dsub_rn(lo, r) : (r > hi ? __dsub_rn(r, hi) : 0.0);
}

// node b (canonical id) of `level`; its children are the slots [nfirst[b], nfirst[b+1]) (slot_end for the
// last node of the level)
__device__ __forceinline__ void ess_node(i64 b, i64 b1, int level, u32 slot_end, const EssArgs& A)
{
    const u32 slot = A.node_slot[b];
    if (A.state[slot] != 1) return;
    bool accept = false;
    if (level < kMaxLevel && A.theta > 0.0) {
        const double4 q = A.rec64[slot];
        double rc = ldexp(A.L, -level) / A.theta;
        if (A.mac == 1) rc = __dadd_rn(rc, A.delta64[b]);
        const double dx = ess_axis_dist(q.x, A.blo[0], A.bhi[0]);
        const double dy = ess_axis_dist(q.y, A.blo[1], A.bhi[1]);
        const double dz = ess_axis_dist(q.z, A.blo[2], A.bhi[2]);
        const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
        accept = d2 > __dmul_rn(rc, rc);
    }
    if (accept) { A.emit[slot] = 1u; return; }
    const u32 first = A.nfirst[b];
    const u32 cnt = (b + 1 < b1 ? A.nfirst[b + 1] : slot_end) - first;
    for (u32 j = 0; j < cnt; ++j) {
        const u32 c = first + j;
        if (A.aux[c].count > 0u) A.state[c] = 1;      // internal child: tested when its level runs
        else A.emit[c] = 1u;                          // leaf cell
    }
}

__global__ void __launch_bounds__(256)
ess_level_kernel(i64 b0, i64 b1, int level, u32 slot_end, const EssArgs A)
{
    const i64 b = b0 + (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (b < b1) ess_node(b, b1, level, slot_end, A);
}

// a run of small levels, root side first, in ONE block (a level is complete before the next starts)
constexpr int kEssSmallNodes = 1024;
__global__ void __launch_bounds__(1024)
ess_small_kernel(const SmallLevels sl, const EssArgs A)
{
    for (int k = 0; k < sl.nlev; ++k) {
        for (i64 b = (i64)sl.b0[k] + threadIdx.x; b < (i64)sl.b1[k]; b += blockDim.x)
            ess_node(b, sl.b1[k], sl.level[k], sl.slot_end[k], A);
        __threadfence_block();
        __syncthreads();
    }
}

// out[4k..4k+3] = (x, y, z, m) of the k-th essential slot; pos = exclusive scan of emit
__global__ void __launch_bounds__(256)
ess_gather_kernel(const u32* __restrict__ pos, i64 nslots, const u32* __restrict__ total_p,
                  const double4* __restrict__ rec64, double* __restrict__ out, i64 cap)
{
    const i64 s = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= nslots) return;
    const u32 p = pos[s];
    const u32 nxt = s + 1 < nslots ? pos[s + 1] : *total_p;
    if (nxt != p && (i64)p < cap) {
        const double2* q = reinterpret_cast<const double2*>(rec64 + s);
        double2* o = reinterpret_cast<double2*>(out + 4 * (i64)p);
        o[0] = q[0];
        o[1] = q[1];
    }
}

}  // namespace bh
