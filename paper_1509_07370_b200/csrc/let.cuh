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
// copied to the host: the records are compacted on the device (count -> scan -> gather) in ascending
// slot order = ascending (level, first sorted cell), ready to be handed to the exchange.
#pragma once
#include "common.cuh"
#include "scan.cuh"
#include "tree.cuh"

namespace bh {

struct EssArgs {
    const u32* nfirst; const u32* node_slot; const double4* rec64; const double* delta64; const WalkAux* aux;
    unsigned char* state;     // per slot: 1 = reached internal node (to be tested at its level), 2 = essential
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
    if (accept) { A.state[slot] = 2; return; }
    const u32 first = A.nfirst[b];
    const u32 cnt = (b + 1 < b1 ? A.nfirst[b + 1] : slot_end) - first;
    for (u32 j = 0; j < cnt; ++j) {
        const u32 c = first + j;
        A.state[c] = A.aux[c].count > 0u ? 1 : 2;     // internal child: tested when its level runs; leaf cell: essential
    }
}

__global__ void __launch_bounds__(256)
ess_level_kernel(i64 b0, i64 b1, int level, u32 slot_end, const EssArgs A)
{
    chain_enter();
    const i64 b = b0 + (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (b < b1) ess_node(b, b1, level, slot_end, A);
}

// a run of small levels, root side first, in ONE block (a level is complete before the next starts)
constexpr int kEssSmallNodes = 1024;
__global__ void __launch_bounds__(1024)
ess_small_kernel(const SmallLevels sl, const EssArgs A)
{
    chain_enter();
    for (int k = 0; k < sl.nlev; ++k) {
        for (i64 b = (i64)sl.b0[k] + threadIdx.x; b < (i64)sl.b1[k]; b += blockDim.x)
            ess_node(b, sl.b1[k], sl.level[k], sl.slot_end[k], A);
        __threadfence_block();
        __syncthreads();
    }
}

// ---- compaction of the essential slots, in slot order -------------------------------------------------
// A block owns kEssTile consecutive slots, a thread 16 of them (one 16-byte load of state bytes).
// ess_count_kernel: essential slots per block; (device scan of the block counts); ess_gather_kernel:
// out[4k..4k+3] = (x, y, z, m) of the k-th essential slot.  19 MB of flags are read twice at 16.8 M cells.
constexpr int kEssThreads = 256;
constexpr int kEssTile = kEssThreads * 16;

__device__ __forceinline__ uint4 ess_load_flags(const unsigned char* state, i64 s0, i64 nslots)
{
    if (s0 + 16 <= nslots) return *reinterpret_cast<const uint4*>(state + s0);
    unsigned char b[16];
    #pragma unroll
    for (int i = 0; i < 16; ++i) b[i] = s0 + i < nslots ? state[s0 + i] : 0;
    uint4 v;
    memcpy(&v, b, 16);
    return v;
}
__device__ __forceinline__ u32 ess_twos(u32 w) { return (w >> 1) & 0x01010101u; }   // bytes are 0, 1 or 2

__global__ void __launch_bounds__(kEssThreads)
ess_count_kernel(const unsigned char* __restrict__ state, i64 nslots, u32* __restrict__ block_count)
{
    chain_enter();
    __shared__ u32 s_warp[9];
    const i64 s0 = ((i64)blockIdx.x * kEssThreads + threadIdx.x) * 16;
    const uint4 v = ess_load_flags(state, s0, nslots);
    const u32 c = __popc(ess_twos(v.x)) + __popc(ess_twos(v.y)) + __popc(ess_twos(v.z)) + __popc(ess_twos(v.w));
    u32 total;
    block_excl_scan_256(c, total, s_warp);
    if (threadIdx.x == 0) block_count[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kEssThreads)
ess_gather_kernel(const unsigned char* __restrict__ state, i64 nslots, const u32* __restrict__ block_base,
                  const double4* __restrict__ rec64, double* __restrict__ out, i64 cap)
{
    chain_enter();
    __shared__ u32 s_warp[9];
    const i64 s0 = ((i64)blockIdx.x * kEssThreads + threadIdx.x) * 16;
    const uint4 v = ess_load_flags(state, s0, nslots);
    const u32 w[4] = {ess_twos(v.x), ess_twos(v.y), ess_twos(v.z), ess_twos(v.w)};
    const u32 c = __popc(w[0]) + __popc(w[1]) + __popc(w[2]) + __popc(w[3]);
    u32 total;
    i64 p = (i64)block_base[blockIdx.x] + block_excl_scan_256(c, total, s_warp);
    if (c == 0u) return;
    #pragma unroll
    for (int i = 0; i < 16; ++i) {
        if ((w[i >> 2] >> (8 * (i & 3))) & 1u) {
            if (p < cap) {
                const double2* q = reinterpret_cast<const double2*>(rec64 + s0 + i);
                double2* o = reinterpret_cast<double2*>(out + 4 * p);
                o[0] = q[0];
                o[1] = q[1];
            }
            ++p;
        }
    }
}

}  // namespace bh
