// walk.cuh -- steps a6 + a7: the group tree walk (§3.3) and the scatter of Phi.
//
// What is kept from the paper's kernel: one warp owns 32 neighbouring (Morton-consecutive) target
// cells; the traversal stack lives in shared memory and is shared by the warp; a node is used only
// if EVERY lane accepts it (the all() vote), otherwise the whole warp opens it;
// potentials are accumulated in registers.
// What differs (the paper's design is for a Fermi C2075, where lane 0 alone walks the tree):
//  * The traversal is lane-parallel: each step pops up to 4 opened nodes and tests their <= 32
//    children at once, one child per lane.  The vote of DESIGN.md W2 ("all members pass
//    d^2 > r_c^2") is decided without touching the members whenever the group's bounding box
//    proves it: fp32 rounding is monotone, so the fp32 d^2 evaluated at the box's nearest (farthest)
//    point bounds every member's fp32 d^2 from below (above).  Only nodes between the two bounds
//    take the per-member test + __all_sync vote.
//  * Accepted nodes and leaf cells are appended to two interaction lists in shared memory, stored
//    as pairs (x0,x1,y0,y1 | z0,z1,m0,m1), and evaluated with lane = target using packed
//    fp32x2 arithmetic (FADD2/FMUL2/FFMA2, sm_100) and one MUFU.RSQ per interaction.
//  * Partial sums are fp32 over one list flush (<= 128 entries, 4 accumulators) and are flushed
//    into an fp64 sum per target, which keeps the summation error near 1e-7 relative.
//  * Phi is written straight to the original cell order (step a7 is fused: no extra pass).
// ALU-bound: 13 flops per interaction by the north-star convention; MUFU (16 rsqrt/clk/SM) is the
// co-limiter.
#pragma once
#include "common.cuh"
#include "tree.cuh"

namespace bh {

constexpr int kWalkWarps = 8;                 // warps (= groups) per CTA
constexpr int kListCap = 128;                 // entries per interaction list (per warp)
constexpr int kListFlushAt = kListCap - 32;   // a traversal step appends <= 32 entries
constexpr int kStackPerLevel = 36;            // stack entries a level can leave behind (<= 3 + 32)

struct WalkParams {
    const float4* rec;        // [n_slots] (x, y, z, m) of every node / leaf-cell slot
    const WalkAux* aux;       // [n_slots]
    const float4* leafrec;    // [n] sorted cells (targets)
    const u32* idx;           // [n] original index of sorted slot
    double* phi;              // [n] original order
    uint4* gcount;            // [ngroups] {accepted, leaf, opened, exact-tested}
    i64 n;
    i64 ngroups;
    float inv_theta;          // (float)(1/theta); +inf for theta = 0
    int mac;                  // BH_MAC_*
    double negG;
    int stack_cap;            // entries per warp
};

__host__ __device__ inline size_t walk_smem_per_warp(int stack_cap)
{
    return (size_t)stack_cap * sizeof(uint2) + 2 * (size_t)kListCap * 16;
}

__device__ __forceinline__ float rsqrt_approx(float v)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
    return r;
}

// Evaluates `cnt` list entries for this lane's target.  List layout per PAIR p (8 floats):
// x[2p], x[2p+1], y[2p], y[2p+1], z[2p], z[2p+1], m[2p], m[2p+1].  The list is padded to a multiple
// of 4 entries with zero-mass far-away dummies by the caller.  CHECKED: skip pairs at zero distance
// (the target's own cell and coincident cells, W3).
template <bool CHECKED>
__device__ __forceinline__ double eval_list(const float* __restrict__ list, int cnt, float2 npx, float2 npy,
                                            float2 npz)
{
    float2 s0 = make_float2(0.f, 0.f), s1 = make_float2(0.f, 0.f);
    const int nquads = (cnt + 3) >> 2;
    const float4* L4 = reinterpret_cast<const float4*>(list);
    #pragma unroll 2
    for (int q = 0; q < nquads; ++q) {
        const float4 a0 = L4[4 * q + 0], b0 = L4[4 * q + 1];
        const float4 a1 = L4[4 * q + 2], b1 = L4[4 * q + 3];
        float2 dx0 = __fadd2_rn(make_float2(a0.x, a0.y), npx);
        float2 dy0 = __fadd2_rn(make_float2(a0.z, a0.w), npy);
        float2 dz0 = __fadd2_rn(make_float2(b0.x, b0.y), npz);
        float2 dx1 = __fadd2_rn(make_float2(a1.x, a1.y), npx);
        float2 dy1 = __fadd2_rn(make_float2(a1.z, a1.w), npy);
        float2 dz1 = __fadd2_rn(make_float2(b1.x, b1.y), npz);
        float2 d0 = __fmul2_rn(dx0, dx0);
        float2 d1 = __fmul2_rn(dx1, dx1);
        d0 = __ffma2_rn(dy0, dy0, d0);
        d1 = __ffma2_rn(dy1, dy1, d1);
        d0 = __ffma2_rn(dz0, dz0, d0);
        d1 = __ffma2_rn(dz1, dz1, d1);
        float2 r0 = make_float2(rsqrt_approx(d0.x), rsqrt_approx(d0.y));
        float2 r1 = make_float2(rsqrt_approx(d1.x), rsqrt_approx(d1.y));
        if (CHECKED) {
            r0.x = d0.x >= 1.17549435e-38f ? r0.x : 0.f;
            r0.y = d0.y >= 1.17549435e-38f ? r0.y : 0.f;
            r1.x = d1.x >= 1.17549435e-38f ? r1.x : 0.f;
            r1.y = d1.y >= 1.17549435e-38f ? r1.y : 0.f;
        }
        s0 = __ffma2_rn(make_float2(b0.z, b0.w), r0, s0);
        s1 = __ffma2_rn(make_float2(b1.z, b1.w), r1, s1);
    }
    return ((double)s0.x + (double)s0.y) + ((double)s1.x + (double)s1.y);
}

__device__ __forceinline__ void list_store(float* list, int e, float4 r)
{
    float* p = list + (e >> 1) * 8 + (e & 1);
    p[0] = r.x; p[2] = r.y; p[4] = r.z; p[6] = r.w;
}

// pads [cnt, roundup4(cnt)) with zero-mass entries far away (finite d^2, no NaN)
__device__ __forceinline__ void list_pad(float* list, int cnt)
{
    const int e = cnt + (int)lane_id();
    if (e < ((cnt + 3) & ~3)) list_store(list, e, make_float4(3.0e18f, 3.0e18f, 3.0e18f, 0.f));
}

__device__ __forceinline__ float warp_min(float v)
{
    #pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}
__device__ __forceinline__ float warp_max(float v)
{
    #pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
    return v;
}

__global__ void __launch_bounds__(kWalkWarps * 32)
walk_group32_kernel(const WalkParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5;
    const u32 lane = lane_id();
    const i64 g = (i64)blockIdx.x * kWalkWarps + warp;
    if (g >= P.ngroups) return;                       // whole warp leaves; no block-level sync below

    unsigned char* my = smem_raw + (size_t)warp * walk_smem_per_warp(P.stack_cap);
    float* nlist = reinterpret_cast<float*>(my);                       // accepted internal nodes
    float* llist = nlist + kListCap * 4;                               // leaf cells
    uint2* stack = reinterpret_cast<uint2*>(llist + kListCap * 4);     // (first child slot, count)

    // ---- the 32 targets of this group (W-rule 1): sorted slots [32g, 32g+32) ----
    const i64 s = g * 32 + lane;
    const int nt = (int)min((i64)32, P.n - g * 32);
    const bool live = (int)lane < nt;
    const float4 tp = __ldg(P.leafrec + (live ? s : g * 32));
    const float px = tp.x, py = tp.y, pz = tp.z;
    // bounding box of the live targets
    const float bxl = warp_min(px), bxh = warp_max(px);
    const float byl = warp_min(py), byh = warp_max(py);
    const float bzl = warp_min(pz), bzh = warp_max(pz);
    const float2 npx = make_float2(-px, -px), npy = make_float2(-py, -py), npz = make_float2(-pz, -pz);

    double acc = 0.0;
    int n_node = 0, n_leaf = 0;                 // list fill (warp-uniform)
    u32 c_acc = 0, c_leaf = 0, c_open = 0, c_exact = 0;
    int sp = 0;
    if (P.n >= 2) {                             // root is tested like any other node (W-rule 2)
        if (lane == 0) stack[0] = make_uint2(0u, 1u);
        sp = 1;
    }
    __syncwarp();

    const u32 lt = lanemask_lt();
    const int sub = lane >> 3, j = lane & 7;
    while (sp > 0) {
        // ---- pop up to 4 opened nodes; lane (sub, j) takes child j of entry sub ----
        int npop = sp < 4 ? sp : 4;
        uint2 e = make_uint2(0u, 0u);
        if (sub < npop) e = stack[sp - 1 - sub];
        u32 jj = (u32)j;
        if (__any_sync(0xffffffffu, e.y > 8u)) {
            // rare: a bucket of > 8 coincident cells is near the top; serve the top entry alone,
            // 32 children per step, shrinking it in place while more than 32 remain
            e = stack[sp - 1];
            jj = lane;
            npop = 1;
            __syncwarp();
            if (e.y > 32u) {
                if (lane == 0) stack[sp - 1] = make_uint2(e.x + 32u, e.y - 32u);
                e.y = 32u;
                npop = 0;
            }
        }
        sp -= npop;
        __syncwarp();
        const bool have = jj < e.y;
        const u32 slot = e.x + jj;
        float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
        WalkAux a; a.size = 0.f; a.delta = 0.f; a.first = 0u; a.count = 0u;
        if (have) {
            r = __ldg(P.rec + slot);
            const uint4 t = __ldg(reinterpret_cast<const uint4*>(P.aux + slot));
            a.size = __uint_as_float(t.x); a.delta = __uint_as_float(t.y); a.first = t.z; a.count = t.w;
        }
        const bool internal = have && a.count > 0u;
        const bool is_leaf = have && a.count == 0u;
        // ---- opening test (W-rule 2, fp32 decision W8): r_c = l*(1/theta) [+ delta] ----
        float rc = __fmul_rn(a.size, P.inv_theta);
        if (P.mac == 1) rc = __fadd_rn(rc, a.delta);
        const float rc2 = __fmul_rn(rc, rc);
        bool accept = false, amb = false;
        if (internal) {
            const float ax = __fsub_rn(bxl, r.x), bx = __fsub_rn(bxh, r.x);
            const float ay = __fsub_rn(byl, r.y), by = __fsub_rn(byh, r.y);
            const float az = __fsub_rn(bzl, r.z), bz = __fsub_rn(bzh, r.z);
            const float nx = fmaxf(0.f, fmaxf(ax, -bx)), fx = fmaxf(-ax, bx);
            const float ny = fmaxf(0.f, fmaxf(ay, -by)), fy = fmaxf(-ay, by);
            const float nz = fmaxf(0.f, fmaxf(az, -bz)), fz = fmaxf(-az, bz);
            const float d2min = __fmaf_rn(nz, nz, __fmaf_rn(ny, ny, __fmul_rn(nx, nx)));
            const float d2max = __fmaf_rn(fz, fz, __fmaf_rn(fy, fy, __fmul_rn(fx, fx)));
            accept = d2min > rc2;                    // every member passes
            amb = !accept && (d2max > rc2);          // some member might pass, some might not
        }
        // ---- nodes the box cannot decide: per-member test + vote ----
        u32 am = __ballot_sync(0xffffffffu, amb);
        c_exact += __popc(am);
        while (am) {
            const int src = __ffs(am) - 1;
            am &= am - 1;
            const float qx = __shfl_sync(0xffffffffu, r.x, src);
            const float qy = __shfl_sync(0xffffffffu, r.y, src);
            const float qz = __shfl_sync(0xffffffffu, r.z, src);
            const float q2 = __shfl_sync(0xffffffffu, rc2, src);
            const float dx = __fsub_rn(px, qx), dy = __fsub_rn(py, qy), dz = __fsub_rn(pz, qz);
            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            const bool ok = __all_sync(0xffffffffu, !live || d2 > q2);
            if ((int)lane == src) accept = ok;
        }
        const bool open = internal && !accept;
        // ---- append accepted nodes and leaf cells to the lists; push opened nodes ----
        const u32 m_acc = __ballot_sync(0xffffffffu, internal && accept);
        const u32 m_leaf = __ballot_sync(0xffffffffu, is_leaf);
        const u32 m_open = __ballot_sync(0xffffffffu, open);
        if (internal && accept) list_store(nlist, n_node + __popc(m_acc & lt), r);
        if (is_leaf) list_store(llist, n_leaf + __popc(m_leaf & lt), r);
        const bool bucket = open && !(a.size < __int_as_float(0x7f800000));
        if (open) stack[sp + __popc(m_open & lt)] = make_uint2(a.first, a.count);
        sp += __popc(m_open);
        n_node += __popc(m_acc);
        n_leaf += __popc(m_leaf);
        c_acc += __popc(m_acc);
        c_leaf += __popc(m_leaf);
        c_open += __popc(m_open) - __popc(__ballot_sync(0xffffffffu, bucket));
        __syncwarp();
        // ---- evaluate a list before the next step could overflow it ----
        if (n_node > kListFlushAt) {
            list_pad(nlist, n_node);
            __syncwarp();
            acc += eval_list<false>(nlist, n_node, npx, npy, npz);
            n_node = 0;
            __syncwarp();
        }
        if (n_leaf > kListFlushAt) {
            list_pad(llist, n_leaf);
            __syncwarp();
            acc += eval_list<true>(llist, n_leaf, npx, npy, npz);
            n_leaf = 0;
            __syncwarp();
        }
    }
    if (n_node > 0) {
        list_pad(nlist, n_node);
        __syncwarp();
        acc += eval_list<false>(nlist, n_node, npx, npy, npz);
    }
    if (n_leaf > 0) {
        list_pad(llist, n_leaf);
        __syncwarp();
        acc += eval_list<true>(llist, n_leaf, npx, npy, npz);
    }
    // ---- a7: Phi_t = -G * sum, written in the original cell order (W-rule 4) ----
    if (live) P.phi[__ldg(P.idx + s)] = P.negG * acc;
    if (lane == 0) P.gcount[g] = make_uint4(c_acc, c_leaf, c_open, c_exact);
}

// per-target interaction counts / int64 group counts from the uint4 group counters
__global__ void __launch_bounds__(256)
group_counts_export_kernel(const uint4* __restrict__ gcount, i64 ngroups, i64* __restrict__ out)
{
    const i64 g = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= ngroups) return;
    const uint4 c = gcount[g];
    out[3 * g + 0] = c.x; out[3 * g + 1] = c.y; out[3 * g + 2] = c.z;
}

__global__ void __launch_bounds__(256)
per_target_counts_kernel(const uint4* __restrict__ gcount, const u32* __restrict__ idx, i64 n, int group,
                         u32* __restrict__ out)
{
    const i64 s = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const uint4 c = gcount[s / group];
    out[idx[s]] = c.x + c.y;
}

// totals[0..3] = sum of the four group counters; totals[4] = sum over targets of (acc + leaf)
__global__ void __launch_bounds__(256)
group_counts_total_kernel(const uint4* __restrict__ gcount, i64 ngroups, i64 n, int group,
                          unsigned long long* __restrict__ totals)
{
    unsigned long long t[5] = {0, 0, 0, 0, 0};
    for (i64 g = (i64)blockIdx.x * blockDim.x + threadIdx.x; g < ngroups; g += (i64)gridDim.x * blockDim.x) {
        const uint4 c = gcount[g];
        const i64 members = min((i64)group, n - g * group);
        t[0] += c.x; t[1] += c.y; t[2] += c.z; t[3] += c.w;
        t[4] += (unsigned long long)(c.x + c.y) * (unsigned long long)members;
    }
    #pragma unroll
    for (int k = 0; k < 5; ++k) {
        #pragma unroll
        for (int o = 16; o > 0; o >>= 1) t[k] += __shfl_xor_sync(0xffffffffu, t[k], o);
        if (lane_id() == 0 && t[k]) atomicAdd(&totals[k], t[k]);
    }
}

}  // namespace bh
