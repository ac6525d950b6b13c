// walk.cuh -- steps a6 + a7: the group tree walk (§3.3) and the scatter of Phi.
//
// What is kept from the paper's kernel: 32 neighbouring (Morton-consecutive) target cells form a
// group that shares one traversal; the traversal stack lives in shared memory; a node is used only
// if EVERY member of the group accepts it (the all() vote), otherwise the whole
// group opens it; potentials are accumulated in registers.
// What differs (the paper's design is for a Fermi C2075, where lane 0 alone walks the tree):
//  * One warp walks TWO adjacent groups A = 2w, B = 2w+1 at once (lane = one target of A and one of
//    B).  The two groups keep their own votes -- every decision below is taken per group, so the
//    result is the one of DESIGN.md W1-W4 -- but they share the traversal: a stack entry carries
//    the set of groups that still need the subtree, and a node both groups accept (about 3/4 of
//    all list entries on the grid workloads) is fetched from shared memory once and evaluated for
//    both targets (packed fp32x2 arithmetic FADD2/FFMA2, sm_100; one MUFU.RSQ per interaction).
//  * The traversal is lane-parallel: each step pops up to 4 stack entries and tests their <= 32
//    children at once, one child per lane.  The vote ("all members have d^2 > r_c^2") is decided
//    without touching the members whenever the group's bounding box proves it: fp32 rounding is
//    monotone, so the fp32 d^2 evaluated at the box's nearest (farthest) point bounds every
//    member's fp32 d^2 from below (above).  Only nodes between the two bounds take the per-member
//    test + __all_sync vote.
//  * Accepted nodes and leaf cells go to interaction lists in shared memory: U2 (both groups),
//    UA / UB (one group only) -- regions of ONE SoA block, so an append is four stores at one
//    computed index whatever the list; evaluated two ENTRIES per packed instruction against a
//    scalar target coordinate, U2 for the lane's two targets from the same loads -- and C (leaf
//    cells inside a group's bounding box -- the only ones that can be a target's own cell or
//    coincide with it -- evaluated with the zero-distance mask of W3).
//  * The member votes of one step are batched: each lane collects its member's failures as a bit
//    per undecided node (the sign bit of bits(d^2) + ~bits(r_c^2), moved in by a funnel shift) and
//    one OR-reduction per group replaces a vote per node.
//  * The kernel counts, per group, the list entries it evaluates (geval): the tests hold that count
//    against the oracle's accepted + leaf, and it is the numerator of the reported roofline.
//  * PERIODIC instantiation (App. A): records are moved to the periodic image nearest the pair, entries
//    on the seam are voted and evaluated with a per-member minimum image, and every entry adds the
//    Ewald correction looked up in the context's field array (ewald.cuh).
//  * Partial sums are fp32 over one list flush (<= 128 entries, 4 accumulators) and are flushed
//    into an fp64 sum per target, which keeps the summation error near 1e-7 relative.
//  * Phi is written straight to the original cell order (step a7 is fused: no extra pass).
// ALU-bound: 13 flops per interaction by the north-star convention; MUFU (16 rsqrt/clk/SM) is the
// co-limiter.
// BH_OPT_GROUP = 1 (W5, the textbook per-target walk) is walk_single_kernel below.
#pragma once
#include "common.cuh"
#include "ewald.cuh"
#include "tree.cuh"

namespace bh {

constexpr int kWalkWarps = 4;                 // warps (= group pairs) per CTA
constexpr int kU2Cap = 128;                   // entries of the both-groups list
constexpr int kU1Cap = 64;                    // entries of each one-group list
constexpr int kSoaCap = kU2Cap + 2 * kU1Cap;  // the three unchecked lists share ONE SoA block x[256] y[256] z[256] m[256]:
constexpr int kOffUA = kU2Cap;                //   U2 at [0, 128), UA at [128, 192), UB at [192, 256) of every component,
constexpr int kOffUB = kU2Cap + kU1Cap;       //   so an append is four stores at one computed index whatever the list
constexpr int kCCap = 64;                     // entries of the checked list (float4 + group mask)
constexpr int kStepMax = 32;                  // a traversal step appends <= 32 entries to any list
constexpr int kStackPerLevel = 36;            // stack entries a level can leave behind (<= 3 + 32)
constexpr u32 kCountMask = 0x3fffffffu;       // stack entry .y = child count | group set << 30
constexpr float kTinyD2 = 1.0e-36f;           // keeps d^2 of the unchecked lists off zero

struct WalkParams {
    const float4* rec;        // [n_slots] (x, y, z, m) of every node / leaf-cell slot
    const WalkAux* aux;       // [n_slots]
    const u32* leaf_slot;     // [n] slot of sorted cell s (the targets are read from rec)
    SortedView sv;            // sorted cells: original index of sorted slot s
    double* phi;              // [n] original order
    double* acc;              // bh_field only: [3n] (gx, gy, gz) per cell, original order
    uint4* gcount;            // [ngroups] {accepted, leaf, opened, exact-tested}
    u32* geval;               // [ngroups] list entries the Phi kernel itself evaluated for the group
    i64 n;
    i64 ngroups;
    float inv_theta;          // (float)(1/theta); +inf for theta = 0
    int mac;                  // BH_MAC_*
    double negG;
    int stack_cap;            // entries per warp
    u32 ntargets;             // only cells with original index < ntargets are targets (bh_set_num_targets)
    u32 nslots;               // checked build: every slot read must be below this
    EwaldTab ew;              // PERIODIC instantiations only: the Ewald field array (ewald.cuh)
};

__host__ __device__ inline size_t walk_smem_per_warp(int stack_cap)
{
    return (size_t)kSoaCap * 16 + (size_t)kCCap * 16 + (size_t)kCCap * 4 + 32 * 16 +
           (size_t)stack_cap * sizeof(uint2);
}

__device__ __forceinline__ float rsqrt_approx(float v)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(v));
    return r;
}

__device__ __forceinline__ float2 splat2(float v) { return make_float2(v, v); }

// ---- unchecked lists: SoA (x[CAP] y[CAP] z[CAP] m[CAP]), evaluated four entries per iteration ------
// The packed fp32x2 operands are two ENTRIES (adjacent registers of one 16-byte shared load), the
// target's coordinates are loop-invariant splatted pairs: no per-entry register shuffling.
// Lists are padded to a multiple of 4 entries by the caller.
struct Tgt2 { float2 x, y, z; };           // (-p, -p) per coordinate of one target

__device__ __forceinline__ void quad_body(const float4 x, const float4 y, const float4 z, const float4 m,
                                          const Tgt2& t, float2& s0, float2& s1)
{
    const float2 dx0 = __fadd2_rn(make_float2(x.x, x.y), t.x), dx1 = __fadd2_rn(make_float2(x.z, x.w), t.x);
    const float2 dy0 = __fadd2_rn(make_float2(y.x, y.y), t.y), dy1 = __fadd2_rn(make_float2(y.z, y.w), t.y);
    const float2 dz0 = __fadd2_rn(make_float2(z.x, z.y), t.z), dz1 = __fadd2_rn(make_float2(z.z, z.w), t.z);
    float2 d0 = __ffma2_rn(dx0, dx0, splat2(kTinyD2));
    float2 d1 = __ffma2_rn(dx1, dx1, splat2(kTinyD2));
    d0 = __ffma2_rn(dy0, dy0, d0);
    d1 = __ffma2_rn(dy1, dy1, d1);
    d0 = __ffma2_rn(dz0, dz0, d0);
    d1 = __ffma2_rn(dz1, dz1, d1);
    const float2 r0 = make_float2(rsqrt_approx(d0.x), rsqrt_approx(d0.y));
    const float2 r1 = make_float2(rsqrt_approx(d1.x), rsqrt_approx(d1.y));
    s0 = __ffma2_rn(make_float2(m.x, m.y), r0, s0);
    s1 = __ffma2_rn(make_float2(m.z, m.w), r1, s1);
}

// one target
template <int CAP>
__device__ __forceinline__ double eval_soa(const float* __restrict__ L, int cnt, const Tgt2& t)
{
    const float4* X = reinterpret_cast<const float4*>(L);
    const float4* Y = reinterpret_cast<const float4*>(L + CAP);
    const float4* Z = reinterpret_cast<const float4*>(L + 2 * CAP);
    const float4* M = reinterpret_cast<const float4*>(L + 3 * CAP);
    float2 s0 = splat2(0.f), s1 = splat2(0.f);
    const int nq = (cnt + 3) >> 2;
    #pragma unroll 2
    for (int q = 0; q < nq; ++q) quad_body(X[q], Y[q], Z[q], M[q], t, s0, s1);
    return ((double)s0.x + (double)s0.y) + ((double)s1.x + (double)s1.y);
}

// two targets (the lane's member of group A and of group B) from the same loads
template <int CAP>
__device__ __forceinline__ void eval_soa2(const float* __restrict__ L, int cnt, const Tgt2& tA, const Tgt2& tB,
                                          double& accA, double& accB)
{
    const float4* X = reinterpret_cast<const float4*>(L);
    const float4* Y = reinterpret_cast<const float4*>(L + CAP);
    const float4* Z = reinterpret_cast<const float4*>(L + 2 * CAP);
    const float4* M = reinterpret_cast<const float4*>(L + 3 * CAP);
    float2 a0 = splat2(0.f), a1 = splat2(0.f), b0 = splat2(0.f), b1 = splat2(0.f);
    const int nq = (cnt + 3) >> 2;
    #pragma unroll 2
    for (int q = 0; q < nq; ++q) {
        const float4 x = X[q], y = Y[q], z = Z[q], m = M[q];
        quad_body(x, y, z, m, tA, a0, a1);
        quad_body(x, y, z, m, tB, b0, b1);
    }
    accA += ((double)a0.x + (double)a0.y) + ((double)a1.x + (double)a1.y);
    accB += ((double)b0.x + (double)b0.y) + ((double)b1.x + (double)b1.y);
}

// ---- C: leaf cells inside a group's bounding box; zero-distance pairs are skipped (W3) ----------
__device__ __forceinline__ void eval_c(const float4* __restrict__ L, const u32* __restrict__ Lm, int cnt,
                                       const float2 npx, const float2 npy, const float2 npz, double& accA,
                                       double& accB, u32& evA, u32& evB)
{
    float2 s = splat2(0.f);
    for (int e = 0; e < cnt; ++e) {
        const float4 v = L[e];
        const u32 mk = Lm[e];
        evA += mk & 1u; evB += mk >> 1;               // every lane sees every entry: warp-uniform
        const float2 dx = __fadd2_rn(splat2(v.x), npx);
        const float2 dy = __fadd2_rn(splat2(v.y), npy);
        const float2 dz = __fadd2_rn(splat2(v.z), npz);
        float2 d2 = __fmul2_rn(dx, dx);
        d2 = __ffma2_rn(dy, dy, d2);
        d2 = __ffma2_rn(dz, dz, d2);
        float2 r = make_float2(rsqrt_approx(d2.x), rsqrt_approx(d2.y));
        r.x = (d2.x >= 1.17549435e-38f && (mk & 1u)) ? r.x : 0.f;
        r.y = (d2.y >= 1.17549435e-38f && (mk & 2u)) ? r.y : 0.f;
        s = __ffma2_rn(splat2(v.w), r, s);
    }
    accA += (double)s.x;
    accB += (double)s.y;
}

// ---- NEXT-4 (bh_field): the same lists, Phi with the same arithmetic, plus g = -grad Phi ----------
// Every entry contributes the gradient of its monopole term: sum of w * (r_j - r_t), w = m/d^3 =
// (m * rinv) * (rinv * rinv); three packed multiplies and three packed fmas more per entry pair.
struct Grad2 { float2 x, y, z; };
__device__ __forceinline__ Grad2 grad_zero()
{
    Grad2 g; g.x = g.y = g.z = splat2(0.f); return g;
}
__device__ __forceinline__ void grad_flush(const Grad2& g, double* acc3)
{
    acc3[0] += (double)g.x.x + (double)g.x.y;
    acc3[1] += (double)g.y.x + (double)g.y.y;
    acc3[2] += (double)g.z.x + (double)g.z.y;
}

__device__ __forceinline__ void quad_body_g(const float4 x, const float4 y, const float4 z, const float4 m,
                                            const Tgt2& t, float2& s0, float2& s1, Grad2& g)
{
    const float2 dx0 = __fadd2_rn(make_float2(x.x, x.y), t.x), dx1 = __fadd2_rn(make_float2(x.z, x.w), t.x);
    const float2 dy0 = __fadd2_rn(make_float2(y.x, y.y), t.y), dy1 = __fadd2_rn(make_float2(y.z, y.w), t.y);
    const float2 dz0 = __fadd2_rn(make_float2(z.x, z.y), t.z), dz1 = __fadd2_rn(make_float2(z.z, z.w), t.z);
    float2 d0 = __ffma2_rn(dx0, dx0, splat2(kTinyD2));
    float2 d1 = __ffma2_rn(dx1, dx1, splat2(kTinyD2));
    d0 = __ffma2_rn(dy0, dy0, d0);
    d1 = __ffma2_rn(dy1, dy1, d1);
    d0 = __ffma2_rn(dz0, dz0, d0);
    d1 = __ffma2_rn(dz1, dz1, d1);
    const float2 r0 = make_float2(rsqrt_approx(d0.x), rsqrt_approx(d0.y));
    const float2 r1 = make_float2(rsqrt_approx(d1.x), rsqrt_approx(d1.y));
    const float2 m0 = make_float2(m.x, m.y), m1 = make_float2(m.z, m.w);
    s0 = __ffma2_rn(m0, r0, s0);
    s1 = __ffma2_rn(m1, r1, s1);
    const float2 w0 = __fmul2_rn(__fmul2_rn(m0, r0), __fmul2_rn(r0, r0));
    const float2 w1 = __fmul2_rn(__fmul2_rn(m1, r1), __fmul2_rn(r1, r1));
    g.x = __ffma2_rn(dx1, w1, __ffma2_rn(dx0, w0, g.x));
    g.y = __ffma2_rn(dy1, w1, __ffma2_rn(dy0, w0, g.y));
    g.z = __ffma2_rn(dz1, w1, __ffma2_rn(dz0, w0, g.z));
}

template <int CAP>
__device__ __forceinline__ double eval_soa_g(const float* __restrict__ L, int cnt, const Tgt2& t, double* acc3)
{
    const float4* X = reinterpret_cast<const float4*>(L);
    const float4* Y = reinterpret_cast<const float4*>(L + CAP);
    const float4* Z = reinterpret_cast<const float4*>(L + 2 * CAP);
    const float4* M = reinterpret_cast<const float4*>(L + 3 * CAP);
    float2 s0 = splat2(0.f), s1 = splat2(0.f);
    Grad2 g = grad_zero();
    const int nq = (cnt + 3) >> 2;
    #pragma unroll 2
    for (int q = 0; q < nq; ++q) quad_body_g(X[q], Y[q], Z[q], M[q], t, s0, s1, g);
    grad_flush(g, acc3);
    return ((double)s0.x + (double)s0.y) + ((double)s1.x + (double)s1.y);
}

template <int CAP>
__device__ __forceinline__ void eval_soa2_g(const float* __restrict__ L, int cnt, const Tgt2& tA, const Tgt2& tB,
                                            double& accA, double& accB, double* gA, double* gB)
{
    const float4* X = reinterpret_cast<const float4*>(L);
    const float4* Y = reinterpret_cast<const float4*>(L + CAP);
    const float4* Z = reinterpret_cast<const float4*>(L + 2 * CAP);
    const float4* M = reinterpret_cast<const float4*>(L + 3 * CAP);
    float2 a0 = splat2(0.f), a1 = splat2(0.f), b0 = splat2(0.f), b1 = splat2(0.f);
    Grad2 ga = grad_zero(), gb = grad_zero();
    const int nq = (cnt + 3) >> 2;
    for (int q = 0; q < nq; ++q) {
        const float4 x = X[q], y = Y[q], z = Z[q], m = M[q];
        quad_body_g(x, y, z, m, tA, a0, a1, ga);
        quad_body_g(x, y, z, m, tB, b0, b1, gb);
    }
    accA += ((double)a0.x + (double)a0.y) + ((double)a1.x + (double)a1.y);
    accB += ((double)b0.x + (double)b0.y) + ((double)b1.x + (double)b1.y);
    grad_flush(ga, gA);
    grad_flush(gb, gB);
}

__device__ __forceinline__ void eval_c_g(const float4* __restrict__ L, const u32* __restrict__ Lm, int cnt,
                                         const float2 npx, const float2 npy, const float2 npz, double& accA,
                                         double& accB, double* gA, double* gB, u32& evA, u32& evB)
{
    float2 s = splat2(0.f), gx = splat2(0.f), gy = splat2(0.f), gz = splat2(0.f);
    for (int e = 0; e < cnt; ++e) {
        const float4 v = L[e];
        const u32 mk = Lm[e];
        evA += mk & 1u; evB += mk >> 1;
        const float2 dx = __fadd2_rn(splat2(v.x), npx);
        const float2 dy = __fadd2_rn(splat2(v.y), npy);
        const float2 dz = __fadd2_rn(splat2(v.z), npz);
        float2 d2 = __fmul2_rn(dx, dx);
        d2 = __ffma2_rn(dy, dy, d2);
        d2 = __ffma2_rn(dz, dz, d2);
        float2 r = make_float2(rsqrt_approx(d2.x), rsqrt_approx(d2.y));
        r.x = (d2.x >= 1.17549435e-38f && (mk & 1u)) ? r.x : 0.f;
        r.y = (d2.y >= 1.17549435e-38f && (mk & 2u)) ? r.y : 0.f;
        s = __ffma2_rn(splat2(v.w), r, s);
        const float2 w = __fmul2_rn(__fmul2_rn(splat2(v.w), r), __fmul2_rn(r, r));
        gx = __ffma2_rn(dx, w, gx); gy = __ffma2_rn(dy, w, gy); gz = __ffma2_rn(dz, w, gz);
    }
    accA += (double)s.x;
    accB += (double)s.y;
    gA[0] += (double)gx.x; gA[1] += (double)gy.x; gA[2] += (double)gz.x;
    gB[0] += (double)gx.y; gB[1] += (double)gy.y; gB[2] += (double)gz.y;
}

// ---- PERIODIC (App. A): every entry contributes m (1/d + corr1(d_vec/L)/L) = m f_EF (Eq. A.1) -------------------
// The unchecked lists hold entries already moved to the periodic image nearest the pair of groups, and only
// entries for which that image is the minimum image for EVERY member, so plain differences are minimum-image
// displacements.  One entry at a time: the table lookup (one 32-byte record, ewald.cuh) dominates.
template <int CAP, bool NESTED>
__device__ __forceinline__ void eval_soa2_pn(const float* __restrict__ L, int cnt, const float4 tA, const float4 tB,
                                            const EwaldTab& T, double& accA, double& accB, bool doA, bool doB)
{
    // 1/d and corr1/L are added per entry BEFORE the sum: far entries nearly cancel (f_EF is small where 1/d is
    // not), two separate fp32 sums would each carry the rounding of a total ~100 x larger than their difference
    float sa = 0.f, sb = 0.f;
    #pragma unroll 1
    for (int e = 0; e < cnt; ++e) {
        const float x = L[e], y = L[CAP + e], z = L[2 * CAP + e], m = L[3 * CAP + e];
        if (doA) {
            const float dx = x - tA.x, dy = y - tA.y, dz = z - tA.z;
            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmaf_rn(dx, dx, kTinyD2)));
            sa = __fmaf_rn(m, __fmaf_rn(ewald_corr<NESTED>(T, dx, dy, dz), T.invL, rsqrt_approx(d2)), sa);
        }
        if (doB) {
            const float dx = x - tB.x, dy = y - tB.y, dz = z - tB.z;
            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmaf_rn(dx, dx, kTinyD2)));
            sb = __fmaf_rn(m, __fmaf_rn(ewald_corr<NESTED>(T, dx, dy, dz), T.invL, rsqrt_approx(d2)), sb);
        }
    }
    accA += (double)sa;
    accB += (double)sb;
}

// checked list under periodic boundaries: explicit minimum image per target; the own cell and zero-distance
// pairs keep their image / background part m corr1(0)/L (reading P5) and drop only 1/d
template <bool NESTED>
__device__ __forceinline__ void eval_c_pn(const float4* __restrict__ L, const u32* __restrict__ Lm, int cnt, const float4 tA,
                                         const float4 tB, const EwaldTab& T, double& accA, double& accB, u32& evA, u32& evB)
{
    float sa = 0.f, sb = 0.f;
    for (int e = 0; e < cnt; ++e) {
        const float4 v = L[e];
        const u32 mk = Lm[e];
        evA += mk & 1u; evB += mk >> 1;
        {
            const float dx = wrap_mi(v.x - tA.x, T.L, T.invL), dy = wrap_mi(v.y - tA.y, T.L, T.invL), dz = wrap_mi(v.z - tA.z, T.L, T.invL);
            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, dx * dx));
            const float ri = d2 >= 1.17549435e-38f ? rsqrt_approx(d2) : 0.f;
            if (mk & 1u) sa = __fmaf_rn(v.w, __fmaf_rn(ewald_corr<NESTED>(T, dx, dy, dz), T.invL, ri), sa);
        }
        {
            const float dx = wrap_mi(v.x - tB.x, T.L, T.invL), dy = wrap_mi(v.y - tB.y, T.L, T.invL), dz = wrap_mi(v.z - tB.z, T.L, T.invL);
            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, dx * dx));
            const float ri = d2 >= 1.17549435e-38f ? rsqrt_approx(d2) : 0.f;
            if (mk & 2u) sb = __fmaf_rn(v.w, __fmaf_rn(ewald_corr<NESTED>(T, dx, dy, dz), T.invL, ri), sb);
        }
    }
    accA += (double)sa;
    accB += (double)sb;
}

// one grid (the default) or nested grids: chosen once per list, not per interaction
template <int CAP>
__device__ __forceinline__ void eval_soa2_p(const float* __restrict__ L, int cnt, const float4 tA, const float4 tB,
                                            const EwaldTab& T, double& accA, double& accB, bool doA, bool doB)
{
    if (T.nref > 1) eval_soa2_pn<CAP, true>(L, cnt, tA, tB, T, accA, accB, doA, doB);
    else eval_soa2_pn<CAP, false>(L, cnt, tA, tB, T, accA, accB, doA, doB);
}

__device__ __forceinline__ void eval_c_p(const float4* __restrict__ L, const u32* __restrict__ Lm, int cnt, const float4 tA,
                                         const float4 tB, const EwaldTab& T, double& accA, double& accB, u32& evA, u32& evB)
{
    if (T.nref > 1) eval_c_pn<true>(L, Lm, cnt, tA, tB, T, accA, accB, evA, evB);
    else eval_c_pn<false>(L, Lm, cnt, tA, tB, T, accA, accB, evA, evB);
}

// packed minimum image: d - L rint(d / L), rint by the 1.5 * 2^23 trick (|d / L| is far below 2^22)
__device__ __forceinline__ float2 wrap_mi2(float2 d, float L, float invL)
{
    const float2 big = splat2(12582912.f);
    const float2 q = __fadd2_rn(__fadd2_rn(__fmul2_rn(d, splat2(invL)), big), splat2(-12582912.f));
    return __ffma2_rn(splat2(-L), q, d);
}

template <int CAP>
__device__ __forceinline__ void soa_store(float* L, int e, float4 r)
{
    L[e] = r.x; L[CAP + e] = r.y; L[2 * CAP + e] = r.z; L[3 * CAP + e] = r.w;
}

// zero-mass entries far away (finite d^2, no NaN) up to the next multiple of 4
template <int CAP>
__device__ __forceinline__ void soa_pad(float* L, int cnt)
{
    const int e = cnt + (int)lane_id();
    if (e < ((cnt + 3) & ~3)) soa_store<CAP>(L, e, make_float4(3.0e18f, 3.0e18f, 3.0e18f, 0.f));
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

// fp32 d^2 at the nearest / farthest point of the boxes of groups A (.x) and B (.y) from q, with the
// rounding sequence of W8 (monotone in every |component|, so they bound every member's fp32 d^2).
struct Box2 { float2 xl, xh, yl, yh, zl, zh; };

__device__ __forceinline__ void box_d2(const float4 q, const Box2& b, float2& d2min, float2& d2max)
{
    const float2 nqx = splat2(-q.x), nqy = splat2(-q.y), nqz = splat2(-q.z);
    const float2 ax = __fadd2_rn(b.xl, nqx), bx = __fadd2_rn(b.xh, nqx);
    const float2 ay = __fadd2_rn(b.yl, nqy), by = __fadd2_rn(b.yh, nqy);
    const float2 az = __fadd2_rn(b.zl, nqz), bz = __fadd2_rn(b.zh, nqz);
    const float2 nx = make_float2(fmaxf(0.f, fmaxf(ax.x, -bx.x)), fmaxf(0.f, fmaxf(ax.y, -bx.y)));
    const float2 ny = make_float2(fmaxf(0.f, fmaxf(ay.x, -by.x)), fmaxf(0.f, fmaxf(ay.y, -by.y)));
    const float2 nz = make_float2(fmaxf(0.f, fmaxf(az.x, -bz.x)), fmaxf(0.f, fmaxf(az.y, -bz.y)));
    const float2 fx = make_float2(fmaxf(-ax.x, bx.x), fmaxf(-ax.y, bx.y));
    const float2 fy = make_float2(fmaxf(-ay.x, by.x), fmaxf(-ay.y, by.y));
    const float2 fz = make_float2(fmaxf(-az.x, bz.x), fmaxf(-az.y, bz.y));
    d2min = __ffma2_rn(nz, nz, __ffma2_rn(ny, ny, __fmul2_rn(nx, nx)));
    d2max = __ffma2_rn(fz, fz, __ffma2_rn(fy, fy, __fmul2_rn(fx, fx)));
}

// COUNT = false: the hot kernel -- builds the lists, evaluates them, writes Phi.
// COUNT = true : the same traversal and the same decisions, but it only counts (W6): per group
//                {internal nodes accepted, leaf cells summed, internal nodes opened, nodes that
//                needed the per-member test}; no lists, no arithmetic on masses, no Phi.
// SUBSET = true: only cells with original index < P.ntargets are targets (bh_set_num_targets); the
//                default instantiation carries none of that code.
// ACC = true   : bh_field -- additionally g = -grad Phi on the same lists (NEXT-4); its own register budget.
// PERIODIC     : periodic boundaries (App. A, NEXT-3; the cube of the build is the periodic box): every child record
//                is first moved to the image nearest the centre of the pair's bounding box.  Where that image is the
//                minimum image for every member (|q' - c|_a + half-width_a < L/2 on all axes) the step runs exactly as
//                in the isolated case; a child on the seam (half a box away along some axis) takes the per-member test
//                with an explicit minimum image per member and, if used, goes to the checked list, which wraps per
//                target.  Every entry is evaluated as m (1/d + corr1/L) with the table lookup of ewald.cuh.
template <bool COUNT, bool SUBSET = false, bool ACC = false, bool PERIODIC = false>
__global__ void __launch_bounds__(kWalkWarps * 32, 24 / kWalkWarps)
walk_pair_kernel(const WalkParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5;
    const u32 lane = lane_id();
    const i64 pr = (i64)blockIdx.x * kWalkWarps + warp;       // pair of groups (2 pr, 2 pr + 1)
    const i64 gA = 2 * pr, gB = gA + 1;
    if (gA >= P.ngroups) return;                      // whole warp leaves; no block-level sync below

    unsigned char* my = smem_raw + (size_t)warp * walk_smem_per_warp(P.stack_cap);
    float* U2 = reinterpret_cast<float*>(my);                           // both groups (SoA block, component stride kSoaCap)
    float* UA = U2 + kOffUA;                                            // group A only (same block)
    float* UB = U2 + kOffUB;                                            // group B only (same block)
    float4* C = reinterpret_cast<float4*>(U2 + 4 * kSoaCap);            // checked leaf cells
    u32* Cm = reinterpret_cast<u32*>(C + kCCap);                        //   and the groups they serve
    float4* amb = reinterpret_cast<float4*>(Cm + kCCap);                // nodes awaiting the member vote
    uint2* stack = reinterpret_cast<uint2*>(amb + 32);                  // (first child slot, count | groups << 30)

    // ---- the targets (W-rule 1): group g = sorted slots [32g, 32g+32) ----
    const bool hasB = gB < P.ngroups;
    const int ntA = (int)min((i64)32, P.n - gA * 32);
    const int ntB = hasB ? (int)min((i64)32, P.n - gB * 32) : 0;
    const bool liveA = (int)lane < ntA, liveB = (int)lane < ntB;
    const i64 sA = gA * 32 + lane, sB = gB * 32 + lane;
    if (SUBSET) {
        // source-only cells (essential nodes received from other domains) sit in long runs
        // of the sorted order: a pair of groups without a single target has nothing to compute
        const bool want = (liveA && sv_idx(P.sv, sA) < P.ntargets) || (liveB && sv_idx(P.sv, sB) < P.ntargets);
        if (!__any_sync(0xffffffffu, want)) {
            if (lane == 0) {
                if (COUNT) {
                    P.gcount[gA] = make_uint4(0u, 0u, 0u, 0u);
                    if (hasB) P.gcount[gB] = make_uint4(0u, 0u, 0u, 0u);
                } else {
                    P.geval[gA] = 0u;
                    if (hasB) P.geval[gB] = 0u;
                }
            }
            return;
        }
    }
    const float4 tA = __ldg(P.rec + __ldg(P.leaf_slot + (liveA ? sA : gA * 32)));
    const float4 tB = __ldg(P.rec + __ldg(P.leaf_slot + (liveB ? sB : (hasB ? gB * 32 : gA * 32))));
    Box2 box;                                         // bounding boxes of the live targets of A and B
    box.xl = make_float2(warp_min(tA.x), warp_min(tB.x)); box.xh = make_float2(warp_max(tA.x), warp_max(tB.x));
    box.yl = make_float2(warp_min(tA.y), warp_min(tB.y)); box.yh = make_float2(warp_max(tA.y), warp_max(tB.y));
    box.zl = make_float2(warp_min(tA.z), warp_min(tB.z)); box.zh = make_float2(warp_max(tA.z), warp_max(tB.z));
    const float2 npx = make_float2(-tA.x, -tB.x), npy = make_float2(-tA.y, -tB.y), npz = make_float2(-tA.z, -tB.z);
    Tgt2 TA, TB;                                      // splatted per target, for the entry-packed lists
    TA.x = splat2(-tA.x); TA.y = splat2(-tA.y); TA.z = splat2(-tA.z);
    TB.x = splat2(-tB.x); TB.y = splat2(-tB.y); TB.z = splat2(-tB.z);

    // PERIODIC: centre and half-widths of the pair's bounding box, the reach within which the image nearest the
    // centre is every member's minimum image (a relative 1e-5 of L/2 is kept clear for the fp32 roundings)
    float pcx = 0.f, pcy = 0.f, pcz = 0.f, phx = 0.f, phy = 0.f, phz = 0.f, reach = 0.f;
    if (PERIODIC) {
        const float x0 = fminf(box.xl.x, box.xl.y), x1 = fmaxf(box.xh.x, box.xh.y);
        const float y0 = fminf(box.yl.x, box.yl.y), y1 = fmaxf(box.yh.x, box.yh.y);
        const float z0 = fminf(box.zl.x, box.zl.y), z1 = fmaxf(box.zh.x, box.zh.y);
        pcx = 0.5f * (x0 + x1); pcy = 0.5f * (y0 + y1); pcz = 0.5f * (z0 + z1);
        phx = 0.5f * (x1 - x0); phy = 0.5f * (y1 - y0); phz = 0.5f * (z1 - z0);
        reach = 0.5f * P.ew.L * (1.0f - 1.0e-5f);
    }

    double accA = 0.0, accB = 0.0;
    double grA[3] = {0.0, 0.0, 0.0}, grB[3] = {0.0, 0.0, 0.0};   // ACC: sums of w (r_j - r_t)
    int nU2 = 0, nUA = 0, nUB = 0, nC = 0;          // list fill (warp-uniform)
    u32 evA = 0, evB = 0;                           // list entries evaluated so far for A / B (unpadded, warp-uniform)
    u32 cAccA = 0, cLeafA = 0, cOpenA = 0, cExA = 0;  // COUNT: per-lane partial counters
    u32 cAccB = 0, cLeafB = 0, cOpenB = 0, cExB = 0;
    int sp = 0;
    if (P.n >= 2) {                             // root is tested like any other node (W-rule 2)
        if (lane == 0) stack[0] = make_uint2(0u, 1u | ((hasB ? 3u : 1u) << 30));
        sp = 1;
    }
    __syncwarp();

    const u32 lt = (1u << lane) - 1u;
    const int sub = lane >> 3, j = lane & 7;
    const float inv_theta = P.inv_theta;
    const bool mac94 = P.mac == 1;
    const float4* __restrict__ rec = P.rec;
    const uint4* __restrict__ aux = reinterpret_cast<const uint4*>(P.aux);
    while (sp > 0) {
        // ---- pop up to 4 entries; lane (sub, j) takes child j of entry sub ----
        int npop = sp < 4 ? sp : 4;
        uint2 e = make_uint2(0u, 0u);
        if (sub < npop) e = stack[sp - 1 - sub];
        u32 jj = (u32)j;
        if (__any_sync(0xffffffffu, (e.y & kCountMask) > 8u)) {
            // rare: a bucket of > 8 coincident cells is near the top; serve the top entry alone,
            // 32 children per step, shrinking it in place while more than 32 remain
            e = stack[sp - 1];
            jj = lane;
            npop = 1;
            __syncwarp();
            if ((e.y & kCountMask) > 32u) {
                if (lane == 0) stack[sp - 1] = make_uint2(e.x + 32u, e.y - 32u);
                e.y = (e.y & ~kCountMask) | 32u;
                npop = 0;
            }
        }
        sp -= npop;
        __syncwarp();
        const bool have = jj < (e.y & kCountMask);
        const u32 msk = have ? (e.y >> 30) : 0u;        // groups that want this child
        const u32 slot = e.x + jj;
        float4 r = make_float4(0.f, 0.f, 0.f, 0.f);
        uint4 t = make_uint4(0u, 0u, 0u, 0u);           // {size, delta, first child, child count}
        BH_DCHECK(!have || slot < P.nslots);
        if (have) { r = __ldg(rec + slot); t = __ldg(aux + slot); }
        const bool internal = t.w > 0u;
        const bool leaf = have && !internal;
        bool seam = false;                              // PERIODIC: the nearest image is not every member's minimum image
        if (PERIODIC) {
            // r - L rint((r - c)/L): a record that needs no shift stays bit-identical (the own-cell check relies on it)
            r.x = __fmaf_rn(-P.ew.L, rint_magic((r.x - pcx) * P.ew.invL), r.x);
            r.y = __fmaf_rn(-P.ew.L, rint_magic((r.y - pcy) * P.ew.invL), r.y);
            r.z = __fmaf_rn(-P.ew.L, rint_magic((r.z - pcz) * P.ew.invL), r.z);
            const float ix = r.x - pcx, iy = r.y - pcy, iz = r.z - pcz;
            seam = have && (fabsf(ix) + phx > reach || fabsf(iy) + phy > reach || fabsf(iz) + phz > reach);
        }
        // ---- opening test (W-rule 2, fp32 decision W8): r_c = l*(1/theta) [+ delta] ----
        float rc = __fmul_rn(__uint_as_float(t.x), inv_theta);
        if (mac94) rc = __fadd_rn(rc, __uint_as_float(t.y));
        const float rc2 = __fmul_rn(rc, rc);
        float2 d2min, d2max;
        box_d2(r, box, d2min, d2max);
        u32 accm = 0u, ambm = 0u;                       // groups that accept / need the member vote
        if (internal) {
            accm = ((d2min.x > rc2 ? 1u : 0u) | (d2min.y > rc2 ? 2u : 0u)) & msk;     // every member passes
            ambm = ((d2max.x > rc2 ? 1u : 0u) | (d2max.y > rc2 ? 2u : 0u)) & msk & ~accm;
            if (PERIODIC && seam) { accm = 0u; ambm = msk; }                         // the box bounds do not hold on the seam
        }
        // ---- nodes a box cannot decide: per-member test + vote ----
        const u32 bAmb = __ballot_sync(0xffffffffu, ambm != 0u);
        if (bAmb) {
            const int myr = __popc(bAmb & lt);
            // .w = ~bits(r_c^2): for non-negative floats d^2 <= r_c^2 iff bits(d^2) + ~bits(r_c^2) < 0 as integers
            if (ambm) amb[myr] = make_float4(r.x, r.y, r.z, __uint_as_float(~__float_as_uint(rc2)));
            __syncwarp();
            const int na = __popc(bAmb);
            BH_DCHECK(na >= 1 && na <= 32);
            // failA / failB collect, one bit per undecided node (node i at bit na - 1 - i), whether this lane's
            // member of A / B does NOT pass it (the sign bit of the integer difference is shifted in); one
            // OR-reduction per group then replaces a vote per node
            u32 failA = 0u, failB = 0u;
            #pragma unroll 4
            for (int i = 0; i < na; ++i) {
                const float4 q = amb[i];
                float2 dx = __fadd2_rn(splat2(q.x), npx), dy = __fadd2_rn(splat2(q.y), npy),
                       dz = __fadd2_rn(splat2(q.z), npz);
                if (PERIODIC) {                           // the member's own minimum image (a no-op off the seam)
                    dx = wrap_mi2(dx, P.ew.L, P.ew.invL); dy = wrap_mi2(dy, P.ew.L, P.ew.invL); dz = wrap_mi2(dz, P.ew.L, P.ew.invL);
                }
                const float2 d2 = __ffma2_rn(dz, dz, __ffma2_rn(dy, dy, __fmul2_rn(dx, dx)));
                failA = __funnelshift_l(__float_as_uint(d2.x) + __float_as_uint(q.w), failA, 1);
                failB = __funnelshift_l(__float_as_uint(d2.y) + __float_as_uint(q.w), failB, 1);
            }
            const u32 resA = ~__reduce_or_sync(0xffffffffu, liveA ? failA : 0u);
            const u32 resB = ~__reduce_or_sync(0xffffffffu, liveB ? failB : 0u);
            const int bit = na - 1 - myr;
            accm |= ambm & (((resA >> bit) & 1u) | (((resB >> bit) & 1u) << 1));
            if (COUNT) { cExA += ambm & 1u; cExB += ambm >> 1; }
            __syncwarp();
        }
        const u32 om = internal ? (msk & ~accm) : 0u;                   // groups that open the node
        // ---- push opened nodes ----
        const u32 bOp = __ballot_sync(0xffffffffu, om != 0u);
        if (om) stack[sp + __popc(bOp & lt)] = make_uint2(t.z, t.w | (om << 30));
        sp += __popc(bOp);
        BH_DCHECK(sp <= P.stack_cap);
        if (COUNT) {
            const bool bucket = internal && !(__uint_as_float(t.x) < __int_as_float(0x7f800000));
            cAccA += accm & 1u; cAccB += accm >> 1;
            if (leaf) { cLeafA += msk & 1u; cLeafB += msk >> 1; }
            if (!bucket) { cOpenA += om & 1u; cOpenB += om >> 1; }
            __syncwarp();
            continue;
        }
        // ---- append accepted nodes and leaf cells to the lists ----
        // leaf cells inside a group's box may be a target's own cell or coincide with one
        const u32 cmask = internal ? accm : msk;                        // groups that take this child as a list entry
        const bool danger = (leaf && (((msk & 1u) && !(d2min.x > 0.f)) || ((msk & 2u) && !(d2min.y > 0.f)))) ||
                            (PERIODIC && seam && cmask != 0u);           // seam entries are wrapped per target
        const u32 um = danger ? 0u : cmask;                             // 3: both groups, 1: A only, 2: B only
        const u32 b1 = __ballot_sync(0xffffffffu, um & 1u);
        const u32 b2 = __ballot_sync(0xffffffffu, um & 2u);
        const u32 same = ((um & 1u) ? b1 : ~b1) & ((um & 2u) ? b2 : ~b2);   // lanes that append to the same list
        const int cU2 = __popc(b1 & b2), cUA = __popc(b1 & ~b2), cUB = __popc(b2 & ~b1);
        if (um) {
            const int at = (um == 3u ? nU2 : (um == 1u ? kOffUA + nUA : kOffUB + nUB)) + __popc(same & lt);
            soa_store<kSoaCap>(U2, at, r);
        }
        nU2 += cU2; nUA += cUA; nUB += cUB;
        BH_DCHECK(nU2 <= kU2Cap && nUA <= kU1Cap && nUB <= kU1Cap);
        const u32 bC = __ballot_sync(0xffffffffu, danger);
        if (bC) {                                                       // rare: only next to the groups' own cells
            if (danger) { const int at = nC + __popc(bC & lt); C[at] = r; Cm[at] = cmask; }
            nC += __popc(bC);
            BH_DCHECK(nC <= kCCap);
        }
        __syncwarp();
        // ---- evaluate a list before the next step could overflow it ----
        if ((((nUA | nUB | nC) >> 5) != 0) || nU2 >= kU2Cap - kStepMax) {
            if (nU2 >= kU2Cap - kStepMax) {
                soa_pad<kSoaCap>(U2, nU2);
                __syncwarp();
                if (PERIODIC) eval_soa2_p<kSoaCap>(U2, nU2, tA, tB, P.ew, accA, accB, true, true);
                else if (ACC) eval_soa2_g<kSoaCap>(U2, nU2, TA, TB, accA, accB, grA, grB);
                else eval_soa2<kSoaCap>(U2, nU2, TA, TB, accA, accB);
                evA += (u32)nU2; evB += (u32)nU2;
                nU2 = 0;
            }
            if (nUA >= kU1Cap - kStepMax) {
                soa_pad<kSoaCap>(UA, nUA);
                __syncwarp();
                if (PERIODIC) eval_soa2_p<kSoaCap>(UA, nUA, tA, tB, P.ew, accA, accB, true, false);
                else accA += ACC ? eval_soa_g<kSoaCap>(UA, nUA, TA, grA) : eval_soa<kSoaCap>(UA, nUA, TA);
                evA += (u32)nUA;
                nUA = 0;
            }
            if (nUB >= kU1Cap - kStepMax) {
                soa_pad<kSoaCap>(UB, nUB);
                __syncwarp();
                if (PERIODIC) eval_soa2_p<kSoaCap>(UB, nUB, tA, tB, P.ew, accA, accB, false, true);
                else accB += ACC ? eval_soa_g<kSoaCap>(UB, nUB, TB, grB) : eval_soa<kSoaCap>(UB, nUB, TB);
                evB += (u32)nUB;
                nUB = 0;
            }
            if (nC >= kCCap - kStepMax) {
                if (PERIODIC) eval_c_p(C, Cm, nC, tA, tB, P.ew, accA, accB, evA, evB);
                else if (ACC) eval_c_g(C, Cm, nC, npx, npy, npz, accA, accB, grA, grB, evA, evB);
                else eval_c(C, Cm, nC, npx, npy, npz, accA, accB, evA, evB);
                nC = 0;
            }
            __syncwarp();
        }
    }
    if (COUNT) {
        cAccA = __reduce_add_sync(0xffffffffu, cAccA); cLeafA = __reduce_add_sync(0xffffffffu, cLeafA);
        cOpenA = __reduce_add_sync(0xffffffffu, cOpenA); cExA = __reduce_add_sync(0xffffffffu, cExA);
        cAccB = __reduce_add_sync(0xffffffffu, cAccB); cLeafB = __reduce_add_sync(0xffffffffu, cLeafB);
        cOpenB = __reduce_add_sync(0xffffffffu, cOpenB); cExB = __reduce_add_sync(0xffffffffu, cExB);
        if (lane == 0) {
            P.gcount[gA] = make_uint4(cAccA, cLeafA, cOpenA, cExA);
            if (hasB) P.gcount[gB] = make_uint4(cAccB, cLeafB, cOpenB, cExB);
        }
        return;
    }
    if (nU2 > 0) {
        soa_pad<kSoaCap>(U2, nU2);
        __syncwarp();
        if (PERIODIC) eval_soa2_p<kSoaCap>(U2, nU2, tA, tB, P.ew, accA, accB, true, true);
        else if (ACC) eval_soa2_g<kSoaCap>(U2, nU2, TA, TB, accA, accB, grA, grB);
        else eval_soa2<kSoaCap>(U2, nU2, TA, TB, accA, accB);
    }
    if (nUA > 0) {
        soa_pad<kSoaCap>(UA, nUA);
        __syncwarp();
        if (PERIODIC) eval_soa2_p<kSoaCap>(UA, nUA, tA, tB, P.ew, accA, accB, true, false);
        else accA += ACC ? eval_soa_g<kSoaCap>(UA, nUA, TA, grA) : eval_soa<kSoaCap>(UA, nUA, TA);
    }
    if (nUB > 0) {
        soa_pad<kSoaCap>(UB, nUB);
        __syncwarp();
        if (PERIODIC) eval_soa2_p<kSoaCap>(UB, nUB, tA, tB, P.ew, accA, accB, false, true);
        else accB += ACC ? eval_soa_g<kSoaCap>(UB, nUB, TB, grB) : eval_soa<kSoaCap>(UB, nUB, TB);
    }
    if (nC > 0) {
        if (PERIODIC) eval_c_p(C, Cm, nC, tA, tB, P.ew, accA, accB, evA, evB);
        else if (ACC) eval_c_g(C, Cm, nC, npx, npy, npz, accA, accB, grA, grB, evA, evB);
        else eval_c(C, Cm, nC, npx, npy, npz, accA, accB, evA, evB);
    }
    // the kernel answers for its own lists: entries it evaluated for each group (= accepted + leaf of W6)
    if (lane == 0) {
        P.geval[gA] = evA + (u32)(nU2 + nUA);
        if (hasB) P.geval[gB] = evB + (u32)(nU2 + nUB);
    }
    // ---- a7: Phi_t = -G * sum, written in the original cell order (W-rule 4) ----
    // bh_field: g_t = -grad Phi_t = G * sum w (r_j - r_t)
    if (liveA) {
        const u32 o = sv_idx(P.sv, sA);
        if (!SUBSET || o < P.ntargets) {
            P.phi[o] = P.negG * accA;
            if (ACC) { P.acc[3 * (size_t)o] = -P.negG * grA[0]; P.acc[3 * (size_t)o + 1] = -P.negG * grA[1]; P.acc[3 * (size_t)o + 2] = -P.negG * grA[2]; }
        }
    }
    if (liveB) {
        const u32 o = sv_idx(P.sv, sB);
        if (!SUBSET || o < P.ntargets) {
            P.phi[o] = P.negG * accB;
            if (ACC) { P.acc[3 * (size_t)o] = -P.negG * grB[0]; P.acc[3 * (size_t)o + 1] = -P.negG * grB[1]; P.acc[3 * (size_t)o + 2] = -P.negG * grB[2]; }
        }
    }
}

// ---- BH_OPT_GROUP = 1 (W5): every target walks alone --------------------------------------------
// The textbook per-particle Barnes-Hut: one thread per target, depth-first with a private stack of
// sibling runs (one entry per level), the same fp32 decision (W8) and the same zero-distance rule
// (W3).  A check / comparison mode, not tuned: threads of a warp diverge.
constexpr int kSingleStack = 3 * (kMaxLevel + 2);

__global__ void __launch_bounds__(128)
walk_single_kernel(const WalkParams P)
{
    const i64 s = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P.n) return;
    if (sv_idx(P.sv, s) >= P.ntargets) { P.gcount[s] = make_uint4(0u, 0u, 0u, 0u); P.geval[s] = 0u; return; }
    const float4 tp = __ldg(P.rec + __ldg(P.leaf_slot + s));
    u32 st_first[kSingleStack], st_count[kSingleStack];
    int sp = 0;
    if (P.n >= 2) { st_first[0] = 0u; st_count[0] = 1u; sp = 1; }
    double acc = 0.0;
    float part = 0.f;
    int npart = 0;
    double g[3] = {0.0, 0.0, 0.0};
    float gp[3] = {0.f, 0.f, 0.f};
    u32 c_acc = 0, c_leaf = 0, c_open = 0;
    while (sp > 0) {
        const u32 slot = st_first[sp - 1];
        if (--st_count[sp - 1] == 0u) --sp; else ++st_first[sp - 1];
        const float4 r = __ldg(P.rec + slot);
        const uint4 t = __ldg(reinterpret_cast<const uint4*>(P.aux + slot));
        const float size = __uint_as_float(t.x), delta = __uint_as_float(t.y);
        const u32 first = t.z, count = t.w;
        const float dx = __fsub_rn(tp.x, r.x), dy = __fsub_rn(tp.y, r.y), dz = __fsub_rn(tp.z, r.z);
        const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
        bool use;
        if (count == 0u) {                       // leaf cell: summed unless at zero distance (W3)
            ++c_leaf;
            use = d2 >= 1.17549435e-38f;
        } else {
            float rc = __fmul_rn(size, P.inv_theta);
            if (P.mac == 1) rc = __fadd_rn(rc, delta);
            use = d2 > __fmul_rn(rc, rc);
            if (use) ++c_acc;
            else {
                if (size < __int_as_float(0x7f800000)) ++c_open;
                st_first[sp] = first; st_count[sp] = count; ++sp;
            }
        }
        if (use) {
            const float ri = rsqrt_approx(d2);
            part = __fmaf_rn(r.w, ri, part);
            if (P.acc) {                                   // bh_field: w (r_j - r_t), w = m / d^3
                const float wgt = __fmul_rn(__fmul_rn(r.w, ri), __fmul_rn(ri, ri));
                gp[0] = __fmaf_rn(-dx, wgt, gp[0]); gp[1] = __fmaf_rn(-dy, wgt, gp[1]); gp[2] = __fmaf_rn(-dz, wgt, gp[2]);
            }
            if (++npart == 32) {
                acc += (double)part; part = 0.f; npart = 0;
                g[0] += (double)gp[0]; g[1] += (double)gp[1]; g[2] += (double)gp[2];
                gp[0] = gp[1] = gp[2] = 0.f;
            }
        }
    }
    acc += (double)part;
    const u32 o = sv_idx(P.sv, s);
    if (P.phi) P.phi[o] = P.negG * acc;
    if (P.acc)
        for (int k = 0; k < 3; ++k) P.acc[3 * (size_t)o + k] = -P.negG * (g[k] + (double)gp[k]);
    P.gcount[s] = make_uint4(c_acc, c_leaf, c_open, 0u);
    P.geval[s] = c_acc + c_leaf;
}

// the Phi kernel's own per-group entry counts as plain u32 (bh_last_group_evaluated)
__global__ void __launch_bounds__(256)
group_eval_export_kernel(const u32* __restrict__ geval, i64 ngroups, u32* __restrict__ out)
{
    const i64 g = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (g < ngroups) out[g] = geval[g];
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
per_target_counts_kernel(const uint4* __restrict__ gcount, const SortedView sv, i64 n, int group,
                         u32* __restrict__ out)
{
    const i64 s = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    const uint4 c = gcount[s / group];
    out[sv_idx(sv, s)] = c.x + c.y;
}

// totals[0..3] = sum of the four group counters of the count-only twin; totals[4] = sum over targets of their
// (acc + leaf); totals[5] = the same sum taken from the Phi kernel's own per-group entry counts (geval)
__global__ void __launch_bounds__(256)
group_counts_total_kernel(const uint4* __restrict__ gcount, const u32* __restrict__ geval, i64 ngroups, i64 n,
                          int group, unsigned long long* __restrict__ totals)
{
    unsigned long long t[6] = {0, 0, 0, 0, 0, 0};
    for (i64 g = (i64)blockIdx.x * blockDim.x + threadIdx.x; g < ngroups; g += (i64)gridDim.x * blockDim.x) {
        const uint4 c = gcount[g];
        const i64 members = min((i64)group, n - g * group);
        t[0] += c.x; t[1] += c.y; t[2] += c.z; t[3] += c.w;
        t[4] += (unsigned long long)(c.x + c.y) * (unsigned long long)members;
        t[5] += (unsigned long long)geval[g] * (unsigned long long)members;
    }
    #pragma unroll
    for (int k = 0; k < 6; ++k) {
        #pragma unroll
        for (int o = 16; o > 0; o >>= 1) t[k] += __shfl_xor_sync(0xffffffffu, t[k], o);
        if (lane_id() == 0 && t[k]) atomicAdd(&totals[k], t[k]);
    }
}

}  // namespace bh
