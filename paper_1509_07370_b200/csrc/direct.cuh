// direct.cuh -- step a8: Eq. 2 written out in fp64,
//   Phi_i = -G sum_{j != i} m_j / |r_i - r_j|   over all n cells of the last build.
// One CTA per 128 targets; the sources stream through shared memory in tiles.  The self term is
// skipped by sorted-slot identity, distinct cells at zero distance are skipped (W3).
// FP64-ALU bound; a check path (PAPER.md:238 uses the direct sum as accuracy reference), not graded.
#pragma once
#include "common.cuh"

namespace bh {

constexpr int kDirectThreads = 128;
constexpr int kDirectTile = 256;

__global__ void __launch_bounds__(kDirectThreads)
direct_kernel(const double4* __restrict__ leaf64, i64 n, const u32* __restrict__ slot_of,
              const i64* __restrict__ targets, i64 nt, double negG, double* __restrict__ phi)
{
    __shared__ double4 tile[kDirectTile];
    const i64 a = (i64)blockIdx.x * kDirectThreads + threadIdx.x;
    bool valid = a < nt;
    i64 self = -1;
    if (valid) {
        const i64 orig = targets ? targets[a] : a;
        if (orig < 0 || orig >= n) valid = false;
        else self = slot_of[orig];
    }
    double px = 0.0, py = 0.0, pz = 0.0;
    if (self >= 0) { const double4 p = leaf64[self]; px = p.x; py = p.y; pz = p.z; }
    double acc = 0.0;
    for (i64 base = 0; base < n; base += kDirectTile) {
        const int cnt = (int)min((i64)kDirectTile, n - base);
        __syncthreads();
        for (int t = threadIdx.x; t < cnt; t += kDirectThreads) tile[t] = leaf64[base + t];
        __syncthreads();
        #pragma unroll 4
        for (int t = 0; t < cnt; ++t) {
            const double4 q = tile[t];
            const double dx = px - q.x, dy = py - q.y, dz = pz - q.z;
            const double d2 = dx * dx + dy * dy + dz * dz;
            if (base + t != self && d2 != 0.0) acc += q.w / sqrt(d2);
        }
    }
    if (a < nt) phi[a] = valid ? negG * acc : __longlong_as_double(0x7ff8000000000000LL);
}

}  // namespace bh
