// ewald.cuh -- periodic boundaries (Appendix A).
//
// "In case of periodic boundary conditions, a node's or data cell's contribution to the gravitational
// potential of a data cell changes to phi = G M f_EF(r)" (Eq. A.1), f_EF the Ewald field (Eq. A.2-A.3:
// erf / erfc split of 1/r, short-range sum A_S over the images, long-range sum A_L from the Poisson
// summation formula).  "The Ewald field is calculated once on startup and stored in a large array
// representing a hierarchy of nested grids ... evaluation ... carried out during the respective tree walk
// using quadratic interpolation".  DESIGN.md readings P1-P5:
//   P1  f_EF(r) = psi1(r/L)/L, psi1 the Ewald sum of 1/r in the unit cube with a neutralising background;
//   P2  the array holds the SMOOTH part corr1(u) = psi1(u) - 1/|u| (finite at 0); the walk adds 1/d itself;
//   P3  octant u_a >= 0 (corr1 is even), `nref` grids of N^3 points, spacing h_k = (1/2)/(N-2)/2^k: grid 0
//       reaches one point past the face of the minimum-image cell, grid k refines the corner around u = 0;
//   P4  quadratic through the 3 points per axis around the NEAREST grid point (central differences);
//   P5  minimum-image displacements everywhere; the own cell and zero-distance pairs contribute m corr1(0)/L.
// What differs from the paper's layout: besides the grid values (fp64, kept for bh_ewald_table) the device keeps,
// per grid point, the TEN coefficients of its quadratic in one 32-byte record: value and first differences in fp32,
// the six second differences in fp16 scaled by a power of two (they multiply offsets |t| <= 1/2 twice: their
// rounding stays below 1e-7 of 1/L).  A lookup is ONE 32-byte load of one aligned sector instead of a 19-point
// gather -- the periodic walk is bound by L1 sectors per lookup (profiles/r2_periodic_ncu.md).
#pragma once
#include <cuda_fp16.h>
#include "common.cuh"

namespace bh {

constexpr double kEwaldAlpha = 2.5;     // splitting parameter a = alpha L (the field does not depend on it)
constexpr int kEwaldSeries = 5;         // |n_i|, |h_i| <= 5 ("gpuEwaldSeriesN"): both tails < 1e-13

// corr1 at one point of the octant (fp64).  Real-space and reciprocal sums are written separately; the
// reciprocal sum uses the product form of cos(2 pi h.u) over the eight sign combinations of h.
__device__ inline double ewald_corr1_point(double ux, double uy, double uz)
{
    const double pi = 3.14159265358979323846;
    const double a = kEwaldAlpha;
    const int S = kEwaldSeries;
    const double d0 = sqrt(ux * ux + uy * uy + uz * uz);
    double real = 0.0;
    for (int i = -S; i <= S; ++i)
        for (int j = -S; j <= S; ++j)
            for (int k = -S; k <= S; ++k) {
                if (i == 0 && j == 0 && k == 0) continue;
                const double dx = ux - i, dy = uy - j, dz = uz - k;
                const double d = sqrt(dx * dx + dy * dy + dz * dz);
                real += erfc(a * d) / d;
            }
    // the n = 0 image without its singular part: erfc(a d)/d - 1/d = -erf(a d)/d -> -2a/sqrt(pi)
    real += d0 > 0.0 ? -erf(a * d0) / d0 : -2.0 * a / sqrt(pi);
    double recip = 0.0;
    for (int i = 0; i <= S; ++i)
        for (int j = 0; j <= S; ++j)
            for (int k = 0; k <= S; ++k) {
                const int h2 = i * i + j * j + k * k;
                if (h2 == 0) continue;
                // sum over the sign combinations of (i, j, k): 2^(#nonzero) cos cos cos
                const double mult = (i ? 2.0 : 1.0) * (j ? 2.0 : 1.0) * (k ? 2.0 : 1.0);
                recip += mult * exp(-pi * pi * h2 / (a * a)) / (pi * h2) * cos(2.0 * pi * i * ux) * cos(2.0 * pi * j * uy) *
                         cos(2.0 * pi * k * uz);
            }
    return real + recip - pi / (a * a);
}

// grid values: table[((lev * N + k) * N + j) * N + i] = corr1(i h, j h, k h), h = (1/2)/(N-2)/2^lev
__global__ void __launch_bounds__(128)
ewald_table_kernel(int N, int nref, double* __restrict__ table)
{
    const i64 total = (i64)nref * N * N * N;
    const i64 id = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= total) return;
    const int i = (int)(id % N), j = (int)((id / N) % N), k = (int)((id / ((i64)N * N)) % N);
    const int lev = (int)(id / ((i64)N * N * N));
    const double h = 0.5 / (N - 2) / (double)(1 << lev);
    table[id] = ewald_corr1_point(i * h, j * h, k * h);
}

__device__ __forceinline__ double ewald_tab_at(const double* t, int N, int i, int j, int k)
{
    i = i < 0 ? -i : i; j = j < 0 ? -j : j; k = k < 0 ? -k : k;          // corr1 is even
    return t[((i64)k * N + j) * N + i];
}

// one grid point's quadratic, in grid units d_a = |u_a|/h - i_a:
//   C0 + Dx dx + Dy dy + Dz dz + (hxx dx^2 + hyy dy^2 + hzz dz^2 + hxy dx dy + hxz dx dz + hyz dy dz) / S_lev,
//   hxx = S_lev Dxx/2 etc.; S_lev = s2 * 4^lev with s2 the power of two below 1/h_0^2 (second differences are
//   O(10 h^2): the scaled values sit in fp16's normal range)
struct __align__(32) EwaldRec {
    float c0, dx, dy, dz;
    __half2 hxx_yy, hzz_xy, hxz_yz;
    u32 pad;
};

__host__ __device__ inline float ewald_s2(int N)
{
    float s = 1.f;
    const float lim = 4.f * (float)(N - 2) * (float)(N - 2);          // 1/h_0^2
    while (2.f * s <= lim) s *= 2.f;
    return s;
}

// per grid point (i, j, k <= N - 2) the quadratic around it
__global__ void __launch_bounds__(128)
ewald_coef_kernel(int N, int nref, const double* __restrict__ table, EwaldRec* __restrict__ coef)
{
    const int M = N - 1;
    const i64 total = (i64)nref * M * M * M;
    const i64 id = (i64)blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= total) return;
    const int i = (int)(id % M), j = (int)((id / M) % M), k = (int)((id / ((i64)M * M)) % M);
    const int lev = (int)(id / ((i64)M * M * M));
    const double* t = table + (i64)lev * N * N * N;
    const double C0 = ewald_tab_at(t, N, i, j, k);
    const double xp = ewald_tab_at(t, N, i + 1, j, k), xm = ewald_tab_at(t, N, i - 1, j, k);
    const double yp = ewald_tab_at(t, N, i, j + 1, k), ym = ewald_tab_at(t, N, i, j - 1, k);
    const double zp = ewald_tab_at(t, N, i, j, k + 1), zm = ewald_tab_at(t, N, i, j, k - 1);
    const double Dxy = 0.25 * (ewald_tab_at(t, N, i + 1, j + 1, k) - ewald_tab_at(t, N, i + 1, j - 1, k) -
                               ewald_tab_at(t, N, i - 1, j + 1, k) + ewald_tab_at(t, N, i - 1, j - 1, k));
    const double Dxz = 0.25 * (ewald_tab_at(t, N, i + 1, j, k + 1) - ewald_tab_at(t, N, i + 1, j, k - 1) -
                               ewald_tab_at(t, N, i - 1, j, k + 1) + ewald_tab_at(t, N, i - 1, j, k - 1));
    const double Dyz = 0.25 * (ewald_tab_at(t, N, i, j + 1, k + 1) - ewald_tab_at(t, N, i, j + 1, k - 1) -
                               ewald_tab_at(t, N, i, j - 1, k + 1) + ewald_tab_at(t, N, i, j - 1, k - 1));
    const double S = (double)ewald_s2(N) * (double)(1 << (2 * lev));
    EwaldRec r;
    r.c0 = (float)C0; r.dx = (float)(0.5 * (xp - xm)); r.dy = (float)(0.5 * (yp - ym)); r.dz = (float)(0.5 * (zp - zm));
    r.hxx_yy = __floats2half2_rn((float)(S * 0.5 * (xp - 2.0 * C0 + xm)), (float)(S * 0.5 * (yp - 2.0 * C0 + ym)));
    r.hzz_xy = __floats2half2_rn((float)(S * 0.5 * (zp - 2.0 * C0 + zm)), (float)(S * Dxy));
    r.hxz_yz = __floats2half2_rn((float)(S * Dxz), (float)(S * Dyz));
    r.pad = 0u;
    coef[id] = r;
}

// what the walk needs of the table
struct EwaldTab {
    const EwaldRec* coef; // [nref][M][M][M], M = N - 1
    float s0;             // grid-0 units per unit length: 2 (N - 2) / L
    float invL;
    float L;
    float top;            // (float)(N - 2): the largest nearest-point index
    int M, MM, M3;        // M = N - 1 and its powers
    int nref;
    float inv_s2;         // 1 / ewald_s2(N)
    int ktop;             // bit pattern of 1.5 * 2^23 + (N - 2): the clamp of the nearest-point index
    u32 cbias;            // bits(1.5 * 2^23) * (M^2 + M + 1) mod 2^32
};

// corr1(r/L) for a minimum-image displacement (dx, dy, dz), |d_a| <= L/2 (+ rounding), fp32; the caller divides by L.
// NESTED = false: one grid (nref = 1, the default) -- the level selection is compiled out (as predicated
// instructions it cost a fifth of the lookup's issue slots).
template <bool NESTED>
__device__ __forceinline__ float ewald_corr(const EwaldTab& T, float dx, float dy, float dz)
{
    float s = T.s0, inv_s = T.inv_s2;
    u32 off = T.cbias;
    if (NESTED) {
        // finest grid with max_a |u_a| 2^lev <= N - 2: floor(log2(top / m)) from the difference of the bit patterns
        const float m = fmaxf(fmaxf(fabsf(dx), fabsf(dy)), fmaxf(fabsf(dz), 1.0e-30f)) * T.s0;
        const int e = (int)(__float_as_uint(T.top) - __float_as_uint(m)) >> 23;
        const int lev = min(T.nref - 1, max(e, 0));
        s *= __int_as_float((127 + lev) << 23);
        inv_s *= __int_as_float((127 - 2 * lev) << 23);
        off -= (u32)lev * (u32)T.M3;
    }
    // nearest grid point without the conversion pipe: x + 1.5 * 2^23 rounds x to the nearest (even on ties) integer for
    // 0 <= x < 2^22 and leaves it in the low mantissa bits; the offset from that point comes out of one fma (no
    // rounding of |d| s in between).
    // No clamp: |d_a| s <= (N - 2)(1 + a few ulp) rounds to at most N - 2, the last point that has a record.
    const float big = 12582912.f;
    const int bx = (int)__float_as_uint(__fmaf_rn(fabsf(dx), s, big));
    const int by = (int)__float_as_uint(__fmaf_rn(fabsf(dy), s, big));
    const int bz = (int)__float_as_uint(__fmaf_rn(fabsf(dz), s, big));
    BH_DCHECK(bx <= T.ktop && by <= T.ktop && bz <= T.ktop);
    const float tx = __fmaf_rn(fabsf(dx), s, big - __uint_as_float((u32)bx));
    const float ty = __fmaf_rn(fabsf(dy), s, big - __uint_as_float((u32)by));
    const float tz = __fmaf_rn(fabsf(dz), s, big - __uint_as_float((u32)bz));
    // the index in wrapping u32 arithmetic: cbias = bits(big) * (M^2 + M + 1) takes the three exponent fields out
    const u32 idx = (u32)bz * (u32)T.MM + ((u32)by * (u32)T.M + ((u32)bx - off));
    u32 w0, w1, w2, w3, w4, w5, w6;
    [[maybe_unused]] u32 w7;                            // the record's padding word
    asm("ld.global.nc.v8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
        : "=r"(w0), "=r"(w1), "=r"(w2), "=r"(w3), "=r"(w4), "=r"(w5), "=r"(w6), "=r"(w7) : "l"(T.coef + idx));
    const float2 xxyy = __half22float2(*reinterpret_cast<const __half2*>(&w4));
    const float2 zzxy = __half22float2(*reinterpret_cast<const __half2*>(&w5));
    const float2 xzyz = __half22float2(*reinterpret_cast<const __half2*>(&w6));
    // explicit fmas: the same bits whatever the compiler would contract (the checked build must agree, test_gpu_checked)
    const float qx = __fmaf_rn(xzyz.x, tz, __fmaf_rn(zzxy.y, ty, xxyy.x * tx));
    const float qy = __fmaf_rn(xzyz.y, tz, xxyy.y * ty);
    const float q = __fmaf_rn(tx, qx, __fmaf_rn(ty, qy, tz * (zzxy.x * tz)));
    const float lin = __fmaf_rn(tz, __uint_as_float(w3), __fmaf_rn(ty, __uint_as_float(w2), __fmaf_rn(tx, __uint_as_float(w1), __uint_as_float(w0))));
    return __fmaf_rn(q, inv_s, lin);
}

// minimum image of a displacement, fp32: d - L rint(d / L)
// rint(v) for |v| < 2^22 on the FMA pipe (1.5 * 2^23 trick) instead of FRND on the conversion pipe
__device__ __forceinline__ float rint_magic(float v) { return (v + 12582912.f) - 12582912.f; }

__device__ __forceinline__ float wrap_mi(float d, float L, float invL) { return __fmaf_rn(-L, rint_magic(d * invL), d); }

// n = 1 under periodic boundaries: the lone cell still feels its own images, Phi = -G m corr1(0)/L
__global__ void periodic_single_kernel(const double4* __restrict__ rec64, const double* __restrict__ table, double L,
                                       double negG, double* __restrict__ phi)
{
    phi[0] = negG * rec64[0].w * table[0] / L;
}

}  // namespace bh
