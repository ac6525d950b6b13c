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
// What differs from the paper's layout: besides the grid values (fp64, kept for bh_export of the table) the
// device keeps, per grid point, the TEN coefficients of its quadratic in fp32 (three float4): a lookup is three
// 16-byte loads from one 48-byte record and nine FMAs instead of a 19-point gather.
#pragma once
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

// per grid point (i, j, k <= N - 2) the quadratic around it, in grid units d_a = |u_a|/h - i_a:
//   c0 = (C0, Dx, Dy, Dz), c1 = (Dxx/2, Dyy/2, Dzz/2, Dxy), c2 = (Dxz, Dyz, 0, 0)
__global__ void __launch_bounds__(128)
ewald_coef_kernel(int N, int nref, const double* __restrict__ table, float4* __restrict__ coef)
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
    coef[3 * id + 0] = make_float4((float)C0, (float)(0.5 * (xp - xm)), (float)(0.5 * (yp - ym)), (float)(0.5 * (zp - zm)));
    coef[3 * id + 1] = make_float4((float)(0.5 * (xp - 2.0 * C0 + xm)), (float)(0.5 * (yp - 2.0 * C0 + ym)),
                                   (float)(0.5 * (zp - 2.0 * C0 + zm)), (float)Dxy);
    coef[3 * id + 2] = make_float4((float)Dxz, (float)Dyz, 0.f, 0.f);
}

// what the walk needs of the table
struct EwaldTab {
    const float4* coef;   // [nref][M][M][M][3], M = N - 1
    float s0;             // grid-0 units per unit length: 2 (N - 2) / L
    float invL;
    float L;
    float top;            // (float)(N - 2): the largest nearest-point index
    int M;
    int nref;
};

// corr1(r/L)/L for a minimum-image displacement (dx, dy, dz), |d_a| <= L/2 (+ rounding), fp32
__device__ __forceinline__ float ewald_corr(const EwaldTab& T, float dx, float dy, float dz)
{
    float ax = fabsf(dx) * T.s0, ay = fabsf(dy) * T.s0, az = fabsf(dz) * T.s0;
    int lev = 0;
    if (T.nref > 1) {
        // finest grid with max_a |u_a| 2^lev <= N - 2: floor(log2(top / m)) from the difference of the bit patterns
        const float m = fmaxf(fmaxf(ax, ay), fmaxf(az, 1.0e-30f));
        const int e = (int)(__float_as_uint(T.top) - __float_as_uint(m)) >> 23;
        lev = min(T.nref - 1, max(e, 0));
        const float sc = __int_as_float((127 + lev) << 23);
        ax *= sc; ay *= sc; az *= sc;
    }
    const float fx = fminf(rintf(ax), T.top), fy = fminf(rintf(ay), T.top), fz = fminf(rintf(az), T.top);
    const float tx = ax - fx, ty = ay - fy, tz = az - fz;
    const int idx = ((lev * T.M + (int)fz) * T.M + (int)fy) * T.M + (int)fx;
    const float4 c0 = __ldg(T.coef + 3 * idx), c1 = __ldg(T.coef + 3 * idx + 1), c2 = __ldg(T.coef + 3 * idx + 2);
    const float v = c0.x + tx * (c0.y + tx * c1.x + ty * c1.w + tz * c2.x) + ty * (c0.z + ty * c1.y + tz * c2.y) +
                    tz * (c0.w + tz * c1.z);
    return v * T.invL;
}

// minimum image of a displacement, fp32: d - L rint(d / L)
__device__ __forceinline__ float wrap_mi(float d, float L, float invL) { return __fmaf_rn(-L, rintf(d * invL), d); }

// n = 1 under periodic boundaries: the lone cell still feels its own images, Phi = -G m corr1(0)/L
__global__ void periodic_single_kernel(const double4* __restrict__ rec64, const double* __restrict__ table, double L,
                                       double negG, double* __restrict__ phi)
{
    phi[0] = negG * rec64[0].w * table[0] / L;
}

}  // namespace bh
