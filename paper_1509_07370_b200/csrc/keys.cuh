// keys.cuh -- step a1: 63-bit Morton keys of the cells inside the caller's cube.
// The paper only names the Morton curve; the exact expression is DESIGN.md K1-K2:
//   s = 2^21 / L (fp64, computed once on the host);  t = (v - v0) * s as one fp64 subtract and one
//   fp64 multiply (round-to-nearest, NO fma contraction);  q = floor(t) clamped to [0, 2^21-1]
//   (NaN -> 0);  key bit 3k+0/1/2 = bit k of qx/qy/qz.
// The permutation starts as the identity and is never stored: the first sort pass uses the element index.
// HBM-bound stream: 24 B read + 8 B written per cell.
#pragma once
#include "common.cuh"

namespace bh {

struct KeyReduce {      // device-resident reduction results of the key pass
    u64 key_or;
    u64 key_and;
    u64 n_clamped;
};

__device__ __forceinline__ u64 spread21(u32 v)
{
    u64 x = v & 0x1fffffu;
    x = (x | (x << 32)) & 0x001f00000000ffffULL;
    x = (x | (x << 16)) & 0x001f0000ff0000ffULL;
    x = (x | (x << 8)) & 0x100f00f00f00f00fULL;
    x = (x | (x << 4)) & 0x10c30c30c30c30c3ULL;
    x = (x | (x << 2)) & 0x1249249249249249ULL;
    return x;
}

__device__ __forceinline__ u32 quantise(double v, double v0, double s, u32& clamped)
{
    double t = __dmul_rn(__dsub_rn(v, v0), s);   // K1: no contraction, no reassociation
    double f = floor(t);
    if (!(f >= 0.0)) { clamped = 1; return 0u; }            // negative or NaN
    if (f > 2097151.0) { clamped = 1; return 2097151u; }
    return (u32)f;
}

__device__ __forceinline__ u64 morton_key(double x, double y, double z, double x0, double y0, double z0,
                                          double s, u32& clamped)
{
    u32 qx = quantise(x, x0, s, clamped);
    u32 qy = quantise(y, y0, s, clamped);
    u32 qz = quantise(z, z0, s, clamped);
    return spread21(qx) | (spread21(qy) << 1) | (spread21(qz) << 2);
}

// Persistent grid-stride kernel; VEC = 2 uses 16-byte loads/stores (needs 16 B aligned inputs).
template <int VEC>
__global__ void __launch_bounds__(256)
morton_keys_kernel(const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
                   i64 n, double x0, double y0, double z0, double s,
                   u64* __restrict__ keys, KeyReduce* __restrict__ red)
{
    chain_enter();
    u64 k_or = 0, k_and = ~0ULL;
    u32 n_cl = 0;
    const i64 stride = (i64)gridDim.x * blockDim.x;
    if (VEC == 2) {
        const i64 nv = n >> 1;
        for (i64 v = (i64)blockIdx.x * blockDim.x + threadIdx.x; v < nv; v += stride) {
            double2 xx = ld_stream(reinterpret_cast<const double2*>(x) + v);
            double2 yy = ld_stream(reinterpret_cast<const double2*>(y) + v);
            double2 zz = ld_stream(reinterpret_cast<const double2*>(z) + v);
            u32 c0 = 0, c1 = 0;
            u64 ka = morton_key(xx.x, yy.x, zz.x, x0, y0, z0, s, c0);
            u64 kb = morton_key(xx.y, yy.y, zz.y, x0, y0, z0, s, c1);
            reinterpret_cast<ulonglong2*>(keys)[v] = make_ulonglong2(ka, kb);
            k_or |= ka | kb;
            k_and &= ka & kb;
            n_cl += c0 + c1;
        }
        if ((n & 1) && blockIdx.x == 0 && threadIdx.x == 0) {   // odd tail
            u32 c0 = 0;
            u64 ka = morton_key(x[n - 1], y[n - 1], z[n - 1], x0, y0, z0, s, c0);
            keys[n - 1] = ka;
            k_or |= ka; k_and &= ka; n_cl += c0;
        }
    } else {
        for (i64 i = (i64)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
            u32 c0 = 0;
            u64 ka = morton_key(x[i], y[i], z[i], x0, y0, z0, s, c0);
            keys[i] = ka;
            k_or |= ka; k_and &= ka; n_cl += c0;
        }
    }
    // warp then block reduction, one set of atomics per block
    #pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        k_or |= __shfl_xor_sync(0xffffffffu, k_or, o);
        k_and &= __shfl_xor_sync(0xffffffffu, k_and, o);
        n_cl += __shfl_xor_sync(0xffffffffu, n_cl, o);
    }
    __shared__ u64 s_or[8], s_and[8];
    __shared__ u32 s_cl[8];
    const int w = threadIdx.x >> 5;
    if (lane_id() == 0) { s_or[w] = k_or; s_and[w] = k_and; s_cl[w] = n_cl; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int i = 1; i < (int)(blockDim.x >> 5); ++i) { k_or |= s_or[i]; k_and &= s_and[i]; n_cl += s_cl[i]; }
        atomicOr(&red->key_or, k_or);
        atomicAnd(&red->key_and, k_and);
        if (n_cl) atomicAdd(&red->n_clamped, (u64)n_cl);
    }
}

}  // namespace bh
