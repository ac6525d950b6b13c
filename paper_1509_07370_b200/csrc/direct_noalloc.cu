// direct_noalloc.cu -- bh_direct_noalloc: the direct sum of Eq. 2 for callers that cannot allocate
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// bh_potential_direct (bh.cu / direct.cuh) sums over a packed fp64 copy of the cells -- one double4 (x, y, z, m) per
// cell -- that it allocates in its context on first use.  This variant keeps that packed copy in a FILE-SCOPE
// `static __device__` array of BH_NOALLOC_MAX_N records (1 MiB; every GPU that loads libbh holds it until the
// process exits) and takes everything else from the caller.  It calls no cudaMalloc / cudaFree and no library
// routine that allocates; it creates no context, stream or event.
//
// The array's name in HOST code is a host-side stand-in, not a device address: the kernels get the address that
// cudaGetSymbolAddress returns, looked up once per device with that device current (noalloc_scratch below).
//
// Sharing: every call on a device uses the same array.  Nothing in it has to start at zero -- the pack kernel
// overwrites records [0, n) before the sum kernel of the same call reads exactly those; records at and beyond n keep
// an earlier call's contents and are never read.  Two calls that overlap on the GPU (different streams, or
// different host threads without ordering between their streams) RACE on the array: the caller orders them.
//
// This file shares nothing with the context code path of bh.cu: its own kernels, no context, no DevBuf.
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>

#include <mutex>

#include "../../include/bh.h"

namespace {

constexpr int kNaThreads = 128;      // targets per CTA
constexpr int kNaTile = 256;         // sources staged in shared memory at a time
constexpr int kNaMaxDevices = 64;

// the scratch: packed (x, y, z, m) of the cells of the call in flight, original order
static __device__ __align__(256) double4 g_noalloc_scratch[BH_NOALLOC_MAX_N];

thread_local char t_msg[256] = "";

std::mutex s_mu;
double4* s_scratch_ptr[kNaMaxDevices] = {};    // device address of g_noalloc_scratch, per device ordinal

__global__ void __launch_bounds__(256)
noalloc_pack_kernel(const double* __restrict__ x, const double* __restrict__ y, const double* __restrict__ z,
                    const double* __restrict__ m, int n, double4* __restrict__ rec)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) rec[i] = make_double4(x[i], y[i], z[i], m[i]);
}

// Phi_i = -G sum_{j != i} m_j / |r_i - r_j| in fp64; the self term is skipped by index identity, distinct cells
// at zero distance are skipped (W3) -- the rules of direct_kernel (direct.cuh), sources in original order.
__global__ void __launch_bounds__(kNaThreads)
noalloc_direct_kernel(const double4* __restrict__ rec, int n, double negG, double* __restrict__ phi)
{
    __shared__ double4 tile[kNaTile];
    const int i = blockIdx.x * kNaThreads + threadIdx.x;
    double px = 0.0, py = 0.0, pz = 0.0;
    if (i < n) { const double4 p = rec[i]; px = p.x; py = p.y; pz = p.z; }
    double acc = 0.0;
    for (int base = 0; base < n; base += kNaTile) {
        const int cnt = n - base < kNaTile ? n - base : kNaTile;
        __syncthreads();
        for (int t = threadIdx.x; t < cnt; t += kNaThreads) tile[t] = rec[base + t];
        __syncthreads();
        #pragma unroll 4
        for (int t = 0; t < cnt; ++t) {
            const double4 q = tile[t];
            const double dx = px - q.x, dy = py - q.y, dz = pz - q.z;
            const double d2 = dx * dx + dy * dy + dz * dz;
            if (base + t != i && d2 != 0.0) acc += q.w / sqrt(d2);
        }
    }
    if (i < n) phi[i] = negG * acc;
}

int fail_cuda(const char* where, cudaError_t e)
{
    snprintf(t_msg, sizeof(t_msg), "%s: %s", where, cudaGetErrorString(e));
    return BH_ERR_CUDA;
}

// set-up, once per device, with that device current: the device address of the static array
int noalloc_scratch(int device, double4** out)
{
    std::lock_guard<std::mutex> lock(s_mu);
    if (!s_scratch_ptr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess) return fail_cuda("cudaGetSymbolAddress(g_noalloc_scratch)", e);
        if (!p) { snprintf(t_msg, sizeof(t_msg), "cudaGetSymbolAddress returned a null address"); return BH_ERR_CUDA; }
        s_scratch_ptr[device] = static_cast<double4*>(p);
    }
    *out = s_scratch_ptr[device];
    return BH_OK;
}

int run(int device, cudaStream_t st, const double* x, const double* y, const double* z, const double* m, int n,
        double G, double* phi)
{
    double4* rec = nullptr;
    const int rc = noalloc_scratch(device, &rec);
    if (rc != BH_OK) return rc;
    noalloc_pack_kernel<<<(n + 255) / 256, 256, 0, st>>>(x, y, z, m, n, rec);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda("noalloc_pack_kernel", e);
    noalloc_direct_kernel<<<(n + kNaThreads - 1) / kNaThreads, kNaThreads, 0, st>>>(rec, n, -G, phi);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_cuda("noalloc_direct_kernel", e);
    return BH_OK;
}

}  // namespace

extern "C" {

const char* bh_noalloc_last_error(void) { return t_msg; }

int bh_direct_noalloc(int device, void* cuda_stream, const double* x, const double* y, const double* z, const double* m,
                      int64_t n, double G, double* phi)
{
    t_msg[0] = 0;
    if (device < 0 || device >= kNaMaxDevices || n < 0 || G != G) {
        snprintf(t_msg, sizeof(t_msg), "bh_direct_noalloc: bad device, negative n or NaN G");
        return BH_ERR_INVALID_ARG;
    }
    if (n > (int64_t)BH_NOALLOC_MAX_N) {
        snprintf(t_msg, sizeof(t_msg), "bh_direct_noalloc: n = %lld exceeds BH_NOALLOC_MAX_N = %d (the size of the static "
                 "scratch array); use bh_build + bh_potential_direct", (long long)n, (int)BH_NOALLOC_MAX_N);
        return BH_ERR_TOO_LARGE;
    }
    if (n == 0) return BH_OK;
    if (!x || !y || !z || !m || !phi) {
        snprintf(t_msg, sizeof(t_msg), "bh_direct_noalloc: null pointer");
        return BH_ERR_INVALID_ARG;
    }
    int prev = -1;
    cudaError_t e = cudaGetDevice(&prev);
    if (e != cudaSuccess) return fail_cuda("cudaGetDevice", e);
    if (prev != device && (e = cudaSetDevice(device)) != cudaSuccess) return fail_cuda("cudaSetDevice", e);
    const int rc = run(device, static_cast<cudaStream_t>(cuda_stream), x, y, z, m, (int)n, G, phi);
    if (prev != device) cudaSetDevice(prev);
    return rc;
}

}  // extern "C"
