// bh.cu -- host side of libbh: the C ABI declared in include/bh.h.
// Every step of the path runs in the kernels of keys.cuh / sort.cuh / scan.cuh / tree.cuh /
// walk.cuh / direct.cuh; this file owns buffers, launches and the two scalar read-backs of bh_build.
#include "../../include/bh.h"

#include <math.h>
#include <new>
#include <stdio.h>
#include <string.h>

#include "common.cuh"
#include "direct.cuh"
#include "ewald.cuh"
#include "keys.cuh"
#include "let.cuh"
#include "scan.cuh"
#include "sort.cuh"
#include "tree.cuh"
#include "walk.cuh"

using namespace bh;

namespace {

struct DevBuf {                 // grow-only device buffer
    void* p = nullptr;
    size_t cap = 0;
    cudaError_t ensure(size_t bytes)
    {
        if (bytes <= cap) return cudaSuccess;
        if (p) { cudaError_t e = cudaFree(p); p = nullptr; cap = 0; if (e != cudaSuccess) return e; }
        size_t want = bytes + bytes / 16 + 256;
        cudaError_t e = cudaMalloc(&p, want);
        if (e != cudaSuccess) { p = nullptr; return e; }
        cap = want;
        return cudaSuccess;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
    template <typename T> T* as() const { return reinterpret_cast<T*>(p); }
};

struct DeviceScalars {          // small device-resident results read back by the host
    KeyReduce keyred;
    u32 topo_rows[kTopoDigits + 1];   // row starts of the scanned level histogram + grand total (filled in the host mirror only:
                                      // topo_totals_kernel writes them there itself)
    u32 scan_total;
    u32 max_bucket;
    u32 spec_ok;                      // gate of the kernels enqueued on speculated level totals (topo_totals_kernel)
    unsigned long long totals[6];     // sums of the four twin counters, twin interactions, the Phi kernel's own interactions
};

enum { EV_B0, EV_KEYS, EV_SORT, EV_PERM, EV_TOPO, EV_MOM, EV_W0, EV_W1,
       EV_H0, EV_HC0, EV_HXYZ, EV_HM, EV_HD0, EV_HD1, EV_HEND, EV_COUNT };   // EV_H*: bh_solve_host


}  // namespace

struct bh_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    int mac = BH_MAC_BH86;
    int group = 32;
    bool built = false;
    bool walked = false;
    int walk_group = 32;
    bool periodic = false;                // BH_OPT_PERIODIC: the cube of the build is a periodic box (App. A)
    bool walk_periodic = false;           // ... of the last walk (the count pass repeats it)
    int ew_N = 66, ew_nref = 1;           // BH_OPT_EWALD_N / _NREF: points per axis and nested grids of the field array
    int ew_ready_N = 0, ew_ready_nref = 0;
    DevBuf ew_table, ew_coef;             // grid values (fp64) and per-point quadratic records (EwaldRec)
    bool counts_valid = false;            // gcount holds the counters of the last walk
    double walk_theta = 0.0;              // arguments of the last bh_potential (the count pass repeats its walk)
    int walk_mac = BH_MAC_BH86;
    char cuda_msg[256] = {0};

    // problem
    i64 n = 0, nn = 0, nslots = 0;
    int depth = 0, maxlevel = 0, sort_passes = 0;
    i64 n_clamped = 0, max_bucket = 1;
    double cube[4] = {0, 0, 0, 1};
    TopoLevels lv = {};                   // canonical-id and slot bases per level

    // per cell
    DevBuf keysA, keysB, idxA, idxB;      // ping-pong (key, index)
    SortedView sv = {};                   // the sorted cells as the sort left them (packed / generic / identity)
    DevBuf clev, leaf_slot;               // c(s); slot of sorted cell s
    DevBuf leaf64, slot_of;               // bh_potential_direct's own copies (built on its first call)
    bool direct_ready = false;
    // sort / scan scratch
    DevBuf hist, scan_scratch;
    // per node (canonical order)
    DevBuf nlo, nfirst, node_slot, delta64;
    // per slot
    DevBuf rec64, rec, aux;
    KeyReduce plan_hint = {};             // key OR / AND of the last build: the next build sorts on them
    bool plan_hint_valid = false;         // without waiting for its own (checked at the second read-back)
    u32 rows_hint[kTopoDigits + 1] = {0}; // level totals (scanned row starts) of the last build: the next build of as
    i64 rows_hint_n = -1;                 // many cells enqueues assign + moments on them before its own arrive
    i64 aux_dirty_nn = -1;                // aux is zero except on node_slot[0, aux_dirty_nn); -1: unknown, clear all
    // walk
    i64 ntargets = -1;                    // bh_set_num_targets: cells [0, ntargets) are targets; -1 = all
    DevBuf ess_state, ess_emit;           // bh_essential_nodes: per-slot flags
    DevBuf gcount;                        // W6 counters of the count-only twin (lazy)
    DevBuf geval;                         // list entries the Phi kernel itself evaluated, per group
    DevBuf scalars;                       // DeviceScalars
    DeviceScalars* h_scalars = nullptr;   // pinned host mirror
    DevBuf stage[4];                      // bh_solve_host staging (x, y, z, m) and phi
    DevBuf stage_phi;
    cudaStream_t copy_stream = nullptr;   // bh_solve_host: the host->device copies run beside the build
    cudaEvent_t assign_wait = nullptr;    // set by bh_solve_host: the masses land after the positions; the first kernel
                                          // that reads m (the assigning kernel) waits for this event
    bool host_timed = false;

    cudaEvent_t ev[EV_COUNT] = {nullptr};
    bool ev_build = false, ev_walk = false;
    bool ev_phases = false;               // the per-phase events of the last build were recorded (BH_OPT_PASS_TIMING)
    int launches_build = 0, launches_walk = 0;

    // BH_OPT_PASS_TIMING: one event after every kernel of bh_build (a reporting mode: the events add gaps)
    bool pass_timing = false;
    static constexpr int kMaxPasses = 96;
    cudaEvent_t pev[kMaxPasses] = {nullptr};
    char pname[kMaxPasses][24];
    double pbytes[kMaxPasses];
    int npass = 0;
};

namespace {

int cuda_fail(bh_ctx* c, cudaError_t e, const char* where)
{
    if (c) snprintf(c->cuda_msg, sizeof(c->cuda_msg), "%.160s: %.80s", where, cudaGetErrorString(e));
    cudaGetLastError();   // clear sticky-free errors
    return e == cudaErrorMemoryAllocation ? BH_ERR_OOM : BH_ERR_CUDA;
}

#define BH_CUDA(call)                                                    \
    do {                                                                 \
        cudaError_t e__ = (call);                                        \
        if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call);       \
    } while (0)

// per-pass timing: closes the pass `name` (everything enqueued since the previous mark) with an event
void pass_mark(bh_ctx* ctx, const char* name, double alg_bytes)
{
    if (!ctx->pass_timing || ctx->npass >= bh_ctx::kMaxPasses) return;
    const int k = ctx->npass;
    if (!ctx->pev[k] && cudaEventCreate(&ctx->pev[k]) != cudaSuccess) { cudaGetLastError(); return; }
    snprintf(ctx->pname[k], sizeof(ctx->pname[k]), "%s", name);
    ctx->pbytes[k] = alg_bytes;
    cudaEventRecord(ctx->pev[k], ctx->stream);
    ctx->npass = k + 1;
}

inline unsigned blocks_for(i64 n, int threads) { return (unsigned)((n + threads - 1) / threads); }

bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

int persistent_grid(const bh_ctx* ctx, int per_sm)
{
    int sms = 148;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ctx->device);
    return sms * per_sm;
}


// a5: moments of every level, deepest first; runs of small levels share one single-block launch
int launch_moments(bh_ctx* ctx, const u32* gate = nullptr)
{
    cudaStream_t st = ctx->stream;
    DeviceScalars* ds = ctx->scalars.as<DeviceScalars>();
    MomentArgs MA;
    MA.sv = ctx->sv; MA.nlo = ctx->nlo.as<u32>(); MA.nfirst = ctx->nfirst.as<u32>();
    MA.node_slot = ctx->node_slot.as<u32>(); MA.rec64 = ctx->rec64.as<double4>();
    MA.delta64 = ctx->delta64.as<double>(); MA.rec = ctx->rec.as<float4>(); MA.aux = ctx->aux.as<WalkAux>();
    MA.max_bucket = &ds->max_bucket;
    MA.x0 = ctx->cube[0]; MA.y0 = ctx->cube[1]; MA.z0 = ctx->cube[2]; MA.L = ctx->cube[3];
    MA.gate = gate;
    SmallLevels sl;
    sl.nlev = 0;
    double small_bytes = 0.0;
    for (int l = ctx->maxlevel; l >= -1; --l) {
        const i64 b0 = l >= 0 ? ctx->lv.node_base[l] : 0, b1 = l >= 0 ? ctx->lv.node_base[l + 1] : 0;
        const bool small = l >= 0 && b1 - b0 <= kSmallLevelNodes;
        // 32 B per leaf cell read + 72 B per node (fp64 moments + packed record); the children
        // of level l are the level-(l+1) entities, of which the level-(l+1) nodes are not leaf cells
        double lvl_bytes = 0.0;
        if (l >= 0) {
            const double kids = (double)ctx->lv.slot_base[l + 2] - (double)ctx->lv.slot_base[l + 1];
            const double inner = l + 1 < kNumLevels ? (double)ctx->lv.node_base[l + 2] - (double)ctx->lv.node_base[l + 1] : 0.0;
            lvl_bytes = 32.0 * (kids - inner) + 72.0 * (double)(b1 - b0);
        }
        if ((!small || l < 0) && sl.nlev > 0) {          // flush the pending run of small levels
            BH_CUDA(launch_chain(moments_small_kernel, dim3(1), dim3(kMomSmallThreads), 0, st, sl, MA));
            ctx->launches_build += 1;
            char nm[24];
            snprintf(nm, sizeof(nm), "moments_L%d-%d", sl.level[sl.nlev - 1], sl.level[0]);
            pass_mark(ctx, nm, small_bytes);
            small_bytes = 0.0;
            sl.nlev = 0;
        }
        if (l < 0 || b1 == b0) continue;
        if (small) {
            sl.level[sl.nlev] = l; sl.b0[sl.nlev] = (u32)b0; sl.b1[sl.nlev] = (u32)b1;
            sl.slot_end[sl.nlev] = ctx->lv.slot_base[l + 2];
            ++sl.nlev;
            small_bytes += lvl_bytes;
        } else {
            BH_CUDA(launch_chain(moments_kernel, dim3(blocks_for(b1 - b0, 128)), dim3(128), 0, st, b0, b1, l,
                                 ctx->lv.slot_base[l + 2], MA));
            ctx->launches_build += 1;
            char nm[24];
            snprintf(nm, sizeof(nm), "moments_L%d", l);
            pass_mark(ctx, nm, lvl_bytes);
        }
    }
    return BH_OK;
}

}  // namespace

extern "C" {

const char* bh_strerror(int code)
{
    switch (code) {
        case BH_OK: return "ok";
        case BH_ERR_INVALID_ARG: return "invalid argument";
        case BH_ERR_NOT_BUILT: return "no tree: call bh_build first";
        case BH_ERR_CUDA: return "CUDA runtime error (see bh_last_cuda_error)";
        case BH_ERR_OOM: return "out of memory";
        case BH_ERR_TOO_LARGE: return "problem too large for this call";
        default: return "unknown error code";
    }
}

const char* bh_last_cuda_error(const bh_ctx* ctx) { return ctx ? ctx->cuda_msg : ""; }

int bh_create(bh_ctx** out, int device, void* cuda_stream)
{
    if (!out) return BH_ERR_INVALID_ARG;
    *out = nullptr;
    int count = 0;
    cudaError_t e = cudaGetDeviceCount(&count);
    if (e != cudaSuccess) { cudaGetLastError(); return BH_ERR_CUDA; }   // no CPU fallback
    if (device < 0 || device >= count) return BH_ERR_INVALID_ARG;
    bh_ctx* ctx = new (std::nothrow) bh_ctx;
    if (!ctx) return BH_ERR_OOM;
    ctx->device = device;
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    int rc = BH_OK;
    do {
        if ((e = cudaSetDevice(device)) != cudaSuccess) { rc = cuda_fail(ctx, e, "cudaSetDevice"); break; }
        int major = 0;
        cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, device);
        if (major != 10) {
            snprintf(ctx->cuda_msg, sizeof(ctx->cuda_msg), "device %d is sm_%d0; libbh is built for sm_100a only",
                     device, major);
            rc = BH_ERR_CUDA;
            break;
        }
        for (int i = 0; i < EV_COUNT; ++i)
            if ((e = cudaEventCreate(&ctx->ev[i])) != cudaSuccess) { rc = cuda_fail(ctx, e, "cudaEventCreate"); break; }
        if (rc) break;
        if ((e = cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking)) != cudaSuccess) { rc = cuda_fail(ctx, e, "cudaStreamCreate"); break; }
        if ((e = ctx->scalars.ensure(sizeof(DeviceScalars))) != cudaSuccess) { rc = cuda_fail(ctx, e, "cudaMalloc"); break; }
        if ((e = cudaMallocHost(&ctx->h_scalars, sizeof(DeviceScalars))) != cudaSuccess) { rc = cuda_fail(ctx, e, "cudaMallocHost"); break; }
        // kernels whose dynamic shared memory exceeds the 48 KB default
        const int walk_smem = 227 * 1024;
        const struct { const void* fn; int bytes; const char* what; } big_smem[] = {
            {(const void*)radix_onesweep_kernel<kGenericFirst>, (int)sort_smem_bytes(false), "sort"},
            {(const void*)radix_onesweep_kernel<kGeneric>, (int)sort_smem_bytes(false), "sort"},
            {(const void*)radix_onesweep_kernel<kPackedFirst>, (int)sort_smem_bytes(true), "sort"},
            {(const void*)radix_onesweep_kernel<kPacked>, (int)sort_smem_bytes(true), "sort"},
            {(const void*)walk_pair_kernel<false>, walk_smem, "walk"},
            {(const void*)walk_pair_kernel<true>, walk_smem, "walk count"},
            {(const void*)walk_pair_kernel<false, true>, walk_smem, "walk subset"},
            {(const void*)walk_pair_kernel<true, true>, walk_smem, "walk subset count"},
            {(const void*)walk_pair_kernel<false, false, true>, walk_smem, "walk field"},
            {(const void*)walk_pair_kernel<false, true, true>, walk_smem, "walk field subset"},
            {(const void*)walk_pair_kernel<false, false, false, true>, walk_smem, "walk periodic"},
            {(const void*)walk_pair_kernel<true, false, false, true>, walk_smem, "walk periodic count"},
        };
        for (const auto& k : big_smem) {
            if ((e = cudaFuncSetAttribute(k.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, k.bytes)) != cudaSuccess) {
                rc = cuda_fail(ctx, e, k.what);
                break;
            }
        }
    } while (0);
    if (rc != BH_OK) { bh_destroy(ctx); return rc; }
    *out = ctx;
    return BH_OK;
}

int bh_destroy(bh_ctx* ctx)
{
    if (!ctx) return BH_OK;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    DevBuf* all[] = {&ctx->keysA, &ctx->keysB, &ctx->idxA, &ctx->idxB, &ctx->clev, &ctx->leaf_slot, &ctx->leaf64,
                     &ctx->slot_of, &ctx->hist, &ctx->scan_scratch, &ctx->nlo, &ctx->nfirst, &ctx->node_slot,
                     &ctx->delta64, &ctx->rec64, &ctx->rec, &ctx->aux, &ctx->gcount, &ctx->geval, &ctx->scalars, &ctx->stage[0],
                     &ctx->stage[1], &ctx->stage[2], &ctx->stage[3], &ctx->stage_phi, &ctx->ess_state, &ctx->ess_emit,
                     &ctx->ew_table, &ctx->ew_coef};
    for (DevBuf* b : all) b->release();
    if (ctx->h_scalars) cudaFreeHost(ctx->h_scalars);
    if (ctx->copy_stream) { cudaStreamSynchronize(ctx->copy_stream); cudaStreamDestroy(ctx->copy_stream); }
    for (int i = 0; i < EV_COUNT; ++i) if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    for (int i = 0; i < bh_ctx::kMaxPasses; ++i) if (ctx->pev[i]) cudaEventDestroy(ctx->pev[i]);
    delete ctx;
    return BH_OK;
}

int bh_set_option(bh_ctx* ctx, int key, int value)
{
    if (!ctx) return BH_ERR_INVALID_ARG;
    if (key == BH_OPT_MAC && (value == BH_MAC_BH86 || value == BH_MAC_BARNES94)) { ctx->mac = value; return BH_OK; }
    if (key == BH_OPT_GROUP && (value == 32 || value == 1)) { ctx->group = value; return BH_OK; }
    if (key == BH_OPT_PERIODIC && (value == 0 || value == 1)) { ctx->periodic = value != 0; return BH_OK; }
    if (key == BH_OPT_EWALD_N && value >= 6 && value <= 258) { ctx->ew_N = value; return BH_OK; }
    if (key == BH_OPT_EWALD_NREF && value >= 1 && value <= 8) { ctx->ew_nref = value; return BH_OK; }
    if (key == BH_OPT_PASS_TIMING && (value == 0 || value == 1)) { ctx->pass_timing = value != 0; ctx->npass = 0; return BH_OK; }
    return BH_ERR_INVALID_ARG;
}

int bh_build(bh_ctx* ctx, const double* x, const double* y, const double* z, const double* m, int64_t n,
             const double cube[4])
{
    if (!ctx || !x || !y || !z || !m || !cube) return BH_ERR_INVALID_ARG;
    if (n >= (1LL << 30) && n < 2147483648LL) return BH_ERR_TOO_LARGE;   // 30-bit tile counters of the sort
    if (n <= 0 || n >= 2147483648LL || !(cube[3] > 0.0) || !isfinite(cube[0]) || !isfinite(cube[1]) ||
        !isfinite(cube[2]) || !isfinite(cube[3]))
        return BH_ERR_INVALID_ARG;
    ctx->built = false;
    ctx->walked = false;
    ctx->launches_build = 0;
    BH_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    DeviceScalars* ds = ctx->scalars.as<DeviceScalars>();
    ctx->n = n;
    memcpy(ctx->cube, cube, sizeof(double) * 4);

    // ---- buffers that depend on n only ----
    BH_CUDA(ctx->keysA.ensure(sizeof(u64) * n));
    BH_CUDA(ctx->keysB.ensure(sizeof(u64) * n));
    BH_CUDA(ctx->clev.ensure((size_t)n + 16));
    BH_CUDA(ctx->leaf_slot.ensure(sizeof(u32) * n));
    {
        const size_t he = sort_hist_elems(n) > topo_hist_elems(n) ? sort_hist_elems(n) : topo_hist_elems(n);
        BH_CUDA(ctx->hist.ensure(sizeof(u32) * (he + 4)));
        BH_CUDA(ctx->scan_scratch.ensure(sizeof(u32) * (scan_scratch_elems((i64)he) + 4)));
    }
    ctx->direct_ready = false;

    BH_CUDA(cudaEventRecord(ctx->ev[EV_B0], st));
    // The sort plan (which key bits vary) and the constant key bits come from the OR / AND of all keys.
    // A solver called every time step sees the same mesh again and again, so the first
    // attempt takes them from the previous build and runs keys -> sort -> count without a host round
    // trip; the real OR / AND arrive with the second read-back and must match, else the build is redone
    // from the keys with the values just read (any plan yields memory-safe, merely useless, passes).
    i64 nchunks = 0;
    unsigned tgrid = 0;
    int aux_cleared = 0;
    int launches_front = 0;
    bool spec_rows = false;
    // Everything after the level totals: sizes, assign + permute (a4 + a3), moments (a5).  `rows` are the scanned
    // row starts -- this build's own, read back, or (gate != null) the previous build's, enqueued before this build's
    // arrive; the kernels then run only if the device finds the two equal (topo_totals_kernel sets *gate).
    auto finish = [&](const u32* rows, const u32* gate) -> int {
        u32* hist = ctx->hist.as<u32>();
        ctx->launches_build = launches_front + aux_cleared + 1 + 3 + 1 + 1;   // keys + sort; count, scan, totals, assign
        // The device scan runs in u32.  Every histogram row sums to at most n < 2^30, so consecutive row
        // starts differ by less than 2^30 and the true 64-bit starts follow from the differences mod 2^32.
        unsigned long long true_rows[kTopoDigits + 1];
        true_rows[0] = rows[0];
        for (int d = 1; d <= kTopoDigits; ++d) true_rows[d] = true_rows[d - 1] + (u32)(rows[d] - rows[d - 1]);
        if (true_rows[kSlotLevels] >= (1ULL << 32)) {          // slots are u32: n + n_nodes must stay below 2^32
            snprintf(ctx->cuda_msg, sizeof(ctx->cuda_msg), "n + n_nodes = %llu needs more than 32-bit slots",
                     true_rows[kSlotLevels]);
            return BH_ERR_TOO_LARGE;
        }
        const i64 nslots = (i64)true_rows[kSlotLevels];       // entities of all levels = n + n_nodes
        const i64 nn = (i64)(true_rows[kTopoDigits] - true_rows[kSlotLevels]);
        for (int l = 0; l <= kSlotLevels; ++l) ctx->lv.slot_base[l] = rows[l];
        for (int l = 0; l <= kNumLevels; ++l) ctx->lv.node_base[l] = (u32)(rows[kSlotLevels + l] - nslots);
        ctx->maxlevel = 0; ctx->depth = 0;
        for (int l = 0; l < kNumLevels; ++l)
            if (ctx->lv.node_base[l + 1] > ctx->lv.node_base[l]) { ctx->maxlevel = l; if (l < kMaxLevel) ctx->depth = l; }
        ctx->nn = nn;
        ctx->nslots = nslots;
        if (nslots != n + nn) {
            snprintf(ctx->cuda_msg, sizeof(ctx->cuda_msg), "topology: %lld entities for %lld cells + %lld nodes",
                     (long long)nslots, (long long)n, (long long)nn);
            return BH_ERR_CUDA;
        }

        {
            const bool grow = sizeof(WalkAux) * (size_t)nslots > ctx->aux.cap;
            BH_CUDA(ctx->aux.ensure(sizeof(WalkAux) * nslots));
            if (grow || ctx->aux_dirty_nn < 0) BH_CUDA(cudaMemsetAsync(ctx->aux.p, 0, ctx->aux.cap, st));
            ctx->aux_dirty_nn = -1;                            // unknown until this build's moments are launched
        }
        BH_CUDA(ctx->nlo.ensure(sizeof(u32) * nn));
        BH_CUDA(ctx->nfirst.ensure(sizeof(u32) * (nn + 4)));
        BH_CUDA(ctx->node_slot.ensure(sizeof(u32) * nn));
        BH_CUDA(ctx->delta64.ensure(sizeof(double) * nn));
        BH_CUDA(ctx->rec64.ensure(sizeof(double4) * nslots));
        BH_CUDA(ctx->rec.ensure(sizeof(float4) * nslots));

        pass_mark(ctx, "aux_clear+readback", 0.0);      // node-slot aux clearing and the idle wait for the level totals
        if (ctx->assign_wait) BH_CUDA(cudaStreamWaitEvent(st, ctx->assign_wait, 0));   // bh_solve_host: m is still landing
        BH_CUDA(launch_chain(topo_assign_kernel, dim3(tgrid), dim3(kTopoThreads), 0, st,
                             ctx->clev.as<signed char>(), n, ctx->sv, x, y, z, m, hist, nchunks, (u32)nslots,
                             ctx->leaf_slot.as<u32>(), ctx->node_slot.as<u32>(), ctx->nfirst.as<u32>(), ctx->nlo.as<u32>(),
                             ctx->rec64.as<double4>(), ctx->rec.as<float4>(), gate));
        pass_mark(ctx, "assign_permute", 84.0 * (double)n + 24.0 * (double)nn);   // a3 84 B/cell + a4 24 B/node
        if (ctx->pass_timing) BH_CUDA(cudaEventRecord(ctx->ev[EV_TOPO], st));

        // ---- a5: moments ----
        { int rc = launch_moments(ctx, gate); if (rc != BH_OK) return rc; }
        ctx->aux_dirty_nn = nn;
        return BH_OK;
    };
    for (int attempt = 0;; ++attempt) {
        const bool speculate = attempt == 0 && ctx->plan_hint_valid;
        ctx->launches_build = 0;
        ctx->npass = 0;
        // A speculated plan is known before the keys exist: every memset is issued first, and the kernels from the
        // keys to the level totals form one chain of dependent launches (launch_chain / chain_enter, common.cuh)
        // with no copy or memset in between; the key reduction is then read back together with the level totals.
        KeyReduce kr = ctx->plan_hint;
        SortPlan plan = make_sort_plan(kr.key_or ^ kr.key_and, n);
        if (speculate && plan.npasses > 0)
            BH_CUDA(cudaMemsetAsync(ctx->hist.p, 0, sizeof(u32) * sort_pass_words(n) * (size_t)plan.npasses, st));
        BH_CUDA(cudaMemsetAsync(ds, 0, sizeof(DeviceScalars), st));
        BH_CUDA(cudaMemsetAsync(&ds->keyred.key_and, 0xff, sizeof(u64), st));   // key_and starts as all ones

        // ---- a1: Morton keys ----
        const double s = 2097152.0 / cube[3];      // K1: s = 2^21 / L in fp64
        {
            const int grid = persistent_grid(ctx, 8);
            if (aligned16(x) && aligned16(y) && aligned16(z)) {
                BH_CUDA(launch_chain(morton_keys_kernel<2>, dim3(grid), dim3(256), 0, st, x, y, z, n, cube[0], cube[1],
                                     cube[2], s, ctx->keysA.as<u64>(), &ds->keyred));
            } else {
                BH_CUDA(launch_chain(morton_keys_kernel<1>, dim3(grid), dim3(256), 0, st, x, y, z, n, cube[0], cube[1],
                                     cube[2], s, ctx->keysA.as<u64>(), &ds->keyred));
            }
        }
        ctx->launches_build += 1;
        pass_mark(ctx, "keys", 36.0 * (double)n);
        if (ctx->pass_timing) BH_CUDA(cudaEventRecord(ctx->ev[EV_KEYS], st));   // an event between two kernels breaks their chain

        // read-back 1: which key bits vary (decides the radix passes) and the clamp count
        if (!speculate) {
            BH_CUDA(cudaMemcpyAsync(&ctx->h_scalars->keyred, &ds->keyred, sizeof(KeyReduce), cudaMemcpyDeviceToHost, st));
            BH_CUDA(cudaStreamSynchronize(st));
            kr = ctx->h_scalars->keyred;
            plan = make_sort_plan(kr.key_or ^ kr.key_and, n);
        }
        ctx->sort_passes = plan.npasses;

        // ---- a2: radix sort of (key, index) ----
        if (plan.npasses > 0 && !plan.packed) {      // the permutation is stored only when the key window left beside the index is too narrow
            BH_CUDA(ctx->idxA.ensure(sizeof(u32) * n));
            BH_CUDA(ctx->idxB.ensure(sizeof(u32) * n));
        }
        BH_CUDA(radix_sort_pairs(ctx->keysA.as<u64>(), ctx->idxA.as<u32>(), ctx->keysB.as<u64>(), ctx->idxB.as<u32>(), n,
                                 plan, ctx->hist.as<u32>(), /*scratch_is_clear=*/speculate, persistent_grid(ctx, 8), st,
                                 [ctx](const char* nm, double b) { pass_mark(ctx, nm, b); }));
        ctx->launches_build += plan.npasses ? 1 + plan.npasses : 0;   // histogram + one kernel per pass
        launches_front = ctx->launches_build;
        {
            const bool odd = plan.npasses & 1;
            const u64* kres = odd ? ctx->keysB.as<u64>() : ctx->keysA.as<u64>();
            SortedView& sv = ctx->sv;
            sv.packed = nullptr; sv.keys = nullptr; sv.idx = nullptr; sv.cbits = 0; sv.lo = 0; sv.ib = plan.ib;
            if (plan.npasses == 0) sv.keys = kres;                      // identity: all keys equal
            else if (plan.packed) {
                sv.packed = kres;
                sv.lo = plan.lo;
                sv.cbits = kr.key_and & ~(((~0ULL) >> plan.ib) << plan.lo);
            } else {
                sv.keys = kres;
                sv.idx = odd ? ctx->idxB.as<u32>() : ctx->idxA.as<u32>();
            }
        }
        if (ctx->pass_timing) BH_CUDA(cudaEventRecord(ctx->ev[EV_SORT], st));

        // ---- a4: topology (a3, the permutation of the cell data, is fused into the assigning kernel) ----
        ctx->nn = 0; ctx->nslots = 0; ctx->depth = 0; ctx->maxlevel = 0; ctx->max_bucket = 1;
        memset(&ctx->lv, 0, sizeof(ctx->lv));
        if (n >= 2) {
            nchunks = topo_chunks(n);
            tgrid = blocks_for(nchunks, kTopoThreads / 32);
            u32* hist = ctx->hist.as<u32>();
            BH_CUDA(launch_chain(topo_count_kernel, dim3(tgrid), dim3(kTopoThreads), 0, st, ctx->sv, n,
                                 ctx->clev.as<signed char>(), hist, nchunks));
            pass_mark(ctx, "topo_count", 8.0 * (double)n);
            BH_CUDA(exclusive_scan_u32(hist, hist, (i64)kTopoDigits * nchunks, ctx->scan_scratch.as<u32>(),
                                       &ds->scan_total, st));
            // the level totals of the previous build are expected again if that build had as many cells and this
            // one already speculates its sort plan (the same mesh as last time)
            spec_rows = speculate && ctx->rows_hint_n == n;
            TotalsHint hint;
            memcpy(hint.rows, ctx->rows_hint, sizeof(hint.rows));
            hint.key_or = kr.key_or; hint.key_and = kr.key_and; hint.check = spec_rows ? 1 : 0;
            BH_CUDA(launch_chain(topo_totals_kernel, dim3(1), dim3(64), 0, st, hist, nchunks, &ds->scan_total,
                                 ctx->h_scalars->topo_rows, hint, &ds->keyred,
                                 speculate ? &ctx->h_scalars->keyred : nullptr, &ds->spec_ok));
            pass_mark(ctx, "topo_scan", 0.0);
            // read-back 2: entities and nodes per level (sizes every node / slot array) and, under a speculated
            // plan, the key reduction of THIS build -- written by the kernel itself into the pinned host mirror
            // (device-accessible under unified addressing), so no copy stands on the stream
        } else if (speculate)
            BH_CUDA(cudaMemcpyAsync(&ctx->h_scalars->keyred, &ds->keyred, sizeof(KeyReduce), cudaMemcpyDeviceToHost, st));
        BH_CUDA(cudaEventRecord(ctx->ev[EV_PERM], st));
        // aux must be zero on every leaf slot; only the node slots of the previous build are not.  Clearing
        // them runs on the device while the host waits for the read-back and prepares the next launches.
        if (ctx->aux_dirty_nn > 0) {
            aux_clear_kernel<<<blocks_for(ctx->aux_dirty_nn, 256), 256, 0, st>>>(ctx->node_slot.as<u32>(), ctx->aux_dirty_nn,
                                                                                ctx->aux.as<WalkAux>());
            BH_CUDA(cudaGetLastError());
            ctx->aux_dirty_nn = 0;
            aux_cleared = 1;
        }
        // speculated level totals: assign and the moments are enqueued now, on the previous build's totals and
        // behind a device-side gate, and the host's wait for the read-back below runs under them
        if (spec_rows) { int rc = finish(ctx->rows_hint, &ds->spec_ok); if (rc != BH_OK) return rc; }
        BH_CUDA(cudaEventSynchronize(ctx->ev[EV_PERM]));
        {
            const KeyReduce& real = ctx->h_scalars->keyred;
            const bool hit = real.key_or == kr.key_or && real.key_and == kr.key_and;
            ctx->plan_hint = real;
            ctx->plan_hint_valid = true;
            ctx->n_clamped = (i64)real.n_clamped;
            if (hit) break;
            if (spec_rows) ctx->aux_dirty_nn = 0;    // the gate was closed (the key reduction differs): aux is untouched
            spec_rows = false;
        }
    }   // attempt
    if (n >= 2) {
        const bool hit_rows = spec_rows && memcmp(ctx->h_scalars->topo_rows, ctx->rows_hint, sizeof(ctx->rows_hint)) == 0;
        if (spec_rows && !hit_rows) ctx->aux_dirty_nn = 0;     // the gated kernels wrote nothing: aux is still all zero
        if (!hit_rows) { int rc = finish(ctx->h_scalars->topo_rows, nullptr); if (rc != BH_OK) return rc; }
        memcpy(ctx->rows_hint, ctx->h_scalars->topo_rows, sizeof(ctx->rows_hint));
        ctx->rows_hint_n = n;
    } else {
        // n = 1: no tree (T-rule 1); the lone cell's record is kept for bh_essential_nodes
        if (ctx->assign_wait) BH_CUDA(cudaStreamWaitEvent(st, ctx->assign_wait, 0));
        BH_CUDA(ctx->rec64.ensure(sizeof(double4)));
        const double* src[4] = {x, y, z, m};
        for (int a = 0; a < 4; ++a)
            BH_CUDA(cudaMemcpyAsync(ctx->rec64.as<double>() + a, src[a], sizeof(double), cudaMemcpyDeviceToDevice, st));
        BH_CUDA(cudaEventRecord(ctx->ev[EV_TOPO], st));
    }
    BH_CUDA(cudaEventRecord(ctx->ev[EV_MOM], st));
    ctx->ev_build = true;
    ctx->ev_phases = ctx->pass_timing || n < 2;
    ctx->built = true;
    return BH_OK;
}

int bh_update_masses(bh_ctx* ctx, const double* m)
{
    if (!ctx || !m) return BH_ERR_INVALID_ARG;
    if (!ctx->built) return BH_ERR_NOT_BUILT;
    BH_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    ctx->walked = false;
    ctx->counts_valid = false;
    ctx->direct_ready = false;
    ctx->launches_build = 0;
    BH_CUDA(cudaEventRecord(ctx->ev[EV_B0], st));
    for (int k = EV_KEYS; k <= EV_TOPO; ++k) BH_CUDA(cudaEventRecord(ctx->ev[k], st));
    ctx->ev_phases = true;
    if (ctx->n >= 2) {
        mass_update_kernel<<<blocks_for(ctx->n, 256), 256, 0, st>>>(ctx->sv, ctx->leaf_slot.as<u32>(), m, ctx->n,
                                                                   ctx->rec64.as<double4>(), ctx->rec.as<float4>());
        BH_CUDA(cudaGetLastError());
        ctx->launches_build += 1;
        { int rc = launch_moments(ctx); if (rc != BH_OK) return rc; }
    }
    BH_CUDA(cudaEventRecord(ctx->ev[EV_MOM], st));
    return BH_OK;
}

int bh_set_num_targets(bh_ctx* ctx, int64_t ntargets)
{
    if (!ctx || ntargets < -1) return BH_ERR_INVALID_ARG;
    ctx->ntargets = ntargets;
    ctx->walked = false;
    ctx->counts_valid = false;
    return BH_OK;
}

int bh_essential_nodes(bh_ctx* ctx, const double box_lo[3], const double box_hi[3], double theta, double* out,
                       int64_t cap, int64_t* count)
{
    if (!ctx || !box_lo || !box_hi || !count || cap < 0 || (cap > 0 && !out) || !(theta >= 0.0)) return BH_ERR_INVALID_ARG;
    for (int a = 0; a < 3; ++a) if (!(box_lo[a] <= box_hi[a])) return BH_ERR_INVALID_ARG;
    if (cap > 0 && !aligned16(out)) return BH_ERR_INVALID_ARG;
    if (!ctx->built) return BH_ERR_NOT_BUILT;
    BH_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    *count = 0;
    if (ctx->n == 1) {                       // a lone cell is sent as it is
        *count = 1;
        if (cap < 1) return BH_ERR_TOO_LARGE;
        BH_CUDA(cudaMemcpyAsync(out, ctx->rec64.p, sizeof(double) * 4, cudaMemcpyDeviceToDevice, st));
        return BH_OK;
    }
    const i64 nslots = ctx->nslots;
    const i64 nblk = (nslots + kEssTile - 1) / kEssTile;
    BH_CUDA(ctx->ess_state.ensure((size_t)nslots + 16));
    BH_CUDA(ctx->ess_emit.ensure(sizeof(u32) * ((size_t)nblk + 4)));                 // essential slots per block
    BH_CUDA(ctx->scan_scratch.ensure(sizeof(u32) * (scan_scratch_elems(nblk) + 4)));
    BH_CUDA(cudaMemsetAsync(ctx->ess_state.p, 0, (size_t)nslots, st));
    BH_CUDA(cudaMemsetAsync(ctx->ess_state.p, 1, 1, st));        // the root (slot 0) is tested like any node
    EssArgs A;
    A.nfirst = ctx->nfirst.as<u32>(); A.node_slot = ctx->node_slot.as<u32>(); A.rec64 = ctx->rec64.as<double4>();
    A.delta64 = ctx->delta64.as<double>(); A.aux = ctx->aux.as<WalkAux>();
    A.state = ctx->ess_state.as<unsigned char>();
    for (int a = 0; a < 3; ++a) { A.blo[a] = box_lo[a]; A.bhi[a] = box_hi[a]; }
    A.theta = theta; A.L = ctx->cube[3]; A.mac = ctx->mac;
    SmallLevels sl;
    sl.nlev = 0;
    for (int l = 0; l <= ctx->maxlevel + 1; ++l) {      // root side first; one extra turn flushes the last run
        const bool last = l > ctx->maxlevel;
        const i64 b0 = last ? 0 : ctx->lv.node_base[l], b1 = last ? 0 : ctx->lv.node_base[l + 1];
        const bool small = !last && b1 - b0 <= kEssSmallNodes;
        if ((!small || last) && sl.nlev > 0) {
            BH_CUDA(launch_chain(ess_small_kernel, dim3(1), dim3(1024), 0, st, sl, A));
            sl.nlev = 0;
        }
        if (last || b1 == b0) continue;
        if (small) {
            sl.level[sl.nlev] = l; sl.b0[sl.nlev] = (u32)b0; sl.b1[sl.nlev] = (u32)b1;
            sl.slot_end[sl.nlev] = ctx->lv.slot_base[l + 2];
            ++sl.nlev;
        } else {
            BH_CUDA(launch_chain(ess_level_kernel, dim3(blocks_for(b1 - b0, 256)), dim3(256), 0, st, b0, b1, l,
                                 ctx->lv.slot_base[l + 2], A));
        }
    }
    u32* blk = ctx->ess_emit.as<u32>();
    BH_CUDA(launch_chain(ess_count_kernel, dim3((unsigned)nblk), dim3(kEssThreads), 0, st, A.state, nslots, blk));
    // the number of entries goes straight into the pinned host mirror (device-accessible): no copy on the stream
    BH_CUDA(exclusive_scan_u32(blk, blk, nblk, ctx->scan_scratch.as<u32>(), &ctx->h_scalars->scan_total, st));
    if (cap > 0)
        BH_CUDA(launch_chain(ess_gather_kernel, dim3((unsigned)nblk), dim3(kEssThreads), 0, st, A.state, nslots, blk,
                             ctx->rec64.as<double4>(), out, cap));
    BH_CUDA(cudaStreamSynchronize(st));
    *count = (int64_t)ctx->h_scalars->scan_total;
    return *count > cap ? BH_ERR_TOO_LARGE : BH_OK;
}

}  // extern "C" (reopened below)

namespace {

// The Ewald field array of the context's (N, nref): built on first use and whenever the options changed
// ("calculated once on startup").  Box units, so it does not depend on the cube.
int ensure_ewald(bh_ctx* ctx)
{
    if (ctx->ew_ready_N == ctx->ew_N && ctx->ew_ready_nref == ctx->ew_nref) return BH_OK;
    const int N = ctx->ew_N, nref = ctx->ew_nref, M = N - 1;
    const i64 npts = (i64)nref * N * N * N, ncoef = (i64)nref * M * M * M;
    BH_CUDA(ctx->ew_table.ensure(sizeof(double) * npts));
    BH_CUDA(ctx->ew_coef.ensure(sizeof(EwaldRec) * ncoef));
    ewald_table_kernel<<<blocks_for(npts, 128), 128, 0, ctx->stream>>>(N, nref, ctx->ew_table.as<double>());
    BH_CUDA(cudaGetLastError());
    ewald_coef_kernel<<<blocks_for(ncoef, 128), 128, 0, ctx->stream>>>(N, nref, ctx->ew_table.as<double>(), ctx->ew_coef.as<EwaldRec>());
    BH_CUDA(cudaGetLastError());
    ctx->ew_ready_N = N;
    ctx->ew_ready_nref = nref;
    return BH_OK;
}

// Launches the walk of the last build on the context's stream.  count_only: the traversal of
// walk_pair_kernel<true> (same decisions, no arithmetic on masses), filling ctx->gcount.
int launch_walk(bh_ctx* ctx, double theta, double G, double* phi, int group, int mac, bool count_only,
                double* acc = nullptr, bool periodic = false)
{
    cudaStream_t st = ctx->stream;
    const i64 n = ctx->n;
    if (periodic) {
        // the periodic walk is the group walk for Phi over all cells (no per-target mode, no field, no source-only cells)
        if (group != 32 || acc || (ctx->ntargets >= 0 && ctx->ntargets < n)) return BH_ERR_INVALID_ARG;
        int rc = ensure_ewald(ctx);
        if (rc != BH_OK) return rc;
    }
    const i64 ngroups = (n + group - 1) / group;
    BH_CUDA(ctx->gcount.ensure(sizeof(uint4) * ngroups));
    BH_CUDA(ctx->geval.ensure(sizeof(u32) * ngroups));
    if (n == 1) {   // T-rule 1: a lone cell has no tree; Phi = 0
        if (!count_only && !periodic) BH_CUDA(cudaMemsetAsync(phi, 0, sizeof(double), st));
        if (!count_only && periodic) {      // the lone cell still feels its own images (reading P5)
            periodic_single_kernel<<<1, 1, 0, st>>>(ctx->rec64.as<double4>(), ctx->ew_table.as<double>(), ctx->cube[3], -G, phi);
            BH_CUDA(cudaGetLastError());
        }
        if (!count_only && acc) BH_CUDA(cudaMemsetAsync(acc, 0, 3 * sizeof(double), st));
        BH_CUDA(cudaMemsetAsync(ctx->gcount.p, 0, sizeof(uint4), st));
        if (!count_only) BH_CUDA(cudaMemsetAsync(ctx->geval.p, 0, sizeof(u32), st));
        return BH_OK;
    }
    WalkParams P;
    P.rec = ctx->rec.as<float4>();
    P.aux = ctx->aux.as<WalkAux>();
    P.leaf_slot = ctx->leaf_slot.as<u32>();
    P.sv = ctx->sv;
    P.phi = phi;
    P.acc = acc;
    P.gcount = ctx->gcount.as<uint4>();
    P.geval = ctx->geval.as<u32>();
    P.n = n;
    P.ngroups = ngroups;
    P.inv_theta = (float)(1.0 / theta);
    P.mac = mac;
    P.negG = -G;
    P.stack_cap = 0;
    P.ntargets = ctx->ntargets < 0 ? 0xffffffffu : (u32)(ctx->ntargets < n ? ctx->ntargets : n);
    P.nslots = (u32)ctx->nslots;
    memset(&P.ew, 0, sizeof(P.ew));
    if (periodic) {
        P.ew.coef = ctx->ew_coef.as<EwaldRec>();
        P.ew.L = (float)ctx->cube[3];
        P.ew.invL = (float)(1.0 / ctx->cube[3]);
        P.ew.s0 = (float)(2.0 * (ctx->ew_N - 2) / ctx->cube[3]);
        P.ew.top = (float)(ctx->ew_N - 2);
        P.ew.M = ctx->ew_N - 1;
        P.ew.MM = P.ew.M * P.ew.M;
        P.ew.M3 = P.ew.MM * P.ew.M;
        P.ew.cbias = 0x4b400000u * (u32)(P.ew.MM + P.ew.M + 1);
        P.ew.nref = ctx->ew_nref;
        P.ew.inv_s2 = 1.f / ewald_s2(ctx->ew_N);
        P.ew.ktop = 0x4b400000 + (ctx->ew_N - 2);
    }
    if (group == 32) {
        i64 cap = (i64)kStackPerLevel * (ctx->maxlevel + 2) + 32;
        cap = (cap + 1) & ~1LL;
        const size_t smem = walk_smem_per_warp((int)cap) * kWalkWarps;
        if (smem > 227 * 1024) return BH_ERR_TOO_LARGE;
        P.stack_cap = (int)cap;
        const i64 npairs = (ngroups + 1) / 2;
        const bool subset = P.ntargets != 0xffffffffu;
        if (periodic && count_only)
            walk_pair_kernel<true, false, false, true><<<blocks_for(npairs, kWalkWarps), kWalkWarps * 32, smem, st>>>(P);
        else if (periodic)
            walk_pair_kernel<false, false, false, true><<<blocks_for(npairs, kWalkWarps), kWalkWarps * 32, smem, st>>>(P);
        else if (count_only && subset)
            walk_pair_kernel<true, true><<<blocks_for(npairs, kWalkWarps), kWalkWarps * 32, smem, st>>>(P);
        else if (count_only)
            walk_pair_kernel<true><<<blocks_for(npairs, kWalkWarps), kWalkWarps * 32, smem, st>>>(P);
        else if (acc && subset)
            walk_pair_kernel<false, true, true><<<blocks_for(npairs, kWalkWarps), kWalkWarps * 32, smem, st>>>(P);
        else if (acc)
            walk_pair_kernel<false, false, true><<<blocks_for(npairs, kWalkWarps), kWalkWarps * 32, smem, st>>>(P);
        else if (subset)
            walk_pair_kernel<false, true><<<blocks_for(npairs, kWalkWarps), kWalkWarps * 32, smem, st>>>(P);
        else
            walk_pair_kernel<false><<<blocks_for(npairs, kWalkWarps), kWalkWarps * 32, smem, st>>>(P);
    } else {
        walk_single_kernel<<<blocks_for(n, 128), 128, 0, st>>>(P);   // counts as it goes
    }
    BH_CUDA(cudaGetLastError());
    return BH_OK;
}

// The per-group counters (W6) are not kept by the hot kernel: the first call that asks for them
// repeats the walk of the last bh_potential in count-only mode.
int ensure_counts(bh_ctx* ctx)
{
    if (ctx->counts_valid) return BH_OK;
    int rc = launch_walk(ctx, ctx->walk_theta, 0.0, nullptr, ctx->walk_group, ctx->walk_mac, true, nullptr, ctx->walk_periodic);
    if (rc == BH_OK) ctx->counts_valid = true;
    return rc;
}

}  // namespace

extern "C" {

static int potential_impl(bh_ctx* ctx, double theta, double G, double* phi, double* acc)
{
    if (!ctx || !phi || !(theta >= 0.0) || isnan(G)) return BH_ERR_INVALID_ARG;
    if (!ctx->built) return BH_ERR_NOT_BUILT;
    BH_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const int group = ctx->group;
    ctx->launches_walk = 0;
    ctx->walked = false;
    BH_CUDA(cudaEventRecord(ctx->ev[EV_W0], st));
    int rc = launch_walk(ctx, theta, G, phi, group, ctx->mac, false, acc, ctx->periodic);
    if (rc != BH_OK) return rc;
    ctx->walk_periodic = ctx->periodic;
    ctx->launches_walk = ctx->n > 1 ? 1 : 0;
    BH_CUDA(cudaEventRecord(ctx->ev[EV_W1], st));
    ctx->ev_walk = true;
    ctx->walked = true;
    ctx->walk_group = group;
    ctx->walk_theta = theta;
    ctx->walk_mac = ctx->mac;
    ctx->counts_valid = group != 32 || ctx->n == 1;   // the per-target walk and n = 1 fill gcount themselves
    return BH_OK;
}

int bh_potential(bh_ctx* ctx, double theta, double G, double* phi)
{
    return potential_impl(ctx, theta, G, phi, nullptr);
}

int bh_field(bh_ctx* ctx, double theta, double G, double* phi, double* acc)
{
    if (!acc) return BH_ERR_INVALID_ARG;
    return potential_impl(ctx, theta, G, phi, acc);
}

int bh_potential_direct(bh_ctx* ctx, double G, const int64_t* targets, int64_t nt, double* phi)
{
    if (!ctx || !phi || isnan(G)) return BH_ERR_INVALID_ARG;
    if (!ctx->built) return BH_ERR_NOT_BUILT;
    if (!targets) {
        if (ctx->n > BH_DIRECT_ALL_MAX) return BH_ERR_TOO_LARGE;
        nt = ctx->n;
    } else if (nt < 0) return BH_ERR_INVALID_ARG;
    if (nt == 0) return BH_OK;
    BH_CUDA(cudaSetDevice(ctx->device));
    if (!ctx->direct_ready) {     // sorted fp64 copy of the cells + inverse permutation, once per build
        BH_CUDA(ctx->leaf64.ensure(sizeof(double4) * ctx->n));
        BH_CUDA(ctx->slot_of.ensure(sizeof(u32) * ctx->n));
        if (ctx->n == 1) {
            BH_CUDA(cudaMemsetAsync(ctx->leaf64.p, 0, sizeof(double4), ctx->stream));
            BH_CUDA(cudaMemsetAsync(ctx->slot_of.p, 0, sizeof(u32), ctx->stream));
        } else {
            direct_prepare_kernel<<<blocks_for(ctx->n, 256), 256, 0, ctx->stream>>>(
                ctx->sv, ctx->leaf_slot.as<u32>(), ctx->rec64.as<double4>(), ctx->n, ctx->leaf64.as<double4>(),
                ctx->slot_of.as<u32>());
            BH_CUDA(cudaGetLastError());
        }
        ctx->direct_ready = true;
    }
    direct_kernel<<<blocks_for(nt, kDirectThreads), kDirectThreads, 0, ctx->stream>>>(
        ctx->leaf64.as<double4>(), ctx->n, ctx->slot_of.as<u32>(), reinterpret_cast<const i64*>(targets), nt, -G, phi);
    BH_CUDA(cudaGetLastError());
    return BH_OK;
}

}  // extern "C" (reopened below)

namespace {

// host -> device / device -> host on `st`.  Pinned buffers are copied by one asynchronous DMA; for pageable ones the
// runtime stages the copy itself.  (Staging pageable buffers here through two pinned 16 MB chunks, the CPU's memcpy of
// one chunk beside the DMA of the other, was measured against that on turb256: 78 ms per call against 71 ms -- the CPU
// copy at ~11 GB/s bounds both, and the runtime's device -> host path is twice as fast -- so it was dropped.)
int h2d(bh_ctx* ctx, void* dst, const void* src, size_t bytes, cudaStream_t st)
{
    BH_CUDA(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, st));
    return BH_OK;
}
int d2h(bh_ctx* ctx, void* dst, const void* src, size_t bytes, cudaStream_t st)
{
    BH_CUDA(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st));
    return BH_OK;
}

}  // namespace

extern "C" {

int bh_solve_host(bh_ctx* ctx, const double* x, const double* y, const double* z, const double* m, int64_t n,
                  const double cube[4], double theta, double G, double* phi)
{
    if (!ctx || !x || !y || !z || !m || !cube || !phi || n <= 0 || n >= 2147483648LL) return BH_ERR_INVALID_ARG;
    BH_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream, cs = ctx->copy_stream;
    for (int k = 0; k < 4; ++k) BH_CUDA(ctx->stage[k].ensure(sizeof(double) * n));
    BH_CUDA(ctx->stage_phi.ensure(sizeof(double) * n));
    ctx->host_timed = false;
    // The copies run on their own stream, positions first: the build (keys, sort, counting -- none of which
    // reads a mass) starts as soon as x, y, z have landed, the assigning kernel waits for m.
    BH_CUDA(cudaEventRecord(ctx->ev[EV_H0], st));
    BH_CUDA(cudaStreamWaitEvent(cs, ctx->ev[EV_H0], 0));           // the staging buffers may still be in use on `st`
    BH_CUDA(cudaEventRecord(ctx->ev[EV_HC0], cs));
    const double* src[4] = {x, y, z, m};
    for (int k = 0; k < 4; ++k) {
        int rc = h2d(ctx, ctx->stage[k].p, src[k], sizeof(double) * n, cs);
        if (rc != BH_OK) return rc;
        if (k == 2) BH_CUDA(cudaEventRecord(ctx->ev[EV_HXYZ], cs));
    }
    BH_CUDA(cudaEventRecord(ctx->ev[EV_HM], cs));
    BH_CUDA(cudaStreamWaitEvent(st, ctx->ev[EV_HXYZ], 0));
    BH_CUDA(cudaEventRecord(ctx->ev[EV_HD0], st));
    ctx->assign_wait = ctx->ev[EV_HM];
    int rc = bh_build(ctx, ctx->stage[0].as<double>(), ctx->stage[1].as<double>(), ctx->stage[2].as<double>(),
                      ctx->stage[3].as<double>(), n, cube);
    ctx->assign_wait = nullptr;
    if (rc != BH_OK) { cudaStreamSynchronize(cs); return rc; }
    rc = bh_potential(ctx, theta, G, ctx->stage_phi.as<double>());
    if (rc != BH_OK) { cudaStreamSynchronize(cs); return rc; }
    BH_CUDA(cudaEventRecord(ctx->ev[EV_HD1], st));
    rc = d2h(ctx, phi, ctx->stage_phi.p, sizeof(double) * n, st);
    if (rc != BH_OK) return rc;
    BH_CUDA(cudaEventRecord(ctx->ev[EV_HEND], st));
    BH_CUDA(cudaStreamSynchronize(st));
    ctx->host_timed = true;
    return BH_OK;
}

int bh_host_breakdown(bh_ctx* ctx, float ms[4])
{
    if (!ctx || !ms) return BH_ERR_INVALID_ARG;
    if (!ctx->host_timed) return BH_ERR_NOT_BUILT;
    BH_CUDA(cudaSetDevice(ctx->device));
    BH_CUDA(cudaEventElapsedTime(&ms[0], ctx->ev[EV_HC0], ctx->ev[EV_HM]));     // host -> device, all four arrays
    BH_CUDA(cudaEventElapsedTime(&ms[1], ctx->ev[EV_HD0], ctx->ev[EV_HD1]));    // build + walk, from the arrival of x, y, z
    BH_CUDA(cudaEventElapsedTime(&ms[2], ctx->ev[EV_HD1], ctx->ev[EV_HEND]));   // device -> host
    BH_CUDA(cudaEventElapsedTime(&ms[3], ctx->ev[EV_H0], ctx->ev[EV_HEND]));    // whole call on the device
    return BH_OK;
}

int bh_get_build_passes(bh_ctx* ctx, bh_pass* out, int cap, int* count)
{
    if (!ctx || !count || cap < 0 || (cap > 0 && !out)) return BH_ERR_INVALID_ARG;
    if (!ctx->built) return BH_ERR_NOT_BUILT;
    BH_CUDA(cudaSetDevice(ctx->device));
    BH_CUDA(cudaStreamSynchronize(ctx->stream));
    *count = ctx->npass;
    for (int k = 0; k < ctx->npass && k < cap; ++k) {
        memset(&out[k], 0, sizeof(out[k]));
        snprintf(out[k].name, sizeof(out[k].name), "%s", ctx->pname[k]);
        out[k].alg_bytes = ctx->pbytes[k];
        cudaEventElapsedTime(&out[k].ms, k == 0 ? ctx->ev[EV_B0] : ctx->pev[k - 1], ctx->pev[k]);
    }
    cudaGetLastError();
    return ctx->npass > cap ? BH_ERR_TOO_LARGE : BH_OK;
}

int bh_ewald_table(bh_ctx* ctx, double* out, int64_t cap, int* N, int* nref)
{
    if (!ctx || cap < 0 || (cap > 0 && !out)) return BH_ERR_INVALID_ARG;
    BH_CUDA(cudaSetDevice(ctx->device));
    { int rc = ensure_ewald(ctx); if (rc != BH_OK) return rc; }
    if (N) *N = ctx->ew_N;
    if (nref) *nref = ctx->ew_nref;
    const i64 npts = (i64)ctx->ew_nref * ctx->ew_N * ctx->ew_N * ctx->ew_N;
    if (cap < npts) return BH_ERR_TOO_LARGE;
    BH_CUDA(cudaMemcpyAsync(out, ctx->ew_table.p, sizeof(double) * npts, cudaMemcpyDeviceToDevice, ctx->stream));
    return BH_OK;
}

int bh_tree_sizes(const bh_ctx* ctx, int64_t* n, int64_t* n_nodes, int64_t* n_slots)
{
    if (!ctx) return BH_ERR_INVALID_ARG;
    if (!ctx->built) return BH_ERR_NOT_BUILT;
    if (n) *n = ctx->n;
    if (n_nodes) *n_nodes = ctx->nn;
    if (n_slots) *n_slots = ctx->nslots;
    return BH_OK;
}

int bh_export_tree(bh_ctx* ctx, uint64_t* keys, uint32_t* perm, int32_t* level, uint64_t* prefix, int64_t* lo,
                   int64_t* hi, int32_t* nchild, double* M, double* Rx, double* Ry, double* Rz, double* delta)
{
    if (!ctx) return BH_ERR_INVALID_ARG;
    if (!ctx->built) return BH_ERR_NOT_BUILT;
    BH_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    if (keys || perm) {
        export_sorted_kernel<<<blocks_for(ctx->n, 256), 256, 0, st>>>(ctx->sv, ctx->n, reinterpret_cast<u64*>(keys), perm);
        BH_CUDA(cudaGetLastError());
    }
    if (ctx->nn > 0) {
        export_nodes_kernel<<<blocks_for(ctx->nn, 256), 256, 0, st>>>(
            ctx->nn, ctx->n, ctx->lv, ctx->sv, ctx->nlo.as<u32>(), ctx->nfirst.as<u32>(), ctx->node_slot.as<u32>(),
            ctx->rec64.as<double4>(), ctx->delta64.as<double>(), level, reinterpret_cast<u64*>(prefix),
            reinterpret_cast<i64*>(lo), reinterpret_cast<i64*>(hi), nchild, M, Rx, Ry, Rz, delta);
        BH_CUDA(cudaGetLastError());
    }
    return BH_OK;
}

int bh_last_group_counts(bh_ctx* ctx, int64_t* counts)
{
    if (!ctx || !counts) return BH_ERR_INVALID_ARG;
    if (!ctx->walked) return BH_ERR_NOT_BUILT;
    BH_CUDA(cudaSetDevice(ctx->device));
    { int rc = ensure_counts(ctx); if (rc != BH_OK) return rc; }
    const i64 ng = (ctx->n + ctx->walk_group - 1) / ctx->walk_group;
    group_counts_export_kernel<<<blocks_for(ng, 256), 256, 0, ctx->stream>>>(ctx->gcount.as<uint4>(), ng,
                                                                             reinterpret_cast<i64*>(counts));
    BH_CUDA(cudaGetLastError());
    return BH_OK;
}

int bh_last_group_evaluated(bh_ctx* ctx, uint32_t* per_group)
{
    if (!ctx || !per_group) return BH_ERR_INVALID_ARG;
    if (!ctx->walked) return BH_ERR_NOT_BUILT;
    BH_CUDA(cudaSetDevice(ctx->device));
    const i64 ng = (ctx->n + ctx->walk_group - 1) / ctx->walk_group;
    group_eval_export_kernel<<<blocks_for(ng, 256), 256, 0, ctx->stream>>>(ctx->geval.as<u32>(), ng, per_group);
    BH_CUDA(cudaGetLastError());
    return BH_OK;
}

int bh_last_walk_group(const bh_ctx* ctx)
{
    if (!ctx) return BH_ERR_INVALID_ARG;
    if (!ctx->walked) return BH_ERR_NOT_BUILT;
    return ctx->walk_group;
}

int bh_last_interactions(bh_ctx* ctx, uint32_t* per_target)
{
    if (!ctx || !per_target) return BH_ERR_INVALID_ARG;
    if (!ctx->walked) return BH_ERR_NOT_BUILT;
    BH_CUDA(cudaSetDevice(ctx->device));
    { int rc = ensure_counts(ctx); if (rc != BH_OK) return rc; }
    per_target_counts_kernel<<<blocks_for(ctx->n, 256), 256, 0, ctx->stream>>>(ctx->gcount.as<uint4>(), ctx->sv,
                                                                               ctx->n, ctx->walk_group, per_target);
    BH_CUDA(cudaGetLastError());
    return BH_OK;
}

int bh_get_stats(bh_ctx* ctx, bh_stats* out)
{
    if (!ctx || !out) return BH_ERR_INVALID_ARG;
    memset(out, 0, sizeof(*out));
    if (!ctx->built) return BH_ERR_NOT_BUILT;
    BH_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    DeviceScalars* ds = ctx->scalars.as<DeviceScalars>();
    if (ctx->walked) {
        { int rc = ensure_counts(ctx); if (rc != BH_OK) return rc; }
        const i64 ng = (ctx->n + ctx->walk_group - 1) / ctx->walk_group;
        BH_CUDA(cudaMemsetAsync(ds->totals, 0, sizeof(ds->totals), st));
        group_counts_total_kernel<<<persistent_grid(ctx, 2), 256, 0, st>>>(ctx->gcount.as<uint4>(), ctx->geval.as<u32>(),
                                                                          ng, ctx->n, ctx->walk_group, ds->totals);
        BH_CUDA(cudaGetLastError());
        BH_CUDA(cudaMemcpyAsync(ctx->h_scalars->totals, ds->totals, sizeof(ds->totals), cudaMemcpyDeviceToHost, st));
    }
    BH_CUDA(cudaMemcpyAsync(&ctx->h_scalars->max_bucket, &ds->max_bucket, sizeof(u32), cudaMemcpyDeviceToHost, st));
    BH_CUDA(cudaStreamSynchronize(st));
    ctx->max_bucket = ctx->h_scalars->max_bucket > 1 ? ctx->h_scalars->max_bucket : 1;
    out->n = ctx->n;
    out->n_nodes = ctx->nn;
    out->n_slots = ctx->nslots;
    out->depth = ctx->depth;
    out->sort_passes = ctx->sort_passes;
    out->n_clamped = ctx->n_clamped;
    out->max_bucket = ctx->max_bucket;
    if (ctx->walked) {
        out->n_accepted = (i64)ctx->h_scalars->totals[0];
        out->n_leaf = (i64)ctx->h_scalars->totals[1];
        out->n_opened = (i64)ctx->h_scalars->totals[2];
        out->n_exact_tests = (i64)ctx->h_scalars->totals[3];
        out->interactions = (double)ctx->h_scalars->totals[5];          // counted by the Phi kernel itself
        out->interactions_counted = (double)ctx->h_scalars->totals[4];  // counted by the count-only twin
        out->walk_group = ctx->walk_group;
    }
    if (ctx->ev_build) {
        // the per-phase events sit between kernels and would break the chain of dependent launches, so an
        // ordinary build records only its two ends; BH_OPT_PASS_TIMING turns the phases (and the passes) on
        if (ctx->ev_phases) {
            cudaEventElapsedTime(&out->ms_keys, ctx->ev[EV_B0], ctx->ev[EV_KEYS]);
            cudaEventElapsedTime(&out->ms_sort, ctx->ev[EV_KEYS], ctx->ev[EV_SORT]);
            cudaEventElapsedTime(&out->ms_count, ctx->ev[EV_SORT], ctx->ev[EV_PERM]);
            cudaEventElapsedTime(&out->ms_assign, ctx->ev[EV_PERM], ctx->ev[EV_TOPO]);
            cudaEventElapsedTime(&out->ms_moments, ctx->ev[EV_TOPO], ctx->ev[EV_MOM]);
        }
        cudaEventElapsedTime(&out->ms_build_total, ctx->ev[EV_B0], ctx->ev[EV_MOM]);
    }
    if (ctx->ev_walk) cudaEventElapsedTime(&out->ms_walk, ctx->ev[EV_W0], ctx->ev[EV_W1]);
    out->launches_build = ctx->launches_build;
    out->launches_walk = ctx->launches_walk;
    cudaGetLastError();
    return BH_OK;
}

}  // extern "C"
