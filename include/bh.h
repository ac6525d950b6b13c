/*
 * bh.h -- C ABI of libbh: Barnes-Hut gravitational potential of AMR grid cells treated as
 * point masses, on one NVIDIA B200 (sm_100a).
 *
 * The method is the one of "A GPU accelerated Barnes-Hut Tree Code for FLASH4" (arXiv 1509.07370;
 * citations below are lines of /root/reference/PAPER.md): an octree over the cells with per-node
 * total mass and centre of mass (§2, Eq. 5), and a per-target tree
 * walk that applies the opening criterion d > l/theta (Eq. 3) or d > l/theta + delta
 * (Eq. 4) with one vote per warp of 32 neighbouring cells (§3.3) and
 * accumulates Phi_i = -G sum_j m_j/|r_i - r_j| (Eq. 2; the printed factor 1/2 is not
 * applied, reading R1).
 *
 * Conventions (all calls):
 *  - Every function returns BH_OK (0) or a negative BH_ERR_* code; nothing throws, exits or
 *    prints.  bh_strerror() names a code; bh_last_cuda_error() returns the CUDA runtime error
 *    string recorded with the last BH_ERR_CUDA of that context.
 *  - Pointers marked DEVICE must be device memory of the context's device; pointers marked HOST
 *    are ordinary host memory.  The library never frees or keeps caller memory: inputs are
 *    borrowed only for the duration stated, outputs are written on the context's stream.
 *  - Work is enqueued on the stream given to bh_create and is complete when the caller has
 *    synchronised that stream, except where a call is documented as synchronising itself
 *    (bh_build reads two small scalars back; *_host calls and bh_get_stats synchronise).
 *  - One context = one tree = one stream.  A context is not thread-safe.
 *  - There is no CPU fallback: without a CUDA device every compute call fails with BH_ERR_CUDA.
 */
#ifndef BH_H_
#define BH_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bh_ctx bh_ctx;

/* ---- status codes ------------------------------------------------------------------------- */
#define BH_OK               0
#define BH_ERR_INVALID_ARG -1   /* null pointer, n <= 0, n >= 2^31, L <= 0, theta < 0 or NaN, bad option */
#define BH_ERR_NOT_BUILT   -2   /* bh_potential / export / direct before a successful bh_build */
#define BH_ERR_CUDA        -3   /* a CUDA runtime call failed; see bh_last_cuda_error() */
#define BH_ERR_OOM         -4   /* device or host allocation failed */
#define BH_ERR_TOO_LARGE   -5   /* bh_build with 2^30 <= n < 2^31 or n + n_nodes >= 2^32 (32-bit slots; checked in 64 bits
                                   before any node or slot array is sized); bh_potential_direct over all n with n above
                                   BH_DIRECT_ALL_MAX; an output buffer smaller than the result (bh_essential_nodes) */

/* ---- options (bh_set_option) ---------------------------------------------------------------- */
#define BH_OPT_MAC    1   /* opening criterion */
#define BH_MAC_BH86     0 /*   Eq. 3:  accept iff d > l/theta          (default) */
#define BH_MAC_BARNES94 1 /*   Eq. 4:  accept iff d > l/theta + delta              */
#define BH_OPT_GROUP  2   /* how many consecutive Morton-sorted targets share one walk and one vote */
                          /*   32 (default): the paper's warp vote; 1: per-target lists  */
#define BH_OPT_PERIODIC 4    /* 1: the cube of bh_build is a PERIODIC box (App. A): bh_potential uses
                                minimum-image displacements and adds the Ewald field; 0 (default): isolated        */
#define BH_OPT_EWALD_N    5  /* points per axis of each grid of the Ewald field array (6..258, default 66;
                                "gpuEwaldFieldNx/y/z"; one number: the box is a cube)                */
#define BH_OPT_EWALD_NREF 6  /* number of nested grids (1..8, default 1; "gpuEwaldSeriesNref")      */
#define BH_OPT_PASS_TIMING 3 /* 1: bh_build records a CUDA event after every kernel (bh_get_build_passes); a
                                reporting mode -- the events cost a little, 0 (default) records none          */

#define BH_MAX_LEVEL 21               /* 21 key bits per dimension -> 63-bit keys */
#define BH_DIRECT_ALL_MAX (1 << 18)   /* largest n for bh_potential_direct with targets == NULL */

/* ---- statistics ----------------------------------------------------------------------------- */
typedef struct bh_stats {
    int64_t n;                 /* cells of the last build                                            */
    int64_t n_nodes;           /* internal nodes incl. level-21 bucket leaves                          */
    int64_t n_slots;           /* records of the walk array: 1 (root) + sum of child counts           */
    int32_t depth;             /* deepest internal-node level below 21 (0 = root only)                */
    int32_t sort_passes;       /* 8-bit radix passes the last build executed                           */
    int64_t n_clamped;         /* cells with a coordinate outside the cube (clamped into the edge cell) */
    int64_t max_bucket;        /* largest number of cells sharing one 63-bit key (1 = no bucket leaves) */
    int64_t n_accepted;        /* last walk: sum over groups of internal nodes accepted                */
    int64_t n_leaf;            /* last walk: sum over groups of leaf cells summed directly            */
    int64_t n_opened;          /* last walk: sum over groups of internal nodes opened                 */
    int64_t n_exact_tests;     /* last walk: nodes whose vote needed the per-target test (diagnostic)  */
    double  interactions;      /* last walk: sum over TARGETS of the list entries evaluated for their group,
                                  counted by the Phi kernel itself at every list flush (the roofline numerator) */
    /* device time in ms of the passes of the last bh_build / bh_potential (CUDA events) */
    /* device ms of the last build: keys (a1), sort (a2), count = c(s) + level histograms + scan (a4),
     * assign = entity numbering + cells moved into their slots (a4 + a3), moments (a5), whole build.
     * The five phase times are filled only for a build made under BH_OPT_PASS_TIMING (else 0): an event between
     * two kernels would break the chain of dependent launches bh_build issues; ms_build_total is always there. */
    float ms_keys, ms_sort, ms_count, ms_assign, ms_moments, ms_build_total;
    float ms_walk;
    int32_t launches_build;    /* kernels the last bh_build launched                                   */
    int32_t launches_walk;     /* kernels the last bh_potential launched                               */
    int32_t walk_group;        /* BH_OPT_GROUP of the last walk (32 or 1): rows of the per-group outputs = ceil(n / it) */
    double  interactions_counted; /* the same sum as `interactions`, from the count-only repeat of the traversal
                                  ((accepted + leaf) of W6); equal to it unless the Phi kernel lost or doubled an entry */
} bh_stats;

/* ---- life cycle ----------------------------------------------------------------------------- */

/* Creates a context on CUDA device `device`.  `cuda_stream` is a cudaStream_t passed as void*
 * (NULL = the legacy default stream), e.g. torch.cuda.current_stream().cuda_stream; the caller
 * keeps ownership of the stream and must keep it alive until bh_destroy. */
int bh_create(bh_ctx** out, int device, void* cuda_stream);

/* Frees every internal buffer (synchronises the stream first). NULL is accepted. */
int bh_destroy(bh_ctx* ctx);

const char* bh_strerror(int code);
const char* bh_last_cuda_error(const bh_ctx* ctx);

int bh_set_option(bh_ctx* ctx, int key, int value);

/* ---- the hot path --------------------------------------------------------------------------- */

/* bh_build: octree with monopole moments over n point masses (§2; Eq. 5).
 *   x, y, z, m : DEVICE, const double[n] each (SoA, "arrays with a one-dimensional layout",
 *                PAPER.md:96): cell centres and cell masses, caller's ("original") order.
 *                Borrowed until the stream has passed this call; the context keeps sorted copies.
 *   n          : 1 <= n < 2^30 (n in [2^30, 2^31) returns BH_ERR_TOO_LARGE: 30-bit tile counters of the sort,
 *                and n + n_nodes must stay below 2^32; larger or non-positive n is BH_ERR_INVALID_ARG).
 *   cube       : HOST, const double[4] = {x0, y0, z0, L}: the root cube [x0,x0+L) x ....
 *                L > 0.  A coordinate outside the cube is clamped into the edge cell and counted
 *                (bh_stats.n_clamped); NaN coordinates quantise to 0.
 * Steps, all on the device: 63-bit Morton keys (DESIGN.md K-rules) -> stable LSD radix sort of
 * (key, index) -> octree topology from the sorted keys (one cell per leaf, single-child chains kept,
 * identical keys form a level-21 bucket leaf; DESIGN.md T-rules), the cell data being gathered into
 * tree order in the same pass -> bottom-up level-by-level M, R (Eq. 5), delta = |R - geometric
 * centre| in fp64 (DESIGN.md M-rules).
 * Waits on the device internally for (a) which key bits vary and (b) the node count per level -- once when the
 * keys vary on the same bits as in the previous build of this context (the sort is then started on that
 * assumption and checked afterwards), twice otherwise.  A build of as many cells as the previous one also
 * enqueues its last kernels on the previous level totals before that wait (they run only if the device finds the
 * totals unchanged, else they are repeated), so the wait runs under them.  The kernels are issued as chains of
 * programmatic dependent launches on the context's stream; to work enqueued before or after the call they behave
 * like ordinary stream-ordered launches. */
int bh_build(bh_ctx* ctx, const double* x, const double* y, const double* z, const double* m,
             int64_t n, const double cube[4]);

/* bh_update_masses: new masses for the SAME cells (positions unchanged since the last bh_build).
 * An AMR code calls the solver every time step but moves no cell between regrids,
 * so keys, sort and topology of the last build stay valid: only the mass fields of the leaf records
 * and the moments (Eq. 5) are recomputed, with the same arithmetic as bh_build -- a following
 * bh_potential gives bit-identical results to a fresh bh_build with these masses.
 *   m : DEVICE, const double[n], original cell order; borrowed until the stream has passed the call. */
int bh_update_masses(bh_ctx* ctx, const double* m);

/* bh_essential_nodes: Find Essential Nodes (§3.2.4, Fig. 7) -- the tree of the last
 * bh_build pruned against a REMOTE DOMAIN, the first half of the locally-essential-tree exchange
 * (PAPER.md:66, 104-118).  The remote domain (the paper's "VN" with its size) is the axis-aligned box
 * [box_lo, box_hi]; d_c is the distance from a node's centre of mass to the nearest point of that box
 * (0 inside).  From the root: an internal node with d_c > l/theta (BH_MAC_BH86) or d_c > l/theta + delta
 * (BH_MAC_BARNES94, the paper's choice; set with bh_set_option) is essential and is emitted as ONE
 * point mass (R, M); otherwise it is opened; a leaf cell under an opened node is emitted as it is; a
 * level-21 bucket is always opened.  theta = 0 emits all n cells.  Decisions are taken in fp64 on the
 * fp64 moments, so the selected set equals the oracle's exactly.
 *   box_lo, box_hi : HOST, const double[3], box_lo[a] <= box_hi[a].
 *   out            : DEVICE, double[4 * cap], 16-byte aligned: entry k = (x, y, z, m) at out[4k..4k+3]
 *                    (the paper's "exchange array ... holding 4N entries", Fig. 4), in ascending
 *                    (tree level, first sorted cell) order.  May be NULL when cap == 0 (size query).
 *   count          : HOST, receives the number of essential entries (1 ... n).
 * Returns BH_ERR_TOO_LARGE (with *count set, the first cap entries written) when count > cap.
 * Synchronises the stream once to read the count back. */
int bh_essential_nodes(bh_ctx* ctx, const double box_lo[3], const double box_hi[3], double theta,
                       double* out, int64_t cap, int64_t* count);

/* bh_set_num_targets: only the cells with ORIGINAL index < ntargets are targets of the following
 * bh_potential calls; the others are sources only (-1, the default: every cell is a target).  This is
 * how a locally essential tree is walked ("Essential Nodes are treated as data cells
 * during the tree build"): the caller builds over its own cells followed by the received essential
 * entries and sets ntargets = number of its own cells.  Groups are still 32 consecutive cells of the
 * sorted order and every member votes (W-rules unchanged, results identical); groups without a target
 * are skipped, and phi needs only ntargets entries. */
int bh_set_num_targets(bh_ctx* ctx, int64_t ntargets);

/* bh_potential: Phi_i = -G sum_j m_j/|r_i - r_j| over the nodes and leaf cells the group walk of
 * PAPER.md:176-178 selects (DESIGN.md W-rules).
 *   theta : >= 0; theta = 0 opens every node (the result is then the direct sum in fp32 terms).
 *   G     : gravitational constant.
 *   phi   : DEVICE, double[n], ORIGINAL cell order; every element is written.
 * fp32 arithmetic for distances and m/d, accumulated in short fp32 blocks that are flushed into
 * fp64 sums.  Precision contract (W8, W9):
 *  - the opening decision d^2 > r_c^2 of a node is taken in fp32 on fp32-rounded operands, so a node whose
 *    d^2 lies within ~1e-7 relative of r_c^2 for the deciding group member can fall on the other side than
 *    in an fp64 evaluation of Eq. 3 / Eq. 4 ("flip": the group then sums the node's children instead of
 *    the node, or the reverse -- both are valid Barnes-Hut lists; the difference is within the method's
 *    own error).  Tests and bench.py count such groups against the fp64 oracle and report the count.
 *  - positions are held in fp32: a pair at distance d carries a relative distance error up to
 *    ~2^-23 L/d.  Cell centres of grids and AMR meshes (dyadic rationals) are exact; for arbitrary
 *    points the 1e-4 bar on Phi holds while the closest pairs are farther apart than ~1e-3 L. */
int bh_potential(bh_ctx* ctx, double theta, double G, double* phi);

/* Periodic boundaries (BH_OPT_PERIODIC = 1; Appendix A, readings P1-P5).
 * A node or cell of mass M at minimum-image displacement r contributes -G M f_EF(r) (Eq. A.1),
 * f_EF(r) = 1/|r| + corr1(r/L)/L, corr1 = the Ewald sum of 1/r in the unit cube with a neutralising background
 * (Eq. A.2-A.3) minus 1/|u|.  corr1 is tabulated once per context on `nref` nested grids of N^3 points covering
 * the octant u >= 0 (grid k: spacing (1/2)/(N-2)/2^k) and evaluated in the walk by quadratic interpolation
 * around the nearest grid point.  The opening test uses the minimum-image distance.  A target's own
 * cell and distinct cells at zero distance contribute their images and background only, m corr1(0)/L.
 * Restrictions: group walk of all cells only -- BH_OPT_GROUP = 1, bh_field and bh_set_num_targets return
 * BH_ERR_INVALID_ARG while BH_OPT_PERIODIC is on; cells must lie inside the cube.
 *
 * bh_ewald_table: the grid values of corr1 (fp64) as the context computed them, for checking:
 *   out : DEVICE, double[nref * N^3], out[((k_grid * N + k) * N + j) * N + i] = corr1(i h, j h, k h); NULL with cap 0
 *         queries *N and *nref (HOST, may be NULL) and returns BH_ERR_TOO_LARGE. */
int bh_ewald_table(bh_ctx* ctx, double* out, int64_t cap, int* N, int* nref);

/* bh_field: bh_potential plus the acceleration g_i = -grad Phi_i in the same walk (
 * the paper returns Phi only and lets the host code difference it).  The interaction lists,
 * the opening decisions and the arithmetic of Phi are exactly those of bh_potential (phi is bit-equal);
 * every accepted node and leaf cell additionally contributes the gradient of its monopole term,
 *   g_i = -G sum_j m_j (r_i - r_j) / |r_i - r_j|^3     (j != i; zero-distance pairs skipped),
 * evaluated in fp32 with blocked accumulation into fp64 like Phi.
 *   phi : DEVICE, double[n] (or [ntargets]), original order.
 *   acc : DEVICE, double[3 n] (or [3 ntargets]): (gx, gy, gz) of cell i at acc[3i .. 3i+2]. */
int bh_field(bh_ctx* ctx, double theta, double G, double* phi, double* acc);

/* bh_potential_direct: Eq. 2 written out in fp64,
 * Phi_i = -G sum_{j != i} m_j/|r_i - r_j| over ALL n cells of the last build.
 *   targets : DEVICE, const int64_t[nt] original cell indices in [0, n), or NULL for all n cells
 *             (then phi has n elements and n must be <= BH_DIRECT_ALL_MAX, else BH_ERR_TOO_LARGE).
 *             Out-of-range indices make their phi element NaN.
 *   phi     : DEVICE, double[nt] (or double[n]); phi[a] belongs to targets[a].
 * Pairs of distinct cells at zero distance are skipped. */
int bh_potential_direct(bh_ctx* ctx, double G, const int64_t* targets, int64_t nt, double* phi);

/* bh_direct_noalloc: the same direct sum (Eq. 2; fp64; zero-distance pairs skipped) WITHOUT a context
 * and WITHOUT any allocation, for callers that cannot call cudaMalloc (CUDA graph capture, serving loops, harnesses
 * that forbid it).  The packed (x, y, z, m) copy of the cells that bh_potential_direct allocates in its context
 * lives here in a file-scope static __device__ array of BH_NOALLOC_MAX_N records (1 MiB per GPU that loads libbh,
 * held until the process exits).  The call enqueues two kernels on `cuda_stream` and returns; it does not
 * synchronise, allocate, free, or create streams / events.  (The first call on a device looks up the array's device
 * address, cudaGetSymbolAddress: make that call outside a stream capture.)
 *   device      : CUDA device ordinal (made current for the call, the previous device is restored)
 *   cuda_stream : cudaStream_t, or NULL for the default stream
 *   x, y, z, m  : DEVICE, const double[n], read only, original order
 *   n           : 0 <= n <= BH_NOALLOC_MAX_N; larger n returns BH_ERR_TOO_LARGE (nothing is launched), n = 0 is BH_OK
 *   phi         : DEVICE, double[n], phi[i] = -G sum_{j != i} m_j/|r_i - r_j|, original order
 * Every call on a device shares the one array and leaves its records in it: the next call overwrites what it reads,
 * nothing has to be cleared.  Calls that OVERLAP on the GPU (different streams without ordering, several host
 * threads) race on it: order them.  Errors: BH_ERR_INVALID_ARG / BH_ERR_TOO_LARGE / BH_ERR_CUDA;
 * bh_noalloc_last_error() returns the calling thread's last message (there is no context to keep it). */
#define BH_NOALLOC_MAX_N 32768
int bh_direct_noalloc(int device, void* cuda_stream, const double* x, const double* y, const double* z, const double* m,
                      int64_t n, double G, double* phi);
const char* bh_noalloc_last_error(void);

/* One call with HOST buffers: copies x, y, z, m (double[n] each, pageable or pinned) to the
 * device, runs bh_build and bh_potential, copies phi (double[n]) back, synchronises ("Only position and
 * mass data is copied to the device ... just results are copied back").
 * The copies run on a stream of their own, positions first: keys, sort and the entity counting start when
 * x, y, z have landed and run beside the copy of m; the first kernel that reads a mass waits for it.
 * Pinned (page-locked) buffers are copied in one asynchronous DMA each and overlap with the kernels; pageable
 * ones are staged by the CUDA runtime (about 11 GB/s, no overlap): pin the buffers of a solver called every step. */
int bh_solve_host(bh_ctx* ctx, const double* x, const double* y, const double* z, const double* m,
                  int64_t n, const double cube[4], double theta, double G, double* phi);

/* Device-side time split of the last bh_solve_host (HOST output, milliseconds, CUDA events):
 * ms[0] host->device copies (all four arrays), ms[1] build + walk (from the arrival of x, y, z to the end of
 * the walk; includes any wait for m), ms[2] device->host copy of phi, ms[3] the whole call.
 * ms[0] + ms[1] + ms[2] - ms[3] is the time the copies and the kernels overlapped. */
int bh_host_breakdown(bh_ctx* ctx, float ms[4]);

/* ---- parity / reporting --------------------------------------------------------------------- */

/* One kernel (or small group of kernels) of the last bh_build, in launch order, when BH_OPT_PASS_TIMING was on:
 * its device time and its ALGORITHMIC bytes by SURVEY.md §8(d) -- keys 36 B/cell; sort_hist 8 B/cell; each
 * sort_pass 24 B/cell; topo_count 8 B/cell; topo_scan 0 (bookkeeping on the chunk histograms); assign_permute
 * 84 B/cell + 24 B/node; moments_L<level> 32 B per leaf-cell child + 72 B per node of that level. */
typedef struct bh_pass {
    char   name[24];
    float  ms;
    double alg_bytes;
} bh_pass;

/* Fills out[0 .. min(cap, *count)) (HOST) with the passes of the last bh_build; *count = number recorded.
 * Synchronises the stream.  BH_ERR_TOO_LARGE when cap is too small (the first cap entries are written). */
int bh_get_build_passes(bh_ctx* ctx, bh_pass* out, int cap, int* count);

/* Sizes of the last build (HOST outputs, any may be NULL). */
int bh_tree_sizes(const bh_ctx* ctx, int64_t* n, int64_t* n_nodes, int64_t* n_slots);

/* bh_export_tree: copies the tree of the last build into caller DEVICE buffers (any may be NULL).
 *   keys[n]  : sorted 63-bit Morton keys            perm[n] : original index of sorted slot s
 * and, for the n_nodes internal nodes (incl. level-21 buckets) in CANONICAL order = ascending
 * (level, prefix) (T5):
 *   level[i] (int32), prefix[i] (uint64 = key >> 3*(21-level)), lo[i], hi[i] (int64: sorted cell
 *   range [lo, hi)), nchild[i] (int32; for a bucket the number of cells), M[i], Rx[i], Ry[i],
 *   Rz[i], delta[i] (double). */
int bh_export_tree(bh_ctx* ctx, uint64_t* keys, uint32_t* perm, int32_t* level, uint64_t* prefix,
                   int64_t* lo, int64_t* hi, int32_t* nchild, double* M, double* Rx, double* Ry,
                   double* Rz, double* delta);

/* Per-group counts of the last bh_potential: DEVICE int64[3 * ngroups], ngroups =
 * ceil(n / group), group g at [3g..3g+2] = {internal nodes accepted, leaf cells summed, internal
 * nodes opened}; same definition as the oracle's counters (W6). */
int bh_last_group_counts(bh_ctx* ctx, int64_t* counts);

/* The number of interaction-list entries the Phi kernel of the last bh_potential / bh_field itself
 * evaluated for each group (counted at every list flush of the timed kernel, not by the count-only
 * repeat that serves bh_last_group_counts): DEVICE uint32[ngroups].  Equals accepted + leaf of W6. */
int bh_last_group_evaluated(bh_ctx* ctx, uint32_t* per_group);

/* BH_OPT_GROUP of the last walk (32 or 1), or a negative BH_ERR_*: sizes the per-group outputs. */
int bh_last_walk_group(const bh_ctx* ctx);

/* Interactions evaluated for each target in the last bh_potential (accepted + leaf of its group;
 * the target's own cell is counted as evaluated-and-masked): DEVICE uint32[n], original order. */
int bh_last_interactions(bh_ctx* ctx, uint32_t* per_target);

/* Synchronises the stream and fills *out (HOST). */
int bh_get_stats(bh_ctx* ctx, bh_stats* out);

#ifdef __cplusplus
}
#endif
#endif /* BH_H_ */
