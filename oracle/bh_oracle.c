/*
 * bh_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded fp64 CPU Barnes-Hut written from the paper
 * (arxiv 1509.07370, /root/reference/PAPER.md) and the readings of SURVEY.md §8(c) / DESIGN.md.
 * It shares no code, header, table or helper with the CUDA library under paper_1509_07370_b200/.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * call it.  Compile with:  gcc -O2 -ffp-contract=off -fPIC -shared -o libbh_oracle.so bh_oracle.c -lm
 * (-ffp-contract=off: the key expression below must not be fused, K-rule 1).
 *
 * What each function follows:
 *   orc_keys      63-bit Morton key of a point in the caller's cube.  The paper only names the
 *                 Morton curve; the exact expression is DESIGN.md reading K1-K2.
 *   orc_build     keys -> stable sort by (key, index) -> octree "recursively divided into eight sub
 *                 cells ... until only one particle is left for every sub cell" (§2);
 *                 per node total mass and centre of mass, Eq. 5, and
 *                 delta = |com - geometric centre|.
 *   orc_potential stack-based depth-first walk (§3.3) with the opening test
 *                 d > l/theta (Eq. 3) or d > l/theta + delta (Eq. 4);
 *                 a group of `group` consecutive sorted targets shares the walk and a node is used
 *                 only if EVERY member accepts it (the all() vote).
 *                 Phi_i = -G sum m_j/|r_i - r_j| (Eq. 2, without the printed 1/2: reading).
 *   orc_direct    Eq. 2 written out: Phi_i = -G sum_{j != i} m_j/|r_i - r_j|.
 *   orc_essential_nodes  Find Essential Nodes (§3.2.4): the tree pruned against a remote
 *                 domain box with the minimum-distance form of the opening test (E1-E4).
 *   orc_field / orc_direct_acc  the acceleration g = -grad Phi on the walk's own interaction lists and by
 *                 direct summation (the Phi arithmetic of orc_potential is untouched).
 *   orc_ewald_psi / orc_ewald_corr / orc_ewald_table / orc_ewald_interp / orc_potential_periodic
 *                 periodic boundaries (App. A, Eq. A.1-A.3): the Ewald
 *                 field of 1/r in a cubic box, its nested-grid table, quadratic interpolation, and the group
 *                 walk with minimum-image displacements (readings P1-P5).
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): keys vs closed form on 2^k grids and a per-bit
 * interleave; tree vs a recursive brute-force partition in numpy; node counts (n-1)/7 on grids;
 * moments vs flat sums; theta=0 walk == direct sum bit for bit in sorted order; convergence with
 * theta; uniform-sphere and MacLaurin closed forms; essential nodes vs a brute-force partition on integer
 * coordinates, the 1..n limits of PAPER.md:106, mass conservation and the potential inside the box
 * (tests/test_oracle_essential.py); accelerations vs a numpy brute force, the numerical gradient of the
 * direct-sum potential, Newton's third law and the two-body / uniform-sphere closed forms
 * (tests/test_oracle_field.py); the Ewald field vs its independence of alpha over a decade, a brute-force
 * shell-summed lattice sum, the simple-cubic Madelung constant 2.8372974795, zero mean against the cube
 * constant 2.3800774, the Laplacian 4 pi, cubic symmetry and periodicity; the table and its interpolation vs
 * the exact field; the periodic walk vs the exact Ewald direct sum, translation invariance and the closed
 * form of a uniform periodic lattice (tests/test_oracle_ewald.py); the mac_fp32 branch of group_accepts vs
 * an independent numpy-float32 restatement incl. one-ulp threshold scans (tests/test_oracle_walk.py,
 * tests/fp32_decision.py).  No function here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_MAXLEVEL 21
#define ORC_MAC_BH86 0     /* Eq. 3 */
#define ORC_MAC_BARNES94 1 /* Eq. 4 */

typedef struct {
    int32_t level;       /* 0 = root; 21 = bucket leaf (>= 2 cells with identical keys) */
    uint64_t prefix;     /* key >> 3*(21-level) */
    int64_t lo, hi;      /* sorted cell range [lo, hi) */
    int64_t child[8];    /* per octant: -1 absent; >= 0 node index; <= -2 leaf cell with sorted slot -(c+2) */
    double M, R[3];      /* Eq. 5 */
    double delta;        /* |R - geometric centre| */
    double size;         /* l = L / 2^level */
    double centre[3];    /* geometric centre */
} orc_node;

typedef struct {
    int64_t n;
    double cube[4];
    uint64_t *key;       /* sorted keys */
    uint32_t *perm;      /* perm[s] = original index of sorted slot s */
    double *x, *y, *z, *m; /* sorted copies */
    orc_node *node;
    int64_t n_nodes, cap_nodes;
    int64_t n_clamped;
    int32_t depth;       /* deepest internal-node level */
} orc_tree;

/* ---- keys (K1-K2) ------------------------------------------------------------------ */
static uint64_t quantise(double v, double v0, double s, int *clamped)
{
    /* t = (v - v0) * s : one subtract, one multiply, round-to-nearest, no contraction */
    double d = v - v0;
    double t = d * s;
    double f = floor(t);
    if (!(f >= 0.0)) { /* negative or NaN */
        if (clamped) *clamped = 1;
        return 0;
    }
    if (f > 2097151.0) {
        if (clamped) *clamped = 1;
        return 2097151u;
    }
    return (uint64_t)f;
}

static uint64_t interleave3(uint64_t qx, uint64_t qy, uint64_t qz)
{
    /* bit (3k+0) = bit k of qx, (3k+1) = bit k of qy, (3k+2) = bit k of qz, k = 0..20 */
    uint64_t key = 0;
    for (int k = 0; k < 21; ++k) {
        key |= ((qx >> k) & 1ull) << (3 * k + 0);
        key |= ((qy >> k) & 1ull) << (3 * k + 1);
        key |= ((qz >> k) & 1ull) << (3 * k + 2);
    }
    return key;
}

int orc_keys(const double *x, const double *y, const double *z, int64_t n, const double *cube,
             uint64_t *keys, int64_t *n_clamped)
{
    if (!x || !y || !z || !cube || !keys || n < 0 || !(cube[3] > 0.0)) return -1;
    double s = 2097152.0 / cube[3];
    int64_t nc = 0;
    for (int64_t i = 0; i < n; ++i) {
        int c = 0;
        uint64_t qx = quantise(x[i], cube[0], s, &c);
        uint64_t qy = quantise(y[i], cube[1], s, &c);
        uint64_t qz = quantise(z[i], cube[2], s, &c);
        keys[i] = interleave3(qx, qy, qz);
        nc += c;
    }
    if (n_clamped) *n_clamped = nc;
    return 0;
}

/* ---- sort (S-rule): ascending key, ties by ascending original index -------------------------- */
typedef struct { uint64_t key; uint32_t idx; } orc_kv;

static int cmp_kv(const void *a, const void *b)
{
    const orc_kv *p = (const orc_kv *)a, *q = (const orc_kv *)b;
    if (p->key < q->key) return -1;
    if (p->key > q->key) return 1;
    if (p->idx < q->idx) return -1;
    if (p->idx > q->idx) return 1;
    return 0;
}

int orc_sort(const uint64_t *keys, int64_t n, uint32_t *perm)
{
    if (!keys || !perm || n < 0) return -1;
    orc_kv *kv = (orc_kv *)malloc(sizeof(orc_kv) * (size_t)(n > 0 ? n : 1));
    if (!kv) return -2;
    for (int64_t i = 0; i < n; ++i) { kv[i].key = keys[i]; kv[i].idx = (uint32_t)i; }
    qsort(kv, (size_t)n, sizeof(orc_kv), cmp_kv);
    for (int64_t i = 0; i < n; ++i) perm[i] = kv[i].idx;
    free(kv);
    return 0;
}

/* ---- tree (T-rules) and moments (M-rules) ---------------------------------------------------- */
static int64_t new_node(orc_tree *t)
{
    if (t->n_nodes == t->cap_nodes) {
        int64_t cap = t->cap_nodes ? 2 * t->cap_nodes : 1024;
        orc_node *p = (orc_node *)realloc(t->node, sizeof(orc_node) * (size_t)cap);
        if (!p) return -1;
        t->node = p;
        t->cap_nodes = cap;
    }
    return t->n_nodes++;
}

/* Builds the node owning sorted range [lo, hi) (hi - lo >= 2) at `level`; returns its index.
 * the cube "is then recursively divided into eight sub cells ... until only one
 * particle is left for every sub cell".  Single-child chains are kept (T-rule 2). */
static int64_t build_node(orc_tree *t, int32_t level, int64_t lo, int64_t hi)
{
    int64_t id = new_node(t);
    if (id < 0) return -1;
    {
        orc_node *nd = &t->node[id];
        nd->level = level;
        nd->prefix = (level == 0) ? 0 : (t->key[lo] >> (3 * (ORC_MAXLEVEL - level)));
        nd->lo = lo;
        nd->hi = hi;
        for (int c = 0; c < 8; ++c) nd->child[c] = -1;
        /* geometric centre (T-rule 4): de-interleave the prefix */
        uint64_t px = 0, py = 0, pz = 0;
        for (int k = 0; k < level; ++k) {
            px |= ((nd->prefix >> (3 * k + 0)) & 1ull) << k;
            py |= ((nd->prefix >> (3 * k + 1)) & 1ull) << k;
            pz |= ((nd->prefix >> (3 * k + 2)) & 1ull) << k;
        }
        nd->size = ldexp(t->cube[3], -level);
        nd->centre[0] = t->cube[0] + ((double)px + 0.5) * nd->size;
        nd->centre[1] = t->cube[1] + ((double)py + 0.5) * nd->size;
        nd->centre[2] = t->cube[2] + ((double)pz + 0.5) * nd->size;
        nd->M = 0.0;
        nd->R[0] = nd->R[1] = nd->R[2] = 0.0;
        nd->delta = 0.0;
    }
    if (level > t->depth && level < ORC_MAXLEVEL) t->depth = level;

    double M = 0.0, S[3] = {0.0, 0.0, 0.0};
    if (level == ORC_MAXLEVEL) {
        /* bucket leaf (T-rule 3): cells with identical keys; moments from the cells in order */
        for (int64_t s = lo; s < hi; ++s) {
            M += t->m[s];
            S[0] += t->m[s] * t->x[s];
            S[1] += t->m[s] * t->y[s];
            S[2] += t->m[s] * t->z[s];
        }
    } else {
        int shift = 3 * (ORC_MAXLEVEL - level - 1);
        int64_t a = lo;
        while (a < hi) {
            int oct = (int)((t->key[a] >> shift) & 7ull);
            int64_t b = a + 1;
            while (b < hi && (int)((t->key[b] >> shift) & 7ull) == oct) ++b;
            if (b - a == 1) {
                t->node[id].child[oct] = -(a + 2); /* leaf cell, sorted slot a */
                M += t->m[a];
                S[0] += t->m[a] * t->x[a];
                S[1] += t->m[a] * t->y[a];
                S[2] += t->m[a] * t->z[a];
            } else {
                int64_t c = build_node(t, level + 1, a, b);
                if (c < 0) return -1;
                t->node[id].child[oct] = c;
                /* Eq. 5 from the children's moments, ascending octant order (M-rule 1) */
                M += t->node[c].M;
                S[0] += t->node[c].M * t->node[c].R[0];
                S[1] += t->node[c].M * t->node[c].R[1];
                S[2] += t->node[c].M * t->node[c].R[2];
            }
            a = b;
        }
    }
    orc_node *nd = &t->node[id];
    nd->M = M;
    if (M != 0.0) {
        nd->R[0] = S[0] / M; /* Eq. 5: R = (1/M) sum m_i r_i */
        nd->R[1] = S[1] / M;
        nd->R[2] = S[2] / M;
        double ex = nd->R[0] - nd->centre[0], ey = nd->R[1] - nd->centre[1], ez = nd->R[2] - nd->centre[2];
        nd->delta = sqrt(ex * ex + ey * ey + ez * ez);
    } else { /* M-rule 2: zero-mass node */
        nd->R[0] = nd->centre[0];
        nd->R[1] = nd->centre[1];
        nd->R[2] = nd->centre[2];
        nd->delta = 0.0;
    }
    return id;
}

void orc_free(orc_tree *t)
{
    if (!t) return;
    free(t->key); free(t->perm); free(t->x); free(t->y); free(t->z); free(t->m); free(t->node);
    free(t);
}

orc_tree *orc_build(const double *x, const double *y, const double *z, const double *m, int64_t n,
                    const double *cube)
{
    if (!x || !y || !z || !m || !cube || n <= 0 || n >= 2147483648ll || !(cube[3] > 0.0)) return NULL;
    orc_tree *t = (orc_tree *)calloc(1, sizeof(orc_tree));
    if (!t) return NULL;
    t->n = n;
    memcpy(t->cube, cube, sizeof(double) * 4);
    uint64_t *k0 = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)n);
    t->key = (uint64_t *)malloc(sizeof(uint64_t) * (size_t)n);
    t->perm = (uint32_t *)malloc(sizeof(uint32_t) * (size_t)n);
    t->x = (double *)malloc(sizeof(double) * (size_t)n);
    t->y = (double *)malloc(sizeof(double) * (size_t)n);
    t->z = (double *)malloc(sizeof(double) * (size_t)n);
    t->m = (double *)malloc(sizeof(double) * (size_t)n);
    if (!k0 || !t->key || !t->perm || !t->x || !t->y || !t->z || !t->m) { free(k0); orc_free(t); return NULL; }
    orc_keys(x, y, z, n, cube, k0, &t->n_clamped);
    if (orc_sort(k0, n, t->perm) != 0) { free(k0); orc_free(t); return NULL; }
    for (int64_t s = 0; s < n; ++s) {
        uint32_t i = t->perm[s];
        t->key[s] = k0[i];
        t->x[s] = x[i]; t->y[s] = y[i]; t->z[s] = z[i]; t->m[s] = m[i];
    }
    free(k0);
    t->depth = 0;
    if (n >= 2) { /* T-rule 1: root is an internal node iff n >= 2 */
        if (build_node(t, 0, 0, n) < 0) { orc_free(t); return NULL; }
    }
    return t;
}

int64_t orc_num_cells(const orc_tree *t) { return t ? t->n : -1; }
int64_t orc_num_nodes(const orc_tree *t) { return t ? t->n_nodes : -1; }  /* incl. level-21 buckets */
int64_t orc_num_clamped(const orc_tree *t) { return t ? t->n_clamped : -1; }
int32_t orc_depth(const orc_tree *t) { return t ? t->depth : -1; }

int orc_get_sorted(const orc_tree *t, uint64_t *keys, uint32_t *perm)
{
    if (!t) return -1;
    if (keys) memcpy(keys, t->key, sizeof(uint64_t) * (size_t)t->n);
    if (perm) memcpy(perm, t->perm, sizeof(uint32_t) * (size_t)t->n);
    return 0;
}

/* canonical order (T-rule 5): by (level, prefix) */
typedef struct { int32_t level; uint64_t prefix; int64_t id; } orc_ord;
static int cmp_ord(const void *a, const void *b)
{
    const orc_ord *p = (const orc_ord *)a, *q = (const orc_ord *)b;
    if (p->level != q->level) return p->level < q->level ? -1 : 1;
    if (p->prefix != q->prefix) return p->prefix < q->prefix ? -1 : 1;
    return 0;
}

/* Fills caller arrays of length orc_num_nodes() in canonical order.  Any pointer may be NULL. */
int orc_export_nodes(const orc_tree *t, int32_t *level, uint64_t *prefix, int64_t *lo, int64_t *hi,
                     double *M, double *Rx, double *Ry, double *Rz, double *delta, int32_t *nchild)
{
    if (!t) return -1;
    int64_t nn = t->n_nodes;
    orc_ord *o = (orc_ord *)malloc(sizeof(orc_ord) * (size_t)(nn > 0 ? nn : 1));
    if (!o) return -2;
    for (int64_t i = 0; i < nn; ++i) { o[i].level = t->node[i].level; o[i].prefix = t->node[i].prefix; o[i].id = i; }
    qsort(o, (size_t)nn, sizeof(orc_ord), cmp_ord);
    for (int64_t i = 0; i < nn; ++i) {
        const orc_node *nd = &t->node[o[i].id];
        if (level) level[i] = nd->level;
        if (prefix) prefix[i] = nd->prefix;
        if (lo) lo[i] = nd->lo;
        if (hi) hi[i] = nd->hi;
        if (M) M[i] = nd->M;
        if (Rx) Rx[i] = nd->R[0];
        if (Ry) Ry[i] = nd->R[1];
        if (Rz) Rz[i] = nd->R[2];
        if (delta) delta[i] = nd->delta;
        if (nchild) {
            int c = 0;
            if (nd->level == ORC_MAXLEVEL) c = (int)(nd->hi - nd->lo);
            else for (int k = 0; k < 8; ++k) c += nd->child[k] != -1;
            nchild[i] = c;
        }
    }
    free(o);
    return 0;
}

/* ---- walk (W-rules) ---------------------------------------------------------------------------- */
/* A leaf cell j reached through an opened parent: every member t != j adds m_j/|r_t - r_j|
 * (Eq. 2, j != i by sorted slot; distinct cells at zero distance are skipped, W-rule 3). */
/* g (may be NULL): per member 3 sums of m_j (r_j - r_t)/d^3, the acceleration before the factor G
 * (NEXT-4: g_t = -grad Phi_t = -G sum_j m_j (r_t - r_j)/|r_t - r_j|^3). */
static void add_leaf_cell(const orc_tree *t, int64_t j, int64_t t0, int nt, double *acc, double *g)
{
    for (int a = 0; a < nt; ++a) {
        int64_t s = t0 + a;
        if (s == j) continue;
        double dx = t->x[s] - t->x[j], dy = t->y[s] - t->y[j], dz = t->z[s] - t->z[j];
        double d2 = dx * dx + dy * dy + dz * dz;
        if (d2 == 0.0) continue;
        acc[a] += t->m[j] / sqrt(d2);
        if (g) {
            double w = t->m[j] / (d2 * sqrt(d2));
            g[3 * a + 0] -= w * dx; g[3 * a + 1] -= w * dy; g[3 * a + 2] -= w * dz;
        }
    }
}

/* Is node nd accepted by EVERY member of the group (the all() vote)?
 * Eq. 3: d > l/theta;  Eq. 4: d > l/theta + delta;  compared as d^2 > r_c^2, strict. */
static int group_accepts(const orc_tree *t, const orc_node *nd, double theta, int mac, int mac_fp32,
                         int64_t t0, int nt)
{
    if (theta == 0.0) return 0; /* r_c = +inf: open everything */
    if (!mac_fp32) {
        double rc = nd->size / theta;
        if (mac == ORC_MAC_BARNES94) rc += nd->delta;
        double rc2 = rc * rc;
        for (int a = 0; a < nt; ++a) {
            int64_t s = t0 + a;
            double dx = t->x[s] - nd->R[0], dy = t->y[s] - nd->R[1], dz = t->z[s] - nd->R[2];
            double d2 = dx * dx + dy * dy + dz * dz;
            if (!(d2 > rc2)) return 0;
        }
        return 1;
    }
    /* mac_fp32: the decision taken in the kernel's arithmetic type (reading W8):
     * operands rounded to fp32, r_c = l*(1/theta) (+ delta), d2 = fma(dz,dz,fma(dy,dy,dx*dx)). */
    float rc = (float)nd->size * (float)(1.0 / theta);
    if (mac == ORC_MAC_BARNES94) rc = rc + (float)nd->delta;
    float rc2 = rc * rc;
    float nx = (float)nd->R[0], ny = (float)nd->R[1], nz = (float)nd->R[2];
    for (int a = 0; a < nt; ++a) {
        int64_t s = t0 + a;
        float dx = (float)t->x[s] - nx, dy = (float)t->y[s] - ny, dz = (float)t->z[s] - nz;
        float d2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        if (!(d2 > rc2)) return 0;
    }
    return 1;
}

/* Walks groups [group_begin, group_end) of `group` consecutive sorted targets (W-rule 1).
 * phi_orig: length n, ORIGINAL order; only the walked targets are written.
 * counts (may be NULL): per walked group {accepted nodes, leaf cells summed, opened nodes}. */
static int walk_groups(const orc_tree *t, double theta, double G, int mac, int group, int mac_fp32,
                       int64_t group_begin, int64_t group_end, double *phi_orig, int64_t *counts,
                       double *acc_orig /* NULL or [3n]: (gx, gy, gz) per cell, ORIGINAL order */)
{
    if (!t || !phi_orig || !(theta >= 0.0) || group < 1) return -1;
    int64_t n = t->n;
    int64_t ngroups = (n + group - 1) / group;
    if (group_end < 0 || group_end > ngroups) group_end = ngroups;
    if (group_begin < 0) group_begin = 0;
    /* stack of child references: >= 0 internal node / bucket index, <= -2 leaf cell -(slot+2).
     * depth-first: at most 7 waiting siblings per level plus the current entry */
    int64_t stack[8 * (ORC_MAXLEVEL + 2)];
    double *acc = (double *)malloc(sizeof(double) * (size_t)group);
    double *gr = acc_orig ? (double *)malloc(sizeof(double) * 3 * (size_t)group) : NULL;
    if (!acc || (acc_orig && !gr)) { free(acc); free(gr); return -2; }
    for (int64_t g = group_begin; g < group_end; ++g) {
        int64_t t0 = g * group, t1 = t0 + group;
        if (t1 > n) t1 = n;
        int nt = (int)(t1 - t0);
        for (int a = 0; a < nt; ++a) acc[a] = 0.0;
        if (gr) for (int a = 0; a < 3 * nt; ++a) gr[a] = 0.0;
        int64_t n_acc = 0, n_leaf = 0, n_open = 0;
        int sp = 0;
        if (n >= 2) stack[sp++] = 0; /* root tested like any other node (W-rule 2); n = 1: Phi = 0 */
        while (sp > 0) {
            int64_t e = stack[--sp];
            if (e <= -2) { /* leaf cell */
                add_leaf_cell(t, -(e + 2), t0, nt, acc, gr);
                ++n_leaf;
                continue;
            }
            const orc_node *nd = &t->node[e];
            if (nd->level == ORC_MAXLEVEL) { /* bucket leaf: all its cells summed directly (T-rule 3) */
                for (int64_t j = nd->lo; j < nd->hi; ++j) {
                    add_leaf_cell(t, j, t0, nt, acc, gr);
                    ++n_leaf;
                }
                continue;
            }
            if (group_accepts(t, nd, theta, mac, mac_fp32, t0, nt)) {
                for (int a = 0; a < nt; ++a) { /* every member adds M_N/|r_t - R_N| */
                    int64_t s = t0 + a;
                    double dx = t->x[s] - nd->R[0], dy = t->y[s] - nd->R[1], dz = t->z[s] - nd->R[2];
                    acc[a] += nd->M / sqrt(dx * dx + dy * dy + dz * dz);
                    if (gr) { /* the node acts as the point mass (R, M) */
                        double d2 = dx * dx + dy * dy + dz * dz;
                        double w = nd->M / (d2 * sqrt(d2));
                        gr[3 * a + 0] -= w * dx; gr[3 * a + 1] -= w * dy; gr[3 * a + 2] -= w * dz;
                    }
                }
                ++n_acc;
                continue;
            }
            ++n_open; /* opened for the whole group: children pop in ascending octant order */
            for (int c = 7; c >= 0; --c)
                if (nd->child[c] != -1) stack[sp++] = nd->child[c];
        }
        for (int a = 0; a < nt; ++a) phi_orig[t->perm[t0 + a]] = -G * acc[a]; /* W-rule 4 */
        if (gr)
            for (int a = 0; a < nt; ++a)
                for (int k = 0; k < 3; ++k) acc_orig[3 * (int64_t)t->perm[t0 + a] + k] = G * gr[3 * a + k];
        if (counts) {
            int64_t *c = counts + 3 * (g - group_begin);
            c[0] = n_acc; c[1] = n_leaf; c[2] = n_open;
        }
    }
    free(acc);
    free(gr);
    return 0;
}

int orc_potential(const orc_tree *t, double theta, double G, int mac, int group, int mac_fp32,
                  int64_t group_begin, int64_t group_end, double *phi_orig, int64_t *counts)
{
    return walk_groups(t, theta, G, mac, group, mac_fp32, group_begin, group_end, phi_orig, counts, NULL);
}

/* NEXT-4 (the paper returns Phi and lets the host code difference it):
 * the same walk, the same interaction lists, additionally g_t = -grad Phi_t evaluated on every
 * accepted node and leaf cell as the gradient of its monopole term: -G M (r_t - R)/|r_t - R|^3. */
int orc_field(const orc_tree *t, double theta, double G, int mac, int group, int mac_fp32,
              int64_t group_begin, int64_t group_end, double *phi_orig, double *acc_orig, int64_t *counts)
{
    if (!acc_orig) return -1;
    return walk_groups(t, theta, G, mac, group, mac_fp32, group_begin, group_end, phi_orig, counts, acc_orig);
}

/* ---- direct summation, Eq. 2 written out ------------------------------------------
 * Phi_i = -G sum_{j != i} m_j/|r_i - r_j| over ALL n sources, for the listed targets (original
 * indices; targets == NULL: all n, phi has length n).  Sources are visited in original order.
 * Distinct cells at zero distance are skipped, as in the walk. */
int orc_direct(const double *x, const double *y, const double *z, const double *m, int64_t n, double G,
               const int64_t *targets, int64_t nt, double *phi)
{
    if (!x || !y || !z || !m || !phi || n <= 0) return -1;
    int64_t count = targets ? nt : n;
    for (int64_t a = 0; a < count; ++a) {
        int64_t i = targets ? targets[a] : a;
        if (i < 0 || i >= n) return -1;
        double s = 0.0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double dx = x[i] - x[j], dy = y[i] - y[j], dz = z[i] - z[j];
            double d2 = dx * dx + dy * dy + dz * dz;
            if (d2 == 0.0) continue;
            s += m[j] / sqrt(d2);
        }
        phi[a] = -G * s;
    }
    return 0;
}

/* ---- Find Essential Nodes (§3.2.4, Fig. 7) -------------
 * The local tree pruned against a remote domain: "Nodes and data cells are treated as essential if
 * they pass the opening angle test ... a slightly modified version of the opening angle criterion ...
 * we refer to the minimum distance d_c between the nodes center of mass and the VN".
 * Reading (E1-E4): the remote domain ("VN" extent) is the axis-aligned box [blo, bhi];
 * d_c = distance from the node's centre of mass R to the nearest point of the box (0 inside it).
 * Depth-first from the root: an internal node with d_c > l/theta (+ delta with Eq. 4) is essential
 * and is sent as ONE point mass (R, M); otherwise it is opened and its children are examined; a
 * leaf cell reached through an opened parent is essential as it is; a level-21 bucket is always
 * opened (all its cells are sent).  theta = 0 opens everything (all n cells are sent).  Decisions
 * in fp64, compared as d_c^2 > r_c^2 (strict), every product and sum rounded separately.
 * Output: entries in ascending (level, first sorted cell) order -- level of a leaf cell = its
 * parent's level + 1 -- as rec[4k..4k+3] = (x, y, z, m) ("exchange array ... 4N entries", Fig. 4),
 * plus (optionally) level[k], lo[k], hi[k] (sorted cell range the entry stands for).
 * Returns the number of entries (they never exceed n), or < 0 on a bad argument. */
typedef struct { int32_t level; int64_t lo, hi; double r[4]; } orc_ess;

static int cmp_ess(const void *a, const void *b)
{
    const orc_ess *p = (const orc_ess *)a, *q = (const orc_ess *)b;
    if (p->level != q->level) return p->level < q->level ? -1 : 1;
    if (p->lo != q->lo) return p->lo < q->lo ? -1 : 1;
    return 0;
}

static double box_dist2(const double R[3], const double *blo, const double *bhi)
{
    double d2 = 0.0;
    for (int a = 0; a < 3; ++a) {
        double d = 0.0;
        if (R[a] < blo[a]) d = blo[a] - R[a];
        else if (R[a] > bhi[a]) d = R[a] - bhi[a];
        d2 = d2 + d * d;
    }
    return d2;
}

int64_t orc_essential_nodes(const orc_tree *t, const double *blo, const double *bhi, double theta, int mac,
                            double *rec, int32_t *level, int64_t *lo, int64_t *hi)
{
    if (!t || !blo || !bhi || !rec || !(theta >= 0.0)) return -1;
    for (int a = 0; a < 3; ++a) if (!(blo[a] <= bhi[a])) return -1;
    int64_t n = t->n;
    orc_ess *out = (orc_ess *)malloc(sizeof(orc_ess) * (size_t)(n > 0 ? n : 1));
    if (!out) return -2;
    int64_t cnt = 0;
    if (n == 1) { /* a lone cell has no tree (T-rule 1): it is sent as it is */
        orc_ess e = {1, 0, 1, {t->x[0], t->y[0], t->z[0], t->m[0]}};
        out[cnt++] = e;
    }
    int64_t stack[8 * (ORC_MAXLEVEL + 2)];
    int32_t slev[8 * (ORC_MAXLEVEL + 2)]; /* level of the stacked child reference */
    int sp = 0;
    if (n >= 2) { stack[sp] = 0; slev[sp] = 0; ++sp; }
    while (sp > 0) {
        --sp;
        int64_t e = stack[sp];
        int32_t lev = slev[sp];
        if (e <= -2) { /* leaf cell */
            int64_t j = -(e + 2);
            orc_ess q = {lev, j, j + 1, {t->x[j], t->y[j], t->z[j], t->m[j]}};
            out[cnt++] = q;
            continue;
        }
        const orc_node *nd = &t->node[e];
        if (nd->level == ORC_MAXLEVEL) { /* bucket: always opened */
            for (int64_t j = nd->lo; j < nd->hi; ++j) {
                orc_ess q = {ORC_MAXLEVEL + 1, j, j + 1, {t->x[j], t->y[j], t->z[j], t->m[j]}};
                out[cnt++] = q;
            }
            continue;
        }
        int accept = 0;
        if (theta > 0.0) {
            double rc = nd->size / theta;
            if (mac == ORC_MAC_BARNES94) rc = rc + nd->delta;
            accept = box_dist2(nd->R, blo, bhi) > rc * rc;
        }
        if (accept) {
            orc_ess q = {nd->level, nd->lo, nd->hi, {nd->R[0], nd->R[1], nd->R[2], nd->M}};
            out[cnt++] = q;
            continue;
        }
        for (int c = 7; c >= 0; --c)
            if (nd->child[c] != -1) { stack[sp] = nd->child[c]; slev[sp] = nd->level + 1; ++sp; }
    }
    qsort(out, (size_t)cnt, sizeof(orc_ess), cmp_ess);
    for (int64_t k = 0; k < cnt; ++k) {
        for (int a = 0; a < 4; ++a) rec[4 * k + a] = out[k].r[a];
        if (level) level[k] = out[k].level;
        if (lo) lo[k] = out[k].lo;
        if (hi) hi[k] = out[k].hi;
    }
    free(out);
    return cnt;
}

/* ---- direct summation of the acceleration (NEXT-4): g_i = -grad Phi_i of Eq. 2 written out ---------
 * g_i = -G sum_{j != i} m_j (r_i - r_j)/|r_i - r_j|^3, acc[3a..3a+2] for the a-th target (original
 * indices; targets == NULL: all n).  Sources in original order; zero-distance pairs skipped. */
int orc_direct_acc(const double *x, const double *y, const double *z, const double *m, int64_t n, double G,
                   const int64_t *targets, int64_t nt, double *acc)
{
    if (!x || !y || !z || !m || !acc || n <= 0) return -1;
    int64_t count = targets ? nt : n;
    for (int64_t a = 0; a < count; ++a) {
        int64_t i = targets ? targets[a] : a;
        if (i < 0 || i >= n) return -1;
        double sx = 0.0, sy = 0.0, sz = 0.0;
        for (int64_t j = 0; j < n; ++j) {
            if (j == i) continue;
            double dx = x[i] - x[j], dy = y[i] - y[j], dz = z[i] - z[j];
            double d2 = dx * dx + dy * dy + dz * dz;
            if (d2 == 0.0) continue;
            double w = m[j] / (d2 * sqrt(d2));
            sx -= w * dx; sy -= w * dy; sz -= w * dz;
        }
        acc[3 * a + 0] = G * sx; acc[3 * a + 1] = G * sy; acc[3 * a + 2] = G * sz;
    }
    return 0;
}

/* ==== periodic boundaries (Appendix A) =====================
 * "In case of periodic boundary conditions, a node's or data cell's contribution to the gravitational
 * potential of a data cell changes to phi = G M f_EF(r)" (Eq. A.1), f_EF the Ewald field:
 * Eq. A.2 splits 1/r = erf(alpha r)/r + erfc(alpha r)/r and Eq. A.3 sums a short-range part A_S over the
 * periodic images and a long-range part A_L obtained with the Poisson summation formula.  The paper prints
 * neither A_S nor A_L nor alpha; reading (P1), the standard Ewald sum of 1/r in a cubic box of
 * edge L with a neutralising uniform background, in box units u = r/L, a = alpha L:
 *   psi1(u) = sum_n erfc(a |u - n|)/|u - n|                               (A_S, images n in Z^3)
 *           + (1/pi) sum_{h != 0} exp(-pi^2 |h|^2 / a^2)/|h|^2 cos(2 pi h.u) (A_L, wave vectors h in Z^3)
 *           - pi / a^2                                                      (background: zero mean over the box)
 * f_EF(r) = psi1(r/L)/L, and a source of mass M at displacement r contributes -G M f_EF(r) to Phi (sign as in
 * reading R1).  Both index ranges are the cube |n_i|, |h_i| <= nser ("gpuEwaldSeriesN ... controls the range
 * of the indices i1, i2, i3").  psi1 does not depend on a once the sums have converged. */
double orc_ewald_psi(const double *u, double a, int nser)
{
    const double pi = 3.14159265358979323846;
    double s = 0.0;
    for (int i = -nser; i <= nser; ++i)
        for (int j = -nser; j <= nser; ++j)
            for (int k = -nser; k <= nser; ++k) {
                double dx = u[0] - i, dy = u[1] - j, dz = u[2] - k;
                double d = sqrt(dx * dx + dy * dy + dz * dz);
                s += erfc(a * d) / d;                                        /* A_S */
                int h2 = i * i + j * j + k * k;
                if (h2 > 0)                                                  /* A_L */
                    s += exp(-pi * pi * h2 / (a * a)) / (pi * h2) * cos(2.0 * pi * (i * u[0] + j * u[1] + k * u[2]));
            }
    return s - pi / (a * a);
}

/* The smooth part that is tabulated: corr1(u) = psi1(u) - 1/|u| for u inside the box, and its limit at
 * u = 0 (erfc(a d)/d - 1/d -> -2a/sqrt(pi)).  The singular 1/|u| is the isolated-boundary term the walk
 * evaluates directly; reading P2: the field array holds f_EF with that term taken out. */
double orc_ewald_corr(const double *u, double a, int nser)
{
    const double pi = 3.14159265358979323846;
    double d0 = sqrt(u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
    if (d0 > 0.0) return orc_ewald_psi(u, a, nser) - 1.0 / d0;
    double s = 0.0;
    for (int i = -nser; i <= nser; ++i)
        for (int j = -nser; j <= nser; ++j)
            for (int k = -nser; k <= nser; ++k) {
                int h2 = i * i + j * j + k * k;
                if (h2 == 0) continue;
                double d = sqrt((double)h2);
                s += erfc(a * d) / d + exp(-pi * pi * h2 / (a * a)) / (pi * h2);
            }
    return s - pi / (a * a) - 2.0 * a / sqrt(pi);
}

/* "The Ewald field is calculated once on startup and stored in a large array representing a hierarchy of
 * nested grids".  Reading P3: corr1 is even in every coordinate, so the array covers the
 * octant u_a >= 0; grid `lev` (0 .. nref-1, "gpuEwaldSeriesNref ... the number of nested grids") has N
 * points per axis ("gpuEwaldFieldNx/y/z"; one N here, the box is a cube) at u = i * h_lev,
 * h_lev = (1/2) / (N - 2) / 2^lev: grid 0 reaches ONE point past the face of the minimum-image cell
 * (u = 1/2 is its point N - 2; corr1 is smooth there but not mirror symmetric, because 1/|u| is not), so the
 * 3-point stencil of any |u_a| <= 1/2 lies inside it; every further grid refines the corner of the previous one
 * around u = 0 by a factor of two.  table[((lev * N + k) * N + j) * N + i] = corr1(i h, j h, k h). */
int orc_ewald_table(int N, int nref, double a, int nser, double *table)
{
    if (N < 4 || nref < 1 || !(a > 0.0) || nser < 1 || !table) return -1;
    for (int lev = 0; lev < nref; ++lev) {
        double h = 0.5 / (N - 2) / (double)(1 << lev);
        double *t = table + (size_t)lev * N * N * N;
        for (int k = 0; k < N; ++k)
            for (int j = 0; j <= k; ++j)
                for (int i = 0; i <= j; ++i) { /* corr1 is symmetric under permutations of the axes */
                    double u[3] = {i * h, j * h, k * h};
                    double v = orc_ewald_corr(u, a, nser);
                    int p[3] = {i, j, k};
                    static const int perm[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
                    for (int q = 0; q < 6; ++q)
                        t[((size_t)p[perm[q][2]] * N + p[perm[q][1]]) * N + p[perm[q][0]]] = v;
                }
    }
    return 0;
}

/* "... carried out during the respective tree walk using quadratic interpolation".
 * Reading P4 (the stencil is not given): on the finest grid that holds the point with its stencil, take the
 * NEAREST grid point i0 per axis and the quadratic through the 3 points per axis around it,
 *   corr(u) ~ C0 + sum_a Da d_a + 1/2 sum_a Daa d_a^2 + sum_{a<b} Dab d_a d_b,   d_a = |u_a|/h - i0_a in [-1/2, 1/2],
 *   Da = (C[+a] - C[-a])/2,  Daa = C[+a] - 2 C0 + C[-a],  Dab = (C[+a+b] - C[+a-b] - C[-a+b] + C[-a-b])/4.
 * Index -1 mirrors to +1 (corr1 is even); the nearest point never exceeds N - 2, so index N - 1 is the last one
 * read.  u must be a minimum-image displacement in box units, |u_a| <= 1/2. */
static double tab_at(const double *t, int N, int i, int j, int k)
{
    int v[3] = {i, j, k};
    for (int c = 0; c < 3; ++c)
        if (v[c] < 0) v[c] = -v[c];
    i = v[0]; j = v[1]; k = v[2];
    return t[((size_t)k * N + j) * N + i];
}

double orc_ewald_interp(const double *table, int N, int nref, const double *u)
{
    double ax = fabs(u[0]), ay = fabs(u[1]), az = fabs(u[2]);
    double mx = ax > ay ? (ax > az ? ax : az) : (ay > az ? ay : az);
    int lev = 0; /* finest grid whose interior (nearest point <= N - 2) holds the point: mx <= 1/2^(l+1) */
    for (int l = nref - 1; l > 0; --l) {
        double h = 0.5 / (N - 2) / (double)(1 << l);
        if (mx <= (N - 2) * h) { lev = l; break; }
    }
    double h = 0.5 / (N - 2) / (double)(1 << lev);
    const double *t = table + (size_t)lev * N * N * N;
    double p[3] = {ax / h, ay / h, az / h};
    int i0[3]; double d[3];
    for (int c = 0; c < 3; ++c) {
        i0[c] = (int)floor(p[c] + 0.5);
        if (i0[c] > N - 2) i0[c] = N - 2;
        d[c] = p[c] - i0[c];
    }
    int i = i0[0], j = i0[1], k = i0[2];
    double C0 = tab_at(t, N, i, j, k);
    double xp = tab_at(t, N, i + 1, j, k), xm = tab_at(t, N, i - 1, j, k);
    double yp = tab_at(t, N, i, j + 1, k), ym = tab_at(t, N, i, j - 1, k);
    double zp = tab_at(t, N, i, j, k + 1), zm = tab_at(t, N, i, j, k - 1);
    double Dx = 0.5 * (xp - xm), Dy = 0.5 * (yp - ym), Dz = 0.5 * (zp - zm);
    double Dxx = xp - 2.0 * C0 + xm, Dyy = yp - 2.0 * C0 + ym, Dzz = zp - 2.0 * C0 + zm;
    double Dxy = 0.25 * (tab_at(t, N, i + 1, j + 1, k) - tab_at(t, N, i + 1, j - 1, k) - tab_at(t, N, i - 1, j + 1, k) + tab_at(t, N, i - 1, j - 1, k));
    double Dxz = 0.25 * (tab_at(t, N, i + 1, j, k + 1) - tab_at(t, N, i + 1, j, k - 1) - tab_at(t, N, i - 1, j, k + 1) + tab_at(t, N, i - 1, j, k - 1));
    double Dyz = 0.25 * (tab_at(t, N, i, j + 1, k + 1) - tab_at(t, N, i, j + 1, k - 1) - tab_at(t, N, i, j - 1, k + 1) + tab_at(t, N, i, j - 1, k - 1));
    return C0 + Dx * d[0] + Dy * d[1] + Dz * d[2] + 0.5 * (Dxx * d[0] * d[0] + Dyy * d[1] * d[1] + Dzz * d[2] * d[2]) +
           Dxy * d[0] * d[1] + Dxz * d[0] * d[2] + Dyz * d[1] * d[2];
}

/* The group walk under periodic boundaries (W-rules unchanged except, reading P5):
 *  - every displacement is the MINIMUM IMAGE one, d_a -> d_a - L nearbyint(d_a / L), in the opening test
 *    (Eq. 3 / Eq. 4 with that distance) and in the sums;
 *  - an accepted node or a leaf cell contributes M (1/d + corr1(d_vec/L)/L) = M f_EF (Eq. A.1), corr1 taken
 *    from the table by quadratic interpolation;
 *  - the target's own cell, and a distinct cell at zero distance, contribute their images and background
 *    only: m corr1(0)/L (the 1/d term is dropped as in W-rule 3).
 * table: orc_ewald_table(N, nref, ...).  The cube of the tree is the periodic box. */
static double wrap_mi(double d, double L) { return d - L * nearbyint(d / L); }

int orc_potential_periodic(const orc_tree *t, double theta, double G, int mac, int group, const double *table,
                           int N, int nref, int64_t group_begin, int64_t group_end, double *phi_orig, int64_t *counts)
{
    if (!t || !phi_orig || !table || !(theta >= 0.0) || group < 1) return -1;
    int64_t n = t->n;
    double L = t->cube[3];
    int64_t ngroups = (n + group - 1) / group;
    if (group_end < 0 || group_end > ngroups) group_end = ngroups;
    if (group_begin < 0) group_begin = 0;
    int64_t stack[8 * (ORC_MAXLEVEL + 2)];
    double *acc = (double *)malloc(sizeof(double) * (size_t)group);
    if (!acc) return -2;
    const double zero[3] = {0.0, 0.0, 0.0};
    double c0 = orc_ewald_interp(table, N, nref, zero) / L;
    for (int64_t g = group_begin; g < group_end; ++g) {
        int64_t t0 = g * group, t1 = t0 + group;
        if (t1 > n) t1 = n;
        int nt = (int)(t1 - t0);
        for (int a = 0; a < nt; ++a) acc[a] = 0.0;
        int64_t n_acc = 0, n_leaf = 0, n_open = 0;
        int sp = 0;
        if (n >= 2) stack[sp++] = 0;
        else acc[0] = t->m[0] * c0; /* a lone cell still feels its own images */
        while (sp > 0) {
            int64_t e = stack[--sp];
            const orc_node *nd = e >= 0 ? &t->node[e] : NULL;
            if (e <= -2 || nd->level == ORC_MAXLEVEL) { /* leaf cell, or every cell of a bucket */
                int64_t j0 = e <= -2 ? -(e + 2) : nd->lo, j1 = e <= -2 ? j0 + 1 : nd->hi;
                for (int64_t j = j0; j < j1; ++j) {
                    for (int a = 0; a < nt; ++a) {
                        int64_t s = t0 + a;
                        double r[3] = {wrap_mi(t->x[s] - t->x[j], L), wrap_mi(t->y[s] - t->y[j], L), wrap_mi(t->z[s] - t->z[j], L)};
                        double d2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
                        if (s == j || d2 == 0.0) { acc[a] += t->m[j] * c0; continue; }
                        double u[3] = {r[0] / L, r[1] / L, r[2] / L};
                        acc[a] += t->m[j] * (1.0 / sqrt(d2) + orc_ewald_interp(table, N, nref, u) / L);
                    }
                    ++n_leaf;
                }
                continue;
            }
            int accept = theta > 0.0;
            if (accept) {
                double rc = nd->size / theta;
                if (mac == ORC_MAC_BARNES94) rc += nd->delta;
                for (int a = 0; a < nt && accept; ++a) {
                    int64_t s = t0 + a;
                    double dx = wrap_mi(t->x[s] - nd->R[0], L), dy = wrap_mi(t->y[s] - nd->R[1], L), dz = wrap_mi(t->z[s] - nd->R[2], L);
                    if (!(dx * dx + dy * dy + dz * dz > rc * rc)) accept = 0;
                }
            }
            if (accept) {
                for (int a = 0; a < nt; ++a) {
                    int64_t s = t0 + a;
                    double r[3] = {wrap_mi(t->x[s] - nd->R[0], L), wrap_mi(t->y[s] - nd->R[1], L), wrap_mi(t->z[s] - nd->R[2], L)};
                    double u[3] = {r[0] / L, r[1] / L, r[2] / L};
                    acc[a] += nd->M * (1.0 / sqrt(r[0] * r[0] + r[1] * r[1] + r[2] * r[2]) + orc_ewald_interp(table, N, nref, u) / L);
                }
                ++n_acc;
                continue;
            }
            ++n_open;
            for (int c = 7; c >= 0; --c)
                if (nd->child[c] != -1) stack[sp++] = nd->child[c];
        }
        for (int a = 0; a < nt; ++a) phi_orig[t->perm[t0 + a]] = -G * acc[a];
        if (counts) {
            int64_t *c = counts + 3 * (g - group_begin);
            c[0] = n_acc; c[1] = n_leaf; c[2] = n_open;
        }
    }
    free(acc);
    return 0;
}
