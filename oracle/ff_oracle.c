/*
 * ff_oracle.c -- the ORACLE: a plain, slow, fp64 CPU statement of what the hot
 * path of arxiv 1212.2934 computes (dipole field + dipole force on N magnetic
 * particles, all-pairs and Barnes-Hut).
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no
 * code with paper_1212_2934_b200/csrc (the CUDA path) and is never a fallback.
 *
 * All citations are lines of /root/reference/PAPER.md ("PAPER.md:n").
 * Readings of passages where the paper is silent are the O3-O5 / Q1-Q8
 * readings of SURVEY.md 8(c), restated in DESIGN.md.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"):
 *   ffo_pair ............ closed forms of one/two dipoles, finite-difference
 *                         gradient tying Eq. 12 to Eq. 11, antisymmetry
 *   ffo_allpairs ........ independent numpy einsum, sum f = 0, torque balance,
 *                         rotation/translation covariance, straight-chain sums
 *   ffo_tree_build ...... independent brute-force prefix grouping, hand-made
 *                         inputs, partition invariants
 *   ffo_tree_moments .... math.fsum root sums, single-particle nodes, Eq. 14
 *   ffo_bh_eval ......... theta = 0 == all-pairs, N <= N_leaf == all-pairs,
 *                         independently written recursive list builder on
 *                         N <= 64, far-cluster limit, (28 pi/3) theta^-3 count
 *   member_accepts ...... the opening test ON its threshold (tests/test_oracle_walk.py): exact equality
 *                         s^2 == theta^2 d2 opens, one fp32 step beyond accepts, one short opens, and two
 *                         targets found by a seeded search on which the fused order of O5 and three rounded
 *                         squares added left to right decide differently (decisions taken from exact-rational
 *                         fma in tests/helpers.py)
 *   Q output (scale) .... independent numpy sum of squared terms (all-pairs and the list builder's lists),
 *                         exact-rational closed form on the straight chain (tests/test_oracle_scale.py)
 *   first-order cell term (O1b, not in the paper): central differences of Eq. 11-12 in the source
 *                         position, error order (s/d)^2 on the far cluster and on a two-particle cell, theta = 0
 *                         unchanged, D against numpy (tests/test_oracle_first_order.py)
 *   BH-vs-all-pairs error SIZE: parity unpinned by the paper (PAPER.md:233,
 *                         239 only say "almost identical"); reported, not gated.
 *
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fopenmp -shared -fPIC (see
 * oracle/__init__.py).  -ffp-contract=off and no -ffast-math are REQUIRED: the
 * fp32 key quantisation (O3) and the fp32 opening test (O5) are defined by
 * their exact IEEE operation order.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define FFO_MAX_LEVEL 10          /* 30-bit key = 10 octant digits (O3) */

/* ------------------------------------------------------------------ O1 --
 * Pair terms, reduced units.  With rho = rho_k - rho_j:
 *   Eq. 11:  h_kj = [3 rho (u_j.rho) - u_j rho^2] / rho^5
 *   Eq. 12:  f_kj = 3 [rho (u_j.u_k) + u_k (u_j.rho) + u_j (u_k.rho)] / rho^5
 *                                 - 15 rho (u_k.rho)(u_j.rho) / rho^7
 * h and f are ADDED to (accumulated into) the output arguments.
 */
static void pair_accumulate(const double rk[3], const double uk[3],
                            const double rj[3], const double uj[3],
                            double h[3], double f[3], double* q /* NULL or [2] */)
{
    double rho[3] = { rk[0] - rj[0], rk[1] - rj[1], rk[2] - rj[2] };
    double r2 = rho[0] * rho[0] + rho[1] * rho[1] + rho[2] * rho[2];
    double r = sqrt(r2);
    double r5 = r2 * r2 * r;
    double r7 = r5 * r2;
    double uj_rho = uj[0] * rho[0] + uj[1] * rho[1] + uj[2] * rho[2];
    double uk_rho = uk[0] * rho[0] + uk[1] * rho[1] + uk[2] * rho[2];
    double uj_uk = uj[0] * uk[0] + uj[1] * uk[1] + uj[2] * uk[2];
    double th2 = 0.0, tf2 = 0.0;
    for (int a = 0; a < 3; ++a) {
        double th = (3.0 * rho[a] * uj_rho - uj[a] * r2) / r5;
        double tf = 3.0 * (rho[a] * uj_uk + uk[a] * uj_rho + uj[a] * uk_rho) / r5
                    - 15.0 * rho[a] * uk_rho * uj_rho / r7;
        h[a] += th;
        f[a] += tf;
        th2 += th * th; tf2 += tf * tf;
    }
    /* not part of the method: the squared magnitudes of the terms, summed per target, give the
     * scale Q_k = sqrt(sum_j |t_kj|^2) against which the tests measure rounding error when the
     * terms of a sum cancel (error metric) */
    if (q) { q[0] += th2; q[1] += tf2; }
}

/* public single-pair entry: h, f are OVERWRITTEN with the pair terms */
void ffo_pair(const double rk[3], const double uk[3], const double rj[3], const double uj[3],
              double h[3], double f[3])
{
    h[0] = h[1] = h[2] = 0.0;
    f[0] = f[1] = f[2] = 0.0;
    pair_accumulate(rk, uk, rj, uj, h, f, NULL);
}

/* ----------------------------------------------------------------- O1b --
 * First-order correction of a cell's pseudo-particle (NOT in the paper, whose cell is the
 * lowest-order term only).  A cell's exact field at a target is sum_i T(rho_k - rho_i) u_i with
 * the dipole tensor of Eq. 11, T_ab(r) = (3 r_a r_b - delta_ab r^2) / r^5.  Expanding each rho_i = rho' + d_i about
 * the cell centre rho' of Eq. 14, with R = rho_k - rho':
 *     h_a = T_ab(R) u'_b  -  S_abc(R) D_cb  +  O(d^2),        D_cb = sum_i d_ic u_ib,
 *     S_abc = dT_ab/dr_c = 3 (delta_ab r_c + delta_ac r_b + delta_bc r_a) / r^5 - 15 r_a r_b r_c / r^7
 * (the same S that gives Eq. 12: f_a = S_abc u_kb u_jc).  The force on the target dipole is f_a = u_kb d(h_b)/dr_a:
 *     f_a = S_abc u_kb u'_c  -  U_abcd u_kb D_cd,
 *     U_abcd = dS_bcd/dr_a = 3 (d_ab d_cd + d_ac d_bd + d_ad d_bc) / r^5
 *              - 15 (d_ab r_c r_d + d_ac r_b r_d + d_ad r_b r_c + d_bc r_a r_d + d_bd r_a r_c + d_cd r_a r_b) / r^7
 *              + 105 r_a r_b r_c r_d / r^9                                         (d_xy = Kronecker delta).
 * Written out as plain loops over the tensor components.  D is the full 3x3 tensor here; the tree stores its
 * symmetric part only (S and U are symmetric in the contracted index pairs, so the antisymmetric part drops out).
 * The correction terms are ADDED to h, f.
 */
static double kd(int a, int b) { return a == b ? 1.0 : 0.0; }

static void first_order_accumulate(const double rk[3], const double uk[3], const double rc[3], const double D[3][3],
                                   double h[3], double f[3], double* q /* NULL or [2] */)
{
    double r[3] = { rk[0] - rc[0], rk[1] - rc[1], rk[2] - rc[2] };
    double r2 = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
    double rr = sqrt(r2), r5 = r2 * r2 * rr, r7 = r5 * r2, r9 = r7 * r2;
    double th2 = 0.0, tf2 = 0.0;
    for (int a = 0; a < 3; ++a) {
        double dh = 0.0, df = 0.0;
        for (int b = 0; b < 3; ++b)
            for (int c = 0; c < 3; ++c) {
                double S = 3.0 * (kd(a, b) * r[c] + kd(a, c) * r[b] + kd(b, c) * r[a]) / r5 - 15.0 * r[a] * r[b] * r[c] / r7;
                dh -= S * D[c][b];
                for (int d = 0; d < 3; ++d) {
                    double U = 3.0 * (kd(a, b) * kd(c, d) + kd(a, c) * kd(b, d) + kd(a, d) * kd(b, c)) / r5
                               - 15.0 * (kd(a, b) * r[c] * r[d] + kd(a, c) * r[b] * r[d] + kd(a, d) * r[b] * r[c]
                                         + kd(b, c) * r[a] * r[d] + kd(b, d) * r[a] * r[c] + kd(c, d) * r[a] * r[b]) / r7
                               + 105.0 * r[a] * r[b] * r[c] * r[d] / r9;
                    df -= U * uk[b] * D[c][d];
                }
            }
        h[a] += dh; f[a] += df;
        th2 += dh * dh; tf2 += df * df;
    }
    if (q) { q[0] += th2; q[1] += tf2; }
}

/* public entry for the pins: h, f are OVERWRITTEN with the first-order terms of a cell at rc with tensor D (row major) */
void ffo_first_order(const double rk[3], const double uk[3], const double rc[3], const double D9[9], double h[3], double f[3])
{
    double D[3][3];
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) D[a][b] = D9[3 * a + b];
    h[0] = h[1] = h[2] = 0.0;
    f[0] = f[1] = f[2] = 0.0;
    first_order_accumulate(rk, uk, rc, D, h, f, NULL);
}

static void widen3(const float* src, int64_t i, double out[3])
{
    out[0] = (double)src[3 * i]; out[1] = (double)src[3 * i + 1]; out[2] = (double)src[3 * i + 2];
}

static int pick_threads(int nthreads)
{
#ifdef _OPENMP
    return nthreads > 0 ? nthreads : omp_get_max_threads();
#else
    (void)nthreads;
    return 1;
#endif
}

int ffo_max_threads(void) { return pick_threads(0); }

/* ------------------------------------------------------------------ O2 --
 * All-pairs: h_k = sum_{j != k} h_kj (Eq. 10 without h_ext) and
 * f_k = sum_{j != k} f_kj (Eq. 12), j in index order, self excluded BY INDEX
 * as in Algorithm 1 line 5.  `targets` (nt entries, NULL = all
 * N) selects which k are evaluated; row t of H/F belongs to targets[t].
 */
int ffo_allpairs(int64_t N, const float* pos, const float* mom,
                 int64_t nt, const int64_t* targets, double* H, double* F, double* Q /* NULL or [nt][2] */,
                 int nthreads)
{
    if (N <= 0 || !pos || !mom || !H || !F) return -1;
    if (!targets) nt = N;
    int nth = pick_threads(nthreads);
    (void)nth;
#pragma omp parallel for schedule(dynamic, 16) num_threads(nth)
    for (int64_t t = 0; t < nt; ++t) {
        int64_t k = targets ? targets[t] : t;
        double rk[3], uk[3], h[3] = { 0, 0, 0 }, f[3] = { 0, 0, 0 }, q[2] = { 0, 0 };
        widen3(pos, k, rk); widen3(mom, k, uk);
        for (int64_t j = 0; j < N; ++j) {
            if (j == k) continue;
            double rj[3], uj[3];
            widen3(pos, j, rj); widen3(mom, j, uj);
            pair_accumulate(rk, uk, rj, uj, h, f, q);
        }
        for (int a = 0; a < 3; ++a) { H[3 * t + a] = h[a]; F[3 * t + a] = f[a]; }
        if (Q) { Q[2 * t] = sqrt(q[0]); Q[2 * t + 1] = sqrt(q[1]); }
    }
    return 0;
}

/* ------------------------------------------------------------------ O3 --
 * Tree (a cubic "main cell" divided into eight sub-cells,
 * re-divided while a sub-cell holds more than one particle).
 */
typedef struct {
    int64_t first, count;     /* sorted-slot range [first, first+count) */
    int32_t level;            /* 0 = root */
    uint32_t prefix;          /* top 3*level key bits */
    int32_t is_leaf;
    int64_t child[8];         /* node index per octant, -1 = empty sub-cell */
    double sum_u[3], sum_p[3];/* O4: fp64 sums in the fixed recursion order */
    float cen[3], mu[3];      /* O4: rho' and u' rounded once to fp32 */
    double sum_pu[6];         /* O4b: fp64 sums of the symmetrised products rho_i (x) u_i, order xx yy zz xy xz yz */
    float dsym[6];            /* O4b: first-order cell tensor D (symmetric part), rounded once to fp32 */
} ffo_node;

typedef struct ffo_tree {
    int64_t N;
    int nleaf;
    float lo[3], S;           /* root cube: origin = min corner, side S */
    uint32_t* key;            /* sorted keys */
    int64_t* perm;            /* perm[s] = caller index of sorted slot s */
    float* spos;              /* sorted positions [N][3] (fp32, as given) */
    float* smom;              /* sorted moments (set by ffo_tree_moments) */
    ffo_node* node; int64_t n_nodes, cap_nodes;
    int has_moments;
} ffo_tree;

typedef struct { uint32_t key; int64_t idx; } key_idx;

static int cmp_key_idx(const void* a, const void* b)
{
    const key_idx* x = (const key_idx*)a; const key_idx* y = (const key_idx*)b;
    if (x->key != y->key) return x->key < y->key ? -1 : 1;
    return x->idx < y->idx ? -1 : (x->idx > y->idx);   /* ties keep caller order: stable */
}

/* spread the low 10 bits of v so that bit b lands on bit 3b */
static uint32_t spread10(uint32_t v)
{
    uint32_t r = 0;
    for (int b = 0; b < 10; ++b) r |= ((v >> b) & 1u) << (3 * b);
    return r;
}

static int64_t new_node(ffo_tree* t)
{
    if (t->n_nodes == t->cap_nodes) {
        int64_t cap = t->cap_nodes ? 2 * t->cap_nodes : 1024;
        ffo_node* p = (ffo_node*)realloc(t->node, (size_t)cap * sizeof(ffo_node));
        if (!p) return -1;
        t->node = p; t->cap_nodes = cap;
    }
    return t->n_nodes++;
}

/* octant digit of a key at level l (1..10): bits [3(10-l), 3(10-l)+2] = 4x+2y+z */
static int digit_at(uint32_t key, int level) { return (int)((key >> (3 * (FFO_MAX_LEVEL - level))) & 7u); }

/* Subdivide the cell (level, prefix) holding sorted slots [first, first+count). */
static int64_t build_cell(ffo_tree* t, int level, uint32_t prefix, int64_t first, int64_t count)
{
    int64_t id = new_node(t);
    if (id < 0) return -1;
    {
        ffo_node* n = &t->node[id];
        memset(n, 0, sizeof(*n));
        n->first = first; n->count = count; n->level = level; n->prefix = prefix;
        for (int o = 0; o < 8; ++o) n->child[o] = -1;
        n->is_leaf = !(count > t->nleaf && level < FFO_MAX_LEVEL);
        if (n->is_leaf) return id;
    }
    int64_t s = first, end = first + count;
    for (int o = 0; o < 8; ++o) {
        int64_t b = s;
        while (s < end && digit_at(t->key[s], level + 1) == o) ++s;
        if (s > b) {
            int64_t c = build_cell(t, level + 1, (prefix << 3) | (uint32_t)o, b, s - b);
            if (c < 0) return -1;
            t->node[id].child[o] = c;     /* re-index: realloc may have moved the pool */
        }
    }
    return id;
}

void ffo_tree_free(ffo_tree* t)
{
    if (!t) return;
    free(t->key); free(t->perm); free(t->spos); free(t->smom); free(t->node); free(t);
}

/*
 * Bounding box (kernel 1) -> root cube -> 30-bit keys -> stable
 * order -> recursive subdivision.  The quantisation is fp32 with this exact
 * operation order (no contraction):
 *    inv = fl(1024 / S);  q_a = min(1023, (int)floor(fl(fl(pos_a - lo_a) * inv)))
 * key bit 3b+2 = bit b of q_x, 3b+1 of q_y, 3b of q_z.
 */
ffo_tree* ffo_tree_build(int64_t N, const float* pos, int nleaf)
{
    if (N <= 0 || !pos || nleaf < 1) return NULL;
    ffo_tree* t = (ffo_tree*)calloc(1, sizeof(ffo_tree));
    if (!t) return NULL;
    t->N = N; t->nleaf = nleaf;
    float lo[3], hi[3];
    for (int a = 0; a < 3; ++a) lo[a] = hi[a] = pos[a];
    for (int64_t i = 1; i < N; ++i)
        for (int a = 0; a < 3; ++a) {
            float v = pos[3 * i + a];
            if (v < lo[a]) lo[a] = v;
            if (v > hi[a]) hi[a] = v;
        }
    float S = 0.0f;
    for (int a = 0; a < 3; ++a) { float e = hi[a] - lo[a]; if (e > S) S = e; }
    if (!(S > 0.0f)) S = 1.0f;
    t->S = S;
    for (int a = 0; a < 3; ++a) t->lo[a] = lo[a];

    key_idx* ki = (key_idx*)malloc((size_t)N * sizeof(key_idx));
    t->key = (uint32_t*)malloc((size_t)N * sizeof(uint32_t));
    t->perm = (int64_t*)malloc((size_t)N * sizeof(int64_t));
    t->spos = (float*)malloc((size_t)N * 3 * sizeof(float));
    if (!ki || !t->key || !t->perm || !t->spos) { free(ki); ffo_tree_free(t); return NULL; }
    float inv = 1024.0f / S;
    for (int64_t i = 0; i < N; ++i) {
        uint32_t q[3];
        for (int a = 0; a < 3; ++a) {
            float d = pos[3 * i + a] - lo[a];
            float g = d * inv;
            int v = (int)floorf(g);
            if (v > 1023) v = 1023;
            if (v < 0) v = 0;
            q[a] = (uint32_t)v;
        }
        ki[i].key = (spread10(q[0]) << 2) | (spread10(q[1]) << 1) | spread10(q[2]);
        ki[i].idx = i;
    }
    qsort(ki, (size_t)N, sizeof(key_idx), cmp_key_idx);
    for (int64_t s = 0; s < N; ++s) {
        t->key[s] = ki[s].key; t->perm[s] = ki[s].idx;
        for (int a = 0; a < 3; ++a) t->spos[3 * s + a] = pos[3 * ki[s].idx + a];
    }
    free(ki);
    if (build_cell(t, 0, 0u, 0, N) != 0) { ffo_tree_free(t); return NULL; }
    return t;
}

int64_t ffo_tree_num_nodes(const ffo_tree* t) { return t->n_nodes; }
int64_t ffo_tree_num_particles(const ffo_tree* t) { return t->N; }

void ffo_tree_bbox(const ffo_tree* t, float lo[3], float* S)
{
    for (int a = 0; a < 3; ++a) lo[a] = t->lo[a];
    *S = t->S;
}

void ffo_tree_keys(const ffo_tree* t, uint32_t* key, int64_t* perm)
{
    if (key) memcpy(key, t->key, (size_t)t->N * sizeof(uint32_t));
    if (perm) memcpy(perm, t->perm, (size_t)t->N * sizeof(int64_t));
}

/* Node list in creation order = pre-order = sorted by (first, level): the canonical topology. */
void ffo_tree_nodes(const ffo_tree* t, int64_t* first, int64_t* count, int32_t* level,
                    uint32_t* prefix, int32_t* is_leaf, int64_t* child /* [n][8] */)
{
    for (int64_t i = 0; i < t->n_nodes; ++i) {
        const ffo_node* n = &t->node[i];
        if (first) first[i] = n->first;
        if (count) count[i] = n->count;
        if (level) level[i] = n->level;
        if (prefix) prefix[i] = n->prefix;
        if (is_leaf) is_leaf[i] = n->is_leaf;
        if (child) for (int o = 0; o < 8; ++o) child[8 * i + o] = n->child[o];
    }
}

/* ------------------------------------------------------------------ O4 --
 * Pseudo-particle of every cell: u' = sum of the moments
 * of the cell's particles, rho' = (sum rho_i) / N' (Eq. 14, unweighted).
 * fp64 sums in a FIXED order -- leaf: particles left to right in sorted order;
 * internal: children in octant order 0..7, ((c0 + c1) + c2) + ... -- then one
 * fp64 divide and ONE rounding to fp32.  The fp32 values are the node data.
 */
/* symmetrised products of one particle, order xx yy zz xy xz yz: rho_a u_a and (rho_a u_b + rho_b u_a) / 2.
 * Products of two fp32 values are exact in fp64; the sum of two of them is rounded once; the halving is exact. */
static void sym_products(const float* p, const float* u, double out[6])
{
    double px = p[0], py = p[1], pz = p[2], ux = u[0], uy = u[1], uz = u[2];
    out[0] = px * ux; out[1] = py * uy; out[2] = pz * uz;
    out[3] = (px * uy + py * ux) * 0.5;
    out[4] = (px * uz + pz * ux) * 0.5;
    out[5] = (py * uz + pz * uy) * 0.5;
}

static void moments_cell(ffo_tree* t, int64_t id)
{
    ffo_node* n = &t->node[id];
    double su[3], sp[3], spu[6];
    if (n->is_leaf) {
        for (int a = 0; a < 3; ++a) {
            su[a] = (double)t->smom[3 * n->first + a];
            sp[a] = (double)t->spos[3 * n->first + a];
        }
        sym_products(t->spos + 3 * n->first, t->smom + 3 * n->first, spu);
        for (int64_t s = n->first + 1; s < n->first + n->count; ++s) {
            double pu[6];
            sym_products(t->spos + 3 * s, t->smom + 3 * s, pu);
            for (int a = 0; a < 3; ++a) {
                su[a] += (double)t->smom[3 * s + a];
                sp[a] += (double)t->spos[3 * s + a];
            }
            for (int a = 0; a < 6; ++a) spu[a] += pu[a];
        }
    } else {
        int started = 0;
        for (int o = 0; o < 8; ++o) {
            int64_t c = n->child[o];
            if (c < 0) continue;
            moments_cell(t, c);
            n = &t->node[id];
            const ffo_node* cn = &t->node[c];
            for (int a = 0; a < 3; ++a) {
                if (!started) { su[a] = cn->sum_u[a]; sp[a] = cn->sum_p[a]; }
                else { su[a] += cn->sum_u[a]; sp[a] += cn->sum_p[a]; }
            }
            for (int a = 0; a < 6; ++a) {
                if (!started) spu[a] = cn->sum_pu[a];
                else spu[a] += cn->sum_pu[a];
            }
            started = 1;
        }
    }
    double cen[3];
    for (int a = 0; a < 3; ++a) {
        n->sum_u[a] = su[a]; n->sum_p[a] = sp[a];
        n->mu[a] = (float)su[a];
        cen[a] = sp[a] / (double)n->count;
        n->cen[a] = (float)cen[a];
    }
    /* O4b: D = sum_i (rho_i - rho') (x) u_i, symmetric part = sum of the symmetrised products minus the symmetrised
     * rho' (x) u' (fp64 rho' before its rounding, fp64 u'), each operation rounded once in fp64, the result once to fp32 */
    static const int ia[6] = { 0, 1, 2, 0, 0, 1 }, ib[6] = { 0, 1, 2, 1, 2, 2 };
    for (int c = 0; c < 6; ++c) {
        n->sum_pu[c] = spu[c];
        double cu = c < 3 ? cen[ia[c]] * su[ib[c]] : (cen[ia[c]] * su[ib[c]] + cen[ib[c]] * su[ia[c]]) * 0.5;
        n->dsym[c] = (float)(spu[c] - cu);
    }
}

int ffo_tree_moments(ffo_tree* t, const float* mom)
{
    if (!t || !mom) return -1;
    if (!t->smom) t->smom = (float*)malloc((size_t)t->N * 3 * sizeof(float));
    if (!t->smom) return -1;
    for (int64_t s = 0; s < t->N; ++s)
        for (int a = 0; a < 3; ++a) t->smom[3 * s + a] = mom[3 * t->perm[s] + a];
    moments_cell(t, 0);
    t->has_moments = 1;
    return 0;
}

/* O4b node data: dsym [n][6] fp32 in the order xx yy zz xy xz yz */
void ffo_tree_node_dsym(const ffo_tree* t, float* dsym)
{
    for (int64_t i = 0; i < t->n_nodes; ++i)
        for (int c = 0; c < 6; ++c) dsym[6 * i + c] = t->node[i].dsym[c];
}

void ffo_tree_node_moments(const ffo_tree* t, double* sum_u, double* sum_p, float* mu, float* cen)
{
    for (int64_t i = 0; i < t->n_nodes; ++i) {
        const ffo_node* n = &t->node[i];
        for (int a = 0; a < 3; ++a) {
            if (sum_u) sum_u[3 * i + a] = n->sum_u[a];
            if (sum_p) sum_p[3 * i + a] = n->sum_p[a];
            if (mu) mu[3 * i + a] = n->mu[a];
            if (cen) cen[3 * i + a] = n->cen[a];
        }
    }
}

/* ------------------------------------------------------------------ O5 --
 * Traversal: from the root, use the pseudo-particle when the
 * particle is "far enough", otherwise check the sub-cells; a single-particle
 * leaf is used directly.  The paper gives no criterion (reading Q1): cell
 * side s over distance d to the pseudo-particle, accept iff s/d < theta.
 * Targets are handled in groups of W consecutive sorted slots (reading Q2;
 * W = 1 is the literal per-particle walk).  Per group and node:
 *   leaf ........ its particles are summed directly (O1), j = k skipped by index
 *   internal .... OPEN if its slot range contains a member of the group (Q3),
 *                 else ACCEPT for the whole group iff EVERY member accepts,
 *                 else OPEN.
 * A member at fp32 position p accepts the node with fp32 centre c iff, in
 * fp32 with exactly this operation order,
 *     dx = fl(px - cx), dy, dz likewise;  d2 = fma(dz, dz, fma(dy, dy, fl(dx*dx)));
 *     fl(s_l * s_l) < fl(fl(theta * theta) * d2)          (strict; equality opens)
 * with s_l = S * 2^-l (exact).  An accepted node contributes one O1 term per
 * member with (u_j, rho_j) := (u', rho') (the fp32 node data widened to fp64).
 */
typedef struct {
    const ffo_tree* t;
    float th2;
    int order;                /* 0 = the paper's cell (Eq. 14); 1 = plus the first-order term O1b */
    int64_t g0, g1;           /* group = sorted slots [g0, g1) */
    double* h; double* f;     /* [g1-g0][3] accumulators (NULL when only listing) */
    double* q;                /* [g1-g0][2] squared term magnitudes (error-metric scale) */
    uint64_t n_cell, n_part, n_mac;
    /* optional interaction lists (for tests) */
    int64_t* cells; int64_t n_cells_out, cap_cells;
    int64_t* parts; int64_t n_parts_out, cap_parts;
} walk_ctx;

static int member_accepts(const float* p, const float* c, float s2, float th2)
{
    float dx = p[0] - c[0];
    float dy = p[1] - c[1];
    float dz = p[2] - c[2];
    float xx = dx * dx;
    float d2 = fmaf(dz, dz, fmaf(dy, dy, xx));
    float rhs = th2 * d2;
    return s2 < rhs;
}

static void visit(walk_ctx* w, int64_t id)
{
    const ffo_tree* t = w->t;
    const ffo_node* n = &t->node[id];
    if (n->is_leaf) {
        for (int64_t j = n->first; j < n->first + n->count; ++j) {
            if (w->parts && w->n_parts_out < w->cap_parts) w->parts[w->n_parts_out] = j;
            if (w->parts) w->n_parts_out++;
            if (!w->h) continue;
            double rj[3], uj[3];
            widen3(t->spos, j, rj); widen3(t->smom, j, uj);
            for (int64_t k = w->g0; k < w->g1; ++k) {
                if (j == k) continue;                      /* Alg. 1 line 5 */
                double rk[3], uk[3];
                widen3(t->spos, k, rk); widen3(t->smom, k, uk);
                pair_accumulate(rk, uk, rj, uj, w->h + 3 * (k - w->g0), w->f + 3 * (k - w->g0), w->q + 2 * (k - w->g0));
                w->n_part++;
            }
        }
        return;
    }
    int open = (n->first < w->g1) && (n->first + n->count > w->g0);   /* holds a member: Q3 */
    if (!open) {
        float s = ldexpf(t->S, -n->level);
        float s2 = s * s;
        int all = 1;
        for (int64_t k = w->g0; k < w->g1; ++k)
            if (!member_accepts(t->spos + 3 * k, n->cen, s2, w->th2)) { all = 0; break; }
        w->n_mac++;
        if (all) {
            if (w->cells && w->n_cells_out < w->cap_cells) w->cells[w->n_cells_out] = id;
            if (w->cells) w->n_cells_out++;
            if (w->h) {
                double rj[3] = { n->cen[0], n->cen[1], n->cen[2] };
                double uj[3] = { n->mu[0], n->mu[1], n->mu[2] };
                for (int64_t k = w->g0; k < w->g1; ++k) {
                    double rk[3], uk[3];
                    widen3(t->spos, k, rk); widen3(t->smom, k, uk);
                    if (!w->order) {
                        pair_accumulate(rk, uk, rj, uj, w->h + 3 * (k - w->g0), w->f + 3 * (k - w->g0), w->q + 2 * (k - w->g0));
                    } else {
                        /* the cell's term = pseudo-particle + first-order correction; its magnitude enters q as ONE term */
                        double th[3] = { 0, 0, 0 }, tf[3] = { 0, 0, 0 };
                        double D[3][3] = { { n->dsym[0], n->dsym[3], n->dsym[4] },
                                           { n->dsym[3], n->dsym[1], n->dsym[5] },
                                           { n->dsym[4], n->dsym[5], n->dsym[2] } };
                        pair_accumulate(rk, uk, rj, uj, th, tf, NULL);
                        first_order_accumulate(rk, uk, rj, D, th, tf, NULL);
                        double* hh = w->h + 3 * (k - w->g0); double* ff = w->f + 3 * (k - w->g0); double* qq = w->q + 2 * (k - w->g0);
                        for (int a = 0; a < 3; ++a) {
                            hh[a] += th[a]; ff[a] += tf[a];
                            qq[0] += th[a] * th[a]; qq[1] += tf[a] * tf[a];
                        }
                    }
                }
                w->n_cell += (uint64_t)(w->g1 - w->g0);
            }
            return;
        }
    }
    for (int o = 0; o < 8; ++o)
        if (n->child[o] >= 0) visit(w, n->child[o]);
}

/*
 * Barnes-Hut field + force.  groups (ng entries, NULL = every group) selects
 * which groups of W sorted slots are evaluated.  H, F: [N][3] fp64 in CALLER
 * order (O6); rows of targets outside the selected groups are left untouched.
 * counters[0] = accepted cell terms summed over targets, [1] = direct
 * particle terms summed over targets (self excluded), [2] = opening tests
 * (group, internal node not holding a member) evaluated.
 */
int ffo_bh_eval_order(const ffo_tree* t, float theta, int W, int order, int64_t ng, const int64_t* groups,
                      double* H, double* F, double* Q /* NULL or [N][2], caller order */, uint64_t counters[3], int nthreads)
{
    if (!t || !t->has_moments || W < 1 || !(theta >= 0.0f) || !H || !F || order < 0 || order > 1) return -1;
    int64_t n_groups = (t->N + W - 1) / W;
    if (!groups) ng = n_groups;
    float th2 = theta * theta;
    uint64_t c0 = 0, c1 = 0, c2 = 0;
    int nth = pick_threads(nthreads);
    (void)nth;
#pragma omp parallel for schedule(dynamic, 4) reduction(+ : c0, c1, c2) num_threads(nth)
    for (int64_t gi = 0; gi < ng; ++gi) {
        int64_t g = groups ? groups[gi] : gi;
        if (g < 0 || g >= n_groups) continue;
        walk_ctx w;
        memset(&w, 0, sizeof(w));
        w.t = t; w.th2 = th2; w.order = order;
        w.g0 = g * W; w.g1 = w.g0 + W < t->N ? w.g0 + W : t->N;
        int64_t m = w.g1 - w.g0;
        double* acc = (double*)calloc((size_t)m * 8, sizeof(double));
        w.h = acc; w.f = acc + 3 * m; w.q = acc + 6 * m;
        visit(&w, 0);
        for (int64_t k = w.g0; k < w.g1; ++k) {
            for (int a = 0; a < 3; ++a) {
                H[3 * t->perm[k] + a] = w.h[3 * (k - w.g0) + a];
                F[3 * t->perm[k] + a] = w.f[3 * (k - w.g0) + a];
            }
            if (Q) {
                Q[2 * t->perm[k]] = sqrt(w.q[2 * (k - w.g0)]);
                Q[2 * t->perm[k] + 1] = sqrt(w.q[2 * (k - w.g0) + 1]);
            }
        }
        free(acc);
        c0 += w.n_cell; c1 += w.n_part; c2 += w.n_mac;
    }
    if (counters) { counters[0] = c0; counters[1] = c1; counters[2] = c2; }
    return 0;
}

/* the paper's cell (order 0) */
int ffo_bh_eval(const ffo_tree* t, float theta, int W, int64_t ng, const int64_t* groups,
                double* H, double* F, double* Q, uint64_t counters[3], int nthreads)
{
    return ffo_bh_eval_order(t, theta, W, 0, ng, groups, H, F, Q, counters, nthreads);
}

/*
 * Interaction lists of one group (for the brute-force pins): accepted node
 * indices and the sorted slots of every particle reached through a leaf
 * (members included; the self term is excluded per member at evaluation).
 * Returns 0; *n_cells / *n_parts receive the full counts even if they exceed
 * the caps.
 */
int ffo_bh_group_lists(const ffo_tree* t, float theta, int W, int64_t g,
                       int64_t* cells, int64_t cap_cells, int64_t* n_cells,
                       int64_t* parts, int64_t cap_parts, int64_t* n_parts)
{
    if (!t || W < 1 || !(theta >= 0.0f)) return -1;
    if (!t->has_moments) return -1;        /* centres rho' are needed by the opening test */
    walk_ctx w;
    memset(&w, 0, sizeof(w));
    w.t = t; w.th2 = theta * theta;
    w.g0 = g * W; w.g1 = w.g0 + W < t->N ? w.g0 + W : t->N;
    static int64_t dummy;
    w.cells = cells ? cells : &dummy; w.cap_cells = cells ? cap_cells : 0;
    w.parts = parts ? parts : &dummy; w.cap_parts = parts ? cap_parts : 0;
    visit(&w, 0);
    *n_cells = w.n_cells_out; *n_parts = w.n_parts_out;
    return 0;
}
