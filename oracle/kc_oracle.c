/*
 * kc_oracle.c — CPU ORACLE for the exact 2-nearest-neighbour certificate path.
 *
 * TEST INFRASTRUCTURE ONLY.  This file is the plain, slow, obviously-correct
 * restatement of what arxiv/paper_2606_18314 ("Repair Entropy in Dynamic
 * Geometric Nearest-Neighbour Structures") defines.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may build, load or call it.  It shares no code, header, table or helper with
 * the CUDA library under paper_2606_18314_b200/csrc/ and neither includes the
 * other.  The product path never routes through it.
 *
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -fopenmp -shared -fPIC
 *        (no FMA contraction, no flush-to-zero, IEEE binary32 throughout).
 *
 * Citations are PAPER.md:<line> (+ section) and SURVEY.md §8(c) reading ids
 * (O1..O8 oracle clauses, A1..A18 readings), restated in DESIGN.md.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): hand-worked dyadic scenes
 * (tests/golden/), Theorem-1 tightness construction, lattice
 * closed forms, entropy closed forms, Theorem 3, Lemma 1 invariant, brute
 * force vs k-d tree vs scipy fp64; the K-list certificate (orc_bruteforce_topk)
 * by hand-worked lists with bit patterns, a numpy lexsort restatement, K = 2 =
 * Definition 1 and the stability of the (K-1)-NN set beyond 4 eps.  No function
 * here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_NOIDX INT32_MAX

/* ---------------------------------------------------------------- O1 ------
 * Squared distance, north_star: ((dx*dx)+(dy*dy))+(dz*dz), every operation a
 * separately rounded binary32 op (this translation unit is compiled with
 * -ffp-contract=off so gcc cannot fuse the multiply and the add).
 * Definition 1's distances are sqrtf of this.                */
static inline float sq2(const float *a, const float *b)
{
    float dx = a[0] - b[0];
    float dy = a[1] - b[1];
    float xx = dx * dx;
    float yy = dy * dy;
    return xx + yy;
}
static inline float sq3(const float *a, const float *b)
{
    float dx = a[0] - b[0];
    float dy = a[1] - b[1];
    float dz = a[2] - b[2];
    float xx = dx * dx;
    float yy = dy * dy;
    float zz = dz * dz;
    float xy = xx + yy;
    return xy + zz;
}
float orc_sqdist(const float *a, const float *b, int d)
{
    return d == 2 ? sq2(a, b) : sq3(a, b);
}

/* running two smallest keys under the total order (s, j) — reading A2:
 * equal squared distances are broken by the smaller index.                  */
typedef struct { float s1, s2; int32_t j1, j2; } top2;

static inline void top2_init(top2 *t)
{
    t->s1 = INFINITY; t->s2 = INFINITY; t->j1 = ORC_NOIDX; t->j2 = ORC_NOIDX;
}
static inline void top2_offer(top2 *t, float s, int32_t j)
{
    if (s < t->s1 || (s == t->s1 && j < t->j1)) {
        t->s2 = t->s1; t->j2 = t->j1; t->s1 = s; t->j1 = j;
    } else if (s < t->s2 || (s == t->s2 && j < t->j2)) {
        t->s2 = s; t->j2 = j;
    }
}
/* O2 (Definition 1): nn = j1, d1 = sqrtf(s1), d2 = sqrtf(s2),
 * c = d2 - d1 (one rounded subtraction).  N = 2 gives d2 = c = +inf (A4).   */
static inline void top2_store(const top2 *t, int64_t i, int32_t *nn, int32_t *nn2,
                              float *d1, float *d2, float *c)
{
    float a = sqrtf(t->s1), b = sqrtf(t->s2);
    nn[i] = t->j1 == ORC_NOIDX ? -1 : t->j1;
    if (nn2) nn2[i] = t->j2 == ORC_NOIDX ? -1 : t->j2;
    d1[i] = a; d2[i] = b; c[i] = b - a;
}

/* ---------------------------------------------------------------- O2 ------
 * Brute force: for every i, scan every j != i (A3: only j = i is excluded; a
 * coincident point is a legitimate neighbour at distance 0).  O(N^2).       */
int orc_bruteforce_top2(const float *p, int64_t N, int d, int32_t *nn, int32_t *nn2,
                        float *d1, float *d2, float *c, int nthreads)
{
    if (!p || !nn || !d1 || !d2 || !c || N < 2 || (d != 2 && d != 3)) return -1;
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(static) num_threads(nthreads)
    for (int64_t i = 0; i < N; ++i) {
        top2 t; top2_init(&t);
        const float *pi = p + i * d;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            float s = d == 2 ? sq2(pi, p + j * d) : sq3(pi, p + j * d);
            top2_offer(&t, s, (int32_t)j);
        }
        top2_store(&t, i, nn, nn2, d1, d2, c);
    }
    return 0;
}

/* Same definition for a subset of query indices q[0..nq) against all N points
 * (used to check sampled outputs at sizes where N^2 is out of reach).
 * Outputs are indexed by position in q.                                     */
int orc_bruteforce_top2_subset(const float *p, int64_t N, int d, const int32_t *q, int64_t nq,
                               int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c,
                               int nthreads)
{
    if (!p || !q || !nn || !d1 || !d2 || !c || N < 2 || (d != 2 && d != 3)) return -1;
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(dynamic, 4) num_threads(nthreads)
    for (int64_t k = 0; k < nq; ++k) {
        int64_t i = q[k];
        top2 t; top2_init(&t);
        const float *pi = p + i * d;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            float s = d == 2 ? sq2(pi, p + j * d) : sq3(pi, p + j * d);
            top2_offer(&t, s, (int32_t)j);
        }
        top2_store(&t, k, nn, nn2, d1, d2, c);
    }
    return 0;
}

/* ------------------------------------------------ NEXT #4: K-list certificate
 * "Richer geometric certificates (... k-nearest-neighbour graphs ...) are left
 * open" (Limitations); the paper studies "k=2 certificates", i.e.
 * the list of the 2 smallest keys (Definition 1).  Reading R20
 * (DESIGN.md): the K-list certificate of point i is the list of the K smallest
 * keys (s(i,j), j), j != i, in ascending order of the same total order (O1, A2,
 * A3): ids nnk[0..K), distances dk[q] = sqrtf(s_q), and the clearance of its
 * (K-1)-nearest-neighbour SET,  ck = dk[K-1] - dk[K-2]  (one rounded
 * subtraction).  K = 2 is Definition 1 exactly (nn = nnk[0], d1, d2, c).  A
 * missing entry (fewer than K other points) has id -1 and distance +inf, and
 * ck = +inf whenever dk[K-1] = +inf.
 * Written as the definition: collect every key, keep the list sorted by plain
 * insertion.  q == NULL means every point is a query.  O(nq N K).            */
int orc_bruteforce_topk(const float *p, int64_t N, int d, int K, const int32_t *q, int64_t nq,
                        int32_t *nnk, float *dk, float *ck, int nthreads)
{
    if (!p || !nnk || !dk || !ck || N < 2 || (d != 2 && d != 3) || K < 2 || K > 64) return -1;
    if (!q) nq = N;
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(dynamic, 4) num_threads(nthreads)
    for (int64_t k = 0; k < nq; ++k) {
        int64_t i = q ? q[k] : k;
        float ls[64];
        int32_t lj[64];
        int n = 0;                                   /* entries held, ascending in (s, j) */
        const float *pi = p + i * d;
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            float s = d == 2 ? sq2(pi, p + j * d) : sq3(pi, p + j * d);
            int pos = n;                             /* first position whose key is larger */
            while (pos > 0 && (s < ls[pos - 1] || (s == ls[pos - 1] && (int32_t)j < lj[pos - 1]))) --pos;
            if (pos >= K) continue;
            int last = n < K ? n : K - 1;
            for (int t = last; t > pos; --t) { ls[t] = ls[t - 1]; lj[t] = lj[t - 1]; }
            ls[pos] = s; lj[pos] = (int32_t)j;
            if (n < K) ++n;
        }
        for (int t = 0; t < K; ++t) {
            nnk[k * K + t] = t < n ? lj[t] : -1;
            dk[k * K + t] = t < n ? sqrtf(ls[t]) : INFINITY;
        }
        float a = dk[k * K + K - 2], b = dk[k * K + K - 1];
        ck[k] = isinf(b) ? INFINITY : b - a;
    }
    return 0;
}

/* ---------------------------------------------------------------- O7 ------
 * k-d tree ("Exact nearest neighbours for ground truth are
 * computed with a k-d tree"): median split on the widest axis, leaves of at
 * most KD_LEAF points scanned with O1 under the (s, j) order.  A subtree is
 * skipped only if a DOUBLE-precision lower bound on the squared distance to
 * its bounding box exceeds s2*(1+1e-6) + 1e-37, never at equality, so neither
 * fp32 rounding of s nor the index tie rule can be pruned away.  Checked
 * bitwise against orc_bruteforce_top2 before it is trusted (tests).         */
#define KD_LEAF 12
typedef struct {
    int32_t lo, hi;        /* range in perm */
    int32_t left, right;   /* child node ids, -1 for a leaf */
    double bmin[3], bmax[3];
} kdnode;
typedef struct {
    const float *p; int d; int64_t N;
    int32_t *perm; kdnode *nodes; int32_t n_nodes, cap_nodes;
} kdtree;

static inline int kd_less(const kdtree *t, int32_t a, int32_t b, int ax)
{
    float xa = t->p[(int64_t)a * t->d + ax], xb = t->p[(int64_t)b * t->d + ax];
    return xa < xb || (xa == xb && a < b);
}
/* quickselect: place the k-th smallest (by coordinate ax, then index) at k  */
static void kd_select(kdtree *t, int32_t lo, int32_t hi, int32_t k, int ax)
{
    int32_t *a = t->perm;
    while (hi - lo > 1) {
        int32_t mid = lo + (hi - lo) / 2, last = hi - 1, tmp;
        /* median of three as pivot, moved to a[last] */
        if (kd_less(t, a[mid], a[lo], ax)) { tmp = a[mid]; a[mid] = a[lo]; a[lo] = tmp; }
        if (kd_less(t, a[last], a[lo], ax)) { tmp = a[last]; a[last] = a[lo]; a[lo] = tmp; }
        if (kd_less(t, a[last], a[mid], ax)) { tmp = a[last]; a[last] = a[mid]; a[mid] = tmp; }
        tmp = a[mid]; a[mid] = a[last]; a[last] = tmp;
        int32_t piv = a[last], st = lo;
        for (int32_t i = lo; i < last; ++i)
            if (kd_less(t, a[i], piv, ax)) { tmp = a[i]; a[i] = a[st]; a[st] = tmp; ++st; }
        tmp = a[st]; a[st] = a[last]; a[last] = tmp;
        if (k == st) return;
        if (k < st) hi = st; else lo = st + 1;
    }
}
static int32_t kd_build(kdtree *t, int32_t lo, int32_t hi)
{
    int32_t id = t->n_nodes++;
    kdnode *n = &t->nodes[id];
    n->lo = lo; n->hi = hi; n->left = n->right = -1;
    for (int a = 0; a < 3; ++a) { n->bmin[a] = INFINITY; n->bmax[a] = -INFINITY; }
    for (int32_t k = lo; k < hi; ++k)
        for (int a = 0; a < t->d; ++a) {
            double x = t->p[(int64_t)t->perm[k] * t->d + a];
            if (x < n->bmin[a]) n->bmin[a] = x;
            if (x > n->bmax[a]) n->bmax[a] = x;
        }
    if (hi - lo <= KD_LEAF) return id;
    int ax = 0; double ext = -1.0;
    for (int a = 0; a < t->d; ++a)
        if (n->bmax[a] - n->bmin[a] > ext) { ext = n->bmax[a] - n->bmin[a]; ax = a; }
    if (!(ext > 0.0)) return id;              /* all coincident: keep as one leaf */
    int32_t mid = lo + (hi - lo) / 2;
    kd_select(t, lo, hi, mid, ax);
    int32_t l = kd_build(t, lo, mid);
    int32_t r = kd_build(t, mid, hi);
    t->nodes[id].left = l; t->nodes[id].right = r;   /* nodes[] never moves */
    return id;
}
static inline double kd_lb(const kdnode *n, const float *x, int d)
{
    double s = 0.0;
    for (int a = 0; a < d; ++a) {
        double v = x[a], g = 0.0;
        if (v < n->bmin[a]) g = n->bmin[a] - v; else if (v > n->bmax[a]) g = v - n->bmax[a];
        s += g * g;
    }
    return s;
}
static void kd_query(const kdtree *t, int32_t id, int32_t i, const float *x, top2 *best)
{
    const kdnode *n = &t->nodes[id];
    if (kd_lb(n, x, t->d) > (double)best->s2 * (1.0 + 1e-6) + 1e-37) return;
    if (n->left < 0) {
        for (int32_t k = n->lo; k < n->hi; ++k) {
            int32_t j = t->perm[k];
            if (j == i) continue;
            const float *pj = t->p + (int64_t)j * t->d;
            float s = t->d == 2 ? sq2(x, pj) : sq3(x, pj);
            top2_offer(best, s, j);
        }
        return;
    }
    double ll = kd_lb(&t->nodes[n->left], x, t->d), lr = kd_lb(&t->nodes[n->right], x, t->d);
    if (ll <= lr) { kd_query(t, n->left, i, x, best); kd_query(t, n->right, i, x, best); }
    else          { kd_query(t, n->right, i, x, best); kd_query(t, n->left, i, x, best); }
}
/* q == NULL: all N points (outputs indexed by point); else the nq listed
 * queries (outputs indexed by position in q).                               */
int orc_kdtree_top2(const float *p, int64_t N, int d, const int32_t *q, int64_t nq,
                    int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c, int nthreads)
{
    if (!p || !nn || !d1 || !d2 || !c || N < 2 || N > INT32_MAX - 1 || (d != 2 && d != 3)) return -1;
    if (nthreads < 1) nthreads = 1;
    kdtree t; t.p = p; t.d = d; t.N = N; t.n_nodes = 0;
    t.cap_nodes = (int32_t)(2 * (N / (KD_LEAF / 2) + 2));
    t.perm = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    t.nodes = (kdnode *)malloc(sizeof(kdnode) * (size_t)t.cap_nodes);
    if (!t.perm || !t.nodes) { free(t.perm); free(t.nodes); return -2; }
    for (int64_t i = 0; i < N; ++i) t.perm[i] = (int32_t)i;
    kd_build(&t, 0, (int32_t)N);
    int64_t M = q ? nq : N;
#pragma omp parallel for schedule(dynamic, 256) num_threads(nthreads)
    for (int64_t k = 0; k < M; ++k) {
        int32_t i = q ? q[k] : (int32_t)k;
        top2 b; top2_init(&b);
        kd_query(&t, 0, i, p + (int64_t)i * d, &b);
        top2_store(&b, k, nn, nn2, d1, d2, c);
    }
    free(t.perm); free(t.nodes);
    return 0;
}

/* ---------------------------------------------------------------- O3 ------
 * Algorithm 1 line 1 and PAPER.md:41:
 * eps_t = max_i ||p'_i - p_i||, each norm = sqrtf(O1).                      */
float orc_max_displacement(const float *p, const float *p2, int64_t N, int d)
{
    float e = 0.0f;
    for (int64_t i = 0; i < N; ++i) {
        float s = d == 2 ? sq2(p2 + i * d, p + i * d) : sq3(p2 + i * d, p + i * d);
        float r = sqrtf(s);
        if (r > e) e = r;
    }
    return e;
}

/* ---------------------------------------------------------------- O4 ------
 * Algorithm 1 line 2: F = { i : d2_i - d1_i <= 4 eps }.
 * Inclusive, because Lemma 1 is safe only for c_i > 4 eps.
 * thr = 4*eps is an exact scaling in binary32.  Returns |F|.                */
int64_t orc_frontier(const float *c, int64_t N, float eps, uint8_t *flags)
{
    float thr = 4.0f * eps;
    int64_t n = 0;
    for (int64_t i = 0; i < N; ++i) {
        uint8_t f = c[i] <= thr ? 1 : 0;
        if (flags) flags[i] = f;
        n += f;
    }
    return n;
}

/* ------------------------------------------------------------ O5 / A6 -----
 * Uniform grid ("resolution is chosen so the mean cell
 * occupancy is a small constant").  Reading A6: the same G on every axis,
 * the smallest integer with G^d >= ceil(N/occ); cubic cells of width
 * h = max_a(hi_a - lo_a)/G * (1 + 2^-20) evaluated in double and rounded to
 * binary32 once; inv_h = 1/h in double from the rounded h, rounded once.    */
typedef struct {
    int32_t d; int32_t G[3];
    float lo[3]; float h; float inv_h;
} orc_geom;

void orc_bbox(const float *p, int64_t N, int d, float lo[3], float hi[3])
{
    for (int a = 0; a < 3; ++a) { lo[a] = 0.0f; hi[a] = 0.0f; }
    for (int a = 0; a < d; ++a) { lo[a] = INFINITY; hi[a] = -INFINITY; }
    for (int64_t i = 0; i < N; ++i)
        for (int a = 0; a < d; ++a) {
            float x = p[i * d + a];
            if (x < lo[a]) lo[a] = x;
            if (x > hi[a]) hi[a] = x;
        }
}
int orc_geom_from_bbox(int64_t N, int d, const float lo[3], const float hi[3], double occ,
                       orc_geom *g)
{
    if (!g || !lo || !hi || N < 1 || (d != 2 && d != 3) || !(occ > 0.0)) return -1;
    int64_t target = (int64_t)ceil((double)N / occ);
    if (target < 1) target = 1;
    int64_t G = 1;
    for (;;) {
        int64_t v = 1;
        for (int a = 0; a < d; ++a) v *= G;
        if (v >= target) break;
        ++G;
    }
    double ext = 0.0;
    for (int a = 0; a < d; ++a) {
        double e = (double)hi[a] - (double)lo[a];
        if (e > ext) ext = e;
    }
    double hd = ext > 0.0 ? ext / (double)G * (1.0 + 1.0 / 1048576.0) : 1.0;
    g->d = d;
    g->G[0] = (int32_t)G; g->G[1] = (int32_t)G; g->G[2] = d == 3 ? (int32_t)G : 1;
    for (int a = 0; a < 3; ++a) g->lo[a] = a < d ? lo[a] : 0.0f;
    g->h = (float)hd;
    g->inv_h = (float)(1.0 / (double)g->h);
    return 0;
}
/* O5: per axis t = fl(fl(x - lo) * inv_h), k = clamp(floorf(t), 0, G-1);
 * linear id = (kz*G1 + ky)*G0 + kx.                                         */
void orc_cell_ids(const float *p, int64_t N, const orc_geom *g, int32_t *cell)
{
    for (int64_t i = 0; i < N; ++i) {
        int32_t k[3] = {0, 0, 0};
        for (int a = 0; a < g->d; ++a) {
            float u = p[i * g->d + a] - g->lo[a];
            float t = u * g->inv_h;
            float f = floorf(t);
            int32_t v = f < 0.0f ? 0 : (f > (float)(g->G[a] - 1) ? g->G[a] - 1 : (int32_t)f);
            k[a] = v;
        }
        cell[i] = (k[2] * g->G[1] + k[1]) * g->G[0] + k[0];
    }
}

/* ---------------------------------------------------------------- O6 ------
 * Definition 2: q_k = fraction of the frontier in occupied
 * cell k; H = -sum q_k log q_k / log C, C = number of cells occupied by ANY
 * point.  Written here literally as the sum over cells of -q log q (double).
 * Readings: n = |F| = 0 -> H = 0; C <= 1 -> H = 0; also m = #cells the
 * frontier meets (Theorem 3).                                 */
int orc_entropy(const int32_t *cell_all, int64_t N, const int32_t *F, int64_t nF, int64_t Ctot,
                double *H, int32_t *m_cells, int32_t *C_occ)
{
    if (!cell_all || !H || Ctot < 1 || nF < 0 || (nF > 0 && !F)) return -1;
    int32_t *tot = (int32_t *)calloc((size_t)Ctot, sizeof(int32_t));
    int32_t *k = (int32_t *)calloc((size_t)Ctot, sizeof(int32_t));
    if (!tot || !k) { free(tot); free(k); return -2; }
    for (int64_t i = 0; i < N; ++i) tot[cell_all[i]]++;
    for (int64_t f = 0; f < nF; ++f) k[cell_all[F[f]]]++;
    int64_t C = 0, m = 0;
    double S = 0.0;
    for (int64_t cix = 0; cix < Ctot; ++cix) {
        if (tot[cix] > 0) ++C;
        if (k[cix] > 0) {
            ++m;
            double q = (double)k[cix] / (double)nF;
            S -= q * log(q);
        }
    }
    *H = (nF == 0 || C <= 1) ? 0.0 : S / log((double)C);
    if (m_cells) *m_cells = (int32_t)m;
    if (C_occ) *C_occ = (int32_t)C;
    free(tot); free(k);
    return 0;
}

int orc_num_procs(void)
{
#ifdef _OPENMP
    return omp_get_num_procs();
#else
    return 1;
#endif
}
