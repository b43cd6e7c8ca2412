/*
 * kc.h — C-ABI of the B200 (sm_100a) kinetic 2-NN certificate library (libkc.so).
 *
 * What it computes: the per-step exact 2-nearest-neighbour certificate maintenance of
 * "Repair Entropy in Dynamic Geometric Nearest-Neighbour Structures" (arxiv/paper_2606_18314):
 * for N moving points in d = 2 or 3 the certificate (nn_i, d1_i <= d2_i), the clearance
 * c_i = d2_i - d1_i (Definition 1), the candidate repair frontier
 * F = {i : c_i <= 4 eps} (Lemma 1; Algorithm 1 line 2), the
 * normalised frontier entropy H(F) over the index cells (Definition 2), and the
 * frontier-only repair against a resident uniform grid (Algorithm 1 lines 3-7).
 *
 * Conventions (all entry points):
 *  - Pointers are DEVICE pointers owned by the caller unless the comment says "host".
 *    The library never frees or keeps a caller pointer beyond the call's stream work.
 *  - Positions are contiguous row-major float32 [N][d] (d = 2 or 3).  Indices are int32.
 *    Outputs are indexed by the ORIGINAL point id.  nn2 (runner-up index) may be NULL.
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Every call is
 *    asynchronous on that stream; no call synchronises the host except kc_grid_info and
 *    kc_fp32_probe, which say so.  Counts that one call produces and the next consumes
 *    (|F|, eps_t) stay on the device.
 *  - Arithmetic (north_star): squared distance
 *    s = ((dx*dx)+(dy*dy))+(dz*dz) with separately rounded binary32 ops (no FMA, no FTZ);
 *    the two smallest keys under the total order (s, j) (equal s: smaller index first);
 *    d1 = sqrtf(s1), d2 = sqrtf(s2) correctly rounded, c = d2 - d1.  Only j = i is excluded;
 *    coincident points are neighbours at distance 0.  N = 2 gives d2 = c = +inf, nn2 = -1.
 *  - Errors: every function returns a kc_status.  KC_EINVAL for a bad argument (d not in {2,3},
 *    N < 2, a required pointer NULL or misaligned, workspace too small ...); KC_ENOMEM when a
 *    device allocation fails; KC_ECUDA when the CUDA runtime reports an error (text in
 *    kc_last_error()); KC_EREBUILD when the resident grid cannot serve the call (not built yet,
 *    N differs from the build, or a whole-set search is asked of an incrementally updated
 *    grid) and the caller must call kc_grid_build / kc_cert_grid_rebuild first.
 *    Non-finite coordinates are a precondition violation: no crash, unspecified certificates.
 *  - There is no CPU fallback anywhere in this library.
 */
#ifndef KC_H_
#define KC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    KC_OK = 0,
    KC_EINVAL = -1,
    KC_ENOMEM = -2,
    KC_ECUDA = -3,
    KC_EREBUILD = -4
} kc_status;

/* Uniform-grid geometry ("a uniform grid whose resolution is chosen so the mean
 * cell occupancy is a small constant").  Cubic cells of width h; cell of x on axis a is
 * clamp(floorf(fl(fl(x - lo[a]) * inv_h)), 0, G[a]-1); linear id = (kz*G[1] + ky)*G[0] + kx.
 * Points outside the box are filed in the nearest boundary cell (the search stays exact). */
typedef struct {
    int32_t d;          /* 2 or 3 */
    int32_t G[3];       /* cells per axis; G[2] = 1 when d = 2 */
    float lo[3];        /* grid origin */
    float h;            /* cell width */
    float inv_h;        /* binary32 nearest to 1/h */
} kc_geom;

/* Opaque resident grid: library-owned device buffers sized at creation. */
typedef struct kc_grid kc_grid;

/* Host-side snapshot of the grid's device counters (kc_grid_info). */
typedef struct {
    int64_t n_points;    /* N of the last build */
    int64_t n_cells;     /* G[0]*G[1]*G[2] */
    int32_t c_occ;       /* C: cells holding >= 1 point, as of the last build or the last
                          * kc_frontier_entropy call, whichever is later */
    int32_t max_occ;     /* largest cell occupancy seen by the last build */
    int32_t n_misfiled;  /* points re-filed into overflow chains since the last build */
    int32_t built;       /* 1 once kc_grid_build has run */
    int32_t dirty;       /* 1 once kc_frontier_repair has updated the grid since the build */
    int32_t n_stragglers;/* queries of the last search that needed more than the solo rings */
    int32_t n_heavy;     /* level-0 cells the last build subdivided (two-level index) */
    int32_t n_leaves;    /* leaves of the last build: undivided cells + sub-cells */
    int32_t heavy_T;     /* build-time record count from which a cell is subdivided */
    int32_t n_handed;    /* queries the ring search handed to the brute-force pass since the last build */
    int32_t n_deferred;  /* d = 3, grids of >= 100,000 points with subdivided cells: queries that the whole-set
                          * search / the slot sweep left to their second kernel since the last build */
} kc_grid_info_t;

/* ---- host utilities -------------------------------------------------------------------- */

const char *kc_version(void);
/* host; thread-local text of the last KC_ECUDA / KC_EINVAL raised on this thread. */
const char *kc_last_error(void);

/* host.  Geometry for a bounding box [lo, hi] (host float[3] each; entries beyond d ignored):
 * the same G on every axis, the smallest integer with G^d >= ceil(N/occ) (occ = target mean
 * occupancy, 2.0 in BASELINE.json's configs); h = max_a(hi[a]-lo[a])/G*(1+2^-20) evaluated in
 * double and rounded once; inv_h = 1/h from the rounded h (reading A6 of PAPER.md:27).
 * A degenerate box (all extents 0) gets h = 1. */
kc_status kc_geom_from_bbox(int64_t N, int d, const float *lo, const float *hi, double occ,
                            kc_geom *out);

/* device.  Exact per-axis min / max of p: lo_hi[0..2] = min, lo_hi[3..5] = max (device float[6];
 * unused axes 0).  For callers that refit the geometry to moved points. */
kc_status kc_bbox(const float *p, int64_t N, int d, float *lo_hi, void *stream);

/* p: device.  Geometry for point sets whose density is far from uniform (reading R24 of
 * PAPER.md:27, "the resolution is set so that the mean cell occupancy is a small constant"): the
 * occupancy is measured against the MEDIAN density of the occupied volume, so that points packed into
 * clusters of negligible volume do not shrink the cells of everything else.  R = the largest integer
 * with R^d * 64 <= N (at most 32 for d = 3, 256 for d = 2); the points are counted in the R^d cells of
 * kc_geom_from_bbox(R^d, d, lo, hi, 1.0) over their bounding box (kc_bbox); med = the lower median of
 * the non-zero counts, n_eff = med * R^d; k = log2(N / n_eff) rounded to the nearest integer and
 * clamped to 0..2 (k grows while 2 (n_eff 2^k)^2 < N^2, in integers); *out = kc_geom_from_bbox(
 * ceil(N / 2^k), d, lo, hi, occ).  A uniform set, or R < 2, gives k = 0: exactly the geometry of
 * kc_geom_from_bbox on the bounding box.  A setup call: it allocates and frees its own scratch
 * (R^d ints), launches 4 kernels on `stream` and SYNCHRONISES it twice; not capturable. */
kc_status kc_geom_by_median_density(const float *p, int64_t N, int d, double occ, void *stream,
                                    kc_geom *out);

/* ---- A0: Algorithm 1 line 1, eps_t = max_i ||p'_i - p_i|| ----------------- */
/* eps_out: device float[1].  Each norm is sqrtf of the squared distance defined above. */
kc_status kc_max_displacement(const float *p, const float *p2, int64_t N, int d, float *eps_out,
                              void *stream);

/* ---- A1: exact all-pairs certificates ("exact N x N pass", Table 2) ---------- */
/* Workspace the tiled kernel needs for (N, d), in bytes (host; 0 only for invalid arguments).
 * WORKSPACE CONTRACT (all kc_cert_allpairs* entry points and kc_frontier_oracle): the caller
 * zero-fills a workspace ONCE, when it is allocated (cudaMemset, torch.zeros); after that it may be
 * passed to any sequence of these calls, for any N, d and start mode, one call at a time (calls on
 * one stream, or otherwise ordered).  Its first 16 + KC_AP_TICKET_BYTES bytes hold the counters of
 * the split launches and nothing else; every call leaves them zero, so no call spends a launch on
 * clearing them.  A counter value that a zero-filled workspace cannot hold never reaches a merge:
 * the kernel reports it through a per-process error word in pinned host memory (no trap, the CUDA
 * context stays usable), leaves the certificates of that query block unspecified, and the NEXT
 * all-pairs call of the process returns KC_EINVAL without running, after clearing the counters of
 * the workspace it was given; the call after that works again.  (The error word is allocated by
 * the first of these calls that runs outside a stream capture.) */
#define KC_AP_TICKET_BYTES (148 * 8 * 8 * 4)
size_t kc_cert_allpairs_workspace(int64_t N, int d);
/* nn,d1,d2,c: device [N]; nn2 device [N] or NULL; workspace: device, 16-byte aligned, >= the size
 * above. */
kc_status kc_cert_allpairs(const float *p, int64_t N, int d, int32_t *nn, int32_t *nn2, float *d1,
                           float *d2, float *c, void *workspace, size_t workspace_bytes,
                           void *stream);

/* A1 for callers that cannot allocate device memory (code under CUDA-graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): the same pass as kc_cert_allpairs (Table 2;
 * same kernels, bit-identical certificates) with its workspace in a file-scope device array of the
 * library instead of a caller-allocated one.  The call makes no cudaMalloc / cudaFree / cudaHostAlloc
 * and calls no allocating routine: one cudaMemsetAsync of the workspace's counters (75,792 B; the array
 * keeps the last call's contents and the counters must start at zero) and the kernels of
 * kc_cert_allpairs, all on `stream`.
 *   p: device float[N*d] (8-byte aligned); nn, d1, d2, c: device [N]; nn2: device [N] or NULL: the
 *   caller's, as in kc_cert_allpairs.
 *   LIMIT: 2 <= N <= kc_cert_allpairs_static_max_n() = 65,536 (the array is 5 MiB; every GPU that loads
 *   the library holds it until exit).  A larger N returns KC_EINVAL with a message naming the limit
 *   and nothing is launched.
 *   SHARED STATE: every call on a device uses the same array.  Calls on one stream (or otherwise
 *   ordered) are fine, back to back; calls that OVERLAP on the GPU (two streams, two host threads,
 *   two replays of a captured graph in flight) race on it and their results are unspecified.
 *   The device address of the array is looked up once per device (cudaGetSymbolAddress, on the first
 *   call with that device current). */
int64_t kc_cert_allpairs_static_max_n(void);
kc_status kc_cert_allpairs_static(const float *p, int64_t N, int d, int32_t *nn, int32_t *nn2, float *d1,
                                  float *d2, float *c, void *stream);

/* A1 started from a kinetic bound.  The certificate logic of Lemma 1: a step in
 * which no point moves by more than eps changes every pairwise distance by at most 2 eps, so the
 * new second-neighbour distance of point i is at most d2_prev[i] + 2 eps.  Given such a bound per
 * point (d2_prev: device float[N], any upper bounds on the previous second-neighbour distances,
 * e.g. the maintained certificates; eps: device float[1], e.g. kc_max_displacement's output), the
 * N x N pass evaluates the same N(N-1) pairs but offers only candidates inside the bound to the
 * top-2 insertion, which a cold start pays ~2 ln N times per point (and, with 32 independent
 * lanes per warp, in almost every step when N is small).  The result never depends on the bound:
 * a point for which fewer than two candidates fall inside it (the bound was wrong, NaN, or
 * stale) is recomputed from scratch in the same call.  Output and workspace as kc_cert_allpairs. */
kc_status kc_cert_allpairs_bounded(const float *p, int64_t N, int d, const float *d2_prev,
                                   const float *eps, int32_t *nn, int32_t *nn2, float *d1, float *d2,
                                   float *c, void *workspace, size_t workspace_bytes, void *stream);

/* A1 started from two known points per query.  Two distinct points a, b other than i at squared
 * distances s_a <= s_b (at the CURRENT positions p) prove that i's second neighbour is no farther
 * than b, so the top-2 list (s_a, a), (s_b, b) is a valid start of the N x N pass: the same
 * N(N-1) pairs are evaluated, only candidates that beat the list reach the insertion.  In a
 * maintenance loop the natural seeds are the point's previous neighbours nn, nn2 (the certificate
 * of Definition 1): after a small step they are still near, and unlike the kinetic
 * bound no eps_t is needed.  seed1, seed2: device int32[N], ANY ids; an id that is out of range,
 * equal to i or (for seed2) equal to seed1[i] is ignored, so the result never depends on the seeds.
 * Output and workspace as kc_cert_allpairs. */
kc_status kc_cert_allpairs_seeded(const float *p, int64_t N, int d, const int32_t *seed1,
                                  const int32_t *seed2, int32_t *nn, int32_t *nn2, float *d1, float *d2,
                                  float *c, void *workspace, size_t workspace_bytes, void *stream);

/* ---- NEXT #1: frontier oracle (PAPER.md:69 rtx_frontier_oracle) -------------------------- */
/* Relabel the queries q[0..*nq) (device int32, distinct ids; *nq read on the device, at most
 * nq_max) against ALL N points by tiled brute force, O(|q| N).  Results are written in place at
 * the query ids (nn[q[k]] ...), other entries are untouched.  workspace: device scratch of at
 * least kc_frontier_oracle_workspace(N, d, nq_max) bytes, 16-byte aligned. */
size_t kc_frontier_oracle_workspace(int64_t N, int d, int64_t nq_max);
kc_status kc_frontier_oracle(const float *p, int64_t N, int d, const int32_t *q, const int32_t *nq,
                             int64_t nq_max, int32_t *nn, int32_t *nn2, float *d1, float *d2,
                             float *c, void *workspace, size_t workspace_bytes, void *stream);

/* ---- A2/A3: uniform grid build and whole-set search (PAPER.md:27, :69 rtx_grid_rebuild) --- */
/* Allocates every device buffer for up to N_max points on geometry *geom (host pointer,
 * copied).  *out receives the handle.  Uses the current CUDA device. */
kc_status kc_grid_create(kc_grid **out, int64_t N_max, const kc_geom *geom);
kc_status kc_grid_destroy(kc_grid *g);
/* Bytes of device memory the grid holds (host). */
size_t kc_grid_bytes(const kc_grid *g);
/* host.  Parameters of the two-level index ("a hierarchical GPU index ... could lower its constant
 * further"): a cell that holds at least heavy_T records at build time is subdivided
 * into S^d sub-cells, S = floor((count / sub_occ)^(1/d)) >= 2, and its records are sorted by
 * sub-cell, so the searches prune inside it.  Defaults: sub_occ = 4; heavy_T = 128 for d = 3 and
 * INT_MAX (no second level) for d = 2, where the whole-set search prunes cell by cell instead;
 * heavy_T is raised to sub_occ * 2^(d+1) if smaller.  (Every search that enters a subdivided cell
 * from outside prunes by sub-cell; the d = 3 whole-set search and slot sweep serve a cell's OWN
 * queries through its sub-cells from max(heavy_T, 256) records on, through the 3^d block of whole
 * cells below that.)  Results never depend on these values.
 * Takes effect with the next kc_grid_build (the grid counts as not built until then). */
kc_status kc_grid_set_index(kc_grid *g, int heavy_T, int sub_occ);

/* A2: cell id per point, per-cell histogram, exclusive scan, scatter into cell-sorted arrays (a
 * counting sort in two levels: the records of a subdivided cell are sorted by sub-cell).
 * After it the grid is resident at positions p (copied; p may be freed afterwards). */
kc_status kc_grid_build(kc_grid *g, const float *p, int64_t N, void *stream);
/* A3: certificates of all N points of a freshly built grid by an exact, unbounded search of the
 * grid (Corollary 1: the block is widened until the second neighbour is
 * provably enclosed; never a search cap).  The 3^d block of the query's leaf first (its sub-cell's
 * block inside a subdivided cell); then d = 3: every cell of the index box
 * [cell(q - r), cell(q + r)] per axis, r >= d2 rounded outwards (the filing function is monotone,
 * so nothing within r can lie outside that box); d = 2 and the fallback of d = 3: wider Chebyshev
 * rings until the distance to the nearest unscanned cell face, shrunk by a rounding slack,
 * exceeds d2, strictly.  Straggler hand-off (this call, kc_frontier_search and
 * kc_frontier_repair): on a grid of >= 200,000 points a query whose rings have reached radius 24
 * (d = 2) / 8 (d = 3) without meeting that bound -- an isolated point, for which ring r costs one
 * thread O(r^(d-1)) dependent row visits -- is put on a list of up to 1,024 queries and finished by a
 * brute-force pass of the whole GPU over all records (the definition of the certificate, so the same
 * bits), launched behind the search kernel; a query that finds the list full goes on with its rings.
 * kc_grid_info_t::n_handed counts them.  KC_EREBUILD if the grid is not freshly built. */
kc_status kc_cert_grid_search(kc_grid *g, int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c,
                              void *stream);
/* A2 + A3 in one call: the O(N) rebuild strategy. */
kc_status kc_cert_grid_rebuild(kc_grid *g, const float *p, int64_t N, int32_t *nn, int32_t *nn2,
                               float *d1, float *d2, float *c, void *stream);

/* ---- A4: Algorithm 1 line 2, F = { i : c_i <= 4 eps } ----------------------- */
/* eps: device float[1] (e.g. kc_max_displacement's output).  flags: device uint8[N] or NULL.
 * F: device int32[N] (capacity N), filled with the frontier ids, ascending inside each block of
 * 1024 ids, blocks in arbitrary order.  nF: device int32[1], set to |F|. */
kc_status kc_frontier_classify(const float *c, int64_t N, const float *eps, uint8_t *flags,
                               int32_t *F, int32_t *nF, void *stream);

/* ---- NEXT #2: frontier from a per-point motion budget ----------------------- */
/* The grid must be resident at p (the pre-step positions; KC_EREBUILD otherwise).  With
 * delta_k = ||p2_k - p_k||, a = nn_i, Delta_B(i) = max delta_k over the points filed in the 3^d cell
 * block of i's cell and R = fl(fl(h (1 - 2^-8)) - max_axis slk) (slk = (|lo| + G h) 2^-20 rounded up):
 *   safe_local(i)  =  c_i > fl(fl(fl(fl(2 delta_i) + delta_a) + Delta_B) K) + m_i
 *                 and  R  > fl(fl(fl(fl(d1_i + fl(2 delta_i)) + delta_a) + eps) K) + m_i,
 *   K = 1 + 2^-18, m_i = fl(fl(d1_i + c_i) 2^-18), every fl one float32 operation, left to right;
 *   F = { i : not ( c_i > fl(4 eps)  or  safe_local(i) ) }   (a subset of kc_frontier_classify's F).
 * Proof sketch: Lemma 1's triangle inequality with individual displacements; points
 * outside the block are at least R away before the step.  nn, d1, c: device [N], exact pre-step
 * certificates; eps: device float[1] = max_k delta_k; flags / F / nF as kc_frontier_classify. */
kc_status kc_frontier_classify_local(kc_grid *g, const float *p, const float *p2, int64_t N,
                                     const int32_t *nn, const float *d1, const float *c, const float *eps,
                                     uint8_t *flags, int32_t *F, int32_t *nF, void *stream);

/* ---- NEXT #3: multi-step maintenance with the cumulative clock (Appendix A.2) -- */
/* S = sum over steps of eps_s.  A certificate last recomputed at clock value S_i stays valid while
 * S - S_i < c_i / 4 (Theorem 1 applied to the cumulative displacement), so the points to revisit in
 * a step are F = { i : c_i <= 4 (S - S_i) }: the flat GPU form of the paper's expiry min-heap.
 *  c: device float[N], clearances as of each point's last recomputation; stamp: device float[N],
 *  the clock value S_i of that recomputation (kc_clock_stamp);
 *  S_in: device double[1], the clock before this step; eps: device float[1], this step's max
 *  displacement; S_out: device double[1] (must differ from S_in), receives S_in + eps;
 *  flags / F / nF: as kc_frontier_classify.
 * The test is evaluated in double: (double)c_i <= 4.0 * (S_out - (double)stamp_i). */
kc_status kc_frontier_classify_clock(const float *c, const float *stamp, int64_t N, const double *S_in,
                                     const float *eps, double *S_out, uint8_t *flags, int32_t *F,
                                     int32_t *nF, void *stream);
/* stamp[i] = *S rounded toward -inf to float32 (the elapsed clock S - S_i is never under-estimated)
 * for the ids in F (*nF on the device, at most nF_max), or for all N points when F is NULL. */
kc_status kc_clock_stamp(const int32_t *F, const int32_t *nF, int64_t nF_max, int64_t N, const double *S,
                         float *stamp, void *stream);

/* The expiry structure of the clock (Theorem 2: "an expiry heap ... O(|F_t| log N)
 * per step") in data-parallel form: a tournament tree over the point ids with fanout 32.  Level-1
 * node j holds a lower bound of min over points 32j .. 32j+31 of the expiry clock stamp_i + c_i / 4
 * (double, rounded down to float, lowered by a relative 2^-22 and 1e-37: more than every rounding of
 * the flat test), level-2 node k the minimum of level-1 nodes 32k .. 32k+31.
 *   tree: device float[kc_clock_tree_floats(N)] = ceil(N/32) + ceil(N/1024) floats, the caller's.
 *   kc_clock_tree_build: all nodes from c and stamp (O(N)).
 *   kc_frontier_classify_clock_tree: the SAME set F as kc_frontier_classify_clock for the same c, stamp,
 *     S_in, eps (and the same S_out), found by reading the ceil(N/1024) level-2 nodes, the children of
 *     those whose bound is <= S (rounded up to float), and the 32 points of those whose bound is <= S,
 *     to which the flat test is applied as written above.  No flags array (that would be O(N) writes);
 *     F in arbitrary order.  c, stamp and tree must be consistent (built, or updated after every change).
 *   kc_clock_tree_update: after the certificates of the ids in F (*nF on the device, at most nF_max)
 *     have been recomputed and re-stamped: their level-1 and level-2 nodes are recomputed (from all
 *     N points when *nF > N / 16, decided on the device; F = NULL: same as build). */
size_t kc_clock_tree_floats(int64_t N);
kc_status kc_clock_tree_build(const float *c, const float *stamp, int64_t N, float *tree, void *stream);
kc_status kc_frontier_classify_clock_tree(const float *c, const float *stamp, int64_t N, const float *tree,
                                          const double *S_in, const float *eps, double *S_out, int32_t *F,
                                          int32_t *nF, void *stream);
kc_status kc_clock_tree_update(const int32_t *F, const int32_t *nF, int64_t nF_max, const float *c,
                               const float *stamp, int64_t N, float *tree, void *stream);

/* ---- NEXT #2: certificate-failure audit (Definition 2; Table 1) -- */
/* The true repair frontier F_t = { i : nn_post[i] != nn_pre[i] } of a step and the audit of the
 * Lemma-1 rule against it.  nn_pre / nn_post: device int32[N], exact certificates before / after
 * the step; flags: device uint8[N] from kc_frontier_classify (1 = c_i <= 4 eps_t).
 * counts: device int32[4] = { |F_t|, detected = failed and flagged, missed = failed but called safe
 * (Lemma 1 guarantees 0), false = flagged but still valid } (the dataset's n_detect_safe /
 * n_missed_safe / n_false_safe).  Ft: device int32[N] or NULL; receives the ids of
 * F_t in arbitrary order (counts[0] entries), ready for kc_frontier_entropy (H(F_t), P_t = |F_t|/N). */
kc_status kc_failure_audit(const int32_t *nn_pre, const int32_t *nn_post, const uint8_t *flags,
                           int64_t N, int32_t *Ft, int32_t *counts, void *stream);

/* ---- A5: Definition 2, H(F) over the grid's cells ------------------------ */
/* F: device int32 list of DISTINCT point ids, *nF entries (device int32[1]), at most nF_max
 * (host upper bound used only to size launches; pass N if unknown).  Cells are the grid's
 * current filing; C counts cells occupied by any point.  Outputs (device): H double[1]
 * (0 when |F| = 0 or C <= 1), m_cells int32[1] (cells the frontier meets, Theorem 3
 * PAPER.md:187), C_occ int32[1]; m_cells / C_occ may be NULL. */
kc_status kc_frontier_entropy(kc_grid *g, const int32_t *F, const int32_t *nF, int64_t nF_max,
                              double *H, int32_t *m_cells, int32_t *C_occ, void *stream);

/* ---- A6 + A7: Algorithm 1 lines 3-7 -------------------------------------- */
/* Incremental update of the resident grid to positions p_new, then exact re-search of the
 * frontier only.
 *  movers: device int32 list of DISTINCT ids whose position differs from what the grid holds
 *          (*n_movers on the device, at most n_movers_max), or NULL = every point may have
 *          moved.  Movers keep their slot if their cell (and, in a subdivided cell, their
 *          sub-cell) is unchanged; otherwise they are tombstoned and re-filed into their new
 *          cell's overflow chain (line 3).  On a grid of >= 100,000 points an update whose
 *          host-side bound allows at least N/8 movers (d = 3, N >= 2^20: N/32) (n_movers_max, or N
 *          for NULL) re-bins the whole grid at p_new instead (A2, O(N)): cheaper than re-filing that
 *          many points one by one, and the search that follows runs on a fresh grid.
 *  F, nF, nF_max: as for kc_frontier_entropy; the queries to recompute (lines 4-7).
 *  nn, nn2, d1, d2, c: certificates, updated IN PLACE at the ids in F, untouched elsewhere.
 * The search is the same unbounded ring search as A3, over sorted ranges and chains. */
kc_status kc_frontier_repair(kc_grid *g, const float *p_new, int64_t N, const int32_t *movers,
                             const int32_t *n_movers, int64_t n_movers_max, const int32_t *F,
                             const int32_t *nF, int64_t nF_max, int32_t *nn, int32_t *nn2,
                             float *d1, float *d2, float *c, void *stream);

/* The two halves of kc_frontier_repair as separate calls (rows A6 and A7): kc_grid_update brings the
 * resident grid to positions p_new (movers as above); kc_frontier_search re-searches the ids in F
 * against the grid as it stands and updates the certificates in place at those ids.  After the
 * update, kc_frontier_entropy and kc_frontier_search touch disjoint state and may run on two streams. */
kc_status kc_grid_update(kc_grid *g, const float *p_new, int64_t N, const int32_t *movers,
                         const int32_t *n_movers, int64_t n_movers_max, void *stream);
kc_status kc_frontier_search(kc_grid *g, const float *p_new, int64_t N, const int32_t *F, const int32_t *nF,
                             int64_t nF_max, int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c,
                             void *stream);

/* CUDA graphs.  Every call only enqueues kernels and memsets on `stream` (kc_grid_create,
 * kc_grid_info and kc_fp32_probe excepted), takes every device-side count from device memory and
 * keeps no per-call counter on the host, so a sequence of calls can be captured once and replayed
 * with other DATA in the same buffers.  What is decided on the HOST at call (= capture) time, and
 * therefore frozen in a captured graph: the kernel variant chosen from N, nF_max and n_movers_max
 * (host-side bounds), whether kc_grid_update re-bins, and the grid's built / updated state, which
 * must be the same at every replay as at capture (capture a whole step, including the build or the
 * update that precedes a search, as paper_2606_18314_b200/driver.py does).  Work lists that a call
 * fills on the device (the sweep marks, the hand-off list, the list of the d = 3 search's second
 * kernel, the scans' descriptors) are emptied or reset by that call's own kernels. */

/* ---- NEXT #4: K-list certificates ---------------------------------------------------------- */
/* "Richer geometric certificates (Delaunay edges, k-nearest-neighbour graphs, ...) are left open"
 * (PAPER.md:114); the paper's certificate is the list of the TWO smallest keys (Definition 1,
 * PAPER.md:29).  The K-list certificate of point i is the list of the K smallest keys
 * (s(i,j), j), j != i, ascending in the total order of "Arithmetic" above (equal s: smaller id):
 *   nnk[i*K + q]  id of the q-th key, -1 if fewer than q+1 other points exist
 *   dk [i*K + q]  sqrtf of its squared distance (+inf if missing)
 *   ck [i]        dk[i*K+K-1] - dk[i*K+K-2] (one rounded subtraction), +inf if dk[i*K+K-1] = +inf:
 *                 the clearance of the (K-1)-nearest-neighbour SET.  By the argument of Lemma 1
 *                  a step with max displacement eps leaves that set unchanged when
 *                 ck > 4 eps, so ck feeds kc_frontier_classify unchanged.
 * K = 2 gives nn = nnk[2i], nn2 = nnk[2i+1], d1, d2, c of kc_cert_allpairs bit for bit.
 * 2 <= K <= KC_TOPK_MAX.  All pointers device, caller-owned: nnk int32[N*K], dk float32[N*K],
 * ck float32[N], row-major.  kc_cert_allpairs_topk: tiled N x N pass (FP32 ALU bound);
 * workspace: device scratch of at least kc_cert_allpairs_topk_workspace(N, d, K) bytes (0 for
 * large N), 4-byte aligned; seed_ids: NULL, or device int32[N*K] with K known points per query
 * (its list from the grid or from the previous step): the pass starts every list from their exact
 * keys at the current positions, which can never make a result wrong (reading R17 for K keys);
 * ANY ids are allowed (out of range, i itself and repeats are ignored); must not alias nnk.
 * kc_cert_grid_topk: ring-expanding search of a freshly built grid,
 * terminating only when the scanned block's bound exceeds the K-th distance (KC_EREBUILD if the
 * grid was updated incrementally since its build).  Asynchronous on `stream`; KC_EINVAL on a NULL
 * pointer, K out of range, N < 2 or d not in {2,3}. */
#define KC_TOPK_MAX 8
size_t kc_cert_allpairs_topk_workspace(int64_t N, int d, int K);
kc_status kc_cert_allpairs_topk(const float *p, int64_t N, int d, int K, const int32_t *seed_ids, int32_t *nnk,
                                float *dk, float *ck, void *workspace, size_t workspace_bytes, void *stream);
kc_status kc_cert_grid_topk(kc_grid *g, int K, int32_t *nnk, float *dk, float *ck, void *stream);
/* A7 for K keys (Algorithm 1 lines 4-7, on K-list certificates): recompute the
 * lists of the ids F[0..*nF) (device int32, *nF read on the device, at most nF_max) against the grid
 * as kc_grid_update left it (p_new: the positions it holds, device [N][d]); rows F[k] of nnk, dk and
 * entry F[k] of ck are overwritten, all others untouched.  With F = {i : ck_i <= 4 eps} the
 * (K-1)-NN set of every other point is still valid (see above).  KC_EREBUILD if the grid was not
 * built for this N. */
kc_status kc_frontier_search_topk(kc_grid *g, const float *p_new, int64_t N, const int32_t *F, const int32_t *nF,
                                  int64_t nF_max, int K, int32_t *nnk, float *dk, float *ck, void *stream);

/* ---- inspection (tests, reports) ---------------------------------------------------------- */
/* Synchronises `stream`, copies the device counters to *out (host). */
kc_status kc_grid_info(kc_grid *g, kc_grid_info_t *out, void *stream);
/* Copies one of the grid's int32 arrays into dst (device int32[capacity], caller-owned),
 * asynchronously on `stream`; *count (host) receives the array length (KC_EINVAL if it exceeds
 * capacity; dst may be NULL to query the length only).
 *  what = 0: cell id of point i, int32[N]      (current filing)
 *         1: cell_start, int32[n_cells+1]      (exclusive scan of the last build's histogram)
 *         2: sorted_idx, int32[N]              (point id in each sorted slot; -1 = tombstone)
 *         3: slot, int32[N]                    (sorted slot of point i; -1 = in an overflow chain)
 *         4: counts, int32[n_cells]            (live occupancy per cell)
 *         5: subinfo, int32[2*n_cells]         (two-level index: per cell {S, first leaf}; meaningful
 *                                               only when kc_grid_info reports n_heavy > 0; S = 0: the
 *                                               cell is one leaf, else it has S^d sub-cells, x fastest)
 *         6: leaf_start, int32[n_cells+N+9]    (exclusive scan of the leaf sizes: the first
 *                                               n_leaves + 1 entries are meaningful) */
kc_status kc_grid_export(const kc_grid *g, int what, int32_t *dst, int64_t capacity, int64_t *count,
                         void *stream);

/* ---- measurement helpers ------------------------------------------------------------------ */
/* host.  Number of CUDA kernels this library has launched in this process so far (bench.py
 * reports the difference over its timed region as gpu_launches). */
uint64_t kc_launch_count(void);
/* Empirical FP32 lane-op rate: `blocks` x 256 threads each run `iters` rounds of 16
 * independent non-fused FADD/FMUL chains; returns separately-rounded FP32 ops/s in *ops_per_s
 * (host double).  Synchronises the stream.  Used only to report the A1 roofline peak. */
kc_status kc_fp32_probe(int blocks, int iters, double *ops_per_s, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* KC_H_ */
