// kc_grid.cuh -- the resident grid's state and the device helpers shared by kc_grid.cu (A2 build,
// A5 entropy, A6 incremental update) and kc_search.cu (A3 / A7 searches).  CUDA side only.
#pragma once
#include <math.h>
#include <stdlib.h>

#include "kc_common.cuh"

namespace kc {

struct Counters {
    int n_misfiled;
    int c_occ;
    int max_occ;
    int n_stragglers;
    int m_cells;
    int n_list2;              // frontier points of the current sweep that live in chains
    int ticket;               // blocks of entropy_collect_kernel that are done (the last one finishes)
    int c_occ_acc;            // recount of the occupied cells in progress (A5 after an incremental update)
    int kmax;                 // largest per-cell frontier count seen by the current A5 call
    int ticket2;              // blocks of the A7 list kernel that are done (the last one empties list2)
    int n_heavy;              // level-0 cells that the last build subdivided (two-level index)
    int n_leaves;             // leaves of the last build: one per undivided cell + S^d per subdivided one
    int n_handoff;            // queries in the hand-off list of the search in progress (zero between calls)
    int ticket3;              // blocks of the hand-off kernel that are done (the last one empties the list)
    int n_handed;             // queries handed to the brute-force pass since the last build
    int scan_ticket;          // block order of the cell scan / the leaf scan of the build in progress
    int lscan_ticket;
    int n_defer;              // queries the leaf search has left to its second kernel (zero between calls)
    int ticket4;              // blocks of that kernel that are done (the last one empties the list)
    int n_deferred;           // queries served by that kernel since the last build
    int defer_next;           // next unserved entry of the list (warps of the second kernel take 32 at a time)
    double big;               // sum k ln k over cells with k >= MHIST (rare)
};

// Two-level index ("a hierarchical GPU index ... could lower its constant further", in
// its grid form).  A level-0 cell that holds at least heavy_T records at build time is subdivided
// into S^d sub-cells, S = floor((count / sub_occ)^(1/d)) >= 2 (sub_occ = 2 records per sub-cell), and its records are sorted by sub-cell
// (x fastest), so a sub-row segment is again ONE contiguous range.  Level-0 contiguity is untouched:
// cell_start[c] .. cell_start[c+1] still holds exactly the records of cell c, and every kernel that
// ignores the second level stays exact.  Leaves (undivided cells and sub-cells) are numbered in
// storage order; leaf_start is the exclusive scan of their sizes, subinfo[c] = {S or 0, first leaf}.
// Sub-cell of coordinate x in cell k of an axis: clamp(floorf(fl(fl(t - k) * S)), 0, S-1) with the
// cell coordinate t = fl(fl(x - lo) * inv_h) of cell_axis(): monotone in x like cell_axis itself.
// Two thresholds (measured on config 5): a cell is SUBDIVIDED from heavy_T records on
// (default 128: whoever visits it from outside prunes by sub-cell), but the leaf search serves the cell's OWN
// queries through its sub-cells only from max(heavy_T, LANE_T_MIN) records on -- below that the 3^d block
// of whole cells is cheaper than the many sub-cells that touch the cell's faces.
constexpr int LANE_T_MIN = 256;
constexpr int KC_INDEX_OFF = 0x7fffffff;          // heavy_T value that switches the second level off

__host__ __device__ inline int sub_res(int cnt, int d, int heavy_T, int sub_occ)
{
    if (cnt < heavy_T) return 0;
    const long long q = cnt / sub_occ;
    int S = d == 2 ? (int)sqrtf((float)q) : (int)cbrtf((float)q);
    if (S < 2) S = 2;
    if (d == 2) {
        while ((long long)(S + 1) * (S + 1) <= q) ++S;
        while (S > 2 && (long long)S * S > q) --S;
    } else {
        while ((long long)(S + 1) * (S + 1) * (S + 1) <= q) ++S;
        while (S > 2 && (long long)S * S * S > q) --S;
    }
    return S;
}
__device__ __forceinline__ int sub_axis(float x, float lo, float inv_h, int k, float fS, int S)
{
    const float t = __fmul_rn(__fsub_rn(x, lo), inv_h);
    const float f = floorf(__fmul_rn(__fsub_rn(t, (float)k), fS));
    return f < 0.0f ? 0 : (f > (float)(S - 1) ? S - 1 : (int)f);
}

struct View {
    int G0, G1, G2;
    float lo0, lo1, lo2, h, inv_h, shrink;
    float slk0, slk1, slk2;   // absolute rounding slack of a computed face / cell boundary per axis
    const int32_t *cell_start;
    const float2 *spos2;
    const float4 *spos4;
    const int32_t *sidx;
    const int32_t *head;
    const int32_t *next;
    const float4 *opos;
    int heavy_T;              // build-time record count from which a level-0 cell is subdivided
    int lane_T;               // >= heavy_T: count from which the leaf search serves a cell's OWN queries through its sub-cells
    const int2 *subinfo;      // per level-0 cell: {S (0 = not subdivided), index of its first leaf}
    const int32_t *leaf_start;   // exclusive scan of the leaf sizes (n_leaves + 1 entries)
    float4 *handoff;          // hand-off list (x, y, z, bits(id)) of ring_continue, or null: rings without limit
    int *n_handoff;           // its length (Counters::n_handoff)
    float4 *defer;            // d = 3: queries whose ball reaches beyond what phase 1 of the leaf search served:
    int *n_defer;             //   two float4 per entry {slot, covered, -, -}, {s1, s2, j1, j2}; length (Counters::n_defer)
};

// Straggler hand-off: a query whose ring search has scanned radius
// HANDOFF_R without meeting its bound (an isolated point: ring r costs O(r^(d-1)) dependent row
// visits of ONE thread, about a thousand by that radius) is appended to a list and finished by a
// brute-force pass of the whole GPU over all records, after the search kernel.  Only on grids of at
// least HANDOFF_MIN_N points (below that the whole grid is a few thousand rows); a list that is full
// leaves the query to the rings.
constexpr int HANDOFF_CAP = 1024;
constexpr int HANDOFF_BLOCKS = 148;              // CTAs of the pass: one record chunk and one partial list each
constexpr int HANDOFF_MIN_N = 200000;
constexpr int HANDOFF_R2 = 24, HANDOFF_R3 = 8;
struct HandoffPart { float s1, s2; int j1, j2; };


}  // namespace kc

struct kc_grid {
    kc_geom geom;
    int64_t N_max, n_cells, N;
    int built, dirty;
    size_t bytes;
    int32_t *cell, *counts, *cell_start, *sidx, *slot, *head, *next, *mlist, *fcount, *mhist;
    unsigned long long *scan_desc;   // look-back descriptors of the build's two scans (cells, then leaves)
    int2 *subinfo;            // two-level index, see View
    int32_t *leaf_cnt, *leaf_start, *leafid;   // leaf sizes, their scan (doubles as scatter cursors), leaf of point i
    int64_t n_leaves_max;
    int heavy_T, sub_occ;
    int32_t *mark;            // per sorted slot: 1 while a sweep has it as a query (zero between calls)
    int32_t *list2;           // frontier points of the current sweep that live in chains
    float4 *handoff;          // hand-off list of the search in progress (HANDOFF_CAP entries; grids of
    kc::HandoffPart *handoff_part;   //   >= HANDOFF_MIN_N points only) and the pass's partial lists [CAP][BLOCKS]
    float *delta;             // NEXT #2: displacement of every point in the current step
    unsigned *cellmax;        // NEXT #2: largest displacement (float bits) per cell
    float2 *spos2;
    float4 *spos4, *opos;
    float4 *defer;            // d = 3: list of the leaf search's second kernel (2 float4 per point)
    kc::Counters *ctr;
    int n_scan_blocks;
};

namespace kc {

inline View make_view(const kc_grid *g)
{
    View v;
    v.G0 = g->geom.G[0]; v.G1 = g->geom.G[1]; v.G2 = g->geom.G[2];
    v.lo0 = g->geom.lo[0]; v.lo1 = g->geom.lo[1]; v.lo2 = g->geom.lo[2];
    v.h = g->geom.h; v.inv_h = g->geom.inv_h;
    int Gm = v.G0 > v.G1 ? v.G0 : v.G1;
    if (v.G2 > Gm) Gm = v.G2;
    // rounding slack of the ring bound: computed cell faces are off by O(u*G) cell widths
    v.shrink = 1.0f - (1.0f / 512.0f + (float)Gm * (1.0f / 524288.0f));
    const int Ga[3] = {v.G0, v.G1, v.G2};
    float slk[3];
    for (int a = 0; a < 3; ++a) {
        double t = (fabs((double)g->geom.lo[a]) + (double)Ga[a] * (double)g->geom.h) / 1048576.0;
        slk[a] = nextafterf((float)t, INFINITY);
    }
    v.slk0 = slk[0]; v.slk1 = slk[1]; v.slk2 = slk[2];
    v.cell_start = g->cell_start;
    v.spos2 = g->spos2; v.spos4 = g->spos4; v.sidx = g->sidx;
    v.head = g->head; v.next = g->next; v.opos = g->opos;
    v.heavy_T = g->heavy_T; v.lane_T = g->heavy_T > LANE_T_MIN ? g->heavy_T : LANE_T_MIN;
    v.subinfo = g->subinfo; v.leaf_start = g->leaf_start;
    v.handoff = nullptr; v.n_handoff = nullptr;       // (the callers that launch the hand-off pass set them)
    v.defer = g->defer; v.n_defer = &g->ctr->n_defer;
    return v;
}

// Append `id` to list[] for the lanes with `want` set: one atomic per warp on the shared cursor
// (every lane of the warp must call it).
__device__ __forceinline__ void warp_append(bool want, int id, int32_t *list, int *cursor)
{
    const unsigned m = __ballot_sync(0xffffffffu, want);
    if (!m) return;
    const int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
    int base = 0;
    if (lane == leader) base = atomicAdd(cursor, __popc(m));
    base = __shfl_sync(0xffffffffu, base, leader);
    if (want) list[base + __popc(m & ((1u << lane) - 1))] = id;
}

template <int D>
__device__ __forceinline__ int cell_of(const View &v, float x, float y, float z)
{
    int kx = cell_axis(x, v.lo0, v.inv_h, v.G0);
    int ky = cell_axis(y, v.lo1, v.inv_h, v.G1);
    int kz = D == 3 ? cell_axis(z, v.lo2, v.inv_h, v.G2) : 0;
    return (kz * v.G1 + ky) * v.G0 + kx;
}

// d = 3: the fraction 1 / div of the points from which a frontier list goes to the slot sweep (kc_search.cu)
// and an update re-bins the grid (kc_grid.cu): lists of up to WPQ_MAX ids get one WARP per query, which wins
// on small grids; beyond that one THREAD per query is slow on clustered cells and the sweep on a fresh grid
// wins down to N / 32 (measured on config 5 and config 4, DESIGN.md section 5 A7).
constexpr int WPQ_MAX = 32768;                       // A7: id lists up to this long get one warp per query
inline int list_div3(int64_t N)
{
    const int64_t d = N / WPQ_MAX;
    return (int)(d < 8 ? 8 : (d > 32 ? 32 : d));
}

inline int blocks_for(int64_t n, int threads, int cap = 148 * 16)
{
    int64_t b = (n + threads - 1) / threads;
    if (b < 1) b = 1;
    return (int)(b < cap ? b : cap);
}

inline kc_status check_certs(const int32_t *nn, const float *d1, const float *d2, const float *c, const char *who)
{
    if (!nn || !d1 || !d2 || !c) {
        set_error("%s: nn, d1, d2, c must be non-NULL", who);
        return KC_EINVAL;
    }
    return KC_OK;
}

}  // namespace kc
