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
    double big;               // sum k ln k over cells with k >= MHIST (rare)
};

struct View {
    int G0, G1, G2;
    float lo0, lo1, lo2, h, inv_h, shrink;
    float slk0, slk1, slk2;   // absolute rounding slack of a computed face / cell boundary per axis
    int dense_thr;            // a row range of at least this many records is handled as dense (A3)
    int wpq_max;              // id lists up to this long are served one warp per query (A7)
    const int32_t *cell_start;
    const float2 *spos2;
    const float4 *spos4;
    const int32_t *sidx;
    const int32_t *head;
    const int32_t *next;
    const float4 *opos;
};

}  // namespace kc

struct kc_grid {
    kc_geom geom;
    int64_t N_max, n_cells, N;
    int built, dirty;
    size_t bytes;
    int32_t *cell, *counts, *cell_start, *sidx, *slot, *head, *next, *mlist, *fcount, *mhist;
    int32_t *blocksums;
    int32_t *mark;            // per sorted slot: epoch of the last sweep that queried it
    int32_t *list2;           // frontier points of the current sweep that live in chains
    float *delta;             // NEXT #2: displacement of every point in the current step
    unsigned *cellmax;        // NEXT #2: largest displacement (float bits) per cell
    int epoch;
    float2 *spos2;
    float4 *spos4, *opos;
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
    static const int dense_env = getenv("KC_DENSE_THR") ? atoi(getenv("KC_DENSE_THR")) : 0;
    v.dense_thr = dense_env > 0 ? dense_env : 128;
    static const int wpq_env = getenv("KC_WPQ_MAX") ? atoi(getenv("KC_WPQ_MAX")) : -1;
    v.wpq_max = wpq_env >= 0 ? wpq_env : 32768;
    v.cell_start = g->cell_start;
    v.spos2 = g->spos2; v.spos4 = g->spos4; v.sidx = g->sidx;
    v.head = g->head; v.next = g->next; v.opos = g->opos;
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
