// kc_search.cu -- A3 whole-set ring search, A7 frontier-only search, K-list searches through the
// resident grid.  Contract: include/kc.h.  Layout of the grid: kc_grid.cuh / kc_grid.cu.
#include "kc_grid.cuh"

using namespace kc;

namespace {

// ------------------------------------------------------------------ A3 / A7 ring search
// Exact top-2 of query (qx,qy,qz), excluding point id `self`, over the grid's sorted ranges and
// (if chains) its overflow chains.  Corollary 1: the block is widened until
// the second neighbour is provably enclosed.
//
// Filing invariant: every record listed in cell k of an axis has a coordinate x with
// cell_axis(x) = k, and cell_axis is monotone, so for a query in cell c < k the real distance
// along that axis is at least  face(k) - q  minus the rounding of the computed face and cell id:
//     x - q >= fl(face_k - q)(1 - u) - u(|lo| + 5.01 G h),      u = 2^-24
// (3 roundings in cell_axis move a cell boundary by <= 3.01 u G h, 2 roundings in
// face_k = fl(lo + fl(k h)) move the face by <= u(|lo| + 2 G h)).  gap_lb() therefore subtracts
// the absolute slack slk = (|lo| + G h) 2^-20 and multiplies by shrink = 1 - 2^-9 - G 2^-19,
// which also covers the <= 3u relative undershoot of an fp32 squared distance.  Points outside
// the grid box are filed in boundary cells; only faces between two cells are ever used, so the
// bound holds for them too (clamping is monotone).
//
// Two uses of the bound, both strict (a tie at equal distance must still be seen, the index
// decides it):
//  * cell pruning inside the 3^d block: a cell whose box is provably farther than the current
//    second-best (sum over axes of the squared shrunk gaps > s2) is skipped.  The query's own
//    cell is scanned first, then its row neighbours, then the other rows nearest first, so in
//    dense cells (occupancy >> 1, d2 << h) most of the block is never touched;
//  * termination: after the Chebyshev-radius-r block is done, every unscanned point lies beyond
//    a block face interior to the grid; stop only when s2 < (min face distance)^2, else scan
//    ring r+1.  No face left = whole grid scanned = stop.  Never a cap.
//
// Candidate ranges are scanned 4 records per step from a 4-aligned start: records in front of the
// range belong to neighbouring cells and the records behind the last slot are NaN padding, so
// the extra ones are either legitimate candidates or inert (every comparison with NaN is false).
// A candidate can therefore be offered more than once; the insertion skips ids already held.
__device__ __forceinline__ void offer_once(Top2 &best, float s, int j, int self)
{
    if (s <= best.s2 && j >= 0 && j != self && j != best.j1 && j != best.j2) best.offer(s, j);
}
template <int D>
__device__ __noinline__ Top2 slow_offer4(const View &v, Top2 best, int t, float s0, float s1,
                                         float s2, float s3, int self)
{
    // the smallest of the four first, retired with NaN (fminf skips it), until none qualifies: the
    // lanes on this path stay in step whichever of their four candidates it is about
    float m = fminf(fminf(s0, s1), fminf(s2, s3));
    while (m <= best.s2) {
        const bool p0 = s0 == m, p1 = !p0 && s1 == m, p2 = !p0 && !p1 && s2 == m;
        const int k = p0 ? 0 : (p1 ? 1 : (p2 ? 2 : 3));
        const float qn = __int_as_float(0x7fc00000);
        s0 = p0 ? qn : s0; s1 = p1 ? qn : s1; s2 = p2 ? qn : s2; s3 = (p0 || p1 || p2) ? s3 : qn;
        const int j = D == 2 ? v.sidx[t + k] : __float_as_int(v.spos4[t + k].w);
        offer_once(best, m, j, self);
        m = fminf(fminf(s0, s1), fminf(s2, s3));
    }
    return best;
}
template <int D>
__device__ __forceinline__ void scan_range(const View &v, int b, int e, float qx, float qy, float qz,
                                           int self, Top2 &best)
{
    for (int t = b & ~3; t < e; t += 4) {
        float s0, s1, s2, s3;
        if (D == 2) {
            const float4 A = *reinterpret_cast<const float4 *>(v.spos2 + t);       // x0 y0 x1 y1
            const float4 B = *reinterpret_cast<const float4 *>(v.spos2 + t + 2);   // x2 y2 x3 y3
            s0 = sqd2(qx, qy, A.x, A.y); s1 = sqd2(qx, qy, A.z, A.w);
            s2 = sqd2(qx, qy, B.x, B.y); s3 = sqd2(qx, qy, B.z, B.w);
        } else {
            const float4 c0 = v.spos4[t], c1 = v.spos4[t + 1], c2 = v.spos4[t + 2], c3 = v.spos4[t + 3];
            s0 = sqd3(qx, qy, qz, c0.x, c0.y, c0.z); s1 = sqd3(qx, qy, qz, c1.x, c1.y, c1.z);
            s2 = sqd3(qx, qy, qz, c2.x, c2.y, c2.z); s3 = sqd3(qx, qy, qz, c3.x, c3.y, c3.z);
        }
        float m = fminf(fminf(s0, s1), fminf(s2, s3));
        if (m <= best.s2) best = slow_offer4<D>(v, best, t, s0, s1, s2, s3, self);
    }
}
template <int D>
__device__ __forceinline__ void scan_chain(const View &v, int cidx, float qx, float qy, float qz,
                                           int self, Top2 &best)
{
    for (int e = v.head[cidx]; e >= 0; e = v.next[e]) {
        float4 c = v.opos[e];
        float s = D == 2 ? sqd2(qx, qy, c.x, c.y) : sqd3(qx, qy, qz, c.x, c.y, c.z);
        offer_once(best, s, e, self);
    }
}

__device__ __forceinline__ float face_at(float lo, int k, float h)
{
    return __fadd_rn(lo, __fmul_rn((float)k, h));
}
// lower bound of the real axis distance behind a computed face at computed distance `gap`
__device__ __forceinline__ float gap_lb(const View &v, float gap, float slk)
{
    return __fmul_rn(fmaxf(__fsub_rn(gap, slk), 0.0f), v.shrink);
}
// squared lower bounds of the axis distance from the query to its six neighbour cells
struct Gaps { float xm, xp, ym, yp, zm, zp; };
template <int D>
__device__ __forceinline__ Gaps make_gaps(const View &v, float qx, float qy, float qz, int cx, int cy, int cz)
{
    Gaps g;
    float t;
    t = gap_lb(v, __fsub_rn(qx, face_at(v.lo0, cx, v.h)), v.slk0); g.xm = __fmul_rn(t, t);
    t = gap_lb(v, __fsub_rn(face_at(v.lo0, cx + 1, v.h), qx), v.slk0); g.xp = __fmul_rn(t, t);
    t = gap_lb(v, __fsub_rn(qy, face_at(v.lo1, cy, v.h)), v.slk1); g.ym = __fmul_rn(t, t);
    t = gap_lb(v, __fsub_rn(face_at(v.lo1, cy + 1, v.h), qy), v.slk1); g.yp = __fmul_rn(t, t);
    g.zm = 0.f; g.zp = 0.f;
    if (D == 3) {
        t = gap_lb(v, __fsub_rn(qz, face_at(v.lo2, cz, v.h)), v.slk2); g.zm = __fmul_rn(t, t);
        t = gap_lb(v, __fsub_rn(face_at(v.lo2, cz + 1, v.h), qz), v.slk2); g.zp = __fmul_rn(t, t);
    }
    return g;
}
// The 3^(d-1) - 1 rows of the block other than the query's own, nearest first: offsets (oy, oz)
// packed two bits each as offset + 1.
//   k:   0       1       2       3       4        5        6        7
//  oy:  -1      +1       0       0      -1       +1       -1       +1
//  oz:   0       0      -1      +1      -1       -1       +1       +1
constexpr unsigned ROW_OY = 0u | (2u << 2) | (1u << 4) | (1u << 6) | (0u << 8) | (2u << 10) | (0u << 12) | (2u << 14);
constexpr unsigned ROW_OZ = 1u | (1u << 2) | (0u << 4) | (2u << 6) | (0u << 8) | (0u << 10) | (2u << 12) | (2u << 14);
__device__ __forceinline__ int row_oy(int k) { return (int)((ROW_OY >> (2 * k)) & 3u) - 1; }
__device__ __forceinline__ int row_oz(int k) { return (int)((ROW_OZ >> (2 * k)) & 3u) - 1; }

// distance (lower bound) from the query to the nearest face of the cell box
// [x0,x1]x[y0,y1]x[z0,z1] that is interior to the grid (+inf if the box covers the grid)
template <int D>
__device__ __forceinline__ float box_bound(const View &v, float qx, float qy, float qz, int x0,
                                           int x1, int y0, int y1, int z0, int z1)
{
    float bound = CUDART_INF_F;
    if (x0 >= 1) bound = fminf(bound, gap_lb(v, __fsub_rn(qx, face_at(v.lo0, x0, v.h)), v.slk0));
    if (x1 < v.G0 - 1) bound = fminf(bound, gap_lb(v, __fsub_rn(face_at(v.lo0, x1 + 1, v.h), qx), v.slk0));
    if (y0 >= 1) bound = fminf(bound, gap_lb(v, __fsub_rn(qy, face_at(v.lo1, y0, v.h)), v.slk1));
    if (y1 < v.G1 - 1) bound = fminf(bound, gap_lb(v, __fsub_rn(face_at(v.lo1, y1 + 1, v.h), qy), v.slk1));
    if (D == 3) {
        if (z0 >= 1) bound = fminf(bound, gap_lb(v, __fsub_rn(qz, face_at(v.lo2, z0, v.h)), v.slk2));
        if (z1 < v.G2 - 1) bound = fminf(bound, gap_lb(v, __fsub_rn(face_at(v.lo2, z1 + 1, v.h), qz), v.slk2));
    }
    return bound;
}
__device__ __forceinline__ bool bound_ok(float bound, float s2)
{
    if (bound == CUDART_INF_F) return true;               // nothing left outside the scanned box
    return bound > 0.0f && s2 < __fmul_rn(bound, bound);
}

// ---- second level: a subdivided cell ------------------------------------------------------------
// Sub-cell boundary a (0..S) of cell k on an axis, in x-space: lo + (k S + a)(h / S).  The records
// filed in sub-cells >= a have cell coordinate t >= k + (a/S)(1 - u) (one more rounding than the
// level-0 filing: fl(fl(t - k) S), where t - k is exact), i.e. x >= lo + (k + a/S) h - 4.02 u G h;
// the computed boundary is off by <= u(|lo| + 4 G h) (hs = h/S, the product and the sum are rounded,
// k S + a < 2^27 is converted with relative error u).  Together <= u(|lo| + 8.1 G h), inside the
// slack slk = 16 u (|lo| + G h) that gap_lb() already subtracts for the level-0 faces, so the same
// gap_lb() gives a valid lower bound of the real axis distance behind a sub-cell boundary.
struct SubAx {
    float lo, q, slk;
    int base;                                  // k * S
    int u;                                     // sub-cell of the query's projection into the cell
};
__device__ __forceinline__ float sub_face(const SubAx &a, int idx, float hs)
{
    return __fadd_rn(a.lo, __fmul_rn((float)(a.base + idx), hs));
}
// squared lower bound of the axis distance from the query to every record in sub-cells < idx
__device__ __forceinline__ float sub_low2(const View &v, const SubAx &a, int idx, float hs)
{
    const float t = gap_lb(v, __fsub_rn(a.q, sub_face(a, idx, hs)), a.slk);
    return __fmul_rn(t, t);
}
// ... to every record in sub-cells >= idx
__device__ __forceinline__ float sub_high2(const View &v, const SubAx &a, int idx, float hs)
{
    const float t = gap_lb(v, __fsub_rn(sub_face(a, idx, hs), a.q), a.slk);
    return __fmul_rn(t, t);
}
__device__ __forceinline__ float sub_gap2(const View &v, const SubAx &a, int idx, float hs)
{
    return idx == a.u ? 0.0f : (idx < a.u ? sub_low2(v, a, idx + 1, hs) : sub_high2(v, a, idx, hs));
}
// Exact visit of a subdivided level-0 cell (cid = linear id, (kx, ky, kz) its coordinates, cend the
// end of its record range).  The query may lie inside the cell or in a neighbour.  While nothing
// bounds the search yet (s2 = +inf) the 3^d sub-block around the query's projection is scanned; if
// that still leaves s2 = +inf the whole cell is.  Then every sub-row that the ball of radius
// sqrt(s2) around the query can reach is scanned over the x-range it can reach, each test strict
// and against the current s2 (which only shrinks), skipping what the first step covered.
template <int D>
__device__ __noinline__ Top2 visit_heavy(const View &v, int cid, int kx, int ky, int kz, int cend,
                                         float qx, float qy, float qz, int self, Top2 best)
{
    const int2 si = v.subinfo[cid];
    const int S = si.x;
    const int32_t *__restrict__ ss = v.leaf_start + si.y;
    const float fS = (float)S;
    const float hs = __fdiv_rn(v.h, fS);
    SubAx ax, ay, az;
    ax.lo = v.lo0; ax.q = qx; ax.slk = v.slk0; ax.base = kx * S; ax.u = sub_axis(qx, v.lo0, v.inv_h, kx, fS, S);
    ay.lo = v.lo1; ay.q = qy; ay.slk = v.slk1; ay.base = ky * S; ay.u = sub_axis(qy, v.lo1, v.inv_h, ky, fS, S);
    az.lo = v.lo2; az.q = qz; az.slk = v.slk2; az.base = kz * S; az.u = D == 3 ? sub_axis(qz, v.lo2, v.inv_h, kz, fS, S) : 0;
    int px0 = 0, px1 = -1, py0 = 0, py1 = -1, pz0 = 0, pz1 = -1;      // block already scanned (empty)
    // No bound yet, or a poor one (worse than two sub-cell widths: a sparse point beside a dense cell):
    // the sub-cells nearest to the query first, so that the sweep below prunes against a bound of the
    // cell's own scale instead of scanning a third of it at the latency of one thread.
    if (!(best.s2 < __fmul_rn(4.0f, __fmul_rn(hs, hs)))) {
        px0 = max(ax.u - 1, 0); px1 = min(ax.u + 1, S - 1);
        py0 = max(ay.u - 1, 0); py1 = min(ay.u + 1, S - 1);
        pz0 = D == 3 ? max(az.u - 1, 0) : 0; pz1 = D == 3 ? min(az.u + 1, S - 1) : 0;
        for (int z = pz0; z <= pz1; ++z)
            for (int y = py0; y <= py1; ++y) {
                const int row = (z * S + y) * S;
                scan_range<D>(v, ss[row + px0], ss[row + px1 + 1], qx, qy, qz, self, best);
            }
        if (best.s2 == CUDART_INF_F) {
            scan_range<D>(v, ss[0], cend, qx, qy, qz, self, best);
            return best;
        }
    }
    int z0 = 0, z1 = 0;
    if (D == 3) {
        z0 = az.u; z1 = az.u;
        while (z0 > 0 && !(best.s2 < sub_low2(v, az, z0, hs))) --z0;
        while (z1 < S - 1 && !(best.s2 < sub_high2(v, az, z1 + 1, hs))) ++z1;
    }
    for (int z = z0; z <= z1; ++z) {
        const float gz2 = D == 3 ? sub_gap2(v, az, z, hs) : 0.0f;
        if (best.s2 < gz2) continue;
        int y0 = ay.u, y1 = ay.u;
        while (y0 > 0 && !(best.s2 < __fadd_rn(gz2, sub_low2(v, ay, y0, hs)))) --y0;
        while (y1 < S - 1 && !(best.s2 < __fadd_rn(gz2, sub_high2(v, ay, y1 + 1, hs)))) ++y1;
        for (int y = y0; y <= y1; ++y) {
            const float rb2 = __fadd_rn(gz2, sub_gap2(v, ay, y, hs));
            if (best.s2 < rb2) continue;
            int x0 = ax.u, x1 = ax.u;
            while (x0 > 0 && !(best.s2 < __fadd_rn(rb2, sub_low2(v, ax, x0, hs)))) --x0;
            while (x1 < S - 1 && !(best.s2 < __fadd_rn(rb2, sub_high2(v, ax, x1 + 1, hs)))) ++x1;
            const int row = (z * S + y) * S;
            if (y >= py0 && y <= py1 && z >= pz0 && z <= pz1) {
                if (x0 < px0) scan_range<D>(v, ss[row + x0], ss[row + px0], qx, qy, qz, self, best);
                if (x1 > px1) scan_range<D>(v, ss[row + px1 + 1], ss[row + x1 + 1], qx, qy, qz, self, best);
            } else {
                scan_range<D>(v, ss[row + x0], ss[row + x1 + 1], qx, qy, qz, self, best);
            }
        }
    }
    return best;
}
// One level-0 cell: its whole record range [b, e), or its sub-cells when it is subdivided.
template <int D>
__device__ __forceinline__ void visit_cell(const View &v, int cid, int kx, int ky, int kz, int b, int e,
                                           float qx, float qy, float qz, int self, Top2 &best)
{
    if (e - b < v.heavy_T) scan_range<D>(v, b, e, qx, qy, qz, self, best);
    else best = visit_heavy<D>(v, cid, kx, ky, kz, e, qx, qy, qz, self, best);
}
// Cells x0..x1 of one grid row (rowbase = linear id of its first cell).
template <int D>
__device__ __forceinline__ void visit_row(const View &v, bool chains, int rowbase, int ky, int kz, int x0, int x1,
                                          float qx, float qy, float qz, int self, Top2 &best)
{
    const int32_t *cs = v.cell_start + rowbase;
    const int b = cs[x0], e = cs[x1 + 1];
    if (e - b < v.heavy_T) {                        // no subdivided cell among them
        scan_range<D>(v, b, e, qx, qy, qz, self, best);
    } else {
        int lo = b;
        for (int x = x0; x <= x1; ++x) {
            const int hi = x == x1 ? e : cs[x + 1];
            if (hi > lo) visit_cell<D>(v, rowbase + x, x, ky, kz, lo, hi, qx, qy, qz, self, best);
            lo = hi;
        }
    }
    if (chains)
        for (int x = x0; x <= x1; ++x) scan_chain<D>(v, rowbase + x, qx, qy, qz, self, best);
}

// Squared lower bound (R7's face bound: slack, shrink) of the axis distance from the query coordinate q in
// cell c to anything filed in cell k of that axis.
__device__ __forceinline__ float axis_gap2(const View &v, float q, float lo, float slk, int k, int c)
{
    if (k == c) return 0.0f;
    const float g = k > c ? __fsub_rn(face_at(lo, k, v.h), q) : __fsub_rn(q, face_at(lo, k + 1, v.h));
    const float t = gap_lb(v, g, slk);
    return __fmul_rn(t, t);
}
// Cells xa..xb of one row of a ring.  A sparse row (the usual case: rings are for isolated queries) is one
// range; a row that holds many records -- the ring of a sparse point beside a dense cluster contains the
// cluster's core -- goes cell by cell, each tested against the current bound (rowgap2 = squared lower bound
// of the row's distance in y and z), subdivided cells through visit_heavy.
constexpr int RING_ROW_DENSE = 64;
template <int D, bool PRUNE>
__device__ __forceinline__ void ring_cells(const View &v, bool chains, int rowbase, int y, int z, int xa, int xb,
                                           float rowgap2, float qx, float qy, float qz, int self, int cx, Top2 &best)
{
    const int32_t *cs = v.cell_start + rowbase;
    const int b = cs[xa], e = cs[xb + 1];
    if (!PRUNE || e - b <= RING_ROW_DENSE) {
        scan_range<D>(v, b, e, qx, qy, qz, self, best);
    } else {
        for (int x = xa; x <= xb; ++x) {
            if (best.s2 < __fadd_rn(rowgap2, axis_gap2(v, qx, v.lo0, v.slk0, x, cx))) continue;
            const int cb = cs[x], ce = cs[x + 1];
            if (ce > cb) visit_cell<D>(v, rowbase + x, x, y, z, cb, ce, qx, qy, qz, self, best);
        }
    }
    if (chains)
        for (int x = xa; x <= xb; ++x) scan_chain<D>(v, rowbase + x, qx, qy, qz, self, best);
}

// Chebyshev rings r = 2, 3, ... around the query's own cell, entered with the radius-1 block
// already done; leaves as soon as the bound of the scanned block allows it.  (Rare path: kept out
// of line, state passed by value.)
struct RingOut { Top2 best; int r; };
template <int D, bool PRUNE>
__device__ __noinline__ RingOut ring_continue(const View &v, bool chains, float qx, float qy, float qz,
                                              int self, int cx, int cy, int cz, Top2 best, bool warp_wide)
{
    int r = 1;
    for (;;) {
        int z0 = D == 3 ? max(cz - r, 0) : 0, z1 = D == 3 ? min(cz + r, v.G2 - 1) : 0;
        int y0 = max(cy - r, 0), y1 = min(cy + r, v.G1 - 1);
        int x0 = max(cx - r, 0), x1 = min(cx + r, v.G0 - 1);
        if (bound_ok(box_bound<D>(v, qx, qy, qz, x0, x1, y0, y1, z0, z1), best.s2)) break;
        if (v.handoff && r == (D == 3 ? HANDOFF_R3 : HANDOFF_R2)) {
            // an isolated query: the brute-force pass behind this kernel finishes it (the certificate
            // the caller stores now is overwritten there).  warp_wide: all 32 lanes are here with the
            // same query (the list kernel), lane 0 speaks for them.
            const bool speaker = !warp_wide || (threadIdx.x & 31) == 0;
            int idx = HANDOFF_CAP;
            if (speaker) idx = atomicAdd(v.n_handoff, 1);
            if (warp_wide) idx = __shfl_sync(0xffffffffu, idx, 0);
            if (idx < HANDOFF_CAP) {                   // (a full list leaves the query to the rings)
                if (speaker) v.handoff[idx] = make_float4(qx, qy, qz, __int_as_float(self));
                ++r;
                break;
            }
        }
        ++r;
        // ring r: shell rows get the full segment, inner rows only the two end cells
        z0 = D == 3 ? max(cz - r, 0) : 0; z1 = D == 3 ? min(cz + r, v.G2 - 1) : 0;
        y0 = max(cy - r, 0); y1 = min(cy + r, v.G1 - 1);
        x0 = max(cx - r, 0); x1 = min(cx + r, v.G0 - 1);
        // PRUNE (the list kernels of A7): rows and, in rows that hold many records, cells are tested against
        // the current bound -- the ring of a sparse query beside a dense cluster contains the cluster's core.
        // The whole-set kernels keep the plain form: their ring queries hide behind the other warps, and the
        // longer code measured 13 % on the whole kernel (register allocation of the caller).
        for (int z = z0; z <= z1; ++z) {
            const float gz = PRUNE && D == 3 ? axis_gap2(v, qz, v.lo2, v.slk2, z, cz) : 0.0f;
            if (PRUNE && best.s2 < gz) continue;                 // (strict: nothing behind that face can enter)
            for (int y = y0; y <= y1; ++y) {
                const float gy = PRUNE ? __fadd_rn(gz, axis_gap2(v, qy, v.lo1, v.slk1, y, cy)) : 0.0f;
                if (PRUNE && best.s2 < gy) continue;
                int rowbase = (z * v.G1 + y) * v.G0;
                bool shell = (D == 3 && (z == cz - r || z == cz + r)) || y == cy - r || y == cy + r;
                if (shell) {
                    ring_cells<D, PRUNE>(v, chains, rowbase, y, z, x0, x1, gy, qx, qy, qz, self, cx, best);
                } else {
                    if (cx - r >= 0) ring_cells<D, PRUNE>(v, chains, rowbase, y, z, cx - r, cx - r, gy, qx, qy, qz, self, cx, best);
                    if (cx + r <= v.G0 - 1) ring_cells<D, PRUNE>(v, chains, rowbase, y, z, cx + r, cx + r, gy, qx, qy, qz, self, cx, best);
                }
            }
        }
    }
    RingOut o;
    o.best = best; o.r = r;
    return o;
}
// final check of the radius-1 block, then wider rings if the bound requires them
template <int D, bool PRUNE = false>
__device__ __forceinline__ int finish_block(const View &v, bool chains, float qx, float qy, float qz, int self,
                                            int cx, int cy, int cz, Top2 &best, bool warp_wide = false)
{
    const int z0 = D == 3 ? max(cz - 1, 0) : 0, z1 = D == 3 ? min(cz + 1, v.G2 - 1) : 0;
    const int y0 = max(cy - 1, 0), y1 = min(cy + 1, v.G1 - 1);
    const int x0 = max(cx - 1, 0), x1 = min(cx + 1, v.G0 - 1);
    if (bound_ok(box_bound<D>(v, qx, qy, qz, x0, x1, y0, y1, z0, z1), best.s2)) return 1;
    const RingOut o = ring_continue<D, PRUNE>(v, chains, qx, qy, qz, self, cx, cy, cz, best, warp_wide);
    best = o.best;
    return o.r;
}

// One thread per query, straight from global memory (A7, and A3's comparison variant): own
// cell, row neighbours, other rows nearest first, every cell subject to pruning; then rings.
template <int D, bool PRUNE = false>
__device__ int block_search(const View &v, bool chains, float qx, float qy, float qz, int self,
                            int cx, int cy, int cz, Top2 &best)
{
    const Gaps g = make_gaps<D>(v, qx, qy, qz, cx, cy, cz);
    const int rb0 = (cz * v.G1 + cy) * v.G0;
    {
        const int32_t *cs = v.cell_start + rb0 + cx;
        const int s0 = cs[0], s1 = cs[1];
        visit_cell<D>(v, rb0 + cx, cx, cy, cz, s0, s1, qx, qy, qz, self, best);
        if (chains) scan_chain<D>(v, rb0 + cx, qx, qy, qz, self, best);
        if (cx > 0 && !(best.s2 < g.xm)) {
            visit_cell<D>(v, rb0 + cx - 1, cx - 1, cy, cz, cs[-1], s0, qx, qy, qz, self, best);
            if (chains) scan_chain<D>(v, rb0 + cx - 1, qx, qy, qz, self, best);
        }
        if (cx < v.G0 - 1 && !(best.s2 < g.xp)) {
            visit_cell<D>(v, rb0 + cx + 1, cx + 1, cy, cz, s1, cs[2], qx, qy, qz, self, best);
            if (chains) scan_chain<D>(v, rb0 + cx + 1, qx, qy, qz, self, best);
        }
    }
#pragma unroll 1
    for (int k = 0; k < (D == 3 ? 8 : 2); ++k) {
        const int oy = row_oy(k), oz = row_oz(k);
        const int y = cy + oy, z = cz + oz;
        if (y < 0 || y >= v.G1 || z < 0 || z >= v.G2) continue;
        const float rb2 = __fadd_rn(oy < 0 ? g.ym : (oy > 0 ? g.yp : 0.f), oz < 0 ? g.zm : (oz > 0 ? g.zp : 0.f));
        if (best.s2 < rb2) continue;
        int x0 = cx, x1 = cx;
        if (cx > 0 && !(best.s2 < __fadd_rn(rb2, g.xm))) x0 = cx - 1;
        if (cx < v.G0 - 1 && !(best.s2 < __fadd_rn(rb2, g.xp))) x1 = cx + 1;
        visit_row<D>(v, chains, (z * v.G1 + y) * v.G0, y, z, x0, x1, qx, qy, qz, self, best);
    }
    return finish_block<D, PRUNE>(v, chains, qx, qy, qz, self, cx, cy, cz, best);
}

// ---- A3 / A7, phased -------------------------------------------------------------------------
// One thread per query.  The search of a query is a handful of short record ranges; what costs is
// not the arithmetic but the control flow around them, which differs from lane to lane.  So every
// lane first QUEUES the ranges it needs (own row or, in a subdivided cell, the 3^d sub-block; after
// that, with a finite second-best, every cell / sub-row it cannot rule out) in a small
// shared-memory list, and the warp then scans all lists in ONE loop, four records per lane and
// step: the distance arithmetic and the loads, three quarters of the instructions, run with the
// lanes in step, only the range bookkeeping diverges.  Pruning is decided when a range is queued,
// against the second-best of the moment: an upper bound of the final one, so every test stays a
// valid strict lower-bound test (see gap_lb above).
constexpr int PS_THREADS = 128;
#ifndef RL_STEP8
#define RL_STEP8 1
#endif
constexpr int RL_CAP = 16;                       // ranges a lane can queue between two scans

struct Qry { float x, y, z; int self; };
// A lane's queue is bounded in entries (RL_CAP) and in records (RL_BUDGET): a query whose ball holds more
// than that -- a sparse point next to a dense cluster, with the poor bound its own cell gave it -- would scan
// it all at the latency of one thread, against a bound that no longer shrinks what was queued.  Such a lane
// drops its queue (big) and runs the ring search instead, which prunes cell by cell and sub-row by sub-row
// against the current bound.
constexpr int RL_BUDGET = 768;
struct Lane { int2 *rl; int cnt; int tot; int last_e; bool big; };   // entry i of this thread's list: rl[i * PS_THREADS]
__device__ __forceinline__ void lane_reset(Lane &L) { L.cnt = 0; L.tot = 0; L.last_e = -1; L.big = false; }

template <int D>
__device__ __forceinline__ void rl_push(const View &v, Lane &L, int b, int e, const Qry &q, Top2 &best)
{
    if (b >= e || L.big) return;
    L.tot += e - b;
    if (L.cnt > 0 && b == L.last_e) {            // continues the previous range (full sub-rows of one cell)
        L.rl[(L.cnt - 1) * PS_THREADS].y = e;
        L.last_e = e;
        if (L.tot > RL_BUDGET) { L.big = true; L.cnt = 0; }
        return;
    }
    if (L.cnt == RL_CAP || L.tot > RL_BUDGET) {
        L.big = true;
        L.cnt = 0;
        return;
    }
    L.rl[L.cnt * PS_THREADS] = make_int2(b, e);
    L.last_e = e;
    ++L.cnt;
}
// All 32 lanes of the warp call this; a lane without ranges just waits for the others.  d = 3 records
// are one float4 each, so a range is entered at its first record; d = 2 records are read two per
// float4, so a range is entered at the even slot at or below its first record.  Records behind the
// end of a range (up to 3) are other cells' records or the NaN padding: candidates or inert.
template <int D>
__device__ __forceinline__ void rl_scan(const View &v, Lane &L, const Qry &q, Top2 &best)
{
    int idx = 0, t = 0, e = 0;
    for (;;) {
        if (t >= e && idx < L.cnt) {
            const int2 r = L.rl[idx * PS_THREADS];
            ++idx;
            t = D == 2 ? (r.x & ~1) : r.x;
            e = r.y;
        }
        const bool work = t < e;
        if (!__any_sync(0xffffffffu, work)) break;
        if (work) {
            float s0, s1, s2, s3;
            if (D == 2) {
                const float4 A = *reinterpret_cast<const float4 *>(v.spos2 + t);
                const float4 B = *reinterpret_cast<const float4 *>(v.spos2 + t + 2);
                s0 = sqd2(q.x, q.y, A.x, A.y); s1 = sqd2(q.x, q.y, A.z, A.w);
                s2 = sqd2(q.x, q.y, B.x, B.y); s3 = sqd2(q.x, q.y, B.z, B.w);
            } else if (RL_STEP8 && t + 4 < e) {
                // eight records per round trip (a queue is scanned at the latency of its loads)
                const float4 c0 = v.spos4[t], c1 = v.spos4[t + 1], c2 = v.spos4[t + 2], c3 = v.spos4[t + 3];
                const float4 c4 = v.spos4[t + 4], c5 = v.spos4[t + 5], c6 = v.spos4[t + 6], c7 = v.spos4[t + 7];
                s0 = sqd3(q.x, q.y, q.z, c0.x, c0.y, c0.z); s1 = sqd3(q.x, q.y, q.z, c1.x, c1.y, c1.z);
                s2 = sqd3(q.x, q.y, q.z, c2.x, c2.y, c2.z); s3 = sqd3(q.x, q.y, q.z, c3.x, c3.y, c3.z);
                const float m0 = fminf(fminf(s0, s1), fminf(s2, s3));
                if (m0 <= best.s2) best = slow_offer4<D>(v, best, t, s0, s1, s2, s3, q.self);
                t += 4;
                s0 = sqd3(q.x, q.y, q.z, c4.x, c4.y, c4.z); s1 = sqd3(q.x, q.y, q.z, c5.x, c5.y, c5.z);
                s2 = sqd3(q.x, q.y, q.z, c6.x, c6.y, c6.z); s3 = sqd3(q.x, q.y, q.z, c7.x, c7.y, c7.z);
            } else {
                const float4 c0 = v.spos4[t], c1 = v.spos4[t + 1], c2 = v.spos4[t + 2], c3 = v.spos4[t + 3];
                s0 = sqd3(q.x, q.y, q.z, c0.x, c0.y, c0.z); s1 = sqd3(q.x, q.y, q.z, c1.x, c1.y, c1.z);
                s2 = sqd3(q.x, q.y, q.z, c2.x, c2.y, c2.z); s3 = sqd3(q.x, q.y, q.z, c3.x, c3.y, c3.z);
            }
            const float m = fminf(fminf(s0, s1), fminf(s2, s3));
            if (m <= best.s2) best = slow_offer4<D>(v, best, t, s0, s1, s2, s3, q.self);
            t += 4;
        }
    }
    L.cnt = 0; L.tot = 0; L.last_e = -1;
}

// ---- A3, warp-tiled: the whole-set search of a freshly built grid --------------------------
// A warp owns 32 consecutive sorted slots.  Slots are cell-sorted, so the lanes of one grid row
// form a contiguous lane segment, and what they need from any row of the 3^d block is ONE
// contiguous record range [B, E) of the sorted array (cells xf-1 .. xl+1 of that row).
//  * sparse row (E - B < dense_thr records): the warp loads the range into its shared-memory tile
//    with coalesced loads (one global round trip instead of one per candidate) and every lane
//    scans its own 3-cell sub-range [b, e) from shared memory, 4 records per step;
//  * dense row (a few cells under 32 lanes, occupancy >> 1, d2 << h): cell pruning pays.  In the
//    lanes' own row the own cell is scanned first, then only the row neighbours a lane cannot
//    rule out; in the other rows only the cells it cannot rule out.  What is left after pruning
//    is long ranges for a few lanes; a tile pass would cost as much as if all 32 lanes needed
//    them, so such a pass is served cooperatively instead: for each lane that still has a range,
//    all 32 lanes take different records of it (coalesced, straight from global memory) and the
//    two best are extracted with warp reductions.
// Lanes whose radius-1 block does not satisfy the bound continue with the ring loop (rare).
constexpr int WT_TILE = 128;   // records per warp tile

template <int D>
__device__ __forceinline__ void tile_scan(const float2 *tp2, const float4 *tp4, const int *tidx, int lb,
                                          int le, float qx, float qy, float qz, int self, Top2 &best)
{
    for (int t = lb; t < le; t += 4) {
        float s0, s1, s2, s3;
        int j0, j1, j2, j3;
        if (D == 2) {
            const float2 c0 = tp2[t], c1 = tp2[t + 1], c2 = tp2[t + 2], c3 = tp2[t + 3];
            s0 = sqd2(qx, qy, c0.x, c0.y); s1 = sqd2(qx, qy, c1.x, c1.y);
            s2 = sqd2(qx, qy, c2.x, c2.y); s3 = sqd2(qx, qy, c3.x, c3.y);
        } else {
            const float4 c0 = tp4[t], c1 = tp4[t + 1], c2 = tp4[t + 2], c3 = tp4[t + 3];
            s0 = sqd3(qx, qy, qz, c0.x, c0.y, c0.z); s1 = sqd3(qx, qy, qz, c1.x, c1.y, c1.z);
            s2 = sqd3(qx, qy, qz, c2.x, c2.y, c2.z); s3 = sqd3(qx, qy, qz, c3.x, c3.y, c3.z);
            j0 = __float_as_int(c0.w); j1 = __float_as_int(c1.w);
            j2 = __float_as_int(c2.w); j3 = __float_as_int(c3.w);
        }
        float m = fminf(fminf(s0, s1), fminf(s2, s3));
        if (m <= best.s2) {
            if (D == 2) { j0 = tidx[t]; j1 = tidx[t + 1]; j2 = tidx[t + 2]; j3 = tidx[t + 3]; }
            // Usually one of the four qualifies: offer the smallest, retire it (NaN: fminf skips it),
            // and look again.  Every lane on this path runs the same instructions whichever of its four
            // candidates it is about; the top-2 does not depend on the order of the offers.
            do {
                const bool p0 = s0 == m, p1 = !p0 && s1 == m, p2 = !p0 && !p1 && s2 == m;
                const int jm = p0 ? j0 : (p1 ? j1 : (p2 ? j2 : j3));
                const float qn = __int_as_float(0x7fc00000);
                s0 = p0 ? qn : s0; s1 = p1 ? qn : s1; s2 = p2 ? qn : s2; s3 = (p0 || p1 || p2) ? s3 : qn;
                offer_once(best, m, jm, self);
                m = fminf(fminf(s0, s1), fminf(s2, s3));
            } while (m <= best.s2);
        }
    }
}

// Tile pass: records [B, E) (warp-uniform) go through the warp's tile, every lane scans its own
// (up to two) ranges [b1,e1), [b2,e2) (empty when b >= e).  Called by all 32 lanes.
template <int D>
__device__ __forceinline__ void tile_pass(const View &v, int N, int lane, float2 *tp2, float4 *tp4, int *tix,
                                          int B, int E, int b1, int e1, int b2, int e2, float qx, float qy,
                                          float qz, int self, Top2 &best)
{
    const float qnan = __int_as_float(0x7fc00000);
    for (int T0 = B; T0 < E; T0 += WT_TILE) {
        const int T1 = T0 + WT_TILE;
        const int lb1 = max(b1, T0), le1 = min(e1, T1), lb2 = max(b2, T0), le2 = min(e2, T1);
        if (E - B > WT_TILE && !__any_sync(0xffffffffu, lb1 < le1 || lb2 < le2)) continue;
        const int need = min(WT_TILE, E - T0 + 3);               // records of this tile anyone can touch
#pragma unroll
        for (int k = lane; k < WT_TILE; k += 32) {
            const int g = T0 + k;
            if (k < need) {
                if (D == 3) {
                    tp4[k] = g < N ? v.spos4[g] : make_float4(qnan, qnan, qnan, __int_as_float(-1));
                } else {
                    tp2[k] = g < N ? v.spos2[g] : make_float2(qnan, qnan);
                    tix[k] = g < N ? v.sidx[g] : -1;
                }
            }
        }
        __syncwarp();
        if (lb1 < le1) tile_scan<D>(tp2, tp4, tix, lb1 - T0, le1 - T0, qx, qy, qz, self, best);
        if (lb2 < le2) tile_scan<D>(tp2, tp4, tix, lb2 - T0, le2 - T0, qx, qy, qz, self, best);
        __syncwarp();
    }
}

// Warp-cooperative scan of one lane's range: all 32 lanes take different records of [b, e) for the
// query of lane L (coalesced loads straight from global memory) and keep their own partial top-2.
template <int D>
__device__ __forceinline__ void coop_range(const View &v, int lane, int b, int e, float qx, float qy,
                                           float qz, int self, float thr, int h1, int h2, Top2 &tmp)
{
    for (int t = b + lane; t < e; t += 32) {
        float s;
        int j;
        if (D == 2) {
            const float2 c = v.spos2[t];
            j = v.sidx[t];                         // issued with the position: one round trip
            s = sqd2(qx, qy, c.x, c.y);
        } else {
            const float4 c = v.spos4[t];
            s = sqd3(qx, qy, qz, c.x, c.y, c.z);
            j = __float_as_int(c.w);
        }
        if (s <= thr && j >= 0 && j != self && j != h1 && j != h2) tmp.offer(s, j);
    }
}
// store_cert with the L2 evict_last policy.  The certificates of a slot-ordered sweep go to ids
// all over the five output arrays, four bytes at a time: a 32-byte sector of an output array is
// completed by eight writes spread over the whole kernel, and a sector that L2 evicts half-written
// costs a fill and a second write-back (ncu, 4,194,304 points: 723 MB written for 84 MB of output).
// The outputs (84 MB) fit the 126 MB L2 if the streamed grid data does not push them out.
__device__ __forceinline__ void st_keep(void *p, unsigned v, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.b32 [%0], %1, %2;" ::"l"(p), "r"(v), "l"(pol) : "memory");
}
__device__ __forceinline__ void store_cert_keep(const Top2 &t, int i, int32_t *nn, int32_t *nn2, float *d1,
                                                float *d2, float *c)
{
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    const float a = __fsqrt_rn(t.s1), b = __fsqrt_rn(t.s2);
    st_keep(nn + i, (unsigned)(t.j1 == KC_NOIDX ? -1 : t.j1), pol);
    if (nn2) st_keep(nn2 + i, (unsigned)(t.j2 == KC_NOIDX ? -1 : t.j2), pol);
    st_keep(d1 + i, __float_as_uint(a), pol);
    st_keep(d2 + i, __float_as_uint(b), pol);
    st_keep(c + i, __float_as_uint(__fsub_rn(b, a)), pol);
}

// ---- d = 2: the row-segment kernel with cell-wise pruning of dense rows -------------------------
// In the plane the leaf-tiled kernel below loses to this older one on clustered data (config 5,
// d = 2: 0.75 vs 0.68 ms): cells of 10-70 records are too small for a second level, and what pays
// there is pruning cell by cell plus the warp-cooperative scan of the few long ranges that survive
// it.  A warp owns 32 consecutive sorted slots; the lanes of one grid row form a segment whose 3-cell
// windows are one contiguous range per row: sparse rows go through the tile whole, dense rows
// (>= WT_DENSE records) own cell first, then only the cells a lane cannot rule out.  The second level
// of the index is ignored (level-0 ranges are contiguous whatever the order inside a cell).
constexpr int WT_WARPS = 4;
constexpr int SW_WORDS = 8;                        // sweep: a warp owns up to 32 * SW_WORDS consecutive slots
// Slots per sweep warp, in units of 32: as many as hold about one warp of marked slots (measured on
// config 5: a second round per warp costs more than idle lanes, so the count aims below 32).
__device__ __forceinline__ int sweep_words(int N, int nF)
{
    return (int)min((int64_t)SW_WORDS, max((int64_t)1, (int64_t)N * 9 / ((int64_t)max(nF, 1) * 10)));
}
constexpr int WT_DENSE = 128;

// Dense pass: every lane brings up to two ranges left after pruning.  Served lane by lane by the
// whole warp when that is cheaper than a tile pass over the hull [B, E) (issue-slot estimates:
// tile pass ~11 per record of the longest lane, cooperative ~45 per served lane + 12 per 32
// records).  Called by all 32 lanes.
template <int D>
__device__ __forceinline__ void dense_pass(const View &v, int N, int lane, float2 *tp2, float4 *tp4, int *tix,
                                           int b1, int e1, int b2, int e2, float qx, float qy, float qz,
                                           int self, Top2 &best)
{
    const bool h1 = b1 < e1, h2 = b2 < e2;
    const int len = (h1 ? e1 - b1 : 0) + (h2 ? e2 - b2 : 0);
    const unsigned active = __ballot_sync(0xffffffffu, len > 0);
    if (!active) return;
    const int maxlen = __reduce_max_sync(0xffffffffu, len);
    const int sumlen = __reduce_add_sync(0xffffffffu, len);
    if (__popc(active) * 360 + sumlen * 3 < maxlen * 88) {
        for (unsigned a = active; a; a &= a - 1) {
            const int L = __ffs(a) - 1;
            const float Lx = __shfl_sync(0xffffffffu, qx, L), Ly = __shfl_sync(0xffffffffu, qy, L);
            const float Lz = D == 3 ? __shfl_sync(0xffffffffu, qz, L) : 0.f;
            const int Lself = __shfl_sync(0xffffffffu, self, L);
            const float thr = __shfl_sync(0xffffffffu, best.s2, L);
            const int Lj1 = __shfl_sync(0xffffffffu, best.j1, L), Lj2 = __shfl_sync(0xffffffffu, best.j2, L);
            const int Lb1 = __shfl_sync(0xffffffffu, b1, L), Le1 = __shfl_sync(0xffffffffu, e1, L);
            const int Lb2 = __shfl_sync(0xffffffffu, b2, L), Le2 = __shfl_sync(0xffffffffu, e2, L);
            Top2 tmp;
            tmp.init();
            coop_range<D>(v, lane, Lb1, Le1, Lx, Ly, Lz, Lself, thr, Lj1, Lj2, tmp);
            coop_range<D>(v, lane, Lb2, Le2, Lx, Ly, Lz, Lself, thr, Lj1, Lj2, tmp);
            float sa, sb;
            int ja, jb;
            warp_pop(tmp, sa, ja);
            warp_pop(tmp, sb, jb);
            if (lane == L) {
                if (ja != KC_NOIDX) best.offer(sa, ja);
                if (jb != KC_NOIDX) best.offer(sb, jb);
            }
        }
        return;
    }
    const int B = __reduce_min_sync(0xffffffffu, min(h1 ? b1 : 0x7fffffff, h2 ? b2 : 0x7fffffff));
    const int E = __reduce_max_sync(0xffffffffu, max(h1 ? e1 : 0, h2 ? e2 : 0));
    tile_pass<D>(v, N, lane, tp2, tp4, tix, B, E, b1, e1, b2, e2, qx, qy, qz, self, best);
}

// SWEEP = false: A3, every slot of a freshly built grid is a query.
// SWEEP = true:  A7 for a large frontier: the same slot-ordered sweep over the incrementally
//   updated grid, but only the slots marked with this call's epoch are queries (their lanes stay
//   idle otherwise; warps without a marked slot leave at once), tombstones are inert records and
//   the overflow chains of every visited cell are scanned too.  Runs only when *nF * sweep_div >= N
//   (the list kernel serves smaller frontiers and the frontier points that live in chains).
template <int D, bool SWEEP, bool FRESH>
__global__ void __launch_bounds__(32 * WT_WARPS)
search_tiled_kernel(View v, int N, Counters *ctr, int32_t *mark,
                    const int32_t *__restrict__ nF, int sweep_div, int32_t *nn, int32_t *nn2, float *d1,
                    float *d2, float *c)
{
    __shared__ __align__(16) float4 s_p4[D == 3 ? WT_WARPS : 1][D == 3 ? WT_TILE + 4 : 1];
    __shared__ __align__(16) float2 s_p2[D == 2 ? WT_WARPS : 1][D == 2 ? WT_TILE + 4 : 1];
    __shared__ int s_ix[D == 2 ? WT_WARPS : 1][D == 2 ? WT_TILE + 4 : 1];
    if (SWEEP && (int64_t)*nF * sweep_div < N) return;
    const bool chains = SWEEP && !FRESH && ctr->n_misfiled > 0;   // FRESH: no incremental update since the build
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const float qnan = __int_as_float(0x7fc00000);
    float4 *tp4 = s_p4[D == 3 ? warp : 0];
    float2 *tp2 = s_p2[D == 2 ? warp : 0];
    int *tix = s_ix[D == 2 ? warp : 0];
    // the whole tile starts inert: a short range leaves records behind it untouched
    for (int k = lane; k < WT_TILE + 4; k += 32) {
        if (D == 3) tp4[k] = make_float4(qnan, qnan, qnan, __int_as_float(-1));
        else { tp2[k] = make_float2(qnan, qnan); tix[k] = -1; }
    }
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s - lane >= N) return;                     // whole warp past the end
    const int sc = min(s, N - 1);                  // tail lanes mirror the last slot (no store)
    float qx, qy, qz = 0.f;
    int self;
    if (D == 2) {
        float2 q = v.spos2[sc];
        qx = q.x; qy = q.y; self = v.sidx[sc];
    } else {
        float4 q = v.spos4[sc];
        qx = q.x; qy = q.y; qz = q.z; self = __float_as_int(q.w);
    }
    const int cx = cell_axis(qx, v.lo0, v.inv_h, v.G0);
    const int cy = cell_axis(qy, v.lo1, v.inv_h, v.G1);
    const int cz = D == 3 ? cell_axis(qz, v.lo2, v.inv_h, v.G2) : 0;
    const int rowid = cz * v.G1 + cy;
    const bool has_l = cx > 0, has_r = cx < v.G0 - 1;
    Top2 best;
    best.init();
    // queries of this warp (marked slots are never tombstones, so their cells are in slot order)
    const bool query = SWEEP ? (s < N && mark[sc] != 0) : true;
    if (SWEEP && query) mark[sc] = 0;              // the marks are all zero again when the sweep ends
    unsigned todo = __ballot_sync(0xffffffffu, query);
    while (todo) {
        const int leader = __ffs(todo) - 1;
        const int R = __shfl_sync(0xffffffffu, rowid, leader);
        const unsigned seg = __ballot_sync(0xffffffffu, rowid == R) & todo;
        const int first = __ffs(seg) - 1, last = 31 - __clz(seg);
        const int xf = __shfl_sync(0xffffffffu, cx, first), xl = __shfl_sync(0xffffffffu, cx, last);
        const int ry = __shfl_sync(0xffffffffu, cy, first), rz = __shfl_sync(0xffffffffu, cz, first);
        const bool mine = (seg >> lane) & 1u;
        const int ux0 = max(xf - 1, 0), ux1 = min(xl + 1, v.G0 - 1);
#pragma unroll 1
        for (int k = -1; k < (D == 3 ? 8 : 2); ++k) {          // k = -1: the lanes' own row
            const int oy = k < 0 ? 0 : row_oy(k), oz = k < 0 ? 0 : row_oz(k);
            const int y = ry + oy, z = rz + oz;
            if (y < 0 || y >= v.G1 || z < 0 || z >= v.G2) continue;
            const int32_t *crow = v.cell_start + (z * v.G1 + y) * v.G0;
            if (chains && mine)
                for (int x = has_l ? cx - 1 : cx; x <= (has_r ? cx + 1 : cx); ++x)
                    scan_chain<D>(v, (z * v.G1 + y) * v.G0 + x, qx, qy, qz, self, best);
            const int B = crow[ux0], E = crow[ux1 + 1];
            if (B == E) continue;
            if (E - B < WT_DENSE) {
                int b = 0, e = 0;
                if (mine) { b = crow[has_l ? cx - 1 : cx]; e = crow[has_r ? cx + 2 : cx + 1]; }
                tile_pass<D>(v, N, lane, tp2, tp4, tix, B, E, b, e, 0, 0, qx, qy, qz, self, best);
                continue;
            }
            const Gaps g = make_gaps<D>(v, qx, qy, qz, cx, cy, cz);
            if (k < 0) {
                int s0 = 0, s1 = 0;
                if (mine) { s0 = crow[cx]; s1 = crow[cx + 1]; }
                tile_pass<D>(v, N, lane, tp2, tp4, tix, crow[xf], crow[xl + 1], s0, s1, 0, 0, qx, qy, qz, self, best);
                int bl = 0, el = 0, br = 0, er = 0;
                if (mine && has_l && !(best.s2 < g.xm)) { bl = crow[cx - 1]; el = s0; }
                if (mine && has_r && !(best.s2 < g.xp)) { br = s1; er = crow[cx + 2]; }
                dense_pass<D>(v, N, lane, tp2, tp4, tix, bl, el, br, er, qx, qy, qz, self, best);
            } else {
                int b = 0, e = 0;
                if (mine) {
                    const float rb2 = __fadd_rn(oy < 0 ? g.ym : (oy > 0 ? g.yp : 0.f), oz < 0 ? g.zm : (oz > 0 ? g.zp : 0.f));
                    if (!(best.s2 < rb2)) {
                        int x0 = cx, x1 = cx + 1;
                        if (has_l && !(best.s2 < __fadd_rn(rb2, g.xm))) x0 = cx - 1;
                        if (has_r && !(best.s2 < __fadd_rn(rb2, g.xp))) x1 = cx + 2;
                        b = crow[x0]; e = crow[x1];
                    }
                }
                dense_pass<D>(v, N, lane, tp2, tp4, tix, b, e, 0, 0, qx, qy, qz, self, best);
            }
        }
        todo &= ~seg;
    }
    if (!query) return;
    const int r = finish_block<D>(v, chains, qx, qy, qz, self, cx, cy, cz, best);
    if (s >= N) return;
    if (r > 2) atomicAdd(&ctr->n_stragglers, 1);
    store_cert_keep(best, self, nn, nn2, d1, d2, c);
}

// ---- A3 / A7, leaf-tiled: the kernel behind kc_cert_grid_search and the slot sweep of A7 ---------
// A warp owns 32 consecutive sorted slots.  Slots are sorted by leaf, so the windows the lanes need
// from one row of their 3^d blocks (3 cells of a grid row for a lane in an undivided cell, 3
// sub-cells of a sub-row of its own cell for a lane in a subdivided cell) lie close together in
// the sorted arrays.  Phase 1, warp-uniform control flow: every lane computes its window for each of
// the 3^(d-1) rows (all start indices are fetched in one round trip), and row by row the hull of the
// lanes' windows goes through the warp's shared-memory tile (coalesced loads) and every lane scans
// its own window of it.  Phase 2, per lane and only where needed: a lane whose block bound already
// exceeds its second-best is done; the others queue what phase 1 did not serve -- windows that
// hold a subdivided cell, everything outside the 3^d sub-block of a lane in a subdivided cell --
// range by range with every pruning test applied, and the queues are scanned by the warp in step.
constexpr int LT_WARPS = 4;
// A7: when the slot sweep serves a frontier: grids of >= SWEEP_MIN_N points, frontier of >= N / div points.
// Measured on config 5 (4,194,304 points, fresh grid, a random subset as the frontier; DESIGN.md section 5 A7):
// d = 2: the list kernels win up to a quarter of the points (12.5 %: 0.26 vs 0.43 ms; 30 %: 0.53 vs 0.48);
// d = 3: one thread per query on clustered cells is slow (10 %: 0.96 ms, the sweep 0.44), so the sweep takes
// over as soon as the list is too long for one WARP per query (WPQ_MAX), down to N / 32 (3 %: 0.37 vs 0.37).
constexpr int SWEEP_MIN_N = 200000, SWEEP_DIV2 = 4;   // (d = 3: list_div3, kc_grid.cuh)
#ifndef LT_MIN_BLOCKS
#define LT_MIN_BLOCKS 8
#endif
constexpr int LT_HULL_MAX = 4096;                 // a longer hull (lanes far apart in memory) is left to phase 2
static_assert(32 * LT_WARPS == PS_THREADS, "the range queues are strided by PS_THREADS");

// index (k of phase 1) of the block row at offset (oy, oz): k = 0 own row, k >= 1: row_oy/row_oz(k-1)
__device__ __forceinline__ int block_row_index(int oy, int oz)
{
    // (oz+1)*3 + (oy+1) -> k, 4 bits each: {5,3,6, 1,0,2, 7,4,8}
    const unsigned long long tab = 0x5ull | (0x3ull << 4) | (0x6ull << 8) | (0x1ull << 12) | (0x0ull << 16) |
                                   (0x2ull << 20) | (0x7ull << 24) | (0x4ull << 28) | (0x8ull << 32);
    return (int)((tab >> (4 * ((oz + 1) * 3 + oy + 1))) & 15ull);
}
// Sub-rows of the subdivided cell cid = (kx, ky, kz) inside the index box of the ball, minus the
// sub-block [bx0,bx1]x[by0,by1]x[bz0,bz1] if has_block (served by phase 1).
template <int D>
__device__ __forceinline__ void ball_sub(const View &v, Lane &L, int cid, int kx, int ky, int kz, const float (&lo)[3],
                                         const float (&hi)[3], bool has_block, int bx0, int bx1, int by0, int by1,
                                         int bz0, int bz1, const Qry &q, Top2 &best)
{
    const int2 si = v.subinfo[cid];
    const int S = si.x;
    const int32_t *__restrict__ ss = v.leaf_start + si.y;
    const float fS = (float)S;
    const int x0 = sub_axis(lo[0], v.lo0, v.inv_h, kx, fS, S), x1 = sub_axis(hi[0], v.lo0, v.inv_h, kx, fS, S);
    const int y0 = sub_axis(lo[1], v.lo1, v.inv_h, ky, fS, S), y1 = sub_axis(hi[1], v.lo1, v.inv_h, ky, fS, S);
    const int z0 = D == 3 ? sub_axis(lo[2], v.lo2, v.inv_h, kz, fS, S) : 0;
    const int z1 = D == 3 ? sub_axis(hi[2], v.lo2, v.inv_h, kz, fS, S) : 0;
    for (int z = z0; z <= z1; ++z)
        for (int y = y0; y <= y1; ++y) {
            if (L.big) return;                   // (queue dropped: nothing more to collect)
            const int row = (z * S + y) * S;
            if (has_block && y >= by0 && y <= by1 && z >= bz0 && z <= bz1) {
                if (x0 < bx0) rl_push<D>(v, L, ss[row + x0], ss[row + min(x1, bx0 - 1) + 1], q, best);
                if (x1 > bx1) rl_push<D>(v, L, ss[row + max(x0, bx1 + 1)], ss[row + x1 + 1], q, best);
            } else {
                rl_push<D>(v, L, ss[row + x0], ss[row + x1 + 1], q, best);
            }
        }
}
// Cells xa..xb of grid row (y, z) inside the ball's index box.
template <int D>
__device__ __forceinline__ void ball_cells(const View &v, Lane &L, bool chains, int y, int z, int xa, int xb,
                                           const float (&lo)[3], const float (&hi)[3], const Qry &q, Top2 &best)
{
    if (xa > xb) return;
    const int rowbase = (z * v.G1 + y) * v.G0;
    const int32_t *cs = v.cell_start + rowbase;
    const int b = cs[xa], e = cs[xb + 1];
    if (e - b < v.heavy_T) {
        rl_push<D>(v, L, b, e, q, best);
    } else {
        int lo_s = b;
        for (int x = xa; x <= xb && !L.big; ++x) {
            const int hi_s = x == xb ? e : cs[x + 1];
            if (hi_s - lo_s >= v.heavy_T) ball_sub<D>(v, L, rowbase + x, x, y, z, lo, hi, false, 0, 0, 0, 0, 0, 0, q, best);
            else rl_push<D>(v, L, lo_s, hi_s, q, best);
            lo_s = hi_s;
        }
    }
    if (chains)
        for (int x = xa; x <= xb; ++x) scan_chain<D>(v, rowbase + x, q.x, q.y, q.z, q.self, best);
}
// What the ball of a query still needs beyond phase 1: nothing, ranges to queue (ball_box), or the
// ring search (no bound yet, or an index box of too many cells: an isolated point).
enum { BALL_DONE = 0, BALL_MORE = 1, BALL_RINGS = 2, BALL_BIG = 3 };
struct BallBox {
    float lo[3], hi[3];
    int X0, X1, Y0, Y1, Z0, Z1;
};
template <int D>
__device__ __forceinline__ int ball_state(const View &v, const Qry &q, const Top2 &best, int cx, int cy, int cz,
                                          bool heavy, unsigned covered, int S, int ux, int uy, int uz, BallBox &B)
{
    if (best.s2 == CUDART_INF_F) return BALL_RINGS;
    // r >= the real distance of anything whose computed squared distance is <= s2 (fp32 rounding
    // of s: relative 3u, or absolute 2^-149 per operation in the denormal range)
    const float r = __fadd_ru(__fmul_ru(__fsqrt_ru(best.s2), 1.0009765625f), 8.470329e-22f);
    B.lo[0] = __fsub_rd(q.x, r); B.hi[0] = __fadd_ru(q.x, r);
    B.lo[1] = __fsub_rd(q.y, r); B.hi[1] = __fadd_ru(q.y, r);
    B.lo[2] = D == 3 ? __fsub_rd(q.z, r) : 0.f; B.hi[2] = D == 3 ? __fadd_ru(q.z, r) : 0.f;
    B.X0 = cell_axis(B.lo[0], v.lo0, v.inv_h, v.G0); B.X1 = cell_axis(B.hi[0], v.lo0, v.inv_h, v.G0);
    B.Y0 = cell_axis(B.lo[1], v.lo1, v.inv_h, v.G1); B.Y1 = cell_axis(B.hi[1], v.lo1, v.inv_h, v.G1);
    B.Z0 = D == 3 ? cell_axis(B.lo[2], v.lo2, v.inv_h, v.G2) : 0; B.Z1 = D == 3 ? cell_axis(B.hi[2], v.lo2, v.inv_h, v.G2) : 0;
    if ((int64_t)(B.X1 - B.X0 + 1) * (B.Y1 - B.Y0 + 1) * (B.Z1 - B.Z0 + 1) > 64) return BALL_RINGS;
    // the common case: the box lies inside what phase 1 served
    const bool in_block = B.X0 >= cx - 1 && B.X1 <= cx + 1 && B.Y0 >= cy - 1 && B.Y1 <= cy + 1 && B.Z0 >= cz - 1 && B.Z1 <= cz + 1;
    if (!heavy && in_block && covered == (D == 3 ? 0x7ffffffu : 0x1ffu)) return BALL_DONE;
    if (heavy && B.X0 == cx && B.X1 == cx && B.Y0 == cy && B.Y1 == cy && B.Z0 == cz && B.Z1 == cz) {
        const float fS = (float)S;
        if (sub_axis(B.lo[0], v.lo0, v.inv_h, cx, fS, S) >= ux - 1 && sub_axis(B.hi[0], v.lo0, v.inv_h, cx, fS, S) <= ux + 1 &&
            sub_axis(B.lo[1], v.lo1, v.inv_h, cy, fS, S) >= uy - 1 && sub_axis(B.hi[1], v.lo1, v.inv_h, cy, fS, S) <= uy + 1 &&
            (D == 2 || (sub_axis(B.lo[2], v.lo2, v.inv_h, cz, fS, S) >= uz - 1 &&
                        sub_axis(B.hi[2], v.lo2, v.inv_h, cz, fS, S) <= uz + 1)))
            return BALL_DONE;      // (on an updated grid the caller still scans the own cell's chain)
    }
    return BALL_MORE;
}
// A query whose ball box holds more than a lane's queue may hold (a sparse point beside a dense cluster:
// most of the box lies outside the ball): the cells of the box one by one, each row and cell tested
// against the CURRENT bound (strict), subdivided cells through visit_heavy, which prunes sub-row by
// sub-row.  Whatever phase 1 has offered already is skipped by id.  (Rare path: out of line.)
template <int D>
__device__ __noinline__ Top2 box_visit(const View &v, bool chains, float qx, float qy, float qz, int self, int cx,
                                       int cy, int cz, int X0, int X1, int Y0, int Y1, int Z0, int Z1, Top2 best)
{
    for (int z = Z0; z <= Z1; ++z) {
        const float gz = D == 3 ? axis_gap2(v, qz, v.lo2, v.slk2, z, cz) : 0.0f;
        if (best.s2 < gz) continue;
        for (int y = Y0; y <= Y1; ++y) {
            const float gy = __fadd_rn(gz, axis_gap2(v, qy, v.lo1, v.slk1, y, cy));
            if (best.s2 < gy) continue;
            const int rowbase = (z * v.G1 + y) * v.G0;
            const int32_t *cs = v.cell_start + rowbase;
            for (int x = X0; x <= X1; ++x) {
                if (best.s2 < __fadd_rn(gy, axis_gap2(v, qx, v.lo0, v.slk0, x, cx))) continue;
                const int b = cs[x], e = cs[x + 1];
                if (e > b) visit_cell<D>(v, rowbase + x, x, y, z, b, e, qx, qy, qz, self, best);
                if (chains) scan_chain<D>(v, rowbase + x, qx, qy, qz, self, best);
            }
        }
    }
    return best;
}
// Queues what the ball needs beyond phase 1.  Returns BALL_DONE (everything the ball needs is served or
// queued), BALL_RINGS (no bound yet / a box of too many cells: the ring search) or BALL_BIG (the box B
// holds more than a lane's queue may hold: box_visit).
template <int D>
__device__ __forceinline__ int ball_box(const View &v, Lane &L, bool chains, const Qry &q, Top2 &best, int cx, int cy,
                                        int cz, bool heavy, unsigned covered, int cs0, int cs1, int S,
                                        const int32_t *ss, int ux, int uy, int uz, BallBox &B)
{
    const int st = ball_state<D>(v, q, best, cx, cy, cz, heavy, covered, S, ux, uy, uz, B);
    if (st == BALL_RINGS) return BALL_RINGS;
    if (st == BALL_DONE) {
        if (heavy && chains) scan_chain<D>(v, (cz * v.G1 + cy) * v.G0 + cx, q.x, q.y, q.z, q.self, best);
        return BALL_DONE;
    }
    const float (&lo)[3] = B.lo, (&hi)[3] = B.hi;
    const int X0 = B.X0, X1 = B.X1, Y0 = B.Y0, Y1 = B.Y1, Z0 = B.Z0, Z1 = B.Z1;
    // Row by row, the cells X0..X1 in maximal runs of cells phase 1 has NOT served (one call site of
    // ball_cells: the kernel's code stays small).  Served: for a light lane the cells cx-1..cx+1 of a
    // block row whose `covered` bit is set (their chains too); for a lane in a subdivided cell the
    // 3^d sub-block of its own cell, so that cell goes through its sub-cells minus the sub-block.
    for (int z = Z0; z <= Z1; ++z)
        for (int y = Y0; y <= Y1; ++y) {
            const int oy = y - cy, oz = z - cz;
            const bool near = oy >= -1 && oy <= 1 && oz >= -1 && oz <= 1;
            const unsigned cv = (!heavy && near) ? (covered >> (3 * block_row_index(oy, oz))) & 7u : 0u;
            const bool own_row = heavy && oy == 0 && oz == 0;
            if (L.big) return BALL_BIG;          // queue dropped: the caller walks the box (box_visit)
            int xa = X0;
            for (int x = X0; x <= X1 + 1; ++x) {
                const bool own = own_row && x == cx;
                const bool served = x >= cx - 1 && x <= cx + 1 && ((cv >> (x - cx + 1)) & 1u);
                if (x <= X1 && !own && !served) continue;
                if (xa < x) ball_cells<D>(v, L, chains, y, z, xa, x - 1, lo, hi, q, best);
                xa = x + 1;
                if (own && x <= X1) {
                    if (chains) scan_chain<D>(v, (z * v.G1 + y) * v.G0 + cx, q.x, q.y, q.z, q.self, best);
                    ball_sub<D>(v, L, (z * v.G1 + y) * v.G0 + cx, cx, cy, cz, lo, hi, true, max(ux - 1, 0),
                                min(ux + 1, S - 1), max(uy - 1, 0), min(uy + 1, S - 1), D == 3 ? max(uz - 1, 0) : 0,
                                D == 3 ? min(uz + 1, S - 1) : 0, q, best);
                }
            }
        }
    return L.big ? BALL_BIG : BALL_DONE;
}

// The search of one round: lane `lane` serves the query at sorted slot sc (query = false: the lane only
// takes part in the warp-wide steps).  Called by all 32 lanes.
template <int D, int MODE>
__device__ __forceinline__ void leaf_search_round(const View &v, int N, Counters *ctr, bool chains, bool defer_mode, int lane,
                                                  float2 *tp2, float4 *tp4, int *tix, Lane &L, int sc, bool query,
                                                  int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c)
{
    constexpr int NR = D == 3 ? 9 : 3;             // rows of a 3^d block
    if (!__any_sync(0xffffffffu, query)) return;
    Qry q;
    q.z = 0.f;
    if (D == 2) {
        const float2 t = v.spos2[sc];
        q.x = t.x; q.y = t.y; q.self = v.sidx[sc];
    } else {
        const float4 t = v.spos4[sc];
        q.x = t.x; q.y = t.y; q.z = t.z; q.self = __float_as_int(t.w);
    }
    const int cx = cell_axis(q.x, v.lo0, v.inv_h, v.G0);
    const int cy = cell_axis(q.y, v.lo1, v.inv_h, v.G1);
    const int cz = D == 3 ? cell_axis(q.z, v.lo2, v.inv_h, v.G2) : 0;
    const int cellid = (cz * v.G1 + cy) * v.G0 + cx;
    const bool has_l = cx > 0, has_r = cx < v.G0 - 1;
    int cs0 = 0, cs1 = 0;
    if (query) { cs0 = v.cell_start[cellid]; cs1 = v.cell_start[cellid + 1]; }
    const bool heavy = query && cs1 - cs0 >= v.lane_T;
    int S = 0, ux = 0, uy = 0, uz = 0;
    const int32_t *ss = v.leaf_start;
    if (heavy) {
        const int2 si = v.subinfo[cellid];
        S = si.x; ss += si.y;
        const float fS = (float)S;
        ux = sub_axis(q.x, v.lo0, v.inv_h, cx, fS, S);
        uy = sub_axis(q.y, v.lo1, v.inv_h, cy, fS, S);
        uz = D == 3 ? sub_axis(q.z, v.lo2, v.inv_h, cz, fS, S) : 0;
    }
    Top2 best;
    best.init();
    // phase 1a: this lane's window in every row of its block (k = 0: its own row); covered = rows
    // that need nothing more (light lanes: served by the tile or outside the grid)
    unsigned covered = 0;
    if (query) {
#pragma unroll
        for (int k = 0; k < NR; ++k) {
            const int oy = k == 0 ? 0 : row_oy(k - 1), oz = k == 0 ? 0 : row_oz(k - 1);
            int b = 0, e = 0;
            if (heavy) {
                const int y = uy + oy, z = uz + oz;
                if (y >= 0 && y < S && z >= 0 && z < (D == 3 ? S : 1)) {
                    const int32_t *srow = ss + (z * S + y) * S;
                    b = srow[max(ux - 1, 0)]; e = srow[min(ux + 1, S - 1) + 1];
                }
            } else {
                const int y = cy + oy, z = cz + oz;
                if (y >= 0 && y < v.G1 && z >= 0 && z < v.G2) {
                    const int32_t *crow = v.cell_start + (z * v.G1 + y) * v.G0;
                    b = crow[has_l ? cx - 1 : cx]; e = crow[has_r ? cx + 2 : cx + 1];
                    if (e - b < v.lane_T) {
                        covered |= 7u << (3 * k);
                    } else if (k == 0) {
                        // a long window (dense cells, or a subdivided one): the ball of phase 2 prunes
                        // it; here only the own cell, which gives that ball its radius
                        b = crow[cx]; e = crow[cx + 1];
                        covered |= 2u << (3 * k);            // (the own cell of a light lane is undivided)
                    } else {
                        b = 0; e = 0;
                    }
                } else {
                    covered |= 7u << (3 * k);
                }
            }
            L.rl[(RL_CAP - 1 - k) * PS_THREADS] = make_int2(b, e);    // top of the queue's storage: the
        }                                                              // queue itself holds < RL_CAP - NR here
    }
    // phase 1b: row by row through the tile
    float gym = 0.f, gyp = 0.f, gzm = 0.f, gzp = 0.f;
#pragma unroll 1
    for (int k = 0; k < NR; ++k) {
        int2 w = make_int2(0, 0);
        if (query) w = L.rl[(RL_CAP - 1 - k) * PS_THREADS];
        if (k == 1 && query && !heavy) {
            // squared lower bounds of the distance to the neighbouring rows (see gap_lb), from the
            // second-best the own row has given: a row that lies provably farther is skipped
            float t;
            t = gap_lb(v, __fsub_rn(q.y, face_at(v.lo1, cy, v.h)), v.slk1); gym = __fmul_rn(t, t);
            t = gap_lb(v, __fsub_rn(face_at(v.lo1, cy + 1, v.h), q.y), v.slk1); gyp = __fmul_rn(t, t);
            if (D == 3) {
                t = gap_lb(v, __fsub_rn(q.z, face_at(v.lo2, cz, v.h)), v.slk2); gzm = __fmul_rn(t, t);
                t = gap_lb(v, __fsub_rn(face_at(v.lo2, cz + 1, v.h), q.z), v.slk2); gzp = __fmul_rn(t, t);
            }
        }
        if (k >= 1 && !heavy && w.x < w.y) {
            const int oy = row_oy(k - 1), oz = row_oz(k - 1);
            const float rb2 = __fadd_rn(oy < 0 ? gym : (oy > 0 ? gyp : 0.f), oz < 0 ? gzm : (oz > 0 ? gzp : 0.f));
            if (best.s2 < rb2) w.y = w.x;                       // (its cells stay marked as served)
        }
        const bool has = w.x < w.y;
        if (chains && query && !heavy && ((covered >> (3 * k)) & 7u)) {
            // the overflow chains of the served cells (a cell without sorted records may still hold
            // re-filed points)
            const int oy = k == 0 ? 0 : row_oy(k - 1), oz = k == 0 ? 0 : row_oz(k - 1);
            const int y = cy + oy, z = cz + oz;
            if (y >= 0 && y < v.G1 && z >= 0 && z < v.G2)
                for (int x = has_l ? cx - 1 : cx; x <= (has_r ? cx + 1 : cx); ++x)
                    if ((covered >> (3 * k + x - cx + 1)) & 1u)
                        scan_chain<D>(v, (z * v.G1 + y) * v.G0 + x, q.x, q.y, q.z, q.self, best);
        }
        // the lanes in undivided cells and those in subdivided cells look at different places: one
        // hull each (a hull that is still long -- lanes in two grid rows -- goes to the queues)
#pragma unroll 1
        for (int grp = 0; grp < 2; ++grp) {
            const bool in = has && heavy == (grp == 1);
            const int B = __reduce_min_sync(0xffffffffu, in ? w.x : 0x7fffffff);
            const int E = __reduce_max_sync(0xffffffffu, in ? w.y : 0);
            if (B >= E) continue;
            if (E - B > LT_HULL_MAX) {                          // (rare; the queue's storage holds the windows)
                if (in) scan_range<D>(v, w.x, w.y, q.x, q.y, q.z, q.self, best);
                continue;
            }
            tile_pass<D>(v, N, lane, tp2, tp4, tix, B, E, in ? w.x : 0, in ? w.y : 0, 0, 0, q.x, q.y, q.z, q.self, best);
        }
    }
    // phase 2: the ball.  Every record that can still enter the list lies within r = d2 (as of now)
    // of the query, so on every axis its coordinate lies in [q - r, q + r], and because the filing
    // functions cell_axis / sub_axis are monotone, its cell (sub-cell) index lies between the
    // indices of those two end points: the candidates are the cells of an index box.  No face
    // arithmetic and no slack are involved: the end points are rounded outwards.  A query whose box
    // lies inside what phase 1 served (the common case) is done; the others -- a fifth of the
    // queries of config 5, a few lanes of every warp -- go to a list with what they have found, and
    // ball_finish_kernel serves that list with full warps.
    // On a grid without (many) subdivided cells few queries get here and the list would only expose
    // their latency: there every lane queues and scans its own ranges on the spot (defer_mode false).
    bool defer = false, rings = false;
    BallBox B;
    lane_reset(L);
    if (query) {
        if (defer_mode) {
            const int st = ball_state<D>(v, q, best, cx, cy, cz, heavy, covered, S, ux, uy, uz, B);
            defer = st == BALL_MORE;
            rings = st == BALL_RINGS;
            if (st == BALL_DONE && heavy && chains) scan_chain<D>(v, cellid, q.x, q.y, q.z, q.self, best);
        } else {
            const int st = ball_box<D>(v, L, chains, q, best, cx, cy, cz, heavy, covered, cs0, cs1, S, ss, ux, uy, uz, B);
            rings = st != BALL_DONE;             // (a queue that overflows, on these small or uniform grids: the rings too)
        }
    }
    if (!defer_mode && __any_sync(0xffffffffu, L.cnt > 0)) rl_scan<D>(v, L, q, best);
    if (query && !defer) {
        if (rings) {
            // no bound yet, or a ball of many cells (an isolated point): the classic ring search (here
            // and not in the second kernel, where its serial rings would be the tail of a short kernel)
            const int r = block_search<D>(v, chains, q.x, q.y, q.z, q.self, cx, cy, cz, best);
            if (r > 2) atomicAdd(&ctr->n_stragglers, 1);
        }
        store_cert_keep(best, q.self, nn, nn2, d1, d2, c);
    }
    const unsigned dm = __ballot_sync(0xffffffffu, defer);
    if (dm) {
        const int leader = __ffs(dm) - 1;
        int base = 0;
        if (lane == leader) base = atomicAdd(v.n_defer, __popc(dm));
        base = __shfl_sync(0xffffffffu, base, leader);
        if (defer) {
            float4 *e = v.defer + 2 * (size_t)(base + __popc(dm & ((1u << lane) - 1)));
            e[0] = make_float4(__int_as_float(sc), __uint_as_float(covered), 0.f, 0.f);
            e[1] = make_float4(best.s1, best.s2, __int_as_float(best.j1), __int_as_float(best.j2));
        }
    }
}

// The second kernel of the leaf search: the queries phase 1 could not finish, 32 list entries per warp.
// Every lane queues what its ball needs beyond phase 1 (ball_box), the warp scans the queues in step,
// the few queries without a bound or with a wide box run the ring search.  The block that finishes
// last empties the list.
// Resident blocks only; a warp takes the next 32 entries from a shared counter, so that the expensive
// tail of the list (the queries of the densest cells) spreads over all SMs.
constexpr int BF_PER_SM = 14;
constexpr int DEFER_MIN_N = 100000;              // smaller grids are launch-bound: no second kernel
inline int bf_blocks(int n) { return min(148 * BF_PER_SM, (n + PS_THREADS - 1) / PS_THREADS); }
#ifndef BF_MIN_BLOCKS
#define BF_MIN_BLOCKS 8
#endif
template <int D>
__global__ void __launch_bounds__(PS_THREADS, BF_MIN_BLOCKS)
ball_finish_kernel(const __grid_constant__ View v, int N, Counters *ctr, int may_chain, int32_t *nn, int32_t *nn2,
                   float *d1, float *d2, float *c)
{
    __shared__ int2 s_rl[RL_CAP * PS_THREADS];
    const int n = ctr->n_defer;
    if (n == 0) return;                            // (every CTA sees the same count: it changes below only)
    const bool chains = may_chain && ctr->n_misfiled > 0;
    const int lane = threadIdx.x & 31;
    Lane L;
    L.rl = s_rl + threadIdx.x;
    lane_reset(L);
#pragma unroll 1
    for (;;) {
        int base = 0;
        if (lane == 0) base = atomicAdd(&ctr->defer_next, 32);
        base = __shfl_sync(0xffffffffu, base, 0);
        if (base >= n) break;
        const bool query = base + lane < n;
        const int ent = min(base + lane, n - 1);
        const float4 e0 = v.defer[2 * (size_t)ent], e1 = v.defer[2 * (size_t)ent + 1];
        const int sc = __float_as_int(e0.x);
        const unsigned covered = __float_as_uint(e0.y);
        Top2 best;
        best.s1 = e1.x; best.s2 = e1.y; best.j1 = __float_as_int(e1.z); best.j2 = __float_as_int(e1.w);
        Qry q;
        q.z = 0.f;
        if (D == 2) {
            const float2 t = v.spos2[sc];
            q.x = t.x; q.y = t.y; q.self = v.sidx[sc];
        } else {
            const float4 t = v.spos4[sc];
            q.x = t.x; q.y = t.y; q.z = t.z; q.self = __float_as_int(t.w);
        }
        const int cx = cell_axis(q.x, v.lo0, v.inv_h, v.G0);
        const int cy = cell_axis(q.y, v.lo1, v.inv_h, v.G1);
        const int cz = D == 3 ? cell_axis(q.z, v.lo2, v.inv_h, v.G2) : 0;
        const int cellid = (cz * v.G1 + cy) * v.G0 + cx;
        const int cs0 = v.cell_start[cellid], cs1 = v.cell_start[cellid + 1];
        const bool heavy = cs1 - cs0 >= v.lane_T;
        int S = 0, ux = 0, uy = 0, uz = 0;
        const int32_t *ss = v.leaf_start;
        if (heavy) {
            const int2 si = v.subinfo[cellid];
            S = si.x; ss += si.y;
            const float fS = (float)S;
            ux = sub_axis(q.x, v.lo0, v.inv_h, cx, fS, S);
            uy = sub_axis(q.y, v.lo1, v.inv_h, cy, fS, S);
            uz = D == 3 ? sub_axis(q.z, v.lo2, v.inv_h, cz, fS, S) : 0;
        }
        // (an entry is here because ball_state said BALL_MORE in the first kernel; state and inputs are the
        // same, so ball_box never asks for the ring search -- those queries ran it there; a lane whose
        // queue overflows walks its box instead, see Lane)
        lane_reset(L);
        BallBox B;
        int st = BALL_DONE;
        if (query) st = ball_box<D>(v, L, chains, q, best, cx, cy, cz, heavy, covered, cs0, cs1, S, ss, ux, uy, uz, B);
        if (__any_sync(0xffffffffu, L.cnt > 0)) rl_scan<D>(v, L, q, best);
        if (query) {
            if (st == BALL_BIG) best = box_visit<D>(v, chains, q.x, q.y, q.z, q.self, cx, cy, cz, B.X0, B.X1, B.Y0, B.Y1, B.Z0, B.Z1, best);
            store_cert_keep(best, q.self, nn, nn2, d1, d2, c);
        }
        __syncwarp();
    }
    __syncthreads();
    if (threadIdx.x == 0 && atomicAdd(&ctr->ticket4, 1) == (int)gridDim.x - 1) {
        ctr->n_deferred += n;
        ctr->n_defer = 0;
        ctr->defer_next = 0;
        ctr->ticket4 = 0;
    }
}

// MODE 0: A3, thread t serves slot t.  MODE 1 / 2: the slot sweep of A7 on an updated / a fresh grid.  A
// warp of the sweep owns 32 * SW_WORDS consecutive slots and serves the marked ones among them 32 at a
// time, in slot order (the k-th marked slot goes to lane k mod 32 of round k / 32): every round runs
// with full lanes whatever the frontier's density, and its queries are still neighbours in the sorted
// arrays, which is all the tile passes need.  The marks are cleared on the way (all zero between calls).
template <int D, int MODE>
__global__ void __launch_bounds__(32 * LT_WARPS, LT_MIN_BLOCKS)
search_leaf_kernel(const __grid_constant__ View v, int N, Counters *ctr, int32_t *mark,
                   const int32_t *__restrict__ nF, int sweep_div, int32_t *nn, int32_t *nn2, float *d1,
                   float *d2, float *c)
{
    __shared__ __align__(16) float4 s_p4[D == 3 ? LT_WARPS : 1][D == 3 ? WT_TILE + 4 : 1];
    __shared__ __align__(16) float2 s_p2[D == 2 ? LT_WARPS : 1][D == 2 ? WT_TILE + 4 : 1];
    __shared__ int s_ix[D == 2 ? LT_WARPS : 1][D == 2 ? WT_TILE + 4 : 1];
    __shared__ int2 s_rl[RL_CAP * PS_THREADS];
    if (MODE != 0 && (int64_t)*nF * sweep_div < N) return;
    // the sweep has two instantiations, both launched; the frontier's density decides which one runs
    if (MODE != 0 && (sweep_words(N, *nF) == 1) != (MODE <= 2)) return;
    const bool chains = (MODE == 1 || MODE == 3) && ctr->n_misfiled > 0;     // MODE 2, 4: a fresh grid has no chains (compile-time)
    // with subdivided cells that hold at least N / 32 points, the queries phase 1 cannot finish go to the second kernel
    const bool defer_mode = N >= DEFER_MIN_N && (int64_t)ctr->n_heavy * v.heavy_T * 32 >= N;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const float qnan = __int_as_float(0x7fc00000);
    float4 *tp4 = s_p4[D == 3 ? warp : 0];
    float2 *tp2 = s_p2[D == 2 ? warp : 0];
    int *tix = s_ix[D == 2 ? warp : 0];
    for (int k = lane; k < WT_TILE + 4; k += 32) {          // the tile starts inert
        if (D == 3) tp4[k] = make_float4(qnan, qnan, qnan, __int_as_float(-1));
        else { tp2[k] = make_float2(qnan, qnan); tix[k] = -1; }
    }
    Lane L;
    L.rl = s_rl + threadIdx.x;
    lane_reset(L);
    if (MODE <= 2) {
        const int s = blockIdx.x * blockDim.x + threadIdx.x;
        if (s - lane >= N) return;                 // whole warp past the end
        const int sc = min(s, N - 1);
        bool query = s < N;
        if (MODE != 0) {
            query = query && mark[sc] != 0;
            if (query) mark[sc] = 0;               // the marks are all zero again when the sweep ends
        }
        leaf_search_round<D, MODE>(v, N, ctr, chains, defer_mode, lane, tp2, tp4, tix, L, sc, query, nn, nn2, d1, d2, c);
        return;
    }
    // (the sweep's bookkeeping lives in shared memory: nothing of it stays in registers across a round)
    __shared__ unsigned s_mask[LT_WARPS][SW_WORDS];
    __shared__ int s_tot[LT_WARPS], s_r0[LT_WARPS], s_sw[LT_WARPS];
    {
        const int sw = sweep_words(N, *nF);
        const int wbase = (blockIdx.x * LT_WARPS + warp) * (32 * sw);
        if (wbase >= N) return;
        int total = 0;
        for (int k = 0; k < sw; ++k) {
            const int s = wbase + 32 * k + lane;
            const bool mk = s < N && mark[s] != 0;
            if (mk) mark[s] = 0;                   // the marks are all zero again when the sweep ends
            const unsigned b = __ballot_sync(0xffffffffu, mk);
            if (lane == 0) s_mask[warp][k] = b;
            total += __popc(b);
        }
        if (lane == 0) { s_tot[warp] = total; s_r0[warp] = 0; s_sw[warp] = sw; }
        __syncwarp();
    }
#pragma unroll 1
    for (;;) {
        const int r0 = s_r0[warp], total = s_tot[warp], sw = s_sw[warp];
        if (r0 >= total) break;
        const int wbase = (blockIdx.x * LT_WARPS + warp) * (32 * sw);
        int t = r0 + lane, sc = wbase;
        const bool query = t < total;
        for (int k = 0; k < sw; ++k) {
            const unsigned b = s_mask[warp][k];
            const int cnt = __popc(b);
            if (query && t >= 0 && t < cnt) sc = wbase + 32 * k + (int)__fns(b, 0, t + 1);
            t -= cnt;
        }
        __syncwarp();
        if (lane == 0) s_r0[warp] = r0 + 32;
        __syncwarp();
        leaf_search_round<D, MODE>(v, N, ctr, chains, defer_mode, lane, tp2, tp4, tix, L, sc, query, nn, nn2, d1, d2, c);
        __syncwarp();
    }
}

// A7, large frontier: stamp the slots of the frontier points with this call's epoch; frontier
// points that live in an overflow chain have no slot and go to the list kernel (list2).
__global__ void __launch_bounds__(256)
mark_frontier_kernel(const int32_t *__restrict__ F, const int32_t *__restrict__ nF, int N, int sweep_div,
                     const int32_t *__restrict__ slot, int32_t *mark, int32_t *list2,
                     Counters *ctr)
{
    const int n = *nF;
    if ((int64_t)n * sweep_div < N) return;
    const int stride = gridDim.x * blockDim.x;
    for (int f0 = blockIdx.x * blockDim.x; f0 < n; f0 += stride) {     // warp-uniform trip count
        const int f = f0 + threadIdx.x;
        int i = -1;
        bool chain = false;
        if (f < n) {
            i = F[f];
            const int sl = slot[i];
            if (sl >= 0) mark[sl] = 1;
            else chain = true;
        }
        warp_append(chain, i, list2, &ctr->n_list2);
    }
}

// ---- warp per query ---------------------------------------------------------------------------
// One warp serves one query, one lane per cell of the 3^d block: every lane fetches its cell's
// record range and chain head at once (one memory round trip for the whole block instead of one
// per row), the own cell is scanned first by the whole warp, then every lane prunes its cell
// against the second-best found so far; short surviving ranges are scanned by their lanes, long
// ones (dense cells) by the whole warp, and two warp reductions extract the two smallest keys.
// No lane ever waits for another query's insertions, and the order of the queries is irrelevant,
// which is what a frontier list in id order needs (A7).
template <int D>
__device__ __forceinline__ void lane_offer(Top2 &tmp, float s, int j, float thr, int self)
{
    insert_bf(tmp, s, j, s <= thr && j >= 0 && j != self);
}
template <int D>
__device__ int wpq_search(const View &v, bool chains, int lane, float qx, float qy, float qz, int self,
                          Top2 &best)
{
    constexpr int NC = D == 3 ? 27 : 9, OWN = NC / 2;
    const int cx = cell_axis(qx, v.lo0, v.inv_h, v.G0);
    const int cy = cell_axis(qy, v.lo1, v.inv_h, v.G1);
    const int cz = D == 3 ? cell_axis(qz, v.lo2, v.inv_h, v.G2) : 0;
    const int ox = lane % 3 - 1, oy = (lane / 3) % 3 - 1, oz = D == 3 ? lane / 9 - 1 : 0;
    const int x = cx + ox, y = cy + oy, z = cz + oz;
    const bool valid = lane < NC && x >= 0 && x < v.G0 && y >= 0 && y < v.G1 && z >= 0 && z < v.G2;
    const int cid = valid ? (z * v.G1 + y) * v.G0 + x : 0;
    int b = 0, e = 0, hd = -1;
    if (valid) {
        b = v.cell_start[cid]; e = v.cell_start[cid + 1];
        if (chains) hd = v.head[cid];
    }
    // own cell: the whole warp
    Top2 tmp;
    tmp.init();
    const int ob = __shfl_sync(0xffffffffu, b, OWN), oe = __shfl_sync(0xffffffffu, e, OWN);
    coop_range<D>(v, lane, ob, oe, qx, qy, qz, self, CUDART_INF_F, KC_NOIDX, KC_NOIDX, tmp);
    if (lane == OWN)
        for (int c = hd; c >= 0; c = v.next[c]) {
            const float4 o = v.opos[c];
            lane_offer<D>(tmp, D == 2 ? sqd2(qx, qy, o.x, o.y) : sqd3(qx, qy, qz, o.x, o.y, o.z), c, CUDART_INF_F, self);
        }
    float sa, sb;
    int ja, jb;
    warp_pop(tmp, sa, ja);
    warp_pop(tmp, sb, jb);
    best.s1 = sa; best.j1 = ja; best.s2 = sb; best.j2 = jb;         // ordered: sa <= sb (or none)
    const float thr = best.s2;
    // the other cells: prune, then short ranges by their lanes, long ones by the warp
    const Gaps g = make_gaps<D>(v, qx, qy, qz, cx, cy, cz);
    const float lb2 = __fadd_rn(__fadd_rn(ox < 0 ? g.xm : (ox > 0 ? g.xp : 0.f), oy < 0 ? g.ym : (oy > 0 ? g.yp : 0.f)),
                                oz < 0 ? g.zm : (oz > 0 ? g.zp : 0.f));
    const bool need = valid && lane != OWN && !(thr < lb2);
    const int len = need ? e - b : 0;
    tmp.init();
    for (unsigned m = __ballot_sync(0xffffffffu, len > 16); m; m &= m - 1) {
        const int L = __ffs(m) - 1;
        coop_range<D>(v, lane, __shfl_sync(0xffffffffu, b, L), __shfl_sync(0xffffffffu, e, L), qx, qy, qz, self,
                      thr, KC_NOIDX, KC_NOIDX, tmp);
    }
    if (len <= 16)
        for (int t0 = b; t0 < b + len; t0 += 4) {        // 4 records per round trip, loads issued together
            const float qnan = __int_as_float(0x7fc00000);
            float4 c[4];
            int j[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const bool ok = t0 + k < b + len;
                if (D == 2) {
                    const float2 r = ok ? v.spos2[t0 + k] : make_float2(qnan, qnan);
                    c[k] = make_float4(r.x, r.y, 0.f, 0.f);
                    j[k] = ok ? v.sidx[t0 + k] : -1;
                } else {
                    c[k] = ok ? v.spos4[t0 + k] : make_float4(qnan, qnan, qnan, __int_as_float(-1));
                    j[k] = __float_as_int(c[k].w);
                }
            }
#pragma unroll
            for (int k = 0; k < 4; ++k)
                lane_offer<D>(tmp, D == 2 ? sqd2(qx, qy, c[k].x, c[k].y) : sqd3(qx, qy, qz, c[k].x, c[k].y, c[k].z),
                              j[k], thr, self);
        }
    if (need)
        for (int c = hd; c >= 0; c = v.next[c]) {
            const float4 o = v.opos[c];
            lane_offer<D>(tmp, D == 2 ? sqd2(qx, qy, o.x, o.y) : sqd3(qx, qy, qz, o.x, o.y, o.z), c, thr, self);
        }
    warp_pop(tmp, sa, ja);
    warp_pop(tmp, sb, jb);
    if (ja != KC_NOIDX) best.offer(sa, ja);
    if (jb != KC_NOIDX) best.offer(sb, jb);
    // every lane holds the same state: the rare ring continuation runs redundantly on all of them
    return finish_block<D, true>(v, chains, qx, qy, qz, self, cx, cy, cz, best, true);
}

// The list kernel is the last reader of list2 (the chain residents of a swept frontier): the block
// that finishes last empties the list, so that every kc_frontier_search call starts from an empty
// one whatever preceded it (every block has read the count before it takes its ticket).  Only a
// call whose frontier was swept can have filled the list, so only such a call takes tickets (one
// atomic per block on one address: 17 us for 4,736 blocks).
__device__ __forceinline__ void list2_done(Counters *ctr)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        if (atomicAdd(&ctr->ticket2, 1) == (int)gridDim.x - 1) {
            ctr->n_list2 = 0;
            ctr->ticket2 = 0;
        }
    }
}
template <int D>
__global__ void __launch_bounds__(128)
search_wpq_kernel(View v, const float *__restrict__ p_new, int N, const int32_t *__restrict__ F,
                  const int32_t *__restrict__ nF, const int32_t *__restrict__ list2, int sweep_div,
                  Counters *ctr, int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c)
{
    const int lane = threadIdx.x & 31;
    const int w0 = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
    // a large frontier is served by the slot sweep; only its chain residents (list2) come here
    const bool swept = sweep_div > 0 && (int64_t)*nF * sweep_div >= N;
    const int n = swept ? ctr->n_list2 : *nF;
    const int32_t *__restrict__ Q = swept ? list2 : F;
    const bool chains = ctr->n_misfiled > 0;
    if (n > WPQ_MAX) {
        // long list: one thread per query keeps more queries in flight
        for (int f = blockIdx.x * blockDim.x + threadIdx.x; f < n; f += gridDim.x * blockDim.x) {
            const int i = Q[f];
            const float qx = p_new[(int64_t)i * D], qy = p_new[(int64_t)i * D + 1];
            const float qz = D == 3 ? p_new[(int64_t)i * D + 2] : 0.f;
            Top2 best;
            best.init();
            const int cx = cell_axis(qx, v.lo0, v.inv_h, v.G0);
            const int cy = cell_axis(qy, v.lo1, v.inv_h, v.G1);
            const int cz = D == 3 ? cell_axis(qz, v.lo2, v.inv_h, v.G2) : 0;
            const int r = block_search<D, true>(v, chains, qx, qy, qz, i, cx, cy, cz, best);
            if (r > 2) atomicAdd(&ctr->n_stragglers, 1);
            store_cert(best, i, nn, nn2, d1, d2, c);
        }
        if (swept) list2_done(ctr);
        return;
    }
    for (int f = w0; f < n; f += nw) {
        const int i = Q[f];
        const float qx = p_new[(int64_t)i * D], qy = p_new[(int64_t)i * D + 1];
        const float qz = D == 3 ? p_new[(int64_t)i * D + 2] : 0.f;
        Top2 best;
        const int r = wpq_search<D>(v, chains, lane, qx, qy, qz, i, best);
        if (lane == 0) {
            if (r > 2) atomicAdd(&ctr->n_stragglers, 1);
            store_cert(best, i, nn, nn2, d1, d2, c);
        }
    }
    if (swept) list2_done(ctr);
}

// ---- NEXT #4: K-list certificates through the grid ---------------------------------------------
// One thread per sorted slot of a freshly built grid: own cell, then Chebyshev rings, until the
// bound of the scanned block exceeds the K-th best distance (the same strict test as A3, with
// s_K in the place of s_2: every unscanned point is then strictly farther than the K-th key).
template <int D, int K>
__device__ __forceinline__ void topk_scan_cells(const View &v, int rowbase, int x0, int x1, float qx, float qy,
                                                float qz, int self, TopK<K> &best)
{
    const int b = v.cell_start[rowbase + x0], e = v.cell_start[rowbase + x1 + 1];
    for (int t = b; t < e; ++t) {
        float s;
        int j;
        if (D == 2) {
            const float2 c = v.spos2[t];
            s = sqd2(qx, qy, c.x, c.y);
            j = v.sidx[t];
        } else {
            const float4 c = v.spos4[t];
            s = sqd3(qx, qy, qz, c.x, c.y, c.z);
            j = __float_as_int(c.w);
        }
        if (s <= best.s[K - 1] && j >= 0 && j != self) best.offer(s, j);
    }
}
template <int D, int K>
__device__ __forceinline__ void topk_scan_chains(const View &v, int rowbase, int x0, int x1, float qx, float qy,
                                                 float qz, int self, TopK<K> &best)
{
    for (int x = x0; x <= x1; ++x)
        for (int e = v.head[rowbase + x]; e >= 0; e = v.next[e]) {
            const float4 c = v.opos[e];
            const float s = D == 2 ? sqd2(qx, qy, c.x, c.y) : sqd3(qx, qy, qz, c.x, c.y, c.z);
            if (s <= best.s[K - 1] && e != self) best.offer(s, e);
        }
}
// K-list ring search of one query: own cell, then Chebyshev rings until the bound of the scanned block
// exceeds the K-th best squared distance (the same strict test as A3, with s_K in the place of s_2:
// every unscanned point is then strictly farther than the K-th key); with `chains` the overflow chains
// of every visited cell are scanned too (incrementally updated grid, tombstones are inert records).
template <int D, int K>
__device__ __forceinline__ void topk_visit(const View &v, bool chains, int rowbase, int x0, int x1, float qx, float qy,
                                           float qz, int self, TopK<K> &best)
{
    topk_scan_cells<D, K>(v, rowbase, x0, x1, qx, qy, qz, self, best);
    if (chains) topk_scan_chains<D, K>(v, rowbase, x0, x1, qx, qy, qz, self, best);
}
template <int D, int K>
__device__ __forceinline__ void topk_ring_search(const View &v, bool chains, float qx, float qy, float qz, int self,
                                                 TopK<K> &best)
{
    const int cx = cell_axis(qx, v.lo0, v.inv_h, v.G0);
    const int cy = cell_axis(qy, v.lo1, v.inv_h, v.G1);
    const int cz = D == 3 ? cell_axis(qz, v.lo2, v.inv_h, v.G2) : 0;
    topk_visit<D, K>(v, chains, (cz * v.G1 + cy) * v.G0, cx, cx, qx, qy, qz, self, best);
    for (int r = 0;;) {
        int z0 = D == 3 ? max(cz - r, 0) : 0, z1 = D == 3 ? min(cz + r, v.G2 - 1) : 0;
        int y0 = max(cy - r, 0), y1 = min(cy + r, v.G1 - 1);
        int x0 = max(cx - r, 0), x1 = min(cx + r, v.G0 - 1);
        if (bound_ok(box_bound<D>(v, qx, qy, qz, x0, x1, y0, y1, z0, z1), best.s[K - 1])) break;
        ++r;
        // ring r: shell rows get the full segment, inner rows only the two end cells
        z0 = D == 3 ? max(cz - r, 0) : 0; z1 = D == 3 ? min(cz + r, v.G2 - 1) : 0;
        y0 = max(cy - r, 0); y1 = min(cy + r, v.G1 - 1);
        x0 = max(cx - r, 0); x1 = min(cx + r, v.G0 - 1);
        for (int z = z0; z <= z1; ++z)
            for (int y = y0; y <= y1; ++y) {
                const int rowbase = (z * v.G1 + y) * v.G0;
                const bool shell = (D == 3 && (z == cz - r || z == cz + r)) || y == cy - r || y == cy + r;
                if (shell) {
                    topk_visit<D, K>(v, chains, rowbase, x0, x1, qx, qy, qz, self, best);
                } else {
                    if (cx - r >= 0) topk_visit<D, K>(v, chains, rowbase, cx - r, cx - r, qx, qy, qz, self, best);
                    if (cx + r <= v.G0 - 1) topk_visit<D, K>(v, chains, rowbase, cx + r, cx + r, qx, qy, qz, self, best);
                }
            }
    }
}
// One thread per sorted slot of a freshly built grid.
template <int D, int K>
__global__ void __launch_bounds__(128)
search_topk_kernel(View v, int N, int32_t *__restrict__ nnk, float *__restrict__ dk, float *__restrict__ ck)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= N) return;
    float qx, qy, qz = 0.f;
    int self;
    if (D == 2) {
        const float2 q = v.spos2[s];
        qx = q.x; qy = q.y; self = v.sidx[s];
    } else {
        const float4 q = v.spos4[s];
        qx = q.x; qy = q.y; qz = q.z; self = __float_as_int(q.w);
    }
    TopK<K> best;
    best.init();
    topk_ring_search<D, K>(v, false, qx, qy, qz, self, best);
    best.store(self, nnk, dk, ck);
}
// K-list repair (A7 for K keys): one thread per id of the list, against the incrementally updated grid.
template <int D, int K>
__global__ void __launch_bounds__(128)
search_topk_list_kernel(View v, const float *__restrict__ p_new, const int32_t *__restrict__ F,
                        const int32_t *__restrict__ nF, const Counters *ctr, int32_t *__restrict__ nnk,
                        float *__restrict__ dk, float *__restrict__ ck)
{
    const int n = *nF;
    const bool chains = ctr->n_misfiled > 0;
    for (int f = blockIdx.x * blockDim.x + threadIdx.x; f < n; f += gridDim.x * blockDim.x) {
        const int self = F[f];
        const float qx = p_new[(int64_t)self * D], qy = p_new[(int64_t)self * D + 1];
        const float qz = D == 3 ? p_new[(int64_t)self * D + 2] : 0.f;
        TopK<K> best;
        best.init();
        topk_ring_search<D, K>(v, chains, qx, qy, qz, self, best);
        best.store(self, nnk, dk, ck);
    }
}
template <int D>
bool dispatch_list_topk(int K, const View &v, const float *p_new, const int32_t *F, const int32_t *nF, int64_t nF_max,
                        const Counters *ctr, int32_t *nnk, float *dk, float *ck, cudaStream_t st)
{
    int64_t want = (nF_max + 127) / 128;
    const int nb = (int)(want < 1 ? 1 : (want < 148 * 16 ? want : 148 * 16));
    switch (K) {
    case 2: search_topk_list_kernel<D, 2><<<nb, 128, 0, st>>>(v, p_new, F, nF, ctr, nnk, dk, ck); return true;
    case 3: search_topk_list_kernel<D, 3><<<nb, 128, 0, st>>>(v, p_new, F, nF, ctr, nnk, dk, ck); return true;
    case 4: search_topk_list_kernel<D, 4><<<nb, 128, 0, st>>>(v, p_new, F, nF, ctr, nnk, dk, ck); return true;
    case 5: search_topk_list_kernel<D, 5><<<nb, 128, 0, st>>>(v, p_new, F, nF, ctr, nnk, dk, ck); return true;
    case 6: search_topk_list_kernel<D, 6><<<nb, 128, 0, st>>>(v, p_new, F, nF, ctr, nnk, dk, ck); return true;
    case 7: search_topk_list_kernel<D, 7><<<nb, 128, 0, st>>>(v, p_new, F, nF, ctr, nnk, dk, ck); return true;
    case 8: search_topk_list_kernel<D, 8><<<nb, 128, 0, st>>>(v, p_new, F, nF, ctr, nnk, dk, ck); return true;
    default: return false;
    }
}
template <int D>
bool dispatch_grid_topk(int K, const View &v, int n, int32_t *nnk, float *dk, float *ck, cudaStream_t st)
{
    const int nb = (n + 127) / 128;
    switch (K) {
    case 2: search_topk_kernel<D, 2><<<nb, 128, 0, st>>>(v, n, nnk, dk, ck); return true;
    case 3: search_topk_kernel<D, 3><<<nb, 128, 0, st>>>(v, n, nnk, dk, ck); return true;
    case 4: search_topk_kernel<D, 4><<<nb, 128, 0, st>>>(v, n, nnk, dk, ck); return true;
    case 5: search_topk_kernel<D, 5><<<nb, 128, 0, st>>>(v, n, nnk, dk, ck); return true;
    case 6: search_topk_kernel<D, 6><<<nb, 128, 0, st>>>(v, n, nnk, dk, ck); return true;
    case 7: search_topk_kernel<D, 7><<<nb, 128, 0, st>>>(v, n, nnk, dk, ck); return true;
    case 8: search_topk_kernel<D, 8><<<nb, 128, 0, st>>>(v, n, nnk, dk, ck); return true;
    default: return false;
    }
}

}  // namespace

// ====================================================================== C-ABI
// ---- straggler hand-off: brute force for the queries ring_continue gave up on ---------------------
// The whole GPU scans every record of the grid once per batch of HO_BATCH listed queries: CTA b owns
// one chunk of the records -- the sorted array (tombstones are inert) followed by the chain residents
// (mlist) -- keeps the two smallest keys (s, j) of every query of the batch over its chunk and writes
// them to part[query][b]; the CTA that finishes last merges the HANDOFF_BLOCKS partial lists of
// every query and stores its certificate: the definition itself, so the result is the one the rings
// would have reached.  That CTA also empties the list: every search call starts from an empty one.
// (One batch reads the records from HBM, later ones find them in L2.)
namespace {
constexpr int HO_THREADS = 512, HO_BATCH = 8;
template <int D>
__global__ void __launch_bounds__(HO_THREADS)
handoff_kernel(const View v, int N, const int32_t *__restrict__ mlist, Counters *ctr, HandoffPart *part,
               int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c)
{
    __shared__ float s_s[HO_BATCH][2 * HO_THREADS / 32];
    __shared__ int s_j[HO_BATCH][2 * HO_THREADS / 32];
    __shared__ bool s_last;
    const int n = min(ctr->n_handoff, HANDOFF_CAP);
    if (n == 0) return;                            // (every CTA sees the same count: it changes below only)
    const int nm = ctr->n_misfiled, total = N + nm;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nb = gridDim.x;
    const int chunk = (total + nb - 1) / nb;
    const int r0 = blockIdx.x * chunk, r1 = min(r0 + chunk, total);
    for (int f0 = 0; f0 < n; f0 += HO_BATCH) {
        float qx[HO_BATCH], qy[HO_BATCH], qz[HO_BATCH];
        int self[HO_BATCH];
        Top2 t[HO_BATCH];
#pragma unroll
        for (int k = 0; k < HO_BATCH; ++k) {
            const float4 q = v.handoff[min(f0 + k, n - 1)];
            qx[k] = q.x; qy[k] = q.y; qz[k] = q.z; self[k] = __float_as_int(q.w);
            t[k].init();
        }
        for (int r = r0 + threadIdx.x; r < r1; r += HO_THREADS) {
            float x, y, z = 0.f;
            int j;
            if (r >= N) {
                j = mlist[r - N];
                const float4 o = v.opos[j];
                x = o.x; y = o.y; z = o.z;
            } else if (D == 2) {
                const float2 o = v.spos2[r];
                x = o.x; y = o.y; j = v.sidx[r];
            } else {
                const float4 o = v.spos4[r];
                x = o.x; y = o.y; z = o.z; j = __float_as_int(o.w);
            }
#pragma unroll
            for (int k = 0; k < HO_BATCH; ++k) {
                const float s = D == 2 ? sqd2(qx[k], qy[k], x, y) : sqd3(qx[k], qy[k], qz[k], x, y, z);
                insert_bf(t[k], s, j, j >= 0 && j != self[k]);
            }
        }
#pragma unroll
        for (int k = 0; k < HO_BATCH; ++k) {
            float sa, sb;
            int ja, jb;
            warp_pop(t[k], sa, ja);
            warp_pop(t[k], sb, jb);
            if (lane == 0) { s_s[k][2 * w] = sa; s_j[k][2 * w] = ja; s_s[k][2 * w + 1] = sb; s_j[k][2 * w + 1] = jb; }
        }
        __syncthreads();
        if (threadIdx.x < HO_BATCH && f0 + threadIdx.x < n) {
            const int k = threadIdx.x;
            Top2 best;
            best.init();
            for (int e = 0; e < 2 * HO_THREADS / 32; ++e)
                if (s_j[k][e] != KC_NOIDX) best.offer(s_s[k][e], s_j[k][e]);
            HandoffPart o;
            o.s1 = best.s1; o.s2 = best.s2; o.j1 = best.j1; o.j2 = best.j2;
            part[(size_t)(f0 + k) * nb + blockIdx.x] = o;
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicAdd(&ctr->ticket3, 1) == nb - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    for (int f = threadIdx.x; f < n; f += HO_THREADS) {
        Top2 best;
        best.init();
        for (int b = 0; b < nb; ++b) {
            const HandoffPart o = part[(size_t)f * nb + b];
            if (o.j1 != KC_NOIDX) best.offer(o.s1, o.j1);
            if (o.j2 != KC_NOIDX) best.offer(o.s2, o.j2);
        }
        store_cert(best, __float_as_int(v.handoff[f].w), nn, nn2, d1, d2, c);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        ctr->n_handed += n;
        ctr->n_handoff = 0;
        ctr->ticket3 = 0;
    }
}
// Grids that hand off (kc_grid.cuh): the view carries the list, and the pass runs behind the search
// kernels of the call (it returns at once when the list is empty).
inline bool hands_off(const kc_grid *g) { return g->N >= HANDOFF_MIN_N && g->handoff != nullptr; }
inline void view_handoff(const kc_grid *g, View &v)
{
    if (hands_off(g)) { v.handoff = g->handoff; v.n_handoff = &g->ctr->n_handoff; }
}
inline void launch_handoff(const kc_grid *g, const View &v, int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c,
                           cudaStream_t st)
{
    if (!hands_off(g)) return;
    if (g->geom.d == 2)
        handoff_kernel<2><<<HANDOFF_BLOCKS, HO_THREADS, 0, st>>>(v, (int)g->N, g->mlist, g->ctr, g->handoff_part, nn, nn2, d1, d2, c);
    else
        handoff_kernel<3><<<HANDOFF_BLOCKS, HO_THREADS, 0, st>>>(v, (int)g->N, g->mlist, g->ctr, g->handoff_part, nn, nn2, d1, d2, c);
    count_launches(1);
}
}  // namespace

extern "C" kc_status kc_cert_grid_search(kc_grid *g, int32_t *nn, int32_t *nn2, float *d1, float *d2,
                                         float *c, void *stream)
{
    if (!g) { set_error("kc_cert_grid_search: NULL grid"); return KC_EINVAL; }
    kc_status s = check_certs(nn, d1, d2, c, "kc_cert_grid_search");
    if (s != KC_OK) return s;
    if (!g->built || g->dirty) {
        set_error("kc_cert_grid_search: grid is not freshly built");
        return KC_EREBUILD;
    }
    cudaStream_t st = (cudaStream_t)stream;
    View v = make_view(g);
    view_handoff(g, v);
    const int n = (int)g->N;
    const int nb = (n + PS_THREADS - 1) / PS_THREADS, tb = 32 * WT_WARPS;
    if (g->geom.d == 2) search_tiled_kernel<2, false, true><<<(n + tb - 1) / tb, tb, 0, st>>>(v, n, g->ctr, nullptr, nullptr, 0, nn, nn2, d1, d2, c);
    else {
        search_leaf_kernel<3, 0><<<nb, PS_THREADS, 0, st>>>(v, n, g->ctr, nullptr, nullptr, 0, nn, nn2, d1, d2, c);
        if (n >= DEFER_MIN_N) {
            ball_finish_kernel<3><<<bf_blocks(n), PS_THREADS, 0, st>>>(v, n, g->ctr, 0, nn, nn2, d1, d2, c);
            count_launches(1);
        }
    }
    count_launches(1);
    launch_handoff(g, v, nn, nn2, d1, d2, c, st);
    KC_LAUNCH_CHECK("kc_cert_grid_search");
    return KC_OK;
}

extern "C" kc_status kc_cert_grid_rebuild(kc_grid *g, const float *p, int64_t N, int32_t *nn,
                                          int32_t *nn2, float *d1, float *d2, float *c, void *stream)
{
    kc_status s = check_certs(nn, d1, d2, c, "kc_cert_grid_rebuild");
    if (s != KC_OK) return s;
    s = kc_grid_build(g, p, N, stream);
    if (s != KC_OK) return s;
    return kc_cert_grid_search(g, nn, nn2, d1, d2, c, stream);
}

extern "C" kc_status kc_cert_grid_topk(kc_grid *g, int K, int32_t *nnk, float *dk, float *ck, void *stream)
{
    if (!g || !nnk || !dk || !ck || K < 2 || K > KC_TOPK_MAX) {
        set_error("kc_cert_grid_topk: bad argument (need grid, nnk, dk, ck, 2 <= K <= %d)", KC_TOPK_MAX);
        return KC_EINVAL;
    }
    if (!g->built || g->dirty) {
        set_error("kc_cert_grid_topk: grid is not freshly built");
        return KC_EREBUILD;
    }
    const View v = make_view(g);
    if (g->geom.d == 2) dispatch_grid_topk<2>(K, v, (int)g->N, nnk, dk, ck, (cudaStream_t)stream);
    else dispatch_grid_topk<3>(K, v, (int)g->N, nnk, dk, ck, (cudaStream_t)stream);
    count_launches(1);
    KC_LAUNCH_CHECK("kc_cert_grid_topk");
    return KC_OK;
}

extern "C" kc_status kc_frontier_search_topk(kc_grid *g, const float *p_new, int64_t N, const int32_t *F,
                                             const int32_t *nF, int64_t nF_max, int K, int32_t *nnk, float *dk,
                                             float *ck, void *stream)
{
    if (!g || !p_new || !F || !nF || nF_max < 0 || !nnk || !dk || !ck || K < 2 || K > KC_TOPK_MAX) {
        set_error("kc_frontier_search_topk: bad argument (2 <= K <= %d)", KC_TOPK_MAX);
        return KC_EINVAL;
    }
    if (!g->built || N != g->N) {
        set_error("kc_frontier_search_topk: grid not built for this N");
        return KC_EREBUILD;
    }
    if (nF_max == 0) return KC_OK;
    const View v = make_view(g);
    if (g->geom.d == 2) dispatch_list_topk<2>(K, v, p_new, F, nF, nF_max, g->ctr, nnk, dk, ck, (cudaStream_t)stream);
    else dispatch_list_topk<3>(K, v, p_new, F, nF, nF_max, g->ctr, nnk, dk, ck, (cudaStream_t)stream);
    count_launches(1);
    KC_LAUNCH_CHECK("kc_frontier_search_topk");
    return KC_OK;
}

// A7, Algorithm 1 lines 4-7: re-search the frontier only.  On a large grid a
// frontier of at least N / sweep_div points (decided on the device from *nF) is served in slot
// order by the tiled sweep, anything else straight from the id list (one warp per query while the
// list is short: latency; one thread per query when it is long: throughput); both kernels are
// launched when the host bound allows either.
extern "C" kc_status kc_frontier_search(kc_grid *g, const float *p_new, int64_t N, const int32_t *F,
                                        const int32_t *nF, int64_t nF_max, int32_t *nn, int32_t *nn2,
                                        float *d1, float *d2, float *c, void *stream)
{
    if (!g || !p_new || !F || !nF || nF_max < 0) {
        set_error("kc_frontier_search: bad argument");
        return KC_EINVAL;
    }
    kc_status s = check_certs(nn, d1, d2, c, "kc_frontier_search");
    if (s != KC_OK) return s;
    if (!g->built || N != g->N) {
        set_error("kc_frontier_search: grid not built for this N");
        return KC_EREBUILD;
    }
    if (nF_max == 0) return KC_OK;
    cudaStream_t st = (cudaStream_t)stream;
    View v = make_view(g);
    view_handoff(g, v);
    const int n = (int)N;
    // slot sweep: grids of at least SWEEP_MIN_N points, frontier of at least N / div points
    // (the host bound decides whether the sweep kernels are launched, the device count whether they run)
    const int div = g->geom.d == 2 ? SWEEP_DIV2 : list_div3(N);
    const int sweep_div = N >= SWEEP_MIN_N && nF_max * (int64_t)div >= N ? div : 0;
    if (sweep_div > 0) {
        mark_frontier_kernel<<<blocks_for(nF_max, 256, 148 * 8), 256, 0, st>>>(F, nF, n, sweep_div, g->slot, g->mark, g->list2, g->ctr);
        // a grid that is fresh (built or re-binned, not updated incrementally) has no tombstones and
        // no chains: the sweep then is the whole-set kernel with a query mask.  d = 3: two launches, of
        // which the device runs one: a frontier of more than 45 % of the points is served slot by slot,
        // a thinner one by the compacting instantiation (a warp owns >= 64 slots there: a smaller grid).
        // (d = 2: compaction measured no gain on the row-segment kernel, 0.43 vs 0.45 ms at 12.5 %.)
        const int tb = 32 * WT_WARPS, nbt = (n + tb - 1) / tb;
        const int nb = (n + PS_THREADS - 1) / PS_THREADS, nb2 = (n + 2 * PS_THREADS - 1) / (2 * PS_THREADS);
        if (g->geom.d == 2) {
            if (g->dirty) search_tiled_kernel<2, true, false><<<nbt, tb, 0, st>>>(v, n, g->ctr, g->mark, nF, sweep_div, nn, nn2, d1, d2, c);
            else search_tiled_kernel<2, true, true><<<nbt, tb, 0, st>>>(v, n, g->ctr, g->mark, nF, sweep_div, nn, nn2, d1, d2, c);
        } else {
            // (a list buffer too short for the direct kernel's density does not launch it)
            const bool direct = 20 * nF_max > 9 * N;
            if (g->dirty) {
                if (direct) search_leaf_kernel<3, 1><<<nb, PS_THREADS, 0, st>>>(v, n, g->ctr, g->mark, nF, sweep_div, nn, nn2, d1, d2, c);
                search_leaf_kernel<3, 3><<<nb2, PS_THREADS, 0, st>>>(v, n, g->ctr, g->mark, nF, sweep_div, nn, nn2, d1, d2, c);
            } else {
                if (direct) search_leaf_kernel<3, 2><<<nb, PS_THREADS, 0, st>>>(v, n, g->ctr, g->mark, nF, sweep_div, nn, nn2, d1, d2, c);
                search_leaf_kernel<3, 4><<<nb2, PS_THREADS, 0, st>>>(v, n, g->ctr, g->mark, nF, sweep_div, nn, nn2, d1, d2, c);
            }
            ball_finish_kernel<3><<<bf_blocks(n), PS_THREADS, 0, st>>>(v, n, g->ctr, g->dirty ? 1 : 0, nn, nn2, d1, d2, c);   // (n >= SWEEP_MIN_N >= DEFER_MIN_N)
            count_launches(direct ? 2 : 1);
        }
        count_launches(2);
    }
    int blocks = blocks_for(nF_max, 4, 148 * 16);          // short list: one warp per query
    if (nF_max > WPQ_MAX) blocks = max(blocks, blocks_for(nF_max, 128, 148 * 32));
    if (g->geom.d == 2)
        search_wpq_kernel<2><<<blocks, 128, 0, st>>>(v, p_new, n, F, nF, g->list2, sweep_div, g->ctr, nn, nn2, d1, d2, c);
    else
        search_wpq_kernel<3><<<blocks, 128, 0, st>>>(v, p_new, n, F, nF, g->list2, sweep_div, g->ctr, nn, nn2, d1, d2, c);
    count_launches(1);
    launch_handoff(g, v, nn, nn2, d1, d2, c, st);
    KC_LAUNCH_CHECK("kc_frontier_search");
    return KC_OK;
}

// A6 + A7 in one call.
extern "C" kc_status kc_frontier_repair(kc_grid *g, const float *p_new, int64_t N, const int32_t *movers,
                                        const int32_t *n_movers, int64_t n_movers_max, const int32_t *F,
                                        const int32_t *nF, int64_t nF_max, int32_t *nn, int32_t *nn2,
                                        float *d1, float *d2, float *c, void *stream)
{
    if (!F || !nF || nF_max < 0) {
        set_error("kc_frontier_repair: bad argument");
        return KC_EINVAL;
    }
    kc_status s = check_certs(nn, d1, d2, c, "kc_frontier_repair");
    if (s != KC_OK) return s;
    s = kc_grid_update(g, p_new, N, movers, n_movers, n_movers_max, stream);
    if (s != KC_OK) return s;
    return kc_frontier_search(g, p_new, N, F, nF, nF_max, nn, nn2, d1, d2, c, stream);
}
