// kc_allpairs.cu — A1: exact all-pairs top-2 ("exact N x N pass", Table 2
// PAPER.md:116-125) and the query-subset variant (PAPER.md:69 rtx_frontier_oracle).
//
// FP32 CUDA-core kernel (no tensor cores: d = 2/3 is not a dense contraction and the
// |x|^2 - 2x.y form would break bit-exactness; no FMA: the contract forbids contraction).
//   * a CTA owns QPT*128 query points (register tile: QPT queries per thread) and one j-chunk;
//   * j-tiles of TJ points are staged in shared memory as SoA (x[], y[], z[]) so that every
//     lane reads the same address (broadcast, conflict-free) and one LDS.128 feeds 4 candidates;
//   * fast path per (query, 4 candidates): 4 distances, min of them, ONE compare against the
//     current second-best; the exact (s, j)-ordered insertion (ties, self, tail) runs only in the
//     rarely taken slow path (~2 ln N times per query);
//   * j is split across gridDim.y so small N still fills 148 SMs; the CTA that finishes a query
//     block's last chunk merges the partial top-2s under the same total order, so the split never
//     changes a result;
//   * when j is split, a seed pass first gives every query its exact top-2 over the first AP_SEED
//     points (warp-cooperative, branch-free), and every chunk starts from that instead of from
//     +inf: a chunk that starts cold pays ~2 ln(chunk) insertions per lane, and with 32 independent
//     lanes that puts some lane on the insertion path in almost every step of a short chunk.
#include <stdlib.h>

#include <atomic>

#include "kc_common.cuh"

using namespace kc;

namespace {

constexpr int AP_TJ = 1152;   // candidates per shared-memory tile (= one j-chunk of the N = 16,000 step: 18 units of AP_GRAN)
constexpr int AP_SEED = 256;  // points scanned by the seed pass of a j-split launch
constexpr int AP_GRAN = 64;   // chunk granularity of a j-split launch (a multiple of every step size 4*C4)
constexpr int AP_TICKETS = 148 * 8 * 8;   // a j-split launch has fewer query blocks than this (choose_shape)
constexpr int AP_RESIDENT = 12;   // CTAs of 128 threads an SM holds at the kernel's ~48 registers per thread

struct Partial { float s1, s2; int j1, j2; };   // 16 B

typedef unsigned long long u64;

// Packed FP32x2 arithmetic (sm_100a FADD2 / FMUL2 / FFMA2): two separately rounded binary32
// operations per instruction, so the issue slots per pair halve while every result keeps the
// contract's rounding.  ptxas contracts mul.rn.f32x2 + add.rn.f32x2 into FFMA2 even under
// -fmad=false, which would break bit-exactness; the sum is therefore written as
// fma(xx, 1.0, yy) with the 1.0 pair passed at run time: xx*1.0 is exact, so the result is
// round(xx + yy), and a product cannot be folded into the addend of an FMA.
__device__ __forceinline__ u64 sub2(u64 a, u64 b)
{
    u64 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ u64 sqr2(u64 a)
{
    u64 d;
    asm("mul.rn.f32x2 %0, %1, %1;" : "=l"(d) : "l"(a));
    return d;
}
__device__ __forceinline__ u64 addvia1(u64 a, u64 one, u64 b)
{
    u64 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(one), "l"(b));
    return d;
}
__device__ __forceinline__ u64 pack2(float lo, float hi)
{
    u64 d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(lo), "f"(hi));
    return d;
}
__device__ __forceinline__ void unpack2(u64 v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}

template <int D, int THREADS>
__device__ __forceinline__ void load_tile(const float *__restrict__ p, int64_t N, int64_t j0, int tl,
                                          float *sx, float *sy, float *sz)
{
    // pad the tail with +inf: s = +inf never beats a finite second-best, and the slow path
    // rejects j >= N explicitly while second-best is still +inf.
    for (int t = threadIdx.x; t < tl; t += THREADS) {
        int64_t j = j0 + t;
        float x = CUDART_INF_F, y = CUDART_INF_F, z = CUDART_INF_F;
        if (j < N) {
            if (D == 2) {
                float2 v = reinterpret_cast<const float2 *>(p)[j];
                x = v.x; y = v.y;
            } else {
                x = p[j * 3 + 0]; y = p[j * 3 + 1]; z = p[j * 3 + 2];
            }
        }
        sx[t] = x; sy[t] = y;
        if (D == 3) sz[t] = z;
    }
}

// exact (s, j)-ordered insertion of the 4 candidates j..j+3 (rare path)
__device__ __noinline__ Top2 slow_offer4(Top2 best, float s0, float s1, float s2, float s3, int j,
                                         int lim, int self)
{
    // ids already held are skipped: a list seeded from two known points meets them again
    if (s0 <= best.s2 && j + 0 < lim && j + 0 != self && j + 0 != best.j1 && j + 0 != best.j2) best.offer(s0, j + 0);
    if (s1 <= best.s2 && j + 1 < lim && j + 1 != self && j + 1 != best.j1 && j + 1 != best.j2) best.offer(s1, j + 1);
    if (s2 <= best.s2 && j + 2 < lim && j + 2 != self && j + 2 != best.j1 && j + 2 != best.j2) best.offer(s2, j + 2);
    if (s3 <= best.s2 && j + 3 < lim && j + 3 != self && j + 3 != best.j1 && j + 3 != best.j2) best.offer(s3, j + 3);
    return best;
}

// QPT queries per thread against candidates [jbeg, jend), C4 groups of 4 candidates per step.
// One step evaluates QPT*C4*4 pairs straight-line (packed FP32x2), reduces each group to its
// minimum, ORs the QPT*C4 "min <= second-best" predicates and branches ONCE; the exact
// insertion runs only behind that branch.  qi[k] = -1 marks a padding query.
template <int D, int QPT, int C4, int THREADS>
__device__ __forceinline__ void scan_chunk(const float *__restrict__ p, int64_t N, int64_t jbeg,
                                           int64_t jend, const float (&qx)[QPT],
                                           const float (&qy)[QPT], const float (&qz)[QPT],
                                           const int (&qi)[QPT], Top2 (&best)[QPT], float *sx,
                                           float *sy, float *sz, u64 one2)
{
    const int lim = (int)min(N, jend);
    u64 qx2[QPT], qy2[QPT], qz2[QPT];
#pragma unroll
    for (int k = 0; k < QPT; ++k) {
        qx2[k] = pack2(qx[k], qx[k]); qy2[k] = pack2(qy[k], qy[k]); qz2[k] = pack2(qz[k], qz[k]);
    }
    for (int64_t j0 = jbeg; j0 < jend; j0 += AP_TJ) {
        // the chunk's last tile may be short: only whole steps of it are staged and evaluated
        const int tl = (int)min((int64_t)AP_TJ, (jend - j0 + 4 * C4 - 1) / (4 * C4) * (4 * C4));
        __syncthreads();
        load_tile<D, THREADS>(p, lim, j0, tl, sx, sy, sz);
        __syncthreads();
#pragma unroll 1
        for (int t = 0; t < tl; t += 4 * C4) {
            u64 sa[QPT][C4], sb[QPT][C4];
            float m[QPT][C4];
#pragma unroll
            for (int g = 0; g < C4; ++g) {
                const ulonglong2 X = *reinterpret_cast<const ulonglong2 *>(sx + t + 4 * g);
                const ulonglong2 Y = *reinterpret_cast<const ulonglong2 *>(sy + t + 4 * g);
                ulonglong2 Z = make_ulonglong2(0, 0);
                if (D == 3) Z = *reinterpret_cast<const ulonglong2 *>(sz + t + 4 * g);
#pragma unroll
                for (int k = 0; k < QPT; ++k) {
                    u64 a = addvia1(sqr2(sub2(qx2[k], X.x)), one2, sqr2(sub2(qy2[k], Y.x)));
                    u64 b = addvia1(sqr2(sub2(qx2[k], X.y)), one2, sqr2(sub2(qy2[k], Y.y)));
                    if (D == 3) {
                        a = addvia1(a, one2, sqr2(sub2(qz2[k], Z.x)));
                        b = addvia1(b, one2, sqr2(sub2(qz2[k], Z.y)));
                    }
                    sa[k][g] = a; sb[k][g] = b;
                    float s0, s1, s2, s3;
                    unpack2(a, s0, s1);
                    unpack2(b, s2, s3);
                    m[k][g] = fminf(fminf(s0, s1), fminf(s2, s3));
                }
            }
            bool any = false;
#pragma unroll
            for (int k = 0; k < QPT; ++k)
#pragma unroll
                for (int g = 0; g < C4; ++g) any |= (m[k][g] <= best[k].s2);
            if (any) {
#pragma unroll
                for (int k = 0; k < QPT; ++k)
#pragma unroll
                    for (int g = 0; g < C4; ++g)
                        if (m[k][g] <= best[k].s2) {
                            float s0, s1, s2, s3;
                            unpack2(sa[k][g], s0, s1);
                            unpack2(sb[k][g], s2, s3);
                            best[k] = slow_offer4(best[k], s0, s1, s2, s3, (int)(j0 + t + 4 * g), lim, qi[k]);
                        }
            }
        }
    }
}

// Everything a launch needs; passed by value.
struct ApArgs {
    const float *p;
    int64_t N;
    const int32_t *qlist;        // null: queries are 0..N-1
    const int32_t *nq_dev;       // null: nq_host queries
    int64_t nq_host;
    int64_t jchunk, jfirst;      // chunk y scans candidates [jfirst + y*jchunk, +jchunk)
    u64 one2;
    const Partial *seed;         // unbounded j-split: exact top-2 over points [0, jfirst)
    const float *bound_d2;       // kinetic bound (both or neither): every query's second neighbour is
    const float *bound_eps;      //   claimed to lie within bound_d2[i] + 2 * bound_eps[0]
    const int32_t *seed1, *seed2;   // two known points per query (e.g. its previous neighbours), or null
    Partial *part;               // j-split: partial lists [js][nq_host]; null: store certificates
    int32_t *redo, *n_redo;      // queries whose bound admitted fewer than two candidates
    int32_t *tickets;            // j-split: chunks finished per query block (the last one merges and re-zeroes)
    int *errword;                // device error word (kc_common.cuh), or null
    int32_t *nn, *nn2;
    float *d1, *d2, *c;
};

// j-split: the CTA that finishes the last chunk of a query block merges the block's partial lists.
// The counters live in a fixed area at the head of the workspace that holds nothing else, start
// at zero (workspace contract, kc.h) and are put back to zero by the last arrival, so no call has
// to clear them (a memset node or a kernel in front of the pass costs 3-5 us of a 70 us launch).
// A count that cannot occur in a clean area (the caller broke the workspace contract) is reported
// through the device error word and the counter is put back to zero; nothing is merged for that
// query block, so its certificates are unspecified, but the context stays usable (no trap) and the
// next all-pairs call returns KC_EINVAL (run()).
__device__ __forceinline__ bool take_ticket(int32_t *t, int total, int *errword)
{
    const int old = atomicAdd(t, 1);
    if (old < 0 || old >= total) {
        if (errword) *reinterpret_cast<volatile int *>(errword) = KC_DEVERR_TICKETS;
        atomicExch(t, 0);
        return false;
    }
    const bool last = old == total - 1;
    if (last) atomicExch(t, 0);
    return last;
}

// grid = (ceil(nq / (QPT*THREADS)), JS).
template <int D, int QPT, int C4, int THREADS>
__global__ void __launch_bounds__(THREADS, (QPT == 1 && THREADS == 128) ? 12 : 1)
allpairs_kernel(const ApArgs a)
{
    __shared__ __align__(16) float sx[AP_TJ];
    __shared__ __align__(16) float sy[AP_TJ];
    __shared__ __align__(16) float sz[D == 3 ? AP_TJ : 4];
    const float *__restrict__ p = a.p;
    const int64_t nq = a.nq_dev ? (int64_t)*a.nq_dev : a.nq_host;
    const int64_t q0 = blockIdx.x * (int64_t)(QPT * THREADS);
    if (q0 >= nq) return;
    float qx[QPT], qy[QPT], qz[QPT];
    int qi[QPT];
    Top2 best[QPT];
    const float eps2 = a.bound_d2 ? 2.0f * a.bound_eps[0] : 0.f;
#pragma unroll
    for (int k = 0; k < QPT; ++k) {
        int64_t q = q0 + k * THREADS + threadIdx.x;
        int i = -1;
        if (q < nq) i = a.qlist ? a.qlist[q] : (int)q;
        qi[k] = i;
        qx[k] = qy[k] = qz[k] = 0.f;
        best[k].init();
        if (i >= 0) {
            qx[k] = p[(int64_t)i * D + 0];
            qy[k] = p[(int64_t)i * D + 1];
            if (D == 3) qz[k] = p[(int64_t)i * D + 2];
            if (a.seed) {                         // exact top-2 over points [0, jfirst)
                const int4 raw = reinterpret_cast<const int4 *>(a.seed)[q];
                best[k].s1 = __int_as_float(raw.x); best[k].s2 = __int_as_float(raw.y);
                best[k].j1 = raw.z; best[k].j2 = raw.w;
            }
            if (a.seed1) {
                // kc_cert_allpairs_seeded: the exact keys, at the CURRENT positions, of two known
                // points (e.g. the previous neighbours).  Two distinct points other than i at
                // squared distances s_a <= s_b prove s2_i <= s_b, so this start can never be
                // wrong; ids out of range, equal to i or to each other are dropped, and a NaN
                // coordinate seeds nothing.  Every chunk of a j-split starts from the same two.
                const int ids[2] = {a.seed1[i], a.seed2[i]};
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int j = ids[e];
                    if (j >= 0 && j < a.N && j != i && j != best[k].j1) {
                        const float s = D == 2 ? sqd2(qx[k], qy[k], p[(int64_t)j * D], p[(int64_t)j * D + 1])
                                               : sqd3(qx[k], qy[k], qz[k], p[(int64_t)j * D], p[(int64_t)j * D + 1],
                                                      p[(int64_t)j * D + 2]);
                        if (s == s) best[k].offer(s, j);
                    }
                }
            }
            if (a.bound_d2) {
                // start from two placeholders (T, no index): candidates beyond T are never
                // inserted; T is inflated by 2^-9, far above every rounding on the way
                const float b = (a.bound_d2[i] + eps2) * 1.001953125f;
                best[k].s1 = best[k].s2 = b * b;
            }
        }
    }
    const int64_t jbeg = a.jfirst + blockIdx.y * a.jchunk;
    const int64_t jend = min(a.N, jbeg + a.jchunk);
    scan_chunk<D, QPT, C4, THREADS>(p, a.N, jbeg, jend, qx, qy, qz, qi, best, sx, sy, sz, a.one2);
    if (a.part) {
        // j-split: publish this chunk's partial lists; the CTA that takes the last ticket of the
        // query block merges all of them (they are read through L2: other SMs wrote them)
#pragma unroll
        for (int k = 0; k < QPT; ++k) {
            int64_t q = q0 + k * THREADS + threadIdx.x;
            if (qi[k] < 0) continue;
            Partial o;
            o.s1 = best[k].s1; o.s2 = best[k].s2; o.j1 = best[k].j1; o.j2 = best[k].j2;
            a.part[blockIdx.y * a.nq_host + q] = o;
        }
        __shared__ int s_last;
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) s_last = take_ticket(&a.tickets[blockIdx.x], (int)gridDim.y, a.errword);
        __syncthreads();
        if (!s_last) return;
        __threadfence();
#pragma unroll
        for (int k = 0; k < QPT; ++k) {
            int64_t q = q0 + k * THREADS + threadIdx.x;
            if (qi[k] < 0) continue;
            Top2 t;
            t.init();
            // every list starts from the same seed entries (or placeholders): skip ids already
            // held and entries without an index
            for (int y = 0; y < (int)gridDim.y; ++y) {
                const int4 raw = __ldcg(reinterpret_cast<const int4 *>(a.part) + (y * a.nq_host + q));
                const float s1 = __int_as_float(raw.x), s2 = __int_as_float(raw.y);
                if (raw.z != KC_NOIDX && raw.z != t.j1 && raw.z != t.j2) t.offer(s1, raw.z);
                if (raw.w != KC_NOIDX && raw.w != t.j1 && raw.w != t.j2) t.offer(s2, raw.w);
            }
            best[k] = t;
        }
    }
#pragma unroll
    for (int k = 0; k < QPT; ++k) {
        if (qi[k] < 0) continue;
        if (a.bound_d2 && best[k].j2 == KC_NOIDX) a.redo[atomicAdd(a.n_redo, 1)] = qi[k];
        else store_cert(best[k], qi[k], a.nn, a.nn2, a.d1, a.d2, a.c);
    }
}

// Seed pass: one warp per query at a time, the 32 lanes take different candidates of [0, S) and
// keep a private top-2 with branch-free selects; two warp reductions pick the two smallest keys.
template <int D>
__global__ void __launch_bounds__(256)
allpairs_seed_kernel(const ApArgs a, int S, Partial *__restrict__ seed)
{
    __shared__ float sx[AP_SEED], sy[AP_SEED], sz[D == 3 ? AP_SEED : 1];
    const float *__restrict__ p = a.p;
    for (int t = threadIdx.x; t < S; t += blockDim.x) {
        sx[t] = p[(int64_t)t * D]; sy[t] = p[(int64_t)t * D + 1];
        if (D == 3) sz[t] = p[(int64_t)t * D + 2];
    }
    __syncthreads();
    const int64_t nq = a.nq_dev ? (int64_t)*a.nq_dev : a.nq_host;
    const int lane = threadIdx.x & 31;
    const int64_t w0 = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int64_t nw = ((int64_t)gridDim.x * blockDim.x) >> 5;
    for (int64_t q = w0; q < nq; q += nw) {
        const int i = a.qlist ? a.qlist[q] : (int)q;
        const float qx = p[(int64_t)i * D], qy = p[(int64_t)i * D + 1];
        const float qz = D == 3 ? p[(int64_t)i * D + 2] : 0.f;
        Top2 tmp;
        tmp.init();
        for (int t = lane; t < S; t += 32) {
            const float s = D == 2 ? sqd2(qx, qy, sx[t], sy[t]) : sqd3(qx, qy, qz, sx[t], sy[t], sz[t]);
            insert_bf(tmp, s, t, t != i);
        }
        Partial o;
        warp_pop(tmp, o.s1, o.j1);
        warp_pop(tmp, o.s2, o.j2);
        if (lane == 0) seed[q] = o;
    }
}

// Redo pass of a bounded launch: the queries whose bound admitted fewer than two candidates (a
// bound that was not one) are recomputed from scratch, one CTA per query, so that the result
// never depends on the bound.  Empty in normal operation.
template <int D>
__global__ void __launch_bounds__(256)
allpairs_redo_kernel(const ApArgs a)
{
    __shared__ float ws[8][2];
    __shared__ int wj[8][2];
    const float *__restrict__ p = a.p;
    const int n = *a.n_redo;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int r = blockIdx.x; r < n; r += gridDim.x) {
        const int i = a.redo[r];
        const float qx = p[(int64_t)i * D], qy = p[(int64_t)i * D + 1];
        const float qz = D == 3 ? p[(int64_t)i * D + 2] : 0.f;
        Top2 tmp;
        tmp.init();
        for (int64_t t = threadIdx.x; t < a.N; t += 256) {
            const float s = D == 2 ? sqd2(qx, qy, p[t * D], p[t * D + 1])
                                   : sqd3(qx, qy, qz, p[t * D], p[t * D + 1], p[t * D + 2]);
            insert_bf(tmp, s, (int)t, t != i);
        }
        float s1, s2;
        int j1, j2;
        warp_pop(tmp, s1, j1);
        warp_pop(tmp, s2, j2);
        if (lane == 0) { ws[warp][0] = s1; ws[warp][1] = s2; wj[warp][0] = j1; wj[warp][1] = j2; }
        __syncthreads();
        if (threadIdx.x == 0) {
            Top2 t;
            t.init();
            for (int w = 0; w < 8; ++w) {
                if (wj[w][0] != KC_NOIDX) t.offer(ws[w][0], wj[w][0]);
                if (wj[w][1] != KC_NOIDX) t.offer(ws[w][1], wj[w][1]);
            }
            store_cert(t, i, a.nn, a.nn2, a.d1, a.d2, a.c);
        }
        __syncthreads();
    }
}

// Launch shape (a function of the sizes only).
struct Shape { int qpt, c4, threads, js; };

Shape choose_shape(int64_t nq, int64_t N)
{
    Shape s;
    s.qpt = nq >= 148 * 8 * 128 * 2 ? 4 : (nq >= 148 * 4 * 128 ? 2 : 1);
    s.threads = 128;
    s.c4 = s.qpt == 4 ? 2 : (s.qpt == 2 ? 2 : 4);
    // j-split (chunks start from the seed pass or from the caller's bound, so short chunks are
    // fine; granularity AP_GRAN candidates, at least 4 units per chunk).  Few query blocks: as many
    // chunks as make ONE full wave of resident CTAs (a second, partly filled wave of this
    // latency-bound kernel would cost as much as a full one).  Many query blocks: many waves deep.
    int64_t per = (int64_t)s.qpt * s.threads;
    int64_t itiles = (nq + per - 1) / per;
    const int64_t resident = 148 * (int64_t)AP_RESIDENT;
    int64_t want = itiles * 2 <= resident ? resident / itiles : (148 * 8 * 8 + itiles - 1) / itiles;
    int64_t cap = (N - AP_SEED) / (4 * AP_GRAN);
    int64_t js = want < cap ? want : cap;
    if (js < 1) js = 1;
    if (js > 65535) js = 65535;
    if (itiles > AP_TICKETS) js = 1;             // the ticket area holds AP_TICKETS query blocks
    s.js = (int)js;
    return s;
}

// Workspace layout: [n_redo: 16 B][tickets: AP_TICKETS int32, a fixed area that holds nothing
// else][redo ids: nq int32, padded to 16 B][seed: nq][part: js x nq] (the last only for a j-split
// shape).  n_redo is zeroed by a memset in a bounded call; the tickets are zero between calls
// (take_ticket; the caller zero-fills a new workspace once, kc.h).
size_t pad16(size_t b) { return (b + 15) & ~(size_t)15; }
size_t head_bytes(int64_t, const Shape &) { return 16 + (size_t)AP_TICKETS * 4; }
size_t workspace_bytes_for(int64_t nq, const Shape &sh)
{
    return head_bytes(nq, sh) + pad16((size_t)nq * 4) + (size_t)nq * sizeof(Partial) +
           (sh.js > 1 ? (size_t)sh.js * (size_t)nq * sizeof(Partial) : 0);
}

template <int D, int QPT, int C4>
void launch_t(int threads, dim3 grid, cudaStream_t st, const ApArgs &a)
{
    (void)threads;
    allpairs_kernel<D, QPT, C4, 128><<<grid, 128, 0, st>>>(a);
}

template <int D>
kc_status launch(ApArgs a, char *ws, Shape sh, cudaStream_t st, int *errword = nullptr)
{
    const int64_t nq = a.nq_host;
    const bool split = sh.js > 1, bounded = a.bound_d2 != nullptr;
    a.one2 = 0x3f8000003f800000ull;
    a.n_redo = reinterpret_cast<int32_t *>(ws);
    a.tickets = reinterpret_cast<int32_t *>(ws + 16);
    a.errword = errword ? errword : error_word_dev();
    a.redo = reinterpret_cast<int32_t *>(ws + head_bytes(nq, sh));
    Partial *seed = reinterpret_cast<Partial *>(ws + head_bytes(nq, sh) + pad16((size_t)nq * 4));
    const bool idseed = a.seed1 != nullptr;
    if (bounded) KC_CUDA(cudaMemsetAsync(ws, 0, 16, st));
    a.jfirst = split && !bounded && !idseed ? AP_SEED : 0;
    int js = sh.js;
    int64_t jchunk;
    if (split) {
        // equal chunks of whole AP_GRAN units, as many as the shape wants
        const int64_t units = (a.N - a.jfirst + AP_GRAN - 1) / AP_GRAN;
        const int64_t want = js < units ? js : units;
        jchunk = (units + want - 1) / want * AP_GRAN;
    } else {
        jchunk = (a.N + 15) / 16 * 16;
    }
    js = (int)((a.N - a.jfirst + jchunk - 1) / jchunk);
    a.jchunk = jchunk;
    a.seed = nullptr;
    a.part = split ? seed + nq : nullptr;
    int launches = 1;
    if (idseed) {
        // seeds are computed in the pass itself
    } else if (split && !bounded) {
        const int blocks = (int)((nq + 7) / 8 < 148 * 8 ? (nq + 7) / 8 : 148 * 8);
        if (D == 2) allpairs_seed_kernel<2><<<blocks, 256, 0, st>>>(a, (int)a.jfirst, seed);
        else allpairs_seed_kernel<3><<<blocks, 256, 0, st>>>(a, (int)a.jfirst, seed);
        a.seed = seed;
        ++launches;
    }
    const int per = sh.qpt * sh.threads;
    dim3 grid((unsigned)((nq + per - 1) / per), (unsigned)js);
#define KC_AP_CASE(Q, C)                                           \
    if (sh.qpt == Q && sh.c4 == C) {                               \
        launch_t<D, Q, C>(sh.threads, grid, st, a);                \
    } else
    KC_AP_CASE(4, 2) KC_AP_CASE(2, 2) KC_AP_CASE(1, 4)
    {
        set_error("kc_cert_allpairs: unsupported launch shape");
        return KC_EINVAL;
    }
#undef KC_AP_CASE
    if (bounded) {
        const int blocks = (int)(nq < 148 * 4 ? nq : 148 * 4);
        if (D == 2) allpairs_redo_kernel<2><<<blocks, 256, 0, st>>>(a);
        else allpairs_redo_kernel<3><<<blocks, 256, 0, st>>>(a);
        ++launches;
    }
    count_launches(launches);
    KC_LAUNCH_CHECK("kc_cert_allpairs");
    return KC_OK;
}

kc_status run(const char *who, const float *p, int64_t N, int d, const int32_t *q, const int32_t *nq_dev,
              int64_t nq, const float *d2_prev, const float *eps, const int32_t *seed1,
              const int32_t *seed2, int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c,
              void *workspace, size_t workspace_bytes, void *stream)
{
    if (!p || !nn || !d1 || !d2 || !c || N < 2 || N > 0x7ffffff0 || (d != 2 && d != 3) ||
        (reinterpret_cast<uintptr_t>(p) & 7) || (d2_prev != nullptr) != (eps != nullptr)) {
        set_error("%s: bad argument", who);
        return KC_EINVAL;
    }
    const Shape sh = choose_shape(nq, N);
    const size_t need = workspace_bytes_for(nq, sh);
    if (!workspace || workspace_bytes < need || (reinterpret_cast<uintptr_t>(workspace) & 15)) {
        set_error("%s: workspace of %zu bytes (16-byte aligned) required", who, need);
        return KC_EINVAL;
    }
    error_word_init();
    if (error_word_take() == KC_DEVERR_TICKETS) {
        // an earlier all-pairs kernel met split counters that a zero-filled workspace cannot hold:
        // its results are unspecified.  Heal the workspace passed now and report; the call is not run.
        KC_CUDA(cudaMemsetAsync(workspace, 0, 16 + (size_t)AP_TICKETS * 4, (cudaStream_t)stream));
        set_error("%s: an earlier all-pairs call was given a workspace that had not been zero-filled "
                  "(kc.h, workspace contract); its certificates are unspecified.  The counters of the "
                  "workspace passed now have been cleared; call again", who);
        return KC_EINVAL;
    }
    ApArgs a = {};
    a.p = p; a.N = N; a.qlist = q; a.nq_dev = nq_dev; a.nq_host = nq;
    a.bound_d2 = d2_prev; a.bound_eps = eps;
    a.seed1 = seed1; a.seed2 = seed2;
    a.nn = nn; a.nn2 = nn2; a.d1 = d1; a.d2 = d2; a.c = c;
    if (d == 2) return launch<2>(a, (char *)workspace, sh, (cudaStream_t)stream);
    return launch<3>(a, (char *)workspace, sh, (cudaStream_t)stream);
}

}  // namespace

extern "C" size_t kc_cert_allpairs_workspace(int64_t N, int d)
{
    if (N < 2 || (d != 2 && d != 3)) return 0;
    error_word_init();
    return workspace_bytes_for(N, choose_shape(N, N));
}

extern "C" kc_status kc_cert_allpairs(const float *p, int64_t N, int d, int32_t *nn, int32_t *nn2,
                                      float *d1, float *d2, float *c, void *workspace,
                                      size_t workspace_bytes, void *stream)
{
    return run("kc_cert_allpairs", p, N, d, nullptr, nullptr, N, nullptr, nullptr, nullptr, nullptr, nn, nn2, d1, d2, c,
               workspace, workspace_bytes, stream);
}

// ---- A1 without any allocation: the workspace is a file-scope device array ---------------------
// For callers that cannot allocate (kc.h).  Every GPU that loads the library holds these 5 MiB until
// exit.  KC_ALLPAIRS_STATIC_MAX_N = 65,536: the largest workspace_bytes_for(N, choose_shape(N, N)) over
// N <= 65,536 is 4,811,792 B (at N = 56,832).
constexpr int64_t AP_STATIC_MAX_N = 65536;
constexpr size_t AP_STATIC_BYTES = 5u << 20;
static __device__ __align__(256) unsigned char g_ap_static_scratch[AP_STATIC_BYTES];

namespace {
// In host code the array's name is a host-side stand-in: its device address is looked up once per
// device, with that device current.
constexpr int AP_MAX_DEVICES = 64;
std::atomic<void *> g_ap_static_ptr[AP_MAX_DEVICES];

kc_status ap_static_address(char **out)
{
    int dev = -1;
    KC_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= AP_MAX_DEVICES) {
        set_error("kc_cert_allpairs_static: device ordinal %d not supported (< %d)", dev, AP_MAX_DEVICES);
        return KC_EINVAL;
    }
    void *ptr = g_ap_static_ptr[dev].load(std::memory_order_acquire);
    if (!ptr) {
        KC_CUDA(cudaGetSymbolAddress(&ptr, g_ap_static_scratch));
        g_ap_static_ptr[dev].store(ptr, std::memory_order_release);
    }
    *out = static_cast<char *>(ptr);
    return KC_OK;
}
}  // namespace

extern "C" int64_t kc_cert_allpairs_static_max_n(void) { return AP_STATIC_MAX_N; }

extern "C" kc_status kc_cert_allpairs_static(const float *p, int64_t N, int d, int32_t *nn, int32_t *nn2,
                                             float *d1, float *d2, float *c, void *stream)
{
    const char *who = "kc_cert_allpairs_static";
    if (!p || !nn || !d1 || !d2 || !c || N < 2 || (d != 2 && d != 3) || (reinterpret_cast<uintptr_t>(p) & 7)) {
        set_error("%s: bad argument", who);
        return KC_EINVAL;
    }
    if (N > AP_STATIC_MAX_N) {
        set_error("%s: N = %lld exceeds the static scratch's maximum of %lld points; use kc_cert_allpairs "
                  "with a caller-allocated workspace", who, (long long)N, (long long)AP_STATIC_MAX_N);
        return KC_EINVAL;
    }
    const Shape sh = choose_shape(N, N);
    const size_t need = workspace_bytes_for(N, sh);
    if (need > AP_STATIC_BYTES) {
        set_error("%s: N = %lld needs %zu bytes of scratch, the static array holds %zu", who, (long long)N, need,
                  (size_t)AP_STATIC_BYTES);
        return KC_EINVAL;
    }
    char *ws = nullptr;
    const kc_status rc = ap_static_address(&ws);
    if (rc != KC_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    // the array keeps the last call's contents: the counters at its head (n_redo, this variant's error
    // word, the tickets) must start at zero; everything behind them is written before it is read
    KC_CUDA(cudaMemsetAsync(ws, 0, head_bytes(N, sh), st));
    ApArgs a = {};
    a.p = p; a.N = N; a.nq_host = N;
    a.nn = nn; a.nn2 = nn2; a.d1 = d1; a.d2 = d2; a.c = c;
    // the error word of this variant lives in the head's padding (device memory: the pinned host word
    // of the other entry points would be an allocation)
    int *errword = reinterpret_cast<int *>(ws + 8);
    if (d == 2) return launch<2>(a, ws, sh, st, errword);
    return launch<3>(a, ws, sh, st, errword);
}

extern "C" kc_status kc_cert_allpairs_bounded(const float *p, int64_t N, int d, const float *d2_prev,
                                              const float *eps, int32_t *nn, int32_t *nn2, float *d1,
                                              float *d2, float *c, void *workspace,
                                              size_t workspace_bytes, void *stream)
{
    if (!d2_prev || !eps) {
        set_error("kc_cert_allpairs_bounded: d2_prev and eps must be non-NULL");
        return KC_EINVAL;
    }
    return run("kc_cert_allpairs_bounded", p, N, d, nullptr, nullptr, N, d2_prev, eps, nullptr, nullptr, nn, nn2, d1, d2, c,
               workspace, workspace_bytes, stream);
}

extern "C" kc_status kc_cert_allpairs_seeded(const float *p, int64_t N, int d, const int32_t *seed1,
                                             const int32_t *seed2, int32_t *nn, int32_t *nn2, float *d1,
                                             float *d2, float *c, void *workspace, size_t workspace_bytes,
                                             void *stream)
{
    if (!seed1 || !seed2) {
        set_error("kc_cert_allpairs_seeded: seed1 and seed2 must be non-NULL");
        return KC_EINVAL;
    }
    return run("kc_cert_allpairs_seeded", p, N, d, nullptr, nullptr, N, nullptr, nullptr, seed1, seed2, nn, nn2,
               d1, d2, c, workspace, workspace_bytes, stream);
}

// NEXT #1 (PAPER.md:69 rtx_frontier_oracle): relabel a query subset against all N points.
// Same kernel with a query list; the grid is sized by nq_max and CTAs beyond the device-side
// count exit at once.  Small query sets are j-split like small N so they still fill the chip.
extern "C" size_t kc_frontier_oracle_workspace(int64_t N, int d, int64_t nq_max)
{
    if (N < 2 || nq_max < 1 || (d != 2 && d != 3)) return 0;
    error_word_init();
    return workspace_bytes_for(nq_max, choose_shape(nq_max, N));
}

extern "C" kc_status kc_frontier_oracle(const float *p, int64_t N, int d, const int32_t *q,
                                        const int32_t *nq, int64_t nq_max, int32_t *nn, int32_t *nn2,
                                        float *d1, float *d2, float *c, void *workspace,
                                        size_t workspace_bytes, void *stream)
{
    if (!q || !nq || nq_max < 0) {
        set_error("kc_frontier_oracle: bad argument");
        return KC_EINVAL;
    }
    if (nq_max == 0) return KC_OK;
    return run("kc_frontier_oracle", p, N, d, q, nq, nq_max, nullptr, nullptr, nullptr, nullptr, nn, nn2, d1, d2, c,
               workspace, workspace_bytes, stream);
}
