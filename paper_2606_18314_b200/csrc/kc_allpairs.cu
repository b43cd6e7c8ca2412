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
//   * j is split across gridDim.y so small N still fills 148 SMs; partial top-2s are merged by
//     a second kernel under the same total order, so the split never changes a result.
#include <stdlib.h>

#include "kc_common.cuh"

using namespace kc;

namespace {

constexpr int AP_TJ = 1024;   // candidates per shared-memory tile

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
__device__ __forceinline__ void load_tile(const float *__restrict__ p, int64_t N, int64_t j0,
                                          float *sx, float *sy, float *sz)
{
    // pad the tail with +inf: s = +inf never beats a finite second-best, and the slow path
    // rejects j >= N explicitly while second-best is still +inf.
    for (int t = threadIdx.x; t < AP_TJ; t += THREADS) {
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
    if (s0 <= best.s2 && j + 0 < lim && j + 0 != self) best.offer(s0, j + 0);
    if (s1 <= best.s2 && j + 1 < lim && j + 1 != self) best.offer(s1, j + 1);
    if (s2 <= best.s2 && j + 2 < lim && j + 2 != self) best.offer(s2, j + 2);
    if (s3 <= best.s2 && j + 3 < lim && j + 3 != self) best.offer(s3, j + 3);
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
        __syncthreads();
        load_tile<D, THREADS>(p, lim, j0, sx, sy, sz);
        __syncthreads();
#pragma unroll 1
        for (int t = 0; t < AP_TJ; t += 4 * C4) {
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

// grid = (ceil(nq / (QPT*THREADS)), JS).  qlist == nullptr: queries are 0..N-1.
template <int D, int QPT, int C4, int THREADS>
__global__ void __launch_bounds__(THREADS)
allpairs_kernel(const float *__restrict__ p, int64_t N, const int32_t *__restrict__ qlist,
                const int32_t *__restrict__ nq_dev, int64_t nq_host, int64_t jchunk, u64 one2,
                Partial *__restrict__ part, int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c)
{
    __shared__ __align__(16) float sx[AP_TJ];
    __shared__ __align__(16) float sy[AP_TJ];
    __shared__ __align__(16) float sz[D == 3 ? AP_TJ : 4];
    const int64_t nq = nq_dev ? (int64_t)*nq_dev : nq_host;
    const int64_t q0 = blockIdx.x * (int64_t)(QPT * THREADS);
    if (q0 >= nq) return;
    float qx[QPT], qy[QPT], qz[QPT];
    int qi[QPT];
    Top2 best[QPT];
#pragma unroll
    for (int k = 0; k < QPT; ++k) {
        int64_t q = q0 + k * THREADS + threadIdx.x;
        int i = -1;
        if (q < nq) i = qlist ? qlist[q] : (int)q;
        qi[k] = i;
        qx[k] = qy[k] = qz[k] = 0.f;
        if (i >= 0) {
            qx[k] = p[(int64_t)i * D + 0];
            qy[k] = p[(int64_t)i * D + 1];
            if (D == 3) qz[k] = p[(int64_t)i * D + 2];
        }
        best[k].init();
    }
    const int64_t jbeg = blockIdx.y * jchunk;
    const int64_t jend = min(N, jbeg + jchunk);
    scan_chunk<D, QPT, C4, THREADS>(p, N, jbeg, jend, qx, qy, qz, qi, best, sx, sy, sz, one2);
#pragma unroll
    for (int k = 0; k < QPT; ++k) {
        int64_t q = q0 + k * THREADS + threadIdx.x;
        if (qi[k] < 0) continue;
        if (gridDim.y == 1) {
            store_cert(best[k], qi[k], nn, nn2, d1, d2, c);
        } else {
            Partial o;
            o.s1 = best[k].s1; o.s2 = best[k].s2; o.j1 = best[k].j1; o.j2 = best[k].j2;
            part[blockIdx.y * nq_host + q] = o;
        }
    }
}

__global__ void __launch_bounds__(256)
allpairs_merge_kernel(const Partial *__restrict__ part, int64_t nq_host, int js,
                      const int32_t *__restrict__ qlist, const int32_t *__restrict__ nq_dev,
                      int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c)
{
    const int64_t nq = nq_dev ? (int64_t)*nq_dev : nq_host;
    int64_t q = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (q >= nq) return;
    Top2 t;
    t.init();
    for (int s = 0; s < js; ++s) {
        const int4 raw = reinterpret_cast<const int4 *>(part)[s * nq_host + q];
        Top2 o;
        o.s1 = __int_as_float(raw.x); o.s2 = __int_as_float(raw.y); o.j1 = raw.z; o.j2 = raw.w;
        t.merge(o);
    }
    store_cert(t, qlist ? qlist[q] : (int)q, nn, nn2, d1, d2, c);
}

// Launch shape.  Tuning overrides for experiments: KC_AP_QPT, KC_AP_C4, KC_AP_THREADS, KC_AP_JS
// (read once per process).
struct Shape { int qpt, c4, threads, js; };

int env_int(const char *name, int dflt)
{
    const char *v = getenv(name);
    return v && *v ? atoi(v) : dflt;
}

Shape choose_shape(int64_t nq, int64_t N)
{
    static const int e_qpt = env_int("KC_AP_QPT", 0), e_thr = env_int("KC_AP_THREADS", 0),
                     e_js = env_int("KC_AP_JS", 0), e_c4 = env_int("KC_AP_C4", 0);
    Shape s;
    s.qpt = nq >= 148 * 8 * 128 * 2 ? 4 : (nq >= 148 * 4 * 128 ? 2 : 1);
    s.threads = 128;
    if (e_qpt == 1 || e_qpt == 2 || e_qpt == 4) s.qpt = e_qpt;
    s.c4 = s.qpt == 4 ? 2 : (s.qpt == 2 ? 2 : 4);
    if (e_c4 == 1 || e_c4 == 2 || e_c4 == 4) s.c4 = e_c4;
    if (e_thr == 32 || e_thr == 64 || e_thr == 128) s.threads = e_thr;
    // j-split: many waves deep, but every CTA still scans >= 4 tiles (short chunks pay the
    // ~2 ln(n) insertions per lane again in every chunk)
    int64_t per = (int64_t)s.qpt * s.threads;
    int64_t itiles = (nq + per - 1) / per;
    int64_t want = (148 * 8 * 8 + itiles - 1) / itiles;
    int64_t cap = N / (4 * AP_TJ);
    int64_t js = want < cap ? want : cap;
    if (e_js > 0) js = e_js;
    if (js < 1) js = 1;
    if (js > 65535) js = 65535;
    s.js = (int)js;
    return s;
}

template <int D, int QPT, int C4>
void launch_t(int threads, dim3 grid, cudaStream_t st, const float *p, int64_t N, const int32_t *q,
              const int32_t *nq_dev, int64_t nq, int64_t jchunk, Partial *part, int32_t *nn,
              int32_t *nn2, float *d1, float *d2, float *c)
{
    const u64 one2 = 0x3f8000003f800000ull;
    if (threads == 32)
        allpairs_kernel<D, QPT, C4, 32><<<grid, 32, 0, st>>>(p, N, q, nq_dev, nq, jchunk, one2, part, nn, nn2, d1, d2, c);
    else if (threads == 64)
        allpairs_kernel<D, QPT, C4, 64><<<grid, 64, 0, st>>>(p, N, q, nq_dev, nq, jchunk, one2, part, nn, nn2, d1, d2, c);
    else
        allpairs_kernel<D, QPT, C4, 128><<<grid, 128, 0, st>>>(p, N, q, nq_dev, nq, jchunk, one2, part, nn, nn2, d1, d2, c);
}

template <int D>
kc_status launch(const float *p, int64_t N, const int32_t *q, const int32_t *nq_dev, int64_t nq,
                 int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c, Partial *part, Shape sh,
                 cudaStream_t st)
{
    int js = sh.js;
    int64_t jchunk = (N + js - 1) / js;
    jchunk = (jchunk + 15) / 16 * 16;
    js = (int)((N + jchunk - 1) / jchunk);
    const int per = sh.qpt * sh.threads;
    dim3 grid((unsigned)((nq + per - 1) / per), (unsigned)js);
#define KC_AP_CASE(Q, C)                                                                            \
    if (sh.qpt == Q && sh.c4 == C) {                                                                \
        launch_t<D, Q, C>(sh.threads, grid, st, p, N, q, nq_dev, nq, jchunk, part, nn, nn2, d1, d2, c); \
    } else
    KC_AP_CASE(4, 1) KC_AP_CASE(4, 2) KC_AP_CASE(2, 1) KC_AP_CASE(2, 2) KC_AP_CASE(2, 4)
    KC_AP_CASE(1, 1) KC_AP_CASE(1, 2) KC_AP_CASE(1, 4)
    {
        set_error("kc_cert_allpairs: unsupported launch shape");
        return KC_EINVAL;
    }
#undef KC_AP_CASE
    if (js > 1)
        allpairs_merge_kernel<<<(unsigned)((nq + 255) / 256), 256, 0, st>>>(part, nq, js, q, nq_dev, nn, nn2, d1, d2, c);
    count_launches(js > 1 ? 2 : 1);
    KC_LAUNCH_CHECK("kc_cert_allpairs");
    return KC_OK;
}

}  // namespace

extern "C" size_t kc_cert_allpairs_workspace(int64_t N, int d)
{
    if (N < 2 || (d != 2 && d != 3)) return 0;
    int js = choose_shape(N, N).js;
    return js > 1 ? (size_t)js * (size_t)N * sizeof(Partial) : 0;
}

extern "C" kc_status kc_cert_allpairs(const float *p, int64_t N, int d, int32_t *nn, int32_t *nn2,
                                      float *d1, float *d2, float *c, void *workspace,
                                      size_t workspace_bytes, void *stream)
{
    if (!p || !nn || !d1 || !d2 || !c || N < 2 || N > 0x7ffffff0 || (d != 2 && d != 3) ||
        (reinterpret_cast<uintptr_t>(p) & 7)) {
        set_error("kc_cert_allpairs: bad argument");
        return KC_EINVAL;
    }
    size_t need = kc_cert_allpairs_workspace(N, d);
    if (need > 0 && (!workspace || workspace_bytes < need || (reinterpret_cast<uintptr_t>(workspace) & 15))) {
        set_error("kc_cert_allpairs: workspace of %zu bytes (16-byte aligned) required", need);
        return KC_EINVAL;
    }
    Shape sh = choose_shape(N, N);
    cudaStream_t st = (cudaStream_t)stream;
    if (d == 2)
        return launch<2>(p, N, nullptr, nullptr, N, nn, nn2, d1, d2, c, (Partial *)workspace, sh, st);
    return launch<3>(p, N, nullptr, nullptr, N, nn, nn2, d1, d2, c, (Partial *)workspace, sh, st);
}

// NEXT #1 (PAPER.md:69 rtx_frontier_oracle): relabel a query subset against all N points.
// Same kernel with a query list; the grid is sized by nq_max and CTAs beyond the device-side
// count exit at once.  Small query sets are j-split like small N so they still fill the chip.
extern "C" size_t kc_frontier_oracle_workspace(int64_t N, int d, int64_t nq_max)
{
    if (N < 2 || nq_max < 1 || (d != 2 && d != 3)) return 0;
    int js = choose_shape(nq_max, N).js;
    return js > 1 ? (size_t)js * (size_t)nq_max * sizeof(Partial) : 0;
}

extern "C" kc_status kc_frontier_oracle(const float *p, int64_t N, int d, const int32_t *q,
                                        const int32_t *nq, int64_t nq_max, int32_t *nn, int32_t *nn2,
                                        float *d1, float *d2, float *c, void *workspace,
                                        size_t workspace_bytes, void *stream)
{
    if (!p || !q || !nq || !nn || !d1 || !d2 || !c || N < 2 || N > 0x7ffffff0 || nq_max < 0 ||
        (d != 2 && d != 3) || (reinterpret_cast<uintptr_t>(p) & 7)) {
        set_error("kc_frontier_oracle: bad argument");
        return KC_EINVAL;
    }
    if (nq_max == 0) return KC_OK;
    size_t need = kc_frontier_oracle_workspace(N, d, nq_max);
    if (need > 0 && (!workspace || workspace_bytes < need || (reinterpret_cast<uintptr_t>(workspace) & 15))) {
        set_error("kc_frontier_oracle: workspace of %zu bytes (16-byte aligned) required", need);
        return KC_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    Shape sh = choose_shape(nq_max, N);
    if (d == 2) return launch<2>(p, N, q, nq, nq_max, nn, nn2, d1, d2, c, (Partial *)workspace, sh, st);
    return launch<3>(p, N, q, nq, nq_max, nn, nn2, d1, d2, c, (Partial *)workspace, sh, st);
}
