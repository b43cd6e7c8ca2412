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
#include "kc_common.cuh"

using namespace kc;

namespace {

constexpr int AP_THREADS = 128;
constexpr int AP_TJ = 1024;   // candidates per shared-memory tile

struct Partial { float s1, s2; int j1, j2; };   // 16 B

template <int D>
__device__ __forceinline__ void load_tile(const float *__restrict__ p, int64_t N, int64_t j0,
                                          float *sx, float *sy, float *sz)
{
    // pad the tail with +inf: s = +inf never beats a finite second-best, and the slow path
    // rejects j >= N explicitly while second-best is still +inf.
    for (int t = threadIdx.x; t < AP_TJ; t += AP_THREADS) {
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

// QPT queries per thread against candidates [jbeg, jend).  qi[k] = -1 marks a padding query.
template <int D, int QPT>
__device__ __forceinline__ void scan_chunk(const float *__restrict__ p, int64_t N, int64_t jbeg,
                                           int64_t jend, const float (&qx)[QPT],
                                           const float (&qy)[QPT], const float (&qz)[QPT],
                                           const int (&qi)[QPT], Top2 (&best)[QPT], float *sx,
                                           float *sy, float *sz)
{
    for (int64_t j0 = jbeg; j0 < jend; j0 += AP_TJ) {
        __syncthreads();
        load_tile<D>(p, min(N, jend), j0, sx, sy, sz);
        __syncthreads();
#pragma unroll 2
        for (int t = 0; t < AP_TJ; t += 4) {
            const float4 X = *reinterpret_cast<const float4 *>(sx + t);
            const float4 Y = *reinterpret_cast<const float4 *>(sy + t);
            float4 Z = make_float4(0.f, 0.f, 0.f, 0.f);
            if (D == 3) Z = *reinterpret_cast<const float4 *>(sz + t);
#pragma unroll
            for (int k = 0; k < QPT; ++k) {
                float s0, s1, s2, s3;
                if (D == 2) {
                    s0 = sqd2(qx[k], qy[k], X.x, Y.x);
                    s1 = sqd2(qx[k], qy[k], X.y, Y.y);
                    s2 = sqd2(qx[k], qy[k], X.z, Y.z);
                    s3 = sqd2(qx[k], qy[k], X.w, Y.w);
                } else {
                    s0 = sqd3(qx[k], qy[k], qz[k], X.x, Y.x, Z.x);
                    s1 = sqd3(qx[k], qy[k], qz[k], X.y, Y.y, Z.y);
                    s2 = sqd3(qx[k], qy[k], qz[k], X.z, Y.z, Z.z);
                    s3 = sqd3(qx[k], qy[k], qz[k], X.w, Y.w, Z.w);
                }
                float m = fminf(fminf(s0, s1), fminf(s2, s3));
                if (m <= best[k].s2) {
                    const int64_t j = j0 + t;
                    const int64_t lim = min(N, jend);
                    if (s0 <= best[k].s2 && j + 0 < lim && (int)(j + 0) != qi[k]) best[k].offer(s0, (int)(j + 0));
                    if (s1 <= best[k].s2 && j + 1 < lim && (int)(j + 1) != qi[k]) best[k].offer(s1, (int)(j + 1));
                    if (s2 <= best[k].s2 && j + 2 < lim && (int)(j + 2) != qi[k]) best[k].offer(s2, (int)(j + 2));
                    if (s3 <= best[k].s2 && j + 3 < lim && (int)(j + 3) != qi[k]) best[k].offer(s3, (int)(j + 3));
                }
            }
        }
    }
}

// grid = (ceil(nq / (QPT*128)), JS).  qlist == nullptr: queries are 0..N-1.
template <int D, int QPT>
__global__ void __launch_bounds__(AP_THREADS)
allpairs_kernel(const float *__restrict__ p, int64_t N, const int32_t *__restrict__ qlist,
                const int32_t *__restrict__ nq_dev, int64_t nq_host, int64_t jchunk,
                Partial *__restrict__ part, int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c)
{
    __shared__ __align__(16) float sx[AP_TJ];
    __shared__ __align__(16) float sy[AP_TJ];
    __shared__ __align__(16) float sz[D == 3 ? AP_TJ : 4];
    const int64_t nq = nq_dev ? (int64_t)*nq_dev : nq_host;
    const int64_t q0 = blockIdx.x * (int64_t)(QPT * AP_THREADS);
    if (q0 >= nq) return;
    float qx[QPT], qy[QPT], qz[QPT];
    int qi[QPT];
    Top2 best[QPT];
#pragma unroll
    for (int k = 0; k < QPT; ++k) {
        int64_t q = q0 + k * AP_THREADS + threadIdx.x;
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
    scan_chunk<D, QPT>(p, N, jbeg, jend, qx, qy, qz, qi, best, sx, sy, sz);
#pragma unroll
    for (int k = 0; k < QPT; ++k) {
        int64_t q = q0 + k * AP_THREADS + threadIdx.x;
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

// j-split so that the grid is many waves deep but every CTA still scans >= 2 tiles.
inline int choose_js(int64_t nq, int64_t N, int qpt)
{
    int64_t itiles = (nq + qpt * AP_THREADS - 1) / (qpt * AP_THREADS);
    int64_t want = (148 * 8 * 8 + itiles - 1) / itiles;
    int64_t cap = N / (2 * AP_TJ);
    int64_t js = want < cap ? want : cap;
    if (js < 1) js = 1;
    if (js > 65535) js = 65535;
    return (int)js;
}
inline int choose_qpt(int64_t nq) { return nq >= 148 * 8 * 128 * 2 ? 4 : (nq >= 148 * 4 * 128 ? 2 : 1); }

template <int D>
kc_status launch(const float *p, int64_t N, const int32_t *q, const int32_t *nq_dev, int64_t nq,
                 int32_t *nn, int32_t *nn2, float *d1, float *d2, float *c, Partial *part, int js,
                 int qpt, cudaStream_t st)
{
    int64_t jchunk = (N + js - 1) / js;
    jchunk = (jchunk + 3) / 4 * 4;
    js = (int)((N + jchunk - 1) / jchunk);
    dim3 grid((unsigned)((nq + qpt * AP_THREADS - 1) / (qpt * AP_THREADS)), (unsigned)js);
    if (qpt == 4)
        allpairs_kernel<D, 4><<<grid, AP_THREADS, 0, st>>>(p, N, q, nq_dev, nq, jchunk, part, nn, nn2, d1, d2, c);
    else if (qpt == 2)
        allpairs_kernel<D, 2><<<grid, AP_THREADS, 0, st>>>(p, N, q, nq_dev, nq, jchunk, part, nn, nn2, d1, d2, c);
    else
        allpairs_kernel<D, 1><<<grid, AP_THREADS, 0, st>>>(p, N, q, nq_dev, nq, jchunk, part, nn, nn2, d1, d2, c);
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
    int js = choose_js(N, N, choose_qpt(N));
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
    int qpt = choose_qpt(N);
    int js = choose_js(N, N, qpt);
    cudaStream_t st = (cudaStream_t)stream;
    if (d == 2)
        return launch<2>(p, N, nullptr, nullptr, N, nn, nn2, d1, d2, c, (Partial *)workspace, js, qpt, st);
    return launch<3>(p, N, nullptr, nullptr, N, nn, nn2, d1, d2, c, (Partial *)workspace, js, qpt, st);
}

// NEXT #1 (PAPER.md:69 rtx_frontier_oracle): relabel a query subset against all N points.
// Same kernel with a query list; the grid is sized by nq_max and CTAs beyond the device-side
// count exit at once.  Small query sets are j-split like small N so they still fill the chip.
extern "C" size_t kc_frontier_oracle_workspace(int64_t N, int d, int64_t nq_max)
{
    if (N < 2 || nq_max < 1 || (d != 2 && d != 3)) return 0;
    int js = choose_js(nq_max, N, choose_qpt(nq_max));
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
    int qpt = choose_qpt(nq_max);
    int js = choose_js(nq_max, N, qpt);
    if (d == 2) return launch<2>(p, N, q, nq, nq_max, nn, nn2, d1, d2, c, (Partial *)workspace, js, qpt, st);
    return launch<3>(p, N, q, nq, nq_max, nn, nn2, d1, d2, c, (Partial *)workspace, js, qpt, st);
}
