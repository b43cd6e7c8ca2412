// kc_topk.cu — NEXT #4: K-list certificates by a tiled N x N pass (contract: include/kc.h,
// kc_cert_allpairs_topk; reading R20 of DESIGN.md; "k-nearest-neighbour graphs",
// Definition 1 PAPER.md:29 generalised from 2 to K keys).
//
// One thread per query keeps its K best keys in registers; candidates are staged through shared
// memory as SoA tiles so that every lane reads the same address (broadcast) and one LDS.128 feeds
// four candidates; four distances are reduced with FMNMX and compared once with the worst key
// held, the exact (s, j) insertion runs only behind that branch.  For small N the candidates are
// split over gridDim.y and a merge kernel folds the partial lists (any merge order gives the
// same list: the order (s, j) is total).
#include "kc_common.cuh"

using namespace kc;

namespace {

constexpr int TK_THREADS = 128;
constexpr int TK_TILE = 512;

template <int D, int K>
__global__ void __launch_bounds__(TK_THREADS)
allpairs_topk_kernel(const float *__restrict__ p, int N, int chunk, const int32_t *__restrict__ seed_ids,
                     float *__restrict__ ws_s, int32_t *__restrict__ ws_j, int32_t *__restrict__ nnk,
                     float *__restrict__ dk, float *__restrict__ ck)
{
    __shared__ __align__(16) float sx[TK_TILE], sy[TK_TILE], sz[D == 3 ? TK_TILE : 4];
    const float qnan = __int_as_float(0x7fc00000);
    const int i = blockIdx.x * TK_THREADS + threadIdx.x;
    const int ic = i < N ? i : N - 1;
    const float qx = p[(int64_t)ic * D], qy = p[(int64_t)ic * D + 1], qz = D == 3 ? p[(int64_t)ic * D + 2] : 0.f;
    TopK<K> best;
    best.init();
    if (seed_ids && i < N) {
        // K known points per query (e.g. its list from the grid, or from the previous step): their
        // exact keys at the current positions are a valid start whatever they are; ids out of
        // range, equal to i or repeated are dropped, a NaN coordinate seeds nothing
#pragma unroll
        for (int q = 0; q < K; ++q) {
            const int j = seed_ids[(int64_t)i * K + q];
            if (j >= 0 && j < N && j != i && !best.holds(j)) {
                const float s = D == 2 ? sqd2(qx, qy, p[(int64_t)j * D], p[(int64_t)j * D + 1])
                                       : sqd3(qx, qy, qz, p[(int64_t)j * D], p[(int64_t)j * D + 1], p[(int64_t)j * D + 2]);
                if (s == s) best.offer(s, j);
            }
        }
    }
    const bool seeded = seed_ids != nullptr;
    const int j0 = blockIdx.y * chunk, j1 = min(N, j0 + chunk);
    for (int t0 = j0; t0 < j1; t0 += TK_TILE) {
        __syncthreads();
        for (int k = threadIdx.x; k < TK_TILE; k += TK_THREADS) {
            const int j = t0 + k;
            const bool ok = j < j1;                     // the tail is NaN: every comparison false
            sx[k] = ok ? p[(int64_t)j * D] : qnan;
            sy[k] = ok ? p[(int64_t)j * D + 1] : qnan;
            if (D == 3) sz[k] = ok ? p[(int64_t)j * D + 2] : qnan;
        }
        __syncthreads();
        const int n = min(TK_TILE, j1 - t0);
        for (int k = 0; k < n; k += 4) {
            const float4 X = *reinterpret_cast<const float4 *>(sx + k);
            const float4 Y = *reinterpret_cast<const float4 *>(sy + k);
            float s0, s1, s2, s3;
            if (D == 2) {
                s0 = sqd2(qx, qy, X.x, Y.x); s1 = sqd2(qx, qy, X.y, Y.y);
                s2 = sqd2(qx, qy, X.z, Y.z); s3 = sqd2(qx, qy, X.w, Y.w);
            } else {
                const float4 Z = *reinterpret_cast<const float4 *>(sz + k);
                s0 = sqd3(qx, qy, qz, X.x, Y.x, Z.x); s1 = sqd3(qx, qy, qz, X.y, Y.y, Z.y);
                s2 = sqd3(qx, qy, qz, X.z, Y.z, Z.z); s3 = sqd3(qx, qy, qz, X.w, Y.w, Z.w);
            }
            const float m = fminf(fminf(s0, s1), fminf(s2, s3));
            if (m <= best.s[K - 1]) {
                const int jb = t0 + k;
                // a seeded list may already hold the candidate
                if (s0 <= best.s[K - 1] && jb != i && !(seeded && best.holds(jb))) best.offer(s0, jb);
                if (s1 <= best.s[K - 1] && jb + 1 != i && !(seeded && best.holds(jb + 1))) best.offer(s1, jb + 1);
                if (s2 <= best.s[K - 1] && jb + 2 != i && !(seeded && best.holds(jb + 2))) best.offer(s2, jb + 2);
                if (s3 <= best.s[K - 1] && jb + 3 != i && !(seeded && best.holds(jb + 3))) best.offer(s3, jb + 3);
            }
        }
    }
    if (i >= N) return;
    if (gridDim.y == 1) {
        best.store(i, nnk, dk, ck);
        return;
    }
    const int64_t base = ((int64_t)blockIdx.y * N + i) * K;
#pragma unroll
    for (int q = 0; q < K; ++q) { ws_s[base + q] = best.s[q]; ws_j[base + q] = best.j[q]; }
}

template <int K>
__global__ void __launch_bounds__(128)
topk_merge_kernel(int N, int chunks, const float *__restrict__ ws_s, const int32_t *__restrict__ ws_j,
                  int32_t *__restrict__ nnk, float *__restrict__ dk, float *__restrict__ ck)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    TopK<K> best;
    best.init();
    for (int y = 0; y < chunks; ++y) {
        const int64_t base = ((int64_t)y * N + i) * K;
#pragma unroll
        for (int q = 0; q < K; ++q) {
            const int id = ws_j[base + q];
            if (id != KC_NOIDX && !best.holds(id)) best.offer(ws_s[base + q], id);    // chunks share their seeds
        }
    }
    best.store(i, nnk, dk, ck);
}

// candidates per y-block: enough blocks for ~8 CTAs per SM, whole tiles, at least one tile
int topk_chunks(int64_t N)
{
    const int64_t qblocks = (N + TK_THREADS - 1) / TK_THREADS;
    int64_t chunks = (148 * 8 + qblocks - 1) / qblocks;
    const int64_t tiles = (N + TK_TILE - 1) / TK_TILE;
    if (chunks > tiles) chunks = tiles;
    if (chunks > 64) chunks = 64;
    if (chunks < 1) chunks = 1;
    return (int)chunks;
}
int topk_chunk_len(int64_t N, int chunks)
{
    const int64_t tiles = (N + TK_TILE - 1) / TK_TILE;
    return (int)((tiles + chunks - 1) / chunks) * TK_TILE;
}

template <int D, int K>
void launch_topk(const float *p, int N, int chunks, int chunk, const int32_t *seed_ids, float *ws_s, int32_t *ws_j,
                 int32_t *nnk, float *dk, float *ck, cudaStream_t st)
{
    const dim3 grid((N + TK_THREADS - 1) / TK_THREADS, chunks);
    allpairs_topk_kernel<D, K><<<grid, TK_THREADS, 0, st>>>(p, N, chunk, seed_ids, ws_s, ws_j, nnk, dk, ck);
    if (chunks > 1) topk_merge_kernel<K><<<(N + 127) / 128, 128, 0, st>>>(N, chunks, ws_s, ws_j, nnk, dk, ck);
}
template <int D>
bool dispatch_topk(int K, const float *p, int N, int chunks, int chunk, const int32_t *seed_ids, float *ws_s,
                   int32_t *ws_j, int32_t *nnk, float *dk, float *ck, cudaStream_t st)
{
    switch (K) {
    case 2: launch_topk<D, 2>(p, N, chunks, chunk, seed_ids, ws_s, ws_j, nnk, dk, ck, st); return true;
    case 3: launch_topk<D, 3>(p, N, chunks, chunk, seed_ids, ws_s, ws_j, nnk, dk, ck, st); return true;
    case 4: launch_topk<D, 4>(p, N, chunks, chunk, seed_ids, ws_s, ws_j, nnk, dk, ck, st); return true;
    case 5: launch_topk<D, 5>(p, N, chunks, chunk, seed_ids, ws_s, ws_j, nnk, dk, ck, st); return true;
    case 6: launch_topk<D, 6>(p, N, chunks, chunk, seed_ids, ws_s, ws_j, nnk, dk, ck, st); return true;
    case 7: launch_topk<D, 7>(p, N, chunks, chunk, seed_ids, ws_s, ws_j, nnk, dk, ck, st); return true;
    case 8: launch_topk<D, 8>(p, N, chunks, chunk, seed_ids, ws_s, ws_j, nnk, dk, ck, st); return true;
    default: return false;
    }
}

}  // namespace

extern "C" size_t kc_cert_allpairs_topk_workspace(int64_t N, int d, int K)
{
    if (N < 2 || (d != 2 && d != 3) || K < 2 || K > KC_TOPK_MAX) return 0;
    const int chunks = topk_chunks(N);
    return chunks > 1 ? (size_t)chunks * (size_t)N * (size_t)K * 8 : 0;
}

extern "C" kc_status kc_cert_allpairs_topk(const float *p, int64_t N, int d, int K, const int32_t *seed_ids,
                                           int32_t *nnk, float *dk, float *ck, void *workspace,
                                           size_t workspace_bytes, void *stream)
{
    if (!p || !nnk || !dk || !ck || N < 2 || N > 0x7ffffff0 || (d != 2 && d != 3) || K < 2 || K > KC_TOPK_MAX) {
        set_error("kc_cert_allpairs_topk: bad argument (need p, nnk, dk, ck, 2 <= N, d in {2,3}, 2 <= K <= %d)",
                  KC_TOPK_MAX);
        return KC_EINVAL;
    }
    const int chunks = topk_chunks(N);
    const size_t need = kc_cert_allpairs_topk_workspace(N, d, K);
    if (need > 0 && (!workspace || workspace_bytes < need)) {
        set_error("kc_cert_allpairs_topk: workspace of %zu bytes required", need);
        return KC_EINVAL;
    }
    float *ws_s = static_cast<float *>(workspace);
    int32_t *ws_j = reinterpret_cast<int32_t *>(ws_s + (size_t)chunks * (size_t)N * (size_t)K);
    const int chunk = topk_chunk_len(N, chunks);
    cudaStream_t st = (cudaStream_t)stream;
    if (seed_ids == nnk) {
        set_error("kc_cert_allpairs_topk: seed_ids must not alias nnk");
        return KC_EINVAL;
    }
    if (d == 2) dispatch_topk<2>(K, p, (int)N, chunks, chunk, seed_ids, ws_s, ws_j, nnk, dk, ck, st);
    else dispatch_topk<3>(K, p, (int)N, chunks, chunk, seed_ids, ws_s, ws_j, nnk, dk, ck, st);
    count_launches(chunks > 1 ? 2 : 1);
    KC_LAUNCH_CHECK("kc_cert_allpairs_topk");
    return KC_OK;
}
