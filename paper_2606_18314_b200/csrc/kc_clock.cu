// kc_clock.cu -- NEXT #3, the expiry structure of the cumulative clock (Appendix A.2, PAPER.md:177-181,
// Theorem 2: "an expiry heap ... O(|F_t| log N) per step").  See include/kc.h for the contract.
//
// The flat form (kc_frontier_classify_clock, kc_misc.cu) tests all N certificates every step.  A heap
// is a serial structure; its data-parallel form is a TOURNAMENT TREE over the point ids with fanout
// 32: node j of level 1 holds a lower bound of the earliest expiry clock among points 32j .. 32j+31,
// node k of level 2 the minimum of level-1 nodes 32k .. 32k+31.  A step reads the N/1024 level-2
// nodes, opens those whose bound has been reached, in them the level-1 nodes whose bound has been
// reached, and applies the EXACT flat test to the 32 points of each of those: the expired set is the
// flat test's, found with N/1024 + 64 reads per opened node.  After the expired certificates have
// been recomputed and re-stamped their nodes are recomputed bottom-up (idempotent: no atomics).
//
// The bound of point i: e = stamp_i + c_i / 4 in double, rounded down to float and lowered by a
// relative 2^-22 and an absolute 1e-37: far more than the double roundings of the flat test
// c_i <= 4 (S - stamp_i), so "expired by the flat test" implies "bound <= S rounded up to float".
#include <math.h>

#include "kc_grid.cuh"

using namespace kc;

namespace {

__device__ __forceinline__ float expiry_bound(float c, float stamp)
{
    const double e = (double)stamp + 0.25 * (double)c;
    const float kf = __double2float_rd(e);
    if (!(kf < CUDART_INF_F)) return CUDART_INF_F;             // c = +inf: never expires
    return __fsub_rd(__fsub_rd(kf, __fmul_ru(fabsf(kf), 2.384186e-7f)), 1e-37f);
}
__device__ __forceinline__ float warp_min(float x)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x = fminf(x, __shfl_xor_sync(0xffffffffu, x, o));
    return x;
}
// level-1 node j from its 32 points (all 32 lanes of a warp)
__device__ __forceinline__ void node1_from_points(const float *__restrict__ c, const float *__restrict__ stamp,
                                                  int64_t N, int64_t j, float *lv1, int lane)
{
    const int64_t i = j * 32 + lane;
    const float k = i < N ? expiry_bound(c[i], stamp[i]) : CUDART_INF_F;
    const float m = warp_min(k);
    if (lane == 0) lv1[j] = m;
}
// level-2 node k from its 32 children
__device__ __forceinline__ void node2_from_nodes(const float *__restrict__ lv1, int64_t n1, int64_t k, float *lv2,
                                                 int lane)
{
    const int64_t j = k * 32 + lane;
    const float m = warp_min(j < n1 ? lv1[j] : CUDART_INF_F);
    if (lane == 0) lv2[k] = m;
}

// Recompute of level 1 (LEVEL = 1) or level 2 (LEVEL = 2): all nodes when F is null or the list is a
// large part of the points (decided on the device), else the nodes above the listed ids, one warp per
// entry (ids that share a node recompute the same value).
template <int LEVEL>
__global__ void __launch_bounds__(256)
clock_tree_nodes_kernel(const int32_t *__restrict__ F, const int32_t *__restrict__ nF, const float *__restrict__ c,
                        const float *__restrict__ stamp, int64_t N, float *lv1, float *lv2)
{
    const int lane = threadIdx.x & 31;
    const int64_t w0 = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5, nw = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const int64_t n1 = (N + 31) / 32, n2 = (n1 + 31) / 32;
    const int64_t n = F ? (int64_t)*nF : 0;
    if (!F || n * 16 > N) {
        for (int64_t j = w0; j < (LEVEL == 1 ? n1 : n2); j += nw) {
            if (LEVEL == 1) node1_from_points(c, stamp, N, j, lv1, lane);
            else node2_from_nodes(lv1, n1, j, lv2, lane);
        }
        return;
    }
    for (int64_t f = w0; f < n; f += nw) {
        const int64_t i = F[f];
        if (LEVEL == 1) node1_from_points(c, stamp, N, i >> 5, lv1, lane);
        else node2_from_nodes(lv1, n1, i >> 10, lv2, lane);
    }
}

__global__ void clock_tree_zero_kernel(int32_t *nF) { *nF = 0; }

// One warp per level-2 node.
__global__ void __launch_bounds__(256)
classify_clock_tree_kernel(const float *__restrict__ c, const float *__restrict__ stamp, int64_t N,
                           const float *__restrict__ lv1, const float *__restrict__ lv2,
                           const double *__restrict__ S_in, const float *__restrict__ eps, double *S_out,
                           int32_t *__restrict__ F, int32_t *nF)
{
    const double S = *S_in + (double)*eps;
    const float Sf = __double2float_ru(S);
    const int lane = threadIdx.x & 31;
    const int64_t w0 = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5, nw = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const int64_t n1 = (N + 31) / 32, n2 = (n1 + 31) / 32;
    if (w0 == 0 && lane == 0) *S_out = S;
    for (int64_t k = w0; k < n2; k += nw) {
        if (!(lv2[k] <= Sf)) continue;                         // (warp-uniform)
        const int64_t j = k * 32 + lane;
        unsigned open = __ballot_sync(0xffffffffu, j < n1 && lv1[j] <= Sf);
        // bit b of `mine`: point (32 k + b) * 32 + lane is expired (the flat test, as
        // kc_frontier_classify_clock evaluates it); one reservation in F per level-2 node
        unsigned mine = 0;
        while (open) {
            const int b = __ffs(open) - 1;
            open &= open - 1;
            const int64_t i = (k * 32 + b) * 32 + lane;
            if (i < N && (double)c[i] <= 4.0 * (S - (double)stamp[i])) mine |= 1u << b;
        }
        const int cnt = __popc(mine);
        int incl = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        const int total = __shfl_sync(0xffffffffu, incl, 31);
        if (total == 0) continue;
        int base = 0;
        if (lane == 0) base = atomicAdd(nF, total);
        base = __shfl_sync(0xffffffffu, base, 0) + incl - cnt;
        while (mine) {
            const int b = __ffs(mine) - 1;
            mine &= mine - 1;
            F[base++] = (int32_t)((k * 32 + b) * 32 + lane);
        }
    }
}

kc_status check_tree_args(const char *who, const float *c, const float *stamp, int64_t N, const float *tree)
{
    if (!c || !stamp || !tree || N < 1 || N > 0x7fffffff) {
        set_error("%s: bad argument", who);
        return KC_EINVAL;
    }
    return KC_OK;
}
int blocks_of_warps(int64_t warps)
{
    const int64_t b = (warps + 7) / 8;
    return (int)(b < 1 ? 1 : (b < 148 * 8 ? b : 148 * 8));
}

}  // namespace

extern "C" size_t kc_clock_tree_floats(int64_t N)
{
    if (N < 1) return 0;
    const int64_t n1 = (N + 31) / 32, n2 = (n1 + 31) / 32;
    return (size_t)(n1 + n2);
}

extern "C" kc_status kc_clock_tree_update(const int32_t *F, const int32_t *nF, int64_t nF_max, const float *c,
                                          const float *stamp, int64_t N, float *tree, void *stream)
{
    kc_status s = check_tree_args("kc_clock_tree_update", c, stamp, N, tree);
    if (s != KC_OK) return s;
    if (F && (!nF || nF_max < 0)) {
        set_error("kc_clock_tree_update: F without nF");
        return KC_EINVAL;
    }
    if (F && nF_max == 0) return KC_OK;
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n1 = (N + 31) / 32;
    float *lv1 = tree, *lv2 = tree + n1;
    // the grid covers the larger of the two shapes the kernel may take (list / all nodes)
    const int64_t w1 = F ? (nF_max * 16 > N ? n1 : nF_max) : n1;
    const int64_t w2 = F ? (nF_max * 16 > N ? (n1 + 31) / 32 : nF_max) : (n1 + 31) / 32;
    clock_tree_nodes_kernel<1><<<blocks_of_warps(w1), 256, 0, st>>>(F, nF, c, stamp, N, lv1, lv2);
    clock_tree_nodes_kernel<2><<<blocks_of_warps(w2), 256, 0, st>>>(F, nF, c, stamp, N, lv1, lv2);
    count_launches(2);
    KC_LAUNCH_CHECK("kc_clock_tree_update");
    return KC_OK;
}

extern "C" kc_status kc_clock_tree_build(const float *c, const float *stamp, int64_t N, float *tree, void *stream)
{
    return kc_clock_tree_update(nullptr, nullptr, 0, c, stamp, N, tree, stream);
}

extern "C" kc_status kc_frontier_classify_clock_tree(const float *c, const float *stamp, int64_t N, const float *tree,
                                                     const double *S_in, const float *eps, double *S_out,
                                                     int32_t *F, int32_t *nF, void *stream)
{
    kc_status s = check_tree_args("kc_frontier_classify_clock_tree", c, stamp, N, tree);
    if (s != KC_OK) return s;
    if (!S_in || !eps || !S_out || S_in == S_out || !F || !nF) {
        set_error("kc_frontier_classify_clock_tree: bad argument (S_in and S_out must differ)");
        return KC_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n1 = (N + 31) / 32, n2 = (n1 + 31) / 32;
    clock_tree_zero_kernel<<<1, 1, 0, st>>>(nF);
    classify_clock_tree_kernel<<<blocks_of_warps(n2), 256, 0, st>>>(c, stamp, N, tree, tree + n1, S_in, eps, S_out, F, nF);
    count_launches(2);
    KC_LAUNCH_CHECK("kc_frontier_classify_clock_tree");
    return KC_OK;
}
