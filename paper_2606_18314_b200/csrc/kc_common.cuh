// kc_common.cuh — shared device helpers of libkc (CUDA side only; the CPU oracle shares nothing
// with this file).  Arithmetic contract: include/kc.h ("Arithmetic"), north_star.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "../../include/kc.h"

#define KC_NOIDX 0x7fffffff

namespace kc {

void set_error(const char *fmt, ...);
void count_launches(int n);   // host-side tally of kernel launches issued by the library
kc_status cuda_fail(cudaError_t e, const char *where);

// Device-side error word: ONE int per process in pinned host memory that kernels can write through
// its device pointer (zero-copy).  A kernel that meets a state it cannot serve (e.g. a workspace
// that was not zero-filled, kc.h) stores a code there instead of trapping -- a trap would poison
// the CUDA context for the whole process -- and the next libkc call that checks the word reports
// it as a status.  error_word_init() allocates it (cudaHostAlloc: call outside stream capture);
// error_word_dev() is the pointer kernels get (nullptr until initialised: they then skip the store).
enum { KC_DEVERR_NONE = 0, KC_DEVERR_TICKETS = 1 };
void error_word_init();
int *error_word_dev();
int error_word_take();        // host: read and clear (0 when none or not initialised)

#define KC_CUDA(call)                                              \
    do {                                                           \
        cudaError_t e_ = (call);                                   \
        if (e_ != cudaSuccess) return kc::cuda_fail(e_, #call);    \
    } while (0)
#define KC_LAUNCH_CHECK(name)                                      \
    do {                                                           \
        cudaError_t e_ = cudaGetLastError();                       \
        if (e_ != cudaSuccess) return kc::cuda_fail(e_, name);     \
    } while (0)

// Squared distance, separately rounded binary32 ops in the fixed order ((dx*dx)+(dy*dy))+(dz*dz).
// __f*_rn intrinsics are never contracted into FMA by nvcc (and the library is built -fmad=false).
__device__ __forceinline__ float sqd2(float ax, float ay, float bx, float by)
{
    float dx = __fsub_rn(ax, bx), dy = __fsub_rn(ay, by);
    return __fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy));
}
__device__ __forceinline__ float sqd3(float ax, float ay, float az, float bx, float by, float bz)
{
    float dx = __fsub_rn(ax, bx), dy = __fsub_rn(ay, by), dz = __fsub_rn(az, bz);
    return __fadd_rn(__fadd_rn(__fmul_rn(dx, dx), __fmul_rn(dy, dy)), __fmul_rn(dz, dz));
}

// Running two smallest keys under the total order (s, j): equal s -> smaller index first.
struct Top2 {
    float s1, s2;
    int j1, j2;
    __device__ __forceinline__ void init()
    {
        s1 = CUDART_INF_F; s2 = CUDART_INF_F; j1 = KC_NOIDX; j2 = KC_NOIDX;
    }
    __device__ __forceinline__ void offer(float s, int j)
    {
        if (s < s1 || (s == s1 && j < j1)) {
            s2 = s1; j2 = j1; s1 = s; j1 = j;
        } else if (s < s2 || (s == s2 && j < j2)) {
            s2 = s; j2 = j;
        }
    }
    __device__ __forceinline__ void merge(const Top2 &o)
    {
        offer(o.s1, o.j1);
        offer(o.s2, o.j2);
    }
};

// Branch-free (s, j)-ordered insertion (converged code for loops whose lanes all insert).
__device__ __forceinline__ void insert_bf(Top2 &b, float s, int j, bool valid)
{
    const bool lt1 = valid && (s < b.s1 || (s == b.s1 && j < b.j1));
    const bool lt2 = valid && (s < b.s2 || (s == b.s2 && j < b.j2));   // lt1 implies lt2
    const float ns2 = lt1 ? b.s1 : s;
    const int nj2 = lt1 ? b.j1 : j;
    b.s2 = lt2 ? ns2 : b.s2; b.j2 = lt2 ? nj2 : b.j2;
    b.s1 = lt1 ? s : b.s1; b.j1 = lt1 ? j : b.j1;
}
// Smallest key (s, j) over the warp's private lists, removed from the list that held it (all 32
// lanes call it; two calls give the two smallest keys of the union).
__device__ __forceinline__ void warp_pop(Top2 &tmp, float &s, int &j)
{
    const unsigned key = __float_as_uint(tmp.s1);              // s >= 0 or +inf: ordered as unsigned
    const unsigned m = __reduce_min_sync(0xffffffffu, key);
    j = __reduce_min_sync(0xffffffffu, key == m ? tmp.j1 : KC_NOIDX);
    s = __uint_as_float(m);
    if (key == m && tmp.j1 == j) {
        tmp.s1 = tmp.s2; tmp.j1 = tmp.j2;
        tmp.s2 = CUDART_INF_F; tmp.j2 = KC_NOIDX;
    }
}

// Definition 1: d1 = sqrtf(s1), d2 = sqrtf(s2), c = d2 - d1.
__device__ __forceinline__ void store_cert(const Top2 &t, int i, int32_t *nn, int32_t *nn2,
                                           float *d1, float *d2, float *c)
{
    float a = __fsqrt_rn(t.s1), b = __fsqrt_rn(t.s2);
    nn[i] = t.j1 == KC_NOIDX ? -1 : t.j1;
    if (nn2) nn2[i] = t.j2 == KC_NOIDX ? -1 : t.j2;
    d1[i] = a;
    d2[i] = b;
    c[i] = __fsub_rn(b, a);
}

// Block-wide stream compaction shared by the classify kernels (A4 and its clock / local-budget
// forms): every thread of a 256-thread block brings up to 4 consecutive candidate ids as the bits of
// `bits` (id = base + k for bit k); the block reserves one range of list[] with a single atomicAdd
// on *cursor and writes its ids ascending inside it.  Every thread of the block must call it.
__device__ __forceinline__ void block_append_ids(unsigned bits, int64_t base, int32_t *__restrict__ list, int32_t *cursor)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int cnt = __popc(bits);
    int incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    __shared__ int wsum[8];
    __shared__ int bbase;
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    if (threadIdx.x == 0) {
        int tot = 0;
#pragma unroll
        for (int w = 0; w < 8; ++w) { const int t = wsum[w]; wsum[w] = tot; tot += t; }
        bbase = tot ? atomicAdd(cursor, tot) : 0;
    }
    __syncthreads();
    int pos = bbase + wsum[warp] + incl - cnt;
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (bits & (1u << k)) list[pos++] = (int32_t)(base + k);
}

// Cell coordinate on one axis (kc_geom comment): clamp(floorf(fl(fl(x - lo) * inv_h)), 0, G-1).
__device__ __forceinline__ int cell_axis(float x, float lo, float inv_h, int G)
{
    float t = __fmul_rn(__fsub_rn(x, lo), inv_h);
    float f = floorf(t);
    int k = f < 0.0f ? 0 : (f > (float)(G - 1) ? G - 1 : (int)f);
    return k;
}

// NEXT #4 (reading R20): the K smallest keys under the same total order (s, j), ascending.
// K is a compile-time constant, so the list lives in registers; a new key replaces the worst one
// and bubbles up through K-1 compare-exchanges written as selects.
template <int K>
struct TopK {
    float s[K];
    int j[K];
    __device__ __forceinline__ void init()
    {
#pragma unroll
        for (int q = 0; q < K; ++q) { s[q] = CUDART_INF_F; j[q] = KC_NOIDX; }
    }
    __device__ __forceinline__ bool holds(int id) const
    {
        bool h = false;
#pragma unroll
        for (int q = 0; q < K; ++q) h |= j[q] == id;
        return h;
    }
    __device__ __forceinline__ void offer(float x, int id)
    {
        if (!(x < s[K - 1] || (x == s[K - 1] && id < j[K - 1]))) return;
        s[K - 1] = x; j[K - 1] = id;
#pragma unroll
        for (int q = K - 1; q > 0; --q) {
            const bool sw = s[q] < s[q - 1] || (s[q] == s[q - 1] && j[q] < j[q - 1]);
            const float ts = s[q];
            const int tj = j[q];
            s[q] = sw ? s[q - 1] : ts; j[q] = sw ? j[q - 1] : tj;
            s[q - 1] = sw ? ts : s[q - 1]; j[q - 1] = sw ? tj : j[q - 1];
        }
    }
    // dk[q] = sqrtf(s_q); ck = dk[K-1] - dk[K-2], +inf when the list is short (kc.h)
    __device__ __forceinline__ void store(int64_t i, int32_t *nnk, float *dk, float *ck) const
    {
        float dq[K];
#pragma unroll
        for (int q = 0; q < K; ++q) {
            dq[q] = __fsqrt_rn(s[q]);
            nnk[i * K + q] = j[q] == KC_NOIDX ? -1 : j[q];
            dk[i * K + q] = dq[q];
        }
        ck[i] = s[K - 1] == CUDART_INF_F ? CUDART_INF_F : __fsub_rn(dq[K - 1], dq[K - 2]);
    }
};

}  // namespace kc
