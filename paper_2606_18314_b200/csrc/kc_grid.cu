// kc_grid.cu — the resident grid: A2 build (two-level counting sort), A5 frontier entropy, A6
// incremental cell update, NEXT #2 local motion budget.  Searches: kc_search.cu.  Contract: include/kc.h.
//
// Layout in HBM (N points, C_tot level-0 cells; shared declarations in kc_grid.cuh):
//   cell[N]        int32   current filing cell of point i
//   counts[C_tot]  int32   live occupancy per cell (histogram, kept current by A6)
//   cell_start[C_tot+1] int32  exclusive scan of the build histogram
//   subinfo[C_tot] int2    two-level index: {S, first leaf} of every cell (S = 0: not subdivided)
//   leaf_start[n_leaves+1] int32  exclusive scan of the leaf sizes (entry l+1 doubles as the scatter
//                           cursor of leaf l during the build)
//   spos2[N] float2 (d=2) / spos4[N] float4 = (x,y,z,bits(idx)) (d=3)   leaf-sorted positions
//   sidx[N]        int32   point id per sorted slot (-1 = tombstone); d = 2 only: a d = 3 record carries its id
//   slot[N]        int32   sorted slot of point i (-1 = lives in an overflow chain)
//   head[C_tot], next[N], opos[N] float4, mlist[N]   overflow chains of re-filed points (A6)
//   fcount[C_tot], mhist[]  scratch of A5 (always left zeroed)
// Rows of cells along x are contiguous in the sorted arrays (linear id has x fastest), so a
// (2r+1)-cell row segment is ONE contiguous candidate range: two cell_start reads per row; the same
// holds for the sub-cells of a subdivided cell and leaf_start.
#include <new>

#include "kc_grid.cuh"

using namespace kc;

namespace {

constexpr int MHIST = 4096;   // frontier-count histogram bins held exactly; larger counts go to `big`
constexpr int SCAN_CHUNK = 2048;   // entries per scan block (256 threads x 8)
// A6: when an update re-bins instead of re-filing: grids of >= REBIN_MIN_N points, host-side bound of at least
// N / 8 movers (d = 2) or N / list_div3(N) (d = 3: N / 8 on small grids, N / 32 from a million points on, where
// chain residents would be served one thread per query and a fresh grid lets the slot sweep take them:
// 10 % movers of 4,194,304 clustered points 1.15 -> 0.68 ms).
constexpr int64_t REBIN_MIN_N = 100000, REBIN_DIV2 = 8;

// ------------------------------------------------------------------ A2 build
// A counting sort in two levels.  (1) prep: drop the chains of the previous residency, zero the
// histograms.  (2) cell id per point + level-0 histogram (one RED per point).  (3) scan over the
// cells: cell_start, and per cell the sub-resolution S and the index of its first leaf.  (4) only
// if some cell is subdivided: leaf of every point + leaf histogram.  (5) scan over the leaves.
// (6) scatter by leaf (returning atomic on the leaf's cursor).  Without a subdivided cell the
// leaves ARE the cells, steps 4-5 leave at once and the cell scan writes the cursors itself.
__global__ void clear_chains_kernel(const int32_t *__restrict__ mlist, const int32_t *__restrict__ cell,
                                    int32_t *head, const Counters *ctr)
{
    int n = ctr->n_misfiled;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x)
        head[cell[mlist[e]]] = -1;
}
__device__ __forceinline__ void zero_i32(int32_t *a, int64_t n, int64_t t0, int64_t nt)
{
    int4 *a4 = reinterpret_cast<int4 *>(a);                // cudaMalloc'ed: 256-byte aligned
    for (int64_t k = t0; k < n / 4; k += nt) a4[k] = make_int4(0, 0, 0, 0);
    for (int64_t k = (n & ~(int64_t)3) + t0; k < n; k += nt) a[k] = 0;
}
__global__ void __launch_bounds__(256)
build_prep_kernel(const int32_t *__restrict__ mlist, const int32_t *__restrict__ cell, int32_t *head,
                  Counters *ctr, int32_t *counts, int n_cells, int32_t *leaf_cnt, int64_t n_leaves_max,
                  unsigned long long *desc, int n_desc)
{
    const int n = ctr->n_misfiled;
    const int64_t t0 = blockIdx.x * (int64_t)blockDim.x + threadIdx.x, nt = (int64_t)gridDim.x * blockDim.x;
    for (int64_t e = t0; e < n; e += nt) head[cell[mlist[e]]] = -1;
    for (int64_t k = t0; k < n_desc; k += nt) desc[k] = 0ull;       // the scans' descriptors and tickets
    if (t0 == 0) { ctr->scan_ticket = 0; ctr->lscan_ticket = 0; }
    zero_i32(counts, n_cells, t0, nt);
    zero_i32(leaf_cnt, n_leaves_max, t0, nt);
}

template <int D>
__global__ void __launch_bounds__(256)
cellid_hist_kernel(View v, const float *__restrict__ p, int N, int32_t *__restrict__ cell,
                   int32_t *counts, Counters *ctr)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i == 0) {          // the chains were dropped by the previous kernel; the scan recounts C
        ctr->n_misfiled = 0; ctr->c_occ = 0; ctr->max_occ = 0; ctr->n_stragglers = 0;
        ctr->n_list2 = 0; ctr->n_heavy = 0; ctr->n_leaves = 0; ctr->n_handed = 0; ctr->n_deferred = 0;
    }
    if (i >= N) return;
    float x, y, z = 0.f;
    if (D == 2) {
        float2 t = reinterpret_cast<const float2 *>(p)[i];
        x = t.x; y = t.y;
    } else {
        x = p[3 * (int64_t)i]; y = p[3 * (int64_t)i + 1]; z = p[3 * (int64_t)i + 2];
    }
    int cidx = cell_of<D>(v, x, y, z);
    cell[i] = cidx;
    atomicAdd(&counts[cidx], 1);                  // result unused: compiles to a RED
}

__device__ __forceinline__ int ipow_d(int S, int d) { return d == 2 ? S * S : S * S * S; }

// Exclusive scan over the block of one pair per thread; wsum: shared int2[32]; returns this
// thread's exclusive offsets.  Every thread of the block must call it.
__device__ __forceinline__ int2 block_excl_scan2(int a, int b, int2 *wsum)
{
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
    int ia = a, ib = b;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int ta = __shfl_up_sync(0xffffffffu, ia, o), tb = __shfl_up_sync(0xffffffffu, ib, o);
        if (lane >= o) { ia += ta; ib += tb; }
    }
    __syncthreads();                               // wsum may still be read from a previous call
    if (lane == 31) wsum[w] = make_int2(ia, ib);
    __syncthreads();
    if (w == 0) {
        const int2 x = lane < nw ? wsum[lane] : make_int2(0, 0);
        int xa = x.x, xb = x.y;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int ta = __shfl_up_sync(0xffffffffu, xa, o), tb = __shfl_up_sync(0xffffffffu, xb, o);
            if (lane >= o) { xa += ta; xb += tb; }
        }
        wsum[lane] = make_int2(xa - x.x, xb - x.y);   // exclusive warp offsets
    }
    __syncthreads();
    const int2 off = wsum[w];
    return make_int2(off.x + ia - a, off.y + ib - b);
}

// ---- scans in one pass (decoupled look-back) ----------------------------------------------------
// A scan block takes a ticket (blocks with smaller tickets are running or done, so waiting for them
// cannot deadlock), publishes the sums of its chunk, and adds up its predecessors' descriptors until
// it meets one that already carries an inclusive prefix.  A descriptor is one 64-bit word -- state
// (0 nothing yet, 1 the block's own sums, 2 inclusive prefix) in the top two bits, two 31-bit sums
// below -- so a single volatile load or store moves state and values together (no fence needed).
// build_prep_kernel zeroes the descriptors and the tickets.
__device__ __forceinline__ unsigned long long desc_pack(int st, int a, int b)
{
    return ((unsigned long long)st << 62) | ((unsigned long long)(unsigned)a << 31) | (unsigned long long)(unsigned)b;
}
// Called by all 32 lanes of ONE warp of the block: exclusive prefix of block `bid` whose own sums are (a, b).
__device__ __forceinline__ int2 scan_lookback(volatile unsigned long long *desc, int bid, int a, int b)
{
    const int lane = threadIdx.x & 31;
    if (bid == 0) {
        if (lane == 0) desc[0] = desc_pack(2, a, b);
        return make_int2(0, 0);
    }
    if (lane == 0) desc[bid] = desc_pack(1, a, b);
    int ra = 0, rb = 0;
    for (int look = bid - 1;; look -= 32) {
        const int idx = look - lane;               // lane 0 reads the nearest predecessor
        unsigned long long dsc;
        do {
            dsc = idx >= 0 ? desc[idx] : desc_pack(2, 0, 0);
        } while (__any_sync(0xffffffffu, (dsc >> 62) == 0));
        const unsigned full = __ballot_sync(0xffffffffu, (dsc >> 62) == 2);
        const bool take = !full || lane <= __ffs(full) - 1;
        ra += __reduce_add_sync(0xffffffffu, take ? (int)((dsc >> 31) & 0x7fffffffu) : 0);
        rb += __reduce_add_sync(0xffffffffu, take ? (int)(dsc & 0x7fffffffu) : 0);
        if (full) break;
    }
    if (lane == 0) desc[bid] = desc_pack(2, ra + a, rb + b);
    return make_int2(ra, rb);
}

// ---- scan over the cells: {records, leaves} --------------------------------------------------
// Thread t owns 8 consecutive cells of the block's chunk; the chunk goes through shared memory both
// ways so that the global loads and stores are coalesced.  Whether any cell of the grid is
// subdivided is not known before the last block is done, so with the second level enabled a cell
// gets both forms of its output: {cell_start, scatter cursor} for a grid without subdivided cells
// (leaf = cell) and {subinfo, size of the single leaf of an undivided cell} for one with; the leaf
// scan, which runs only in the second case, overwrites every cursor (n_leaves >= n_cells).
__global__ void __launch_bounds__(256)
scan_cells_kernel(const int32_t *__restrict__ counts, int n_cells, int d, int heavy_T, int sub_occ, bool two_level,
                  unsigned long long *desc, int32_t *__restrict__ cell_start, int2 *__restrict__ subinfo,
                  int32_t *__restrict__ leaf_cnt, int32_t *__restrict__ leaf_start, Counters *ctr, int N)
{
    __shared__ int2 wsum[32];
    __shared__ int s_cnt[SCAN_CHUNK];              // counts in, starts out
    __shared__ int2 s_sub[SCAN_CHUNK];
    __shared__ int s_bid;
    __shared__ int2 s_agg, s_pre;
    if (threadIdx.x == 0) s_bid = atomicAdd(&ctr->scan_ticket, 1);
    __syncthreads();
    const int bid = s_bid, cbase = bid * SCAN_CHUNK;
#pragma unroll
    for (int k = 0; k < SCAN_CHUNK / 256; ++k) {
        const int c = cbase + k * 256 + threadIdx.x;
        s_cnt[k * 256 + threadIdx.x] = c < n_cells ? counts[c] : 0;
    }
    __syncthreads();
    const int lbase = threadIdx.x * 8, base = cbase + lbase;
    int v[8], S[8];
    int tsum = 0, tl = 0, occ = 0, mx = 0, hv = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        v[k] = s_cnt[lbase + k];
        S[k] = sub_res(v[k], d, heavy_T, sub_occ);
        tsum += v[k]; occ += v[k] > 0; mx = max(mx, v[k]); hv += S[k] > 0;
        tl += base + k < n_cells ? (S[k] ? ipow_d(S[k], d) : 1) : 0;
    }
    const int2 e = block_excl_scan2(tsum, tl, wsum);      // (syncs: every thread has read its counts)
    if (threadIdx.x == 255) s_agg = make_int2(e.x + tsum, e.y + tl);
    occ = __reduce_add_sync(0xffffffffu, occ);
    hv = __reduce_add_sync(0xffffffffu, hv);
    mx = __reduce_max_sync(0xffffffffu, mx);
    if ((threadIdx.x & 31) == 0) {
        if (occ) atomicAdd(&ctr->c_occ, occ);
        if (hv) atomicAdd(&ctr->n_heavy, hv);
        if (mx) atomicMax(&ctr->max_occ, mx);
    }
    __syncthreads();
    if (threadIdx.x < 32) {
        const int2 pre = scan_lookback(desc, bid, s_agg.x, s_agg.y);
        if (threadIdx.x == 0) s_pre = pre;
    }
    __syncthreads();
    const int2 off = s_pre;
    int run = off.x + e.x, lrun = off.y + e.y;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        s_cnt[lbase + k] = run;
        s_sub[lbase + k] = make_int2(S[k], lrun);
        // an undivided cell of a grid with subdivided cells is one leaf of that size
        if (two_level && !S[k] && base + k < n_cells) leaf_cnt[lrun] = v[k];
        run += v[k];
        lrun += base + k < n_cells ? (S[k] ? ipow_d(S[k], d) : 1) : 0;
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < SCAN_CHUNK / 256; ++k) {
        const int c = cbase + k * 256 + threadIdx.x;
        if (c < n_cells) {
            const int st = s_cnt[k * 256 + threadIdx.x];
            cell_start[c] = st;
            leaf_start[c + 1] = st;                // leaf = cell: the scatter's cursor straight away
            if (two_level) subinfo[c] = s_sub[k * 256 + threadIdx.x];
        }
    }
    if (threadIdx.x == 255 && cbase + SCAN_CHUNK >= n_cells && cbase < n_cells) {   // the last chunk
        ctr->n_leaves = lrun;
        cell_start[n_cells] = N;
        leaf_start[0] = 0;
    }
}
// ---- leaf of every point + leaf histogram (only with subdivided cells) ------------------------
template <int D>
__global__ void __launch_bounds__(256)
leafid_hist_kernel(View v, const float *__restrict__ p, int N, const int32_t *__restrict__ cell,
                   int32_t *leaf_cnt, int32_t *__restrict__ leafid, const Counters *ctr)
{
    if (ctr->n_heavy == 0) return;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int2 si = v.subinfo[cell[i]];
    int leaf = si.y;
    if (si.x) {
        float x, y, z = 0.f;
        if (D == 2) {
            float2 t = reinterpret_cast<const float2 *>(p)[i];
            x = t.x; y = t.y;
        } else {
            x = p[3 * (int64_t)i]; y = p[3 * (int64_t)i + 1]; z = p[3 * (int64_t)i + 2];
        }
        const int S = si.x;
        const float fS = (float)S;
        const int ux = sub_axis(x, v.lo0, v.inv_h, cell_axis(x, v.lo0, v.inv_h, v.G0), fS, S);
        const int uy = sub_axis(y, v.lo1, v.inv_h, cell_axis(y, v.lo1, v.inv_h, v.G1), fS, S);
        const int uz = D == 3 ? sub_axis(z, v.lo2, v.inv_h, cell_axis(z, v.lo2, v.inv_h, v.G2), fS, S) : 0;
        leaf += (uz * S + uy) * S + ux;
        atomicAdd(&leaf_cnt[leaf], 1);            // RED
    }
    leafid[i] = leaf;
}

// ---- scan over the leaves: leaf_start[l + 1] = start of leaf l (the scatter's cursor) ----------
// One pass, as above (second component unused); blocks behind the last leaf leave at once.
__global__ void __launch_bounds__(256)
lscan_kernel(const int32_t *__restrict__ leaf_cnt, unsigned long long *desc, int32_t *__restrict__ leaf_start,
             Counters *ctr)
{
    if (ctr->n_heavy == 0) return;
    __shared__ int2 wsum[32];
    __shared__ int s_cnt[SCAN_CHUNK];              // sizes in, starts out (coalesced both ways)
    __shared__ int s_bid, s_agg, s_pre;
    if (threadIdx.x == 0) s_bid = atomicAdd(&ctr->lscan_ticket, 1);
    __syncthreads();
    const int n = ctr->n_leaves;
    const int bid = s_bid, cbase = bid * SCAN_CHUNK;
    if (cbase >= n) return;
#pragma unroll
    for (int k = 0; k < SCAN_CHUNK / 256; ++k) {
        const int l = cbase + k * 256 + threadIdx.x;
        s_cnt[k * 256 + threadIdx.x] = l < n ? leaf_cnt[l] : 0;
    }
    __syncthreads();
    const int lbase = threadIdx.x * 8;
    int v[8];
    int tsum = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        v[k] = s_cnt[lbase + k];
        tsum += v[k];
    }
    const int2 e = block_excl_scan2(tsum, 0, wsum);
    if (threadIdx.x == 255) s_agg = e.x + tsum;
    __syncthreads();
    if (threadIdx.x < 32) {
        const int2 pre = scan_lookback(desc, bid, s_agg, 0);
        if (threadIdx.x == 0) s_pre = pre.x;
    }
    __syncthreads();
    int run = s_pre + e.x;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        s_cnt[lbase + k] = run;
        run += v[k];
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < SCAN_CHUNK / 256; ++k) {
        const int l = cbase + k * 256 + threadIdx.x;
        if (l < n) leaf_start[l + 1] = s_cnt[k * 256 + threadIdx.x];
    }
}
template <int D>
__global__ void __launch_bounds__(256)
scatter_kernel(const float *__restrict__ p, int N, const int32_t *__restrict__ cell,
               const int32_t *__restrict__ leafid, int32_t *leaf_start, const Counters *ctr,
               float2 *__restrict__ spos2, float4 *__restrict__ spos4, int32_t *__restrict__ sidx,
               int32_t *__restrict__ slot)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < 8) {                                  // inert padding behind the last slot
        const float qnan = __int_as_float(0x7fc00000);
        if (D == 2) spos2[N + i] = make_float2(qnan, qnan);
        else spos4[N + i] = make_float4(qnan, qnan, qnan, __int_as_float(-1));
        sidx[N + i] = -1;
    }
    if (i >= N) return;
    // (inputs are read once: streaming loads, so that they do not push the sorted arrays out of L2)
    const int leaf = ctr->n_heavy ? __ldcs(leafid + i) : __ldcs(cell + i);
    int s = atomicAdd(&leaf_start[leaf + 1], 1);
    // The sorted arrays are written at random slots, a fraction of a 32-byte sector at a time: the
    // stores ask L2 to keep their sectors (evict_last) so that a sector is completed in L2 and
    // written back once instead of being evicted half-written and filled again.
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    if (D == 2) {
        const float2 r = __ldcs(reinterpret_cast<const float2 *>(p) + i);
        asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(spos2 + s), "f"(r.x), "f"(r.y), "l"(pol) : "memory");
        asm volatile("st.global.L2::cache_hint.b32 [%0], %1, %2;" ::"l"(sidx + s), "r"(i), "l"(pol) : "memory");
    } else {
        const float x = __ldcs(p + 3 * (int64_t)i), y = __ldcs(p + 3 * (int64_t)i + 1), z = __ldcs(p + 3 * (int64_t)i + 2);
        asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(spos4 + s), "f"(x), "f"(y), "f"(z),
                     "f"(__int_as_float(i)), "l"(pol) : "memory");   // d = 3: the id travels in the record's fourth word
    }
    __stcs(slot + i, s);
}

// ------------------------------------------------------------------ A6 incremental update
// Algorithm 1 line 3: "update cell_i in G for points that changed cell".
// A mover whose cell is unchanged is overwritten in its sorted slot; one whose cell changed is
// tombstoned (NaN coordinates: every comparison with NaN is false, so it is never selected) and
// appended once to the misfiled list; misfiled points live in per-cell overflow chains that are
// cleared and re-linked every call, O(#misfiled).
template <int D>
__global__ void __launch_bounds__(256)
refresh_kernel(View v, const float *__restrict__ p_new, int N, const int32_t *__restrict__ movers,
               const int32_t *__restrict__ n_movers, int32_t *cell, int32_t *slot, int32_t *sidx,
               float2 *spos2, float4 *spos4, float4 *opos, int32_t *mlist, int32_t *counts,
               Counters *ctr)
{
    const int n = movers ? *n_movers : N;
    const int stride = gridDim.x * blockDim.x;
    for (int k0 = blockIdx.x * blockDim.x; k0 < n; k0 += stride) {     // warp-uniform trip count
        const int k = k0 + threadIdx.x;
        bool misfile = false;
        int i = -1;
        if (k < n) {
            i = movers ? movers[k] : k;
            float x = p_new[(int64_t)i * D], y = p_new[(int64_t)i * D + 1];
            float z = D == 3 ? p_new[(int64_t)i * D + 2] : 0.f;
            int cnew = cell_of<D>(v, x, y, z);
            int cold = cell[i];
            int sl = slot[i];
            bool in_chain = sl < 0;
            if (sl >= 0) {
                bool stay = cnew == cold;
                if (stay && v.cell_start[cold + 1] - v.cell_start[cold] >= v.heavy_T) {
                    // subdivided cell: the record keeps its slot only if it also stays in its
                    // sub-cell (the slot still holds the position it was filed under)
                    const int S = v.subinfo[cold].x;
                    const float fS = (float)S;
                    float ox, oy, oz = 0.f;
                    if (D == 2) { const float2 o = spos2[sl]; ox = o.x; oy = o.y; }
                    else { const float4 o = spos4[sl]; ox = o.x; oy = o.y; oz = o.z; }
                    const int kx = cell_axis(x, v.lo0, v.inv_h, v.G0), ky = cell_axis(y, v.lo1, v.inv_h, v.G1);
                    const int kz = D == 3 ? cell_axis(z, v.lo2, v.inv_h, v.G2) : 0;
                    stay = sub_axis(x, v.lo0, v.inv_h, kx, fS, S) == sub_axis(ox, v.lo0, v.inv_h, kx, fS, S) &&
                           sub_axis(y, v.lo1, v.inv_h, ky, fS, S) == sub_axis(oy, v.lo1, v.inv_h, ky, fS, S) &&
                           (D == 2 || sub_axis(z, v.lo2, v.inv_h, kz, fS, S) == sub_axis(oz, v.lo2, v.inv_h, kz, fS, S));
                }
                if (stay) {
                    if (D == 2) spos2[sl] = make_float2(x, y);
                    else spos4[sl] = make_float4(x, y, z, __int_as_float(i));
                } else {
                    const float qnan = __int_as_float(0x7fc00000);
                    if (D == 2) spos2[sl] = make_float2(qnan, qnan);
                    else spos4[sl] = make_float4(qnan, qnan, qnan, __int_as_float(-1));
                    if (D == 2) sidx[sl] = -1;
                    slot[i] = -1;
                    misfile = true;
                    in_chain = true;
                }
            }
            if (in_chain) opos[i] = make_float4(x, y, z, 0.f);
            if (cnew != cold) {
                cell[i] = cnew;
                // occupancy follows with fire-and-forget REDs; C is recounted by A5 when it is
                // asked for (returning atomics here cost 0.3 ms at 4 M movers)
                atomicSub(&counts[cold], 1);
                atomicAdd(&counts[cnew], 1);
            }
        }
        warp_append(misfile, i, mlist, &ctr->n_misfiled);
    }
}
__global__ void link_chains_kernel(const int32_t *__restrict__ mlist, const int32_t *__restrict__ cell,
                                   int32_t *head, int32_t *next, Counters *ctr)
{
    int n = ctr->n_misfiled;
    if (blockIdx.x == 0 && threadIdx.x == 0) ctr->n_list2 = 0;
    for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n; e += gridDim.x * blockDim.x) {
        int i = mlist[e];
        next[i] = atomicExch(&head[cell[i]], i);
    }
}

// ------------------------------------------------------------------ A5 frontier entropy
// Definition 2 with n = |F|, k = frontier points per cell:
//   H = ( ln n - (1/n) sum_cells k ln k ) / ln C.
// Counts are integers (atomics), the sum is taken over the histogram-of-counts M[k] in a fixed
// order in double, so the result does not depend on atomic ordering.
__global__ void __launch_bounds__(256)
entropy_count_kernel(const int32_t *__restrict__ F, const int32_t *__restrict__ nF,
                     const int32_t *__restrict__ cell, int32_t *fcount, const int32_t *__restrict__ counts,
                     int n_cells, int recount, Counters *ctr)
{
    if (recount) {                      // C = occupied cells at the current filing
        int occ = 0;
        for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n_cells; k += gridDim.x * blockDim.x)
            occ += counts[k] > 0;
        occ = __reduce_add_sync(0xffffffffu, occ);
        if ((threadIdx.x & 31) == 0 && occ) atomicAdd(&ctr->c_occ_acc, occ);
    }
    int n = *nF;
    for (int f = blockIdx.x * blockDim.x + threadIdx.x; f < n; f += gridDim.x * blockDim.x)
        atomicAdd(&fcount[cell[F[f]]], 1);
}
__global__ void __launch_bounds__(256)
entropy_collect_kernel(const int32_t *__restrict__ F, const int32_t *__restrict__ nF,
                       const int32_t *__restrict__ cell, int32_t *fcount, int32_t *mhist, Counters *ctr,
                       int recount, double *H, int32_t *m_cells, int32_t *C_occ)
{
    // almost every cell holds a handful of frontier points, so the low bins of M[k] would take one
    // global atomic per cell on a few addresses: they are aggregated per block in shared memory
    constexpr int LOW = 64;
    __shared__ int low[LOW];
    if (threadIdx.x < LOW) low[threadIdx.x] = 0;
    __syncthreads();
    int n = *nF;
    int m_local = 0;
    int c1 = 0, c2 = 0, c3 = 0, c4 = 0;             // the commonest counts stay in registers
    int kmax_local = 0;
    for (int f = blockIdx.x * blockDim.x + threadIdx.x; f < n; f += gridDim.x * blockDim.x) {
        int k = atomicExch(&fcount[cell[F[f]]], 0);     // first visitor collects and re-zeroes
        if (k > 0) {
            ++m_local;
            kmax_local = max(kmax_local, k);
            c1 += k == 1; c2 += k == 2; c3 += k == 3; c4 += k == 4;
            if (k > 4) {
                if (k < LOW) atomicAdd(&low[k], 1);
                else if (k < MHIST) atomicAdd(&mhist[k], 1);
                else atomicAdd(&ctr->big, (double)k * log((double)k));
            }
        }
    }
    m_local = __reduce_add_sync(0xffffffffu, m_local);
    c1 = __reduce_add_sync(0xffffffffu, c1); c2 = __reduce_add_sync(0xffffffffu, c2);
    c3 = __reduce_add_sync(0xffffffffu, c3); c4 = __reduce_add_sync(0xffffffffu, c4);
    kmax_local = __reduce_max_sync(0xffffffffu, kmax_local);
    if ((threadIdx.x & 31) == 0) {
        if (kmax_local > 4) atomicMax(&ctr->kmax, kmax_local);
        if (m_local) atomicAdd(&ctr->m_cells, m_local);
        if (c1) atomicAdd(&low[1], c1);
        if (c2) atomicAdd(&low[2], c2);
        if (c3) atomicAdd(&low[3], c3);
        if (c4) atomicAdd(&low[4], c4);
    }
    __syncthreads();
    if (threadIdx.x < LOW && low[threadIdx.x]) atomicAdd(&mhist[threadIdx.x], low[threadIdx.x]);
    // the block that takes the last ticket evaluates H from the finished histogram-of-counts
    // (fixed order, double: independent of atomic ordering) and leaves the scratch zeroed
    __shared__ int s_last;
    __shared__ double part[8];
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) s_last = atomicAdd(&ctr->ticket, 1) == (int)gridDim.x - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    double acc = 0.0;
    const int lim = min(MHIST, max(__ldcg(&ctr->kmax), 4) + 1);     // bins above the largest count are empty
    for (int k = threadIdx.x; k < lim; k += 256) {
        int M = __ldcg(&mhist[k]);
        if (M) {
            if (k > 1) acc += (double)M * ((double)k * log((double)k));
            mhist[k] = 0;
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc += __shfl_down_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double S = __ldcg(&ctr->big);
        for (int w = 0; w < 8; ++w) S += part[w];
        int C = ctr->c_occ;
        if (recount) {
            C = __ldcg(&ctr->c_occ_acc);
            ctr->c_occ = C;
            ctr->c_occ_acc = 0;
        }
        double h = 0.0;
        if (n > 0 && C > 1) h = (log((double)n) - S / (double)n) / log((double)C);
        *H = h;
        if (m_cells) *m_cells = __ldcg(&ctr->m_cells);
        if (C_occ) *C_occ = C;
        ctr->m_cells = 0;
        ctr->big = 0.0;
        ctr->ticket = 0;
        ctr->kmax = 0;
    }
}

// ------------------------------------------------------------------ NEXT #2: local motion budget
// "A per-point motion budget would tighten the safe set without affecting the no-miss guarantee"
// (PAPER.md:127).  With delta_k = ||p'_k - p_k|| the displacement of point k, a = nn_i, B(i) the 3^d
// cell block around i's (pre-step) cell and Delta_B(i) = max of delta_k over the points filed in
// B(i), certificate i keeps its nearest neighbour if
//   (1)  c_i > 2 delta_i + delta_a + Delta_B(i)          (every k in the block stays behind a), and
//   (2)  R   > d1_i + 2 delta_i + delta_a + eps_t         (every k outside the block, at distance
//                                                          >= R ~ h before the step, stays behind a),
// by the triangle-inequality argument of Lemma 1 with the individual displacements in
// place of eps.  Lemma 1's own test c_i > 4 eps_t remains a sufficient alternative.  The frontier is
//   F_local = { i : not ( c_i > 4 eps_t  or  ((1) and (2)) ) }  (a subset of Lemma 1's set),
// and it shrinks with the number of movers, which the global rule does not (reading R12).
// All tests in float32, fixed operation order, right-hand sides inflated by K = 1 + 2^-18 plus
// 2^-18 d2_i for the roundings of c, d1, delta (reading R19); the oracle restates them.
__global__ void __launch_bounds__(256)
motion_field_kernel(int D, const float *__restrict__ p, const float *__restrict__ p2, int N,
                    const int32_t *__restrict__ cell, float *__restrict__ delta, unsigned *cellmax)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    float s;
    if (D == 2) s = sqd2(p2[2 * (int64_t)i], p2[2 * (int64_t)i + 1], p[2 * (int64_t)i], p[2 * (int64_t)i + 1]);
    else s = sqd3(p2[3 * (int64_t)i], p2[3 * (int64_t)i + 1], p2[3 * (int64_t)i + 2], p[3 * (int64_t)i],
                  p[3 * (int64_t)i + 1], p[3 * (int64_t)i + 2]);
    const float dl = __fsqrt_rn(s);
    delta[i] = dl;
    if (dl > 0.0f) atomicMax(&cellmax[cell[i]], __float_as_uint(dl));     // delta >= 0: bits are ordered
}

__global__ void __launch_bounds__(256)
classify_local_kernel(View v, float R, int N, const int32_t *__restrict__ cell,
                      const float *__restrict__ delta, const unsigned *__restrict__ cellmax,
                      const int32_t *__restrict__ nn, const float *__restrict__ d1, const float *__restrict__ c,
                      const float *__restrict__ eps, uint8_t *__restrict__ flags, int32_t *__restrict__ F,
                      int32_t *nF)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    bool infr = false;
    if (i < N) {
        const float e = *eps, ci = c[i];
        if (!(ci > __fmul_rn(4.0f, e))) {
            const float K = 1.0f + 1.0f / 262144.0f;
            const int cid = cell[i];
            const int cx = cid % v.G0, cy = (cid / v.G0) % v.G1, cz = cid / (v.G0 * v.G1);
            unsigned mx = 0;
            for (int z = max(cz - 1, 0); z <= min(cz + 1, v.G2 - 1); ++z)
                for (int y = max(cy - 1, 0); y <= min(cy + 1, v.G1 - 1); ++y)
                    for (int x = max(cx - 1, 0); x <= min(cx + 1, v.G0 - 1); ++x)
                        mx = max(mx, cellmax[(z * v.G1 + y) * v.G0 + x]);
            const float dB = __uint_as_float(mx);
            const int a = nn[i];
            const float di = delta[i], da = a >= 0 ? delta[a] : 0.0f, d1i = d1[i];
            const float two = __fmul_rn(2.0f, di);
            const float m = __fmul_rn(__fadd_rn(d1i, ci), 1.0f / 262144.0f);
            const float rhs1 = __fadd_rn(__fmul_rn(__fadd_rn(__fadd_rn(two, da), dB), K), m);
            const float rhs2 = __fadd_rn(__fmul_rn(__fadd_rn(__fadd_rn(__fadd_rn(d1i, two), da), e), K), m);
            infr = !(ci > rhs1 && R > rhs2);
        }
        if (flags) flags[i] = (uint8_t)infr;
    }
    block_append_ids(infr ? 1u : 0u, i, F, nF);      // ids ascending inside the block, one atomicAdd per block
}

__global__ void record_ids_kernel(const float4 *__restrict__ spos4, int n, int32_t *__restrict__ out)
{
    for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < n; t += gridDim.x * blockDim.x)
        out[t] = __float_as_int(spos4[t].w);
}

}  // namespace

// ====================================================================== C-ABI
extern "C" kc_status kc_grid_create(kc_grid **out, int64_t N_max, const kc_geom *geom)
{
    if (!out || !geom || N_max < 2 || N_max > 0x7ffffff0 || (geom->d != 2 && geom->d != 3) ||
        geom->G[0] < 1 || geom->G[1] < 1 || geom->G[2] < 1 || !(geom->h > 0.f) || !(geom->inv_h > 0.f) ||
        (geom->d == 2 && geom->G[2] != 1)) {
        set_error("kc_grid_create: bad argument");
        return KC_EINVAL;
    }
    int64_t n_cells = (int64_t)geom->G[0] * geom->G[1] * geom->G[2];
    int Gm = geom->G[0] > geom->G[1] ? geom->G[0] : geom->G[1];
    if (geom->G[2] > Gm) Gm = geom->G[2];
    if (n_cells > 0x7ffffff0 || Gm > 131072) {
        set_error("kc_grid_create: grid too large");
        return KC_EINVAL;
    }
    kc_grid *g = new (std::nothrow) kc_grid();
    if (!g) return KC_ENOMEM;
    g->geom = *geom;
    g->N_max = N_max; g->n_cells = n_cells; g->N = 0; g->built = 0; g->dirty = 0; g->bytes = 0;
    // leaves: one per undivided cell, S^d <= max(count / sub_occ, 2^d) per subdivided one
    g->n_leaves_max = n_cells + N_max + 8;
    if (g->n_leaves_max > 0x7ffffff0) {
        set_error("kc_grid_create: grid too large");
        delete g;
        return KC_EINVAL;
    }
    // two-level index defaults (measured on config 5): d = 3: cells of >= 128 records
    // are subdivided at ~4 records per sub-cell (LANE_T_MIN in kc_grid.cuh: from where a cell's own
    // queries use the sub-cells); d = 2: off (the plane's whole-set kernel prunes
    // cell by cell instead); kc_grid_set_index changes them
    g->sub_occ = 4;
    g->heavy_T = geom->d == 2 ? KC_INDEX_OFF : 128;
    g->n_scan_blocks = (int)((g->n_leaves_max + SCAN_CHUNK - 1) / SCAN_CHUNK);
    bool ok = true;
    auto alloc = [&](void **p, size_t bytes) {
        *p = nullptr;
        if (!ok) return;
        if (cudaMalloc(p, bytes) != cudaSuccess) { ok = false; *p = nullptr; cudaGetLastError(); return; }
        g->bytes += bytes;
    };
    size_t n = (size_t)N_max, nc = (size_t)n_cells;
    alloc((void **)&g->cell, n * 4);
    alloc((void **)&g->counts, nc * 4); alloc((void **)&g->cell_start, (nc + 1) * 4);
    alloc((void **)&g->sidx, (n + 8) * 4); alloc((void **)&g->slot, n * 4);
    alloc((void **)&g->head, nc * 4); alloc((void **)&g->next, n * 4);
    alloc((void **)&g->mlist, n * 4); alloc((void **)&g->fcount, nc * 4);
    alloc((void **)&g->mhist, MHIST * 4);
    alloc((void **)&g->scan_desc, (2 * (size_t)g->n_scan_blocks + 2) * sizeof(unsigned long long));
    alloc((void **)&g->subinfo, nc * sizeof(int2));
    alloc((void **)&g->leaf_cnt, (size_t)g->n_leaves_max * 4);
    alloc((void **)&g->leaf_start, ((size_t)g->n_leaves_max + 1) * 4);
    alloc((void **)&g->leafid, n * 4);
    alloc((void **)&g->mark, (n + 8) * 4);
    alloc((void **)&g->list2, n * 4);
    if (N_max >= HANDOFF_MIN_N) {
        alloc((void **)&g->handoff, (size_t)HANDOFF_CAP * sizeof(float4));
        alloc((void **)&g->handoff_part, (size_t)HANDOFF_CAP * HANDOFF_BLOCKS * sizeof(HandoffPart));
    }
    alloc((void **)&g->delta, n * 4); alloc((void **)&g->cellmax, nc * 4);
    g->spos2 = nullptr; g->spos4 = nullptr;
    if (geom->d == 2) alloc((void **)&g->spos2, (n + 8) * sizeof(float2));
    else alloc((void **)&g->spos4, (n + 8) * sizeof(float4));
    alloc((void **)&g->opos, n * sizeof(float4));
    g->defer = nullptr;
    if (geom->d == 3) alloc((void **)&g->defer, 2 * n * sizeof(float4));
    alloc((void **)&g->ctr, sizeof(Counters));
    if (!ok) {
        kc_grid_destroy(g);
        set_error("kc_grid_create: device allocation failed");
        return KC_ENOMEM;
    }
    // one-time initialisation (default stream, synchronous): chains empty, scratch zeroed
    bool e = cudaMemset(g->head, 0xff, nc * 4) != cudaSuccess ||
             cudaMemset(g->fcount, 0, nc * 4) != cudaSuccess ||
             cudaMemset(g->mhist, 0, MHIST * 4) != cudaSuccess ||
             cudaMemset(g->mark, 0, (n + 8) * 4) != cudaSuccess ||
             cudaMemset(g->ctr, 0, sizeof(Counters)) != cudaSuccess ||
             cudaDeviceSynchronize() != cudaSuccess;
    if (e) {
        kc_status s = cuda_fail(cudaGetLastError(), "kc_grid_create init");
        kc_grid_destroy(g);
        return s;
    }
    *out = g;
    return KC_OK;
}

extern "C" kc_status kc_grid_destroy(kc_grid *g)
{
    if (!g) return KC_OK;
    void *ptrs[] = {g->cell, g->counts, g->cell_start, g->sidx, g->slot, g->head, g->next,
                    g->mlist, g->fcount, g->mhist, g->scan_desc, g->subinfo, g->leaf_cnt, g->leaf_start, g->leafid, g->mark, g->list2, g->handoff, g->handoff_part, g->delta, g->cellmax, g->spos2, g->spos4, g->opos, g->defer, g->ctr};
    for (void *p : ptrs)
        if (p) cudaFree(p);
    delete g;
    return KC_OK;
}

extern "C" size_t kc_grid_bytes(const kc_grid *g) { return g ? g->bytes : 0; }

extern "C" kc_status kc_grid_set_index(kc_grid *g, int heavy_T, int sub_occ)
{
    if (!g || sub_occ < 1 || sub_occ > 64 || heavy_T < 1) {
        set_error("kc_grid_set_index: bad argument (1 <= sub_occ <= 64, heavy_T >= 1)");
        return KC_EINVAL;
    }
    const int thr_min = sub_occ << (g->geom.d + 1);      // keeps the leaf count within n_leaves_max
    g->sub_occ = sub_occ;
    g->heavy_T = heavy_T < thr_min ? thr_min : heavy_T;   // (KC_INDEX_OFF = INT_MAX: no second level)
    g->built = 0;                                         // takes effect with the next build
    return KC_OK;
}

extern "C" kc_status kc_grid_build(kc_grid *g, const float *p, int64_t N, void *stream)
{
    if (!g || !p || N < 2 || N > g->N_max || (reinterpret_cast<uintptr_t>(p) & 7)) {
        set_error("kc_grid_build: bad argument (N must be in [2, N_max], p 8-byte aligned)");
        return KC_EINVAL;
    }
    cudaStream_t st = (cudaStream_t)stream;
    View v = make_view(g);
    const int n = (int)N, nc = (int)g->n_cells;
    const int d = g->geom.d, T = g->heavy_T, so = g->sub_occ;
    // upper bound of the number of leaves of THIS build (the device knows the exact count)
    const bool two_level = T != KC_INDEX_OFF;             // off: the leaves are the cells, no second pass
    const int64_t nl_max = two_level ? (int64_t)nc + N + 8 : 0;
    const int ncb = (nc + SCAN_CHUNK - 1) / SCAN_CHUNK, nlb = (int)((nl_max + SCAN_CHUNK - 1) / SCAN_CHUNK);
    unsigned long long *desc_c = g->scan_desc, *desc_l = g->scan_desc + ncb;
    build_prep_kernel<<<blocks_for((nl_max > nc ? nl_max : nc) / 4 + 1, 256, 148 * 8), 256, 0, st>>>(g->mlist, g->cell, g->head, g->ctr,
                                                                              g->counts, nc, g->leaf_cnt, nl_max,
                                                                              g->scan_desc, ncb + nlb);
    if (d == 2) cellid_hist_kernel<2><<<(n + 255) / 256, 256, 0, st>>>(v, p, n, g->cell, g->counts, g->ctr);
    else cellid_hist_kernel<3><<<(n + 255) / 256, 256, 0, st>>>(v, p, n, g->cell, g->counts, g->ctr);
    scan_cells_kernel<<<ncb, 256, 0, st>>>(g->counts, nc, d, T, so, two_level, desc_c, g->cell_start, g->subinfo,
                                           g->leaf_cnt, g->leaf_start, g->ctr, n);
    // second level (these kernels leave at once when no cell is subdivided)
    if (two_level) {
        if (d == 2) leafid_hist_kernel<2><<<(n + 255) / 256, 256, 0, st>>>(v, p, n, g->cell, g->leaf_cnt, g->leafid, g->ctr);
        else leafid_hist_kernel<3><<<(n + 255) / 256, 256, 0, st>>>(v, p, n, g->cell, g->leaf_cnt, g->leafid, g->ctr);
        lscan_kernel<<<nlb, 256, 0, st>>>(g->leaf_cnt, desc_l, g->leaf_start, g->ctr);
    }
    if (d == 2)
        scatter_kernel<2><<<(n + 255) / 256, 256, 0, st>>>(p, n, g->cell, g->leafid, g->leaf_start, g->ctr, g->spos2,
                                                           g->spos4, g->sidx, g->slot);
    else
        scatter_kernel<3><<<(n + 255) / 256, 256, 0, st>>>(p, n, g->cell, g->leafid, g->leaf_start, g->ctr, g->spos2,
                                                           g->spos4, g->sidx, g->slot);
    count_launches(two_level ? 6 : 4);
    KC_LAUNCH_CHECK("kc_grid_build");
    g->N = N; g->built = 1; g->dirty = 0;
    return KC_OK;
}

extern "C" kc_status kc_frontier_classify_local(kc_grid *g, const float *p, const float *p2, int64_t N,
                                                const int32_t *nn, const float *d1, const float *c,
                                                const float *eps, uint8_t *flags, int32_t *F, int32_t *nF,
                                                void *stream)
{
    if (!g || !p || !p2 || !nn || !d1 || !c || !eps || !F || !nF) {
        set_error("kc_frontier_classify_local: bad argument");
        return KC_EINVAL;
    }
    if (!g->built || N != g->N) {
        set_error("kc_frontier_classify_local: grid not resident at p for this N");
        return KC_EREBUILD;
    }
    cudaStream_t st = (cudaStream_t)stream;
    View v = make_view(g);
    // everything outside the 3^d block of a point's cell is at least R away from it
    const float slkmax = fmaxf(v.slk0, fmaxf(v.slk1, v.slk2));
    volatile float hr = g->geom.h * 0.99609375f;          // two separately rounded float32 ops
    const float R = hr - slkmax;
    const int n = (int)N;
    KC_CUDA(cudaMemsetAsync(g->cellmax, 0, (size_t)g->n_cells * 4, st));
    KC_CUDA(cudaMemsetAsync(nF, 0, 4, st));
    motion_field_kernel<<<(n + 255) / 256, 256, 0, st>>>(g->geom.d, p, p2, n, g->cell, g->delta, g->cellmax);
    classify_local_kernel<<<(n + 255) / 256, 256, 0, st>>>(v, R, n, g->cell, g->delta, g->cellmax, nn, d1, c, eps,
                                                           flags, F, nF);
    count_launches(2);
    KC_LAUNCH_CHECK("kc_frontier_classify_local");
    return KC_OK;
}

extern "C" kc_status kc_frontier_entropy(kc_grid *g, const int32_t *F, const int32_t *nF,
                                         int64_t nF_max, double *H, int32_t *m_cells, int32_t *C_occ,
                                         void *stream)
{
    if (!g || !F || !nF || !H || nF_max < 0) {
        set_error("kc_frontier_entropy: bad argument");
        return KC_EINVAL;
    }
    if (!g->built) { set_error("kc_frontier_entropy: grid not built"); return KC_EREBUILD; }
    cudaStream_t st = (cudaStream_t)stream;
    int blocks = blocks_for(nF_max, 256, 148 * 8);
    const int recount = g->dirty;       // a fresh build's scan has counted C already
    if (recount) blocks = max(blocks, blocks_for(g->n_cells, 1024, 148 * 8));
    entropy_count_kernel<<<blocks, 256, 0, st>>>(F, nF, g->cell, g->fcount, g->counts, (int)g->n_cells, recount, g->ctr);
    entropy_collect_kernel<<<blocks, 256, 0, st>>>(F, nF, g->cell, g->fcount, g->mhist, g->ctr, recount, H, m_cells, C_occ);
    count_launches(2);
    KC_LAUNCH_CHECK("kc_frontier_entropy");
    return KC_OK;
}

// A6, Algorithm 1 line 3: unlink every chain, refresh positions / re-file cell
// changers, link again.
extern "C" kc_status kc_grid_update(kc_grid *g, const float *p_new, int64_t N, const int32_t *movers,
                                    const int32_t *n_movers, int64_t n_movers_max, void *stream)
{
    if (!g || !p_new || (movers && (!n_movers || n_movers_max < 0))) {
        set_error("kc_grid_update: bad argument");
        return KC_EINVAL;
    }
    if (!g->built || N != g->N) {
        set_error("kc_grid_update: grid not built for this N");
        return KC_EREBUILD;
    }
    // Most points may have moved on a large grid: re-bin (A2, O(N), ~0.3 ms at 4 M points) instead of
    // re-filing them one by one -- cheaper than the refresh pass itself, no tombstones, no chains,
    // and the frontier search that follows runs on a fresh grid.  (Decided from the host-side bounds.)
    const int64_t nm = movers ? n_movers_max : N;
    if (N >= REBIN_MIN_N && nm * (g->geom.d == 2 ? REBIN_DIV2 : (int64_t)list_div3(N)) >= N) return kc_grid_build(g, p_new, N, stream);
    cudaStream_t st = (cudaStream_t)stream;
    View v = make_view(g);
    const int n = (int)N;
    const int chain_blocks = blocks_for(g->dirty ? N : 1, 256, 148 * 4);
    if (g->dirty) clear_chains_kernel<<<chain_blocks, 256, 0, st>>>(g->mlist, g->cell, g->head, g->ctr);
    count_launches((g->dirty ? 1 : 0) + (nm > 0 ? 1 : 0) + 1);
    if (nm > 0) {
        int blocks = blocks_for(nm, 256, 148 * 16);
        if (g->geom.d == 2)
            refresh_kernel<2><<<blocks, 256, 0, st>>>(v, p_new, n, movers, n_movers, g->cell, g->slot, g->sidx,
                                                      g->spos2, g->spos4, g->opos, g->mlist, g->counts, g->ctr);
        else
            refresh_kernel<3><<<blocks, 256, 0, st>>>(v, p_new, n, movers, n_movers, g->cell, g->slot, g->sidx,
                                                      g->spos2, g->spos4, g->opos, g->mlist, g->counts, g->ctr);
    }
    link_chains_kernel<<<blocks_for(nm > 0 || g->dirty ? N : 1, 256, 148 * 4), 256, 0, st>>>(g->mlist, g->cell, g->head, g->next, g->ctr);
    g->dirty = 1;
    KC_LAUNCH_CHECK("kc_grid_update");
    return KC_OK;
}

extern "C" kc_status kc_grid_info(kc_grid *g, kc_grid_info_t *out, void *stream)
{
    if (!g || !out) { set_error("kc_grid_info: bad argument"); return KC_EINVAL; }
    Counters h;
    KC_CUDA(cudaMemcpyAsync(&h, g->ctr, sizeof(Counters), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    KC_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    out->n_points = g->N; out->n_cells = g->n_cells;
    out->c_occ = h.c_occ; out->max_occ = h.max_occ; out->n_misfiled = h.n_misfiled;
    out->built = g->built; out->dirty = g->dirty; out->n_stragglers = h.n_stragglers; out->n_handed = h.n_handed;
    out->n_heavy = h.n_heavy; out->n_leaves = h.n_heavy ? h.n_leaves : (int32_t)g->n_cells;
    out->heavy_T = g->heavy_T; out->n_deferred = h.n_deferred;
    return KC_OK;
}

extern "C" kc_status kc_grid_export(const kc_grid *g, int what, int32_t *dst, int64_t capacity,
                                    int64_t *count, void *stream)
{
    if (!g || !count) { set_error("kc_grid_export: bad argument"); return KC_EINVAL; }
    const int32_t *src = nullptr;
    int64_t n = 0;
    switch (what) {
    case 0: src = g->cell; n = g->N; break;
    case 1: src = g->cell_start; n = g->n_cells + 1; break;
    case 2:
        n = g->N;
        if (g->geom.d == 3 && dst && capacity >= n) {     // d = 3 keeps the ids inside the records
            record_ids_kernel<<<blocks_for(n, 256, 148 * 8), 256, 0, (cudaStream_t)stream>>>(g->spos4, (int)n, dst);
            *count = n;
            KC_LAUNCH_CHECK("kc_grid_export");
            return KC_OK;
        }
        src = g->sidx;
        break;
    case 3: src = g->slot; n = g->N; break;
    case 4: src = g->counts; n = g->n_cells; break;
    case 5: src = reinterpret_cast<const int32_t *>(g->subinfo); n = 2 * g->n_cells; break;
    case 6: src = g->leaf_start; n = g->n_cells + g->N + 9; break;
    default: set_error("kc_grid_export: unknown array %d", what); return KC_EINVAL;
    }
    *count = n;
    if (!dst) return KC_OK;
    if (capacity < n) { set_error("kc_grid_export: capacity %lld < %lld", (long long)capacity, (long long)n); return KC_EINVAL; }
    KC_CUDA(cudaMemcpyAsync(dst, src, (size_t)n * 4, cudaMemcpyDeviceToDevice, (cudaStream_t)stream));
    return KC_OK;
}
