// query3.cu -- S:8(a) A6 (2pCF sweep), A7 (3pCF intersection + histogram), A10 (fold + flush).
//
// "for each hub i and each neighbor j in N(i), it checks whether a second neighbor k in N(i)
// with k > j is also in N(j).  If so, the triangle (i,j,k) is counted in the (r_ij, r_ik, r_jk) bin."
// the hub tail {k in N(i): k > j} and N(j) are both sorted, so the membership tests are one
// sorted-set intersection per hub-spoke pair.  With oriented storage (A-15) every triangle i<j<k is
// found exactly once (A-1).
//
// Mapping (differs from the paper's OpenACC gang-per-hub / lane-per-candidate binary search):
// persistent CTAs pull hubs from a global counter in spatial order (so concurrently resident hubs share
// spoke rows in L2), the hub row (ids, bins, weights) is staged once in shared memory, each warp owns
// hub-spoke pairs, and hits go to a per-CTA shared-memory uint32 histogram flushed with uint64 atomics.
#include "internal.cuh"

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <type_traits>

namespace {

#ifndef GR_LONG_U
#define GR_LONG_U 8      // windows in flight per trip on long rows
#endif
constexpr int Q3_THREADS = 256;
constexpr int Q3_WARPS = Q3_THREADS / 32;

struct Q3Params {
    int nb;
    int nh;             // nb^3
    int row_cap;        // entries of the staged hub row
    int smem_hist;      // 1: uint32 histogram in shared memory
    int weighted;
    int want_counts;
    int n_slabs;        // fp64 slabs in g_w (a CTA adds to slab blockIdx % n_slabs)
    int equi;           // equilateral restriction (S:8(f)-3): count only b_ij == b_ik == b_jk, histogram over b_ij (nh = nb)
    unsigned long long flush;   // drain the shared uint32 histogram before the CTA's hit budget passes this
};

__device__ __forceinline__ unsigned lane_id() { return threadIdx.x & 31; }

// lower_bound of key in sorted smem array a[lo,hi)
__device__ __forceinline__ int lower_bound_s(const int32_t *a, int lo, int hi, int32_t key)
{
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if (a[mid] < key) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// ---- 3pCF, lane-parallel binary search variant ("GPU binary-search kernels") ------------------------
template <bool WEIGHTED>
__global__ void __launch_bounds__(Q3_THREADS)
k_3pcf_bsearch(GrView v, Q3Params p, unsigned int *__restrict__ hub_counter,
               unsigned long long *__restrict__ g_cnt, double *__restrict__ g_w)
{
    extern __shared__ __align__(16) unsigned char smem[];
    // layout: [w row_cap*8] [idx row_cap*4] [hist nh*4] [bin row_cap]
    double *a_w = (double *)smem;
    int32_t *a_idx = (int32_t *)(smem + (WEIGHTED ? (size_t)p.row_cap * 8 : 0));
    uint32_t *hist = (uint32_t *)(a_idx + p.row_cap);
    uint8_t *a_bin = (uint8_t *)(hist + (p.smem_hist ? p.nh : 0));
    __shared__ int s_slot;
    unsigned long long budget = 0;      // CTA-uniform: upper bound of the hits added since the last flush

    const int nb = p.nb;
    const int warp = threadIdx.x >> 5, lane = lane_id();
    if (p.smem_hist)
        for (int t = threadIdx.x; t < p.nh; t += Q3_THREADS) hist[t] = 0;
    double *my_w = WEIGHTED ? g_w + (size_t)(blockIdx.x % p.n_slabs) * p.nh : nullptr;
    __syncthreads();

    for (;;) {
        if (threadIdx.x == 0) s_slot = v.s_lo + (int)atomicAdd(hub_counter, 1u);
        __syncthreads();
        const int s = s_slot;
        if (s >= v.s_hi) break;
        const int32_t i = v.order[s];
        const bool mine = (i >= v.h_lo && i < v.h_hi) && GR_HUB_SELECTED(v, i);
        const int64_t rb = mine ? v.ptr[i] : 0, re = mine ? v.ptr[i + 1] : 0;
        const int n = (int)(re - rb);
        if (n >= 2) {
            // uint32 histogram overflow guard: a hub adds at most n(n-1)/2 hits
            if (p.smem_hist) {
                unsigned long long add = (unsigned long long)n * (n - 1) / 2;
                if (budget + add > p.flush) {
                    for (int t = threadIdx.x; t < p.nh; t += Q3_THREADS) {
                        uint32_t c = hist[t];
                        if (c) { atomicAdd(&g_cnt[t], (unsigned long long)c); hist[t] = 0; }
                    }
                    budget = 0;
                }
                budget += add;
            }
            const int32_t *gi = v.idx_h + (rb - v.e0_h);
            const uint8_t *gb = v.bin_h + (rb - v.e0_h);
            for (int t = threadIdx.x; t < n; t += Q3_THREADS) {
                int32_t k = gi[t];
                a_idx[t] = k;
                a_bin[t] = gb[t];
                if (WEIGHTED) a_w[t] = v.w[k];
            }
            __syncthreads();
            const double wi = WEIGHTED ? v.w[i] : 1.0;
            for (int a = warp; a < n - 1; a += Q3_WARPS) {
                const int32_t j = a_idx[a];
                if (j < v.c_lo || j >= v.c_hi) continue;          // foreign spoke
                const int64_t jb = v.ptr[j], je = v.ptr[j + 1];
                const int nj = (int)(je - jb);
                if (nj == 0) continue;
                const int32_t *B = v.idx_c + (jb - v.e0_c);
                const uint8_t *Bb = v.bin_c + (jb - v.e0_c);
                const int32_t *T = a_idx + a + 1;
                const int nt = n - a - 1;
                const int32_t t_last = T[nt - 1];
                const int bij = (int)a_bin[a];
                const int hbase = bij * nb * nb;
                const double wij = WEIGHTED ? wi * a_w[a] : 1.0;
                int lo = 0;
                for (int t0 = 0; t0 < nj; t0 += 32) {
                    const int t = t0 + lane;
                    int32_t k = (t < nj) ? B[t] : INT32_MAX;
                    int pos = nt;
                    if (k <= t_last) pos = lower_bound_s(T, lo, nt, k);
                    bool hit = (pos < nt) && (T[pos] == k);
                    if (p.equi) hit = hit && (int)Bb[t] == bij && (int)a_bin[a + 1 + pos] == bij;
                    if (hit) {
                        const int h = p.equi ? bij : hbase + (int)a_bin[a + 1 + pos] * nb + (int)Bb[t];
                        if (p.want_counts) {
                            if (p.smem_hist) atomicAdd(&hist[h], 1u);
                            else atomicAdd(&g_cnt[h], 1ull);
                        }
                        if (WEIGHTED) atomicAdd(&my_w[h], wij * a_w[a + 1 + pos]);
                    }
                    // every later element of B is larger: the window can start at lane 0's position
                    lo = __shfl_sync(0xffffffffu, pos, 0);
                    if (__shfl_sync(0xffffffffu, k, 31) > t_last) break;
                }
            }
        }
        __syncthreads();
    }
    if (p.smem_hist && p.want_counts) {
        __syncthreads();
        for (int t = threadIdx.x; t < p.nh; t += Q3_THREADS) {
            uint32_t c = hist[t];
            if (c) atomicAdd(&g_cnt[t], (unsigned long long)c);
        }
    }
}

// ---- 3pCF, merge-path variant (the paper's two-pointer walk, partitioned over a warp) ----------------
// BASELINE's sketch of the kernel: a warp takes a hub-spoke pair and intersects the hub tail (shared memory) with
// the spoke row N+(j) by a merge: the row is staged through a per-warp shared buffer in tiles, the part of the
// tail a tile can meet is located with a 32-ary search, the merged sequence of the two pieces is cut into 32
// equal diagonals (one binary search per lane on its diagonal), and every lane walks its piece with the
// two-pointer rule of P:59-70 -- on a tie the row element is consumed first, and a row element is a hit iff the
// current head of the tail equals it, so each triangle is found by exactly one lane.
// The hub row itself arrives by one TMA bulk copy per array (cp.async.bulk -> UBLKCP, mbarrier completion).
// Kept as GRAMSCI_ALGO_MERGEPATH for the ablation DESIGN.md section 6 reports; the slot table beats it.
constexpr int MP_TILE = 512;          // row elements staged per warp and tile

__device__ __forceinline__ void mbar_init(uint64_t *bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)),
                 "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity)
{
    asm volatile(
        "{\n.reg .pred p;\nWAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\nbra WAIT_%=;\nDONE_%=:\n}" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_bulk_g2s(void *dst, const void *src, unsigned bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     (unsigned)__cvta_generic_to_shared(dst)),
                 "l"(src), "r"(bytes), "r"((unsigned)__cvta_generic_to_shared(bar))
                 : "memory");
}

template <bool WEIGHTED>
__global__ void __launch_bounds__(Q3_THREADS)
k_3pcf_merge(GrView v, Q3Params p, unsigned int *__restrict__ hub_counter,
             unsigned long long *__restrict__ g_cnt, double *__restrict__ g_w)
{
    extern __shared__ __align__(16) unsigned char smem[];
    // layout: [w row_cap*8 (W)] [idx raw (row_cap+8)*4] [bin raw row_cap+32] [hist nh*4] [per warp: tile idx, tile bin]
    double *a_w = (double *)smem;
    int32_t *raw_idx = (int32_t *)(smem + (WEIGHTED ? (size_t)p.row_cap * 8 : 0));
    uint8_t *raw_bin = (uint8_t *)(raw_idx + p.row_cap + 8);
    uint32_t *hist = (uint32_t *)(raw_bin + p.row_cap + 32);
    const int warp = threadIdx.x >> 5, lane = lane_id();
    int32_t *t_idx = (int32_t *)(hist + p.nh) + warp * MP_TILE;
    uint8_t *t_bin = (uint8_t *)((int32_t *)(hist + p.nh) + Q3_WARPS * MP_TILE) + warp * MP_TILE;
    __shared__ int s_slot;
    __shared__ __align__(8) uint64_t s_bar;
    unsigned long long budget = 0;
    unsigned phase = 0;

    const int nb = p.nb;
    for (int t = threadIdx.x; t < p.nh; t += Q3_THREADS) hist[t] = 0;
    if (threadIdx.x == 0) {
        mbar_init(&s_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    double *my_w = WEIGHTED ? g_w + (size_t)(blockIdx.x % p.n_slabs) * p.nh : nullptr;
    __syncthreads();

    for (;;) {
        if (threadIdx.x == 0) s_slot = v.s_lo + (int)atomicAdd(hub_counter, 1u);
        __syncthreads();
        const int s = s_slot;
        if (s >= v.s_hi) break;
        const int32_t i = v.order[s];
        const bool mine = (i >= v.h_lo && i < v.h_hi) && GR_HUB_SELECTED(v, i);
        const int64_t rb = mine ? v.ptr[i] : 0, re = mine ? v.ptr[i + 1] : 0;
        const int n = (int)(re - rb);
        if (n >= 2) {
            if (budget + (unsigned long long)n * (n - 1) / 2 > p.flush) {      // uint32 bins cannot wrap
                for (int t = threadIdx.x; t < p.nh; t += Q3_THREADS) {
                    const uint32_t c = hist[t];
                    if (c) { atomicAdd(&g_cnt[t], (unsigned long long)c); hist[t] = 0; }
                }
                budget = 0;
            }
            budget += (unsigned long long)n * (n - 1) / 2;
            // ---- hub row by TMA: bulk copies need 16-byte aligned source, destination and size, so each array is
            // copied from its address rounded down and used at the matching offset
            const int32_t *gi = v.idx_h + (rb - v.e0_h);
            const uint8_t *gb = v.bin_h + (rb - v.e0_h);
            const unsigned xi = (unsigned)(((uintptr_t)gi & 15) >> 2), xb = (unsigned)((uintptr_t)gb & 15);
            const unsigned bytes_i = (((unsigned)n + xi) * 4 + 15) & ~15u, bytes_b = ((unsigned)n + xb + 15) & ~15u;
            if (threadIdx.x == 0) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");    // earlier generic reads of the row buffers
                mbar_expect_tx(&s_bar, bytes_i + bytes_b);
                tma_bulk_g2s(raw_idx, (const void *)((uintptr_t)gi & ~(uintptr_t)15), bytes_i, &s_bar);
                tma_bulk_g2s(raw_bin, (const void *)((uintptr_t)gb & ~(uintptr_t)15), bytes_b, &s_bar);
            }
            const int32_t *a_idx = raw_idx + xi;
            const uint8_t *a_bin = raw_bin + xb;
            if (WEIGHTED)
                for (int t = threadIdx.x; t < n; t += Q3_THREADS) a_w[t] = v.w[gi[t]];
            mbar_wait(&s_bar, phase);
            phase ^= 1;
            __syncthreads();

            const double wi = WEIGHTED ? v.w[i] : 1.0;
            for (int a = warp; a < n - 1; a += Q3_WARPS) {
                const int32_t j = a_idx[a];
                if (j < v.c_lo || j >= v.c_hi) continue;          // foreign spoke
                const int64_t jb = v.ptr[j];
                const int nj = (int)(v.ptr[j + 1] - jb);
                const int32_t *B = v.idx_c + (jb - v.e0_c);
                const uint8_t *Bb = v.bin_c + (jb - v.e0_c);
                const int32_t *A = a_idx + a + 1;                 // hub tail {k in N+(i): k > j}
                const int nA = n - a - 1;
                const int32_t a_last = A[nA - 1];
                const int hbase = (int)a_bin[a] * nb * nb;
                const double wij = WEIGHTED ? wi * a_w[a] : 1.0;
                int alo = 0;                                      // tail elements below every later row element
                for (int b0 = 0; b0 < nj && alo < nA; b0 += MP_TILE) {
                    const int nB = min(MP_TILE, nj - b0);
                    __syncwarp();
                    for (int t = lane; t < nB; t += 32) { t_idx[t] = B[b0 + t]; t_bin[t] = Bb[b0 + t]; }
                    __syncwarp();
                    const int32_t b_first = t_idx[0], b_last = t_idx[nB - 1];
                    // 32-ary searches: first tail element >= b_first, first tail element > b_last
                    auto lower = [&](int32_t key, int lo) {        // first x in [lo,nA) with A[x] >= key (nA if none)
                        int hi = nA;                               // candidates [lo,hi), answer in [lo,hi]
                        while (hi > lo) {
                            const int stride = (hi - lo + 31) >> 5;
                            const int x = lo + (lane + 1) * stride - 1;          // 32 probes, the last ones may fall off
                            const int c = __popc(__ballot_sync(0xffffffffu, x < hi && A[x] < key));   // a prefix of lanes
                            hi = min(lo + (c + 1) * stride - 1, hi);   // probe c is >= key (or off the end)
                            lo = lo + c * stride;                      // everything up to probe c-1 is < key
                        }
                        return lo;
                    };
                    alo = lower(b_first, alo);
                    const int ahi = (b_last >= a_last) ? nA : lower(b_last + 1, alo);
                    const int nAt = ahi - alo;
                    if (nAt > 0) {
                        // merge path: diagonal d = lane * L of the (nAt + nB)-long merged sequence
                        const int T = nAt + nB, L = (T + 31) >> 5;
                        const int d0 = min(lane * L, T), d1 = min(d0 + L, T);
                        int lo = max(0, d0 - nB), hi = min(d0, nAt);
                        while (lo < hi) {                              // ties: the row element goes first
                            const int mid = (lo + hi) >> 1;
                            if (A[alo + mid] < t_idx[d0 - 1 - mid]) lo = mid + 1; else hi = mid;
                        }
                        int ia = lo, ib = d0 - lo;
                        for (int step = d0; step < d1; ++step) {
                            const int32_t av = (ia < nAt) ? A[alo + ia] : INT32_MAX;
                            const int32_t bv = (ib < nB) ? t_idx[ib] : INT32_MAX;
                            if (ib < nB && bv <= av) {
                                if (bv == av) {
                                    const int pos = a + 1 + alo + ia;
                                    const int h = hbase + (int)a_bin[pos] * nb + (int)t_bin[ib];
                                    if (p.want_counts) atomicAdd(&hist[h], 1u);
                                    if (WEIGHTED) atomicAdd(&my_w[h], wij * a_w[pos]);
                                }
                                ++ib;
                            } else {
                                ++ia;
                            }
                        }
                    }
                    alo = ahi;
                    if (b_last >= a_last) break;                    // the tail is used up
                }
            }
        }
        __syncthreads();
    }
    __syncthreads();
    for (int t = threadIdx.x; t < p.nh; t += Q3_THREADS) {
        const uint32_t c = hist[t];
        if (c) atomicAdd(&g_cnt[t], (unsigned long long)c);
    }
}

// ---- 3pCF, slot-table variant (default) ------------------------------------------------------------------
// Membership of k in N+(i) is one table lookup instead of a search (the hub-side analogue of the paper's
// lmat idea: spend O(len) setup per hub to make every later test O(1)).  The hub row is scattered
// into a two-level table keyed by d = k - first(N+(i)):  page g = d >> s  ->  chunk pt[g] (0 = page not
// touched by the row), slot (chunk << s) | (d & (2^s - 1)) -> the entry's bin byte (or its position,
// weighted) or EMPTY.  With labels in cell order a row touches few pages (it lives in a handful of runs
// of x-adjacent cells), so the table is a few KB; sizes come from the row statistics of the build.
// Set-up and tear-down touch only the row's own entries (O(len)).
//
// Work mapping: G warps share one hub (G = 1, 2, 4, 8 by table size); each warp takes blocks of 32 spokes:
// the lanes fetch the 32 row heads (ptr[j], ptr[j+1]) at once, then the warp streams the rows N+(j) one
// after the other, 32 elements per window, with the first two windows of the next row already in flight
// (rows are tens of entries long in the 1e6-point configurations, so the ptr -> idx latency chain per row
// is what has to be hidden).  An earlier variant walked the 32 rows as one flat index space (no idle lanes)
// but paid ~57 instructions per window for the bookkeeping; this one needs ~25.
template <int G>
__device__ __forceinline__ void group_sync(int group)
{
    if (G == 1) __syncwarp();
    else if (G == Q3_WARPS) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "r"(G * 32) : "memory");
}

struct T3Params {
    int nb, nh;
    int s;              // page shift
    int pt_len;         // page-table entries (uint16)
    int tab_len;        // slots
    int row_cap;        // staged weights / bins per hub (weighted)
    int want_counts;
    int group_bytes;    // shared memory per group (multiple of 16)
    int hub_batch;      // schedule slots fetched per atomic
    int n_slabs;        // fp64 slabs in g_w (a CTA adds to slab blockIdx % n_slabs)
    unsigned long long flush;   // a warp drains the CTA histogram before its own hit budget passes this
};

template <bool WEIGHTED, int G, int U>      // U = windows in flight per trip on long rows
__global__ void __launch_bounds__(Q3_THREADS)
k_3pcf_table(GrView v, T3Params p, unsigned int *__restrict__ hub_counter,
             unsigned long long *__restrict__ g_cnt, double *__restrict__ g_w)
{
    typedef typename std::conditional<WEIGHTED, uint16_t, uint8_t>::type slot_t;
    constexpr unsigned EMPTY = WEIGHTED ? 0xffffu : 0xffu;
    constexpr int NGROUPS = Q3_WARPS / G;
    extern __shared__ __align__(16) unsigned char smem[];
    // CTA: [hist u32 nh] [group 0] [group 1] ...
    uint32_t *hist = (uint32_t *)smem;
    double *my_w = WEIGHTED ? g_w + (size_t)(blockIdx.x % p.n_slabs) * p.nh : nullptr;   // fp64 partials: a slab per CTA while the byte budget allows (RED.F64)
    const int warp = threadIdx.x >> 5, lane = lane_id();
    const int group = warp / G, gw = warp % G;
    // (plain pointer arithmetic on `smem` only: a round trip through an integer would turn every access
    // below into a generic-address load instead of LDS)
    unsigned char *gs = smem + (((size_t)p.nh * 4 + 15) & ~(size_t)15) + (size_t)group * p.group_bytes;
    // group: [a_w f64 row_cap (W)] [row heads per warp] [pt u16] [tab] [a_bin u8 row_cap (W)]
    double *a_w = (double *)gs;
    unsigned char *q = gs + (WEIGHTED ? (size_t)p.row_cap * 8 : 0);
    int4 *s_head = (int4 *)q + gw * 32;                      q += (size_t)G * 32 * 16;   // (row offset lo, hi, len, b_ij nb^2)
    double *s_wia = (double *)q + gw * 32;                  q += WEIGHTED ? (size_t)G * 32 * 8 : 0;
    uint16_t *pt = (uint16_t *)q;                           q += ((size_t)p.pt_len * 2 + 15) & ~(size_t)15;
    slot_t *tab = (slot_t *)q;                              q += ((size_t)p.tab_len * sizeof(slot_t) + 15) & ~(size_t)15;
    uint8_t *a_bin = (uint8_t *)q;
    __shared__ int s_fetch[NGROUPS];

    for (int t = threadIdx.x; t < p.nh; t += Q3_THREADS) hist[t] = 0;
    for (int t = gw * 32 + lane; t < p.pt_len; t += G * 32) pt[t] = 0;
    for (int t = gw * 32 + lane; t < p.tab_len; t += G * 32) tab[t] = (slot_t)EMPTY;
    __syncthreads();

    const int nb = p.nb, nb2 = nb * nb;
    const int sh = p.s;
    const unsigned pm = (1u << sh) - 1u;
    const unsigned dmax = ((unsigned)p.pt_len - 1u) << sh;  // first key of the sentinel page: always chunk 0 (all EMPTY)
    const unsigned lt_mask = (1u << lane) - 1u, le_mask = (2u << lane) - 1u;
    unsigned long long budget = 0;       // upper bound of the hits this warp added since it last flushed
    // key of a label k in the current hub's table: the largest gap of the row is cut out (rows next to a
    // periodic face reach the far end of the label range):
    //   k <  brk : d = min(k - base, guard)      (labels inside the gap land on the empty guard page)
    //   k >= brk : d = k - brk + off,  off = guard + 2^s
    // previous hub of this group (its table entries are cleared before the next one is set)
    const int32_t *prev_gi = nullptr;
    int prev_n = 0;
    int32_t prev_base = 0, prev_brk = 0;
    unsigned prev_off = 0;

    int s_cur = 0, s_end = 0;
    for (;;) {
        if (s_cur >= s_end) {
            int s0;
            if (G == 1) {
                s0 = (lane == 0) ? (int)atomicAdd(hub_counter, (unsigned)p.hub_batch) : 0;
                s0 = __shfl_sync(0xffffffffu, s0, 0);
            } else {
                if (gw == 0 && lane == 0) s_fetch[group] = (int)atomicAdd(hub_counter, (unsigned)p.hub_batch);
                group_sync<G>(group);
                s0 = s_fetch[group];
                group_sync<G>(group);
            }
            s_cur = v.s_lo + s0;
            s_end = min(s_cur + p.hub_batch, v.s_hi);
            if (s_cur >= v.s_hi) break;
        }
        const int32_t i = v.order[s_cur++];
        const bool mine = (i >= v.h_lo && i < v.h_hi) && GR_HUB_SELECTED(v, i);
        const int64_t rb = mine ? v.ptr[i] : 0, re = mine ? v.ptr[i + 1] : 0;
        const int n = (int)(re - rb);
        if (n < 2) continue;
        const int32_t *gi = v.idx_h + (rb - v.e0_h);
        const uint8_t *gb = v.bin_h + (rb - v.e0_h);
        const int32_t base = gi[0];
        // first largest gap of the row (every warp of the group computes the same values)
        int32_t brk, lowmax;
        {
            int best_gap = 0, best_t = 1;
            int32_t carry = base;
            for (int t0 = 0; t0 < n; t0 += 32) {
                const int t = t0 + lane;
                const int32_t k = (t < n) ? gi[t] : 0;
                int32_t pk = __shfl_up_sync(0xffffffffu, k, 1);
                if (lane == 0) pk = carry;
                const int gap = (t < n) ? k - pk : 0;
                const int m = __reduce_max_sync(0xffffffffu, gap);
                if (m > best_gap) {
                    best_gap = m;
                    best_t = t0 + __ffs(__ballot_sync(0xffffffffu, gap == m)) - 1;
                }
                carry = __shfl_sync(0xffffffffu, k, 31);
            }
            lowmax = gi[best_t - 1];
            brk = gi[best_t];
        }
        const unsigned guard = ((((unsigned)(lowmax - base)) >> sh) + 1u) << sh;
        const unsigned off = guard + (1u << sh);
        const int32_t sub_hi = brk - (int32_t)off;

        // ---- table: clear the previous hub's entries, set this hub's (warp 0 of the group) ----
        group_sync<G>(group);                       // every warp is done looking things up
        if (gw == 0) {
            if (prev_n) {
                int cbase = 0, carry = -1;
                for (int t0 = 0; t0 < prev_n; t0 += 32) {
                    const int t = t0 + lane;
                    const bool ok = t < prev_n;
                    const int32_t k = ok ? prev_gi[t] : prev_base;
                    const unsigned d = (k >= prev_brk) ? (unsigned)(k - prev_brk) + prev_off : (unsigned)(k - prev_base);
                    const int g = (int)(d >> sh);
                    int pg = __shfl_up_sync(0xffffffffu, g, 1);
                    if (lane == 0) pg = carry;
                    const unsigned m = __ballot_sync(0xffffffffu, ok && g != pg);
                    const int ch = cbase + __popc(m & le_mask);
                    if (ok) { tab[((unsigned)ch << sh) | (d & pm)] = (slot_t)EMPTY; pt[g] = 0; }
                    cbase += __popc(m);
                    carry = __shfl_sync(0xffffffffu, g, 31);
                }
                __syncwarp();
            }
            int cbase = 0, carry = -1;
            for (int t0 = 0; t0 < n; t0 += 32) {
                const int t = t0 + lane;
                const bool ok = t < n;
                const int32_t k = ok ? gi[t] : base;
                const unsigned d = (k >= brk) ? (unsigned)(k - sub_hi) : (unsigned)(k - base);
                const int g = (int)(d >> sh);
                int pg = __shfl_up_sync(0xffffffffu, g, 1);
                if (lane == 0) pg = carry;
                const bool np = ok && g != pg;
                const unsigned m = __ballot_sync(0xffffffffu, np);
                const int ch = cbase + __popc(m & le_mask);          // chunks are numbered from 1
                if (np) pt[g] = (uint16_t)((unsigned)ch << sh);      // slot base of the page's chunk
                if (ok) tab[((unsigned)ch << sh) | (d & pm)] = WEIGHTED ? (slot_t)t : (slot_t)gb[t];
                cbase += __popc(m);
                carry = __shfl_sync(0xffffffffu, g, 31);
            }
        }
        if (WEIGHTED)
            for (int t = gw * 32 + lane; t < n; t += G * 32) { a_w[t] = v.w[gi[t]]; a_bin[t] = gb[t]; }
        prev_gi = gi;
        prev_n = n;
        prev_base = base;
        prev_brk = brk;
        prev_off = off;
        group_sync<G>(group);

        const double wi = WEIGHTED ? v.w[i] : 1.0;
        // ---- blocks of 32 spokes: lanes fetch the row heads (ptr[j], ptr[j+1]) of 32 spokes at once, then the
        // warp walks the rows one after the other; the first two windows of the NEXT row are in flight while
        // the current row is looked up (rows are tens of entries long in the 1e6-point configurations)
        auto lookup = [&](int32_t k, unsigned gam, int hb, double wia) {
            const bool hi = k >= brk;
            // one clamp does both ends: below / inside the gap -> guard page, beyond the row -> sentinel page
            const unsigned d = min((unsigned)(k - (hi ? sub_hi : base)), hi ? dmax : guard);
            const unsigned e = tab[(unsigned)pt[d >> sh] | (d & pm)];      // pt holds the slot base, chunk << s
            if (e != EMPTY) {
                if (WEIGHTED) {
                    const int h = hb + (int)a_bin[e] * nb + (int)gam;
                    if (p.want_counts) atomicAdd(&hist[h], 1u);
                    atomicAdd(&my_w[h], wia * a_w[e]);
                } else {
                    atomicAdd(&hist[hb + (int)e * nb + (int)gam], 1u);
                }
            }
        };
        const int32_t dead = base - 1;                 // below the row: lands on the guard page, never a member
        const int32_t last = gi[n - 1];
        for (int a0 = gw * 32; a0 < n - 1; a0 += G * 32) {
            const int a = a0 + lane;
            int nj = 0, hb = 0;
            int64_t jb = 0;
            double wia = 0.0;
            if (a < n - 1) {
                const int32_t j = gi[a];
                if (j >= v.c_lo && j < v.c_hi) {              // foreign spokes are skipped
                    jb = v.ptr[j];
                    nj = (int)(v.ptr[j + 1] - jb);
                }
                hb = (int)gb[a] * nb2;
                if (WEIGHTED) wia = wi * a_w[a];
            }
            const unsigned nz = __ballot_sync(0xffffffffu, nj > 0);
            const int m = __popc(nz);
            if (m == 0) continue;
            __syncwarp();
            if (nj > 0) {
                const int r = __popc(nz & lt_mask);
                s_head[r] = make_int4((int)((jb - v.e0_c) & 0xffffffffll), (int)((jb - v.e0_c) >> 32), nj, hb);
                if (WEIGHTED) s_wia[r] = wia;
            }
            __syncwarp();
            // prologue: first two windows of row 0
            int4 hd = s_head[0];
            double w_cur = WEIGHTED ? s_wia[0] : 0.0;
            const int32_t *pi = v.idx_c + (((long long)hd.y << 32) | (unsigned)hd.x) + lane;
            const uint8_t *pb = v.bin_c + (((long long)hd.y << 32) | (unsigned)hd.x) + lane;
            int32_t k0 = dead, k1 = dead;
            unsigned g0 = 0, g1 = 0;
            if (lane < hd.z) { k0 = pi[0]; g0 = pb[0]; }
            if (lane + 32 < hd.z) { k1 = pi[32]; g1 = pb[32]; }
            for (int q = 0; q < m; ++q) {
                const int njc = hd.z, hbc = hd.w;
                const double wc = w_cur;
                const int32_t *pic = pi;
                const uint8_t *pbc = pb;
                const int32_t c0 = k0, c1 = k1;
                const unsigned e0g = g0, e1g = g1;
                if (q + 1 < m) {                               // next row's first two windows
                    hd = s_head[q + 1];
                    if (WEIGHTED) w_cur = s_wia[q + 1];
                    pi = v.idx_c + (((long long)hd.y << 32) | (unsigned)hd.x) + lane;
                    pb = v.bin_c + (((long long)hd.y << 32) | (unsigned)hd.x) + lane;
                    k0 = dead; k1 = dead;
                    if (lane < hd.z) { k0 = pi[0]; g0 = pb[0]; }
                    if (lane + 32 < hd.z) { k1 = pi[32]; g1 = pb[32]; }
                }
                budget += (unsigned long long)njc;
                lookup(c0, e0g, hbc, wc);
                // rows are sorted: once a window starts beyond the hub's last neighbour nothing further can hit
                if (njc > 32 && __shfl_sync(0xffffffffu, c1, 0) <= last) lookup(c1, e1g, hbc, wc);
                if (njc > 64 && __shfl_sync(0xffffffffu, c1, 31) > last) continue;
                for (int t0 = 64; t0 < njc; t0 += 32 * U) {
                    int32_t kk[U];
                    unsigned gg[U];
#pragma unroll
                    for (int u = 0; u < U; ++u) {
                        kk[u] = dead;
                        gg[u] = 0;
                        if (t0 + 32 * u + lane < njc) { kk[u] = pic[t0 + 32 * u]; gg[u] = pbc[t0 + 32 * u]; }
                    }
#pragma unroll
                    for (int u = 0; u < U; ++u)
                        if (t0 + 32 * u < njc) lookup(kk[u], gg[u], hbc, wc);
                    if (__shfl_sync(0xffffffffu, kk[U - 1], 31) > last) break;     // (a dead lane 31 = end of the row anyway)
                }
            }
            // uint32 bins cannot wrap: any bin holds at most the hits all 8 warps added since their own last
            // flush, and a warp flushes (atomicExch, safe against concurrent adds) before it passes 2^28
            if (budget > p.flush) {
                for (int t = lane; t < p.nh; t += 32) {
                    const uint32_t c = atomicExch(&hist[t], 0u);
                    if (c) atomicAdd(&g_cnt[t], (unsigned long long)c);
                }
                budget = 0;
            }
        }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < p.nh; t += Q3_THREADS) {
        const uint32_t c = hist[t];
        if (c) atomicAdd(&g_cnt[t], (unsigned long long)c);
    }
}

// ---- A10 fold: raw hub-ordered (b_ij, b_ik, b_jk) -> sorted triple (A-5); also sums the weight slots ------
__global__ void k_fold3(int nb, const unsigned long long *__restrict__ raw_cnt, const double *__restrict__ raw_w,
                        int n_slots, unsigned long long *__restrict__ out_cnt, double *__restrict__ out_w)
{
    const int nh = nb * nb * nb;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= nh) return;
    const int a = x / (nb * nb), b = (x / nb) % nb, c = x % nb;
    unsigned long long cnt = 0;
    double ws = 0.0;
    if (a <= b && b <= c) {
        int perm[6][3] = {{a, b, c}, {a, c, b}, {b, a, c}, {b, c, a}, {c, a, b}, {c, b, a}};
        for (int q = 0; q < 6; ++q) {
            bool dup = false;
            for (int r = 0; r < q; ++r)
                dup = dup || (perm[r][0] == perm[q][0] && perm[r][1] == perm[q][1] && perm[r][2] == perm[q][2]);
            if (dup) continue;
            const int y = (perm[q][0] * nb + perm[q][1]) * nb + perm[q][2];
            if (raw_cnt) cnt += raw_cnt[y];
            if (raw_w)
                for (int s = 0; s < n_slots; ++s) ws += raw_w[(size_t)s * nh + y];
        }
    }
    if (out_cnt) out_cnt[x] = cnt;
    if (out_w) out_w[x] = ws;
}

// ---- A6: 2pCF sweep ("a single sweep of the graph") ---------------------------------------------------
__global__ void __launch_bounds__(256)
k_2pcf(GrView v, int nb, int weighted, unsigned long long *__restrict__ g_cnt, double *__restrict__ g_w)
{
    __shared__ unsigned int h_c[GR_MAXBINS + 1];
    __shared__ double h_w[GR_MAXBINS + 1];
    for (int t = threadIdx.x; t < nb; t += blockDim.x) { h_c[t] = 0; h_w[t] = 0.0; }
    __syncthreads();
    const int lane = lane_id();
    const int warps_total = gridDim.x * (blockDim.x >> 5);
    for (int64_t i = v.h_lo + (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < v.h_hi; i += warps_total) {
        const int64_t rb = v.ptr[i], re = v.ptr[i + 1];
        const double wi = weighted ? v.w[i] : 1.0;
        for (int64_t e = rb + lane; e < re; e += 32) {
            const int b = v.bin_h[e - v.e0_h];
            atomicAdd(&h_c[b], 1u);
            if (weighted) atomicAdd(&h_w[b], wi * v.w[v.idx_h[e - v.e0_h]]);
        }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < nb; t += blockDim.x) {
        if (h_c[t]) atomicAdd(&g_cnt[t], (unsigned long long)h_c[t]);
        if (weighted && h_w[t] != 0.0) atomicAdd(&g_w[t], h_w[t]);
    }
}

// ---- exact work counters (S:8(d)): sum over oriented edges of len(N+(j)) and of the tail lengths ----------
__global__ void k_work(GrView v, unsigned long long *__restrict__ out)
{
    const int lane = lane_id();
    const int warps_total = gridDim.x * (blockDim.x >> 5);
    unsigned long long spoke = 0, tail = 0;
    for (int64_t i = v.h_lo + (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < v.h_hi; i += warps_total) {
        const int64_t rb = v.ptr[i], re = v.ptr[i + 1];
        for (int64_t e = rb + lane; e < re; e += 32) {
            const int32_t j = v.idx_h[e - v.e0_h];
            spoke += (unsigned long long)(v.ptr[j + 1] - v.ptr[j]);
            tail += (unsigned long long)(re - e - 1);
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        spoke += __shfl_xor_sync(0xffffffffu, spoke, o);
        tail += __shfl_xor_sync(0xffffffffu, tail, o);
    }
    if (lane == 0) { atomicAdd(&out[0], spoke); atomicAdd(&out[1], tail); }
}

struct Q3Run {
    Q3Params p;
    T3Params t;
    unsigned int *counter;
    unsigned long long *raw_cnt;
    double *raw_w;
    int grid;
    size_t smem;
    int use_table, G, long_rows, use_merge;
};

template <bool W, int U>
void launch_table(const Q3Run *r, const GrView &v, cudaStream_t st)
{
    switch (r->G) {
        case 1: k_3pcf_table<W, 1, U><<<r->grid, Q3_THREADS, r->smem, st>>>(v, r->t, r->counter, r->raw_cnt, r->raw_w); break;
        case 2: k_3pcf_table<W, 2, U><<<r->grid, Q3_THREADS, r->smem, st>>>(v, r->t, r->counter, r->raw_cnt, r->raw_w); break;
        case 4: k_3pcf_table<W, 4, U><<<r->grid, Q3_THREADS, r->smem, st>>>(v, r->t, r->counter, r->raw_cnt, r->raw_w); break;
        default: k_3pcf_table<W, 8, U><<<r->grid, Q3_THREADS, r->smem, st>>>(v, r->t, r->counter, r->raw_cnt, r->raw_w); break;
    }
}

template <bool W, int U>
const void *table_fn(int G)
{
    switch (G) {
        case 1: return (const void *)k_3pcf_table<W, 1, U>;
        case 2: return (const void *)k_3pcf_table<W, 2, U>;
        case 4: return (const void *)k_3pcf_table<W, 4, U>;
        default: return (const void *)k_3pcf_table<W, 8, U>;
    }
}

void tile_3pcf(gramsci_graph *g, const GrView &v, void *user, cudaStream_t st)
{
    Q3Run *r = (Q3Run *)user;
    GR_CUDA(cudaMemsetAsync(r->counter, 0, sizeof(unsigned int), st));
    if (r->use_merge) {
        if (r->p.weighted) k_3pcf_merge<true><<<r->grid, Q3_THREADS, r->smem, st>>>(v, r->p, r->counter, r->raw_cnt, r->raw_w);
        else k_3pcf_merge<false><<<r->grid, Q3_THREADS, r->smem, st>>>(v, r->p, r->counter, r->raw_cnt, r->raw_w);
    } else if (r->use_table) {
        if (r->p.weighted) { if (r->long_rows) launch_table<true, GR_LONG_U>(r, v, st); else launch_table<true, 4>(r, v, st); }
        else { if (r->long_rows) launch_table<false, GR_LONG_U>(r, v, st); else launch_table<false, 4>(r, v, st); }
    } else if (r->p.weighted)
        k_3pcf_bsearch<true><<<r->grid, Q3_THREADS, r->smem, st>>>(v, r->p, r->counter, r->raw_cnt, r->raw_w);
    else
        k_3pcf_bsearch<false><<<r->grid, Q3_THREADS, r->smem, st>>>(v, r->p, r->counter, r->raw_cnt, r->raw_w);
    GR_CUDA(cudaGetLastError());
    g->n_launches += 1;
}

// shared memory of one group of the slot-table kernel for page shift s (0 = does not apply)
size_t table_group_bytes(const gramsci_graph *g, int s, bool weighted, int G, int row_cap, int *pt_len, int *tab_len)
{
    const size_t a16 = 15;
    const int64_t ptl = (int64_t)g->max_ptl[s] + 1;      // + sentinel page
    const int64_t tbl = ((int64_t)g->max_pages[s] + 1) << s;
    if (ptl > (1 << 20) || tbl > 65536 || g->max_pages[s] >= 65535) return 0;      // slot bases are uint16
    *pt_len = (int)ptl;
    *tab_len = (int)tbl;
    size_t b = (size_t)G * 32 * (16 + (weighted ? 8 : 0));
    b += ((size_t)ptl * 2 + a16) & ~a16;
    b += ((size_t)tbl * (weighted ? 2 : 1) + a16) & ~a16;
    if (weighted) b += (size_t)row_cap * 8 + (((size_t)row_cap + a16) & ~a16);
    return (b + a16) & ~a16;
}

struct Q2Run { unsigned long long *cnt; double *w; int weighted; };

void tile_2pcf(gramsci_graph *g, const GrView &v, void *user, cudaStream_t st)
{
    Q2Run *r = (Q2Run *)user;
    // enough CTAs that no shared uint32 bin can wrap (each CTA sees < 2^30 edges)
    int64_t e_tile = g->n_edges;
    int grid = (int)std::max<int64_t>(g->sm_count * 4, (e_tile >> 30) + 1);
    k_2pcf<<<grid, 256, 0, st>>>(v, g->nb, r->weighted, r->cnt, r->w);
    GR_CUDA(cudaGetLastError());
    g->n_launches += 1;
}

void tile_work(gramsci_graph *g, const GrView &v, void *user, cudaStream_t st)
{
    k_work<<<g->sm_count * 4, 256, 0, st>>>(v, (unsigned long long *)user);
    GR_CUDA(cudaGetLastError());
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------
void gr_fold3(gramsci_graph *g, int nb, const unsigned long long *raw_cnt, const double *raw_w, int n_slots,
              uint64_t *d_counts, double *d_wsum)
{
    const int nh = nb * nb * nb;
    k_fold3<<<(nh + 255) / 256, 256, 0, g->stream>>>(nb, raw_cnt, raw_w, n_slots, (unsigned long long *)d_counts, d_wsum);
    GR_CUDA(cudaGetLastError());
}

// the equilateral histogram [nb]: raw bins are final, only the fp64 slabs are summed
__global__ void k_sum_eq(int nb, const unsigned long long *__restrict__ cnt, const double *__restrict__ w, int n_slabs,
                         unsigned long long *__restrict__ out_cnt, double *__restrict__ out_w)
{
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= nb) return;
    if (out_cnt) out_cnt[x] = cnt[x];
    if (out_w) {
        double s = 0.0;
        for (int k = 0; k < n_slabs; ++k) s += w[(size_t)k * nb + x];
        out_w[x] = s;
    }
}

void gr_3pcf(gramsci_graph *g, uint64_t *d_counts, double *d_wsum, int equilateral)
{
    cudaStream_t st = g->stream;
    const int nb = g->nb;
    const int64_t nh64 = equilateral ? (int64_t)nb : (int64_t)nb * nb * nb;
    if (nh64 > (int64_t)1 << 26) GR_FAIL(GRAMSCI_EINVAL, "3pcf: nbins^3 too large");
    const int nh = (int)nh64;
    GrTimer total(st);
    g->n_launches = 0;
    g->staged_bytes = 0;
    if (!d_counts && !d_wsum) { g->t_query_ms = total.stop(); return; }

    // ---- gather kernel (query3g.cu): the default wherever its dense rows apply ----
    if (g->algo == GRAMSCI_ALGO_DEFAULT || g->algo == GRAMSCI_ALGO_GATHER) {
        const char *why = "";
        const size_t planes = (size_t)((!d_wsum || d_counts) ? 1 : 0) + (d_wsum ? 3 : 0);
        const size_t hist_bytes = planes * (size_t)((nh + 32) & ~31) * 4;
        if (gr_gather_applicable(g, d_wsum != nullptr, hist_bytes, &why)) {
            gr_3pcf_gather(g, d_counts, d_wsum, equilateral);
            g->t_query_ms = total.stop();          // includes the one-off expansion of the dense rows
            return;
        }
        if (g->algo == GRAMSCI_ALGO_GATHER)
            GR_FAIL(GRAMSCI_ERANGE, "3pcf: the gather kernel does not apply to this graph (%s)", why);
    }

    Q3Run r;
    r.p.nb = nb; r.p.nh = nh;
    r.p.equi = equilateral ? 1 : 0;
    r.p.weighted = (d_wsum != nullptr) ? 1 : 0;
    r.p.want_counts = (d_counts != nullptr) ? 1 : 0;
    r.p.row_cap = std::max(16, (g->max_row + 15) & ~15);
    const bool W = r.p.weighted != 0;

    // ---- slot-table kernel: page shift s minimising the table, then the smallest group that fits ----
    r.use_table = 0;
    r.G = 8;
    // rows of hundreds of entries and more stream from DRAM (the CSR no longer lives in L2): keep 8 windows in flight
    r.long_rows = (g->n > 0 && g->n_edges / g->n >= 512) ? 1 : 0;
    r.use_merge = (g->algo == GRAMSCI_ALGO_MERGEPATH && !equilateral) ? 1 : 0;
    if (!equilateral && g->algo >= GRAMSCI_ALGO_BITMAP && g->algo <= GRAMSCI_ALGO_TABLE_G8 && g->max_row >= 65535)
        GR_FAIL(GRAMSCI_ERANGE, "3pcf: slot table needs rows shorter than 65535 entries (longest row %d)", g->max_row);
    // (the equilateral restriction exists in the gather kernels and, as the fallback for graphs they do not take, in
    //  the search kernel)
    if (!equilateral && g->algo != GRAMSCI_ALGO_BSEARCH && !r.use_merge && g->max_row >= 2 && g->max_row < 65535) {
        gr_row_stats(g);
        const size_t hist_bytes = (((size_t)nh * 4 + 15) & ~(size_t)15) + 16;
        int best_s = -1, ptl = 0, tbl = 0;
        size_t best = 0;
        for (int s = GR_S_MIN; s <= GR_S_MAX; ++s) {
            int a = 0, b = 0;
            const size_t bytes = table_group_bytes(g, s, W, 1, r.p.row_cap, &a, &b);
            if (bytes && (best_s < 0 || bytes < best)) { best = bytes; best_s = s; ptl = a; tbl = b; }
        }
        if (best_s >= 0) {
            const size_t soft = 100 * 1024;       // two CTAs per SM
            int G = 0;
            const int forced = (g->algo >= GRAMSCI_ALGO_TABLE_G1 && g->algo <= GRAMSCI_ALGO_TABLE_G8) ? (1 << (g->algo - GRAMSCI_ALGO_TABLE_G1)) : 0;
            for (int cand = 1; cand <= 8 && !G; cand *= 2) {
                if (forced && cand != forced) continue;
                const size_t cta = hist_bytes + (size_t)(Q3_WARPS / cand) * table_group_bytes(g, best_s, W, cand, r.p.row_cap, &ptl, &tbl);
                if (cta <= soft || ((cand == 8 || forced) && cta <= g->smem_optin)) G = cand;
            }
            if (G) {
                r.use_table = 1;
                r.G = G;
                r.t.nb = nb; r.t.nh = nh; r.t.s = best_s; r.t.pt_len = ptl; r.t.tab_len = tbl;
                r.t.row_cap = r.p.row_cap; r.t.want_counts = r.p.want_counts;
                r.t.group_bytes = (int)table_group_bytes(g, best_s, W, G, r.p.row_cap, &ptl, &tbl);
                r.t.hub_batch = (G == 8) ? 1 : 4;
                r.smem = hist_bytes + (size_t)(Q3_WARPS / G) * r.t.group_bytes;
            }
        }
        if (!r.use_table && g->algo >= GRAMSCI_ALGO_BITMAP && g->algo <= GRAMSCI_ALGO_TABLE_G8)
            GR_FAIL(GRAMSCI_ERANGE, "3pcf: slot table does not fit in shared memory (longest row %d)", g->max_row);
    }
    const void *fn;
    if (r.use_merge) {
        const size_t rc = (size_t)r.p.row_cap;
        r.smem = (W ? rc * 8 : 0) + (rc + 8) * 4 + rc + 32 + (size_t)nh * 4 + (size_t)Q3_WARPS * MP_TILE * 5 + 64;
        if (r.smem > g->smem_optin)
            GR_FAIL(GRAMSCI_ERANGE, "3pcf: longest row (%d entries) does not fit in shared memory", g->max_row);
        fn = W ? (const void *)k_3pcf_merge<true> : (const void *)k_3pcf_merge<false>;
    } else if (r.use_table) {
        fn = W ? (r.long_rows ? table_fn<true, GR_LONG_U>(r.G) : table_fn<true, 4>(r.G))
               : (r.long_rows ? table_fn<false, GR_LONG_U>(r.G) : table_fn<false, 4>(r.G));
    } else {
        r.p.smem_hist = ((size_t)nh * 4 <= 96 * 1024) ? 1 : 0;
        size_t per_entry = 4 + 1 + (W ? 8 : 0);
        r.smem = (size_t)r.p.row_cap * per_entry + (r.p.smem_hist ? (size_t)nh * 4 : 0) + 64;
        if (r.smem > g->smem_optin)
            GR_FAIL(GRAMSCI_ERANGE, "3pcf: longest row (%d entries) does not fit in shared memory", g->max_row);
        fn = W ? (const void *)k_3pcf_bsearch<true> : (const void *)k_3pcf_bsearch<false>;
    }
    int occ = gr_kernel_occupancy(fn, Q3_THREADS, r.smem);
    occ = std::max(1, std::min(occ, 8));
    r.grid = g->sm_count * occ;

    if (getenv("GRAMSCI_DEBUG"))
        fprintf(stderr, "[gramsci] 3pcf: table=%d G=%d s=%d pt_len=%d tab_len=%d group_bytes=%d smem=%zu occ=%d grid=%d span=%d row=%d\n",
                r.use_table, r.G, r.use_table ? r.t.s : -1, r.use_table ? r.t.pt_len : 0, r.use_table ? r.t.tab_len : 0,
                r.use_table ? r.t.group_bytes : 0, r.smem, occ, r.grid, 0, g->max_row);

    DevBuf<unsigned int> counter;
    DevBuf<unsigned long long> raw_cnt;
    DevBuf<double> raw_w;
    counter.alloc(1);
    raw_cnt.alloc((size_t)nh);
    GR_CUDA(cudaMemsetAsync(raw_cnt.p, 0, sizeof(unsigned long long) * nh, st));
    // fp64 slabs (weighted only): one per CTA while they fit a byte budget, else CTAs share slabs (blockIdx % n)
    const int n_slots = (int)std::max<int64_t>(1, std::min<int64_t>(r.grid, ((int64_t)256 << 20) / ((int64_t)nh * 8)));
    r.p.n_slabs = r.t.n_slabs = n_slots;
    r.p.flush = gr_flush_budget(0xF0000000ull);
    r.t.flush = gr_flush_budget(1ull << 28);
    if (W) {
        raw_w.alloc((size_t)nh * n_slots);
        GR_CUDA(cudaMemsetAsync(raw_w.p, 0, sizeof(double) * (size_t)nh * n_slots, st));
    }
    r.counter = counter.p; r.raw_cnt = raw_cnt.p; r.raw_w = raw_w.p;

    {
        GrTimer en(st);
        gr_for_each_tile(g, false, false, tile_3pcf, &r);
        g->t_enum_ms = en.stop();
    }
    if (equilateral) {
        k_sum_eq<<<(nb + 127) / 128, 128, 0, st>>>(nb, raw_cnt.p, W ? raw_w.p : nullptr, n_slots, (unsigned long long *)d_counts, d_wsum);
        GR_CUDA(cudaGetLastError());
    } else {
        gr_fold3(g, nb, d_counts ? raw_cnt.p : nullptr, W ? raw_w.p : nullptr, n_slots, d_counts, d_wsum);
    }
    g->n_launches += 1;
    GR_CUDA(cudaStreamSynchronize(st));
    g->t_query_ms = total.stop();
}

void gr_2pcf(gramsci_graph *g, uint64_t *d_counts, double *d_wsum)
{
    cudaStream_t st = g->stream;
    GrTimer total(st);
    g->n_launches = 0;
    g->staged_bytes = 0;
    DevBuf<unsigned long long> cnt;
    DevBuf<double> w;
    cnt.alloc(GR_MAXBINS + 1);
    w.alloc(GR_MAXBINS + 1);
    GR_CUDA(cudaMemsetAsync(cnt.p, 0, sizeof(unsigned long long) * (GR_MAXBINS + 1), st));
    GR_CUDA(cudaMemsetAsync(w.p, 0, sizeof(double) * (GR_MAXBINS + 1), st));
    Q2Run r{cnt.p, w.p, d_wsum ? 1 : 0};
    {
        GrTimer en(st);
        gr_for_each_tile(g, false, true, tile_2pcf, &r);    // hub windows only
        g->t_enum_ms = en.stop();
    }
    if (d_counts) GR_CUDA(cudaMemcpyAsync(d_counts, cnt.p, sizeof(uint64_t) * g->nb, cudaMemcpyDeviceToDevice, st));
    if (d_wsum) GR_CUDA(cudaMemcpyAsync(d_wsum, w.p, sizeof(double) * g->nb, cudaMemcpyDeviceToDevice, st));
    GR_CUDA(cudaStreamSynchronize(st));
    g->t_query_ms = total.stop();
}

void gr_work_counters(gramsci_graph *g, uint64_t *spoke_elems, uint64_t *tail_elems)
{
    cudaStream_t st = g->stream;
    DevBuf<unsigned long long> out;
    out.alloc(2);
    GR_CUDA(cudaMemsetAsync(out.p, 0, 16, st));
    gr_for_each_tile(g, false, true, tile_work, out.p);
    unsigned long long h[2];
    GR_CUDA(cudaMemcpyAsync(h, out.p, 16, cudaMemcpyDeviceToHost, st));
    GR_CUDA(cudaStreamSynchronize(st));
    if (spoke_elems) *spoke_elems = h[0];
    if (tail_elems) *tail_elems = h[1];
}
