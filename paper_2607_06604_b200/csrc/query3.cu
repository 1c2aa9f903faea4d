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

namespace {

constexpr int Q3_THREADS = 256;
constexpr int Q3_WARPS = Q3_THREADS / 32;

struct Q3Params {
    int nb;
    int nh;             // nb^3
    int row_cap;        // entries of the staged hub row
    int smem_hist;      // 1: uint32 histogram in shared memory
    int weighted;
    int want_counts;
};

// ---- hub row staging ---------------------------------------------------------------------------------
struct HubRow {
    int32_t *idx;   // [row_cap]
    uint8_t *bin;   // [row_cap]
    double *w;      // [row_cap] (weighted only)
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
    double *my_w = WEIGHTED ? g_w + (size_t)blockIdx.x * p.nh : nullptr;
    __syncthreads();

    for (;;) {
        if (threadIdx.x == 0) s_slot = v.s_lo + (int)atomicAdd(hub_counter, 1u);
        __syncthreads();
        const int s = s_slot;
        if (s >= v.s_hi) break;
        const int32_t i = v.order[s];
        const bool mine = (i >= v.h_lo && i < v.h_hi);
        const int64_t rb = mine ? v.ptr[i] : 0, re = mine ? v.ptr[i + 1] : 0;
        const int n = (int)(re - rb);
        if (n >= 2) {
            // uint32 histogram overflow guard: a hub adds at most n(n-1)/2 hits
            if (p.smem_hist) {
                unsigned long long add = (unsigned long long)n * (n - 1) / 2;
                if (budget + add > 0xF0000000ull) {
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
                const int hbase = (int)a_bin[a] * nb * nb;
                const double wij = WEIGHTED ? wi * a_w[a] : 1.0;
                int lo = 0;
                for (int t0 = 0; t0 < nj; t0 += 32) {
                    const int t = t0 + lane;
                    int32_t k = (t < nj) ? B[t] : INT32_MAX;
                    int pos = nt;
                    if (k <= t_last) pos = lower_bound_s(T, lo, nt, k);
                    const bool hit = (pos < nt) && (T[pos] == k);
                    if (hit) {
                        const int h = hbase + (int)a_bin[a + 1 + pos] * nb + (int)Bb[t];
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
    unsigned int *counter;
    unsigned long long *raw_cnt;
    double *raw_w;
    int grid;
    size_t smem;
    int algo;
};

void tile_3pcf(gramsci_graph *g, const GrView &v, void *user, cudaStream_t st)
{
    Q3Run *r = (Q3Run *)user;
    GR_CUDA(cudaMemsetAsync(r->counter, 0, sizeof(unsigned int), st));
    if (r->p.weighted)
        k_3pcf_bsearch<true><<<r->grid, Q3_THREADS, r->smem, st>>>(v, r->p, r->counter, r->raw_cnt, r->raw_w);
    else
        k_3pcf_bsearch<false><<<r->grid, Q3_THREADS, r->smem, st>>>(v, r->p, r->counter, r->raw_cnt, r->raw_w);
    GR_CUDA(cudaGetLastError());
    g->n_launches += 1;
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
void gr_3pcf(gramsci_graph *g, uint64_t *d_counts, double *d_wsum)
{
    cudaStream_t st = g->stream;
    const int nb = g->nb;
    const int64_t nh64 = (int64_t)nb * nb * nb;
    if (nh64 > (int64_t)1 << 26) GR_FAIL(GRAMSCI_EINVAL, "3pcf: nbins^3 too large");
    const int nh = (int)nh64;
    GrTimer total(st);
    g->n_launches = 0;
    g->staged_bytes = 0;

    Q3Run r;
    r.algo = g->algo;
    r.p.nb = nb; r.p.nh = nh;
    r.p.weighted = (d_wsum != nullptr) ? 1 : 0;
    r.p.want_counts = (d_counts != nullptr) ? 1 : 0;
    r.p.row_cap = std::max(16, (g->max_row + 15) & ~15);
    r.p.smem_hist = ((size_t)nh * 4 <= 96 * 1024) ? 1 : 0;
    size_t per_entry = 4 + 1 + (r.p.weighted ? 8 : 0);
    r.smem = (size_t)r.p.row_cap * per_entry + (r.p.smem_hist ? (size_t)nh * 4 : 0) + 64;
    if (r.smem > g->smem_optin)
        GR_FAIL(GRAMSCI_ERANGE, "3pcf: longest row (%d entries) does not fit in shared memory", g->max_row);
    GR_CUDA(cudaFuncSetAttribute(k_3pcf_bsearch<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)r.smem));
    GR_CUDA(cudaFuncSetAttribute(k_3pcf_bsearch<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)r.smem));
    int occ = 1;
    if (r.p.weighted)
        GR_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_3pcf_bsearch<true>, Q3_THREADS, r.smem));
    else
        GR_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_3pcf_bsearch<false>, Q3_THREADS, r.smem));
    occ = std::max(1, std::min(occ, 8));
    r.grid = g->sm_count * occ;

    DevBuf<unsigned int> counter;
    DevBuf<unsigned long long> raw_cnt;
    DevBuf<double> raw_w;
    counter.alloc(1);
    raw_cnt.alloc((size_t)nh);
    GR_CUDA(cudaMemsetAsync(raw_cnt.p, 0, sizeof(unsigned long long) * nh, st));
    if (r.p.weighted) {
        raw_w.alloc((size_t)nh * r.grid);
        GR_CUDA(cudaMemsetAsync(raw_w.p, 0, sizeof(double) * (size_t)nh * r.grid, st));
    }
    r.counter = counter.p; r.raw_cnt = raw_cnt.p; r.raw_w = raw_w.p;

    {
        GrTimer en(st);
        gr_for_each_tile(g, false, false, tile_3pcf, &r);
        g->t_enum_ms = en.stop();
    }
    k_fold3<<<(nh + 255) / 256, 256, 0, st>>>(nb, raw_cnt.p, r.p.weighted ? raw_w.p : nullptr, r.grid,
                                             (unsigned long long *)d_counts, d_wsum);
    GR_CUDA(cudaGetLastError());
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
