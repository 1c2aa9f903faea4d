// query4.cu -- S:8(a) A8 (4pCF second-level intersection), A9 (parity split), A10 (fold + flush).
//
// tetrahedra are the tuples (i, j1, j2, j3) whose six pairs are all graph edges; P:72-87 finds j3
// by walking three sorted lists at once, P:149 instead precomputes, per hub, the "local connectivity
// matrix lmat(k2,k1)" holding the bin of the edge between two hub neighbours, so that the innermost
// loop is O(1) lookups after C(m,2) membership searches per hub.  This file takes the second design
// and restates it for a CTA:
//
//   phase 1 (per hub i, = the 3pCF membership pass): row a of the local matrix D is
//            D[a][p] = bin of edge (k_a, k_p) if k_p in N+(k_a) else 0xFF,   a < p < n = len(N+(i)),
//            found by one lane-parallel search of every element of N+(k_a) in the staged hub row;
//   phase 2: D also exists as bit rows.  Warps scan the bit rows for local edges (a,b), compact them with
//            ballots into a small queue, and every LANE takes one local edge: the set bits c > b of
//            bits[a] & bits[b] are the 4-cliques i < k_a < k_b < k_c, each found exactly once (oriented
//            storage, A-1, A-15) and histogrammed by its raw 6-tuple (b_ia, b_ib, b_ic, b_ab, b_ac, b_bc)
//            = the order (b12,b13,b14,b23,b24,b34).  (A first version gave a warp to each local edge and
//            streamed the byte rows; with rows of ~50 entries most lanes idled: 37 ms vs now on cfg3.)
//
// Parity (Eq. 3; A-8..A-11): V = (n_a x n_b) . n_c on the pixel-centre unit vectors of the three
// hub spokes, every product and sum rounded separately; the kernel files every hit under the RAW tuple in
// one of three sign classes (V > 0, V < 0, |V| < 1e-9) -- one atomic per hit and kind of output instead of
// separate even and odd updates -- and the fold forms even = pos + neg + degenerate and odd = chi (pos - neg)
// with the chirality factor of the raw tuple, which for the raw tuple t^sigma of a canonical chiral tuple t
// is sgn(sigma) (and 0 for bin-achiral t).
//
// D lives in shared memory when the longest row allows (a few hundred entries), else in a per-CTA slice of a
// global scratch (the paper's "per-gang slice of a global scratch sized from the longest row"),
// written and read by the same CTA only (L1/L2 resident).
// Raw histograms are nb^6 bins -- too large for shared memory (8^6 x 4 B = 1 MiB) -- so hits go to
// global memory with RED atomics, spread over a few shards that the fold sums.
#include "internal.cuh"

#include <algorithm>
#include <cmath>
#include <cstdlib>

namespace {

constexpr int Q4_THREADS = 256;
constexpr int Q4_WARPS = Q4_THREADS / 32;

struct Q4Params {
    int nb;
    int64_t nh;          // nb^6
    int row_cap;         // staged hub row capacity (multiple of 16)
    int parity, weighted, want_counts;
    int n_shards;
    int ncfg;            // LUT path: number of canonical configurations (histograms are indexed by configuration)
    unsigned long long flush;   // LUT path: a warp drains the CTA histograms before its hit budget passes this
    int ooc;             // capped graph: tile (h, c1 <= c2) of P:159 -- spoke rows come from two resident search windows
};

__constant__ int8_t c_perm4[24][4] = {
    {0,1,2,3},{0,1,3,2},{0,2,1,3},{0,2,3,1},{0,3,1,2},{0,3,2,1},{1,0,2,3},{1,0,3,2},{1,2,0,3},{1,2,3,0},
    {1,3,0,2},{1,3,2,0},{2,0,1,3},{2,0,3,1},{2,1,0,3},{2,1,3,0},{2,3,0,1},{2,3,1,0},{3,0,1,2},{3,0,2,1},
    {3,1,0,2},{3,1,2,0},{3,2,0,1},{3,2,1,0}};

__device__ __forceinline__ int lower_bound_s(const int32_t *a, int lo, int hi, int32_t key)
{
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if (a[mid] < key) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// ---- enumeration ---------------------------------------------------------------------------------------
// cnt_e/cnt_o/w_e/w_o: [n_shards][nh] raw histograms (any may be null).
// SMALL: the local matrix D (bytes) and its bit rows live in shared memory (rows up to a few hundred
// entries); otherwise in the CTA's slice of the global scratch.
// LUT: a raw tuple is mapped to its canonical configuration on the spot (lut[x] = configuration id | chirality
// code << 24, built on the device once per graph); counts then go to per-CTA SHARED uint32 / int32 histograms
// over configurations (native ATOMS, hardware-aggregated on equal addresses) and weighted sums to one global
// slab per CTA, instead of one global RED per hit and channel into nb^6 raw bins.  In that mode cnt_e/cnt_o
// are [ncfg] and w_e/w_o are [grid][ncfg]; without it they are [n_shards][nh] raw histograms.
template <bool SMALL, bool LUT>
__global__ void __launch_bounds__(Q4_THREADS)
k_4pcf(GrView v, Q4Params p, unsigned int *__restrict__ hub_counter, uint8_t *scratch, size_t scratch_stride,
       const double *__restrict__ pix_tab, const uint32_t *__restrict__ lut, unsigned long long *__restrict__ cnt_e,
       unsigned long long *__restrict__ cnt_o, double *__restrict__ w_e, double *__restrict__ w_o)
{
    extern __shared__ __align__(16) unsigned char smem[];
    // layout: [tab 256*3*8 (parity)] [w row_cap*8 (weighted)] [idx row_cap*4] [t3 row_cap*4] [queues 8*64*4]
    //         [LUT: h_e ncfg*4, h_o ncfg*4 (parity)] [pix row_cap] [SMALL: D row_cap*row_cap, bits row_cap*(row_cap/32)*4]
    double *s_tab = (double *)smem;
    double *a_w = (double *)(smem + (p.parity ? 256 * 3 * 8 : 0));
    int32_t *a_idx = (int32_t *)((unsigned char *)a_w + (p.weighted ? (size_t)p.row_cap * 8 : 0));
    uint32_t *a_t3 = (uint32_t *)(a_idx + p.row_cap);       // b_ic * nb^3
    uint32_t *s_queue = a_t3 + p.row_cap;                   // per warp: 64 pending local edges (a << 16 | b)
    uint32_t *h_e = s_queue + Q4_WARPS * 64;
    int *h_o = (int *)(h_e + (LUT ? p.ncfg : 0));
    const int ncfg_pad = LUT ? ((p.ncfg * (p.parity ? 2 : 1) + 3) & ~3) : 0;
    uint8_t *a_pix = (uint8_t *)(h_e + ncfg_pad);
    __shared__ int s_slot;

    const int nb = p.nb;
    const uint32_t nb2 = nb * nb, nb3 = nb2 * nb;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const unsigned lt_mask = (1u << lane) - 1u;
    uint8_t *D;
    uint32_t *bits;
    if (SMALL) {
        D = a_pix + p.row_cap;
        bits = (uint32_t *)(D + (size_t)p.row_cap * p.row_cap);
    } else {
        D = scratch + (size_t)blockIdx.x * scratch_stride;
        bits = (uint32_t *)(D + (size_t)p.row_cap * p.row_cap);
    }
    uint32_t *my_q = s_queue + warp * 64;
    if (LUT) {
        if (w_e) w_e += (size_t)blockIdx.x * p.ncfg;
        if (w_o) w_o += (size_t)blockIdx.x * p.ncfg;
        for (int t = threadIdx.x; t < ncfg_pad; t += Q4_THREADS) h_e[t] = 0u;
    } else {
        // raw mode: [n_shards][nh], or [n_shards][3][nh] (sign classes) for the parity split
        const size_t shard = (size_t)(blockIdx.x % p.n_shards) * (size_t)p.nh * (p.parity ? 3 : 1);
        if (cnt_e) cnt_e += shard;
        if (w_e) w_e += shard;
    }
    if (p.parity)
        for (int t = threadIdx.x; t < 256 * 3; t += Q4_THREADS) s_tab[t] = pix_tab[t];
    unsigned long long budget = 0;       // LUT: upper bound of the hits this warp added since it last flushed

    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_slot = v.s_lo + (int)atomicAdd(hub_counter, 1u);
        __syncthreads();
        const int s = s_slot;
        if (s >= v.s_hi) break;
        const int32_t i = v.order[s];
        if (!GR_HUB_SELECTED(v, i)) continue;
        if (i < v.h_lo || i >= v.h_hi) continue;               // hub of another window (capped graphs)
        const int64_t rb = v.ptr[i], re = v.ptr[i + 1];
        const int n = (int)(re - rb);
        if (n < 3) continue;                                   // a 4-clique needs three spokes
        const int ld = (n + 15) & ~15;                         // row stride of D (bytes)
        const int nw = (n + 31) >> 5;                          // row stride of bits (words)
        const int32_t *gi = v.idx_h + (rb - v.e0_h);
        const uint8_t *gb = v.bin_h + (rb - v.e0_h);
        const uint8_t *gp = v.pix_h ? v.pix_h + (rb - v.e0_h) : nullptr;
        for (int t = threadIdx.x; t < n; t += Q4_THREADS) {
            const int32_t k = gi[t];
            a_idx[t] = k;
            a_t3[t] = (uint32_t)gb[t] * nb3;
            if (p.parity) a_pix[t] = gp[t];
            if (p.weighted) a_w[t] = v.w[k];
        }
        {   // D := 0xFF, bits := 0
            const uint4 ff = make_uint4(0xffffffffu, 0xffffffffu, 0xffffffffu, 0xffffffffu);
            uint4 *D4 = (uint4 *)D;
            const int total = (n * ld) >> 4;
            for (int t = threadIdx.x; t < total; t += Q4_THREADS) D4[t] = ff;
            for (int t = threadIdx.x; t < n * nw; t += Q4_THREADS) bits[t] = 0u;
        }
        __syncthreads();

        // ---- phase 1: local connectivity matrix (bytes) and its bit rows ----
        for (int a = warp; a < n - 1; a += Q4_WARPS) {
            const int32_t j = a_idx[a];
            const int64_t jb = v.ptr[j], je = v.ptr[j + 1];
            const int nj = (int)(je - jb);
            const int32_t *B = v.idx_c + (jb - v.e0_c);
            const uint8_t *Bb = v.bin_c + (jb - v.e0_c);
            if (p.ooc) {
                // rows of j1 come from search window c1, rows of j2 from c2; other rows are not resident and
                // not needed: this tile only follows local edges (a, b) with k_a in c1 and k_b in c2
                if (j >= v.c_lo && j < v.c_hi) {
                } else if (j >= v.c2_lo && j < v.c2_hi) {
                    B = v.idx_c2 + (jb - v.e0_c2);
                    Bb = v.bin_c2 + (jb - v.e0_c2);
                } else continue;
            }
            const int32_t t_last = a_idx[n - 1];
            uint8_t *Da = D + (size_t)a * ld;
            uint32_t *Ba = bits + (size_t)a * nw;
            int lo = a + 1;
            for (int t0 = 0; t0 < nj; t0 += 32) {
                const int t = t0 + lane;
                const int32_t k = (t < nj) ? B[t] : INT32_MAX;
                int pos = n;
                if (k <= t_last) pos = lower_bound_s(a_idx, lo, n, k);
                if (pos < n && a_idx[pos] == k) {
                    Da[pos] = Bb[t];
                    atomicOr(&Ba[pos >> 5], 1u << (pos & 31));
                }
                lo = __shfl_sync(0xffffffffu, pos, 0);
                if (__shfl_sync(0xffffffffu, k, 31) > t_last) break;
            }
        }
        __syncthreads();

        // ---- phase 2: triangles of the local graph = 4-cliques under hub i; one LANE per local edge (a,b) ----
        const double wi = p.weighted ? v.w[i] : 1.0;
        auto process = [&](uint32_t pair) -> int {
            int nhit = 0;
            const int a = (int)(pair >> 16), b = (int)(pair & 0xffffu);
            const uint8_t *Da = D + (size_t)a * ld, *Db = D + (size_t)b * ld;
            const uint32_t *Ba = bits + (size_t)a * nw, *Bb2 = bits + (size_t)b * nw;
            const uint32_t base = a_t3[a] * nb2 + a_t3[b] * nb + (uint32_t)Da[b] * nb2;   // b_ia nb^5 + b_ib nb^4 + b_ab nb^2
            double cx = 0, cy = 0, cz = 0, wiab = 1.0;
            if (p.parity) {
                const double *qa = s_tab + 3 * a_pix[a], *qb = s_tab + 3 * a_pix[b];
                cx = __dsub_rn(__dmul_rn(qa[1], qb[2]), __dmul_rn(qa[2], qb[1]));
                cy = __dsub_rn(__dmul_rn(qa[2], qb[0]), __dmul_rn(qa[0], qb[2]));
                cz = __dsub_rn(__dmul_rn(qa[0], qb[1]), __dmul_rn(qa[1], qb[0]));
            }
            if (p.weighted) wiab = wi * a_w[a] * a_w[b];
            for (int w = (b + 1) >> 5; w < nw; ++w) {
                uint32_t common = Ba[w] & Bb2[w];
                if (w == ((b + 1) >> 5)) common &= ~((1u << ((b + 1) & 31)) - 1u);     // only c > b
                while (common) {
                    const int c = (w << 5) + __ffs(common) - 1;
                    common &= common - 1u;
                    const uint32_t x = base + a_t3[c] + (uint32_t)Da[c] * nb + (uint32_t)Db[c];
                    double ww = 0.0;
                    if (p.weighted) ww = wiab * a_w[c];
                    int sg = 0;
                    if (p.parity) {
                        const double *nc = s_tab + 3 * a_pix[c];
                        const double V = __dadd_rn(__dadd_rn(__dmul_rn(cx, nc[0]), __dmul_rn(cy, nc[1])),
                                                   __dmul_rn(cz, nc[2]));
                        if (fabs(V) >= 1e-9) sg = (V > 0.0) ? 1 : -1;
                    }
                    if (LUT) {
                        const uint32_t e = lut[x];
                        const uint32_t cid = e & 0xffffffu;
                        sg *= (int)(e >> 24) - 1;                              // chirality factor of the raw tuple (A-10)
                        ++nhit;
                        if (cnt_e) atomicAdd(&h_e[cid], 1u);
                        if (p.weighted && w_e) atomicAdd(&w_e[cid], ww);
                        if (sg != 0) {
                            if (cnt_o) atomicAdd(&h_o[cid], sg);
                            if (w_o) atomicAdd(&w_o[cid], sg > 0 ? ww : -ww);
                        }
                    } else if (p.parity) {
                        // one RED per hit and kind of output: the hit goes to the class of its sign (V > 0, V < 0,
                        // degenerate); even = sum of the classes, odd = pos - neg, formed by the fold
                        const size_t y = (size_t)(sg > 0 ? 0 : (sg < 0 ? 1 : 2)) * (size_t)p.nh + x;
                        if (cnt_e) atomicAdd(&cnt_e[y], 1ull);
                        if (p.weighted) atomicAdd(&w_e[y], ww);
                    } else {
                        if (cnt_e) atomicAdd(&cnt_e[x], 1ull);
                        if (p.weighted) atomicAdd(&w_e[x], ww);
                    }
                }
            }
            return nhit;
        };
        // LUT: uint32 / int32 bins cannot wrap -- any bin holds at most the hits all 8 warps added since their own
        // last flush, and a warp flushes the CTA histograms (atomicExch, safe against concurrent adds) before it
        // passes 2^27
        auto account = [&](int nhit) {
            if (!LUT) return;
            budget += (unsigned long long)__reduce_add_sync(0xffffffffu, nhit);
            if (budget > p.flush) {
                for (int t = lane; t < p.ncfg; t += 32) {
                    if (cnt_e) { const uint32_t c = atomicExch(&h_e[t], 0u); if (c) atomicAdd(&cnt_e[t], (unsigned long long)c); }
                    if (cnt_o) { const int c = atomicExch(&h_o[t], 0); if (c) atomicAdd(&cnt_o[t], (unsigned long long)(long long)c); }
                }
                budget = 0;
            }
        };
        int qn = 0;                                            // warp-uniform queue fill
        for (int a = warp; a < n - 2; a += Q4_WARPS) {
            const uint32_t *Ba = bits + (size_t)a * nw;
            if (p.ooc && (a_idx[a] < v.c_lo || a_idx[a] >= v.c_hi)) continue;      // j1 belongs to another tile
            for (int w = (a + 1) >> 5; w < nw; ++w) {          // lanes scan the 32 candidates b of word w
                const int bcand = (w << 5) + lane;
                bool edge = bcand > a && bcand < n - 1 && ((Ba[w] >> lane) & 1u);
                if (p.ooc && edge) edge = a_idx[bcand] >= v.c2_lo && a_idx[bcand] < v.c2_hi;   // j2 in window c2
                const unsigned m = __ballot_sync(0xffffffffu, edge);
                if (edge) my_q[qn + __popc(m & lt_mask)] = ((uint32_t)a << 16) | (uint32_t)bcand;
                qn += __popc(m);
                __syncwarp();
                if (qn >= 32) {
                    const uint32_t pr = my_q[lane];
                    const uint32_t rest = my_q[32 + lane];
                    __syncwarp();
                    my_q[lane] = rest;
                    qn -= 32;
                    account(process(pr));
                    __syncwarp();
                }
            }
        }
        if (qn > 0) {
            __syncwarp();
            account((lane < qn) ? process(my_q[lane]) : 0);
        }
    }
    if (LUT) {
        __syncthreads();
        for (int t = threadIdx.x; t < p.ncfg; t += Q4_THREADS) {
            if (cnt_e && h_e[t]) atomicAdd(&cnt_e[t], (unsigned long long)h_e[t]);
            if (cnt_o && h_o[t]) atomicAdd(&cnt_o[t], (unsigned long long)(long long)h_o[t]);
        }
    }
}

// ---- LUT construction: canonical flag per raw tuple, then (after a scan) configuration id and chirality -------
__device__ __forceinline__ void canon4_dev(int nb, int64_t x, int64_t &ymin, int &chi)
{
    int t[6];
    {
        int64_t r = x;
        for (int e = 5; e >= 0; --e) { t[e] = (int)(r % nb); r /= nb; }
    }
    int m[4][4];
    m[0][0] = m[1][1] = m[2][2] = m[3][3] = 0;
    m[0][1] = m[1][0] = t[0]; m[0][2] = m[2][0] = t[1]; m[0][3] = m[3][0] = t[2];
    m[1][2] = m[2][1] = t[3]; m[1][3] = m[3][1] = t[4]; m[2][3] = m[3][2] = t[5];
    ymin = x;
    int npos = 0, nneg = 0;
    bool first = true;
    for (int s = 0; s < 24; ++s) {
        const int8_t *q = c_perm4[s];
        const int u[6] = {m[q[0]][q[1]], m[q[0]][q[2]], m[q[0]][q[3]], m[q[1]][q[2]], m[q[1]][q[3]], m[q[2]][q[3]]};
        int64_t y = 0;
        for (int e = 0; e < 6; ++e) y = y * nb + u[e];
        int inv = 0;
        for (int a = 0; a < 4; ++a)
            for (int b = a + 1; b < 4; ++b) inv += (q[a] > q[b]) ? 1 : 0;
        if (first || y < ymin) { ymin = y; npos = nneg = 0; first = false; }
        if (y == ymin) { if (inv & 1) ++nneg; else ++npos; }
    }
    chi = (npos && nneg) ? 0 : (npos ? 1 : -1);      // parity of the vertex orders reaching the minimum (A-10)
}

__global__ void k_lut_flag(int nb, int64_t nh, int32_t *__restrict__ flag)
{
    const int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= nh) return;
    int64_t ymin;
    int chi;
    canon4_dev(nb, x, ymin, chi);
    flag[x] = (ymin == x) ? 1 : 0;
}

__global__ void k_lut_fill(int nb, int64_t nh, const int32_t *__restrict__ rank, uint32_t *__restrict__ lut,
                           int32_t *__restrict__ dense_of)
{
    const int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= nh) return;
    int64_t ymin;
    int chi;
    canon4_dev(nb, x, ymin, chi);
    lut[x] = (uint32_t)rank[ymin] | ((uint32_t)(chi + 1) << 24);
    if (ymin == x) dense_of[rank[x]] = (int32_t)x;
}

// LUT path fold: per configuration, counts as they are and the per-CTA weight slabs summed
__global__ void k_fold4_cfg(int ncfg, int n_slabs, const int32_t *__restrict__ dense_of,
                            const unsigned long long *__restrict__ cnt_e, const unsigned long long *__restrict__ cnt_o,
                            const double *__restrict__ w_e, const double *__restrict__ w_o,
                            unsigned long long *__restrict__ out_ce, long long *__restrict__ out_co,
                            double *__restrict__ out_we, double *__restrict__ out_wo)
{
    const int c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncfg) return;
    const int64_t x = dense_of[c];
    if (out_ce) out_ce[x] = cnt_e[c];
    if (out_co) out_co[x] = (long long)cnt_o[c];
    if (out_we || out_wo) {
        double se = 0.0, so = 0.0;
        for (int k = 0; k < n_slabs; ++k) {
            if (out_we) se += w_e[(size_t)k * ncfg + c];
            if (out_wo) so += w_o[(size_t)k * ncfg + c];
        }
        if (out_we) out_we[x] = se;
        if (out_wo) out_wo[x] = so;
    }
}

// ---- A10 fold: raw 6-tuples -> canonical configurations (A-7), odd channel with the chirality sign (A-10) ---
__global__ void k_fold4(int nb, int64_t nh, int n_shards, int cls3, const unsigned long long *__restrict__ cnt_e,
                        const unsigned long long *__restrict__ cnt_o, const double *__restrict__ w_e,
                        const double *__restrict__ w_o, unsigned long long *__restrict__ out_ce,
                        long long *__restrict__ out_co, double *__restrict__ out_we, double *__restrict__ out_wo)
{
    const int64_t x = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= nh) return;
    int t[6];
    {
        int64_t r = x;
        for (int e = 5; e >= 0; --e) { t[e] = (int)(r % nb); r /= nb; }
    }
    int m[4][4];
    m[0][0] = m[1][1] = m[2][2] = m[3][3] = 0;
    m[0][1] = m[1][0] = t[0]; m[0][2] = m[2][0] = t[1]; m[0][3] = m[3][0] = t[2];
    m[1][2] = m[2][1] = t[3]; m[1][3] = m[3][1] = t[4]; m[2][3] = m[3][2] = t[5];
    int64_t ys[24];
    bool canonical = true, odd_aut = false;
    for (int s = 0; s < 24; ++s) {
        const int8_t *q = c_perm4[s];
        const int u[6] = {m[q[0]][q[1]], m[q[0]][q[2]], m[q[0]][q[3]], m[q[1]][q[2]], m[q[1]][q[3]], m[q[2]][q[3]]};
        int64_t y = 0;
        for (int e = 0; e < 6; ++e) y = y * nb + u[e];
        ys[s] = y;
        if (y < x) canonical = false;            // base-nb value order == lexicographic order of the tuple
        int inv = 0;
        for (int a = 0; a < 4; ++a)
            for (int b = a + 1; b < 4; ++b) inv += (q[a] > q[b]) ? 1 : 0;
        if (y == x && (inv & 1)) odd_aut = true; // an odd vertex order fixes the tuple: achiral at bin resolution
    }
    unsigned long long ce = 0;
    long long co = 0;
    double we = 0.0, wo = 0.0;
    if (canonical) {
        for (int s = 0; s < 24; ++s) {
            bool dup = false;
            for (int r = 0; r < s; ++r) dup = dup || (ys[r] == ys[s]);
            if (dup) continue;
            const int8_t *q = c_perm4[s];
            int inv = 0;
            for (int a = 0; a < 4; ++a)
                for (int b = a + 1; b < 4; ++b) inv += (q[a] > q[b]) ? 1 : 0;
            const int sg = (inv & 1) ? -1 : 1;
            for (int sh = 0; sh < n_shards; ++sh) {
                if (cls3) {            // parity: raw classes pos / neg / degenerate per shard
                    const size_t y = (size_t)sh * 3 * (size_t)nh + (size_t)ys[s];
                    if (cnt_e) {
                        const unsigned long long cp = cnt_e[y], cn = cnt_e[y + nh], cz = cnt_e[y + 2 * nh];
                        ce += cp + cn + cz;
                        if (!odd_aut) co += (long long)sg * ((long long)cp - (long long)cn);
                    }
                    if (w_e) {
                        const double wp = w_e[y], wn = w_e[y + nh], wz = w_e[y + 2 * nh];
                        we += (wp + wn) + wz;
                        if (!odd_aut) wo += (double)sg * (wp - wn);
                    }
                } else {
                    const size_t y = (size_t)sh * (size_t)nh + (size_t)ys[s];
                    if (cnt_e) ce += cnt_e[y];
                    if (w_e) we += w_e[y];
                }
            }
        }
    }
    if (out_ce) out_ce[x] = ce;
    if (out_co) out_co[x] = co;
    if (out_we) out_we[x] = we;
    if (out_wo) out_wo[x] = wo;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------------
void gr_4pcf(gramsci_graph *g, int parity, uint64_t *d_even_c, int64_t *d_odd_c, double *d_even_w, double *d_odd_w)
{
    cudaStream_t st = g->stream;
    const int nb = g->nb;
    int64_t nh = 1;
    for (int e = 0; e < 6; ++e) nh *= nb;
    GrTimer total(st);
    g->n_launches = 0;
    g->staged_bytes = 0;

    Q4Params p;
    p.nb = nb; p.nh = nh;
    p.parity = parity ? 1 : 0;
    p.weighted = (d_even_w || d_odd_w) ? 1 : 0;
    p.want_counts = (d_even_c || d_odd_c) ? 1 : 0;
    p.row_cap = std::max(16, (g->max_row + 15) & ~15);
    p.flush = gr_flush_budget(1ull << 27);
    p.ooc = g->ooc ? 1 : 0;
    const int channels = (d_even_c ? 1 : 0) + (d_odd_c ? 1 : 0) + (d_even_w ? 1 : 0) + (d_odd_w ? 1 : 0);
    if (channels == 0) { GR_CUDA(cudaStreamSynchronize(st)); g->t_query_ms = total.stop(); return; }
    {   // raw histograms kept per launch: counts and/or weights, three sign classes each for the parity split
        const int kinds = ((d_even_c || d_odd_c) ? 1 : 0) + ((d_even_w || d_odd_w) ? 1 : 0);
        const int64_t per_shard = nh * 8 * kinds * (p.parity ? 3 : 1);
        p.n_shards = (int)std::max<int64_t>(1, std::min<int64_t>(8, ((int64_t)96 << 20) / per_shard));
    }

    const size_t rc = (size_t)p.row_cap;
    if (rc >= 65536) GR_FAIL(GRAMSCI_ERANGE, "4pcf: longest row (%d entries) exceeds 65535", g->max_row);

    // ---- configuration LUT (once per graph): flag canonical tuples, rank them, fill ----
    // (measured slower than plain RED so far -- cfg3 13.3 vs 9.8 ms, cfg4 replica 579 vs 411 ms: the dependent LUT
    //  load sits in every lane's serial hit loop -- so it is opt-in: GRAMSCI_4PCF_LUT=1)
    const char *lut_env = getenv("GRAMSCI_4PCF_LUT");
    const bool want_lut = lut_env && lut_env[0] == '1';
    if (want_lut && nb <= 10 && g->ncfg4 == 0) {
        DevBuf<int32_t> flag, rank;
        flag.alloc((size_t)nh);
        rank.alloc((size_t)nh + 1);
        k_lut_flag<<<(unsigned)((nh + 127) / 128), 128, 0, st>>>(nb, nh, flag.p);
        gr_exclusive_scan_i32(flag.p, nh, rank.p, st);
        int32_t ncfg = 0;
        GR_CUDA(cudaMemcpyAsync(&ncfg, rank.p + nh, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        GR_CUDA(cudaStreamSynchronize(st));
        g->lut4.alloc((size_t)nh);
        g->dense4.alloc((size_t)ncfg);
        k_lut_fill<<<(unsigned)((nh + 127) / 128), 128, 0, st>>>(nb, nh, rank.p, g->lut4.p, g->dense4.p);
        GR_CUDA(cudaGetLastError());
        GR_CUDA(cudaStreamSynchronize(st));
        g->ncfg4 = ncfg;
        g->n_launches += 5;
    }

    // ---- shared memory plan: staged row, queues, (LUT) configuration histograms, (SMALL) local matrix ----
    const size_t mat_bytes = rc * rc + rc * ((rc + 31) / 32) * 4;        // D (bytes) + bit rows
    size_t smem = (p.parity ? 256 * 3 * 8 : 0) + rc * (4 + 4 + 1 + (p.weighted ? 8 : 0)) + Q4_WARPS * 64 * 4 + 64;
    smem = (smem + 15) & ~(size_t)15;
    const size_t hist_bytes = (((size_t)g->ncfg4 * (p.parity ? 2 : 1) + 3) & ~(size_t)3) * 4;
    const bool use_lut = want_lut && g->ncfg4 > 0 && smem + hist_bytes <= 120 * 1024 && (d_even_c || d_odd_c);
    p.ncfg = use_lut ? g->ncfg4 : 0;
    if (use_lut) smem += hist_bytes;
    const bool small = smem + mat_bytes <= 100 * 1024;
    if (small) smem += mat_bytes;
    if (smem > g->smem_optin)
        GR_FAIL(GRAMSCI_ERANGE, "4pcf: longest row (%d entries) does not fit in shared memory", g->max_row);
    const void *fn = small ? (use_lut ? (const void *)k_4pcf<true, true> : (const void *)k_4pcf<true, false>)
                           : (use_lut ? (const void *)k_4pcf<false, true> : (const void *)k_4pcf<false, false>);
    int occ = gr_kernel_occupancy(fn, Q4_THREADS, smem);
    occ = std::max(1, std::min(occ, 8));
    const int grid = g->sm_count * occ;
    const size_t stride = small ? 0 : ((mat_bytes + 255) & ~(size_t)255);

    DevBuf<uint8_t> scratch;
    DevBuf<unsigned int> counter;
    DevBuf<double> tab;
    DevBuf<unsigned long long> ce, co;
    DevBuf<double> we, wo;
    scratch.alloc(stride * grid + 256);
    counter.alloc(1);
    GR_CUDA(cudaMemsetAsync(counter.p, 0, sizeof(unsigned int), st));
    // LUT: counts [ncfg], weights [grid][ncfg]; raw: [n_shards][nh] each
    const size_t raw = (size_t)nh * p.n_shards * (p.parity ? 3 : 1);
    const size_t tot_c = use_lut ? (size_t)p.ncfg : raw;
    const size_t tot_w = use_lut ? (size_t)p.ncfg * grid : raw;
    if (d_even_c || (!use_lut && d_odd_c)) { ce.alloc(tot_c); GR_CUDA(cudaMemsetAsync(ce.p, 0, tot_c * 8, st)); }
    if (use_lut && d_odd_c) { co.alloc(tot_c); GR_CUDA(cudaMemsetAsync(co.p, 0, tot_c * 8, st)); }
    if (d_even_w || d_odd_w) { we.alloc(tot_w); GR_CUDA(cudaMemsetAsync(we.p, 0, tot_w * 8, st)); }
    if (use_lut && d_odd_w) { wo.alloc(tot_w); GR_CUDA(cudaMemsetAsync(wo.p, 0, tot_w * 8, st)); }
    if (p.parity) {
        // pixel-centre unit vectors (A-8): z_c = (iz + 1/2)/8 - 1, phi_c = (iphi + 1/2) pi/8
        std::vector<double> h(256 * 3);
        for (int px = 0; px < 256; ++px) {
            const int iz = px >> 4, ip = px & 15;
            const double zc = ((double)iz + 0.5) / 8.0 - 1.0;
            const double ph = ((double)ip + 0.5) * (3.14159265358979323846 / 8.0);
            const double sq = std::sqrt(1.0 - zc * zc);
            h[3 * px + 0] = sq * std::cos(ph);
            h[3 * px + 1] = sq * std::sin(ph);
            h[3 * px + 2] = zc;
        }
        tab.alloc(256 * 3);
        GR_CUDA(cudaMemcpyAsync(tab.p, h.data(), sizeof(double) * 256 * 3, cudaMemcpyHostToDevice, st));
        GR_CUDA(cudaStreamSynchronize(st));      // h goes out of scope
    }

    struct Run {
        Q4Params p; bool small, use_lut; int grid; size_t smem, stride;
        unsigned int *counter; uint8_t *scratch; const double *tab; const uint32_t *lut;
        unsigned long long *ce, *co; double *we, *wo;
    } run{p, small, use_lut, grid, smem, stride, counter.p, scratch.p, tab.p, g->lut4.p, ce.p, co.p,
          (d_even_w || d_odd_w) ? we.p : nullptr, wo.p};
    // one launch per tile: the whole graph in-core; (hub window, search windows c1 <= c2) under a memory cap
    auto tile_fn = [](gramsci_graph *gg, const GrView &v, void *user, cudaStream_t s) {
        Run &r = *(Run *)user;
        GR_CUDA(cudaMemsetAsync(r.counter, 0, sizeof(unsigned int), s));
        if (r.small && r.use_lut)
            k_4pcf<true, true><<<r.grid, Q4_THREADS, r.smem, s>>>(v, r.p, r.counter, r.scratch, r.stride, r.tab, r.lut, r.ce, r.co, r.we, r.wo);
        else if (r.small)
            k_4pcf<true, false><<<r.grid, Q4_THREADS, r.smem, s>>>(v, r.p, r.counter, r.scratch, r.stride, r.tab, nullptr, r.ce, r.co, r.we, r.wo);
        else if (r.use_lut)
            k_4pcf<false, true><<<r.grid, Q4_THREADS, r.smem, s>>>(v, r.p, r.counter, r.scratch, r.stride, r.tab, r.lut, r.ce, r.co, r.we, r.wo);
        else
            k_4pcf<false, false><<<r.grid, Q4_THREADS, r.smem, s>>>(v, r.p, r.counter, r.scratch, r.stride, r.tab, nullptr, r.ce, r.co, r.we, r.wo);
        GR_CUDA(cudaGetLastError());
        gg->n_launches += 1;
    };
    {
        GrTimer en(st);
        if (g->n > 0) gr_for_each_tile(g, p.parity != 0, false, tile_fn, &run, false, true);
        g->t_enum_ms = en.stop();
    }
    if (use_lut) {
        if (d_even_c) GR_CUDA(cudaMemsetAsync(d_even_c, 0, (size_t)nh * 8, st));
        if (d_odd_c) GR_CUDA(cudaMemsetAsync(d_odd_c, 0, (size_t)nh * 8, st));
        if (d_even_w) GR_CUDA(cudaMemsetAsync(d_even_w, 0, (size_t)nh * 8, st));
        if (d_odd_w) GR_CUDA(cudaMemsetAsync(d_odd_w, 0, (size_t)nh * 8, st));
        k_fold4_cfg<<<(p.ncfg + 127) / 128, 128, 0, st>>>(p.ncfg, grid, g->dense4.p, ce.p, co.p, d_even_w ? we.p : nullptr,
                                                         d_odd_w ? wo.p : nullptr, (unsigned long long *)d_even_c,
                                                         (long long *)d_odd_c, d_even_w, d_odd_w);
    } else {
        k_fold4<<<(unsigned)((nh + 127) / 128), 128, 0, st>>>(nb, nh, p.n_shards, p.parity, ce.p, co.p, we.p, wo.p,
                                                              (unsigned long long *)d_even_c, (long long *)d_odd_c,
                                                              d_even_w, d_odd_w);
    }
    GR_CUDA(cudaGetLastError());
    g->n_launches += 1;
    GR_CUDA(cudaStreamSynchronize(st));
    g->t_query_ms = total.stop();
}
