// query3g.cu -- S:8(a) A7 / A10, gather variant of the 3pCF (the default on spatially relabelled graphs).
//
// "for each hub i and each neighbor j in N(i), it checks whether a second neighbor k in N(i) with k > j is
// also in N(j)."  The membership test is the whole cost.  P:57-70 answers it by walking two sorted
// lists, P:47/P:147 by a binary search, P:149 (4pCF) by a per-hub matrix of precomputed answers.  Here the answers
// are precomputed ONCE per graph as dense cell-block rows (dense.cu): byte (j,k) = bin of edge (j,k) or 0xFF.  For a
// hub i the kernel then visits every pair j < k of N+(i) -- a "wedge" -- and gathers that byte:
//      hit  <=>  dense[row(j) + T[cell(j)][cell(k)] + pos(k)] != 0xFF ;   histogram (b_ij, b_ik, byte) += 1.
// Work = sum_i C(len N+(i), 2) wedges instead of sum_(i,j) len N+(j) streamed list elements (0.63-0.75 x), one byte
// load per wedge instead of a two-level table look-up per element, and no per-row streaming overhead.
//
// Mapping.  Work units are runs of hubs inside ONE cell (dense.cu), pulled by persistent CTAs from a global counter;
// hubs of a cell share the forward stencil, so the CTA builds one 27x27 table T (segment offset of cell o_k inside a
// row of cell o_j, -1 if o_k is not forward of o_j) per cell.  A group of G warps (G = 1 for rows up to a few
// hundred entries, 8 beyond) stages the hub row as (position in its cell | stencil ordinal, bin) words plus, per
// entry, the address of that entry's own dense row (it is a spoke for the later entries).  Lanes own tail entries
// k; the loop runs over spokes j.  Rows of up to 128 entries keep the lane's entries in registers.
//
// Histograms: per-CTA shared uint32 bins (ATOMS.POPC.INC), drained into global uint64 bins between units before a
// budget could wrap them.  Weighted sums: fixed point.  w_i w_j w_k is scaled by a power of two so that
// |x| < 2^40, rounded to the nearest integer and added as three limbs (14 + 14 + 12 signed bits) with three
// native 32-bit shared atomics; 2^17 additions fit before a limb could overflow, units are cut at that many wedges,
// and the drain recombines the limbs exactly (int64), converts once to fp64 and adds to the CTA's global slab.
// Integer addition is associative, so the weighted result no longer depends on atomic order up to the (few) fp64
// additions of the drains; the rounding error per term is <= 2^-41 of the largest product.  Graphs whose weights
// span more than a factor 3.17 in magnitude (so that products span > 32) keep fp64 RED atomics (WMODE 2).
#include "internal.cuh"

#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstdlib>

namespace {

constexpr int G3_THREADS = 256;
constexpr int G3_WARPS = G3_THREADS / 32;
constexpr int LIMB_BITS = 14;
constexpr unsigned LIMB_MASK = (1u << LIMB_BITS) - 1u;
constexpr unsigned long long LIMB_MAX_ADDS = 1ull << 17;

struct G3Params {
    int nb, nh, nhp;        // bins, histogram entries (nb^3, or nb equilateral), words per shared plane
    int row_cap;            // staged hub-row entries per group
    int want_counts;
    int n_slabs;            // fp64 slabs in g_w
    int n_units;
    unsigned long long flush;    // drain the counts before the CTA's wedge budget passes this
    unsigned long long wflush;   // the same for the fixed-point limbs
    double wscale, inv_wscale;
};

struct G3Tables {
    const int32_t *cell_start, *cell_of, *fwd_cell, *fwd_off, *nf, *rowlen;
    const int64_t *dbase;
    const int32_t *unit_lo;
    const unsigned int *unit_w;
};

template <int G>
__device__ __forceinline__ void group_sync(int group)
{
    if (G == 1) __syncwarp();
    else if (G == G3_WARPS) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(group + 1), "r"(G * 32) : "memory");
}

// WMODE: 0 counts only, 1 weighted with fixed-point limbs in shared memory, 2 weighted with fp64 RED atomics.
// EQ: equilateral restriction (S:8(f)-3): only wedges with b_ik == b_ij are followed, only hits with b_jk == b_ij count.
template <int WMODE, int G, bool EQ>
__global__ void __launch_bounds__(G3_THREADS)
k_3pcf_gather(GrView v, G3Params p, G3Tables tb, unsigned int *__restrict__ unit_counter,
              unsigned long long *__restrict__ g_cnt, double *__restrict__ g_w)
{
    constexpr int NGROUPS = G3_WARPS / G;
    extern __shared__ __align__(16) unsigned char smem[];
    // CTA: [hist u32 nhp (counts)] [limbs 3 x nhp (WMODE 1)] [T i32 27x32] [f_start, f_rowlen i32 32 each] [f_dbase i64 32]
    //      then per group: [kw uint2 row_cap] [rbase i64 row_cap] [aw f64 row_cap (weighted)]
    const bool have_cnt = (WMODE == 0) || p.want_counts;
    uint32_t *hist = (uint32_t *)smem;
    uint32_t *limb = hist + (have_cnt ? p.nhp : 0);
    int32_t *T = (int32_t *)(limb + (WMODE == 1 ? 3 * p.nhp : 0));
    int32_t *f_start = T + GR_STENCIL * 32;
    int32_t *f_rowlen = f_start + 32;
    int64_t *f_dbase = (int64_t *)(f_rowlen + 32);
    unsigned char *gs = (unsigned char *)(f_dbase + 32);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int group = warp / G, gw = warp % G;
    const size_t per_entry = 16 + (WMODE ? 8 : 0);
    gs += (size_t)group * p.row_cap * per_entry;
    uint2 *kw = (uint2 *)gs;
    int64_t *rbase = (int64_t *)(kw + p.row_cap);
    double *aw = (double *)(rbase + p.row_cap);
    __shared__ int s_unit;

    const int nb = p.nb, nb2 = nb * nb;
    double *my_w = WMODE ? g_w + (size_t)(blockIdx.x % p.n_slabs) * p.nh : nullptr;
    for (int t = threadIdx.x; t < (have_cnt ? p.nhp : 0) + (WMODE == 1 ? 3 * p.nhp : 0); t += G3_THREADS) hist[t] = 0u;

    // cooperative drain of the shared histograms (all threads; callers synchronise before and after)
    auto drain = [&]() {
        for (int t = threadIdx.x; t < p.nh; t += G3_THREADS) {
            if (have_cnt) {
                const uint32_t c = hist[t];
                if (c) { atomicAdd(&g_cnt[t], (unsigned long long)c); hist[t] = 0u; }
            }
            if (WMODE == 1) {
                const uint32_t s0 = limb[t], s1 = limb[p.nhp + t], s2 = limb[2 * p.nhp + t];
                if (s0 | s1 | s2) {
                    const long long x = (long long)s0 + ((long long)s1 << LIMB_BITS) + ((long long)(int32_t)s2 << (2 * LIMB_BITS));
                    atomicAdd(&my_w[t], (double)x * p.inv_wscale);
                    limb[t] = 0u; limb[p.nhp + t] = 0u; limb[2 * p.nhp + t] = 0u;
                }
            }
        }
    };
    // one hit: counts and weights.  key = raw histogram index; pw = w_i w_j w_k (already times the fixed-point scale, WMODE 1)
    auto record = [&](int key, double pw) {
        if (have_cnt) atomicAdd(&hist[key], 1u);
        if (WMODE == 1) {
            const long long x = __double2ll_rn(pw);
            atomicAdd(&limb[key], (uint32_t)x & LIMB_MASK);
            atomicAdd(&limb[p.nhp + key], (uint32_t)(x >> LIMB_BITS) & LIMB_MASK);
            atomicAdd(&limb[2 * p.nhp + key], (uint32_t)(int32_t)(x >> (2 * LIMB_BITS)));
        } else if (WMODE == 2) {
            atomicAdd(&my_w[key], pw);
        }
    };

    int cur_cell = -1;
    unsigned long long cbudget = 0, wbudget = 0;       // CTA-uniform: wedges since the last drain
    for (;;) {
        __syncthreads();
        if (threadIdx.x == 0) s_unit = (int)atomicAdd(unit_counter, 1u);
        __syncthreads();
        const int u = s_unit;
        if (u >= p.n_units) break;
        const int lo = tb.unit_lo[u], hi = tb.unit_lo[u + 1];
        if (hi <= v.h_lo || lo >= v.h_hi) continue;
        const unsigned long long uw = tb.unit_w[u];
        if (cbudget + uw > p.flush || (WMODE == 1 && wbudget + uw > p.wflush)) {
            drain();
            cbudget = wbudget = 0;
        }
        cbudget += uw;
        wbudget += uw;
        const int c = tb.cell_of[lo];
        const int nfc = tb.nf[c];
        if (c != cur_cell) {
            // ---- forward stencil of the cell and the table T[o_j][o_k] ----
            if (threadIdx.x < 32) {
                const int o = threadIdx.x;
                int fs = INT_MAX, rl = 0;
                int64_t db = 0;
                if (o < nfc) {
                    const int fc = tb.fwd_cell[(int64_t)c * GR_STENCIL + o];
                    fs = tb.cell_start[fc];
                    rl = tb.rowlen[fc];
                    db = tb.dbase[fc];
                }
                f_start[o] = fs; f_rowlen[o] = rl; f_dbase[o] = db;
            }
            for (int x = threadIdx.x; x < GR_STENCIL * 32; x += G3_THREADS) {
                const int oj = x >> 5, ok = x & 31;
                int val = -1;
                if (oj < nfc && ok < nfc && ok >= oj) {
                    const int cj = tb.fwd_cell[(int64_t)c * GR_STENCIL + oj], ck = tb.fwd_cell[(int64_t)c * GR_STENCIL + ok];
                    const int m = tb.nf[cj];
                    for (int t = 0; t < m; ++t) {
                        const int cc = tb.fwd_cell[(int64_t)cj * GR_STENCIL + t];
                        if (cc == ck) { val = tb.fwd_off[(int64_t)cj * GR_STENCIL + t]; break; }
                        if (cc > ck) break;
                    }
                }
                T[x] = val;
            }
            cur_cell = c;
        }
        __syncthreads();

        for (int i = lo + group; i < hi; i += NGROUPS) {
            const bool mine = (i >= v.h_lo && i < v.h_hi) && GR_HUB_SELECTED(v, i);
            const int64_t rb = mine ? v.ptr[i] : 0, re = mine ? v.ptr[i + 1] : 0;
            const int n = (int)(re - rb);
            if (n < 2) continue;
            const int32_t *gi = v.idx_h + (rb - v.e0_h);
            const uint8_t *gb = v.bin_h + (rb - v.e0_h);
            group_sync<G>(group);                       // the previous hub's entries are no longer read
            for (int t = gw * 32 + lane; t < n; t += G * 32) {
                const int32_t k = gi[t];
                const int b = gb[t];
                int o = 0;                               // ordinal of k's cell in the forward stencil: last f_start <= k
#pragma unroll
                for (int step = 16; step > 0; step >>= 1)
                    if (f_start[o + step] <= k) o += step;
                const int pk = k - f_start[o];
                kw[t] = make_uint2((unsigned)pk | ((unsigned)o << 16), EQ ? (unsigned)b : (unsigned)(b * nb));
                // k as a spoke: its own dense row, if that row is resident (out-of-core: search window)
                int64_t ra = -1;
                if (k >= v.c_lo && k < v.c_hi) ra = f_dbase[o] + (int64_t)pk * f_rowlen[o] - v.d0;
                rbase[t] = ra;
                if (WMODE) aw[t] = v.w[k];
            }
            group_sync<G>(group);
            const double wi = WMODE ? v.w[i] * (WMODE == 1 ? p.wscale : 1.0) : 0.0;

            if (G == 1 && n <= 128) {
                // ---- short rows: the lane's tail entries live in registers; loop over spokes ----
                constexpr int R = 4;
                uint2 wk[R];
                double ak[R];
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int t = r * 32 + lane;
                    wk[r] = (t < n) ? kw[t] : make_uint2(0u, 0u);
                    ak[r] = (WMODE && t < n) ? aw[t] : 0.0;
                }
                const int nr = (n + 31) >> 5;
#pragma unroll 2
                for (int a = 0; a < n - 1; ++a) {
                    const int64_t ra = rbase[a];
                    if (ra < 0) continue;
                    const uint2 wa = kw[a];
                    const int32_t *Trow = T + (wa.x >> 16) * 32;
                    const uint8_t *row = v.dense + ra;
                    const int hb = EQ ? (int)wa.y : (int)wa.y * nb;
                    const double wia = WMODE ? wi * aw[a] : 0.0;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        if (r >= nr || r * 32 + 31 <= a) continue;        // warp-uniform
                        const int t = r * 32 + lane;
                        bool act = t > a && t < n;
                        if (EQ) act = act && wk[r].y == wa.y;
                        int off = -1;
                        if (act) off = Trow[wk[r].x >> 16];
                        if (off >= 0) {
                            const unsigned bv = row[off + (int)(wk[r].x & 0xffffu)];
                            if (EQ ? (bv == wa.y) : (bv != 0xffu))
                                record(EQ ? hb : hb + (int)wk[r].y + (int)bv, WMODE ? wia * ak[r] : 0.0);
                        }
                    }
                }
            } else {
                // ---- general rows: spokes dealt to the group's warps, lanes stream the tail from shared memory ----
                unsigned long long hbudget = 0;          // G == 8, WMODE 1: wedges of this hub since the last drain
                for (int a0 = 0; a0 < n - 1; a0 += G) {
                    const int a = a0 + gw;
                    if (WMODE == 1 && G == G3_WARPS) {    // rows beyond 512 entries: drain inside the hub (group == CTA)
                        hbudget += (unsigned long long)G * (unsigned long long)(n - a0);
                        if (hbudget > p.wflush) {
                            __syncthreads();
                            drain();
                            __syncthreads();
                            hbudget = (unsigned long long)G * (unsigned long long)(n - a0);
                            cbudget = wbudget = 0;
                        }
                    }
                    if (a >= n - 1) continue;
                    const int64_t ra = rbase[a];
                    if (ra < 0) continue;
                    const uint2 wa = kw[a];
                    const int32_t *Trow = T + (wa.x >> 16) * 32;
                    const uint8_t *row = v.dense + ra;
                    const int hb = EQ ? (int)wa.y : (int)wa.y * nb;
                    const double wia = WMODE ? wi * aw[a] : 0.0;
#pragma unroll 4
                    for (int t = a + 1 + lane; t < n; t += 32) {
                        const uint2 w = kw[t];
                        if (EQ && w.y != wa.y) continue;
                        const int off = Trow[w.x >> 16];
                        if (off >= 0) {
                            const unsigned bv = row[off + (int)(w.x & 0xffffu)];
                            if (EQ ? (bv == wa.y) : (bv != 0xffu))
                                record(EQ ? hb : hb + (int)w.y + (int)bv, WMODE ? wia * aw[t] : 0.0);
                        }
                    }
                }
            }
        }
    }
    __syncthreads();
    drain();
}

struct G3Run {
    G3Params p;
    G3Tables tb;
    unsigned int *counter;
    unsigned long long *raw_cnt;
    double *raw_w;
    int grid, G, wmode, eq;
    size_t smem;
};

template <int WMODE, bool EQ>
const void *gather_fn(int G)
{
    return G == 1 ? (const void *)k_3pcf_gather<WMODE, 1, EQ> : (const void *)k_3pcf_gather<WMODE, 8, EQ>;
}

const void *gather_fn(int wmode, int G, int eq)
{
    if (eq) return wmode == 0 ? gather_fn<0, true>(G) : wmode == 1 ? gather_fn<1, true>(G) : gather_fn<2, true>(G);
    return wmode == 0 ? gather_fn<0, false>(G) : wmode == 1 ? gather_fn<1, false>(G) : gather_fn<2, false>(G);
}

template <int WMODE, bool EQ>
void launch_gather(const G3Run *r, const GrView &v, cudaStream_t st)
{
    if (r->G == 1)
        k_3pcf_gather<WMODE, 1, EQ><<<r->grid, G3_THREADS, r->smem, st>>>(v, r->p, r->tb, r->counter, r->raw_cnt, r->raw_w);
    else
        k_3pcf_gather<WMODE, 8, EQ><<<r->grid, G3_THREADS, r->smem, st>>>(v, r->p, r->tb, r->counter, r->raw_cnt, r->raw_w);
}

void tile_3pcf_gather(gramsci_graph *g, const GrView &v, void *user, cudaStream_t st)
{
    G3Run *r = (G3Run *)user;
    GR_CUDA(cudaMemsetAsync(r->counter, 0, sizeof(unsigned int), st));
    if (r->eq) {
        if (r->wmode == 0) launch_gather<0, true>(r, v, st);
        else if (r->wmode == 1) launch_gather<1, true>(r, v, st);
        else launch_gather<2, true>(r, v, st);
    } else {
        if (r->wmode == 0) launch_gather<0, false>(r, v, st);
        else if (r->wmode == 1) launch_gather<1, false>(r, v, st);
        else launch_gather<2, false>(r, v, st);
    }
    GR_CUDA(cudaGetLastError());
    g->n_launches += 1;
}

__global__ void k_copy_eq(int nb, const unsigned long long *__restrict__ cnt, const double *__restrict__ w, int n_slabs,
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

}  // namespace

// Can this graph take the gather kernel?  (spatial labels, dense rows built or buildable, rows that fit the staging)
bool gr_gather_applicable(gramsci_graph *g, bool weighted, const char **why)
{
    static const char *none = "";
    if (why) *why = none;
    if (!gr_dense_prepare(g)) { if (why) *why = g->dn.why; return false; }
    const size_t per_entry = 16 + (weighted ? 8 : 0);
    if ((size_t)std::max(16, (g->max_row + 15) & ~15) * per_entry + 64 * 1024 > g->smem_optin) {
        if (why) *why = "longest row does not fit the shared-memory staging of the gather kernel";
        return false;
    }
    return true;
}

void gr_3pcf_gather(gramsci_graph *g, uint64_t *d_counts, double *d_wsum, int equilateral)
{
    cudaStream_t st = g->stream;
    const int nb = g->nb;
    const int nh = equilateral ? nb : nb * nb * nb;
    GrTimer total(st);
    G3Run r;
    r.eq = equilateral ? 1 : 0;
    const bool W = d_wsum != nullptr;
    r.p.nb = nb; r.p.nh = nh; r.p.nhp = (nh + 31) & ~31;
    r.p.want_counts = d_counts ? 1 : 0;
    r.p.row_cap = std::max(16, (g->max_row + 15) & ~15);
    // weights: fixed-point limbs when the products span a factor <= 32 (error <= 2^-41 x 32 of a term), else fp64 RED
    r.wmode = 0;
    r.p.wscale = r.p.inv_wscale = 1.0;
    if (W) {
        const double hi = g->w_absmax, lo = g->w_absmin;
        const char *force = getenv("GRAMSCI_WMODE");
        r.wmode = (lo > 0.0 && hi / lo <= 3.1748 && std::isfinite(hi)) ? 1 : 2;
        if (force && (force[0] == '1' || force[0] == '2') && !(force[0] == '1' && !(lo > 0.0))) r.wmode = force[0] - '0';
        if (r.wmode == 1) {
            int e = 0;
            std::frexp(hi * hi * hi, &e);                  // hi^3 < 2^e
            r.p.wscale = std::ldexp(1.0, 39 - e);          // |x| < 2^39 (+ rounding)
            r.p.inv_wscale = std::ldexp(1.0, e - 39);
        }
    }
    const size_t per_entry = 16 + (r.wmode ? 8 : 0);
    const size_t planes = (size_t)((r.wmode == 0 || d_counts) ? 1 : 0) + (r.wmode == 1 ? 3 : 0);
    const size_t fixed = planes * r.p.nhp * 4 + GR_STENCIL * 32 * 4 + 32 * 4 * 2 + 32 * 8 + 64;
    // G = 1 (a warp per hub, 8 hubs per CTA) while the rows are short; the limbs need rows <= 512 there
    const size_t g1 = fixed + (size_t)G3_WARPS * r.p.row_cap * per_entry;
    r.G = (g1 <= 100 * 1024 && !(r.wmode == 1 && g->max_row > 512) && g->max_row <= 1024) ? 1 : 8;
    if (g->algo_g) r.G = g->algo_g;
    r.smem = fixed + (size_t)(G3_WARPS / r.G) * r.p.row_cap * per_entry;
    if (r.smem > g->smem_optin || planes * r.p.nhp * 4 > 160 * 1024)
        GR_FAIL(GRAMSCI_ERANGE, "3pcf (gather): histogram or longest row (%d entries) does not fit in shared memory", g->max_row);
    const void *fn = gather_fn(r.wmode, r.G, r.eq);
    int occ = gr_kernel_occupancy(fn, G3_THREADS, r.smem);
    occ = std::max(1, std::min(occ, 8));
    r.grid = g->sm_count * occ;

    r.p.flush = gr_flush_budget(0xE0000000ull);
    r.p.wflush = std::min<unsigned long long>(LIMB_MAX_ADDS, gr_flush_budget(LIMB_MAX_ADDS));
    // units: up to 4 hubs per group while rows are short, one hub per CTA when a CTA shares a hub
    const int unit_hubs = (r.G == 1) ? 32 : 2;
    gr_dense_units(g, unit_hubs, r.wmode == 1 ? r.p.wflush : 0xC0000000ull);
    r.p.n_units = g->dn.n_units;
    GrDense &d = g->dn;
    r.tb.cell_start = g->cell_start.p; r.tb.cell_of = g->cell_of.p; r.tb.fwd_cell = d.fwd_cell.p; r.tb.fwd_off = d.fwd_off.p;
    r.tb.nf = d.nf.p; r.tb.rowlen = d.rowlen.p; r.tb.dbase = d.dbase.p; r.tb.unit_lo = d.unit_lo.p; r.tb.unit_w = d.unit_w.p;

    if (getenv("GRAMSCI_DEBUG"))
        fprintf(stderr, "[gramsci] 3pcf gather: G=%d wmode=%d eq=%d smem=%zu occ=%d grid=%d units=%d row=%d dense=%.3f GB (%.2f ms)\n",
                r.G, r.wmode, r.eq, r.smem, occ, r.grid, r.p.n_units, g->max_row, d.total * 1e-9, d.t_build_ms);

    DevBuf<unsigned int> counter;
    DevBuf<unsigned long long> raw_cnt;
    DevBuf<double> raw_w;
    counter.alloc(1);
    raw_cnt.alloc((size_t)nh);
    GR_CUDA(cudaMemsetAsync(raw_cnt.p, 0, sizeof(unsigned long long) * nh, st));
    const int n_slots = (int)std::max<int64_t>(1, std::min<int64_t>(r.grid, ((int64_t)256 << 20) / ((int64_t)nh * 8)));
    r.p.n_slabs = n_slots;
    if (W) {
        raw_w.alloc((size_t)nh * n_slots);
        GR_CUDA(cudaMemsetAsync(raw_w.p, 0, sizeof(double) * (size_t)nh * n_slots, st));
    }
    r.counter = counter.p; r.raw_cnt = raw_cnt.p; r.raw_w = raw_w.p;
    {
        GrTimer en(st);
        gr_for_each_tile(g, false, false, tile_3pcf_gather, &r);
        g->t_enum_ms = en.stop();
    }
    if (equilateral) {
        k_copy_eq<<<(nb + 127) / 128, 128, 0, st>>>(nb, raw_cnt.p, W ? raw_w.p : nullptr, n_slots,
                                                   (unsigned long long *)d_counts, d_wsum);
        GR_CUDA(cudaGetLastError());
    } else {
        gr_fold3(g, nb, d_counts ? raw_cnt.p : nullptr, W ? raw_w.p : nullptr, n_slots, d_counts, d_wsum);
    }
    g->n_launches += 1;
    GR_CUDA(cudaStreamSynchronize(st));
    g->t_query_ms = total.stop();
}
