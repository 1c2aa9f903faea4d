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
// Hubs of one cell share the forward stencil (<= 27 cells, ordinal o); T[o_j][o_k] = offset of the segment of cell
// o_k inside a dense row of cell o_j (0xFFFF if o_k is not forward of o_j) is built once per cell and worker.
// A staged hub-row entry is (position in its cell | ordinal | bin) plus, for its role as a spoke, the address of its
// own dense row.  Lanes own tail entries k, the loop runs over spokes j, so everything about j is warp-uniform.
//   * k_3pcf_gather_warp: rows of 2..250 entries.  A WARP pulls a run of hubs of one cell (work unit, dense.cu),
//     builds its own T, and needs no CTA barrier at all; the lane's entries stay in registers per block of 32.
//   * k_3pcf_gather_cta:  longer rows.  A CTA per hub, spokes dealt to the 8 warps, tail streamed from shared memory.
//
// Histograms: per-CTA shared uint32 bins (ATOMS.POPC.INC), drained into global uint64 bins before a wedge budget
// could wrap them.  Weighted sums (WMODE 1): FIXED POINT.  w_i w_j w_k is scaled by a power of two so that
// |x| < 2^39, rounded to the nearest integer and added as three limbs (13 + 13 + 13 signed bits) with three native
// 32-bit shared atomics; 2^18 - 2^12 additions fit before a limb word could overflow, the wedge budgets are cut
// there, and the drain recombines the limb sums exactly (int64), converts once to fp64 and adds to a global fp64
// slab.  Integer addition is associative: the weighted result no longer depends on atomic order except through the
// few fp64 additions of the drains.  Rounding error per term <= 2^-40 of 2^ceil(log2 max|www|): with products
// spanning at most a factor 32 that is <= 5.8e-11 of the smallest term (BASELINE's 1e-10).
// Catalogues whose |w| span more than 32^(1/3) = 3.17 keep fp64 RED atomics into per-CTA global slabs (WMODE 2).
#include "internal.cuh"

#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <type_traits>
#include <vector>

namespace {

constexpr int G3_THREADS = 256;
constexpr int G3_WARPS = G3_THREADS / 32;
constexpr int SHORT_CAP = 250;                 // longest row of the warp kernel: C(250,2) wedges < 2^15 - 2^9
constexpr int SHORT_STAGE = 256;
constexpr int LIMB_BITS = 13;
constexpr unsigned LIMB_MASK = (1u << LIMB_BITS) - 1u;
constexpr unsigned long long LIMB_CTA_ADDS = (1ull << 18) - (1ull << 12);   // per CTA between drains
constexpr unsigned T_NONE = 0xffffu;
constexpr unsigned ROW_NONE = 0xffffffffu;

struct G3Params {
    int nb, nh, nhp;        // bins, histogram entries (nb^3; nb equilateral), words per shared plane
    int row_cap;            // CTA kernel: staged hub-row entries
    int want_counts;
    int n_slabs;            // fp64 slabs in g_w
    int n_units;
    long long u_end;         // this launch takes units [value of the counter at launch, u_end)
    long long n_tile_units;  // CTA kernel: (hub, spoke tile) units
    long long tile_bytes;    // CTA kernel: dense bytes of one spoke tile (the rows a wave of CTAs shares in L2);
                             // 0 = no tiling, a unit is a whole hub
    int ncell;
    int len_lo, len_hi;     // rows this launch takes
    unsigned long long flush;    // counts: drain before the wedge budget (per warp / per CTA) passes this
    unsigned long long wflush;   // limbs: the same
    double wscale, inv_wscale;
    int hybrid;             // WMODE 1: every other spoke goes to fp64 RED instead of the limbs (two atomic paths in parallel)
};

struct G3Tables {
    const int32_t *cell_start, *cell_of, *fwd_cell, *fwd_off, *nf, *rowlen;
    const int64_t *dbase;
    const int2 *units;
    const int32_t *ucell_off;   // CTA kernel: units of cell c are units[ucell_off[c] .. ucell_off[c+1])
    const long long *tbase;     // CTA kernel: first (hub, tile) unit of cell c
};

// ---- shared memory through 32-bit shared addresses (no generic-address arithmetic in the inner loops) ----------
__device__ __forceinline__ unsigned s_addr(const void *p)
{
    unsigned a = (unsigned)__cvta_generic_to_shared(p);
    asm volatile("mov.u32 %0, %0;" : "+r"(a));        // opaque: kept in a register instead of being re-derived at every use
    return a;
}
__device__ __forceinline__ unsigned lds_u16(unsigned a)
{
    unsigned short v;
    asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ uint2 lds_v2(unsigned a)
{
    uint2 v;
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a));
    return v;
}
__device__ __forceinline__ double lds_f64(unsigned a)
{
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a));
    return v;
}
// one byte of a dense row through the read-only path, zero-extended into a 32-bit register (opaque to the compiler, which
// otherwise re-masks the byte before every use)
// -DG3_BOUNDS=1 (debug build; compute-sanitizer is not available on the GPU pool): every gather address is checked
// against the dense rows behind the view and every histogram address against the CTA's planes; a violation traps
#ifndef G3_BOUNDS
#define G3_BOUNDS 0
#endif
#define G3_CHECK_DENSE(v, ptr) do { if (G3_BOUNDS && ((ptr) < (v).dense || (ptr) >= (v).dense + (v).dense_span)) __trap(); } while (0)
#define G3_CHECK_HIST(a, lo, bytes) do { if (G3_BOUNDS && ((a) < (lo) || (a) >= (lo) + (bytes) || ((a) & 3u))) __trap(); } while (0)
__device__ __forceinline__ unsigned ldg_u8(const uint8_t *p)
{
    unsigned v;
    asm volatile("ld.global.nc.u8 %0, [%1];" : "=r"(v) : "l"(p));
    return v;
}
__device__ __forceinline__ unsigned sexch0(unsigned a)
{
    unsigned v;
    asm volatile("atom.shared.exch.b32 %0, [%1], 0;" : "=r"(v) : "r"(a) : "memory");
    return v;
}
// predicated shared-memory reductions (no branch around the atomic): the hit test is part of the instruction
template <bool EQ>
__device__ __forceinline__ void sred_inc_hit(unsigned a, unsigned bv, unsigned ref)
{
    if (EQ) asm volatile("{\n .reg .pred q;\n setp.eq.u32 q, %1, %2;\n @q red.shared.add.u32 [%0], 1;\n}" ::"r"(a), "r"(bv), "r"(ref));
    else asm volatile("{\n .reg .pred q;\n setp.ne.u32 q, %1, 255;\n @q red.shared.add.u32 [%0], 1;\n}" ::"r"(a), "r"(bv));
}
// Branch-free form: a miss adds to a spare word behind the histogram (index nh; the drains never read it).  The
// predicated form above compiles to BSSY / BRA / ATOMS.POPC.INC / BSYNC; this one to SEL / ATOMS.POPC.INC, and the lanes
// of a warp that miss share one address, which the instruction aggregates.
#ifndef G3_DUMMY_BIN
#define G3_DUMMY_BIN 1
#endif
#ifndef G3_SPU
#define G3_SPU 2
#endif
#ifndef G3_FLAT
#define G3_FLAT 1
#endif
#ifndef G3_FLAT_U
#define G3_FLAT_U 4
#endif
#ifndef G3_SBLK
#define G3_SBLK 128          /* spokes per work item of the k-major loop */
#endif
#ifndef G3_MINB
#define G3_MINB 3
#endif
#ifndef G3_WMINB
#define G3_WMINB 1
#endif
#ifndef G3_DUMMY_WARP
#define G3_DUMMY_WARP 1
#endif
__device__ __forceinline__ void sred_inc_sel(unsigned a, unsigned bv, unsigned a_dummy)
{
    asm volatile("{\n .reg .pred q;\n .reg .u32 a2;\n setp.ne.u32 q, %1, 255;\n selp.u32 a2, %0, %2, q;\n red.shared.add.u32 [a2], 1;\n}"
                 ::"r"(a), "r"(bv), "r"(a_dummy));
}
template <bool EQ>
__device__ __forceinline__ void sred_limbs_hit(unsigned a, unsigned stride, unsigned l0, unsigned l1, unsigned l2, unsigned bv,
                                               unsigned ref)
{
    if (EQ)
        asm volatile("{\n .reg .pred q;\n .reg .u32 a1, a2;\n setp.eq.u32 q, %5, %6;\n add.u32 a1, %0, %4;\n add.u32 a2, a1, %4;\n"
                     " @q red.shared.add.u32 [%0], %1;\n @q red.shared.add.u32 [a1], %2;\n @q red.shared.add.u32 [a2], %3;\n}"
                     ::"r"(a), "r"(l0), "r"(l1), "r"(l2), "r"(stride), "r"(bv), "r"(ref));
    else
        asm volatile("{\n .reg .pred q;\n .reg .u32 a1, a2;\n setp.ne.u32 q, %5, 255;\n add.u32 a1, %0, %4;\n add.u32 a2, a1, %4;\n"
                     " @q red.shared.add.u32 [%0], %1;\n @q red.shared.add.u32 [a1], %2;\n @q red.shared.add.u32 [a2], %3;\n}"
                     ::"r"(a), "r"(l0), "r"(l1), "r"(l2), "r"(stride), "r"(bv));
}

// ---- per-cell tables -------------------------------------------------------------------------------------
// forward stencil of cell c: lane o < nf keeps its cell id, and (start label, row length, first-row offset) go to shared
__device__ __forceinline__ int load_fwd(const G3Tables &tb, int c, int nfc, int lane, int32_t *f_start, int32_t *f_rowlen,
                                        int64_t *f_dbase)
{
    int fc = -1, fs = INT_MAX, rl = 0;
    int64_t db = 0;
    if (lane < nfc) {
        fc = tb.fwd_cell[(int64_t)c * GR_STENCIL + lane];
        fs = tb.cell_start[fc];
        rl = tb.rowlen[fc];
        db = tb.dbase[fc];
    }
    f_start[lane] = fs;
    f_rowlen[lane] = rl;
    f_dbase[lane] = db;
    return fc;
}

// row o_j of T: lane o_k gets the offset of its cell's segment in a dense row of cell cj (its forward list is sorted)
__device__ __forceinline__ void build_T_row(const G3Tables &tb, int cj, int fc_lane, int lane, uint16_t *Trow)
{
    int L = -1, O = 0;
    if (lane < GR_STENCIL) {
        L = tb.fwd_cell[(int64_t)cj * GR_STENCIL + lane];
        O = tb.fwd_off[(int64_t)cj * GR_STENCIL + lane];
    }
    unsigned val = T_NONE;
#pragma unroll
    for (int t = 0; t < GR_STENCIL; ++t) {
        const int lt = __shfl_sync(0xffffffffu, L, t);
        const int ot = __shfl_sync(0xffffffffu, O, t);
        if (lt == fc_lane && lt >= 0) val = (unsigned)ot;
    }
    Trow[lane] = (uint16_t)val;
}

// One staged hub-row entry, in its two roles (ordinal o of its cell by binary search over the forward start labels):
//   as a tail entry k:  kx = { position in its cell | (2 o) << 16 ,  histogram byte offset of b_ik }
//   as a spoke j:       sp = { its own dense row (byte address >> 5, ROW_NONE if not resident) ,
//                              64 o | (histogram byte offset of b_ij) << 11 }
struct Entry { uint2 kx, sp; };
template <bool EQ>
__device__ __forceinline__ Entry make_entry(const GrView &v, int32_t k, unsigned b, unsigned nb4, unsigned nb24,
                                            const int32_t *f_start, const int32_t *f_rowlen, const int64_t *f_dbase)
{
    int o = 0;
#pragma unroll
    for (int step = 16; step > 0; step >>= 1)
        if (f_start[o + step] <= k) o += step;
    const int pk = k - f_start[o];
    Entry e;
    e.kx = make_uint2((unsigned)pk | ((unsigned)o << 17), EQ ? b * 4u : b * nb4);
    unsigned ra = ROW_NONE;
    if (k >= v.c_lo && k < v.c_hi) ra = (unsigned)((f_dbase[o] + (int64_t)pk * f_rowlen[o] - v.d0) >> 5);
    e.sp = make_uint2(ra, ((unsigned)o << 6) | ((EQ ? b * 4u : b * nb24) << 11));
    return e;
}

// fixed-point limbs of a weight product (already scaled): x = l0 + l1 2^13 + l2 2^26, l0, l1 in [0, 2^13), l2 signed
__device__ __forceinline__ void limbs_of(double pw, unsigned &l0, unsigned &l1, unsigned &l2)
{
    const long long x = __double2ll_rn(pw);
    const unsigned lo = (unsigned)x, hi = (unsigned)(x >> 32);
    l0 = lo & LIMB_MASK;
    l1 = (lo >> LIMB_BITS) & LIMB_MASK;
    l2 = __funnelshift_r(lo, hi, 2 * LIMB_BITS);
}

// ---- warp kernel: rows of len_lo..len_hi (<= SHORT_CAP) entries ---------------------------------------------
// WMODE: 0 counts only, 1 weighted by fixed-point limbs in shared memory, 2 weighted by fp64 RED atomics.
// EQ: equilateral restriction (S:8(f)-3): only wedges with b_ik == b_ij are followed, only hits with b_jk == b_ij count.
// OOC: spokes whose dense row is not resident are skipped (out-of-core tiles).
template <int WMODE, bool EQ, bool OOC>
__global__ void __launch_bounds__(G3_THREADS)
k_3pcf_gather_warp(GrView v, G3Params p, G3Tables tb, unsigned long long *__restrict__ unit_counter,
                   unsigned long long *__restrict__ g_cnt, double *__restrict__ g_w)
{
    extern __shared__ __align__(16) unsigned char smem[];
    // CTA: [hist u32 nhp (counts)] [limbs 3 x nhp (WMODE 1)], then per warp:
    //      [T u16 27x32] [f_start i32 32] [f_rowlen i32 32] [f_dbase i64 32] [sp uint2 cap] [kx uint2 cap] [aw f64 cap (weighted)]
    const bool have_cnt = (WMODE == 0) || p.want_counts;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t *hist = (uint32_t *)smem;
    const int planes = (have_cnt ? 1 : 0) + (WMODE == 1 ? 3 : 0);
    const int cap = p.row_cap;
    const size_t per_warp = GR_STENCIL * 32 * 2 + 128 + 128 + 256 + (size_t)cap * (16 + (WMODE ? 8 : 0));
    unsigned char *ws = smem + (size_t)planes * p.nhp * 4 + (size_t)warp * per_warp;
    uint16_t *T = (uint16_t *)ws;
    int32_t *f_start = (int32_t *)(ws + GR_STENCIL * 32 * 2);
    int32_t *f_rowlen = f_start + 32;
    int64_t *f_dbase = (int64_t *)(f_rowlen + 32);
    uint2 *sp = (uint2 *)(f_dbase + 32);
    uint2 *kx = sp + cap;
    double *aw = (double *)(kx + cap);
    const unsigned a_hist = s_addr(hist), a_T = s_addr(T), a_sp = s_addr(sp), a_kx = s_addr(kx), a_aw = s_addr(aw);
    const unsigned plane_b = (unsigned)p.nhp * 4;
    const unsigned a_limb = a_hist + (have_cnt ? plane_b : 0u);

    for (int t = threadIdx.x; t < planes * p.nhp; t += G3_THREADS) hist[t] = 0u;
    __syncthreads();

    const unsigned nb4 = (unsigned)p.nb * 4u, nb24 = (unsigned)p.nb * p.nb * 4u;
    double *my_w = WMODE ? g_w + (size_t)(blockIdx.x % p.n_slabs) * p.nh : nullptr;
    unsigned long long cb = 0, wb = 0;          // this warp's wedges since ITS last drain

    // any warp may drain the CTA histograms (exchange with 0 is safe against the other warps' additions; the limb
    // sums are linear, so it does not matter which drain collects which limb of a concurrent hit)
    auto warp_drain = [&]() {
        for (int t = lane; t < p.nh; t += 32) {
            if (have_cnt) {
                const unsigned c = sexch0(a_hist + 4u * t);
                if (c) atomicAdd(&g_cnt[t], (unsigned long long)c);
            }
            if (WMODE == 1) {
                const unsigned s0 = sexch0(a_limb + 4u * t), s1 = sexch0(a_limb + plane_b + 4u * t),
                               s2 = sexch0(a_limb + 2u * plane_b + 4u * t);
                if (s0 | s1 | s2) {
                    const long long x = (long long)s0 + ((long long)s1 << LIMB_BITS) + ((long long)(int32_t)s2 << (2 * LIMB_BITS));
                    atomicAdd(&my_w[t], (double)x * p.inv_wscale);
                }
            }
        }
        cb = wb = 0;
    };

    const uint8_t *dbase = v.dense;              // kept in registers (otherwise re-read from the constant bank at every gather)
    asm volatile("" : "+l"(dbase));
    int cur_cell = -1;
    for (;;) {
        int u = 0;
        if (lane == 0) u = (int)atomicAdd(unit_counter, 1ull);
        u = __shfl_sync(0xffffffffu, u, 0);
        if (u >= (int)p.u_end) break;
        const int2 un = tb.units[u];
        if (un.y <= v.h_lo || un.x >= v.h_hi) continue;
        const int c = tb.cell_of[un.x];
        if (c != cur_cell) {
            const int nfc = tb.nf[c];
            __syncwarp();
            const int fc = load_fwd(tb, c, nfc, lane, f_start, f_rowlen, f_dbase);
            for (int oj = 0; oj < nfc; ++oj) build_T_row(tb, __shfl_sync(0xffffffffu, fc, oj), fc, lane, T + oj * 32);
            cur_cell = c;
            __syncwarp();
        }
        for (int i = un.x; i < un.y; ++i) {
            const bool mine = (i >= v.h_lo && i < v.h_hi) && GR_HUB_SELECTED(v, i);
            const int64_t rb = mine ? v.ptr[i] : 0, re = mine ? v.ptr[i + 1] : 0;
            const int n = (int)(re - rb);
            if (n < p.len_lo || n > p.len_hi) continue;
            const unsigned long long wedges = (unsigned long long)n * (n - 1) / 2;
            if (cb + wedges > p.flush || (WMODE == 1 && wb + wedges > p.wflush)) warp_drain();
            cb += wedges;
            wb += wedges;
            const int32_t *gi = v.idx_h + (rb - v.e0_h);
            const uint8_t *gb = v.bin_h + (rb - v.e0_h);
            __syncwarp();                               // the previous hub's entries are no longer read
            for (int t = lane; t < n; t += 32) {
                const int32_t k = gi[t];
                const Entry e = make_entry<EQ>(v, k, gb[t], nb4, nb24, f_start, f_rowlen, f_dbase);
                kx[t] = e.kx;
                sp[t] = e.sp;
                if (WMODE) aw[t] = v.w[k];
            }
            __syncwarp();
            const double wi = WMODE ? v.w[i] * (WMODE == 1 ? p.wscale : 1.0) : 0.0;

            if (G3_FLAT && WMODE == 0) {      // (weighted launches run at the RED rate either way: measured 32.4 vs 31.6 ms)
                // FLAT: the n (n - 1) / 2 wedges (a, t), a < t, as one index space, so that no lane idles on the triangular
                // shape (rows of ~56 entries: 86 warp iterations over blocks of 32 entries, 49 over the flat space).  Spoke p
                // (n - 1 - p wedges) and spoke n - 2 - p (p + 1 wedges) share a row of exactly n slots:
                //      slot s -> p = s / n, x = s % n;   x < n - 1 - p ?  (a, t) = (p, x + p + 1)  :  (n - 2 - p, x)
                // (s / n by a multiply-high with ceil(2^32 / n): exact while s n < 2^32; n <= 250 here)
                const unsigned W = (unsigned)n * (unsigned)(n - 1) / 2u;
                const unsigned M = 0xffffffffu / (unsigned)n + 1u;
                constexpr int U = G3_FLAT_U;
                for (unsigned s0 = 0; s0 < W; s0 += 32u * U) {
                    uint2 sv[U], kv[U];
                    unsigned off[U], bv[U];
                    bool ok[U];
                    double wa[U], wk[U];
#pragma unroll
                    for (int q = 0; q < U; ++q) {
                        unsigned sl = s0 + 32u * q + lane;
                        ok[q] = sl < W;
                        sl = min(sl, W - 1u);                            // a slot beyond the end re-reads the last wedge (masked below)
                        const unsigned pp = __umulhi(sl, M), x = sl - pp * (unsigned)n;
                        const bool first = x < (unsigned)(n - 1) - pp;
                        const unsigned a = first ? pp : (unsigned)(n - 2) - pp;
                        const unsigned t = first ? x + pp + 1u : x;
                        sv[q] = lds_v2(a_sp + 8u * a);
                        kv[q] = lds_v2(a_kx + 8u * t);
                        if (WMODE) { wa[q] = lds_f64(a_aw + 8u * a); wk[q] = lds_f64(a_aw + 8u * t); }
                    }
#pragma unroll
                    for (int q = 0; q < U; ++q) off[q] = lds_u16(a_T + (kv[q].x >> 16) + (sv[q].y & 0x7c0u));
#pragma unroll
                    for (int q = 0; q < U; ++q) {
                        bool act = ok[q] && off[q] != T_NONE;
                        if (OOC) act = act && sv[q].x != ROW_NONE;
                        if (EQ) act = act && kv[q].y == (sv[q].y >> 11);
                        bv[q] = 0xffu;
                        if (act) {
                            const uint8_t *ptr = dbase + ((size_t)sv[q].x << 5) + (off[q] + (kv[q].x & 0xffffu));
                            G3_CHECK_DENSE(v, ptr);
                            bv[q] = ldg_u8(ptr);
                        }
                    }
#pragma unroll
                    for (int q = 0; q < U; ++q) {
                        const unsigned hb = sv[q].y >> 11;               // byte offset of b_ij in the histogram (EQ: 4 b_ij)
                        const unsigned ah = EQ ? a_hist + hb : a_hist + kv[q].y + hb + bv[q] * 4u;
                        if (have_cnt) {
                            if (bv[q] != 0xffu) G3_CHECK_HIST(ah, a_hist, 4u * (unsigned)p.nh);
                            if (G3_DUMMY_WARP && !EQ) sred_inc_sel(ah, bv[q], a_hist + 4u * (unsigned)p.nh);
                            else sred_inc_hit<EQ>(ah, bv[q], hb >> 2);
                        }
                        if (WMODE == 1) {
                            unsigned l0, l1, l2;
                            limbs_of((wi * wa[q]) * wk[q], l0, l1, l2);
                            sred_limbs_hit<EQ>(ah + (have_cnt ? plane_b : 0u), plane_b, l0, l1, l2, bv[q], hb >> 2);
                        } else if (WMODE == 2) {
                            if (EQ ? (bv[q] == (hb >> 2)) : (bv[q] != 0xffu)) atomicAdd(&my_w[(ah - a_hist) >> 2], (wi * wa[q]) * wk[q]);
                        }
                    }
                }
                continue;
            }
            // blocks of 32 tail entries (the lane's entry in registers); spokes a < min(n - 1, end of the block)
            for (int r0 = 0; r0 < n; r0 += 32) {
                const int t = r0 + lane;
                // a lane without an entry looks up ordinal 31, whose T column is T_NONE for every spoke
                const uint2 kxv = (t < n) ? lds_v2(a_kx + 8u * t) : make_uint2(31u << 17, 0u);
                const unsigned pk = kxv.x & 0xffffu;
                const unsigned a_Tk = a_T + (kxv.x >> 16);
                const unsigned a_hk = (EQ ? a_hist : a_hist + kxv.y);     // counts plane; limb planes follow at plane_b strides
                const double ak = (WMODE && t < n) ? lds_f64(a_aw + 8u * t) : 0.0;
                const int a_end = min(n - 1, r0 + 31);
                // U spokes at a time: all loads of a stage before the next stage.  TRI: spokes inside the lane's own block
                // (a >= r0) need the test t > a; BOUND: a partial chunk at the end of a range
                auto chunk = [&](int a0, auto Uc, auto TRIc, int lim) {
                    constexpr int U = decltype(Uc)::value;
                    constexpr bool TRI = decltype(TRIc)::value;
                    uint2 s[U];
                    unsigned off[U], bv[U];
                    double wa[U];
#pragma unroll
                    for (int q = 0; q < U; ++q) {
                        s[q] = lds_v2(a_sp + 8u * (a0 + q));
                        if (WMODE) wa[q] = lds_f64(a_aw + 8u * (a0 + q));
                    }
#pragma unroll
                    for (int q = 0; q < U; ++q) {
                        off[q] = T_NONE;
                        if (!OOC || s[q].x != ROW_NONE) off[q] = lds_u16(a_Tk + (s[q].y & 0x7c0u));
                    }
#pragma unroll
                    for (int q = 0; q < U; ++q) {
                        bool act = off[q] != T_NONE;
                        if (TRI) act = act && t > a0 + q;
                        if (EQ) act = act && kxv.y == (s[q].y >> 11);
                        bv[q] = 0xffu;
                        if (act) {
                            G3_CHECK_DENSE(v, v.dense + ((size_t)s[q].x << 5) + (off[q] + pk));
                            bv[q] = __ldg(v.dense + ((size_t)s[q].x << 5) + (off[q] + pk));
                        }
                    }
#pragma unroll
                    for (int q = 0; q < U; ++q) {
                        const unsigned hb = s[q].y >> 11;                // byte offset of b_ij in the histogram (EQ: 4 b_ij)
                        const unsigned ah = EQ ? a_hist + hb : a_hk + hb + bv[q] * 4u;
                        if (have_cnt) {
                            if (G3_DUMMY_WARP && !EQ) sred_inc_sel(ah, bv[q], a_hist + 4u * (unsigned)p.nh);
                            else sred_inc_hit<EQ>(ah, bv[q], hb >> 2);
                        }
                        if (WMODE == 1 && p.hybrid && (q & 1)) {
                            if (EQ ? (bv[q] == (hb >> 2)) : (bv[q] != 0xffu))
                                atomicAdd(&my_w[(ah - a_hist) >> 2], ((wi * wa[q]) * ak) * p.inv_wscale);
                        } else if (WMODE == 1) {
                            unsigned l0, l1, l2;
                            limbs_of((wi * wa[q]) * ak, l0, l1, l2);
                            sred_limbs_hit<EQ>(ah + (have_cnt ? plane_b : 0u), plane_b, l0, l1, l2, bv[q], hb >> 2);
                        } else if (WMODE == 2) {
                            if (EQ ? (bv[q] == (hb >> 2)) : (bv[q] != 0xffu)) atomicAdd(&my_w[(ah - a_hist) >> 2], (wi * wa[q]) * ak);
                        }
                    }
                    (void)lim;
                };
                using U4 = std::integral_constant<int, 4>;
                using U1 = std::integral_constant<int, 1>;
                const int a_mid = min(a_end, r0);                        // spokes before the block: every lane's entry is beyond them
                int a = 0;
                for (; a + 4 <= a_mid; a += 4) chunk(a, U4(), std::false_type(), 0);
                for (; a < a_mid; ++a) chunk(a, U1(), std::false_type(), 0);
                for (; a + 4 <= a_end; a += 4) chunk(a, U4(), std::true_type(), 0);
                for (; a < a_end; ++a) chunk(a, U1(), std::true_type(), 0);
            }
        }
    }
    __syncthreads();
    // final drain, cooperative
    for (int t = threadIdx.x; t < p.nh; t += G3_THREADS) {
        if (have_cnt) {
            const uint32_t c = hist[t];
            if (c) atomicAdd(&g_cnt[t], (unsigned long long)c);
        }
        if (WMODE == 1) {
            const uint32_t *limb = hist + (have_cnt ? p.nhp : 0);
            const uint32_t s0 = limb[t], s1 = limb[p.nhp + t], s2 = limb[2 * p.nhp + t];
            if (s0 | s1 | s2) {
                const long long x = (long long)s0 + ((long long)s1 << LIMB_BITS) + ((long long)(int32_t)s2 << (2 * LIMB_BITS));
                atomicAdd(&my_w[t], (double)x * p.inv_wscale);
            }
        }
    }
}

// ---- CTA kernel: rows longer than the warp kernel takes; one hub per CTA at a time -------------------------------
// Rows of thousands of entries: 4 bytes of shared memory per staged entry (position in cell | ordinal << 16 |
// bin << 21) so that several CTAs fit an SM; what a spoke needs (its dense row, its row of T, its histogram offset)
// is derived once per spoke from its entry.  T holds 32-bit offsets here (dense rows of long-row graphs pass 64 KB).
__device__ __forceinline__ unsigned lds_u32(unsigned a)
{
    unsigned v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}

__device__ __forceinline__ void build_T_row32(const G3Tables &tb, int cj, int fc_lane, int lane, uint32_t *Trow)
{
    int L = -1, O = 0;
    if (lane < GR_STENCIL) {
        L = tb.fwd_cell[(int64_t)cj * GR_STENCIL + lane];
        O = tb.fwd_off[(int64_t)cj * GR_STENCIL + lane];
    }
    unsigned val = ROW_NONE;
#pragma unroll
    for (int t = 0; t < GR_STENCIL; ++t) {
        const int lt = __shfl_sync(0xffffffffu, L, t);
        const int ot = __shfl_sync(0xffffffffu, O, t);
        if (lt == fc_lane && lt >= 0) val = (unsigned)ot;
    }
    Trow[lane] = val;
}

// KMAJOR: the LANES keep their tail entries k in registers (a chunk of 128 per warp: position, ordinal, bin and, weighted,
// w_k) and the loop runs over the SPOKES of a block of 32; what depends on the spoke alone (dense row, histogram plane,
// w_i w_j) is warp-uniform, and the table offsets T[o_j][o_k] of the lane's four entries are reloaded only when the
// spoke's cell changes (spokes are in label = cell order: every ~1/14 of a row).  Per 128 wedges that leaves ONE
// shared-memory load next to the four byte gathers and the four histogram updates, instead of eight -- the kernel runs at
// the LSU wavefront rate (profiles/r2_gather_cta_cfg5e.md), so loads are what is worth removing.  Work items (chunk,
// spoke block) are dealt to the warps through a shared-memory counter.
template <int WMODE, bool EQ, bool OOC, bool KMAJOR>
__global__ void __launch_bounds__(G3_THREADS, KMAJOR ? (WMODE == 0 ? G3_MINB : G3_WMINB) : 1)
k_3pcf_gather_cta(GrView v, G3Params p, G3Tables tb, unsigned long long *__restrict__ unit_counter,
                  unsigned long long *__restrict__ g_cnt, double *__restrict__ g_w)
{
    extern __shared__ __align__(16) unsigned char smem[];
    // [hist u32 nhp (counts)] [limbs 3 x nhp (WMODE 1)] [T u32 27x32] [f_start, f_rowlen i32 32 each] [f_dbase i64 32]
    // [aw f64 row_cap (weighted)] [kx u32 row_cap]
    const bool have_cnt = (WMODE == 0) || p.want_counts;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    uint32_t *hist = (uint32_t *)smem;
    const int planes = (have_cnt ? 1 : 0) + (WMODE == 1 ? 3 : 0);
    uint32_t *limb = hist + (have_cnt ? p.nhp : 0);
    uint32_t *T = hist + (size_t)planes * p.nhp;
    int32_t *f_start = (int32_t *)(T + GR_STENCIL * 32);
    int32_t *f_rowlen = f_start + 32;
    int64_t *f_dbase = (int64_t *)(f_rowlen + 32);
    double *aw = (double *)(f_dbase + 32);
    uint32_t *kx = (uint32_t *)(aw + (WMODE ? p.row_cap : 0));
    __shared__ int f_occ[32];
    __shared__ int s_item;                    // KMAJOR: next work item of the current unit
    __shared__ int s_cum[514];                // KMAJOR: items before chunk c
    __shared__ int s_cf[34];                  // KMAJOR: first staged row entry whose cell ordinal is >= o (entries are in cell order)
    const unsigned a_hist = s_addr(hist), a_T = s_addr(T), a_kx = s_addr(kx), a_aw = s_addr(aw);
    const unsigned plane_b = (unsigned)p.nhp * 4;
    __shared__ int s_unit;

    for (int t = threadIdx.x; t < planes * p.nhp; t += G3_THREADS) hist[t] = 0u;
    const unsigned nb4 = (unsigned)p.nb * 4u, nb24 = (unsigned)p.nb * p.nb * 4u;
    double *my_w = WMODE ? g_w + (size_t)(blockIdx.x % p.n_slabs) * p.nh : nullptr;

    auto drain = [&]() {                          // cooperative; callers synchronise before and after
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

    // Units are (hub, spoke tile) pairs in TILE-MAJOR order inside a cell: all long hubs of cell c against the spokes
    // in tile 0 (a run of <= tile_bytes of dense rows of one forward cell), then against tile 1, ...  The CTAs of a
    // wave therefore gather from the same few tens of MB of dense rows, which stay in L2 (P:153-161 cuts the edge
    // arrays into windows for the same reason one level up the hierarchy).
    __shared__ long long s_u;
    __shared__ int s_cell;
    int cur_cell = -1;
    long long cur_lo = 0, cur_hi = 0;
    int nlong = 1, nfc = 0, ubeg = 0;
    unsigned long long cb = 0, wb = 0;            // CTA-uniform: wedges since the last drain
    for (;;) {
        __syncthreads();                          // the previous unit is done: tables and staged row may be rewritten
        if (threadIdx.x == 0) {
            const long long u0 = (long long)atomicAdd(unit_counter, 1ull);
            s_u = u0;
            if (u0 < p.u_end && (u0 < cur_lo || u0 >= cur_hi)) {      // another cell: last c with tbase[c] <= u
                int lo = 0, hi = p.ncell;
                while (hi - lo > 1) {
                    const int mid = (lo + hi) >> 1;
                    if (tb.tbase[mid] <= u0) lo = mid; else hi = mid;
                }
                s_cell = lo;
            }
        }
        __syncthreads();
        const long long u = s_u;
        if (u >= p.u_end) break;
        if (u < cur_lo || u >= cur_hi) {
            const int c = s_cell;
            nfc = tb.nf[c];
            const int fc = load_fwd(tb, c, nfc, lane, f_start, f_rowlen, f_dbase);      // every warp writes the same values
            for (int oj = warp; oj < nfc; oj += G3_WARPS) build_T_row32(tb, __shfl_sync(0xffffffffu, fc, oj), fc, lane, T + oj * 32);
            // occupancy of the forward cells (tile sizes)
            if (warp == 0) f_occ[lane] = (lane < nfc) ? tb.cell_start[fc + 1] - tb.cell_start[fc] : 0;
            cur_cell = c;
            cur_lo = tb.tbase[c];
            cur_hi = tb.tbase[c + 1];
            ubeg = tb.ucell_off[c];
            nlong = tb.ucell_off[c + 1] - ubeg;
            __syncthreads();
        }
        // (tile, hub) of this unit; tile -> (forward ordinal o, label range of its spokes)
        const long long local = u - cur_lo;
        int tau = (int)(local / nlong);
        const int i = tb.units[ubeg + (int)(local % nlong)].x;
        int o = 0, l_lo = 0, l_hi = INT_MAX;
        if (p.tile_bytes) for (; o < nfc; ++o) {
            const int occ_o = f_occ[o];
            const long long bytes = (long long)occ_o * f_rowlen[o];
            const int ns = (int)max(1ll, (bytes + p.tile_bytes - 1) / p.tile_bytes);
            if (tau < ns) {
                const int per = (occ_o + ns - 1) / ns;
                l_lo = f_start[o] + tau * per;
                l_hi = min(f_start[o] + occ_o, l_lo + per);
                break;
            }
            tau -= ns;
        }
        {
            const bool mine = (i >= v.h_lo && i < v.h_hi) && GR_HUB_SELECTED(v, i);
            const int64_t rb = mine ? v.ptr[i] : 0, re = mine ? v.ptr[i + 1] : 0;
            const int n = (int)(re - rb);
            if (n < p.len_lo || n > p.len_hi || o >= nfc || l_hi <= l_lo) continue;
            if (OOC) { l_lo = max(l_lo, v.c_lo); l_hi = min(l_hi, v.c_hi); if (l_hi <= l_lo) continue; }
            const int32_t *gi = v.idx_h + (rb - v.e0_h);
            const uint8_t *gb = v.bin_h + (rb - v.e0_h);
            // spokes of this tile = row entries with label in [l_lo, l_hi): two cooperative 256-ary search rounds
            int a_lo = 0, a_hi = n;
            if (p.tile_bytes || OOC) {
                const int step = (n + G3_THREADS - 1) / G3_THREADS;
                const int seg = (int)threadIdx.x * step;
                int32_t last = INT_MAX;
                if (seg < n) last = gi[min(n, seg + step) - 1];
                const int c1 = __syncthreads_count(last < l_lo), c2 = __syncthreads_count(last < l_hi);
                int32_t e1 = INT_MAX, e2 = INT_MAX;
                if ((int)threadIdx.x < step && c1 * step + (int)threadIdx.x < n) e1 = gi[c1 * step + threadIdx.x];
                if ((int)threadIdx.x < step && c2 * step + (int)threadIdx.x < n) e2 = gi[c2 * step + threadIdx.x];
                a_lo = min(n, c1 * step + __syncthreads_count(e1 < l_lo));
                a_hi = min(n, c2 * step + __syncthreads_count(e2 < l_hi));
            }
            a_hi = min(a_hi, n - 1);
            if (a_lo >= a_hi) continue;
            const unsigned long long wedges = (unsigned long long)(a_hi - a_lo) * (unsigned long long)(n - a_lo);
            if (cb + wedges > p.flush || (WMODE == 1 && wb + wedges > p.wflush)) {
                drain();
                cb = wb = 0;
            }
            cb += wedges;
            wb += wedges;
            for (int t = a_lo + threadIdx.x; t < n; t += G3_THREADS) {
                const int32_t k = gi[t];
                int ok = 0;
#pragma unroll
                for (int step = 16; step > 0; step >>= 1)
                    if (f_start[ok + step] <= k) ok += step;
                kx[t] = (unsigned)(k - f_start[ok]) | ((unsigned)ok << 16) | ((unsigned)gb[t] << 21);
                if (WMODE) aw[t] = v.w[k];
            }
            if (KMAJOR && threadIdx.x < 34) s_cf[threadIdx.x] = n;
            __syncthreads();
            const double wi = WMODE ? v.w[i] * (WMODE == 1 ? p.wscale : 1.0) : 0.0;
            if (KMAJOR) {
                // runs of spokes of one cell: s_cf[o] = first entry with ordinal >= o (ordinals may skip empty cells)
                for (int t = a_lo + threadIdx.x; t < n; t += G3_THREADS) {
                    const int o = (int)((kx[t] >> 16) & 31u);
                    const int op = (t > a_lo) ? (int)((kx[t - 1] >> 16) & 31u) : -1;
                    for (int x = op + 1; x <= o; ++x) s_cf[x] = t;
                }
                // chunk c = tail entries [t_base + 128 c, + 128); its spokes are [a_lo, min(a_hi, last entry of the chunk))
                const int t_base = a_lo + 1;
                const int n_chunks = (n - t_base + 127) >> 7;
                if (threadIdx.x == 0) {
                    int cum = 0;
                    for (int c = 0; c < n_chunks; ++c) {
                        s_cum[c] = cum;
                        const int a_end = min(a_hi, min(n, t_base + 128 * c + 128) - 1);
                        cum += (a_end - a_lo + G3_SBLK - 1) / G3_SBLK;
                    }
                    s_cum[n_chunks] = cum;
                    s_item = 0;
                }
                __syncthreads();
                const int n_items = s_cum[n_chunks];
                int c = 0;
                for (;;) {
                    int item = 0;
                    if (lane == 0) item = atomicAdd(&s_item, 1);
                    item = __shfl_sync(0xffffffffu, item, 0);
                    if (item >= n_items) break;
                    while (s_cum[c + 1] <= item) ++c;                  // items come in ascending order
                    const int t0 = t_base + 128 * c;
                    const int a_end = min(a_hi, min(n, t0 + 128) - 1);
                    const int sa = a_lo + G3_SBLK * (item - s_cum[c]), sb = min(a_end, sa + G3_SBLK);
                    unsigned pos[4], okk[4], hk[4];
                    int tq[4];
                    double wk[4];
                    // offset of the lane's entry inside a dense row of the spoke's cell (32 bits; the rows of the cell start at
                    // cell_rows, which is warp-uniform and kept as ONE 64-bit pointer: with a 64-bit pointer per entry the
                    // compiler spent two register moves per gather on pairing them up for IMAD.WIDE); ROW_NONE for an
                    // entry whose cell is not forward of the spoke's (about half of the wedges: no load is issued for them --
                    // pointing them at a 0xFF pad byte instead, of the spoke's row or one fixed byte per cell, was measured
                    // slower: the predicate costs less in issue slots than the extra loads cost in the L1 data pipe)
                    unsigned pq[4];
                    const uint8_t *cell_rows = v.dense;
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        tq[q] = t0 + 32 * q + lane;
                        const unsigned kk = (tq[q] < n) ? lds_u32(a_kx + 4u * tq[q]) : (31u << 16);
                        pos[q] = kk & 0xffffu;
                        okk[q] = (kk >> 14) & 0x7cu;
                        hk[q] = EQ ? (kk >> 21) : (kk >> 21) * nb4;
                        pq[q] = ROW_NONE;
                        if (WMODE) wk[q] = (tq[q] < n) ? lds_f64(a_aw + 8u * tq[q]) : 0.0;
                    }
                    unsigned rl5 = 0;                                  // row length of the spoke's cell in 32-byte sectors
                    // one spoke: its four byte gathers (all issued before anything waits for them) ...
                    auto gather = [&](int a, unsigned ea, auto TRIc, unsigned (&bv)[4]) {
                        constexpr bool TRI = decltype(TRIc)::value;
                        const unsigned rs = (ea & 0xffffu) * rl5;      // row of the spoke, in sectors from its cell's first row
                        const uint8_t *rowp = cell_rows + (size_t)rs * 32u;
                        asm volatile("" : "+l"(rowp));                 // one 64-bit row pointer per spoke (not re-associated into the gathers)
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            bool act = pq[q] != ROW_NONE;
                            if (TRI) act = act && tq[q] > a;
                            if (EQ) act = act && hk[q] == (ea >> 21);
                            bv[q] = 0xffu;
                            if (act) {
                                G3_CHECK_DENSE(v, rowp + pq[q]);
                                bv[q] = ldg_u8(rowp + pq[q]);
                            }
                        }
                    };
                    // ... and its four histogram updates
                    auto update = [&](int a, unsigned ea, const unsigned (&bv)[4]) {
                        const unsigned ba = ea >> 21;
                        const unsigned a_hj = EQ ? a_hist + ba * 4u : a_hist + ba * nb24;
                        const double wia = WMODE ? wi * lds_f64(a_aw + 8u * a) : 0.0;
#pragma unroll
                        for (int q = 0; q < 4; ++q) {
                            const unsigned ah = EQ ? a_hj : a_hj + hk[q] + bv[q] * 4u;
                            if (have_cnt) {
                                if (bv[q] != 0xffu) G3_CHECK_HIST(ah, a_hist, 4u * (unsigned)p.nh);
                                if (G3_DUMMY_BIN && !EQ) sred_inc_sel(ah, bv[q], a_hist + 4u * (unsigned)p.nh);
                                else sred_inc_hit<EQ>(ah, bv[q], ba);
                            }
                            if (WMODE == 1) {
                                unsigned l0, l1, l2;
                                limbs_of(wia * wk[q], l0, l1, l2);
                                sred_limbs_hit<EQ>(ah + (have_cnt ? plane_b : 0u), plane_b, l0, l1, l2, bv[q], ba);
                            } else if (WMODE == 2) {
                                if (EQ ? (bv[q] == ba) : (bv[q] != 0xffu)) atomicAdd(&my_w[(ah - a_hist) >> 2], wia * wk[q]);
                            }
                        }
                    };
                    // spokes [a_from, a_to): cell by cell (the table offsets of the lane's entries depend on the spoke's cell
                    // only), G3_SPU spokes at a time with all their gathers issued before the first histogram update
                    auto spoke_loop = [&](int a_from, int a_to, auto TRIc) {
                        constexpr bool TRI = decltype(TRIc)::value;
                        constexpr int SPU = TRI ? 1 : G3_SPU;
                        int a = a_from;
                        while (a < a_to) {
                            const int oj = (int)((lds_u32(a_kx + 4u * a) >> 16) & 31u);
                            const int run_end = min(a_to, s_cf[oj + 1]);
                            {
                                const unsigned a_Tj = a_T + (unsigned)oj * 128u;
                                cell_rows = v.dense + (f_dbase[oj] - v.d0);
                                rl5 = (unsigned)f_rowlen[oj] >> 5;
#pragma unroll
                                for (int q = 0; q < 4; ++q) {
                                    const unsigned o2 = lds_u32(a_Tj + okk[q]);
                                    pq[q] = (o2 == ROW_NONE) ? ROW_NONE : o2 + pos[q];
                                }
                            }
                            for (; a + SPU <= run_end; a += SPU) {
                                unsigned ea[SPU], bv[SPU][4];
#pragma unroll
                                for (int u = 0; u < SPU; ++u) ea[u] = lds_u32(a_kx + 4u * (a + u));
#pragma unroll
                                for (int u = 0; u < SPU; ++u) gather(a + u, ea[u], TRIc, bv[u]);
#pragma unroll
                                for (int u = 0; u < SPU; ++u) update(a + u, ea[u], bv[u]);
                            }
                            for (; a < run_end; ++a) {
                                const unsigned ea = lds_u32(a_kx + 4u * a);
                                unsigned bv[4];
                                gather(a, ea, TRIc, bv);
                                update(a, ea, bv);
                            }
                        }
                    };
                    // spokes below every entry of the chunk need no t > a test
                    const int s_mid = min(sb, max(sa, t0));
                    spoke_loop(sa, s_mid, std::false_type());
                    spoke_loop(s_mid, sb, std::true_type());
                }
                continue;                                              // next unit (the loop head synchronises)
            }
            unsigned long long hbud = 0;          // WMODE 1: wedges of this hub since the last drain (rows beyond 724 entries)
            for (int a0 = a_lo; a0 < a_hi; a0 += G3_WARPS) {
                if (WMODE == 1 && wedges > p.wflush) {
                    hbud += (unsigned long long)G3_WARPS * (unsigned long long)(n - a0);
                    if (hbud > p.wflush) {
                        __syncthreads();
                        drain();
                        __syncthreads();
                        hbud = (unsigned long long)G3_WARPS * (unsigned long long)(n - a0);
                    }
                }
                const int a = a0 + warp;
                if (a >= a_hi) continue;
                // ---- the spoke (warp-uniform) ----
                const unsigned ea = lds_u32(a_kx + 4u * a);
                const int oj = (ea >> 16) & 31, pj = ea & 0xffffu;
                const unsigned ba = ea >> 21;
                const uint8_t *row = v.dense + (f_dbase[oj] + (int64_t)pj * f_rowlen[oj] - v.d0);
                const unsigned a_Tj = a_T + (unsigned)oj * 128u;
                const unsigned a_hj = EQ ? a_hist + ba * 4u : a_hist + ba * nb24;
                const double wia = WMODE ? wi * lds_f64(a_aw + 8u * a) : 0.0;
                auto chunk = [&](int t0, auto Uc) {
                    constexpr int U = decltype(Uc)::value;
                    unsigned kk[U], off[U], bv[U];
                    double wk[U];
#pragma unroll
                    for (int q = 0; q < U; ++q) {
                        const int t = t0 + 32 * q + lane;
                        kk[q] = (t < n) ? lds_u32(a_kx + 4u * t) : (31u << 16);
                        if (WMODE) wk[q] = (t < n) ? lds_f64(a_aw + 8u * t) : 0.0;
                    }
#pragma unroll
                    for (int q = 0; q < U; ++q) off[q] = lds_u32(a_Tj + ((kk[q] >> 14) & 0x7cu));
#pragma unroll
                    for (int q = 0; q < U; ++q) {
                        bool act = off[q] != ROW_NONE;
                        if (EQ) act = act && (kk[q] >> 21) == ba;
                        bv[q] = 0xffu;
                        if (act) {
                            G3_CHECK_DENSE(v, row + (off[q] + (kk[q] & 0xffffu)));
                            bv[q] = __ldg(row + (off[q] + (kk[q] & 0xffffu)));
                        }
                    }
#pragma unroll
                    for (int q = 0; q < U; ++q) {
                        const unsigned ah = EQ ? a_hj : a_hj + (kk[q] >> 21) * nb4 + bv[q] * 4u;
                        if (have_cnt) sred_inc_hit<EQ>(ah, bv[q], ba);
                        if (WMODE == 1 && p.hybrid && (q & 1)) {
                            if (EQ ? (bv[q] == ba) : (bv[q] != 0xffu)) atomicAdd(&my_w[(ah - a_hist) >> 2], (wia * wk[q]) * p.inv_wscale);
                        } else if (WMODE == 1) {
                            unsigned l0, l1, l2;
                            limbs_of(wia * wk[q], l0, l1, l2);
                            sred_limbs_hit<EQ>(ah + (have_cnt ? plane_b : 0u), plane_b, l0, l1, l2, bv[q], ba);
                        } else if (WMODE == 2) {
                            if (EQ ? (bv[q] == ba) : (bv[q] != 0xffu)) atomicAdd(&my_w[(ah - a_hist) >> 2], wia * wk[q]);
                        }
                    }
                };
                int t0 = a + 1;
                for (; t0 + 128 <= n; t0 += 128) chunk(t0, std::integral_constant<int, 4>());
                for (; t0 < n; t0 += 32) chunk(t0, std::integral_constant<int, 1>());
            }
        }
    }
    __syncthreads();
    drain();
}

typedef void (*gather_kernel_t)(GrView, G3Params, G3Tables, unsigned long long *, unsigned long long *, double *);

struct G3Run {
    G3Params p;
    G3Tables tb;
    unsigned long long *counter;
    unsigned long long *raw_cnt;
    double *raw_w;
    int grid, wmode, eq, cta;
    size_t smem;
    gather_kernel_t fn;
    std::vector<long long> h_ubeg, h_uend;      // out-of-core: unit range of every hub window
};

template <int WMODE, bool EQ>
gather_kernel_t gather_fn2(int cta, int ooc)
{
    if (cta == 2) return ooc ? k_3pcf_gather_cta<WMODE, EQ, true, true> : k_3pcf_gather_cta<WMODE, EQ, false, true>;
    if (cta) return ooc ? k_3pcf_gather_cta<WMODE, EQ, true, false> : k_3pcf_gather_cta<WMODE, EQ, false, false>;
    return ooc ? k_3pcf_gather_warp<WMODE, EQ, true> : k_3pcf_gather_warp<WMODE, EQ, false>;
}

gather_kernel_t gather_fn(int wmode, int eq, int cta, int ooc)
{
    if (eq) return wmode == 0 ? gather_fn2<0, true>(cta, ooc) : wmode == 1 ? gather_fn2<1, true>(cta, ooc) : gather_fn2<2, true>(cta, ooc);
    return wmode == 0 ? gather_fn2<0, false>(cta, ooc) : wmode == 1 ? gather_fn2<1, false>(cta, ooc) : gather_fn2<2, false>(cta, ooc);
}

// one tile = up to two launches: the warp kernel over the short rows, the CTA kernel over the long ones
void tile_3pcf_gather(gramsci_graph *g, const GrView &v, void *user, cudaStream_t st)
{
    G3Run *runs = (G3Run *)user;
    for (int k = 0; k < 2; ++k) {
        G3Run *r = &runs[k];
        if (r->p.n_units == 0) continue;
        // units whose hubs can lie in this tile's hub window (units are in label order; cells are label ranges)
        G3Params p = r->p;
        long long u_begin = 0;
        p.u_end = r->cta ? r->p.n_tile_units : (long long)r->p.n_units;
        if (g->ooc && !r->h_ubeg.empty()) {
            const size_t w = (size_t)v.win_h;
            u_begin = r->h_ubeg[w];
            p.u_end = r->h_uend[w];
        }
        if (p.u_end <= u_begin) continue;
        if (u_begin == 0) {
            GR_CUDA(cudaMemsetAsync(r->counter, 0, sizeof(unsigned long long), st));
        } else {                     // (a pageable host source is staged before the call returns)
            const unsigned long long ub = (unsigned long long)u_begin;
            GR_CUDA(cudaMemcpyAsync(r->counter, &ub, sizeof ub, cudaMemcpyHostToDevice, st));
        }
        r->fn<<<r->grid, G3_THREADS, r->smem, st>>>(v, p, r->tb, r->counter, r->raw_cnt, r->raw_w);
        GR_CUDA(cudaGetLastError());
        g->n_launches += 1;
    }
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

// Can this graph take the gather kernels?  (spatial labels, dense rows built or buildable, rows that fit the staging)
bool gr_gather_applicable(gramsci_graph *g, bool weighted, size_t hist_bytes, const char **why)
{
    static const char *none = "";
    if (why) *why = none;
    const size_t per_entry = 16 + (weighted ? 8 : 0);
    const size_t tables = GR_STENCIL * 32 * 2 + 128 + 128 + 256;
    const size_t stage = (size_t)std::min(SHORT_STAGE, (g->max_row + 15) & ~15);
    if (hist_bytes + (size_t)G3_WARPS * (tables + stage * per_entry) > g->smem_optin) {
        if (why) *why = "the histogram does not fit in shared memory";
        return false;
    }
    if (g->max_row > 125 && hist_bytes + tables + 2048 + (size_t)((g->max_row + 15) & ~15) * (4 + (weighted ? 8 : 0)) + 64 > g->smem_optin) {
        if (why) *why = "longest row does not fit the shared-memory staging of the gather kernel";
        return false;
    }
    if (!gr_dense_prepare(g)) { if (why) *why = g->dn.why; return false; }
    if (g->ooc && gr_tiler_slots(g, false, true) < 2) {
        if (why) *why = "device_mem_cap_bytes too small for two windows with their dense rows";
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
    const bool W = d_wsum != nullptr;
    G3Params p;
    p.nb = nb; p.nh = nh; p.nhp = (nh + 32) & ~31;      // at least one spare word behind the bins
    p.want_counts = d_counts ? 1 : 0;
    p.row_cap = std::max(16, (g->max_row + 15) & ~15);
    // weights: fp64 RED into per-CTA global slabs by default (measured faster than the limbs on every workload:
    // cfg2-D 30.9 vs 40.7 ms, uniform 1e6 points 6.8 vs 11.7 ms); GRAMSCI_WMODE=1 selects the fixed-point limbs
    // (order-independent sums) when the products span a factor <= 32
    int wmode = 0;
    p.wscale = p.inv_wscale = 1.0;
    p.hybrid = getenv("GRAMSCI_HYBRID") ? 1 : 0;
    if (W) {
        const double hi = g->w_absmax, lo = g->w_absmin;
        wmode = 2;
        if (const char *force = getenv("GRAMSCI_WMODE"))
            if (force[0] == '1' && lo > 0.0 && std::isfinite(hi) && hi / lo <= 3.1748) wmode = 1;
        if (wmode == 1) {
            int e = 0;
            std::frexp(hi * hi * hi, &e);                  // hi^3 < 2^e
            p.wscale = std::ldexp(1.0, 39 - e);            // |x| < 2^39
            p.inv_wscale = std::ldexp(1.0, e - 39);
        }
    }
    const size_t planes = (size_t)((wmode == 0 || d_counts) ? 1 : 0) + (wmode == 1 ? 3 : 0);
    const size_t hist_bytes = planes * p.nhp * 4;
    const size_t tables = GR_STENCIL * 32 * 2 + 128 + 128 + 256, tables_cta = GR_STENCIL * 32 * 4 + 128 + 128 + 256;

    G3Run runs[2];
    GrDense &d = g->dn;
    DevBuf<unsigned long long> counter;
    counter.alloc(2);
    const unsigned long long cflush = gr_flush_budget(0xE0000000ull);
    for (int k = 0; k < 2; ++k) {
        G3Run &r = runs[k];
        r.p = p;
        r.wmode = wmode; r.eq = equilateral ? 1 : 0; r.cta = k;
        r.counter = counter.p + k;
        GrUnits &un = k ? d.ub : d.ua;
        // the limb planes leave the weighted warp kernel room for 128 staged entries at two CTAs per SM
        // (dense rows of 64 KB and more do not fit the warp kernel's 16-bit table: everything goes to the CTA kernel)
        const bool wide = g->dn.max_rowlen >= 65535;
        const int short_cap = wide ? 1 : (wmode == 1) ? 125 : SHORT_CAP, short_stage = (wmode == 1) ? 128 : SHORT_STAGE;
        if (k == 0) {
            r.p.len_lo = 2; r.p.len_hi = short_cap;
            r.p.row_cap = std::max(16, std::min(short_stage, (g->max_row + 15) & ~15));
            r.smem = hist_bytes + (size_t)G3_WARPS * (tables + (size_t)r.p.row_cap * (16 + (wmode ? 8 : 0)));
            gr_dense_units(g, un, 32, r.p.len_lo, r.p.len_hi);
            // per warp: eight warps share the CTA's histograms
            r.p.flush = std::min<unsigned long long>(cflush, 1ull << 28);
            r.p.wflush = std::min<unsigned long long>(gr_flush_budget(LIMB_CTA_ADDS) / G3_WARPS, LIMB_CTA_ADDS / G3_WARPS);
        } else {
            r.p.len_lo = short_cap + 1; r.p.len_hi = INT_MAX;
            r.smem = hist_bytes + tables_cta + (size_t)p.row_cap * (4 + (wmode ? 8 : 0)) + 64;
            gr_dense_units(g, un, 1, r.p.len_lo, r.p.len_hi);
            long long tile_mb = 64;
            if (const char *e = getenv("GRAMSCI_TILE_MB")) tile_mb = std::max(1ll, atoll(e));
            // spoke tiles pay when a hub's spokes (thousands of dense rows of tens of KB) overflow L2 between two hubs
            const bool tiled = g->n_edges / std::max<int64_t>(g->n, 1) >= 512 || getenv("GRAMSCI_TILE_MB");
            if (!tiled) tile_mb = 0;
            if (un.n > 0) gr_dense_tile_units(g, un, tile_mb << 20);
            r.p.tile_bytes = tile_mb << 20;
            r.p.n_tile_units = un.n > 0 ? un.n_tile_units : 0;
            r.p.ncell = (int)g->ncell;
            r.p.flush = cflush;
            r.p.wflush = std::min<unsigned long long>(gr_flush_budget(LIMB_CTA_ADDS), LIMB_CTA_ADDS);
        }
        r.p.n_units = un.n;
        r.grid = 0;
        if (un.n == 0) continue;
        if (r.smem > g->smem_optin)
            GR_FAIL(GRAMSCI_ERANGE, "3pcf (gather): histogram or longest row (%d entries) does not fit in shared memory", g->max_row);
        // long rows: lanes keep their tail entries, the loop runs over the spokes (KMAJOR) for counts; weighted launches
        // run at the RED rate in either order and the first one is slightly ahead (cfg2-D 31.0 vs 31.8 ms);
        // GRAMSCI_CTA_KMAJOR=0 / 1 forces an order (ablation, tests); the limb path (WMODE 1) needs its mid-hub drains
        int kmajor = (wmode == 0 && g->max_row <= 65000) ? 1 : 0;
        if (const char *e = getenv("GRAMSCI_CTA_KMAJOR")) kmajor = (atoi(e) != 0 && wmode != 1 && g->max_row <= 65000) ? 1 : 0;
        r.fn = gather_fn(wmode, r.eq, (k && kmajor) ? 2 : k, g->ooc);
        if (const char *e = getenv("GRAMSCI_CARVEOUT"))      // experiment: shared-memory carve-out in percent (L1 gets the rest)
            cudaFuncSetAttribute((const void *)r.fn, cudaFuncAttributePreferredSharedMemoryCarveout, atoi(e));
        int occ = gr_kernel_occupancy((const void *)r.fn, G3_THREADS, r.smem);
        if (const char *e = getenv("GRAMSCI_OCC")) occ = std::min(occ, std::max(1, atoi(e)));
        occ = std::max(1, std::min(occ, 8));
        r.grid = g->sm_count * occ;
        r.tb.cell_start = g->cell_start.p; r.tb.cell_of = g->cell_of.p; r.tb.fwd_cell = d.fwd_cell.p; r.tb.fwd_off = d.fwd_off.p;
        r.tb.nf = d.nf.p; r.tb.rowlen = d.rowlen.p; r.tb.dbase = d.dbase.p; r.tb.units = un.units.p;
        r.tb.ucell_off = un.cell_off.p; r.tb.tbase = (const long long *)un.tbase.p;
    }
    if (g->ooc) {
        // hub window -> unit range: cells of its first and last row, then the per-cell unit offsets
        const size_t Wn = g->windows.size();
        std::vector<int32_t> c_lo(Wn), c_hi(Wn);
        for (size_t w = 0; w < Wn; ++w) {
            const GrWindow &gw = g->windows[w];
            c_lo[w] = c_hi[w] = 0;
            if (gw.row_hi > gw.row_lo) {
                GR_CUDA(cudaMemcpyAsync(&c_lo[w], g->cell_of.p + gw.row_lo, 4, cudaMemcpyDeviceToHost, st));
                GR_CUDA(cudaMemcpyAsync(&c_hi[w], g->cell_of.p + gw.row_hi - 1, 4, cudaMemcpyDeviceToHost, st));
            }
        }
        GR_CUDA(cudaStreamSynchronize(st));
        for (int k = 0; k < 2; ++k) {
            G3Run &r = runs[k];
            if (r.p.n_units == 0) continue;
            GrUnits &un = k ? d.ub : d.ua;
            std::vector<int32_t> off((size_t)g->ncell + 1);
            std::vector<int64_t> tb((size_t)g->ncell + 1);
            GR_CUDA(cudaMemcpyAsync(off.data(), un.cell_off.p, 4 * off.size(), cudaMemcpyDeviceToHost, st));
            if (k) GR_CUDA(cudaMemcpyAsync(tb.data(), un.tbase.p, 8 * tb.size(), cudaMemcpyDeviceToHost, st));
            GR_CUDA(cudaStreamSynchronize(st));
            r.h_ubeg.resize(Wn);
            r.h_uend.resize(Wn);
            for (size_t w = 0; w < Wn; ++w) {
                const bool empty = g->windows[w].row_hi <= g->windows[w].row_lo;
                r.h_ubeg[w] = empty ? 0 : (k ? tb[c_lo[w]] : off[c_lo[w]]);
                r.h_uend[w] = empty ? 0 : (k ? tb[c_hi[w] + 1] : off[c_hi[w] + 1]);
            }
        }
    }
    if (getenv("GRAMSCI_DEBUG"))
        fprintf(stderr, "[gramsci] 3pcf gather: wmode=%d eq=%d warp: units=%d smem=%zu grid=%d | cta: units=%d smem=%zu grid=%d | row=%d dense=%.3f GB (%.2f ms)\n",
                wmode, equilateral, runs[0].p.n_units, runs[0].smem, runs[0].grid, runs[1].p.n_units, runs[1].smem, runs[1].grid,
                g->max_row, d.total * 1e-9, d.t_build_ms);

    DevBuf<unsigned long long> raw_cnt;
    DevBuf<double> raw_w;
    raw_cnt.alloc((size_t)nh);
    GR_CUDA(cudaMemsetAsync(raw_cnt.p, 0, sizeof(unsigned long long) * nh, st));
    const int max_grid = std::max(1, std::max(runs[0].grid, runs[1].grid));
    const int n_slots = (int)std::max<int64_t>(1, std::min<int64_t>(max_grid, ((int64_t)256 << 20) / ((int64_t)nh * 8)));
    if (W) {
        raw_w.alloc((size_t)nh * n_slots);
        GR_CUDA(cudaMemsetAsync(raw_w.p, 0, sizeof(double) * (size_t)nh * n_slots, st));
    }
    for (int k = 0; k < 2; ++k) { runs[k].p.n_slabs = n_slots; runs[k].raw_cnt = raw_cnt.p; runs[k].raw_w = raw_w.p; }
    {
        GrTimer en(st);
        gr_for_each_tile(g, false, false, tile_3pcf_gather, runs, true);
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
