// build_graph.cu -- S:8(a) A1-A5: cell binning, neighbour count, offsets scan, fill, per-row sort.
//
// "finds, for each object i, all neighbors within r_max ... stored as a sorted adjacency
// list N(i) = {j1 < j2 < ...} (Eq. 1) ... alongside each neighbor index, the radial-bin index (an
// integer byte) and optionally a direction-pixel byte".  The paper does this on the CPU with a
// kd-tree; here it is a GPU cell list (cells of side >= r_max, 27-cell stencil), an exclusive
// prefix sum for the int64 row offsets ("all edge indexing is 64-bit") and, when labels are
// not in cell order, a segmented bitonic sort of every row.
//
// Bit-exactness against the oracle (readings A-2..A-4, A-8): the squared distance is
// (dx*dx + dy*dy) + dz*dz with every product and sum rounded separately (__dmul_rn/__dadd_rn are
// never contracted into FMAs), compared with squared bin edges computed on the host.
#include "internal.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <atomic>
#include <chrono>
#include <string>
#include <thread>

namespace {

struct BuildParams {
    int64_t n;
    int nb;
    int periodic;
    double box[3], half[3];
    double lo[3], inv_cw[3];
    int nc[3];
    int spatial;
    int want_pix;
};

struct BinEdges { double q[GR_MAXBINS + 1]; };   // squared bin edges (A-3)

// Both structs travel as __grid_constant__ kernel parameters (the parameter bank is constant memory): nothing
// about a build lives in process-global device state, so builds on different streams or host threads do not
// touch each other (include/gramsci.h, THREADS).

// ---- A1: cell ids ------------------------------------------------------------------------------
__device__ __forceinline__ int cell_coord(const BuildParams &c_bp, double x, int c)
{
    int k = (int)floor((x - c_bp.lo[c]) * c_bp.inv_cw[c]);
    k = max(0, min(k, c_bp.nc[c] - 1));
    return k;
}

__global__ void k_cell_id(const __grid_constant__ BuildParams c_bp, const double *__restrict__ pts,
                          int32_t *__restrict__ cell_of, int32_t *__restrict__ cell_cnt)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= c_bp.n) return;
    int cx = cell_coord(c_bp, pts[3 * i + 0], 0), cy = cell_coord(c_bp, pts[3 * i + 1], 1), cz = cell_coord(c_bp, pts[3 * i + 2], 2);
    int id = (cz * c_bp.nc[1] + cy) * c_bp.nc[0] + cx;
    cell_of[i] = id;
    atomicAdd(&cell_cnt[id], 1);
}

__global__ void k_scatter_cells(const int32_t *__restrict__ cell_of, int32_t *__restrict__ cell_fill,
                                int32_t *__restrict__ slot_pt, int64_t n)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int s = atomicAdd(&cell_fill[cell_of[i]], 1);
    slot_pt[s] = (int32_t)i;
}

// gather coordinates (SoA) and labels into slot order
__global__ void k_gather_slots(const double *__restrict__ pts, const int32_t *__restrict__ slot_pt,
                               double *__restrict__ sx, double *__restrict__ sy, double *__restrict__ sz,
                               int32_t *__restrict__ lab, int32_t *__restrict__ caller_of,
                               const int32_t *__restrict__ cell_of, int32_t *__restrict__ cell_of_slot, int64_t n, int spatial)
{
    int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    int32_t i = slot_pt[s];
    if (cell_of_slot) cell_of_slot[s] = cell_of[i];
    sx[s] = pts[3 * (int64_t)i + 0];
    sy[s] = pts[3 * (int64_t)i + 1];
    sz[s] = pts[3 * (int64_t)i + 2];
    lab[s] = spatial ? (int32_t)s : i;
    if (caller_of) caller_of[s] = i;
}

__global__ void k_gather_weights(const double *__restrict__ w, const int32_t *__restrict__ slot_pt,
                                 double *__restrict__ out, int64_t n, int spatial)
{
    int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n) return;
    int32_t i = slot_pt[s];
    out[spatial ? s : (int64_t)i] = w ? w[i] : 1.0;
}

// ---- bounding box of an open catalogue ------------------------------------------------------------
__global__ void k_minmax(const double *__restrict__ pts, int64_t n, double *__restrict__ part)
{
    __shared__ double s[6][256];
    double mn[3] = {INFINITY, INFINITY, INFINITY}, mx[3] = {-INFINITY, -INFINITY, -INFINITY};
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        for (int c = 0; c < 3; ++c) {
            double v = pts[3 * i + c];
            mn[c] = fmin(mn[c], v);
            mx[c] = fmax(mx[c], v);
        }
    for (int c = 0; c < 3; ++c) { s[c][threadIdx.x] = mn[c]; s[3 + c][threadIdx.x] = mx[c]; }
    __syncthreads();
    for (int st = 128; st > 0; st >>= 1) {
        if ((int)threadIdx.x < st)
            for (int c = 0; c < 3; ++c) {
                s[c][threadIdx.x] = fmin(s[c][threadIdx.x], s[c][threadIdx.x + st]);
                s[3 + c][threadIdx.x] = fmax(s[3 + c][threadIdx.x], s[3 + c][threadIdx.x + st]);
            }
        __syncthreads();
    }
    if (threadIdx.x < 6) part[blockIdx.x * 6 + threadIdx.x] = s[threadIdx.x][0];
}

// ---- A3: exclusive prefix sum, int32 counts -> int64 offsets (three-phase scan) -----------------------
constexpr int SCAN_BLOCK = 256, SCAN_ITEMS = 8, SCAN_TILE = SCAN_BLOCK * SCAN_ITEMS;

template <typename InT>
__global__ void k_scan_tile_sums(const InT *__restrict__ in, int64_t n, int64_t *__restrict__ tile_sum)
{
    __shared__ int64_t s[SCAN_BLOCK];
    int64_t base = (int64_t)blockIdx.x * SCAN_TILE;
    int64_t acc = 0;
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        int64_t i = base + (int64_t)k * SCAN_BLOCK + threadIdx.x;
        if (i < n) acc += in[i];
    }
    s[threadIdx.x] = acc;
    __syncthreads();
    for (int st = SCAN_BLOCK / 2; st > 0; st >>= 1) {
        if ((int)threadIdx.x < st) s[threadIdx.x] += s[threadIdx.x + st];
        __syncthreads();
    }
    if (threadIdx.x == 0) tile_sum[blockIdx.x] = s[0];
}

__global__ void k_scan_tile_offsets(int64_t *__restrict__ tile_sum, int64_t n_tiles)
{
    // single block: serial-in-chunks exclusive scan of the tile sums (n_tiles <= ~1e6)
    __shared__ int64_t s[1024];
    __shared__ int64_t carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int64_t base = 0; base < n_tiles; base += 1024) {
        int64_t i = base + threadIdx.x;
        int64_t v = (i < n_tiles) ? tile_sum[i] : 0;
        s[threadIdx.x] = v;
        __syncthreads();
        for (int st = 1; st < 1024; st <<= 1) {
            int64_t t = ((int)threadIdx.x >= st) ? s[threadIdx.x - st] : 0;
            __syncthreads();
            s[threadIdx.x] += t;
            __syncthreads();
        }
        if (i < n_tiles) tile_sum[i] = carry + s[threadIdx.x] - v;
        __syncthreads();
        if (threadIdx.x == 1023) carry += s[1023];
        __syncthreads();
    }
}

template <typename InT, typename OutT>
__global__ void k_scan_apply(const InT *__restrict__ in, int64_t n, const int64_t *__restrict__ tile_off,
                             OutT *__restrict__ out)
{
    // each thread owns SCAN_ITEMS consecutive items
    __shared__ int64_t s[SCAN_BLOCK];
    int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    InT v[SCAN_ITEMS];
    int64_t acc = 0;
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        v[k] = (base + k < n) ? in[base + k] : 0;
        acc += v[k];
    }
    s[threadIdx.x] = acc;
    __syncthreads();
    for (int st = 1; st < SCAN_BLOCK; st <<= 1) {
        int64_t t = ((int)threadIdx.x >= st) ? s[threadIdx.x - st] : 0;
        __syncthreads();
        s[threadIdx.x] += t;
        __syncthreads();
    }
    int64_t run = tile_off[blockIdx.x] + s[threadIdx.x] - acc;
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) out[base + k] = (OutT)run;
        run += v[k];
    }
    if (base <= n - 1 && n - 1 < base + SCAN_ITEMS) out[n] = (OutT)run;   // total
}

template <typename OutT, typename InT = int32_t>
void exclusive_scan(const InT *d_in, int64_t n, OutT *d_out, cudaStream_t st)
{
    if (n == 0) {
        GR_CUDA(cudaMemsetAsync(d_out, 0, sizeof(OutT), st));
        return;
    }
    int64_t tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
    DevBuf<int64_t> ts;
    ts.alloc((size_t)tiles);
    k_scan_tile_sums<InT><<<(unsigned)tiles, SCAN_BLOCK, 0, st>>>(d_in, n, ts.p);
    k_scan_tile_offsets<<<1, 1024, 0, st>>>(ts.p, tiles);
    k_scan_apply<InT, OutT><<<(unsigned)tiles, SCAN_BLOCK, 0, st>>>(d_in, n, ts.p, d_out);
    GR_CUDA(cudaGetLastError());
    GR_CUDA(cudaStreamSynchronize(st));   // ts freed on return
}

// ---- A5: segmented bitonic sort (key int32 ascending, optional two byte payloads) ----------------------
// One CTA per segment.  The network is the all-ascending form of the bitonic sorter (first step of
// every merge stage pairs t with its mirror image, later steps pair t with t^j), so a segment whose
// length is not a power of two is handled by treating the missing tail as +infinity: such pairs are
// already ordered and are skipped.  Segments of at most `cap` entries are sorted in shared memory,
// longer ones (not reached by the paper-shaped workloads) in place in global memory.
constexpr int SORT_SMEM_CAP = 16384;

__device__ __forceinline__ void bitonic_pair(int k, int j, bool first, int t, int &lo, int &hi)
{
    if (first) {                       // j == k/2: mirror pairing inside blocks of k
        int base = (t / j) * k, off = t % j;
        lo = base + off;
        hi = base + k - 1 - off;
    } else {
        lo = ((t & ~(j - 1)) << 1) | (t & (j - 1));
        hi = lo | j;
    }
}

template <typename OffT>
__global__ void __launch_bounds__(256)
k_segsort(const OffT *__restrict__ seg, int64_t seg_lo, int64_t seg_hi, int64_t e0, int cap,
          int32_t *__restrict__ keys, uint8_t *__restrict__ p1, uint8_t *__restrict__ p2)
{
    extern __shared__ unsigned char smem_raw[];
    int32_t *sk = (int32_t *)smem_raw;
    uint16_t *sp = (uint16_t *)(sk + cap);
    const int nt = blockDim.x;
    for (int64_t r = seg_lo + blockIdx.x; r < seg_hi; r += gridDim.x) {
        const int64_t b = (int64_t)seg[r] - e0, e = (int64_t)seg[r + 1] - e0;
        const int len = (int)(e - b);
        if (len < 2) continue;
        int P = 1;
        while (P < len) P <<= 1;
        if (len <= cap) {
            for (int t = threadIdx.x; t < len; t += nt) {
                sk[t] = keys[b + t];
                uint16_t pay = 0;
                if (p1) pay = p1[b + t];
                if (p2) pay |= (uint16_t)p2[b + t] << 8;
                sp[t] = pay;
            }
            __syncthreads();
            for (int k = 2; k <= P; k <<= 1)
                for (int j = k >> 1; j > 0; j >>= 1) {
                    for (int t = threadIdx.x; t < (P >> 1); t += nt) {
                        int lo, hi;
                        bitonic_pair(k, j, j == (k >> 1), t, lo, hi);
                        if (hi < len) {
                            int32_t a = sk[lo], c = sk[hi];
                            if (a > c) {
                                sk[lo] = c; sk[hi] = a;
                                uint16_t pa = sp[lo]; sp[lo] = sp[hi]; sp[hi] = pa;
                            }
                        }
                    }
                    __syncthreads();
                }
            for (int t = threadIdx.x; t < len; t += nt) {
                keys[b + t] = sk[t];
                if (p1) p1[b + t] = (uint8_t)(sp[t] & 0xff);
                if (p2) p2[b + t] = (uint8_t)(sp[t] >> 8);
            }
            __syncthreads();
        } else {
            for (int k = 2; k <= P; k <<= 1)
                for (int j = k >> 1; j > 0; j >>= 1) {
                    for (int t = threadIdx.x; t < (P >> 1); t += nt) {
                        int lo, hi;
                        bitonic_pair(k, j, j == (k >> 1), t, lo, hi);
                        if (hi < len) {
                            int32_t a = keys[b + lo], c = keys[b + hi];
                            if (a > c) {
                                keys[b + lo] = c; keys[b + hi] = a;
                                if (p1) { uint8_t x = p1[b + lo]; p1[b + lo] = p1[b + hi]; p1[b + hi] = x; }
                                if (p2) { uint8_t x = p2[b + lo]; p2[b + lo] = p2[b + hi]; p2[b + hi] = x; }
                            }
                        }
                    }
                    __syncthreads();
                }
        }
    }
}

// ---- A2 / A4: neighbour count and fill ------------------------------------------------------------------
__device__ __forceinline__ int bin_of(const BuildParams &c_bp, const BinEdges &eq, double d2)
{   // b = #{k in [1,nb): q_k <= d2} (A-3); q is non-decreasing so this is an upper bound search
    int lo = 1, hi = c_bp.nb;            // answer = (first k in [1,nb) with q_k > d2) - 1
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if (eq.q[mid] <= d2) lo = mid + 1; else hi = mid;
    }
    return lo - 1;
}

__device__ __forceinline__ int pixel_of(double dx, double dy, double dz, double d2)
{   // A-8: 16 equal-area z bands x 16 phi sectors
    const double r = __dsqrt_rn(d2);
    int iz = 0;
#pragma unroll
    for (int k = 1; k < 16; ++k) iz += (dz >= __dmul_rn((double)k / 8.0 - 1.0, r)) ? 1 : 0;
    const double ax = fabs(dx), ay = fabs(dy);
    int s = 0;
    s += (ay >= __dmul_rn(ax, 0.41421356237309503)) ? 1 : 0;   // tan 22.5 deg
    s += (ay >= __dmul_rn(ax, 1.0)) ? 1 : 0;                   // tan 45 deg
    s += (ay >= __dmul_rn(ax, 2.414213562373095)) ? 1 : 0;     // tan 67.5 deg
    int iphi;
    if (dx >= 0.0) iphi = (dy >= 0.0) ? s : 15 - s;
    else           iphi = (dy >= 0.0) ? 7 - s : 8 + s;
    return 16 * iz + iphi;
}

// One warp per slot s (a point in cell order).  Lanes 0..26 own the stencil cells; duplicates (periodic
// grids with fewer than 3 cells on an axis) are removed with match_any, and the cells are visited in
// ascending id so that in spatial mode (label == slot) the row is emitted already sorted (Eq. 1).
template <bool FILL>
__global__ void __launch_bounds__(256)
k_neighbours(const __grid_constant__ BuildParams c_bp, const __grid_constant__ BinEdges eq,
             const double *__restrict__ sx, const double *__restrict__ sy, const double *__restrict__ sz,
             const int32_t *__restrict__ lab, const int32_t *__restrict__ cell_start,
             int64_t slot_lo, int64_t slot_hi, int32_t row_lo, int32_t row_hi,
             int32_t *__restrict__ deg, const int64_t *__restrict__ ptr, int64_t e0,
             int32_t *__restrict__ idx, uint8_t *__restrict__ bin, uint8_t *__restrict__ pix)
{
    const int lane = threadIdx.x & 31;
    const int64_t s = slot_lo + ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / 32;
    if (s >= slot_hi) return;
    const int32_t li = lab[s];
    if (li < row_lo || li >= row_hi) return;
    const double xi = sx[s], yi = sy[s], zi = sz[s];
    const int cx = cell_coord(c_bp, xi, 0), cy = cell_coord(c_bp, yi, 1), cz = cell_coord(c_bp, zi, 2);
    const int own = (cz * c_bp.nc[1] + cy) * c_bp.nc[0] + cx;

    // stencil cell of this lane
    int id = -1;
    if (lane < 27) {
        int o[3] = {cx + (lane % 3) - 1, cy + ((lane / 3) % 3) - 1, cz + (lane / 9) - 1};
        bool ok = true;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            if (c_bp.periodic) o[c] = (o[c] + c_bp.nc[c]) % c_bp.nc[c];
            else if (o[c] < 0 || o[c] >= c_bp.nc[c]) ok = false;
        }
        if (ok) id = (o[2] * c_bp.nc[1] + o[1]) * c_bp.nc[0] + o[0];
        if (c_bp.spatial && id < own) id = -1;          // label > own label  =>  cell >= own cell
    }
    const unsigned same = __match_any_sync(0xffffffffu, id);
    const bool keep = (id >= 0) && ((__ffs(same) - 1) == lane);
    int rank = 0;
    for (int t = 0; t < 27; ++t) {
        int v = __shfl_sync(0xffffffffu, id, t);
        bool kt = __shfl_sync(0xffffffffu, (int)keep, t);
        rank += (kt && v < id) ? 1 : 0;
    }
    const int ncell = __popc(__ballot_sync(0xffffffffu, keep));
    int cs = 0, ce = 0;
    if (keep) { cs = cell_start[id]; ce = cell_start[id + 1]; }

    int64_t out = 0;
    if (FILL) {
        out = ptr[li] - e0;
        if (ptr[li + 1] == ptr[li]) return;             // empty row (also: a row outside slab + halo of a slab graph)
    }
    int count = 0;
    // The (cell, 32-candidate chunk) pairs are walked as one sequence with the NEXT chunk's label and
    // coordinates already in flight while the current chunk's distances are evaluated (a cell holds about one
    // chunk in the 1e6-point configurations, so without this every chunk pays the full load latency).
    int r = -1, t0 = -32, e = -32;             // last consumed cell rank, chunk start, range end (warp-uniform)
    // Cells adjacent in x have adjacent slot ranges, so a partial chunk at the end of one cell is topped up from
    // the next cell when that one starts where this one ends (a cell holds ~28 points in the 1e6-point
    // configurations: 18 chunks per point without this, ~13 with).
    auto advance = [&]() -> bool {             // move to the next non-empty chunk; false when the stencil is done
        t0 += 32;
        for (;;) {
            if (t0 + 32 <= e) return true;                     // a full chunk is left in the current range
            if (r + 1 >= ncell) return t0 < e;
            const int src = __ffs(__ballot_sync(0xffffffffu, keep && rank == r + 1)) - 1;
            int b2 = __shfl_sync(0xffffffffu, cs, src);
            const int e2 = __shfl_sync(0xffffffffu, ce, src);
            const int cid = __shfl_sync(0xffffffffu, id, src);
            if (c_bp.spatial && cid == own) b2 = (int)s + 1;
            if (t0 >= e) { ++r; t0 = b2; e = e2; continue; }    // range exhausted: jump to the next cell
            if (b2 == e) { ++r; e = e2; continue; }             // next cell is contiguous: extend the range
            return true;                                       // partial chunk, next cell elsewhere
        }
    };
    // loop invariants out of constant memory (the compiler re-issued ~13 constant loads per chunk)
    const bool per = c_bp.periodic != 0;
    const double hx = per ? c_bp.half[0] : INFINITY, hy = per ? c_bp.half[1] : INFINITY, hz = per ? c_bp.half[2] : INFINITY;
    const double bx = c_bp.box[0], by = c_bp.box[1], bz = c_bp.box[2];
    const double q_lo = eq.q[0], q_hi = eq.q[c_bp.nb];
    // separation component a -> b, minimum image when periodic (A-4); half = +inf switches the wrap off
    auto sep = [](double a, double b, double half, double box) -> double {
        double d = __dsub_rn(b, a);
        if (d > half) d = __dsub_rn(d, box);
        else if (d < -half) d = __dadd_rn(d, box);
        return d;
    };
    bool have = advance();
    int n_lj = 0;
    double n_x = 0.0, n_y = 0.0, n_z = 0.0;
    bool n_ok = false;
    if (have) {
        const int t = t0 + lane;
        n_ok = t < e;
        if (n_ok) { n_lj = lab[t]; n_x = sx[t]; n_y = sy[t]; n_z = sz[t]; }
    }
    while (have) {
        const bool ok = n_ok;
        const int lj = n_lj;
        const double xj = n_x, yj = n_y, zj = n_z;
        have = advance();
        n_ok = false;
        if (have) {
            const int t = t0 + lane;
            n_ok = t < e;
            if (n_ok) { n_lj = lab[t]; n_x = sx[t]; n_y = sy[t]; n_z = sz[t]; }
        }
        bool edge = false;
        int bb = 0, pp = 0;
        if (ok && lj > li) {
            // direction lower label -> higher label (hub -> spoke)
            const double dx = sep(xi, xj, hx, bx), dy = sep(yi, yj, hy, by), dz = sep(zi, zj, hz, bz);
            const double d2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
            edge = (d2 >= q_lo) && (d2 < q_hi);                // r_min <= r < r_max (A-2)
            if (FILL && edge) {
                bb = bin_of(c_bp, eq, d2);
                if (c_bp.want_pix) pp = pixel_of(dx, dy, dz, d2);
            }
        }
        const unsigned m = __ballot_sync(0xffffffffu, edge);
        if (FILL) {
            if (edge) {
                const int64_t o = out + __popc(m & ((1u << lane) - 1u));
                idx[o] = lj;
                bin[o] = (uint8_t)bb;
                if (pix) pix[o] = (uint8_t)pp;
            }
            out += __popc(m);
        } else {
            count += __popc(m);
        }
    }
    if (!FILL && lane == 0) deg[li] = count;
}

// ---- slab + halo partition (S:8(e)): work estimate per cell, rows of cells outside slab + halo emptied ----
__global__ void k_cell_cost(int64_t ncell, const int32_t *__restrict__ cell_start, const int32_t *__restrict__ deg,
                            double *__restrict__ cost)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    double s = 0.0;
    for (int i = cell_start[c]; i < cell_start[c + 1]; ++i) s += (double)deg[i] * (double)deg[i];
    cost[c] = s;
}

__global__ void k_mask_deg(int64_t n, const int32_t *__restrict__ cell_of, const uint8_t *__restrict__ keep, int32_t *__restrict__ deg)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n && !keep[cell_of[i]]) deg[i] = 0;
}

// ---- export in caller labels (spatial mode): re-orient every edge to lower caller label ---------------
__global__ void k_export_count(const int64_t *__restrict__ ptr, const int32_t *__restrict__ idx,
                               const int32_t *__restrict__ caller_of, int64_t n, int32_t *__restrict__ deg)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int ci = caller_of[i];
    for (int64_t e = ptr[i]; e < ptr[i + 1]; ++e) {
        int cj = caller_of[idx[e]];
        atomicAdd(&deg[min(ci, cj)], 1);
    }
}

__global__ void k_export_fill(const int64_t *__restrict__ ptr, const int32_t *__restrict__ idx,
                              const uint8_t *__restrict__ bin, const int32_t *__restrict__ caller_of, int64_t n,
                              const int64_t *__restrict__ optr, int32_t *__restrict__ fill,
                              int32_t *__restrict__ oidx, uint8_t *__restrict__ obin)
{
    int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int ci = caller_of[i];
    for (int64_t e = ptr[i]; e < ptr[i + 1]; ++e) {
        int cj = caller_of[idx[e]];
        int lo = min(ci, cj), hi = max(ci, cj);
        int64_t o = optr[lo] + atomicAdd(&fill[lo], 1);
        oidx[o] = hi;
        obin[o] = bin[e];
    }
}

// ---- row statistics for the slot-table 3pCF kernel: one warp per row -------------------------------------
// The kernel keys its table by d(k) = k - first, after cutting the LARGEST gap between consecutive entries
// out of the row (rows of hubs next to a periodic face reach labels at the other end of the label range):
// entries before the gap keep d = k - first, entries from `brk` (first entry after the gap) on get
// d = k - brk + off(s), off(s) = two pages past the page of the last entry before the gap (one guard page).
// For every page shift s this emits   out[2*(s-GR_S_MIN)]   = max over rows of the page-table length
//                                     out[2*(s-GR_S_MIN)+1] = max over rows of the number of touched pages.
__global__ void __launch_bounds__(256)
k_row_stats(const int64_t *__restrict__ ptr, const int32_t *__restrict__ idx, int64_t e0, int32_t row_lo,
            int32_t row_hi, int32_t *__restrict__ out)
{
    __shared__ int s_max[2 * (GR_S_MAX - GR_S_MIN + 1)];
    if (threadIdx.x < 2 * (GR_S_MAX - GR_S_MIN + 1)) s_max[threadIdx.x] = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int64_t r = row_lo + ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / 32;
    int64_t b = 0, e = 0;
    if (r < row_hi) { b = ptr[r] - e0; e = ptr[r + 1] - e0; }
    if (e - b >= 2) {
    const int32_t first = idx[b], last = idx[e - 1];
    // pass 1: first largest gap
    int best_gap = 0;
    int64_t best_t = b + 1;
    int32_t carry = first;
    for (int64_t t0 = b; t0 < e; t0 += 32) {
        const int64_t t = t0 + lane;
        const int32_t k = (t < e) ? idx[t] : 0;
        int32_t prev = __shfl_up_sync(0xffffffffu, k, 1);
        if (lane == 0) prev = carry;
        const int gap = (t < e) ? k - prev : 0;
        const int m = __reduce_max_sync(0xffffffffu, gap);
        if (m > best_gap) {
            best_gap = m;
            best_t = t0 + __ffs(__ballot_sync(0xffffffffu, gap == m)) - 1;
        }
        carry = __shfl_sync(0xffffffffu, k, 31);
    }
    const int32_t lowmax = idx[best_t - 1], brk = idx[best_t];
    // pass 2: touched pages per shift
    int cnt[GR_S_MAX - GR_S_MIN + 1];
#pragma unroll
    for (int s = 0; s <= GR_S_MAX - GR_S_MIN; ++s) cnt[s] = 0;
    int32_t cprev = -1;      // previous entry (label), -1 = none
    for (int64_t t0 = b; t0 < e; t0 += 32) {
        const int64_t t = t0 + lane;
        const bool ok = t < e;
        const int32_t k = ok ? idx[t] : 0;
        int32_t prev = __shfl_up_sync(0xffffffffu, k, 1);
        if (lane == 0) prev = cprev;
#pragma unroll
        for (int s = 0; s <= GR_S_MAX - GR_S_MIN; ++s) {
            const int sh = s + GR_S_MIN;
            // page identity: (side of the gap, page inside that side)
            const int pk = (k >= brk) ? (((k - brk) >> sh) | 0x40000000) : ((k - first) >> sh);
            const int pp = (prev < 0) ? -1 : ((prev >= brk) ? (((prev - brk) >> sh) | 0x40000000) : ((prev - first) >> sh));
            cnt[s] += __popc(__ballot_sync(0xffffffffu, ok && pk != pp));
        }
        cprev = __shfl_sync(0xffffffffu, k, 31);
    }
    if (lane == 0) {
#pragma unroll
        for (int s = 0; s <= GR_S_MAX - GR_S_MIN; ++s) {
            const int sh = s + GR_S_MIN;
            const int ptl = ((lowmax - first) >> sh) + 2 + ((last - brk) >> sh) + 1;   // low pages, guard, high pages
            atomicMax(&s_max[2 * s], ptl);
            atomicMax(&s_max[2 * s + 1], cnt[s]);
        }
    }
    }
    __syncthreads();      // one global atomic per block and value, not per row (same-address atomics serialise in L2)
    if (threadIdx.x < 2 * (GR_S_MAX - GR_S_MIN + 1) && s_max[threadIdx.x] > 0) atomicMax(&out[threadIdx.x], s_max[threadIdx.x]);
}

// which search windows the edges [lo,hi) of a hub window reach: bit c of out[0..] is set iff some neighbour
// label lies in window c (row boundaries wlo[0..W], W <= 1024); tiler.cu visits only those tiles
__global__ void k_need_mask(const int32_t *__restrict__ idx, int64_t lo, int64_t hi, const int32_t *__restrict__ wlo,
                            int W, unsigned int *__restrict__ out)
{
    extern __shared__ unsigned int s_mask[];
    for (int t = threadIdx.x; t < (W + 31) / 32; t += blockDim.x) s_mask[t] = 0;
    __syncthreads();
    for (int64_t e = lo + (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < hi; e += (int64_t)gridDim.x * blockDim.x) {
        const int32_t k = idx[e];
        int a = 0, b = W;                    // largest c with wlo[c] <= k
        while (b - a > 1) {
            const int mid = (a + b) >> 1;
            if (wlo[mid] <= k) a = mid; else b = mid;
        }
        const unsigned bit = 1u << (a & 31);
        if (!(s_mask[a >> 5] & bit)) atomicOr(&s_mask[a >> 5], bit);
    }
    __syncthreads();
    for (int t = threadIdx.x; t < (W + 31) / 32; t += blockDim.x)
        if (s_mask[t]) atomicOr(&out[t], s_mask[t]);
}

inline unsigned blocks_for(int64_t n, int per) { return (unsigned)std::max<int64_t>(1, (n + per - 1) / per); }

// min and max of |w| (fp64 atomics on two words; doubles >= 0 order like their bit patterns)
__global__ void k_abs_minmax(const double *__restrict__ w, int64_t n, double *__restrict__ out)
{
    double mn = INFINITY, mx = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
        const double a = fabs(w[i]);
        mn = fmin(mn, a);
        mx = fmax(mx, a);
    }
    for (int o = 16; o > 0; o >>= 1) {
        mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, o));
        mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMin((unsigned long long *)&out[0], (unsigned long long)__double_as_longlong(mn));
        atomicMax((unsigned long long *)&out[1], (unsigned long long)__double_as_longlong(mx));
    }
}

template <typename OffT>
__global__ void k_seg_max(const OffT *__restrict__ seg, int64_t n, int32_t *__restrict__ out)
{
    int m = 0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        m = max(m, (int)(seg[i + 1] - seg[i]));
    for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(out, m);
}

template <typename OffT>
int seg_max(const OffT *seg, int64_t n, cudaStream_t st)
{
    DevBuf<int32_t> mx;
    mx.alloc(1);
    int h = 0;
    GR_CUDA(cudaMemsetAsync(mx.p, 0, sizeof(int32_t), st));
    if (n > 0) k_seg_max<OffT><<<296, 256, 0, st>>>(seg, n, mx.p);
    GR_CUDA(cudaMemcpyAsync(&h, mx.p, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    GR_CUDA(cudaStreamSynchronize(st));
    return h;
}

// sort every segment [seg[r], seg[r+1]) for r in [seg_lo,seg_hi); max_len = longest segment
template <typename OffT>
void segsort(const OffT *seg, int64_t seg_lo, int64_t seg_hi, int64_t e0, int max_len, int32_t *keys, uint8_t *p1,
             uint8_t *p2, cudaStream_t st)
{
    if (seg_hi <= seg_lo || max_len < 2) return;
    int cap = 64;
    while (cap < max_len && cap < SORT_SMEM_CAP) cap <<= 1;
    size_t smem = (size_t)cap * (sizeof(int32_t) + sizeof(uint16_t));
    GR_CUDA(cudaFuncSetAttribute(k_segsort<OffT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)((size_t)SORT_SMEM_CAP * 6)));
    int threads = std::max(32, std::min(256, cap / 2));
    unsigned grid = (unsigned)std::min<int64_t>(seg_hi - seg_lo, 148 * 32);
    k_segsort<OffT><<<grid, threads, smem, st>>>(seg, seg_lo, seg_hi, e0, cap, keys, p1, p2);
    GR_CUDA(cudaGetLastError());
}

}  // namespace

void gr_exclusive_scan_i32(const int32_t *d_in, int64_t n, int32_t *d_out, cudaStream_t st)
{
    exclusive_scan<int32_t>(d_in, n, d_out, st);
}

template <typename InT, typename OutT>
void gr_exclusive_scan(const InT *d_in, int64_t n, OutT *d_out, cudaStream_t st)
{
    exclusive_scan<OutT, InT>(d_in, n, d_out, st);
}
template void gr_exclusive_scan<int32_t, int32_t>(const int32_t *, int64_t, int32_t *, cudaStream_t);
template void gr_exclusive_scan<int32_t, int64_t>(const int32_t *, int64_t, int64_t *, cudaStream_t);
template void gr_exclusive_scan<int64_t, int64_t>(const int64_t *, int64_t, int64_t *, cudaStream_t);

// ---------------------------------------------------------------------------------------------------
void gr_build(gramsci_graph *g, const double *d_points, const double *d_weights, int n_windows_forced)
{
    const int64_t n = g->n;
    cudaStream_t st = g->stream;
    GrTimer timer(st);
    double launches = 0;

    // --- cell grid (cells of side >= r_max; A1) ---
    double lo[3] = {0, 0, 0}, hi[3] = {1, 1, 1};
    if (g->periodic) {
        for (int c = 0; c < 3; ++c) { lo[c] = 0.0; hi[c] = g->box[c]; }
    } else if (n > 0) {
        const int nbk = 256;
        DevBuf<double> part;
        part.alloc(nbk * 6);
        k_minmax<<<nbk, 256, 0, st>>>(d_points, n, part.p);
        launches += 1;
        std::vector<double> h(nbk * 6);
        GR_CUDA(cudaMemcpyAsync(h.data(), part.p, sizeof(double) * nbk * 6, cudaMemcpyDeviceToHost, st));
        GR_CUDA(cudaStreamSynchronize(st));
        for (int c = 0; c < 3; ++c) { lo[c] = INFINITY; hi[c] = -INFINITY; }
        for (int b = 0; b < nbk; ++b)
            for (int c = 0; c < 3; ++c) {
                lo[c] = std::min(lo[c], h[b * 6 + c]);
                hi[c] = std::max(hi[c], h[b * 6 + 3 + c]);
            }
        for (int c = 0; c < 3; ++c)
            if (!std::isfinite(lo[c]) || !std::isfinite(hi[c])) GR_FAIL(GRAMSCI_EINVAL, "non-finite coordinate");
    }
    BuildParams bp;
    bp.n = n; bp.nb = g->nb; bp.periodic = g->periodic; bp.spatial = g->spatial; bp.want_pix = g->has_pix;
    int64_t ncell = 1;
    // keep the cell count modest: at most ~2 cells per point and 2^22 overall
    const double cell_budget = std::min<double>(4194304.0, std::max<double>(64.0, 2.0 * (double)n));
    double side = g->r_max * 1.000001;
    for (int iter = 0; iter < 64; ++iter) {
        ncell = 1;
        for (int c = 0; c < 3; ++c) {
            double ext = hi[c] - lo[c];
            int k = (ext > 0) ? (int)std::floor(ext / side) : 1;
            k = std::max(1, std::min(k, 1024));
            g->nc[c] = k;
            ncell *= k;
        }
        if ((double)ncell <= cell_budget) break;
        side *= 1.26;
    }
    for (int c = 0; c < 3; ++c) {
        double ext = hi[c] - lo[c];
        g->lo[c] = lo[c];
        g->cw[c] = (ext > 0) ? ext / g->nc[c] : 1.0;
        bp.box[c] = g->box[c]; bp.half[c] = 0.5 * g->box[c];
        bp.lo[c] = g->lo[c]; bp.inv_cw[c] = 1.0 / g->cw[c]; bp.nc[c] = g->nc[c];
        // guard: rounding in (x-lo)*inv_cw must not push two points closer than r_max two cells apart
        bp.inv_cw[c] *= (1.0 - 1e-12);
    }
    BinEdges eq;
    for (int k = 0; k <= GR_MAXBINS; ++k) eq.q[k] = (k <= g->nb) ? g->q[k] : INFINITY;

    g->ptr.alloc((size_t)n + 1);
    g->w.alloc((size_t)n);
    g->order.alloc((size_t)n);
    if (g->spatial) { g->caller_of.alloc((size_t)n); g->cell_of.alloc((size_t)n); }
    if (n == 0) {
        GR_CUDA(cudaMemsetAsync(g->ptr.p, 0, sizeof(int64_t), st));
        g->idx.alloc(0); g->bin.alloc(0);
        if (g->has_pix) g->pix.alloc(0);
        g->windows.clear();
        GrWindow w0; g->windows.push_back(w0);
        g->n_edges = 0; g->max_row = 0;
        GR_CUDA(cudaStreamSynchronize(st));
        g->t_build_ms = timer.stop();
        g->n_launches = launches;
        return;
    }

    // --- counting sort of the points by cell, ascending caller index inside a cell (A1) ---
    DevBuf<int32_t> cell_of, cell_cnt, cell_fill, slot_pt;
    DevBuf<int32_t> &cell_start = g->cell_start;      // kept: the dense cell-block rows are laid out by cell (dense.cu)
    g->ncell = ncell;
    cell_of.alloc((size_t)n);
    cell_cnt.alloc((size_t)ncell);
    cell_start.alloc((size_t)ncell + 1);
    cell_fill.alloc((size_t)ncell + 1);
    slot_pt.alloc((size_t)n);
    GR_CUDA(cudaMemsetAsync(cell_cnt.p, 0, sizeof(int32_t) * ncell, st));
    k_cell_id<<<blocks_for(n, 256), 256, 0, st>>>(bp, d_points, cell_of.p, cell_cnt.p);
    exclusive_scan<int32_t>(cell_cnt.p, ncell, cell_start.p, st);
    GR_CUDA(cudaMemcpyAsync(cell_fill.p, cell_start.p, sizeof(int32_t) * (ncell + 1), cudaMemcpyDeviceToDevice, st));
    k_scatter_cells<<<blocks_for(n, 256), 256, 0, st>>>(cell_of.p, cell_fill.p, slot_pt.p, n);
    segsort<int32_t>(cell_start.p, 0, ncell, 0, seg_max<int32_t>(cell_start.p, ncell, st), slot_pt.p, nullptr, nullptr, st);
    launches += 6;

    DevBuf<double> sx, sy, sz;
    DevBuf<int32_t> lab;
    sx.alloc((size_t)n); sy.alloc((size_t)n); sz.alloc((size_t)n); lab.alloc((size_t)n);
    k_gather_slots<<<blocks_for(n, 256), 256, 0, st>>>(d_points, slot_pt.p, sx.p, sy.p, sz.p, lab.p,
                                                       g->spatial ? g->caller_of.p : nullptr, cell_of.p,
                                                       g->spatial ? g->cell_of.p : nullptr, n, g->spatial);
    k_gather_weights<<<blocks_for(n, 256), 256, 0, st>>>(d_weights, slot_pt.p, g->w.p, n, g->spatial);
    GR_CUDA(cudaMemcpyAsync(g->order.p, lab.p, sizeof(int32_t) * n, cudaMemcpyDeviceToDevice, st));
    launches += 2;

    // --- A2 count, A3 offsets ---
    DevBuf<int32_t> deg;
    deg.alloc((size_t)n);
    const unsigned nblk = blocks_for(n * 32, 256);
    k_neighbours<false><<<nblk, 256, 0, st>>>(bp, eq, sx.p, sy.p, sz.p, lab.p, cell_start.p, 0, n, 0, INT32_MAX, deg.p,
                                              nullptr, 0, nullptr, nullptr, nullptr);
    if (g->slab_count > 1) {
        // equal-work cell ranges (work of a hub ~ its wedges ~ deg^2); this graph owns range slab_index and keeps the
        // rows of its cells and of their forward stencil cells (where the spokes of its hubs live)
        DevBuf<double> cost;
        cost.alloc((size_t)ncell);
        k_cell_cost<<<blocks_for(ncell, 128), 128, 0, st>>>(ncell, cell_start.p, deg.p, cost.p);
        std::vector<double> hc((size_t)ncell);
        std::vector<int32_t> hs((size_t)ncell + 1);
        GR_CUDA(cudaMemcpyAsync(hc.data(), cost.p, sizeof(double) * ncell, cudaMemcpyDeviceToHost, st));
        GR_CUDA(cudaMemcpyAsync(hs.data(), cell_start.p, sizeof(int32_t) * (ncell + 1), cudaMemcpyDeviceToHost, st));
        GR_CUDA(cudaStreamSynchronize(st));
        double total = 0.0;
        for (double x : hc) total += x + 1.0;           // + 1 per cell: empty catalogues still split
        auto boundary = [&](int k) -> int64_t {          // first cell of range k
            if (k <= 0) return 0;
            if (k >= g->slab_count) return ncell;
            const double want = total * (double)k / (double)g->slab_count;
            double acc = 0.0;
            for (int64_t c = 0; c < ncell; ++c) { if (acc >= want) return c; acc += hc[c] + 1.0; }
            return ncell;
        };
        const int64_t c_lo = boundary(g->slab_index), c_hi = boundary(g->slab_index + 1);
        std::vector<uint8_t> keep((size_t)ncell, 0);
        for (int64_t c = c_lo; c < c_hi; ++c) {
            const int cx = (int)(c % g->nc[0]), cy = (int)((c / g->nc[0]) % g->nc[1]), cz = (int)(c / ((int64_t)g->nc[0] * g->nc[1]));
            for (int t = 0; t < 27; ++t) {
                int o[3] = {cx + (t % 3) - 1, cy + ((t / 3) % 3) - 1, cz + (t / 9) - 1};
                bool ok = true;
                for (int a = 0; a < 3; ++a) {
                    if (g->periodic) o[a] = (o[a] + g->nc[a]) % g->nc[a];
                    else if (o[a] < 0 || o[a] >= g->nc[a]) ok = false;
                }
                if (!ok) continue;
                const int64_t id = ((int64_t)o[2] * g->nc[1] + o[1]) * g->nc[0] + o[0];
                if (id >= c) keep[(size_t)id] = 1;
            }
        }
        g->cell_keep.alloc((size_t)ncell);
        GR_CUDA(cudaMemcpyAsync(g->cell_keep.p, keep.data(), (size_t)ncell, cudaMemcpyHostToDevice, st));
        k_mask_deg<<<blocks_for(n, 256), 256, 0, st>>>(n, g->cell_of.p, g->cell_keep.p, deg.p);
        GR_CUDA(cudaStreamSynchronize(st));             // `keep` goes out of scope
        g->hub_lo = hs[(size_t)c_lo];
        g->hub_hi = hs[(size_t)c_hi];
        launches += 2;
    }
    exclusive_scan<int64_t>(deg.p, n, g->ptr.p, st);
    launches += 4;
    int64_t E = 0;
    GR_CUDA(cudaMemcpyAsync(&E, g->ptr.p + n, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    GR_CUDA(cudaStreamSynchronize(st));
    g->max_row = seg_max<int64_t>(g->ptr.p, n, st);
    launches += 1;
    g->n_edges = E;

    // --- windows (row-aligned): one window in-core, several when a memory cap is set ---
    const uint64_t bpe = 5 + (g->has_pix ? 1 : 0);
    std::vector<int64_t> hptr;
    g->windows.clear();
    int W = 1;
    g->ooc = 0;
    if (g->cap_bytes && ((uint64_t)E * bpe > g->cap_bytes || n_windows_forced > 1)) {
        g->ooc = 1;
        // four window buffers must fit under the cap (hub + search, double buffered); on a spatially relabelled
        // graph a window buffer also holds the dense cell-block rows expanded from its CSR rows (gather kernel)
        uint64_t total = (uint64_t)E * bpe;
        if (g->spatial && gr_dense_tables(g)) total += (uint64_t)g->dn.total;
        uint64_t per = g->cap_bytes / 4;
        W = (int)((total + per - 1) / std::max<uint64_t>(per, 1));
        W = std::max(W, 2);
    }
    if (n_windows_forced > 0) { W = n_windows_forced; g->ooc = (g->cap_bytes != 0); }
    if (W > 1 || g->ooc) {
        hptr.resize((size_t)n + 1);
        GR_CUDA(cudaMemcpyAsync(hptr.data(), g->ptr.p, sizeof(int64_t) * (n + 1), cudaMemcpyDeviceToHost, st));
        GR_CUDA(cudaStreamSynchronize(st));
    }
    // The cut is by edges, the buffers also hold dense rows, and a window cannot split a row: the largest window can exceed
    // cap / 4.  W grows until FOUR buffers fit (hub + search + the next tile's two: with three the tiler re-stages a window
    // for nearly every tile -- configs[4] under 24 GiB: 114 GB staged per query with 3 buffers, 1.3 x the CSR with 4).
    for (int attempt = 0;; ++attempt) {
        g->windows.clear();
        if (W <= 1) {
            GrWindow w0;
            w0.row_lo = 0; w0.row_hi = (int32_t)n; w0.e_lo = 0; w0.e_hi = E;
            g->windows.push_back(w0);
        } else {
            // boundaries at the first row starting at or after k*E/W (k = 1..W-1); empty windows are dropped
            int32_t r = 0;
            for (int k = 1; k <= W && r < n; ++k) {
                int32_t r2 = (int32_t)n;
                if (k < W) {
                    const int64_t want = (int64_t)(((__int128)E * k) / W);
                    r2 = (int32_t)(std::lower_bound(hptr.begin(), hptr.begin() + n, want) - hptr.begin());
                    r2 = std::max(r2, r + 1);
                    r2 = (int32_t)std::min<int64_t>(r2, n);
                    if (hptr[r2] == hptr[r] && r2 < n) continue;      // no edges yet: extend this window
                }
                GrWindow w;
                w.row_lo = r;
                w.row_hi = r2;
                w.e_lo = hptr[r] & ~int64_t(15);
                w.e_hi = hptr[r2];
                g->windows.push_back(w);
                r = r2;
            }
        }
        if (g->ooc && g->spatial && gr_dense_tables(g)) {      // dense byte range of every window
            std::vector<int32_t> rows;
            for (auto &w : g->windows) rows.push_back(w.row_lo);
            rows.push_back((int32_t)n);
            std::vector<int64_t> addr(rows.size());
            gr_dense_rowaddrs(g, rows.data(), (int)rows.size(), addr.data());
            for (size_t k = 0; k < g->windows.size(); ++k) { g->windows[k].d_lo = addr[k]; g->windows[k].d_hi = addr[k + 1]; }
        }
        if (!g->ooc || n_windows_forced > 0 || attempt >= 12 || W >= 1000) break;
        int64_t maxbuf = 0;
        for (auto &w : g->windows) maxbuf = std::max<int64_t>(maxbuf, (w.e_hi - w.e_lo) * (int64_t)bpe + (w.d_hi - w.d_lo));
        if ((uint64_t)maxbuf * 4 <= g->cap_bytes) break;
        W = W + std::max(1, W / 8);
    }

    DevBuf<int32_t> stats;
    stats.alloc(32);
    GR_CUDA(cudaMemsetAsync(stats.p, 0, sizeof(int32_t) * 32, st));

    // --- A4 fill (+ A5 sort when labels are not in cell order) per window ---
    if (!g->ooc) {
        g->idx.alloc((size_t)E);
        g->bin.alloc((size_t)E);
        if (g->has_pix) g->pix.alloc((size_t)E);
        k_neighbours<true><<<nblk, 256, 0, st>>>(bp, eq, sx.p, sy.p, sz.p, lab.p, cell_start.p, 0, n, 0, INT32_MAX, nullptr,
                                                 g->ptr.p, 0, g->idx.p, g->bin.p, g->has_pix ? g->pix.p : nullptr);
        launches += 1;
        if (!g->spatial) {
            segsort<int64_t>(g->ptr.p, 0, n, 0, g->max_row, g->idx.p, g->bin.p, g->has_pix ? g->pix.p : nullptr, st);
            launches += 1;
        }
        GR_CUDA(cudaGetLastError());      // (row statistics of the slot-table kernel: on first use, gr_row_stats)
    } else {
        // Every window gets ONE page-locked host block [idx | bin | pix] (entry 0 = edge e_lo).  Page-locking is the
        // slowest step of a capped build (~25 GiB/s on this box, 42 GB for configs[4]), so a background thread prepares
        // the blocks in window order (cached blocks of an earlier graph first) while the device fills the windows;
        // fills go to two staging buffers, and the copy of window k to the host (copy stream) overlaps the fill of k+1.
        const int Wn = (int)g->windows.size();
        if (Wn > 1024) GR_FAIL(GRAMSCI_ENOMEM, "device_mem_cap_bytes too small: %d windows", Wn);
        int64_t maxlen = 0;
        for (auto &w : g->windows) maxlen = std::max(maxlen, w.e_hi - w.e_lo);
        DevBuf<int32_t> widx[2];
        DevBuf<uint8_t> wbin[2], wpix[2];
        for (int k = 0; k < 2; ++k) {
            widx[k].alloc((size_t)maxlen); wbin[k].alloc((size_t)maxlen);
            if (g->has_pix) wpix[k].alloc((size_t)maxlen);
        }
        g->need.assign((size_t)Wn * Wn, 0);
        const int mwords = (Wn + 31) / 32;
        DevBuf<unsigned int> dmask;
        DevBuf<int32_t> dwlo;
        dmask.alloc((size_t)mwords);
        dwlo.alloc((size_t)Wn + 1);
        std::vector<unsigned int> hmask((size_t)mwords);
        {
            std::vector<int32_t> hw((size_t)Wn + 1);
            for (int c = 0; c < Wn; ++c) hw[c] = g->windows[c].row_lo;
            hw[Wn] = (int32_t)n;
            GR_CUDA(cudaMemcpyAsync(dwlo.p, hw.data(), sizeof(int32_t) * (Wn + 1), cudaMemcpyHostToDevice, st));
            GR_CUDA(cudaStreamSynchronize(st));
        }
        struct Pipe {                                   // joined / destroyed before the staging buffers go away
            std::thread th;
            std::atomic<int> ready{0}, failed{0}, stop{0};
            std::string err;
            cudaStream_t cs = nullptr;
            cudaEvent_t filled[2] = {nullptr, nullptr}, copied[2] = {nullptr, nullptr};
            ~Pipe() {
                stop.store(1);
                if (th.joinable()) th.join();
                if (cs) { cudaStreamSynchronize(cs); cudaStreamDestroy(cs); }
                for (int k = 0; k < 2; ++k) { if (filled[k]) cudaEventDestroy(filled[k]); if (copied[k]) cudaEventDestroy(copied[k]); }
            }
        } pipe;
        GR_CUDA(cudaStreamCreateWithFlags(&pipe.cs, cudaStreamNonBlocking));
        for (int k = 0; k < 2; ++k) {
            GR_CUDA(cudaEventCreateWithFlags(&pipe.filled[k], cudaEventDisableTiming));
            GR_CUDA(cudaEventCreateWithFlags(&pipe.copied[k], cudaEventDisableTiming));
        }
        int dev = 0;
        GR_CUDA(cudaGetDevice(&dev));
        const int has_pix = g->has_pix;
        pipe.th = std::thread([g, Wn, dev, has_pix, &pipe] {
            cudaSetDevice(dev);
            for (int k = 0; k < Wn && !pipe.stop.load(); ++k) {
                GrWindow &w = g->windows[k];
                const size_t len = (size_t)(w.e_hi - w.e_lo);
                const size_t sec_i = (len * 4 + 255) & ~size_t(255), sec_b = (len + 255) & ~size_t(255);
                size_t bytes = std::max<size_t>(4096, sec_i + sec_b * (has_pix ? 2 : 1));
                void *blk = gr_pinned_alloc_nothrow(&bytes, &pipe.err);
                if (!blk) { pipe.failed.store(1); return; }
                w.h_block = blk;
                w.h_block_bytes = bytes;
                w.h_idx = (int32_t *)blk;
                w.h_bin = (uint8_t *)blk + sec_i;
                w.h_pix = has_pix ? (uint8_t *)blk + sec_i + sec_b : nullptr;
                pipe.ready.store(k + 1, std::memory_order_release);
            }
        });
        for (int hwin = 0; hwin < Wn; ++hwin) {
            GrWindow &w = g->windows[hwin];
            const int sb = hwin & 1;
            int64_t len = w.e_hi - w.e_lo;
            int64_t s_lo = g->spatial ? w.row_lo : 0, s_hi = g->spatial ? w.row_hi : n;
            unsigned nb2 = blocks_for((s_hi - s_lo) * 32, 256);
            if (hwin >= 2) GR_CUDA(cudaStreamWaitEvent(st, pipe.copied[sb], 0));     // window hwin-2 has left this staging buffer
            k_neighbours<true><<<nb2, 256, 0, st>>>(bp, eq, sx.p, sy.p, sz.p, lab.p, cell_start.p, s_lo, s_hi, w.row_lo, w.row_hi,
                                                    nullptr, g->ptr.p, w.e_lo, widx[sb].p, wbin[sb].p, g->has_pix ? wpix[sb].p : nullptr);
            launches += 1;
            if (!g->spatial) {
                segsort<int64_t>(g->ptr.p, w.row_lo, w.row_hi, w.e_lo, g->max_row, widx[sb].p, wbin[sb].p, g->has_pix ? wpix[sb].p : nullptr, st);
                launches += 1;
            }
            GR_CUDA(cudaEventRecord(pipe.filled[sb], st));
            k_row_stats<<<blocks_for((int64_t)(w.row_hi - w.row_lo) * 32, 256), 256, 0, st>>>(g->ptr.p, widx[sb].p, w.e_lo,
                                                                                           w.row_lo, w.row_hi, stats.p);
            launches += 1;
            int64_t head = hptr[w.row_lo] - w.e_lo;   // entries before the first row belong to the previous window
            // search windows this hub window reaches (exact)
            GR_CUDA(cudaMemsetAsync(dmask.p, 0, sizeof(unsigned int) * mwords, st));
            if (len > head)
                k_need_mask<<<296, 256, sizeof(unsigned int) * mwords, st>>>(widx[sb].p, head, len, dwlo.p, Wn, dmask.p);
            GR_CUDA(cudaMemcpyAsync(hmask.data(), dmask.p, sizeof(unsigned int) * mwords, cudaMemcpyDeviceToHost, st));
            launches += 1;
            // the host block of this window (background thread), then its copy on the copy stream
            while (pipe.ready.load(std::memory_order_acquire) <= hwin) {
                if (pipe.failed.load()) GR_FAIL(GRAMSCI_ENOMEM, "%s", pipe.err.c_str());
                std::this_thread::sleep_for(std::chrono::microseconds(50));
            }
            GR_CUDA(cudaStreamWaitEvent(pipe.cs, pipe.filled[sb], 0));
            if (len > head) {
                GR_CUDA(cudaMemcpyAsync(w.h_idx + head, widx[sb].p + head, (size_t)(len - head) * 4, cudaMemcpyDeviceToHost, pipe.cs));
                GR_CUDA(cudaMemcpyAsync(w.h_bin + head, wbin[sb].p + head, (size_t)(len - head), cudaMemcpyDeviceToHost, pipe.cs));
                if (g->has_pix)
                    GR_CUDA(cudaMemcpyAsync(w.h_pix + head, wpix[sb].p + head, (size_t)(len - head), cudaMemcpyDeviceToHost, pipe.cs));
            }
            GR_CUDA(cudaEventRecord(pipe.copied[sb], pipe.cs));
            GR_CUDA(cudaStreamSynchronize(st));
            for (int c = 0; c < Wn; ++c)
                if (hmask[c >> 5] & (1u << (c & 31))) g->need[(size_t)hwin * Wn + c] = 1;
        }
        GR_CUDA(cudaStreamSynchronize(pipe.cs));
        GR_CUDA(cudaStreamSynchronize(st));
    }
    if (g->ooc) {
        int32_t h[32];
        GR_CUDA(cudaMemcpyAsync(h, stats.p, sizeof h, cudaMemcpyDeviceToHost, st));
        GR_CUDA(cudaStreamSynchronize(st));
        for (int s = GR_S_MIN; s <= GR_S_MAX; ++s) {
            g->max_ptl[s] = h[2 * (s - GR_S_MIN)];
            g->max_pages[s] = h[2 * (s - GR_S_MIN) + 1];
        }
        g->stats_done = 1;
    }
    // range of |w|: the gather kernel accumulates weighted sums in fixed point when the weights are of one scale
    if (d_weights && n > 0) {
        DevBuf<double> mm;
        mm.alloc(2);
        const double init[2] = {INFINITY, 0.0};
        double h[2];
        GR_CUDA(cudaMemcpyAsync(mm.p, init, 16, cudaMemcpyHostToDevice, st));
        k_abs_minmax<<<296, 256, 0, st>>>(g->w.p, n, mm.p);
        GR_CUDA(cudaMemcpyAsync(h, mm.p, 16, cudaMemcpyDeviceToHost, st));
        GR_CUDA(cudaStreamSynchronize(st));
        g->w_absmin = h[0];
        g->w_absmax = h[1];
        launches += 1;
    }
    if (const char *e = getenv("GRAMSCI_GATHER_G")) g->algo_g = (atoi(e) == 1 || atoi(e) == 8) ? atoi(e) : 0;
    g->t_build_ms = timer.stop();
    g->n_launches = launches;
}

// row statistics of the slot-table 3pCF kernel, on first use (in-core graphs; capped graphs gather them in the build)
void gr_row_stats(gramsci_graph *g)
{
    if (g->stats_done || g->ooc || g->n <= 0) return;
    cudaStream_t st = g->stream;
    DevBuf<int32_t> stats;
    stats.alloc(32);
    GR_CUDA(cudaMemsetAsync(stats.p, 0, sizeof(int32_t) * 32, st));
    k_row_stats<<<blocks_for(g->n * 32, 256), 256, 0, st>>>(g->ptr.p, g->idx.p, 0, 0, (int32_t)g->n, stats.p);
    GR_CUDA(cudaGetLastError());
    int32_t h[32];
    GR_CUDA(cudaMemcpyAsync(h, stats.p, sizeof h, cudaMemcpyDeviceToHost, st));
    GR_CUDA(cudaStreamSynchronize(st));
    for (int s = GR_S_MIN; s <= GR_S_MAX; ++s) {
        g->max_ptl[s] = h[2 * (s - GR_S_MIN)];
        g->max_pages[s] = h[2 * (s - GR_S_MIN) + 1];
    }
    g->stats_done = 1;
    g->n_launches += 1;
}

// ---------------------------------------------------------------------------------------------------
void gr_export_csr(const gramsci_graph *g, int64_t *d_ptr, int32_t *d_idx, uint8_t *d_bin, uint8_t *d_pix)
{
    cudaStream_t st = g->stream;
    const int64_t n = g->n, E = g->n_edges;
    if (g->ooc) GR_FAIL(GRAMSCI_EINVAL, "export_csr: not supported for out-of-core graphs");
    if (!g->spatial) {
        if (d_ptr) GR_CUDA(cudaMemcpyAsync(d_ptr, g->ptr.p, sizeof(int64_t) * (n + 1), cudaMemcpyDeviceToDevice, st));
        if (d_idx && E) GR_CUDA(cudaMemcpyAsync(d_idx, g->idx.p, sizeof(int32_t) * E, cudaMemcpyDeviceToDevice, st));
        if (d_bin && E) GR_CUDA(cudaMemcpyAsync(d_bin, g->bin.p, E, cudaMemcpyDeviceToDevice, st));
        if (d_pix && E && g->has_pix) GR_CUDA(cudaMemcpyAsync(d_pix, g->pix.p, E, cudaMemcpyDeviceToDevice, st));
        GR_CUDA(cudaStreamSynchronize(st));
        return;
    }
    DevBuf<int32_t> deg, fill, oidx;
    DevBuf<int64_t> optr;
    DevBuf<uint8_t> obin;
    deg.alloc((size_t)n); fill.alloc((size_t)n); optr.alloc((size_t)n + 1); oidx.alloc((size_t)E); obin.alloc((size_t)E);
    GR_CUDA(cudaMemsetAsync(deg.p, 0, sizeof(int32_t) * std::max<int64_t>(n, 1), st));
    GR_CUDA(cudaMemsetAsync(fill.p, 0, sizeof(int32_t) * std::max<int64_t>(n, 1), st));
    if (n) k_export_count<<<blocks_for(n, 256), 256, 0, st>>>(g->ptr.p, g->idx.p, g->caller_of.p, n, deg.p);
    exclusive_scan<int64_t>(deg.p, n, optr.p, st);
    if (n) {
        k_export_fill<<<blocks_for(n, 256), 256, 0, st>>>(g->ptr.p, g->idx.p, g->bin.p, g->caller_of.p, n, optr.p, fill.p,
                                                          oidx.p, obin.p);
        segsort<int64_t>(optr.p, 0, n, 0, seg_max<int64_t>(optr.p, n, st), oidx.p, obin.p, nullptr, st);
    }
    GR_CUDA(cudaGetLastError());
    if (d_ptr) GR_CUDA(cudaMemcpyAsync(d_ptr, optr.p, sizeof(int64_t) * (n + 1), cudaMemcpyDeviceToDevice, st));
    if (d_idx && E) GR_CUDA(cudaMemcpyAsync(d_idx, oidx.p, sizeof(int32_t) * E, cudaMemcpyDeviceToDevice, st));
    if (d_bin && E) GR_CUDA(cudaMemcpyAsync(d_bin, obin.p, E, cudaMemcpyDeviceToDevice, st));
    GR_CUDA(cudaStreamSynchronize(st));
}
