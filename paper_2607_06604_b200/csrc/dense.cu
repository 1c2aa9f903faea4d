// dense.cu -- dense cell-block rows: the membership structure of the gather 3pCF kernel (query3g.cu).
//
// P:149 keeps, per hub, a "local connectivity matrix lmat(k2,k1)" holding the bin of the edge between two hub
// neighbours so that the innermost loop is an O(1) lookup.  With labels in cell order (S:8(a) A1) the same idea
// works globally: every neighbour k > j of a point j lies in one of the <= 27 stencil cells of j's cell whose id is
// not smaller (the FORWARD stencil), and the labels of a cell are consecutive.  Row j of the dense structure is the
// concatenation, over the forward stencil cells c' of cell(j) in ascending id, of occ(c') bytes:
//     byte (segment c', position q) = bin of the edge (j, cell_start[c'] + q), or 0xFF if there is none.
// "Is (j,k) an edge, and in which bin" is then ONE byte load for any k > j -- the 3pCF becomes, per hub i, a gather
// of the bytes (j,k) over the pairs j < k of N+(i) (query3g.cu).  Rows of one cell share their layout, so the whole
// structure is a set of dense blocks (cell, forward cell); at the ~15 % fill of a 27-cell stencil it takes about
// as much memory as the 5-byte CSR entries it is expanded from (cfg2: 0.40-0.47 GB; cfg5: 66 GB).
//
// The rows are EXPANDED FROM THE CSR (memset + one scatter pass), so the CSR stays the graph's primary form
// (export, 2pCF, 4pCF, the other 3pCF kernels) and the out-of-core tiler can expand a staged CSR window on the
// device instead of streaming dense rows over PCIe.
#include "internal.cuh"

#include <algorithm>
#include <climits>

namespace {

// ---- per-cell layout: sorted forward stencil, segment offsets, row length ----------------------------------
__global__ void k_cell_fwd(int64_t ncell, int ncx, int ncy, int ncz, int periodic, const int32_t *__restrict__ cell_start,
                           int32_t *__restrict__ fwd_cell, int32_t *__restrict__ fwd_off, int32_t *__restrict__ nf,
                           int32_t *__restrict__ rowlen, int64_t *__restrict__ rowbytes, int32_t *__restrict__ stats,
                           const uint8_t *__restrict__ keep)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    const int cx = (int)(c % ncx), cy = (int)((c / ncx) % ncy), cz = (int)(c / ((int64_t)ncx * ncy));
    int ids[GR_STENCIL];
    int m = 0;
    for (int dz = -1; dz <= 1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
            for (int dx = -1; dx <= 1; ++dx) {
                int o[3] = {cx + dx, cy + dy, cz + dz};
                const int nc[3] = {ncx, ncy, ncz};
                bool ok = true;
                for (int a = 0; a < 3; ++a) {
                    if (periodic) o[a] = (o[a] + nc[a]) % nc[a];
                    else if (o[a] < 0 || o[a] >= nc[a]) ok = false;
                }
                if (!ok) continue;
                const int id = (o[2] * ncy + o[1]) * ncx + o[0];
                if (id < (int)c) continue;                        // label k > j  =>  cell(k) >= cell(j)
                bool dup = false;                                // periodic grids with < 3 cells on an axis alias
                for (int t = 0; t < m; ++t) dup = dup || ids[t] == id;
                if (dup) continue;
                int t = m++;
                while (t > 0 && ids[t - 1] > id) { ids[t] = ids[t - 1]; --t; }
                ids[t] = id;
            }
    int off = 0;
    for (int t = 0; t < GR_STENCIL; ++t) {
        if (t < m) {
            fwd_cell[c * GR_STENCIL + t] = ids[t];
            fwd_off[c * GR_STENCIL + t] = off;
            off += cell_start[ids[t] + 1] - cell_start[ids[t]];
        } else {
            fwd_cell[c * GR_STENCIL + t] = -1;
            fwd_off[c * GR_STENCIL + t] = -1;
        }
    }
    const int occ = cell_start[c + 1] - cell_start[c];
    // rows start on 32-byte sectors (row addresses fit 32 bits after >> 5) and end with at least ONE pad byte, which
    // stays 0xFF: the gather kernel points entries that have no segment in a row at it instead of predicating the load
    const int rl = (off + 32) & ~31;
    nf[c] = m;
    rowlen[c] = rl;
    rowbytes[c] = (keep && !keep[c]) ? 0 : (int64_t)occ * rl;      // slab graphs: no dense rows outside slab + halo
    if (occ > 0) {
        atomicMax(&stats[0], occ);
        atomicMax(&stats[1], rl);
    }
}

// ---- expansion: CSR rows -> dense rows (warp per row) -----------------------------------------------------
__global__ void __launch_bounds__(256)
k_dense_scatter(int32_t row_lo, int32_t row_hi, const int64_t *__restrict__ ptr, const int32_t *__restrict__ idx,
                const uint8_t *__restrict__ bin, int64_t e0, const int32_t *__restrict__ cell_of,
                const int32_t *__restrict__ cell_start, const int32_t *__restrict__ fwd_cell,
                const int32_t *__restrict__ fwd_off, const int32_t *__restrict__ nf, const int32_t *__restrict__ rowlen,
                const int64_t *__restrict__ dbase, int64_t d0, uint8_t *__restrict__ out)
{
    const int lane = threadIdx.x & 31;
    const int64_t j = row_lo + ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) / 32;
    if (j >= row_hi) return;
    const int64_t rb = ptr[j], re = ptr[j + 1];
    if (re == rb) return;
    const int c = cell_of[j];
    const int m = nf[c];
    int fs = INT_MAX, fo = 0;
    if (lane < m) {
        fs = cell_start[fwd_cell[(int64_t)c * GR_STENCIL + lane]];
        fo = fwd_off[(int64_t)c * GR_STENCIL + lane];
    }
    uint8_t *row = out + (dbase[c] + (int64_t)((int)j - cell_start[c]) * rowlen[c] - d0);
    for (int64_t eb = rb; eb < re; eb += 32) {            // the whole warp iterates (shuffles below)
        const int64_t e = eb + lane;
        const bool ok = e < re;
        const int32_t k = ok ? idx[e - e0] : INT_MAX - 1;
        int o = -1;
        for (int t = 0; t < m; ++t) o += (__shfl_sync(0xffffffffu, fs, t) <= k) ? 1 : 0;
        o = max(o, 0);
        const int pos = __shfl_sync(0xffffffffu, fo, o) + (k - __shfl_sync(0xffffffffu, fs, o));
        if (ok) row[pos] = bin[e - e0];
    }
}

__global__ void k_rowaddr(const int32_t *__restrict__ rows, int nrows, int64_t n, const int32_t *__restrict__ cell_of,
                          const int32_t *__restrict__ cell_start, const int32_t *__restrict__ rowlen,
                          const int64_t *__restrict__ dbase, int64_t total, int64_t *__restrict__ out)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nrows) return;
    const int32_t j = rows[t];
    if (j >= n) { out[t] = total; return; }
    const int c = cell_of[j];
    out[t] = dbase[c] + (int64_t)(j - cell_start[c]) * rowlen[c];
}

// ---- work units of the gather kernels: runs of hubs inside one cell ------------------------------------------
// Only hubs whose row length lies in [len_lo, len_hi] count (the kernel skips the others): rows of up to a few hundred
// entries go to the warp-per-hub kernel, longer ones to the CTA-per-hub kernel.  A unit closes after max_hubs
// counted hubs.  pass 0 counts the units of every cell, pass 1 writes (first label, last label + 1) at the scanned
// offsets.
__global__ void k_units(int64_t ncell, const int32_t *__restrict__ cell_start, const int64_t *__restrict__ ptr,
                        int max_hubs, int len_lo, int len_hi, int pass, const int32_t *__restrict__ unit_off,
                        int32_t *__restrict__ unit_cnt, int2 *__restrict__ units)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    const int lo = cell_start[c], hi = cell_start[c + 1];
    int nu = 0, hubs = 0, start = lo, last = lo;
    int out = pass ? unit_off[c] : 0;
    for (int i = lo; i < hi; ++i) {
        const int64_t n = ptr[i + 1] - ptr[i];
        if (n < len_lo || n > len_hi) continue;
        if (hubs >= max_hubs) {
            if (pass) units[out++] = make_int2(start, last + 1);
            ++nu; hubs = 0;
        }
        if (hubs == 0) start = i;
        last = i;
        ++hubs;
    }
    if (hubs > 0) {
        if (pass) units[out] = make_int2(start, last + 1);
        ++nu;
    }
    if (!pass) unit_cnt[c] = nu;
}

// (hub, spoke tile) units of the CTA gather kernel: units(c) = #tiles(c) x #listed hubs(c), where the tiles of cell c cut
// the dense rows of every forward cell into runs of at most tile_bytes (the same arithmetic as the kernel's walk)
__global__ void k_tile_units(int64_t ncell, const int32_t *__restrict__ cell_start, const int32_t *__restrict__ fwd_cell,
                             const int32_t *__restrict__ nf, const int32_t *__restrict__ rowlen,
                             const int32_t *__restrict__ ucell_off, long long tile_bytes, int64_t *__restrict__ units)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= ncell) return;
    const int nl = ucell_off[c + 1] - ucell_off[c];
    long long nt = tile_bytes ? 0 : 1;                 // tile_bytes 0: one unit per listed hub
    if (nl > 0 && tile_bytes)
        for (int o = 0; o < nf[c]; ++o) {
            const int fc = fwd_cell[c * GR_STENCIL + o];
            const long long bytes = (long long)(cell_start[fc + 1] - cell_start[fc]) * rowlen[fc];
            nt += max(1ll, (bytes + tile_bytes - 1) / tile_bytes);
        }
    units[c] = nt * nl;
}

inline unsigned blocks_for(int64_t n, int per) { return (unsigned)std::max<int64_t>(1, (n + per - 1) / per); }

}  // namespace

// Layout tables (any spatial graph); false + reason when the structure does not apply.
bool gr_dense_tables(gramsci_graph *g)
{
    GrDense &d = g->dn;
    if (d.state != 0) return d.state > 0;
    d.state = -1;
    if (!g->spatial) { d.why = "labels are not in cell order"; return false; }
    if (g->n <= 0 || g->n_edges <= 0) { d.why = "empty graph"; return false; }
    cudaStream_t st = g->stream;
    const int64_t nc = g->ncell;
    d.fwd_cell.alloc((size_t)nc * GR_STENCIL);
    d.fwd_off.alloc((size_t)nc * GR_STENCIL);
    d.nf.alloc((size_t)nc);
    d.rowlen.alloc((size_t)nc);
    d.dbase.alloc((size_t)nc + 1);
    DevBuf<int64_t> rowbytes;
    DevBuf<int32_t> stats;
    rowbytes.alloc((size_t)nc);
    stats.alloc(2);
    GR_CUDA(cudaMemsetAsync(stats.p, 0, 8, st));
    k_cell_fwd<<<blocks_for(nc, 128), 128, 0, st>>>(nc, g->nc[0], g->nc[1], g->nc[2], g->periodic, g->cell_start.p,
                                                    d.fwd_cell.p, d.fwd_off.p, d.nf.p, d.rowlen.p, rowbytes.p, stats.p,
                                                    g->cell_keep.p);
    GR_CUDA(cudaGetLastError());
    gr_exclusive_scan<int64_t, int64_t>(rowbytes.p, nc, d.dbase.p, st);
    int32_t h[2];
    GR_CUDA(cudaMemcpyAsync(h, stats.p, 8, cudaMemcpyDeviceToHost, st));
    GR_CUDA(cudaMemcpyAsync(&d.total, d.dbase.p + nc, 8, cudaMemcpyDeviceToHost, st));
    GR_CUDA(cudaStreamSynchronize(st));
    d.max_occ = h[0];
    d.max_rowlen = h[1];
    g->n_launches += 4;
    if (d.max_occ >= 65536) { d.why = "a cell holds 65536 points or more"; return false; }
    d.state = 1;
    return true;
}

void gr_dense_rowaddrs(gramsci_graph *g, const int32_t *h_rows, int nrows, int64_t *h_out)
{
    GrDense &d = g->dn;
    DevBuf<int32_t> r;
    DevBuf<int64_t> a;
    r.alloc((size_t)nrows);
    a.alloc((size_t)nrows);
    GR_CUDA(cudaMemcpyAsync(r.p, h_rows, 4 * (size_t)nrows, cudaMemcpyHostToDevice, g->stream));
    k_rowaddr<<<blocks_for(nrows, 128), 128, 0, g->stream>>>(r.p, nrows, g->n, g->cell_of.p, g->cell_start.p, d.rowlen.p,
                                                             d.dbase.p, d.total, a.p);
    GR_CUDA(cudaMemcpyAsync(h_out, a.p, 8 * (size_t)nrows, cudaMemcpyDeviceToHost, g->stream));
    GR_CUDA(cudaStreamSynchronize(g->stream));
}

void gr_dense_expand(gramsci_graph *g, int32_t row_lo, int32_t row_hi, const int32_t *idx, const uint8_t *bin, int64_t e0,
                     uint8_t *out, int64_t d0, int64_t out_bytes, cudaStream_t st)
{
    GrDense &d = g->dn;
    if (row_hi <= row_lo || out_bytes <= 0) return;
    GR_CUDA(cudaMemsetAsync(out, 0xFF, (size_t)out_bytes, st));
    k_dense_scatter<<<blocks_for((int64_t)(row_hi - row_lo) * 32, 256), 256, 0, st>>>(
        row_lo, row_hi, g->ptr.p, idx, bin, e0, g->cell_of.p, g->cell_start.p, d.fwd_cell.p, d.fwd_off.p, d.nf.p,
        d.rowlen.p, d.dbase.p, d0, out);
    GR_CUDA(cudaGetLastError());
    g->n_launches += 2;
}

bool gr_dense_prepare(gramsci_graph *g)
{
    GrDense &d = g->dn;
    if (!gr_dense_tables(g)) return false;
    if (g->ooc || d.bytes.p) return true;
    GrTimer t(g->stream);
    const size_t fr = gr_dev_available();
    if ((size_t)d.total + ((size_t)2 << 30) > fr) {
        d.state = -1;
        d.why = "not enough free device memory for the dense rows";
        return false;
    }
    d.bytes.alloc((size_t)d.total + 64);
    gr_dense_expand(g, 0, (int32_t)g->n, g->idx.p, g->bin.p, 0, d.bytes.p, 0, d.total, g->stream);
    d.t_build_ms = t.stop();
    return true;
}

// work units of hubs with row length in [len_lo, len_hi], at most max_hubs per unit (cached per list)
void gr_dense_units(gramsci_graph *g, GrUnits &u, int max_hubs, int len_lo, int len_hi)
{
    if (u.units.p && u.max_hubs == max_hubs && u.len_lo == len_lo && u.len_hi == len_hi) return;
    cudaStream_t st = g->stream;
    const int64_t nc = g->ncell;
    DevBuf<int32_t> cnt, off;
    cnt.alloc((size_t)nc);
    off.alloc((size_t)nc + 1);
    k_units<<<blocks_for(nc, 128), 128, 0, st>>>(nc, g->cell_start.p, g->ptr.p, max_hubs, len_lo, len_hi, 0, nullptr, cnt.p, nullptr);
    gr_exclusive_scan<int32_t, int32_t>(cnt.p, nc, off.p, st);
    int32_t nu = 0;
    GR_CUDA(cudaMemcpyAsync(&nu, off.p + nc, 4, cudaMemcpyDeviceToHost, st));
    GR_CUDA(cudaStreamSynchronize(st));
    u.units.alloc((size_t)nu + 1);
    u.cell_off.alloc((size_t)nc + 1);
    GR_CUDA(cudaMemcpyAsync(u.cell_off.p, off.p, sizeof(int32_t) * (nc + 1), cudaMemcpyDeviceToDevice, st));
    u.tiles_valid = 0;
    if (nu > 0)
        k_units<<<blocks_for(nc, 128), 128, 0, st>>>(nc, g->cell_start.p, g->ptr.p, max_hubs, len_lo, len_hi, 1, off.p, nullptr, u.units.p);
    GR_CUDA(cudaGetLastError());
    GR_CUDA(cudaStreamSynchronize(st));
    u.n = nu;
    u.max_hubs = max_hubs;
    u.len_lo = len_lo;
    u.len_hi = len_hi;
    g->n_launches += 5;
}

// tile-major (hub, spoke tile) unit bases of a unit list (one hub per unit), for spoke tiles of tile_bytes
void gr_dense_tile_units(gramsci_graph *g, GrUnits &u, long long tile_bytes)
{
    if (u.tile_bytes == tile_bytes && u.tbase.p && u.tiles_valid) return;
    u.tiles_valid = 1;
    cudaStream_t st = g->stream;
    const int64_t nc = g->ncell;
    GrDense &d = g->dn;
    DevBuf<int64_t> per;
    per.alloc((size_t)nc);
    u.tbase.alloc((size_t)nc + 1);
    k_tile_units<<<blocks_for(nc, 128), 128, 0, st>>>(nc, g->cell_start.p, d.fwd_cell.p, d.nf.p, d.rowlen.p, u.cell_off.p,
                                                      tile_bytes, per.p);
    GR_CUDA(cudaGetLastError());
    gr_exclusive_scan<int64_t, int64_t>(per.p, nc, u.tbase.p, st);
    int64_t tot = 0;
    GR_CUDA(cudaMemcpyAsync(&tot, u.tbase.p + nc, 8, cudaMemcpyDeviceToHost, st));
    GR_CUDA(cudaStreamSynchronize(st));
    u.n_tile_units = tot;
    u.tile_bytes = tile_bytes;
    g->n_launches += 4;
}
