// internal.cuh -- shared declarations of the CUDA path (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <string>
#include <vector>

#include "../../include/gramsci.h"

#define GR_MAXBINS 255
#define GR_SM_COUNT_FALLBACK 148
#define GR_S_MIN 4
#define GR_S_MAX 11

// ---- error plumbing --------------------------------------------------------------------------
void gr_set_error(const char *fmt, ...);
struct GrFail { int code; };   // thrown inside the library only; every ABI entry catches it

#define GR_CUDA(call)                                                                         \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess) {                                                              \
            gr_set_error("%s:%d: %s -> %s", __FILE__, __LINE__, #call, cudaGetErrorString(e_)); \
            throw GrFail{e_ == cudaErrorMemoryAllocation ? GRAMSCI_ENOMEM : GRAMSCI_ECUDA};   \
        }                                                                                     \
    } while (0)

#define GR_FAIL(code_, ...)            \
    do {                               \
        gr_set_error(__VA_ARGS__);     \
        throw GrFail{code_};           \
    } while (0)

// ---- device buffer owned by the library --------------------------------------------------------
// Where device memory comes from (include/gramsci.h, gramsci_options.alloc / dealloc):
//  * the caller's allocator hooks when given (PyTorch's caching allocator in the Python binding), else
//  * stream-ordered allocations from a PRIVATE memory pool of the device (cudaMallocFromPoolAsync; release
//    threshold raised so that freed blocks are reused by the next call instead of going back to the driver: a
//    graph build or a query allocates tens of scratch buffers and must not pay a device synchronisation for
//    each).  The device's default pool is left alone; gramsci_release_memory() trims the private one.
// Every ABI entry sets the allocation context of the calling thread (gr_alloc_ctx); all library work runs
// on that stream.
struct GrAllocCtx {
    cudaStream_t stream = nullptr;
    void *(*alloc)(size_t, void *, void *) = nullptr;
    void (*dealloc)(void *, void *, void *) = nullptr;
    void *user = nullptr;
};
GrAllocCtx &gr_alloc_ctx();
inline cudaStream_t &gr_alloc_stream() { return gr_alloc_ctx().stream; }
void *gr_dev_alloc(size_t bytes, const GrAllocCtx &ctx, int *kind);     // kind: 0 cudaMalloc, 1 pool, 2 hook
void gr_dev_free(void *p, const GrAllocCtx &ctx, int kind);
size_t gr_dev_available();                     // driver-free bytes + freed blocks cached in the private pool

template <typename T>
struct DevBuf {
    T *p = nullptr;
    size_t n = 0;
    GrAllocCtx ctx;
    int kind = 0;
    DevBuf() {}
    DevBuf(const DevBuf &) = delete;
    DevBuf &operator=(const DevBuf &) = delete;
    ~DevBuf() { release(); }
    void alloc(size_t count) {
        release();
        n = count;
        size_t bytes = (count ? count : 1) * sizeof(T);
        bytes = (bytes + 255) & ~size_t(255);          // tail padding: aligned vector loads may over-read
        ctx = gr_alloc_ctx();
        p = (T *)gr_dev_alloc(bytes + 256, ctx, &kind);
    }
    void release() {
        if (p) gr_dev_free(p, ctx, kind);
        p = nullptr;
        n = 0;
    }
};

// One contiguous range of CSR rows whose edge arrays sit in one buffer (device or pinned host).
struct GrWindow {
    int32_t row_lo = 0, row_hi = 0;   // rows [row_lo,row_hi)
    int64_t e_lo = 0, e_hi = 0;       // edges [e_lo,e_hi), e_lo rounded down to a multiple of 16
    int64_t d_lo = 0, d_hi = 0;       // dense cell-block rows of these rows: bytes [d_lo,d_hi) (spatial graphs)
    // out-of-core: the window's edge arrays in ONE page-locked host block [idx | bin | pix]; entry 0 = edge e_lo
    void *h_block = nullptr;
    size_t h_block_bytes = 0;
    int32_t *h_idx = nullptr;
    uint8_t *h_bin = nullptr, *h_pix = nullptr;
};

// hub filter of the enumeration kernels (hub_stride: sampled partial result; shard_*: one shard of a multi-GPU run)
#define GR_HUB_SELECTED(v, i) (((v).hub_stride <= 1 || ((i) % (v).hub_stride) == 0) && \
                               ((v).shard_count <= 1 || ((i) % (v).shard_count) == (v).shard_index))

// Dense cell-block rows (dense.cu).  Row of point j (cell c, position p = j - cell_start[c]) lives at
// dbase[c] + p * rowlen[c] and holds, for every cell c' of the FORWARD stencil of c (the stencil cells with id >= c,
// ascending: fwd_cell[c*27 + o], o < nf[c]) a segment of occ(c') bytes at fwd_off[c*27 + o]: byte q of the segment
// = bin of the edge (j, cell_start[c'] + q) or 0xFF.  This is P:149's lmat idea made global: one byte answers
// "is (j,k) an edge and in which bin" for any k > j.
#define GR_STENCIL 27
struct GrUnits {                           // hub label ranges [x, y) inside one cell
    DevBuf<int2> units;
    DevBuf<int32_t> cell_off;              // [ncell+1] units of cell c are units[cell_off[c] .. cell_off[c+1])
    DevBuf<int64_t> tbase;                 // [ncell+1] CTA kernel: first (hub, spoke tile) unit of cell c
    long long tile_bytes = 0, n_tile_units = 0;
    int tiles_valid = 0;
    int n = 0, max_hubs = 0, len_lo = 0, len_hi = 0;
};
struct GrDense {
    int state = 0;                 // 0 not tried, 1 built, -1 not applicable (reason in `why`)
    const char *why = "";
    DevBuf<int32_t> fwd_cell, fwd_off;     // [ncell*27]
    DevBuf<int32_t> nf, rowlen;            // [ncell]
    DevBuf<int64_t> dbase;                 // [ncell+1] byte offset of the first row of every cell
    DevBuf<uint8_t> bytes;                 // in-core: all rows
    GrUnits ua, ub;                        // work units of the warp-per-hub / CTA-per-hub gather kernels
    int64_t total = 0;
    int32_t max_occ = 0, max_rowlen = 0;
    double t_build_ms = 0;
};

struct gramsci_graph {
    // parameters
    int64_t n = 0;
    int nb = 1;
    int periodic = 0;
    double box[3] = {0, 0, 0};
    double r_min = 0, r_max = 0;
    double q[GR_MAXBINS + 1];      // squared bin edges (A-3)
    int weighted = 0, has_pix = 0, spatial = 0, algo = 0, hub_stride = 1, shard_count = 1, shard_index = 0;
    int slab_count = 1, slab_index = 0;      // slab + halo partition (gramsci_options.slab_count)
    int32_t hub_lo = 0, hub_hi = INT32_MAX;  // hubs this graph owns (internal labels); everything unless slab_count > 1
    DevBuf<uint8_t> cell_keep;               // slab graphs: [ncell] 1 = rows of this cell are stored
    int algo_g = 0;                // gather kernel: forced warps per hub (test knob GRAMSCI_GATHER_G), 0 = choose
    double w_absmin = 1.0, w_absmax = 1.0;   // range of |w| (1 for unit weights): picks fixed-point or fp64 weighted sums
    cudaStream_t stream = nullptr;
    GrAllocCtx actx;               // allocator of this graph (hooks or the private pool), set at build
    int sm_count = GR_SM_COUNT_FALLBACK;
    size_t smem_optin = 0;
    // cell grid
    int nc[3] = {1, 1, 1};
    double lo[3] = {0, 0, 0}, cw[3] = {1, 1, 1};
    // graph (internal labels; `order` lists labels in spatial order = hub schedule)
    int64_t n_edges = 0;
    int32_t max_row = 0;
    DevBuf<int64_t> ptr;           // [n+1]
    DevBuf<int32_t> idx;           // [E]   (in-core only)
    DevBuf<uint8_t> bin, pix;      // [E]
    DevBuf<double> w;              // [n] weights by internal label
    DevBuf<int32_t> order;         // [n] label at spatial slot s
    DevBuf<int32_t> caller_of;     // [n] caller label of internal label (spatial mode), else empty
    // cell list kept for the dense cell-block rows (dense.cu; spatial mode): labels of cell c are
    // [cell_start[c], cell_start[c+1]); cell_of[label] = cell id
    DevBuf<int32_t> cell_start, cell_of;
    int64_t ncell = 0;
    GrDense dn;                    // dense rows + per-cell layout tables (built on first use by the gather kernel)
    // row statistics for the slot-table 3pCF kernel (query3.cu; k_row_stats in build_graph.cu): for page
    // size 2^s labels (s = GR_S_MIN .. GR_S_MAX), the longest page table and the most pages a row touches
    int32_t max_ptl[16] = {0};
    int32_t max_pages[16] = {0};
    int stats_done = 0;
    // 4pCF: raw 6-tuple -> (canonical configuration id | chirality code << 24), and configuration id -> dense
    // index; built on the device at the first 4pCF call (query4.cu)
    DevBuf<uint32_t> lut4;
    DevBuf<int32_t> dense4;
    int ncfg4 = 0;
    // out-of-core state: edge arrays in pinned host memory, cut into row-aligned windows
    uint64_t cap_bytes = 0;
    int ooc = 0;
    std::vector<GrWindow> windows;
    std::vector<uint8_t> need;     // [W*W] need[h*W+c] = 1 iff some edge (i,j) has i in window h, j in window c
    // (the pinned host arrays hang off the windows: GrWindow::h_block)
    // timing of the last calls
    double t_build_ms = 0, t_query_ms = 0, t_enum_ms = 0, n_launches = 0, staged_bytes = 0;
};

// Hit budget after which a kernel drains its shared-memory uint32 histogram into the global uint64 one (bins must
// not wrap).  The defaults are reached only by the largest workloads; the parity tests set the environment
// variable GRAMSCI_FLUSH_BUDGET (read at every query) to a few thousand so that every kernel variant drains many
// times on small inputs and is compared bin by bin with the oracle.
unsigned long long gr_flush_budget(unsigned long long dflt);

// opt the kernel in to `smem` bytes of dynamic shared memory and return its resident CTAs per SM; both driver calls
// are cached per (device, kernel, size) -- they cost a few hundred microseconds per query otherwise (api.cu)
int gr_kernel_occupancy(const void *fn, int threads, size_t smem);

// page-locked host memory for the out-of-core windows (api.cu): anonymous mapping, pages touched by all
// host cores, then cudaHostRegister -- cudaHostAlloc pins at 2.6 GiB/s on this box, this path at ~25 GiB/s
// Freed blocks go to a process-wide cache (like the device pool, so that the next capped build does not pin 42 GB
// again); gramsci_release_memory() unpins and unmaps them.  gr_pinned_alloc_nothrow is for the build's background
// pinning thread (error text returned instead of the thread-local error state); `*bytes` is rounded up to the block
// actually handed out, which is what gr_pinned_free takes back.
void *gr_pinned_alloc_nothrow(size_t *bytes, std::string *err);
void *gr_pinned_alloc(size_t *bytes);
void gr_pinned_free(void *p, size_t bytes);
void gr_pinned_release_cache();

// ---- build_graph.cu -----------------------------------------------------------------------------
void gr_build(gramsci_graph *g, const double *d_points, const double *d_weights, int n_windows_forced);
void gr_row_stats(gramsci_graph *g);
void gr_export_csr(const gramsci_graph *g, int64_t *d_ptr, int32_t *d_idx, uint8_t *d_bin, uint8_t *d_pix);
void gr_exclusive_scan_i32(const int32_t *d_in, int64_t n, int32_t *d_out /*[n+1]*/, cudaStream_t st);

// ---- query kernels ----------------------------------------------------------------------------
// Device views handed to the enumeration kernels: hub rows come from (idx_h,bin_h,pix_h) holding
// edges [e0_h, ...), spoke rows from (idx_c,...) holding edges [e0_c, ...); only spokes with label
// in [c_lo,c_hi) are processed (the out-of-core tile rule).
struct GrView {
    const int64_t *ptr;
    const int32_t *idx_h; const uint8_t *bin_h; const uint8_t *pix_h; int64_t e0_h;
    const int32_t *idx_c; const uint8_t *bin_c; const uint8_t *pix_c; int64_t e0_c;
    int32_t h_lo, h_hi;     // hub rows of this tile (labels), already cut to the hubs the graph owns (slab graphs)
    int32_t win_h;          // index of the hub window of this tile (0 in-core)
    int32_t c_lo, c_hi;     // resident search rows (labels)
    // 4pCF under a memory cap: a SECOND resident search window; a tile (h, c1 <= c2) takes the tetrahedra
    // (i, j1, j2, j3) with i in h, j1 in [c_lo,c_hi) and j2 in [c2_lo,c2_hi).  In-core: the same arrays as idx_c.
    const int32_t *idx_c2; const uint8_t *bin_c2; int64_t e0_c2;
    int32_t c2_lo, c2_hi;
    const int32_t *order;   // hub schedule (labels in spatial order), [n]
    int32_t s_lo, s_hi;     // schedule slots to walk (in-core: [0,n))
    const double *w;        // weights by label or nullptr
    int32_t hub_stride;     // > 1: only hubs with label % hub_stride == 0
    int32_t shard_count, shard_index;   // shard_count > 1: only hubs with label % shard_count == shard_index
    // dense cell-block rows of the resident search rows (gather kernel): row of label j at dense + rowaddr(j) - d0
    const uint8_t *dense; int64_t d0;
    int64_t dense_span;     // bytes of dense rows behind `dense` (bounds checks of the debug build, -DG3_BOUNDS=1)
};

void gr_2pcf(gramsci_graph *g, uint64_t *d_counts, double *d_wsum);
void gr_3pcf(gramsci_graph *g, uint64_t *d_counts, double *d_wsum, int equilateral = 0);
void gr_4pcf(gramsci_graph *g, int parity, uint64_t *d_even_c, int64_t *d_odd_c, double *d_even_w, double *d_odd_w);
void gr_work_counters(gramsci_graph *g, uint64_t *spoke_elems, uint64_t *tail_elems);

// dense.cu: layout tables + dense rows (in-core) for the gather kernel; returns false when not applicable
bool gr_dense_prepare(gramsci_graph *g);
bool gr_dense_tables(gramsci_graph *g);                 // layout tables only (what a capped build needs)
void gr_dense_rowaddrs(gramsci_graph *g, const int32_t *h_rows, int nrows, int64_t *h_out);
// expand the CSR rows [row_lo,row_hi) (edge arrays starting at edge e0) into dense rows at `out` (= row row_lo)
// (`out` + rowaddr(row) - d0 is where a row lands; the first out_bytes bytes of `out` are reset to 0xFF)
void gr_dense_expand(gramsci_graph *g, int32_t row_lo, int32_t row_hi, const int32_t *idx, const uint8_t *bin, int64_t e0,
                     uint8_t *out, int64_t d0, int64_t out_bytes, cudaStream_t st);
void gr_dense_units(gramsci_graph *g, GrUnits &u, int max_hubs, int len_lo, int len_hi);
void gr_dense_tile_units(gramsci_graph *g, GrUnits &u, long long tile_bytes);
// query3g.cu: the gather 3pCF kernel as a tile function
bool gr_gather_applicable(gramsci_graph *g, bool weighted, size_t hist_bytes, const char **why);
void gr_3pcf_gather(gramsci_graph *g, uint64_t *d_counts, double *d_wsum, int equilateral);
void gr_fold3(gramsci_graph *g, int nb, const unsigned long long *raw_cnt, const double *raw_w, int n_slots,
              uint64_t *d_counts, double *d_wsum);
template <typename InT, typename OutT>
void gr_exclusive_scan(const InT *d_in, int64_t n, OutT *d_out, cudaStream_t st);

// tiler.cu: run `tile_fn(view)` over every needed (hub window, search window) tile
struct GrTileRunner;
typedef void (*gr_tile_fn)(gramsci_graph *g, const GrView &v, void *user, cudaStream_t st);
// hub_only: visit each hub window once with no search window (2pCF sweep, work counters)
// pair_search: tiles are (hub window h, search windows c1 <= c2) -- the 4pCF tiling of P:159 (three resident windows)
void gr_for_each_tile(gramsci_graph *g, bool need_pix, bool hub_only, gr_tile_fn fn, void *user, bool need_dense = false,
                      bool pair_search = false);
int gr_tiler_slots(const gramsci_graph *g, bool need_pix, bool need_dense);

// host helpers (canon.cpp part of api.cu)
int gr_canon4(int nb, const int t[6], int c[6]);   // returns chirality factor
int64_t gr_num_configs4(int nb);

struct GrTimer {
    cudaEvent_t a = nullptr, b = nullptr;
    cudaStream_t st;
    explicit GrTimer(cudaStream_t s) : st(s) {
        cudaEventCreate(&a);
        cudaEventCreate(&b);
        cudaEventRecord(a, st);
    }
    double stop() {
        cudaEventRecord(b, st);
        cudaEventSynchronize(b);
        float ms = 0;
        cudaEventElapsedTime(&ms, a, b);
        return ms;
    }
    ~GrTimer() {
        if (a) cudaEventDestroy(a);
        if (b) cudaEventDestroy(b);
    }
};
