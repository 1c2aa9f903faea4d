/*
 * gramsci.h -- C ABI of the B200-native GRAMSCI-style N-point correlation query engine.
 *
 * Citations: P:<n> = PAPER.md line n (arxiv/paper_2607_06604); S:8(c) A-k = SURVEY.md section 8(c)
 * reading k (all restated in DESIGN.md section 3).
 *
 * The library computes, on one CUDA device (sm_100a), binned counts of the 2-, 3- and 4-cliques of
 * the radius graph of a point catalogue, and the parity-decomposed 4-clique counts
 * (P:91-101).  Every step runs in hand-written CUDA kernels; there is no CPU fallback: a call on a
 * machine without a usable CUDA device returns GRAMSCI_ECUDA.
 *
 * POINTERS.  Every data pointer (points, weights, output histograms) may be a DEVICE pointer or a
 * HOST pointer (pageable or pinned); the library asks the CUDA runtime which one it was given
 * (cudaPointerGetAttributes) and stages host buffers through device scratch itself.  `box` and all
 * scalar out-parameters are always HOST pointers.
 *
 * OWNERSHIP.  The caller owns points, weights and every output buffer.  The library owns the graph
 * (opaque handle) and all scratch, and releases them in gramsci_free_graph.  points/weights may be
 * freed as soon as gramsci_build_graph returns (weights are copied, coordinates discarded).
 *
 * OUTPUTS are overwritten (not accumulated) and are complete when the call returns (the call
 * enqueues on the graph's stream and synchronises that stream before returning).  Any output
 * pointer may be NULL to skip that channel.  Layout: dense row-major [nb]^3, index (b1*nb+b2)*nb+b3
 * or [nb]^6 in the order (b12,b13,b14,b23,b24,b34); populated ONLY at canonical configurations
 * (3pCF: sorted triple b1<=b2<=b3, A-5; 4pCF: lexicographic minimum over the 24 vertex orders, A-7),
 * zero elsewhere.
 *
 * ERRORS.  Every function returns a gramsci_status; nothing throws or aborts across the ABI; on
 * failure no output is written.  gramsci_last_error() gives a thread-local message.
 *
 * DETERMINISM.  Unweighted counts are exact integers, identical run to run and with or without a
 * device-memory cap.  Weighted fp64 sums may differ in the last bits with atomic order.
 *
 * THREADS.  The library keeps no process-global device state: build parameters and bin edges travel as
 * kernel arguments, scratch is allocated per call.  Calls on DIFFERENT graphs may run concurrently from
 * different host threads (each on its graph's stream); calls on the SAME graph must be serialised by the
 * caller (a query records its timings and scratch in the graph, which is why the handle is not const
 * in effect).  gramsci_last_error() is thread-local.
 *
 * DEVICE MEMORY.  The graph and all scratch come from the caller's allocator when gramsci_options.alloc /
 * dealloc are set (the Python binding can pass PyTorch's caching allocator), else from a private
 * stream-ordered memory pool of the device (never the device's default pool), which keeps freed blocks
 * for the next call; gramsci_release_memory() returns them to the driver.  HOST MEMORY: only capped graphs use it
 * (one page-locked block per window); freed blocks stay page-locked in a process-wide cache for the next capped
 * build until gramsci_release_memory().
 *
 * ENVIRONMENT (test and ablation knobs, read at query time; none is needed for normal use):
 *   GRAMSCI_FLUSH_BUDGET=n   drain the shared-memory histograms every n hits (parity tests force the drain paths)
 *   GRAMSCI_CTA_KMAJOR=0     long-row gather kernel in its first loop order (one spoke per warp)
 *   GRAMSCI_TILE_MB=n        spoke-tile size of the long-row gather kernel (default 64; forces tiling)
 *   GRAMSCI_WMODE=1          weighted 3pCF sums as fixed-point limbs in shared memory instead of fp64 RED
 *   GRAMSCI_4PCF_LUT=1       4pCF through the configuration look-up table and shared-memory histograms
 *   GRAMSCI_OCC=n, GRAMSCI_CARVEOUT=p, GRAMSCI_HYBRID=1, GRAMSCI_GATHER_G=g   occupancy / carve-out / path experiments
 *   GRAMSCI_TRIM_ON_FREE=1   trim the private device pool to 2 GiB when a graph larger than 4 GiB is freed
 *   GRAMSCI_DEBUG=1          one line per query on stderr (kernel choice, sizes)
 */
#ifndef GRAMSCI_H
#define GRAMSCI_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gramsci_graph gramsci_graph; /* opaque, owned by the library */

typedef enum {
    GRAMSCI_OK = 0,
    GRAMSCI_EINVAL = 1,    /* bad pointer / size / nbins / radii / unsupported combination         */
    GRAMSCI_ERANGE = 2,    /* periodic box with r_max >= min(box)/2 (A-4), or a row too long for smem */
    GRAMSCI_ENOMEM = 3,    /* device or host allocation failed, or device_mem_cap_bytes too small    */
    GRAMSCI_ECUDA = 4,     /* CUDA runtime error, or no CUDA device (see gramsci_last_error)         */
    GRAMSCI_EOVERFLOW = 5  /* N >= 2^31                                                              */
} gramsci_status;

/* 3pCF intersection kernel variants (S:8(f) rank 2 ablation). 0 picks the default. */
enum {
    GRAMSCI_ALGO_DEFAULT = 0,
    GRAMSCI_ALGO_MERGEPATH = 1, /* merge-path partitioned two-pointer walk (P:57-70 on a warp), hub row staged by TMA */
    GRAMSCI_ALGO_BSEARCH = 2,   /* lane-parallel binary search of N+(j) in the hub tail */
    GRAMSCI_ALGO_BITMAP = 3,    /* hub row scattered into a shared-memory slot table, O(1) membership;
                                   the default when the table fits (labels in cell order)               */
    GRAMSCI_ALGO_TABLE_G1 = 4,  /* slot table with a forced number of warps per hub: 1, 2, 4, 8          */
    GRAMSCI_ALGO_TABLE_G2 = 5,
    GRAMSCI_ALGO_TABLE_G4 = 6,
    GRAMSCI_ALGO_TABLE_G8 = 7,
    GRAMSCI_ALGO_GATHER = 8,    /* dense cell-block rows + hub-tail gather (needs spatial labels); the default
                                   when it applies                                                          */
    GRAMSCI_ALGO_MAX = 8
};

typedef struct {       /* zero-initialised struct == defaults */
    void *stream;                  /* cudaStream_t to run on (e.g. torch's current stream); NULL = default stream */
    uint64_t device_mem_cap_bytes; /* 0 = keep the whole CSR resident; else the edge arrays live in pinned
                                      host memory and are streamed through device windows of at most this
                                      many bytes in total (out-of-core tiler)                   */
    int want_pixels;               /* 1 = also store the direction-pixel byte per edge (needed by
                                      gramsci_4pcf_parity); forces caller-label order (A-10)         */
    int relabel;                   /* 0 = default (spatial relabelling unless want_pixels), 1 = force
                                      spatial (cell-order) labels, 2 = force caller labels                 */
    int algo;                      /* GRAMSCI_ALGO_* for gramsci_3pcf                                      */
    int n_windows;                 /* out-of-core only: force this many row windows (0 = derive from cap);
                                      the paper's env-var override, P:159                                 */
    int hub_stride;                /* > 1: enumerate only tuples whose smallest-label vertex i has i % hub_stride
                                      == 0 (a sampled partial result, for checking full-size runs against a
                                      reference that is too slow to run in full).  The label is the INTERNAL
                                      one: the caller's with relabel = 2 / want_pixels, else the cell-order label
                                      that gramsci_export_labels returns                                   */
    int shard_count, shard_index;  /* shard_count > 1: this graph's queries enumerate only the tuples whose hub (the
                                      vertex with the smallest internal label) has label % shard_count ==
                                      shard_index.  The shards partition the tuples: the histograms of shards
                                      0..shard_count-1 add up to the full result, exactly for counts -- one GPU
                                      per shard and one all-reduce of the histogram (S:8(e)); 2pCF is not sharded */
    int slab_count, slab_index;    /* slab_count > 1 (spatial labels only): SLAB + HALO partition for one GPU per slab
                                      (S:8(e), "one hub window per device ... no communication between
                                      tiles").  The cells (in id order = z-slabs of the grid) are cut into slab_count
                                      contiguous ranges of equal estimated work (sum of squared row lengths); this
                                      graph OWNS the hubs of range slab_index and stores only the rows of its own
                                      cells and of the cells its hubs' neighbours lie in (the forward stencil: the
                                      halo) -- every other row is empty, so memory is ~1/slab_count + halo.  All
                                      slabs must be built from the same points in the same order.  The histograms of
                                      the slabs add up to the full result (exactly for counts): one all-reduce.
                                      2pCF counts the edges stored at owned hubs.  Not combinable with shard_count */
    int reserved;                  /* must be 0 */
    /* Device allocator hooks (S:8(b)): both or neither.  alloc returns a DEVICE pointer valid on `stream`
       (256-byte aligned) or NULL; dealloc releases it.  NULL = the library's private memory pool.       */
    void *(*alloc)(size_t bytes, void *stream, void *user);
    void (*dealloc)(void *ptr, void *stream, void *user);
    void *user;
} gramsci_options;

/*
 * Build the radius graph (S:8(a) A1-A5): edge {i,j} iff r_min <= d(i,j) < r_max (A-2), d the
 * Euclidean distance, minimum image per axis when periodic (A-4).  Stored oriented (each edge once,
 * at its lower internal label, A-15) as CSR: ptr int64 [N+1], idx int32 [E] sorted ascending within a
 * row (Eq. 1), bin uint8 [E] = index of the equal-width bin of [r_min,r_max) (A-3: squared
 * distances compared with squared bin edges, no FMA contraction), pix uint8 [E] (A-8) if want_pixels.
 *
 *   points   [N,3] fp64 row-major x,y,z; inside [0,box) per axis when periodic.   HOST or DEVICE.
 *   weights  [N] fp64 (any sign) or NULL = unit weights.                            HOST or DEVICE.
 *   box      HOST double[3] periodic side lengths; NULL or any entry <= 0 = open (non-periodic).
 *   nbins    1..255 (bin index is one byte).
 * Errors: EINVAL (NULL points with N>0, nbins, r_min<0, r_max<=r_min), ERANGE (r_max >= box/2),
 * EOVERFLOW (N >= 2^31), ENOMEM, ECUDA.  On error *out is NULL.
 */
int gramsci_build_graph(const double *points, const double *weights, int64_t N, const double *box,
                        double r_min, double r_max, int nbins, const gramsci_options *opt,
                        gramsci_graph **out);

/* Sizes of a built graph (all out-pointers HOST, any may be NULL). csr_bytes = 5E (+E with pixels).
 * n_edges counts the STORED edges (a slab graph stores the rows of its slab and halo only). */
int gramsci_graph_info(const gramsci_graph *g, int64_t *n_points, int64_t *n_edges, int32_t *max_row,
                       uint64_t *csr_bytes, int32_t *n_windows);

/*
 * Copy the CSR out in CALLER labels (for graph-level parity tests): row i = caller point i, holding
 * the caller labels j > i of its neighbours, ascending.  ptr int64 [N+1], idx int32 [E], bin uint8 [E],
 * pix uint8 [E] (only if built with want_pixels, else untouched).  HOST or DEVICE; any may be NULL.
 * With spatial relabelling the library converts (re-orients and re-sorts) on the device.
 * Not available for graphs built under a device-memory cap (GRAMSCI_EINVAL).
 */
int gramsci_export_csr(const gramsci_graph *g, int64_t *ptr, int32_t *idx, uint8_t *bin, uint8_t *pix);

/* Internal label -> caller label (HOST or DEVICE int32 [N]): caller_of[l] is the index, in the caller's points
 * array, of the point with internal label l.  Identity when the graph keeps caller labels.  With it a caller can
 * reproduce the internal order (hub_stride, shard_* and the hub of a tuple are defined on internal labels). */
int gramsci_export_labels(const gramsci_graph *g, int32_t *caller_of);

/* 2pCF sweep (S:8(a) A6): counts[b] = #edges in bin b, wsum[b] = sum w_i w_j.  [nb] each. */
int gramsci_2pcf(const gramsci_graph *g, uint64_t *counts, double *wsum);

/* 3pCF (S:8(a) A7, A10): every 3-clique once; counts/wsum [nb^3] at sorted triples. */
int gramsci_3pcf(const gramsci_graph *g, uint64_t *counts, double *wsum);

/* Equilateral 3pCF (P:135, P:257 name it as one of the four query kernels; S:8(f)-3): the 3-cliques whose three
 * edges fall in the SAME radial bin, counts/wsum [nb] indexed by that bin -- the diagonal b1 = b2 = b3 of
 * gramsci_3pcf, but enumerated with the restriction inside the kernel: for a hub-spoke pair (i,j) only neighbours k
 * with b_ik == b_ij are followed, and only edges (j,k) with b_jk == b_ij count. */
int gramsci_3pcf_equilateral(const gramsci_graph *g, uint64_t *counts, double *wsum);

/* 4pCF (S:8(a) A8, A10): every 4-clique once; [nb^6] at canonical 6-tuples.
 * Requires nbins <= 16, rows shorter than 65536 entries and a resident graph (no device-memory cap:
 * GRAMSCI_EINVAL otherwise). */
int gramsci_4pcf(const gramsci_graph *g, uint64_t *counts, double *wsum);

/* Parity-decomposed 4pCF (Eq. 3; S:8(a) A9; A-8..A-11): even == gramsci_4pcf; odd adds
 * s = chi(raw tuple) * sign(V) per 4-clique, V from the pixel-centre unit vectors of the three spokes
 * of the smallest-caller-label vertex, s = 0 when |V| < 1e-9 or the configuration is achiral at bin
 * resolution.  Requires a graph built with want_pixels = 1 and nbins <= 16.  [nb^6] each. */
int gramsci_4pcf_parity(const gramsci_graph *g, uint64_t *even_counts, int64_t *odd_counts,
                        double *even_wsum, double *odd_wsum);

/* Number of canonical configurations (3pCF: C(nb+2,3); 4pCF: S4 orbits of bin 6-tuples): 220, 680,
 * 276, ....  Host-only arithmetic. */
int gramsci_num_configs(int npoint /*3|4*/, int nbins, int64_t *n);

/* Gather a dense HOST histogram (elem_bytes = 8) into the lexicographic list of canonical
 * configurations: compact [n_configs] (same element type), config_bins uint8 [n_configs, 3|6].
 * Host-only; either output may be NULL. */
int gramsci_compact(int npoint, int nbins, const void *dense, int elem_bytes, void *compact,
                    uint8_t *config_bins);

/* Disconnected 4pCF, Eq. 4: out[c] = xi(c12)xi(c34) + xi(c13)xi(c24) + xi(c14)xi(c23) on every
 * dense index; xi HOST [nb] -> out HOST [nb^6].  Host-only post-process (S:8(a) "tiny"). */
int gramsci_zeta_disc(int nbins, const double *xi, double *out);

/* Device time (ms, CUDA events on the graph's stream) of the kernels of the most recent call on this
 * graph: what = 0 build (all build kernels), 1 last query total, 2 last query's enumeration kernel(s)
 * only, 3 number of kernel launches of the last call (as a double), 4 out-of-core: bytes staged H2D. */
int gramsci_last_timing(const gramsci_graph *g, int what, double *value);

/* Exact work counters of the 3pCF on this graph (device pre-pass; S:8(d)): spoke_elems = sum over
 * oriented edges (i,j) of len(N+(j)); tail_elems = sum of len(tail_i(j)).  HOST out-pointers. */
int gramsci_work_counters(const gramsci_graph *g, uint64_t *spoke_elems, uint64_t *tail_elems);

/* The hubs a graph owns, as a range [hub_lo, hub_hi) of INTERNAL labels (out-pointers HOST): the whole catalogue
 * [0, N) unless the graph was built with slab_count > 1. */
int gramsci_slab_range(const gramsci_graph *g, int32_t *hub_lo, int32_t *hub_hi);

/*
 * The 2pCF sweep WITHOUT ANY ALLOCATION (csrc/noalloc.cu), for callers that cannot call cudaMalloc: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it.  Same result as gramsci_2pcf.  The accumulators live in a static
 * device array of GRAMSCI_NOALLOC_MAX_BINS bins (2 KB, held by every GPU that loads the library until exit).
 *   - counts [nb] uint64, wsum [nb] fp64: DEVICE buffers on the current device (either may be NULL); host buffers are
 *     rejected (staging them would allocate).  The graph must be resident (no device_mem_cap_bytes) and on the current
 *     device.  EINVAL with a message for nbins > GRAMSCI_NOALLOC_MAX_BINS, capped graphs, host outputs.
 *   - The call ENQUEUES memset + kernel + copies on the graph's stream and does NOT synchronise (no allocation, no event,
 *     no synchronisation: capturable): the outputs are complete once that stream has been synchronised by the caller.
 *     The first call on a device looks up the array's address (cudaGetSymbolAddress): make it once outside a capture.
 *   - All calls on a device share the array (cleared at the start of each call): calls that overlap on the GPU -- different
 *     streams with no ordering between them -- race on it.  Calls on one stream, one after the other, are safe.
 */
#define GRAMSCI_NOALLOC_MAX_BINS 128
int gramsci_2pcf_noalloc(const gramsci_graph *g, uint64_t *counts, double *wsum);

void gramsci_free_graph(gramsci_graph *g);

/* Return the freed blocks of the library's private memory pool on the current device to the driver and unpin the
 * cached host blocks (synchronises the device).  Nothing is returned automatically: a freed graph's memory serves
 * the next build (re-growing the pool for a 108 GB graph costs 2.6 s); call this before handing the device to
 * another allocator.  GRAMSCI_TRIM_ON_FREE=1 restores trimming to 2 GiB whenever a graph larger than 4 GiB is freed. */
int gramsci_release_memory(void);

const char *gramsci_last_error(void); /* thread-local, never NULL */

#ifdef __cplusplus
}
#endif
#endif /* GRAMSCI_H */
