// api.cu -- the C ABI of include/gramsci.h: argument checks, host/device pointer staging, error
// plumbing, and the small host-only helpers (configuration enumeration, Eq. 4 post-process).
#include "internal.cuh"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <thread>
#include <tuple>
#include <vector>
#include <algorithm>
#include <sys/mman.h>

// ---- errors --------------------------------------------------------------------------------------------
static thread_local char t_err[512] = "";

void gr_set_error(const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(t_err, sizeof t_err, fmt, ap);
    va_end(ap);
}

extern "C" const char *gramsci_last_error(void) { return t_err; }

#define GR_API_BEGIN try {
#define GR_API_END                                                        \
    }                                                                     \
    catch (const GrFail &f) { cudaGetLastError(); return f.code; }        \
    catch (const std::bad_alloc &) { gr_set_error("host allocation failed"); return GRAMSCI_ENOMEM; } \
    catch (...) { gr_set_error("unexpected internal error"); return GRAMSCI_ECUDA; }                  \
    return GRAMSCI_OK;

// ---- allocation context / private memory pool ----------------------------------------------------------------
GrAllocCtx &gr_alloc_ctx()
{
    static thread_local GrAllocCtx ctx;
    return ctx;
}

// one private pool per device (nullptr = pools unsupported on that device: plain cudaMalloc)
static std::mutex g_pool_mu;
static std::map<int, cudaMemPool_t> g_pools;

static cudaMemPool_t gr_pool(int dev)
{
    std::lock_guard<std::mutex> lk(g_pool_mu);
    auto it = g_pools.find(dev);
    if (it != g_pools.end()) return it->second;
    cudaMemPool_t pool = nullptr;
    int ok = 0;
    if (cudaDeviceGetAttribute(&ok, cudaDevAttrMemoryPoolsSupported, dev) == cudaSuccess && ok) {
        cudaMemPoolProps props;
        memset(&props, 0, sizeof props);
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        if (cudaMemPoolCreate(&pool, &props) == cudaSuccess) {
            uint64_t thr = UINT64_MAX;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
        } else {
            pool = nullptr;
        }
    }
    cudaGetLastError();
    g_pools[dev] = pool;
    return pool;
}

// device memory a new allocation of the library can draw on: what the driver reports free plus the freed blocks cached
// in the private pool
size_t gr_dev_available()
{
    size_t fr = 0, tot = 0;
    if (cudaMemGetInfo(&fr, &tot) != cudaSuccess) { cudaGetLastError(); return 0; }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return fr;
    cudaMemPool_t pool = gr_pool(dev);
    if (pool) {
        uint64_t res = 0, used = 0;
        if (cudaMemPoolGetAttribute(pool, cudaMemPoolAttrReservedMemCurrent, &res) == cudaSuccess &&
            cudaMemPoolGetAttribute(pool, cudaMemPoolAttrUsedMemCurrent, &used) == cudaSuccess && res > used)
            fr += (size_t)(res - used);
        cudaGetLastError();
    }
    return fr;
}

void *gr_dev_alloc(size_t bytes, const GrAllocCtx &ctx, int *kind)
{
    void *p = nullptr;
    if (ctx.alloc) {
        p = ctx.alloc(bytes, (void *)ctx.stream, ctx.user);
        if (!p) GR_FAIL(GRAMSCI_ENOMEM, "the caller's allocator returned NULL for %zu bytes", bytes);
        *kind = 2;
        return p;
    }
    int dev = 0;
    GR_CUDA(cudaGetDevice(&dev));
    cudaMemPool_t pool = gr_pool(dev);
    if (pool) {
        cudaError_t e = cudaMallocFromPoolAsync(&p, bytes, pool, ctx.stream);
        if (e == cudaErrorMemoryAllocation) {
            // cached free blocks that do not fit this request (another size mix than the last graph's): give them back
            // to the driver and try once more
            cudaGetLastError();
            cudaStreamSynchronize(ctx.stream);
            cudaMemPoolTrimTo(pool, 0);
            e = cudaMallocFromPoolAsync(&p, bytes, pool, ctx.stream);
        }
        GR_CUDA(e);
        *kind = 1;
    } else {
        GR_CUDA(cudaMalloc(&p, bytes));
        *kind = 0;
    }
    return p;
}

void gr_dev_free(void *p, const GrAllocCtx &ctx, int kind)
{
    if (!p) return;
    if (kind == 2) { if (ctx.dealloc) ctx.dealloc(p, (void *)ctx.stream, ctx.user); }
    else if (kind == 1) cudaFreeAsync(p, ctx.stream);
    else cudaFree(p);
}

extern "C" int gramsci_release_memory(void)
{
    GR_API_BEGIN
    int dev = 0;
    GR_CUDA(cudaGetDevice(&dev));
    cudaMemPool_t pool = gr_pool(dev);
    if (pool) {
        GR_CUDA(cudaDeviceSynchronize());
        GR_CUDA(cudaMemPoolTrimTo(pool, 0));
    }
    gr_pinned_release_cache();
    GR_API_END
}

unsigned long long gr_flush_budget(unsigned long long dflt)
{
    const char *e = getenv("GRAMSCI_FLUSH_BUDGET");
    if (!e || !*e) return dflt;
    const unsigned long long v = strtoull(e, nullptr, 10);
    return (v >= 1 && v < dflt) ? v : dflt;
}

// ---- kernel attributes / occupancy, cached ---------------------------------------------------------------------
int gr_kernel_occupancy(const void *fn, int threads, size_t smem)
{
    static std::mutex mu;
    static std::map<std::tuple<int, const void *, size_t>, int> occ_cache;
    static std::map<std::pair<int, const void *>, size_t> smem_set;
    int dev = 0;
    GR_CUDA(cudaGetDevice(&dev));
    std::lock_guard<std::mutex> lk(mu);
    auto &cur = smem_set[std::make_pair(dev, fn)];
    if (smem > cur) {
        GR_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        cur = smem;
    }
    const auto key = std::make_tuple(dev, fn, smem);
    auto it = occ_cache.find(key);
    if (it != occ_cache.end()) return it->second;
    int occ = 0;
    GR_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, threads, smem));
    occ_cache[key] = occ;
    return occ;
}

// ---- page-locked host memory -------------------------------------------------------------------------------
namespace {
struct PinnedBlock { void *p; size_t bytes; };
std::mutex g_pin_mu;
std::vector<PinnedBlock> g_pin_cache;
}

void *gr_pinned_alloc_nothrow(size_t *bytes_io, std::string *err)
{
    size_t bytes = (*bytes_io + 4095) & ~size_t(4095);
    {   // smallest cached block that fits without wasting more than half of it
        std::lock_guard<std::mutex> lk(g_pin_mu);
        int best = -1;
        for (int k = 0; k < (int)g_pin_cache.size(); ++k)
            if (g_pin_cache[k].bytes >= bytes && g_pin_cache[k].bytes <= 2 * bytes + (size_t(1) << 20) &&
                (best < 0 || g_pin_cache[k].bytes < g_pin_cache[best].bytes)) best = k;
        if (best >= 0) {
            PinnedBlock b = g_pin_cache[best];
            g_pin_cache.erase(g_pin_cache.begin() + best);
            *bytes_io = b.bytes;
            return b.p;
        }
    }
    void *p = mmap(nullptr, bytes, PROT_READ | PROT_WRITE, MAP_PRIVATE | MAP_ANONYMOUS, -1, 0);
    if (p == MAP_FAILED) {
        if (err) *err = "out-of-core: cannot map " + std::to_string(bytes) + " bytes of host memory";
        return nullptr;
    }
    madvise(p, bytes, MADV_HUGEPAGE);
    unsigned nt = std::max(1u, std::min(32u, std::thread::hardware_concurrency()));
    if (bytes < (size_t(64) << 20)) nt = 1;
    std::vector<std::thread> th;
    const size_t chunk = ((bytes / nt) + 4095) & ~size_t(4095);
    for (unsigned t = 0; t < nt; ++t)
        th.emplace_back([=] {
            char *c = (char *)p;
            const size_t lo = std::min(bytes, (size_t)t * chunk), hi = std::min(bytes, lo + chunk);
            for (size_t o = lo; o < hi; o += 4096) c[o] = 0;
        });
    for (auto &t : th) t.join();
    cudaError_t e = cudaHostRegister(p, bytes, cudaHostRegisterDefault);
    if (e != cudaSuccess) {
        munmap(p, bytes);
        cudaGetLastError();
        if (err) *err = "out-of-core: cannot page-lock " + std::to_string(bytes) + " bytes of host memory (" + cudaGetErrorString(e) + ")";
        return nullptr;
    }
    *bytes_io = bytes;
    return p;
}

void *gr_pinned_alloc(size_t *bytes)
{
    std::string err;
    void *p = gr_pinned_alloc_nothrow(bytes, &err);
    if (!p) GR_FAIL(GRAMSCI_ENOMEM, "%s", err.c_str());
    return p;
}

void gr_pinned_free(void *p, size_t bytes)
{
    if (!p) return;
    std::vector<PinnedBlock> evict;
    {
        std::lock_guard<std::mutex> lk(g_pin_mu);
        g_pin_cache.push_back({p, (bytes + 4095) & ~size_t(4095)});
        // bound what stays page-locked: 64 GiB (one capped configs[4] graph is 42 GB); the oldest blocks go first
        size_t total = 0;
        for (auto &b : g_pin_cache) total += b.bytes;
        while (total > (size_t(64) << 30) && g_pin_cache.size() > 1) {
            evict.push_back(g_pin_cache.front());
            total -= g_pin_cache.front().bytes;
            g_pin_cache.erase(g_pin_cache.begin());
        }
    }
    for (auto &b : evict) {
        cudaHostUnregister(b.p);
        munmap(b.p, b.bytes);
    }
    if (!evict.empty()) cudaGetLastError();
}

void gr_pinned_release_cache()
{
    std::vector<PinnedBlock> blocks;
    {
        std::lock_guard<std::mutex> lk(g_pin_mu);
        blocks.swap(g_pin_cache);
    }
    for (auto &b : blocks) {
        cudaHostUnregister(b.p);
        munmap(b.p, b.bytes);
    }
    cudaGetLastError();
}

// ---- pointer staging -------------------------------------------------------------------------------------
static bool is_device_ptr(const void *p)
{
    cudaPointerAttributes a;
    cudaError_t e = cudaPointerGetAttributes(&a, p);
    if (e != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// read-only input: returns a device pointer (the caller's, or a staged copy owned by `hold`)
template <typename T>
static const T *stage_in(const T *p, size_t n, DevBuf<T> &hold, cudaStream_t st)
{
    if (!p || n == 0) return p;
    if (is_device_ptr(p)) return p;
    hold.alloc(n);
    GR_CUDA(cudaMemcpyAsync(hold.p, p, n * sizeof(T), cudaMemcpyHostToDevice, st));
    return hold.p;
}

// output: device scratch when the caller's buffer is on the host
template <typename T>
struct OutStage {
    T *user = nullptr, *dev = nullptr;
    size_t n = 0;
    bool host = false;
    DevBuf<T> hold;
    void init(T *p, size_t count) {
        user = p; n = count;
        if (!p) return;
        host = !is_device_ptr(p);
        if (host) { hold.alloc(count); dev = hold.p; } else dev = p;
    }
    void finish(cudaStream_t st) {
        if (user && host && n) {
            GR_CUDA(cudaMemcpyAsync(user, dev, n * sizeof(T), cudaMemcpyDeviceToHost, st));
            GR_CUDA(cudaStreamSynchronize(st));
        }
    }
};

static void require_device()
{
    int n = 0;
    cudaError_t e = cudaGetDeviceCount(&n);
    if (e != cudaSuccess || n <= 0) {
        cudaGetLastError();
        GR_FAIL(GRAMSCI_ECUDA, "no usable CUDA device (%s); this library has no CPU fallback",
                e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
    }
}

static int64_t ipow(int b, int e)
{
    int64_t r = 1;
    for (int k = 0; k < e; ++k) r *= b;
    return r;
}

// ---- build -------------------------------------------------------------------------------------------------
extern "C" int gramsci_build_graph(const double *points, const double *weights, int64_t N, const double *box,
                                   double r_min, double r_max, int nbins, const gramsci_options *opt,
                                   gramsci_graph **out)
{
    if (out) *out = nullptr;
    gramsci_graph *g = nullptr;
    GR_API_BEGIN
    if (!out) GR_FAIL(GRAMSCI_EINVAL, "build_graph: out is NULL");
    if (N < 0 || (N > 0 && !points)) GR_FAIL(GRAMSCI_EINVAL, "build_graph: bad points/N");
    if (N >= ((int64_t)1 << 31) - 1) GR_FAIL(GRAMSCI_EOVERFLOW, "build_graph: N >= 2^31");
    if (nbins < 1 || nbins > GR_MAXBINS) GR_FAIL(GRAMSCI_EINVAL, "build_graph: nbins must be in 1..255");
    if (!(r_min >= 0.0) || !(r_max > r_min) || !std::isfinite(r_max))
        GR_FAIL(GRAMSCI_EINVAL, "build_graph: need 0 <= r_min < r_max");
    gramsci_options o;
    memset(&o, 0, sizeof o);
    if (opt) o = *opt;
    if (o.relabel < 0 || o.relabel > 2 || o.algo < 0 || o.algo > GRAMSCI_ALGO_MAX || o.n_windows < 0 || o.hub_stride < 0 ||
        o.shard_count < 0 || o.shard_index < 0 || (o.shard_count > 1 && o.shard_index >= o.shard_count) ||
        o.slab_count < 0 || o.slab_index < 0 || (o.slab_count > 1 && o.slab_index >= o.slab_count) ||
        (o.slab_count > 1 && o.shard_count > 1))
        GR_FAIL(GRAMSCI_EINVAL, "build_graph: bad options");
    require_device();

    g = new gramsci_graph();
    g->n = N; g->nb = nbins; g->r_min = r_min; g->r_max = r_max;
    g->periodic = (box && box[0] > 0.0 && box[1] > 0.0 && box[2] > 0.0) ? 1 : 0;
    if (g->periodic)
        for (int c = 0; c < 3; ++c) {
            g->box[c] = box[c];
            if (!(r_max < 0.5 * box[c])) {
                delete g; g = nullptr;
                GR_FAIL(GRAMSCI_ERANGE, "build_graph: periodic box needs r_max < box/2 (A-4)");
            }
        }
    // squared bin edges (A-3): e_k = r_min + (k (r_max - r_min)) / nb, e_0 = r_min, e_nb = r_max; q_k = e_k^2.
    // volatile keeps every operation a separately rounded fp64 operation whatever the host flags.
    for (int k = 0; k <= nbins; ++k) {
        volatile double span = r_max - r_min;
        volatile double num = (double)k * span;
        volatile double quo = num / (double)nbins;
        volatile double e = r_min + quo;
        if (k == 0) e = r_min;
        if (k == nbins) e = r_max;
        volatile double q = e * e;
        g->q[k] = q;
    }
    g->weighted = weights ? 1 : 0;
    g->has_pix = o.want_pixels ? 1 : 0;
    g->spatial = (o.relabel == 1) ? 1 : (o.relabel == 2) ? 0 : (o.want_pixels ? 0 : 1);
    g->algo = o.algo;
    g->hub_stride = o.hub_stride > 1 ? o.hub_stride : 1;
    g->shard_count = o.shard_count > 1 ? o.shard_count : 1;
    g->shard_index = o.shard_count > 1 ? o.shard_index : 0;
    g->slab_count = o.slab_count > 1 ? o.slab_count : 1;
    g->slab_index = o.slab_count > 1 ? o.slab_index : 0;
    if (g->slab_count > 1 && !g->spatial) {
        delete g; g = nullptr;
        GR_FAIL(GRAMSCI_EINVAL, "build_graph: slab_count needs spatial (cell-order) labels: not with want_pixels / relabel = 2");
    }
    if (g->has_pix && g->spatial) {
        delete g; g = nullptr;
        GR_FAIL(GRAMSCI_EINVAL, "build_graph: want_pixels needs caller labels (A-10): relabel = 1 cannot be combined with it");
    }
    g->stream = (cudaStream_t)o.stream;
    g->cap_bytes = o.device_mem_cap_bytes;
    int dev = 0;
    GR_CUDA(cudaGetDevice(&dev));
    {   // two attributes, cached per device (cudaGetDeviceProperties costs milliseconds per call)
        static std::mutex mu;
        static std::map<int, std::pair<int, size_t>> cache;
        std::lock_guard<std::mutex> lk(mu);
        auto it = cache.find(dev);
        if (it == cache.end()) {
            int sms = 0, optin = 0;
            GR_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
            GR_CUDA(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
            it = cache.emplace(dev, std::make_pair(sms, (size_t)optin)).first;
        }
        g->sm_count = it->second.first;
        g->smem_optin = it->second.second;
    }

    if ((o.alloc != nullptr) != (o.dealloc != nullptr)) {
        delete g; g = nullptr;
        GR_FAIL(GRAMSCI_EINVAL, "build_graph: alloc and dealloc must be given together");
    }
    g->actx.stream = g->stream; g->actx.alloc = o.alloc; g->actx.dealloc = o.dealloc; g->actx.user = o.user;
    gr_alloc_ctx() = g->actx;
    DevBuf<double> hp, hw;
    const double *d_pts = stage_in(points, (size_t)N * 3, hp, g->stream);
    const double *d_w = stage_in(weights, (size_t)N, hw, g->stream);
    gr_build(g, d_pts, d_w, o.n_windows);
    GR_CUDA(cudaStreamSynchronize(g->stream));
    *out = g;
    g = nullptr;
    }
    catch (const GrFail &f) { cudaGetLastError(); if (g) gramsci_free_graph(g); return f.code; }
    catch (const std::bad_alloc &) { gr_set_error("host allocation failed"); if (g) gramsci_free_graph(g); return GRAMSCI_ENOMEM; }
    catch (...) { gr_set_error("unexpected internal error"); if (g) gramsci_free_graph(g); return GRAMSCI_ECUDA; }
    return GRAMSCI_OK;
}

extern "C" void gramsci_free_graph(gramsci_graph *g)
{
    if (!g) return;
    cudaStreamSynchronize(g->stream);
    for (auto &w : g->windows) { gr_pinned_free(w.h_block, w.h_block_bytes); w.h_block = nullptr; }
    // Freed blocks stay in the library's private pool for the next graph: growing the pool again costs more than the whole
    // build (configs[4]: 108 GB of graph, 2.6 s of a 12.7 s step went into re-growing a trimmed pool).  They are invisible to
    // other allocators (PyTorch's) until gramsci_release_memory(); GRAMSCI_TRIM_ON_FREE=1 trims to 2 GiB after graphs > 4 GiB.
    const bool trim = (uint64_t)g->n_edges * 5 > ((uint64_t)4 << 30) && !g->actx.alloc && getenv("GRAMSCI_TRIM_ON_FREE");
    cudaStream_t st = g->stream;
    delete g;
    if (trim) {
        int dev = 0;
        cudaStreamSynchronize(st);
        if (cudaGetDevice(&dev) == cudaSuccess) {
            cudaMemPool_t pool = gr_pool(dev);
            if (pool) cudaMemPoolTrimTo(pool, (size_t)2 << 30);
        }
        cudaGetLastError();
    }
}

extern "C" int gramsci_slab_range(const gramsci_graph *g, int32_t *hub_lo, int32_t *hub_hi)
{
    GR_API_BEGIN
    if (!g) GR_FAIL(GRAMSCI_EINVAL, "slab_range: graph is NULL");
    if (hub_lo) *hub_lo = std::max(0, g->hub_lo);
    if (hub_hi) *hub_hi = (int32_t)std::min<int64_t>(g->n, g->hub_hi);
    GR_API_END
}

extern "C" int gramsci_graph_info(const gramsci_graph *g, int64_t *n_points, int64_t *n_edges, int32_t *max_row,
                                  uint64_t *csr_bytes, int32_t *n_windows)
{
    GR_API_BEGIN
    if (!g) GR_FAIL(GRAMSCI_EINVAL, "graph_info: NULL graph");
    if (n_points) *n_points = g->n;
    if (n_edges) *n_edges = g->n_edges;
    if (max_row) *max_row = g->max_row;
    if (csr_bytes) *csr_bytes = (uint64_t)g->n_edges * (5 + (g->has_pix ? 1 : 0));
    if (n_windows) *n_windows = (int32_t)g->windows.size();
    GR_API_END
}

extern "C" int gramsci_export_csr(const gramsci_graph *g, int64_t *ptr, int32_t *idx, uint8_t *bin, uint8_t *pix)
{
    GR_API_BEGIN
    if (!g) GR_FAIL(GRAMSCI_EINVAL, "export_csr: NULL graph");
    gr_alloc_ctx() = g->actx;
    OutStage<int64_t> op; OutStage<int32_t> oi; OutStage<uint8_t> ob, ox;
    op.init(ptr, (size_t)g->n + 1);
    oi.init(idx, (size_t)g->n_edges);
    ob.init(bin, (size_t)g->n_edges);
    ox.init(g->has_pix ? pix : nullptr, (size_t)g->n_edges);
    gr_export_csr(g, op.dev, oi.dev, ob.dev, ox.dev);
    op.finish(g->stream); oi.finish(g->stream); ob.finish(g->stream); ox.finish(g->stream);
    GR_API_END
}

__global__ void k_iota(int32_t *out, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = (int32_t)i;
}

extern "C" int gramsci_export_labels(const gramsci_graph *g, int32_t *caller_of)
{
    GR_API_BEGIN
    if (!g) GR_FAIL(GRAMSCI_EINVAL, "export_labels: NULL graph");
    gr_alloc_ctx() = g->actx;
    OutStage<int32_t> o;
    o.init(caller_of, (size_t)g->n);
    if (caller_of && g->n > 0) {
        if (g->spatial)
            GR_CUDA(cudaMemcpyAsync(o.dev, g->caller_of.p, sizeof(int32_t) * g->n, cudaMemcpyDeviceToDevice, g->stream));
        else
            k_iota<<<(unsigned)((g->n + 255) / 256), 256, 0, g->stream>>>(o.dev, g->n);
        GR_CUDA(cudaGetLastError());
        GR_CUDA(cudaStreamSynchronize(g->stream));
    }
    o.finish(g->stream);
    GR_API_END
}

// ---- queries -----------------------------------------------------------------------------------------------
extern "C" int gramsci_2pcf(const gramsci_graph *cg, uint64_t *counts, double *wsum)
{
    GR_API_BEGIN
    gramsci_graph *g = const_cast<gramsci_graph *>(cg);
    if (!g) GR_FAIL(GRAMSCI_EINVAL, "2pcf: NULL graph");
    gr_alloc_ctx() = g->actx;
    OutStage<uint64_t> oc; OutStage<double> ow;
    oc.init(counts, (size_t)g->nb);
    ow.init(wsum, (size_t)g->nb);
    gr_2pcf(g, oc.dev, ow.dev);
    oc.finish(g->stream); ow.finish(g->stream);
    GR_API_END
}

extern "C" int gramsci_3pcf(const gramsci_graph *cg, uint64_t *counts, double *wsum)
{
    GR_API_BEGIN
    gramsci_graph *g = const_cast<gramsci_graph *>(cg);
    if (!g) GR_FAIL(GRAMSCI_EINVAL, "3pcf: NULL graph");
    gr_alloc_ctx() = g->actx;
    const size_t nh = (size_t)ipow(g->nb, 3);
    OutStage<uint64_t> oc; OutStage<double> ow;
    oc.init(counts, nh);
    ow.init(wsum, nh);
    gr_3pcf(g, oc.dev, ow.dev);
    oc.finish(g->stream); ow.finish(g->stream);
    GR_API_END
}

extern "C" int gramsci_3pcf_equilateral(const gramsci_graph *cg, uint64_t *counts, double *wsum)
{
    GR_API_BEGIN
    gramsci_graph *g = const_cast<gramsci_graph *>(cg);
    if (!g) GR_FAIL(GRAMSCI_EINVAL, "3pcf_equilateral: NULL graph");
    gr_alloc_ctx() = g->actx;
    OutStage<uint64_t> oc; OutStage<double> ow;
    oc.init(counts, (size_t)g->nb);
    ow.init(wsum, (size_t)g->nb);
    gr_3pcf(g, oc.dev, ow.dev, 1);
    oc.finish(g->stream); ow.finish(g->stream);
    GR_API_END
}

extern "C" int gramsci_4pcf(const gramsci_graph *cg, uint64_t *counts, double *wsum)
{
    GR_API_BEGIN
    gramsci_graph *g = const_cast<gramsci_graph *>(cg);
    if (!g) GR_FAIL(GRAMSCI_EINVAL, "4pcf: NULL graph");
    gr_alloc_ctx() = g->actx;
    if (g->nb > 16) GR_FAIL(GRAMSCI_EINVAL, "4pcf: nbins must be <= 16");
    const size_t nh = (size_t)ipow(g->nb, 6);
    OutStage<uint64_t> oc; OutStage<double> ow;
    oc.init(counts, nh);
    ow.init(wsum, nh);
    gr_4pcf(g, 0, oc.dev, nullptr, ow.dev, nullptr);
    oc.finish(g->stream); ow.finish(g->stream);
    GR_API_END
}

extern "C" int gramsci_4pcf_parity(const gramsci_graph *cg, uint64_t *even_counts, int64_t *odd_counts,
                                   double *even_wsum, double *odd_wsum)
{
    GR_API_BEGIN
    gramsci_graph *g = const_cast<gramsci_graph *>(cg);
    if (!g) GR_FAIL(GRAMSCI_EINVAL, "4pcf_parity: NULL graph");
    gr_alloc_ctx() = g->actx;
    if (g->nb > 16) GR_FAIL(GRAMSCI_EINVAL, "4pcf_parity: nbins must be <= 16");
    if (!g->has_pix || g->spatial)
        GR_FAIL(GRAMSCI_EINVAL, "4pcf_parity: graph must be built with want_pixels=1 in caller-label order (A-10)");
    const size_t nh = (size_t)ipow(g->nb, 6);
    OutStage<uint64_t> oc; OutStage<int64_t> oo; OutStage<double> ow, oow;
    oc.init(even_counts, nh);
    oo.init(odd_counts, nh);
    ow.init(even_wsum, nh);
    oow.init(odd_wsum, nh);
    gr_4pcf(g, 1, oc.dev, oo.dev, ow.dev, oow.dev);
    oc.finish(g->stream); oo.finish(g->stream); ow.finish(g->stream); oow.finish(g->stream);
    GR_API_END
}

extern "C" int gramsci_last_timing(const gramsci_graph *g, int what, double *value)
{
    GR_API_BEGIN
    if (!g || !value) GR_FAIL(GRAMSCI_EINVAL, "last_timing: NULL argument");
    switch (what) {
        case 0: *value = g->t_build_ms; break;
        case 1: *value = g->t_query_ms; break;
        case 2: *value = g->t_enum_ms; break;
        case 3: *value = g->n_launches; break;
        case 4: *value = g->staged_bytes; break;
        default: GR_FAIL(GRAMSCI_EINVAL, "last_timing: unknown selector %d", what);
    }
    GR_API_END
}

extern "C" int gramsci_work_counters(const gramsci_graph *cg, uint64_t *spoke_elems, uint64_t *tail_elems)
{
    GR_API_BEGIN
    gramsci_graph *g = const_cast<gramsci_graph *>(cg);
    if (!g) GR_FAIL(GRAMSCI_EINVAL, "work_counters: NULL graph");
    gr_alloc_ctx() = g->actx;
    gr_work_counters(g, spoke_elems, tail_elems);
    GR_API_END
}

// ---- canonical configurations (host; A-5, A-7, A-10) -------------------------------------------------------
// A 4-point configuration is the orbit of (b01,b02,b03,b12,b13,b23) under relabelling of the four
// vertices; its representative is the lexicographic minimum.  The chirality factor is 0 when
// the minimum is reached by vertex orders of both parities, else the parity of the orders reaching it.
static const int8_t kPerm4[24][4] = {
    {0,1,2,3},{0,1,3,2},{0,2,1,3},{0,2,3,1},{0,3,1,2},{0,3,2,1},{1,0,2,3},{1,0,3,2},{1,2,0,3},{1,2,3,0},
    {1,3,0,2},{1,3,2,0},{2,0,1,3},{2,0,3,1},{2,1,0,3},{2,1,3,0},{2,3,0,1},{2,3,1,0},{3,0,1,2},{3,0,2,1},
    {3,1,0,2},{3,1,2,0},{3,2,0,1},{3,2,1,0}};

int gr_canon4(int nb, const int t[6], int c[6])
{
    (void)nb;
    int m[4][4] = {{0}};
    m[0][1] = m[1][0] = t[0]; m[0][2] = m[2][0] = t[1]; m[0][3] = m[3][0] = t[2];
    m[1][2] = m[2][1] = t[3]; m[1][3] = m[3][1] = t[4]; m[2][3] = m[3][2] = t[5];
    bool have = false;
    int even = 0, odd = 0;
    for (int s = 0; s < 24; ++s) {
        const int8_t *p = kPerm4[s];
        int u[6] = {m[p[0]][p[1]], m[p[0]][p[2]], m[p[0]][p[3]], m[p[1]][p[2]], m[p[1]][p[3]], m[p[2]][p[3]]};
        int cmp = have ? 0 : -1;
        for (int e = 0; e < 6 && have && cmp == 0; ++e) cmp = (u[e] < c[e]) ? -1 : (u[e] > c[e]) ? 1 : 0;
        if (cmp < 0) { memcpy(c, u, sizeof u); have = true; even = odd = 0; cmp = 0; }
        if (cmp == 0) {
            int inv = 0;
            for (int a = 0; a < 4; ++a) for (int b = a + 1; b < 4; ++b) inv += (p[a] > p[b]);
            if (inv & 1) ++odd; else ++even;
        }
    }
    if (even && odd) return 0;
    return even ? 1 : -1;
}

static std::mutex g_cfg_mu;
static std::map<int, int64_t> g_cfg4;

int64_t gr_num_configs4(int nb)
{
    std::lock_guard<std::mutex> lk(g_cfg_mu);
    auto it = g_cfg4.find(nb);
    if (it != g_cfg4.end()) return it->second;
    int64_t n = 0;
    int t[6], c[6];
    const int64_t nh = ipow(nb, 6);
    for (int64_t x = 0; x < nh; ++x) {
        int64_t r = x;
        for (int e = 5; e >= 0; --e) { t[e] = (int)(r % nb); r /= nb; }
        gr_canon4(nb, t, c);
        if (memcmp(t, c, sizeof t) == 0) ++n;
    }
    g_cfg4[nb] = n;
    return n;
}

extern "C" int gramsci_num_configs(int npoint, int nbins, int64_t *n)
{
    GR_API_BEGIN
    if (!n || nbins < 1 || nbins > GR_MAXBINS) GR_FAIL(GRAMSCI_EINVAL, "num_configs: bad arguments");
    if (npoint == 3) *n = (int64_t)nbins * (nbins + 1) * (nbins + 2) / 6;
    else if (npoint == 4) {
        if (nbins > 16) GR_FAIL(GRAMSCI_EINVAL, "num_configs: 4-point needs nbins <= 16");
        *n = gr_num_configs4(nbins);
    } else GR_FAIL(GRAMSCI_EINVAL, "num_configs: npoint must be 3 or 4");
    GR_API_END
}

extern "C" int gramsci_compact(int npoint, int nbins, const void *dense, int elem_bytes, void *compact,
                               uint8_t *config_bins)
{
    GR_API_BEGIN
    if (nbins < 1 || nbins > GR_MAXBINS || elem_bytes != 8 || (compact && !dense))
        GR_FAIL(GRAMSCI_EINVAL, "compact: bad arguments");
    const uint64_t *src = (const uint64_t *)dense;
    uint64_t *dst = (uint64_t *)compact;
    int64_t k = 0;
    if (npoint == 3) {
        for (int a = 0; a < nbins; ++a) for (int b = a; b < nbins; ++b) for (int c = b; c < nbins; ++c) {
            if (dst) dst[k] = src[((int64_t)a * nbins + b) * nbins + c];
            if (config_bins) { config_bins[3 * k] = (uint8_t)a; config_bins[3 * k + 1] = (uint8_t)b; config_bins[3 * k + 2] = (uint8_t)c; }
            ++k;
        }
    } else if (npoint == 4) {
        if (nbins > 16) GR_FAIL(GRAMSCI_EINVAL, "compact: 4-point needs nbins <= 16");
        int t[6], c[6];
        const int64_t nh = ipow(nbins, 6);
        for (int64_t x = 0; x < nh; ++x) {
            int64_t r = x;
            for (int e = 5; e >= 0; --e) { t[e] = (int)(r % nbins); r /= nbins; }
            gr_canon4(nbins, t, c);
            if (memcmp(t, c, sizeof t) != 0) continue;
            if (dst) dst[k] = src[x];
            if (config_bins) for (int e = 0; e < 6; ++e) config_bins[6 * k + e] = (uint8_t)t[e];
            ++k;
        }
    } else GR_FAIL(GRAMSCI_EINVAL, "compact: npoint must be 3 or 4");
    GR_API_END
}

extern "C" int gramsci_zeta_disc(int nbins, const double *xi, double *out)
{
    GR_API_BEGIN
    if (nbins < 1 || nbins > 16 || !xi || !out) GR_FAIL(GRAMSCI_EINVAL, "zeta_disc: bad arguments");
    const int64_t nh = ipow(nbins, 6);
    for (int64_t x = 0; x < nh; ++x) {
        int b[6];
        int64_t r = x;
        for (int e = 5; e >= 0; --e) { b[e] = (int)(r % nbins); r /= nbins; }
        // (b12,b13,b14,b23,b24,b34): xi(r12)xi(r34) + xi(r13)xi(r24) + xi(r14)xi(r23)   (Eq. 4)
        out[x] = xi[b[0]] * xi[b[5]] + xi[b[1]] * xi[b[4]] + xi[b[2]] * xi[b[3]];
    }
    GR_API_END
}
