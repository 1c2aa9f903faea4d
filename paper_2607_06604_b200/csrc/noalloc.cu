// noalloc.cu -- gramsci_2pcf_noalloc: the 2pCF sweep (S:8(a) A6; "a single sweep of the graph") for callers that
// cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
//
// The regular path (gr_2pcf, query3.cu) takes its accumulators -- uint64 [nb] pair counts and fp64 [nb] weighted pair sums,
// filled with global atomics by all CTAs and copied to the caller's buffers afterwards -- from the library's memory pool.
// This variant keeps them in a file-scope __device__ array of GRAMSCI_NOALLOC_MAX_BINS bins (2 KB; every GPU that loads the
// library holds it until exit) and calls no cudaMalloc / cudaFree / pool routine, creates no event and does not
// synchronise: it enqueues  memset(scratch) -> k_2pcf_static -> copy to the caller's DEVICE buffers  on the graph's stream.
//
// `g_scratch` names a host-side stand-in in host code, not a device address: the kernel gets the address that
// cudaGetSymbolAddress returns, looked up once per device with that device current (scratch_of).
// All calls on a device share the array: it keeps the last call's contents (cleared at the start of every call), and two
// calls that overlap on the GPU (different streams, no ordering between them) race on it.
#include "internal.cuh"

#include <algorithm>
#include <mutex>

namespace {

constexpr int NA_MAX_BINS = GRAMSCI_NOALLOC_MAX_BINS;

// [uint64 counts NA_MAX_BINS][fp64 weighted sums NA_MAX_BINS]
static __device__ __align__(256) unsigned char g_scratch[NA_MAX_BINS * 16];

constexpr int NA_MAX_DEVICES = 64;
std::mutex g_mu;
unsigned char *g_addr[NA_MAX_DEVICES];      // device ordinal -> device address of g_scratch on that device (0 = not looked up)

// device address of the scratch array on the CURRENT device (set-up: once per device)
unsigned char *scratch_of(int dev)
{
    if (dev < 0 || dev >= NA_MAX_DEVICES) GR_FAIL(GRAMSCI_EINVAL, "2pcf_noalloc: device ordinal %d out of range", dev);
    std::lock_guard<std::mutex> lk(g_mu);
    if (g_addr[dev]) return g_addr[dev];
    unsigned char *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void **)&p, g_scratch);
    if (e != cudaSuccess || !p) {
        cudaGetLastError();
        GR_FAIL(GRAMSCI_ECUDA, "2pcf_noalloc: cudaGetSymbolAddress(scratch) failed on device %d: %s", dev, cudaGetErrorString(e));
    }
    g_addr[dev] = p;
    return p;
}

// the sweep of k_2pcf (query3.cu) with its global accumulators at `cnt` / `wsum` (the static scratch)
__global__ void __launch_bounds__(256)
k_2pcf_static(const int64_t *__restrict__ ptr, const int32_t *__restrict__ idx, const uint8_t *__restrict__ bin,
              const double *__restrict__ w, int32_t h_lo, int32_t h_hi, int nb, int weighted,
              unsigned long long *__restrict__ cnt, double *__restrict__ wsum)
{
    __shared__ unsigned int h_c[NA_MAX_BINS];
    __shared__ double h_w[NA_MAX_BINS];
    for (int t = threadIdx.x; t < nb; t += blockDim.x) { h_c[t] = 0; h_w[t] = 0.0; }
    __syncthreads();
    const int lane = threadIdx.x & 31;
    const int warps_total = gridDim.x * (blockDim.x >> 5);
    for (int64_t i = h_lo + (int64_t)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); i < h_hi; i += warps_total) {
        const int64_t rb = ptr[i], re = ptr[i + 1];
        const double wi = weighted ? w[i] : 1.0;
        for (int64_t e = rb + lane; e < re; e += 32) {
            const int b = bin[e];
            atomicAdd(&h_c[b], 1u);
            if (weighted) atomicAdd(&h_w[b], wi * w[idx[e]]);
        }
    }
    __syncthreads();
    for (int t = threadIdx.x; t < nb; t += blockDim.x) {
        if (h_c[t]) atomicAdd(&cnt[t], (unsigned long long)h_c[t]);
        if (weighted && h_w[t] != 0.0) atomicAdd(&wsum[t], h_w[t]);
    }
}

bool on_device(const void *p, int dev)
{
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return (a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged) && a.device == dev;
}

}  // namespace

extern "C" int gramsci_2pcf_noalloc(const gramsci_graph *g, uint64_t *counts, double *wsum)
{
    try {
        if (!g) GR_FAIL(GRAMSCI_EINVAL, "2pcf_noalloc: NULL graph");
        if (g->nb > NA_MAX_BINS)
            GR_FAIL(GRAMSCI_EINVAL, "2pcf_noalloc: %d bins exceed GRAMSCI_NOALLOC_MAX_BINS = %d (the static scratch); use gramsci_2pcf",
                    g->nb, NA_MAX_BINS);
        if (g->ooc)
            GR_FAIL(GRAMSCI_EINVAL, "2pcf_noalloc: the graph was built under a device-memory cap (its windows are staged through "
                                    "allocated buffers); use gramsci_2pcf");
        int dev = 0;
        GR_CUDA(cudaGetDevice(&dev));
        if (g->n > 0 && !on_device(g->ptr.p, dev))
            GR_FAIL(GRAMSCI_EINVAL, "2pcf_noalloc: the graph does not live on the current device (%d)", dev);
        if ((counts && !on_device(counts, dev)) || (wsum && !on_device(wsum, dev)))
            GR_FAIL(GRAMSCI_EINVAL, "2pcf_noalloc: outputs must be DEVICE buffers of the current device (staging a host buffer "
                                    "would allocate)");
        if (!counts && !wsum) return GRAMSCI_OK;
        cudaStream_t st = g->stream;
        unsigned char *sc = scratch_of(dev);
        unsigned long long *cnt = (unsigned long long *)sc;
        double *ws = (double *)(sc + (size_t)NA_MAX_BINS * 8);
        GR_CUDA(cudaMemsetAsync(sc, 0, (size_t)NA_MAX_BINS * 16, st));      // the array keeps the last call's contents
        const int32_t h_lo = std::max(0, g->hub_lo), h_hi = (int32_t)std::min<int64_t>(g->n, g->hub_hi);
        if (g->n > 0 && g->n_edges > 0 && h_hi > h_lo) {
            const int grid = (int)std::max<int64_t>(g->sm_count * 4, (g->n_edges >> 30) + 1);
            k_2pcf_static<<<grid, 256, 0, st>>>(g->ptr.p, g->idx.p, g->bin.p, g->w.p, h_lo, h_hi, g->nb, wsum ? 1 : 0, cnt, ws);
            GR_CUDA(cudaGetLastError());
        }
        if (counts) GR_CUDA(cudaMemcpyAsync(counts, cnt, sizeof(uint64_t) * g->nb, cudaMemcpyDeviceToDevice, st));
        if (wsum) GR_CUDA(cudaMemcpyAsync(wsum, ws, sizeof(double) * g->nb, cudaMemcpyDeviceToDevice, st));
    }
    catch (const GrFail &f) { cudaGetLastError(); return f.code; }
    catch (...) { gr_set_error("unexpected internal error"); return GRAMSCI_ECUDA; }
    return GRAMSCI_OK;
}
