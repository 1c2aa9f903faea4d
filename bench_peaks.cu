// bench_peaks.cu -- the in-run peak measurements bench.py puts under its roofline figures (not part of libgramsci.so).
//
// SURVEY 8(d) states the 3pCF roofline on L2->SM bytes and the 4pCF one on the global atomic rate; the driver
// measures only the HBM copy bandwidth (MEASURED_PEAKS.json).  bench.py therefore builds this file into
// libbench_peaks.so (nvcc, sm_100a) and calls it once per run, on the GPU and in the process that reports the
// numbers:
//   peaks_l2_read_gbs(mb)        every CTA streams a working set of `mb` MB (L2 resident after the first pass) with
//                                16-byte loads                                         -> GB/s
//   peaks_red_f64_gops(bins)     fp64 RED into a per-CTA global slab of `bins` bins, 32 active lanes, spread
//                                addresses (the access pattern of the 4pCF and weighted 3pCF kernels)  -> 1e9 RED/s
//   peaks_red_u64_gops(bins)     the same with uint64 RED into ONE shared histogram of `bins` bins
//   peaks_smem_atom_gops(bins)   uint32 shared-memory atomics on `bins` random bins (the 3pCF hit path)
//   peaks_hbm_copy_gbs(mb)       device-to-device copy of `mb` MB (read + write bytes), for the record
// Every loop iteration of the atomic tests also pays an LCG step and a runtime modulo, so those rates are slight
// under-estimates; kernels that do nothing but the atomic can read a little above them.
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

namespace {

__device__ __forceinline__ uint32_t lcg(uint32_t &s) { s = s * 1664525u + 1013904223u; return s >> 8; }

template <int MODE>
__global__ void k_atom(int iters, int nbins, unsigned long long *g64, double *gd, unsigned long long *sink)
{
    extern __shared__ uint32_t h32[];
    if (MODE == 0) for (int t = threadIdx.x; t < nbins; t += blockDim.x) h32[t] = 0;
    __syncthreads();
    uint32_t s = (blockIdx.x * blockDim.x + threadIdx.x) * 2654435761u + 12345u;
    double *myd = gd + (size_t)blockIdx.x * nbins;
    for (int it = 0; it < iters; ++it) {
        const uint32_t r = lcg(s) % nbins;
        if (MODE == 0) atomicAdd(&h32[r], 1u);
        if (MODE == 1) atomicAdd(&myd[r], 1.5);
        if (MODE == 2) atomicAdd(&g64[r], 1ull);
    }
    __syncthreads();
    if (MODE == 0 && threadIdx.x == 0) sink[0] += h32[0];
}

__global__ void k_l2read(const int4 *__restrict__ buf, size_t n16, int reps, int *sink)
{
    int acc = 0;
    for (int r = 0; r < reps; ++r) {
        const size_t off = ((size_t)r * 250112) % n16;        // a different rotation per pass: nothing to hoist
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += (size_t)gridDim.x * blockDim.x) {
            size_t j = i + off;
            if (j >= n16) j -= n16;
            const int4 v = __ldcg(buf + j);
            acc += v.x ^ v.y ^ v.z ^ v.w;
        }
    }
    if (acc == 0x7fffffff) sink[0] = acc;
}

int sm_count()
{
    int dev = 0, n = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
    return n;
}

template <int MODE>
double atom_rate(int nbins, int ctas_per_sm, size_t smem)
{
    const int iters = 4096, grid = sm_count() * ctas_per_sm;
    unsigned long long *g64 = nullptr, *sink = nullptr;
    double *gd = nullptr;
    if (cudaMalloc(&g64, sizeof(unsigned long long) * (size_t)nbins) != cudaSuccess) return -1;
    cudaMalloc(&gd, sizeof(double) * (size_t)nbins * grid);
    cudaMalloc(&sink, 64);
    cudaMemset(g64, 0, sizeof(unsigned long long) * (size_t)nbins);
    cudaMemset(gd, 0, sizeof(double) * (size_t)nbins * grid);
    cudaMemset(sink, 0, 64);
    cudaFuncSetAttribute(k_atom<MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    k_atom<MODE><<<grid, 256, smem>>>(64, nbins, g64, gd, sink);
    cudaDeviceSynchronize();
    double best = 0;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(a);
        k_atom<MODE><<<grid, 256, smem>>>(iters, nbins, g64, gd, sink);
        cudaEventRecord(b);
        if (cudaDeviceSynchronize() != cudaSuccess) { best = -1; break; }
        float ms = 0;
        cudaEventElapsedTime(&ms, a, b);
        const double rate = (double)grid * 256 * iters / (ms * 1e-3) / 1e9;
        if (rate > best) best = rate;
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    cudaFree(g64); cudaFree(gd); cudaFree(sink);
    return best;
}

}  // namespace

extern "C" double peaks_smem_atom_gops(int nbins) { return atom_rate<0>(nbins, 4, (size_t)nbins * 4 + 64); }
extern "C" double peaks_red_f64_gops(int nbins) { return atom_rate<1>(nbins, 4, 64); }
extern "C" double peaks_red_u64_gops(int nbins) { return atom_rate<2>(nbins, 4, 64); }

extern "C" double peaks_l2_read_gbs(int mb)
{
    const size_t n16 = (size_t)mb * (1 << 20) / 16;
    int4 *buf = nullptr;
    int *sk = nullptr;
    if (cudaMalloc(&buf, n16 * 16) != cudaSuccess) return -1;
    cudaMemset(buf, 1, n16 * 16);
    cudaMalloc(&sk, 4);
    const int reps = 100, grid = sm_count() * 8;
    k_l2read<<<grid, 256>>>(buf, n16, 2, sk);
    cudaDeviceSynchronize();
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    double best = 0;
    for (int rep = 0; rep < 3; ++rep) {
        cudaEventRecord(a);
        k_l2read<<<grid, 256>>>(buf, n16, reps, sk);
        cudaEventRecord(b);
        if (cudaDeviceSynchronize() != cudaSuccess) { best = -1; break; }
        float ms = 0;
        cudaEventElapsedTime(&ms, a, b);
        const double gbs = (double)n16 * 16 * reps / (ms * 1e-3) / 1e9;
        if (gbs > best) best = gbs;
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    cudaFree(buf); cudaFree(sk);
    return best;
}

extern "C" double peaks_hbm_copy_gbs(int mb)
{
    const size_t bytes = (size_t)mb << 20;
    char *x = nullptr, *y = nullptr;
    if (cudaMalloc(&x, bytes) != cudaSuccess || cudaMalloc(&y, bytes) != cudaSuccess) { cudaFree(x); return -1; }
    cudaMemset(x, 1, bytes);
    cudaEvent_t a, b;
    cudaEventCreate(&a);
    cudaEventCreate(&b);
    cudaMemcpy(y, x, bytes, cudaMemcpyDeviceToDevice);
    double best = 0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(a);
        cudaMemcpyAsync(y, x, bytes, cudaMemcpyDeviceToDevice);
        cudaEventRecord(b);
        cudaDeviceSynchronize();
        float ms = 0;
        cudaEventElapsedTime(&ms, a, b);
        const double gbs = 2.0 * bytes / (ms * 1e-3) / 1e9;
        if (gbs > best) best = gbs;
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    cudaFree(x); cudaFree(y);
    return best;
}
