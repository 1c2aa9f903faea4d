// ubench_atomics.cu -- stand-alone micro-benchmark of the histogram primitives the enumeration kernels lean
// on (shared uint32 / uint64 / fp64 atomics, global RED into per-CTA slabs and into one shared histogram,
// random shared-memory loads, match.any).  Not part of libgramsci.so.  It is where DESIGN.md section 6 and
// bench.py take the "L2 atomic rate" peak of the 4pCF kernels from (profiles/r1_ubench_atomics.txt):
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o ubench_atomics paper_2607_06604_b200/csrc/ubench_atomics.cu
//   ./ubench_atomics
// Every loop iteration also pays an LCG step and a runtime modulo (~11 cycles per warp instruction, visible
// in the "LDS u32 random" line), so the per-instruction costs are upper bounds.
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define CK(x) do{cudaError_t e=(x); if(e!=cudaSuccess){printf("ERR %s line %d\n",cudaGetErrorString(e),__LINE__);return 1;}}while(0)
__device__ __forceinline__ uint32_t lcg(uint32_t &s){ s = s*1664525u+1013904223u; return s>>8; }

template<int MODE>
__global__ void k(int iters, int nbins, int active, unsigned long long *g64, double *gd, unsigned long long *sink)
{
    extern __shared__ unsigned char sm[];
    uint32_t *h32=(uint32_t*)sm; unsigned long long *h64=(unsigned long long*)sm; double *hd=(double*)sm; uint8_t* h8=(uint8_t*)sm;
    if(MODE<=2||MODE==5||MODE==6||MODE==8) for(int t=threadIdx.x;t<nbins*2;t+=blockDim.x) h32[t]=0;
    __syncthreads();
    uint32_t s = (blockIdx.x*blockDim.x+threadIdx.x)*2654435761u+12345u;
    const int lane=threadIdx.x&31;
    const bool act = lane<active;
    unsigned long long acc=0;
    double *myd = gd + (size_t)blockIdx.x*nbins;
    for(int it=0;it<iters;++it){
        uint32_t r = lcg(s)%nbins;
        if(MODE==0){ if(act) atomicAdd(&h32[r],1u); }
        if(MODE==1){ if(act) atomicAdd(&h64[r],1ull); }
        if(MODE==2){ if(act) atomicAdd(&hd[r],1.5); }
        if(MODE==3){ if(act) atomicAdd(&myd[r],1.5); }
        if(MODE==4){ if(act) atomicAdd(&g64[r],1ull); }
        if(MODE==5){ if(act) acc += h8[r]; }                       // random byte LDS
        if(MODE==6){ uint32_t base = (lcg(s)%nbins)&~255u; uint32_t rr=__shfl_sync(0xffffffffu,base,0)+lane*6+(r&3); if(act) acc += h8[rr%nbins]; } // sorted-local byte LDS
        if(MODE==7){ acc += __match_any_sync(0xffffffffu, r&255); }
        if(MODE==8){ if(act) acc += h32[r]; }                      // random word LDS
        if(MODE==9){ if(act) atomicAdd(&gd[r],1.5); }                // fp64 RED to one shared global hist
    }
    if(acc==0x12345) sink[0]=acc;
    __syncthreads();
    if(MODE<=2 && threadIdx.x==0) sink[1]+=h32[0];
}
// L2 -> SM read bandwidth: every CTA streams the whole working set (<= 64 MB, L2 resident after the first pass)
// with 16-byte loads; DESIGN.md section 6 quotes it next to the HBM copy figure
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

template<int MODE> int run(const char*name,int nbins,int active,size_t smem,int ctas_per_sm, unsigned long long*g64,double*gd,unsigned long long*sink)
{
    int iters=4096; int grid=148*ctas_per_sm;
    CK(cudaFuncSetAttribute(k<MODE>,cudaFuncAttributeMaxDynamicSharedMemorySize,(int)smem));
    cudaEvent_t a,b; cudaEventCreate(&a); cudaEventCreate(&b);
    k<MODE><<<grid,256,smem>>>(64,nbins,active,g64,gd,sink);
    CK(cudaDeviceSynchronize());
    cudaEventRecord(a);
    k<MODE><<<grid,256,smem>>>(iters,nbins,active,g64,gd,sink);
    cudaEventRecord(b); CK(cudaDeviceSynchronize());
    float ms; cudaEventElapsedTime(&ms,a,b);
    double ops=(double)grid*256/32*active*iters;
    double winstr=(double)grid*8*iters;
    printf("%-34s bins=%7d act=%2d ctas/sm=%d  %8.3f ms  %9.3e lane-ops/s  %6.2f ns/warp-instr/SM (~%5.1f cyc @1.9GHz)\n",name,nbins,active,ctas_per_sm,ms,ops/(ms*1e-3), ms*1e6/(winstr/148), ms*1e6/(winstr/148)*1.9);
    return 0;
}
int main(){
    unsigned long long *g64,*sink; double*gd;
    CK(cudaMalloc(&g64,sizeof(unsigned long long)*(1<<22))); CK(cudaMemset(g64,0,sizeof(unsigned long long)*(1<<22)));
    CK(cudaMalloc(&gd,sizeof(double)*4096*148*8)); CK(cudaMemset(gd,0,sizeof(double)*4096*148*8));
    CK(cudaMalloc(&sink,64)); CK(cudaMemset(sink,0,64));
    for(int act: {32,15}){
      run<0>("smem atomicAdd u32",3375,act,3375*8,2,g64,gd,sink);
      run<0>("smem atomicAdd u32",3375,act,3375*8,4,g64,gd,sink);
      run<1>("smem atomicAdd u64",3375,act,3375*8,2,g64,gd,sink);
      run<2>("smem atomicAdd f64 (CAS)",3375,act,3375*8,2,g64,gd,sink);
      run<3>("global RED f64 per-CTA slab",3375,act,1024,2,g64,gd,sink);
      run<3>("global RED f64 per-CTA slab",3375,act,1024,4,g64,gd,sink);
      run<9>("global RED f64 shared hist",3375,act,1024,4,g64,gd,sink);
      run<4>("global RED u64 shared hist",262144,act,1024,4,g64,gd,sink);
      run<4>("global RED u64 shared hist",3375,act,1024,4,g64,gd,sink);
      run<5>("smem LDS u8 random",16384,act,16384*8,1,g64,gd,sink);
      run<6>("smem LDS u8 sorted-local",16384,act,16384*8,1,g64,gd,sink);
      run<8>("smem LDS u32 random",4096,act,4096*8,4,g64,gd,sink);
    }
    run<7>("match_any",256,32,1024,4,g64,gd,sink);
    for (size_t mb : {16, 32, 64}) {
        const size_t n16 = mb * (1 << 20) / 16;
        int4 *buf; int *sk;
        CK(cudaMalloc(&buf, n16 * 16)); CK(cudaMemset(buf, 1, n16 * 16)); CK(cudaMalloc(&sk, 4));
        const int reps = 200;
        k_l2read<<<148 * 8, 256>>>(buf, n16, 2, sk);
        CK(cudaDeviceSynchronize());
        cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
        cudaEventRecord(a);
        k_l2read<<<148 * 8, 256>>>(buf, n16, reps, sk);
        cudaEventRecord(b); CK(cudaDeviceSynchronize());
        float ms; cudaEventElapsedTime(&ms, a, b);
        printf("L2 read, %zu MB working set, 16-byte loads: %.3f ms for %d passes -> %.0f GB/s\n", mb, ms, reps,
               (double)n16 * 16 * reps / (ms * 1e-3) / 1e9);
        cudaFree(buf); cudaFree(sk);
    }
    return 0;
}
