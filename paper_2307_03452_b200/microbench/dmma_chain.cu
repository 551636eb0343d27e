// dmma_chain.cu -- dependent-issue latency of DMMA.8x8x4 on sm_100a: NACC independent accumulator chains per warp, 1-4 warps per
// SM sub-partition.  Standalone: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o dmma_chain dmma_chain.cu && ./dmma_chain
// Result (profiles/r2_dmma_chain.txt): a dependent DMMA issues 26 clocks after its predecessor; one chain per warp already
// saturates the pipe with two or more warps per sub-partition -- accumulator count per warp is not a constraint.
#include <cstdio>
#include <cuda_runtime.h>
__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
template <int NACC>
__global__ void k(double* out, int iters, double a, double b) {
    double c0[NACC], c1[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) { c0[i] = threadIdx.x + i; c1[i] = i; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int i = 0; i < NACC; ++i) dmma(c0[i], c1[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) s += c0[i] + c1[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <int NACC> void run(double* out, int nsm, int warps) {
    const int iters = 20000;
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    k<NACC><<<nsm, warps * 32>>>(out, iters, 1.0000001, 1e-9); cudaDeviceSynchronize();
    cudaEventRecord(e0); k<NACC><<<nsm, warps * 32>>>(out, iters, 1.0000001, 1e-9); cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    double ndmma = 4.0 * NACC * iters;   // per warp
    double clk = ms * 1e-3 * 1.965e9;
    printf("NACC=%d warps/SM=%2d: %.1f clk per DMMA per warp, chain step %.0f clk, SM rate %.2f DMMA/16clk/SMSP\n", NACC, warps, clk / ndmma, clk / ndmma * NACC,
           ndmma * warps / 4.0 / (clk / 16.0));
}
int main() {
    cudaDeviceProp p; cudaGetDeviceProperties(&p, 0); int nsm = p.multiProcessorCount;
    double* out; cudaMalloc(&out, sizeof(double) * nsm * 1024);
    for (int w : {4, 8, 12, 16}) { run<1>(out, nsm, w); run<2>(out, nsm, w); run<3>(out, nsm, w); run<4>(out, nsm, w); run<6>(out, nsm, w); run<8>(out, nsm, w); }
    return 0;
}
