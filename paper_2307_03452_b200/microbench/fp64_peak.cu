// fp64_peak.cu -- FP64 peak microbenchmarks behind DESIGN.md section 6 "Roofline denominator": independent DFMA
// chains vs independent DMMA.8x8x4 chains, with and without shared-memory operand traffic, as a function of
// warps per SM (1 CTA per SM).  Warp counts that are not multiples of 4 show whether the FP64 tensor pipe is
// per SM sub-partition (a sub-partition with one warp more than the others then sets the time).
// Standalone: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o fp64_peak fp64_peak.cu && ./fp64_peak
#include <cstdio>
#include <cuda_runtime.h>
#include <vector>

__device__ __forceinline__ void dmma(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int NACC>
__global__ void k_dfma(double* out, int iters, double a, double b) {
    double acc[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) acc[i] = threadIdx.x + i;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < NACC; ++i) acc[i] = fma(acc[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) s += acc[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <int NACC>
__global__ void k_dmma(double* out, int iters, double a, double b) {
    double c0[NACC], c1[NACC];
#pragma unroll
    for (int i = 0; i < NACC; ++i) { c0[i] = threadIdx.x + i; c1[i] = i; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < NACC; ++i) dmma(c0[i], c1[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NACC; ++i) s += c0[i] + c1[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// DMMA with one LDS.64 per lane per DMMA (B operand from smem), NACC accumulators share... each own B
template <int NACC, int REUSE>
__global__ void k_dmma_lds(double* out, int iters, double a, int stride) {
    extern __shared__ double sm[];
    for (int i = threadIdx.x; i < 8192; i += blockDim.x) sm[i] = 1.0 / (i + 1);
    __syncthreads();
    double c0[NACC * REUSE], c1[NACC * REUSE];
#pragma unroll
    for (int i = 0; i < NACC * REUSE; ++i) { c0[i] = threadIdx.x + i; c1[i] = i; }
    const int lane = threadIdx.x & 31;
    int base = (lane * stride) & 4095;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < NACC; ++i) {
            double b = sm[(base + i * 37 + it) & 8191];
#pragma unroll
            for (int r = 0; r < REUSE; ++r) dmma(c0[i * REUSE + r], c1[i * REUSE + r], a + r, b);
        }
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < NACC * REUSE; ++i) s += c0[i] + c1[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <typename F>
float timeit(F f) {
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    f();
    cudaDeviceSynchronize();
    float best = 1e30f;
    for (int r = 0; r < 5; ++r) {
        cudaEventRecord(e0);
        f();
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    return best;
}

int main() {
    cudaDeviceProp p; cudaGetDeviceProperties(&p, 0);
    printf("%s SMs=%d clock=%d kHz\n", p.name, p.multiProcessorCount, p.clockRate);
    const int nsm = p.multiProcessorCount;
    double* out; cudaMalloc(&out, sizeof(double) * nsm * 8 * 1024);
    const int iters = 20000;
    for (int warps : {1, 2, 3, 4, 5, 6, 8, 11, 12, 16, 32}) {
        const int thr = warps * 32;
        {
            float ms = timeit([&] { k_dfma<16><<<nsm, thr>>>(out, iters, 1.0000001, 1e-9); });
            double fl = 2.0 * 16 * iters * (double)thr * nsm;
            printf("DFMA  warps/SM=%2d  %8.3f ms  %7.2f TFLOP/s\n", warps, ms, fl / ms / 1e9);
        }
        {
            float ms = timeit([&] { k_dmma<16><<<nsm, thr>>>(out, iters, 1.0000001, 1e-9); });
            double fl = 512.0 * 16 * iters * (double)warps * nsm;
            printf("DMMA  warps/SM=%2d  %8.3f ms  %7.2f TFLOP/s\n", warps, ms, fl / ms / 1e9);
        }
        if (warps == 4 || warps == 8 || warps == 11 || warps == 12 || warps == 16) {
            cudaFuncSetAttribute(k_dmma_lds<8, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
            cudaFuncSetAttribute(k_dmma_lds<8, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
            cudaFuncSetAttribute(k_dmma_lds<4, 4>, cudaFuncAttributeMaxDynamicSharedMemorySize, 65536);
            for (int stride : {1, 2, 33}) {
                float ms = timeit([&] { k_dmma_lds<8, 1><<<nsm, thr, 65536>>>(out, iters, 1.0000001, stride); });
                double fl = 512.0 * 8 * iters * (double)warps * nsm;
                printf("DMMA+LDS r1 stride=%2d warps/SM=%2d  %8.3f ms  %7.2f TFLOP/s\n", stride, warps, ms, fl / ms / 1e9);
                ms = timeit([&] { k_dmma_lds<8, 2><<<nsm, thr, 65536>>>(out, iters, 1.0000001, stride); });
                fl = 512.0 * 16 * iters * (double)warps * nsm;
                printf("DMMA+LDS r2 stride=%2d warps/SM=%2d  %8.3f ms  %7.2f TFLOP/s\n", stride, warps, ms, fl / ms / 1e9);
                ms = timeit([&] { k_dmma_lds<4, 4><<<nsm, thr, 65536>>>(out, iters, 1.0000001, stride); });
                fl = 512.0 * 16 * iters * (double)warps * nsm;
                printf("DMMA+LDS r4 stride=%2d warps/SM=%2d  %8.3f ms  %7.2f TFLOP/s\n", stride, warps, ms, fl / ms / 1e9);
            }
        }
    }
    return 0;
}
