// FP64 pipe probe: DFMA and DMMA (mma.sync.m8n8k4.f64) throughput on sm_100a -- the denominator of the "alu" rooflines
// (DESIGN.md section 5.3).  Not part of libbs: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/fp64_peak <this file> && /tmp/fp64_peak
#include <cstdio>
#include <cuda_runtime.h>
__global__ void k_dfma(double* out, int iters) {
    double a[16];
    for (int i = 0; i < 16; ++i) a[i] = threadIdx.x * 1e-3 + i;
    double x = 1.0000001, y = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 16; ++i) a[i] = a[i] * x + y;
    }
    double s = 0;
    for (int i = 0; i < 16; ++i) s += a[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void k_dmma(double* out, int iters) {
    double c[8][2];
    for (int i = 0; i < 8; ++i) c[i][0] = c[i][1] = 0.0;
    double a = threadIdx.x * 1e-3, b = 1.0 + threadIdx.x * 1e-6;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
int main() {
    double* d; cudaMalloc(&d, 148 * 8 * 1024 * 8);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int threads : {128, 256, 512, 1024}) {
        int iters = 20000; float ms;
        k_dfma<<<148, threads>>>(d, 100); cudaDeviceSynchronize();
        cudaEventRecord(e0); k_dfma<<<148, threads>>>(d, iters); cudaEventRecord(e1); cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        double fma = 148.0 * threads * 16.0 * iters;
        printf("DFMA threads=%d: %.3f ms  %.2f TFLOP/s  %.1f DFMA/clk/SM (at 1.965 GHz)\n", threads, ms, 2 * fma / ms / 1e9, fma / 148 / (ms * 1e-3 * 1.965e9));
        k_dmma<<<148, threads>>>(d, 100); cudaDeviceSynchronize();
        cudaEventRecord(e0); k_dmma<<<148, threads>>>(d, iters); cudaEventRecord(e1); cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        double fm2 = 148.0 * (threads / 32) * 8.0 * iters * 256.0;
        printf("DMMA threads=%d: %.3f ms  %.2f TFLOP/s  %.1f FMA/clk/SM\n", threads, ms, 2 * fm2 / ms / 1e9, fm2 / 148 / (ms * 1e-3 * 1.965e9));
    }
    return 0;
}
