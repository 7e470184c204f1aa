// Peak probes behind the roofline denominators of bench.py / DESIGN.md section 6 that MEASURED_PEAKS.json does not carry:
// plain fp64 (DFMA) and fp64 tensor (mma.sync.m8n8k4) throughput, and read / copy bandwidth of L2-resident and
// HBM-resident buffers (21 MB = one factor of config 3).  Stand-alone:
//     nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o /tmp/peak_probe paper_2110_13481_b200/csrc/peak_probe.cu && /tmp/peak_probe
#include <cstdio>
#include <cuda_runtime.h>
__global__ void k_dfma(double* out, int iters) {
    double a[16];
    for (int i = 0; i < 16; i++) a[i] = threadIdx.x * 1e-3 + i;
    const double b = 1.0000001, c = 1e-9;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 16; i++) a[i] = fma(a[i], b, c);
    }
    double s = 0; for (int i = 0; i < 16; i++) s += a[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void k_dmma(double* out, int iters) {
    double c[8][2];
    for (int i = 0; i < 8; i++) c[i][0] = c[i][1] = 0.0;
    double a = threadIdx.x * 1e-3, b = 1.0 + threadIdx.x * 1e-6;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0; for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
__global__ void k_read(const double2* in, size_t n, double* out) {
    double s = 0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) { double2 v = in[i]; s += v.x + v.y; }
    if (s == 123.456) out[0] = s;
}
__global__ void k_copy(const double2* in, double2* outp, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) outp[i] = in[i];
}
int main() {
    double* out; cudaMalloc(&out, 148 * 8 * 1024 * 8);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    for (int warps : {4, 8, 16, 32}) {
        const int iters = 20000, blocks = 148 * 2;
        k_dfma<<<blocks, warps * 32 / 2>>>(out, 100);
        cudaEventRecord(e0); k_dfma<<<blocks, warps * 32 / 2>>>(out, iters); cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        double fl = 2.0 * 16 * iters * (double)blocks * warps * 16;
        printf("DFMA  warps/SM %2d: %.2f TFLOP/s\n", warps, fl / ms / 1e9);
        k_dmma<<<blocks, warps * 32 / 2>>>(out, 100);
        cudaEventRecord(e0); k_dmma<<<blocks, warps * 32 / 2>>>(out, iters); cudaEventRecord(e1); cudaEventSynchronize(e1);
        cudaEventElapsedTime(&ms, e0, e1);
        fl = 2.0 * 256 * 8 * iters * (double)blocks * warps / 2;
        printf("DMMA  warps/SM %2d: %.2f TFLOP/s\n", warps, fl / ms / 1e9);
    }
    for (size_t mb : {21, 42, 84, 512, 4096}) {
        size_t n = mb * 1024 * 1024 / 16; double2 *a, *b; cudaMalloc(&a, n * 16); cudaMalloc(&b, n * 16); cudaMemset(a, 0, n * 16); cudaMemset(b, 0, n*16);
        for (int grid : {148 * 2, 148 * 8}) {
            float best = 1e9, bestc = 1e9;
            for (int rep = 0; rep < 10; rep++) {
                cudaEventRecord(e0); k_read<<<grid, 512>>>(a, n, out); cudaEventRecord(e1); cudaEventSynchronize(e1);
                float ms; cudaEventElapsedTime(&ms, e0, e1); if (ms < best) best = ms;
                cudaEventRecord(e0); k_copy<<<grid, 512>>>(a, b, n); cudaEventRecord(e1); cudaEventSynchronize(e1);
                cudaEventElapsedTime(&ms, e0, e1); if (ms < bestc) bestc = ms;
            }
            printf("read %4zu MB grid %4d: %.1f us = %.0f GB/s ; copy: %.1f us = %.0f GB/s (r+w)\n", mb, grid, best * 1e3, n * 16 / best / 1e6, bestc * 1e3, 2.0 * n * 16 / bestc / 1e6);
        }
        cudaFree(a); cudaFree(b);
    }
    printf("%s\n", cudaGetErrorString(cudaDeviceSynchronize()));
}
