// fp64_peak: register-resident micro-benchmark of the two FP64 pipes of the GPU it runs on -- DFMA (vector) and
// DMMA (mma.sync.m8n8k4.f64, the FP64 tensor path on sm_100a; tcgen05 has no FP64 kind).  bench.py runs it to
// obtain the MEASURED FP64 peak its tensor roofline is quoted against (MEASURED_PEAKS.json has no FP64 figure).
// Prints one JSON line: {"dfma_tflops": .., "dmma_tflops": .., "sms": .., "sm_khz": ..}.
#include <cstdio>
#include <cstdlib>
#include <cuda_runtime.h>

#define CK(x) do { cudaError_t e = (x); if (e != cudaSuccess) { fprintf(stderr, "CUDA error %s at line %d\n", cudaGetErrorString(e), __LINE__); return 1; } } while (0)

__global__ void k_dfma(double *out, int iters, double a, double b) {
    double x[16];
#pragma unroll
    for (int i = 0; i < 16; i++) x[i] = threadIdx.x * 1e-3 + i;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 16; i++) x[i] = fma(x[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 16; i++) s += x[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void k_dmma(double *out, int iters, double a, double b) {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) c[i][0] = c[i][1] = 0.0;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int i = 0; i < 8; i++)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

int main() {
    cudaDeviceProp p;
    CK(cudaGetDeviceProperties(&p, 0));
    const int threads = 256, blocks = p.multiProcessorCount * 4;
    double *out;
    CK(cudaMalloc(&out, (size_t)blocks * threads * sizeof(double)));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    double best[2] = {0, 0};
    for (int which = 0; which < 2; which++) {
        const int iters = which == 0 ? 20000 : 5000;
        const double flop = (which == 0 ? 32.0 : 8 * 2.0 * 8 * 8 * 4 / 32) * (double)iters * blocks * threads;
        for (int r = 0; r < 6; r++) {
            CK(cudaEventRecord(e0));
            if (which == 0) k_dfma<<<blocks, threads>>>(out, iters, 1.0000001, 1e-9);
            else k_dmma<<<blocks, threads>>>(out, iters, 1.0000001, 1e-9);
            CK(cudaEventRecord(e1));
            CK(cudaEventSynchronize(e1));
            float ms;
            CK(cudaEventElapsedTime(&ms, e0, e1));
            const double tf = flop / ms * 1e-9;
            if (r > 0 && tf > best[which]) best[which] = tf;
        }
    }
    printf("{\"dfma_tflops\": %.2f, \"dmma_tflops\": %.2f, \"sms\": %d, \"sm_khz\": %d}\n", best[0], best[1],
           p.multiProcessorCount, p.clockRate);
    return 0;
}
