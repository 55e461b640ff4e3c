// Measures what the integer-only control step of the library rests on (sp2_control.cuh): on B200 an FP64 instruction
// that follows a stretch of non-FP64 work pays a wake-up latency far above its pipeline latency, while back-to-back
// FP64 instructions do not.  Prints "name cycles_per_iteration" lines; built and run by tests/test_probe_hardware.py.
#include <cstdio>
#include <cuda_runtime.h>

__global__ void dense_chain(double* out, long long* cyc, int n) {
    double x = out[0] + threadIdx.x;
    const long long t0 = clock64();
    for (int i = 0; i < n; ++i) x = fma(x, 1.0000001, 1e-9);                 // dependent DFMA chain
    const long long t1 = clock64();
    if (threadIdx.x == 0) cyc[0] = t1 - t0;
    out[threadIdx.x + 1] = x;
}
__global__ void float_chain(double* out, long long* cyc, int n) {
    float f = (float)out[0] + threadIdx.x;
    const long long t0 = clock64();
    for (int i = 0; i < n; ++i) f = fmaf(f, 1.0000001f, 1e-9f);              // dependent FFMA chain
    const long long t1 = clock64();
    if (threadIdx.x == 0) cyc[0] = t1 - t0;
    out[threadIdx.x + 1] = f;
}
// one DFMA, then `gap` dependent FFMAs, repeated
__global__ void sparse_chain(double* out, long long* cyc, int n, int gap) {
    double x = out[0] + threadIdx.x;
    float f = (float)x;
    const long long t0 = clock64();
    for (int i = 0; i < n; ++i) {
        x = fma(x, 1.0000001, 1e-9);
        for (int g = 0; g < gap; ++g) f = fmaf(f, 1.0000001f, 1e-9f);
        f += (float)(i & 1);
    }
    const long long t1 = clock64();
    if (threadIdx.x == 0) cyc[0] = t1 - t0;
    out[threadIdx.x + 1] = x + f;
}

int main() {
    double* out;
    long long *cyc, h;
    cudaMalloc(&out, 1 << 16);
    cudaMalloc(&cyc, 8);
    cudaMemset(out, 0, 1 << 16);
    const int n = 2000;
    for (int rep = 0; rep < 2; ++rep) dense_chain<<<1, 32>>>(out, cyc, n);
    cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost);
    printf("dfma_chain %.2f\n", (double)h / n);
    for (int rep = 0; rep < 2; ++rep) float_chain<<<1, 32>>>(out, cyc, n);
    cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost);
    printf("ffma_chain %.2f\n", (double)h / n);
    const int gaps[4] = {16, 64, 256, 1024};
    for (int gi = 0; gi < 4; ++gi) {
        for (int rep = 0; rep < 2; ++rep) sparse_chain<<<1, 32>>>(out, cyc, 200, gaps[gi]);
        cudaMemcpy(&h, cyc, 8, cudaMemcpyDeviceToHost);
        printf("dfma_plus_%d_ffma %.2f\n", gaps[gi], (double)h / 200);
    }
    return cudaDeviceSynchronize() == cudaSuccess ? 0 : 1;
}
