// Arithmetic-pipe peaks of this B200 for the ALU roofline of the DG kernels: FP64 DFMA, FP64 DMMA
// (mma.sync.m8n8k4.f64), the two mixed 1:1, and FP32 FFMA, each as a register-only dependent-chain loop with
// enough independent chains to cover the pipe latency.  Build and run:
//   nvcc -O3 -gencode arch=compute_100a,code=sm_100a -o /tmp/peaks paper_1610_05023_b200/csrc/ubench/peaks.cu && /tmp/peaks
// Prints one line per pipe: TFLOP/s (2 flop per FMA; 512 flop per DMMA.8x8x4 warp instruction).
#include <cuda_runtime.h>

#include <cstdio>

constexpr int ITER = 4096, CH = 8;

__global__ void k_dfma(double* out, double a, double b) {
    double x[CH];
    for (int i = 0; i < CH; ++i) x[i] = threadIdx.x + i;
    for (int it = 0; it < ITER; ++it)
#pragma unroll
        for (int i = 0; i < CH; ++i) x[i] = fma(x[i], a, b);
    double s = 0;
    for (int i = 0; i < CH; ++i) s += x[i];
    if (s == 12345.678) out[0] = s;
}

__global__ void k_ffma(float* out, float a, float b) {
    float x[CH];
    for (int i = 0; i < CH; ++i) x[i] = threadIdx.x + i;
    for (int it = 0; it < ITER; ++it)
#pragma unroll
        for (int i = 0; i < CH; ++i) x[i] = fmaf(x[i], a, b);
    float s = 0;
    for (int i = 0; i < CH; ++i) s += x[i];
    if (s == 12345.678f) out[0] = s;
}

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c[0]), "+d"(c[1]) : "d"(a), "d"(b));
}

template <bool MIX>
__global__ void k_dmma(double* out, double a, double b) {
    double c[CH][2], x[CH];
    for (int i = 0; i < CH; ++i) { c[i][0] = threadIdx.x; c[i][1] = i; x[i] = i; }
    for (int it = 0; it < ITER; ++it)
#pragma unroll
        for (int i = 0; i < CH; ++i) {
            dmma(c[i], a, b);
            if (MIX) {      // 8 DFMA per lane per DMMA would be 1:1 in flops; 4 is the ratio of the DG kernel's epilogue
                x[i] = fma(x[i], a, b); x[i] = fma(x[i], a, b); x[i] = fma(x[i], a, b); x[i] = fma(x[i], a, b);
            }
        }
    double s = 0;
    for (int i = 0; i < CH; ++i) s += c[i][0] + c[i][1] + x[i];
    if (s == 12345.678) out[0] = s;
}

template <typename F>
double time_ms(F launch) {
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    launch(); launch();
    cudaDeviceSynchronize();
    float best = 1e30f;
    for (int r = 0; r < 5; ++r) {
        cudaEventRecord(e0); launch(); cudaEventRecord(e1); cudaEventSynchronize(e1);
        float ms; cudaEventElapsedTime(&ms, e0, e1);
        if (ms < best) best = ms;
    }
    return best;
}

int main() {
    int sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
    double* d; cudaMalloc(&d, 64);
    const int grid = sms * 8, block = 512;
    const double thr = (double)grid * block;
    double ms;
    ms = time_ms([&] { k_dfma<<<grid, block>>>(d, 1.0000001, 1e-9); });
    printf("fp64 DFMA      : %7.2f TFLOP/s\n", thr * ITER * CH * 2 / ms * 1e-9);
    ms = time_ms([&] { k_dmma<false><<<grid, block>>>(d, 1.0000001, 1e-9); });
    printf("fp64 DMMA 8x8x4: %7.2f TFLOP/s\n", thr / 32 * ITER * CH * 512 / ms * 1e-9);
    ms = time_ms([&] { k_dmma<true><<<grid, block>>>(d, 1.0000001, 1e-9); });
    printf("fp64 DMMA+4DFMA: %7.2f TFLOP/s (both counted)\n", thr * ITER * CH * (16 + 8) / ms * 1e-9);
    ms = time_ms([&] { k_ffma<<<grid, block>>>((float*)d, 1.0000001f, 1e-9f); });
    printf("fp32 FFMA      : %7.2f TFLOP/s\n", thr * ITER * CH * 2 / ms * 1e-9);
    cudaError_t e = cudaDeviceSynchronize();
    printf("sms %d status %s\n", sms, cudaGetErrorString(e));
    return e != cudaSuccess;
}
