// lcf_peaks.cu -- arithmetic-pipe microbenchmarks behind lcf_measure_peak(): the denominators of
// the "alu" rooflines (FP32 FMA for the Gram/projection kernels, FP64 FMA for precision = 1).
// Register-resident dependent-chain FMA loops, 16 independent chains per thread.
#include "lcf_internal.h"

namespace lcf {

constexpr int PK_CHAINS = 16, PK_ITERS = 2048, PK_THREADS = 256;

__global__ void __launch_bounds__(PK_THREADS) peak_ffma(float* out, float a, float b) {
    float acc[PK_CHAINS];
#pragma unroll
    for (int i = 0; i < PK_CHAINS; ++i) acc[i] = (float)(threadIdx.x + i);
#pragma unroll 1
    for (int it = 0; it < PK_ITERS; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < PK_CHAINS; ++i) acc[i] = fmaf(acc[i], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < PK_CHAINS; ++i) s += acc[i];
    if (s == 12345.678f) out[0] = s;  // never true in practice; keeps the chains alive
}

__global__ void __launch_bounds__(PK_THREADS) peak_ffma2(float* out, float a, float b) {
    unsigned long long acc[PK_CHAINS], av, bv;
    asm("mov.b64 %0, {%1, %1};" : "=l"(av) : "f"(a));
    asm("mov.b64 %0, {%1, %1};" : "=l"(bv) : "f"(b));
#pragma unroll
    for (int i = 0; i < PK_CHAINS; ++i) {
        float x = (float)(threadIdx.x + i), y = x + 0.5f;
        asm("mov.b64 %0, {%1, %2};" : "=l"(acc[i]) : "f"(x), "f"(y));
    }
#pragma unroll 1
    for (int it = 0; it < PK_ITERS; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < PK_CHAINS; ++i)
                asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(acc[i]) : "l"(av), "l"(bv));
    }
    float s = 0.f;
#pragma unroll
    for (int i = 0; i < PK_CHAINS; ++i) {
        float x, y;
        asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(acc[i]));
        s += x + y;
    }
    if (s == 12345.678f) out[0] = s;
}

__global__ void __launch_bounds__(PK_THREADS) peak_dfma(float* out, double a, double b) {
    double acc[PK_CHAINS];
#pragma unroll
    for (int i = 0; i < PK_CHAINS; ++i) acc[i] = (double)(threadIdx.x + i);
#pragma unroll 1
    for (int it = 0; it < PK_ITERS; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r)
#pragma unroll
            for (int i = 0; i < PK_CHAINS; ++i) acc[i] = fma(acc[i], a, b);
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < PK_CHAINS; ++i) s += acc[i];
    if (s == 12345.678) out[0] = (float)s;
}

}  // namespace lcf

extern "C" lcf_status lcf_measure_peak(int kind, double* tflops) {
    using namespace lcf;
    if (!tflops || kind < 0 || kind > 2) return LCF_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return LCF_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return LCF_ERR_CUDA;
    float* out = nullptr;
    if (cudaMalloc(&out, 4) != cudaSuccess) return LCF_ERR_ALLOC;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = sms * 8;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0);
        if (kind == 0) peak_ffma<<<blocks, PK_THREADS>>>(out, 0.999f, 0.001f);
        else if (kind == 1) peak_ffma2<<<blocks, PK_THREADS>>>(out, 0.999f, 0.001f);
        else peak_dfma<<<blocks, PK_THREADS>>>(out, 0.999, 0.001);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(out); return LCF_ERR_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        double fl = 2.0 * (double)blocks * PK_THREADS * (double)PK_ITERS * 4.0 * PK_CHAINS * (kind == 1 ? 2.0 : 1.0);
        double tf = fl / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    *tflops = best;
    return cudaGetLastError() == cudaSuccess ? LCF_OK : LCF_ERR_CUDA;
}
