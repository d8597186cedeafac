// lcf_peaks.cu -- arithmetic-pipe microbenchmarks behind lcf_measure_peak(): the denominators of
// the "alu" rooflines (FP32 FMA for the Gram/projection kernels, FP64 FMA for precision = 1).
// Register-resident dependent-chain FMA loops, 16 independent chains per thread.
#include "lcf_internal.h"
#include "lcf_sm100.cuh"

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

// Bare tcgen05.mma.kind::f16 loop: one CTA per SM, operands resident in shared memory (K-major core
// matrices, no swizzle, zeros), 128 x 256 x 16 MMAs alternating between two TMEM accumulators, one
// commit at the end.  No loads, no conversion, no epilogue: the ceiling of the fp16 tensor path that the
// Gram and projection kernels are quoted against.
constexpr int PK_TC_ITERS = 8192;
__global__ void __launch_bounds__(128, 1) peak_tc_f16(float* out) {
    using namespace sm100;
    extern __shared__ __align__(1024) unsigned char pk_smem[];
    unsigned char* sb = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(pk_smem) + 1023) & ~(uintptr_t)1023);
    unsigned char* A = sb;                       // 2 chunks x 128 rows x 16 B = 4 KB
    unsigned char* B = sb + 4096;                // 2 chunks x 256 rows x 16 B = 8 KB
    __shared__ uint64_t bar;
    __shared__ uint32_t tbase;
    const int tid = threadIdx.x, warp = tid >> 5;
    for (int i = tid * 16; i < 12288; i += 128 * 16) *reinterpret_cast<uint4*>(sb + i) = make_uint4(0, 0, 0, 0);
    fence_proxy_async_smem();
    if (tid == 0) { mbar_init(&bar, 1); mbar_fence_init(); }
    if (warp == 0) tmem_alloc<512>(&tbase);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = tbase;
    if (warp == 1) {
        const uint32_t idesc = make_idesc_f16(128, 256, false, false);
        const uint64_t dA = make_smem_desc(smem_u32(A), 128 * 16, 128, SWZ_NONE);
        const uint64_t dB = make_smem_desc(smem_u32(B), 256 * 16, 128, SWZ_NONE);
        if (elect_one()) {
#pragma unroll 1
            for (int it = 0; it < PK_TC_ITERS; it += 2) {
                mma_f16(tmem, dA, dB, idesc, 1u);
                mma_f16(tmem + 256, dA, dB, idesc, 1u);
            }
            mma_commit(&bar);
        }
        __syncwarp();
        mbar_wait(&bar, 0);
        tc_fence_after_sync();
    }
    tc_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_dealloc<512>(tmem);
    if (tid == 0 && out == nullptr) *out = 0.f;  // never
}

}  // namespace lcf

extern "C" lcf_status lcf_measure_peak(int kind, double* tflops) {
    using namespace lcf;
    if (!tflops || kind < 0 || kind > 3) return LCF_ERR_INVALID_ARG;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return LCF_ERR_CUDA;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return LCF_ERR_CUDA;
    float* out = nullptr;
    if (cudaMalloc(&out, 4) != cudaSuccess) return LCF_ERR_ALLOC;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int blocks = kind == 3 ? sms : sms * 8;
    double best = 0.0;
    for (int rep = 0; rep < 4; ++rep) {
        cudaEventRecord(e0);
        if (kind == 3) peak_tc_f16<<<blocks, 128, 12288 + 1024>>>(out);
        else if (kind == 0) peak_ffma<<<blocks, PK_THREADS>>>(out, 0.999f, 0.001f);
        else if (kind == 1) peak_ffma2<<<blocks, PK_THREADS>>>(out, 0.999f, 0.001f);
        else peak_dfma<<<blocks, PK_THREADS>>>(out, 0.999, 0.001);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(out); return LCF_ERR_CUDA; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        double fl = 2.0 * (double)blocks * PK_THREADS * (double)PK_ITERS * 4.0 * PK_CHAINS * (kind == 1 ? 2.0 : 1.0);
        if (kind == 3) fl = (double)blocks * (double)PK_TC_ITERS * 2.0 * 128.0 * 256.0 * 16.0;
        double tf = fl / (ms * 1e-3) / 1e12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(out);
    *tflops = best;
    return cudaGetLastError() == cudaSuccess ? LCF_OK : LCF_ERR_CUDA;
}
