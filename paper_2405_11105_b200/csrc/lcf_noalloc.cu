// lcf_noalloc.cu -- the allocation-free entry point declared in include/lcf_noalloc.h:
//   lcf_gram_global_noalloc   R[i][j] = sum_p conj(S[i][p]) S[j][p]   (Eq. 1) in double,
// a variant of the plan path's CUDA-core Gram (lcf_gram.cu: per-chunk partial sums in a workspace that lcf_plan_create
// allocates, then a fixed-order reduction) whose partial sums live in a file-scope __device__ array instead, so that the call
// never allocates.  Nothing here is used by, or changes, the plan path.
//
// The array's name below is, in HOST code, only a stand-in for the symbol: its device address is taken once per device with
// cudaGetSymbolAddress (with that device current) and handed to the kernels as an ordinary pointer.
#include <cstdio>
#include <mutex>

#include "../../include/lcf_noalloc.h"

#include <cuda_runtime.h>

namespace {

constexpr int NA_MAXN = LCF_NOALLOC_MAX_FRAMES;      // 128 frames
constexpr int NA_SLICES = LCF_NOALLOC_SLICES;        // pixel slices = partial sums per entry of R
constexpr int NA_TILE = 32;                          // a CTA owns a 32 x 32 tile of R for one pixel slice
constexpr int NA_PC = 64;                            // pixels per shared-memory chunk
constexpr int NA_MAXDEV = 64;

// [NA_SLICES][N][N] partial sums of the current call (slice stride NA_MAXN^2): 16 x 128 x 128 x 16 B = 4 MiB per GPU
static __device__ __align__(256) double2 na_scratch[(size_t)NA_SLICES * NA_MAXN * NA_MAXN];

// grid (tiles_i * tiles_j, NA_SLICES), 256 threads = 16 x 16, thread (tx, ty) keeps entries (ty + 16 a, tx + 16 b), a, b in {0, 1}
__global__ void __launch_bounds__(256) na_gram_partial_kernel(const float2* iq, int N, long long P, double2* part) {
    __shared__ float2 A[NA_TILE][NA_PC + 1], B[NA_TILE][NA_PC + 1];       // +1: rows start on different banks
    const int nt = (N + NA_TILE - 1) / NA_TILE;
    const int ti = blockIdx.x / nt, tj = blockIdx.x - ti * nt, s = blockIdx.y;
    const int tid = threadIdx.x, tx = tid & 15, ty = tid >> 4;
    const long long p0 = P * s / NA_SLICES, p1 = P * (s + 1) / NA_SLICES;
    double re[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, im[2][2] = {{0.0, 0.0}, {0.0, 0.0}};
    for (long long pc = p0; pc < p1; pc += NA_PC) {
        __syncthreads();
        for (int e = tid; e < 2 * NA_TILE * NA_PC; e += 256) {
            const int which = e / (NA_TILE * NA_PC), r = (e / NA_PC) % NA_TILE, c = e % NA_PC;   // lanes run over pixels: coalesced
            const int t = (which ? tj : ti) * NA_TILE + r;
            const long long p = pc + c;
            const float2 v = (t < N && p < p1) ? iq[(size_t)t * P + p] : make_float2(0.f, 0.f);
            if (which) B[r][c] = v; else A[r][c] = v;
        }
        __syncthreads();
#pragma unroll 4
        for (int c = 0; c < NA_PC; ++c) {
            const float2 a0 = A[ty][c], a1 = A[ty + 16][c], b0 = B[tx][c], b1 = B[tx + 16][c];
            const double ar[2] = {a0.x, a1.x}, ai[2] = {a0.y, a1.y}, br[2] = {b0.x, b1.x}, bi[2] = {b0.y, b1.y};
#pragma unroll
            for (int a = 0; a < 2; ++a)
#pragma unroll
                for (int b = 0; b < 2; ++b) {                         // conj(a) b = (ar br + ai bi) + i (ar bi - ai br)
                    re[a][b] = fma(ar[a], br[b], fma(ai[a], bi[b], re[a][b]));
                    im[a][b] = fma(ar[a], bi[b], fma(-ai[a], br[b], im[a][b]));
                }
        }
    }
    double2* ps = part + (size_t)s * NA_MAXN * NA_MAXN;
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 2; ++b) {
            const int i = ti * NA_TILE + ty + 16 * a, j = tj * NA_TILE + tx + 16 * b;
            if (i < N && j < N) ps[(size_t)i * N + j] = make_double2(re[a][b], im[a][b]);      // every slot a call reads is written here first
        }
}

// R[e] = sum over the slices in the order 0, 1, ... (deterministic)
__global__ void na_gram_reduce_kernel(const double2* part, int N, double2* R) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= N * N) return;
    double sr = 0.0, si = 0.0;
    for (int s = 0; s < NA_SLICES; ++s) {
        const double2 v = part[(size_t)s * NA_MAXN * NA_MAXN + e];
        sr += v.x; si += v.y;
    }
    R[e] = make_double2(sr, si);
}

std::mutex na_mutex;
double2* na_scratch_addr[NA_MAXDEV] = {};              // device address of na_scratch on device d (0: not taken yet)
thread_local char na_error[256] = "";

#define NA_FAIL(st, ...) do { snprintf(na_error, sizeof(na_error), __VA_ARGS__); return (st); } while (0)

}  // namespace

extern "C" const char* lcf_noalloc_last_error(void) { return na_error; }

extern "C" lcf_status lcf_gram_global_noalloc(const void* iq_dev, int N, long long P, double* R_dev, cudaStream_t stream) {
    na_error[0] = 0;
    if (!iq_dev || !R_dev) NA_FAIL(LCF_ERR_INVALID_ARG, "lcf_gram_global_noalloc: null pointer");
    if (N < 1 || P < 1) NA_FAIL(LCF_ERR_INVALID_ARG, "lcf_gram_global_noalloc: N = %d, P = %lld: both must be at least 1", N, P);
    if (N > NA_MAXN)
        NA_FAIL(LCF_ERR_UNSUPPORTED, "lcf_gram_global_noalloc: N = %d frames is beyond the fixed scratch array (at most %d frames); "
                "nothing was launched -- use a plan (lcf_plan_create) for longer ensembles", N, NA_MAXN);
    if (P > (1LL << 30))
        NA_FAIL(LCF_ERR_UNSUPPORTED, "lcf_gram_global_noalloc: P = %lld pixels is beyond the supported %lld; nothing was launched", P, 1LL << 30);
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= NA_MAXDEV)
        NA_FAIL(LCF_ERR_CUDA, "lcf_gram_global_noalloc: no usable current device (device %d): %s", dev, cudaGetErrorString(e));
    double2* part = nullptr;
    {
        std::lock_guard<std::mutex> lock(na_mutex);
        if (!na_scratch_addr[dev]) {                     // once per device, with that device current
            void* ptr = nullptr;
            e = cudaGetSymbolAddress(&ptr, na_scratch);
            if (e != cudaSuccess || !ptr) {
                cudaGetLastError();
                NA_FAIL(LCF_ERR_CUDA, "lcf_gram_global_noalloc: cudaGetSymbolAddress of the scratch array failed on device %d: %s", dev,
                        cudaGetErrorString(e));
            }
            na_scratch_addr[dev] = static_cast<double2*>(ptr);
        }
        part = na_scratch_addr[dev];
    }
    const int nt = (N + NA_TILE - 1) / NA_TILE;
    na_gram_partial_kernel<<<dim3(nt * nt, NA_SLICES), 256, 0, stream>>>(static_cast<const float2*>(iq_dev), N, P, part);
    e = cudaGetLastError();
    if (e == cudaSuccess) {
        na_gram_reduce_kernel<<<(N * N + 255) / 256, 256, 0, stream>>>(part, N, reinterpret_cast<double2*>(R_dev));
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) NA_FAIL(LCF_ERR_CUDA, "lcf_gram_global_noalloc: kernel launch failed on device %d: %s", dev, cudaGetErrorString(e));
    return LCF_OK;
}
