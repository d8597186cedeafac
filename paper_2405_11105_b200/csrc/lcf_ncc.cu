// lcf_ncc.cu -- method 4 of the paper: the cut-off that minimises the spatial normalised cross-correlation
// of a tissue image and a blood image (Eq. 8), per window, on the GPU.
//
//   u_i = C_w v_i / sigma_i     (C V = U D, lambda_i = sigma_i^2; C_w = W C, Eq. 11)
//   I_T(k) = sum_{i=k-fn+1}^{k} |u_i|     I_B(k) = sum_{i=k+1}^{k+fn} |u_i|     (fn = 5, w_i = 1, clipped to 1..N)
//   k* = argmin_{k=1..N-1}  sum_p I_T I_B / (sqrt(sum_p I_T^2) sqrt(sum_p I_B^2))       (lowest k on ties)
// (readings of the garbled index ranges: DESIGN.md "Readings" 19).  It runs between the EVD and the projection
// when the plan's mode is LCF_HARD_NCC / LCF_SOFT_NCC.  The EVD kernels are launched with all eigen-weights 1,
// so B_k = V_k; then
//   1. ncc_isig_kernel      1 / sigma by rank (0 where lambda <= 1e-12 lambda_1);
//   2. |u_i(p)| for every pixel of every window, components in rank order: the third tall contraction, on the
//      tcgen05 projection pipeline with a magnitude epilogue (lcf_project_tc.cu, MAG variant) -- or, where
//      that kernel is not eligible (odd Nz, tiny shapes), ncc_mag_kernel on the FP32 pipe;
//   3. ncc_sums_kernel      per (window, pixel chunk): thread k keeps sum I_T I_B, sum I_T^2, sum I_B^2 of its k;
//   4. ncc_argmin_kernel    chunks summed in double in a fixed order, the curve, its minimum -> c_k;
//   5. ncc_reweight_kernel  eigen-weights from c_k (hard, or Eq. 9 around it: method 5 as the paper pairs them,
//      PAPER.md:118), B_k = V_k diag(wt).
// Deterministic: no atomics, fixed summation orders.
#include <cfloat>

#include "lcf_internal.h"
#include "lcf_thresh.cuh"

namespace lcf {

constexpr int NCC_FN = 5;                  // singular vectors on either side of the cut
constexpr int NCC_CHUNKS = 32;             // pixel chunks per window in ncc_sums_kernel

// isig[k][r] = 1 / sqrt(lambda_r) for rank r < N with lambda_r > 1e-12 lambda_1, else 0
__global__ void ncc_isig_kernel(const double* lam, int N, int ncol, float* isig) {
    const int k = blockIdx.x;
    const double l1 = lam[(size_t)k * N];
    for (int r = threadIdx.x; r < ncol; r += blockDim.x) {
        float v = 0.f;
        if (r < N) {
            const double l = lam[(size_t)k * N + r];
            if (l > 0.0 && l > 1e-12 * l1) v = (float)(1.0 / sqrt(l));
        }
        isig[(size_t)k * ncol + r] = v;
    }
}

// FP32 fallback of step 2: one CTA per 32 pixels of a window, thread r = rank.
//   mag[(tile_off + q) * ncol + r] = w(p) |sum_t S[t][p] B[t][slot(r)]| / sigma_r
__global__ void __launch_bounds__(256) ncc_mag_kernel(const float2* iq, int N, int Ns, int Nz, int Nx, long long P, const float2* B,
                                                      const int* order, const WinBox* box, const ProjItem* items,
                                                      const double* gz, const double* gx, const float* isig, int ncol, float* mag) {
    extern __shared__ float2 ncc_sm[];                 // [32 pixels][N] samples of the chunk (w applied)
    const ProjItem it = items[blockIdx.x];
    const WinBox bx = box[it.k];
    for (int half = 0; half < 2; ++half) {             // items are 64-pixel chunks: two passes of 32
        const int q00 = it.q0 + 32 * half;
        const int np = it.q1 - q00 < 32 ? it.q1 - q00 : 32;
        if (np <= 0) break;
        __syncthreads();
        for (int e = threadIdx.x; e < np * N; e += blockDim.x) {
            const int t = e / np, j = e - t * np;
            const int q = q00 + j, xr = q / bx.Lz, zr = q - xr * bx.Lz;
            const int x = bx.x0 + xr, z = bx.z0 + zr;
            const float w = (float)(gz[(size_t)bx.kz * Nz + z] * gx[(size_t)bx.kx * Nx + x]);
            const float2 s = iq[(size_t)t * P + (size_t)x * Nz + z];
            ncc_sm[j * N + t] = make_float2(w * s.x, w * s.y);
        }
        __syncthreads();
        for (int r = threadIdx.x; r < N; r += blockDim.x) {
            const int u = order[(size_t)it.k * N + r];
            const float2* Bk = B + (size_t)it.k * N * Ns + u;
            const float is = isig[(size_t)it.k * ncol + r];
            for (int j = 0; j < np; ++j) {
                float ur = 0.f, ui = 0.f;
                for (int t = 0; t < N; ++t) {
                    const float2 b = Bk[(size_t)t * Ns], s = ncc_sm[j * N + t];
                    ur = fmaf(s.x, b.x, fmaf(-s.y, b.y, ur));
                    ui = fmaf(s.x, b.y, fmaf(s.y, b.x, ui));
                }
                mag[((size_t)bx.tile_off + q00 + j) * ncol + r] = sqrtf(ur * ur + ui * ui) * is;
            }
        }
    }
}

// Step 3.  CTA (chunk c, window k), thread k' = candidate cut (1-based k' = threadIdx.x + 1).  The chunk's pixels
// stream through shared memory NCC_ROWS rows at a time (cp.async, two buffers); a row sits between NCC_FN zeros on
// either side, so the clipping of I_T / I_B to 1..N is the padding and every thread adds ten taps with fixed bounds.
constexpr int NCC_ROWS = 32;
constexpr int NCC_PADL = 8;                // floats of zeros before a row (>= NCC_FN - 1, keeps rows 16-byte aligned)
__device__ __forceinline__ void ncc_cp16(float* dst, const float* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__device__ __forceinline__ void ncc_cp4(float* dst, const float* src) {
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src) : "memory");
}
__global__ void __launch_bounds__(256) ncc_sums_kernel(const float* mag, int N, int ncol, const WinBox* box, float* part /* [K][CHUNKS][3][N] */) {
    extern __shared__ __align__(16) float ncc_rows[];  // [2][NCC_ROWS][RS]
    const int k = blockIdx.y, c = blockIdx.x, kk = threadIdx.x + 1;
    const int RS = NCC_PADL + ((ncol + 3) & ~3) + 8;   // row stride: zeros, the row, zeros (>= NCC_FN)
    const WinBox bx = box[k];
    const long long q0 = (long long)bx.Pk * c / NCC_CHUNKS, q1 = (long long)bx.Pk * (c + 1) / NCC_CHUNKS;
    for (int e = threadIdx.x; e < 2 * NCC_ROWS * RS; e += blockDim.x) ncc_rows[e] = 0.f;
    __syncthreads();
    const bool vec = (ncol & 3) == 0;
    auto issue = [&](long long q, int buf) {
        const int nr = q1 - q < NCC_ROWS ? (int)(q1 - q) : NCC_ROWS;
        const float* src = mag + ((size_t)bx.tile_off + q) * ncol;
        float* dst = ncc_rows + (size_t)buf * NCC_ROWS * RS + NCC_PADL;
        if (vec) {
            const int cpr = ncol >> 2;
            for (int e = threadIdx.x; e < nr * cpr; e += blockDim.x) {
                const int r = e / cpr, j = e - r * cpr;
                ncc_cp16(dst + r * RS + 4 * j, src + (size_t)r * ncol + 4 * j);
            }
        } else {
            for (int e = threadIdx.x; e < nr * ncol; e += blockDim.x) {
                const int r = e / ncol, j = e - r * ncol;
                ncc_cp4(dst + r * RS + j, src + (size_t)r * ncol + j);
            }
        }
        asm volatile("cp.async.commit_group;\n" ::: "memory");
    };
    float stb = 0.f, stt = 0.f, sbb = 0.f;
    int buf = 0;
    if (q0 < q1) issue(q0, 0);
    for (long long q = q0; q < q1; q += NCC_ROWS, buf ^= 1) {
        const int nr = q1 - q < NCC_ROWS ? (int)(q1 - q) : NCC_ROWS;
        if (q + NCC_ROWS < q1) {
            issue(q + NCC_ROWS, buf ^ 1);
            asm volatile("cp.async.wait_group 1;\n" ::: "memory");
        } else {
            asm volatile("cp.async.wait_group 0;\n" ::: "memory");
        }
        __syncthreads();
        if (kk <= N - 1) {
            const float* row = ncc_rows + (size_t)buf * NCC_ROWS * RS + NCC_PADL + (kk - 1);
            for (int r = 0; r < nr; ++r, row += RS) {
                float it = 0.f, ib = 0.f;
#pragma unroll
                for (int i = NCC_FN - 1; i >= 0; --i) it += row[-i];            // i = k - fn + 1 .. k, ascending
#pragma unroll
                for (int i = 1; i <= NCC_FN; ++i) ib += row[i];                 // i = k + 1 .. k + fn
                stb = fmaf(it, ib, stb); stt = fmaf(it, it, stt); sbb = fmaf(ib, ib, sbb);
            }
        }
        __syncthreads();                               // the buffer is refilled two iterations on
    }
    if (threadIdx.x < N) {
        float* o = part + ((size_t)k * NCC_CHUNKS + c) * 3 * N + threadIdx.x;
        o[0] = stb; o[N] = stt; o[2 * N] = sbb;
    }
}

// Step 4.  One CTA per window: the curve in double, its minimum (lowest k on ties; a k whose I_T or I_B vanishes
// everywhere is never chosen; if all do, k = 1).
__global__ void ncc_argmin_kernel(const float* part, int N, double* curve /* [K][N] */, int* cut) {
    __shared__ double val[256];
    __shared__ int idx[256];
    const int k = blockIdx.x, t = threadIdx.x;
    double v = HUGE_VAL;
    if (t < N - 1) {
        double stb = 0.0, stt = 0.0, sbb = 0.0;
        for (int c = 0; c < NCC_CHUNKS; ++c) {
            const float* o = part + ((size_t)k * NCC_CHUNKS + c) * 3 * N + t;
            stb += (double)o[0]; stt += (double)o[N]; sbb += (double)o[2 * N];
        }
        if (stt > 0.0 && sbb > 0.0) v = stb / (sqrt(stt) * sqrt(sbb));
    }
    if (t < N) curve[(size_t)k * N + t] = v;
    val[t] = v; idx[t] = t;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (t < o) {
            const double a = val[t], b = val[t + o];
            if (b < a || (b == a && idx[t + o] < idx[t])) { val[t] = b; idx[t] = idx[t + o]; }
        }
        __syncthreads();
    }
    if (t == 0) cut[k] = (val[0] < HUGE_VAL ? idx[0] : 0) + 1;
}

// Step 5.  Eigen-weights from the cut-off, by rank and by slot, and B_k = V_k diag(wt) (B_k holds V_k on entry).
__global__ void ncc_reweight_kernel(int N, int Ns, int soft, double beta, const int* cut, const int* order, double* wt, float* wslot,
                                    double* wslot_dd, float2* B) {
    __shared__ float ws[256];
    const int k = blockIdx.x, t = threadIdx.x;
    const int c = cut[k];
    if (t < Ns) ws[t] = 0.f;
    __syncthreads();
    if (t < N) {
        const double w = thresh_weight(soft != 0, beta, t + 1, c);           // rank t
        const int u = order[(size_t)k * N + t];
        wt[(size_t)k * N + t] = w;
        wslot[(size_t)k * Ns + u] = (float)w;
        wslot_dd[(size_t)k * Ns + u] = w;
        ws[u] = (float)w;
    }
    __syncthreads();
    float2* Bk = B + (size_t)k * N * Ns;
    for (int e = t; e < N * Ns; e += blockDim.x) {
        const float w = ws[e % Ns];
        const float2 v = Bk[e];
        Bk[e] = make_float2(v.x * w, v.y * w);
    }
}

bool ncc_mode(int mode) { return mode == LCF_HARD_NCC || mode == LCF_SOFT_NCC; }

cudaError_t launch_project_tc_mag(lcf_plan* p, const float2* iq, cudaStream_t st);

cudaError_t launch_ncc(lcf_plan* p, const float2* iq, cudaStream_t st) {
    const int N = p->N, ncol = p->ncc_magN;
    if (p->K == 0 || p->sumPk == 0) return cudaSuccess;
    ncc_isig_kernel<<<p->K, 128, 0, st>>>(p->lam_d, N, ncol, p->ncc_isig_d);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (p->proj_tc) {
        e = launch_project_tc_mag(p, iq, st);
    } else {
        if ((size_t)32 * N * sizeof(float2) > 48 * 1024) {           // above 192 frames the chunk needs the opt-in shared-memory size
            e = set_max_dyn_smem(ncc_mag_kernel, p->smem_optin);
            if (e != cudaSuccess) return e;
        }
        ncc_mag_kernel<<<p->n_pitems, 256, (size_t)32 * N * sizeof(float2), st>>>(iq, N, p->Ns, p->Nz, p->Nx, p->P, p->B_d, p->order_d, p->box_d,
                                                                                  p->pitems_d, p->gz_d, p->gx_d, p->ncc_isig_d, ncol, p->ncc_mag_d);
        e = cudaGetLastError();
    }
    if (e != cudaSuccess) return e;
    {
        const int RS = NCC_PADL + ((ncol + 3) & ~3) + 8;
        const size_t sm = (size_t)2 * NCC_ROWS * RS * sizeof(float);          // <= 70 KB at ncol = 256
        const int thr = N <= 128 ? 128 : 256;
        if (sm > 48 * 1024) {
            e = set_max_dyn_smem(ncc_sums_kernel, p->smem_optin);
            if (e != cudaSuccess) return e;
        }
        ncc_sums_kernel<<<dim3(NCC_CHUNKS, p->K), thr, sm, st>>>(p->ncc_mag_d, N, ncol, p->box_d, p->ncc_part_d);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    ncc_argmin_kernel<<<p->K, 256, 0, st>>>(p->ncc_part_d, N, p->ncc_curve_d, p->cut_d);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    ncc_reweight_kernel<<<p->K, 256, 0, st>>>(N, p->Ns, p->thr.mode == LCF_SOFT_NCC ? 1 : 0, p->thr.beta, p->cut_d, p->order_d, p->wt_d,
                                              p->wslot_d, p->wslot_dd_d, p->B_d);
    return cudaGetLastError();
}

}  // namespace lcf
