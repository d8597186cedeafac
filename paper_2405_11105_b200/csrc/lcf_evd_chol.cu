// lcf_evd_chol.cu -- kernel 2+3, fast path (precision 0, N <= 128): batched Hermitian EVD (Eq. 2,
// PAPER.md:48-50) by pivoted Cholesky + one-sided Jacobi, fused with the eigen-weights and the
// projector factor B_k = V_k diag(wt) (Eq. 9).
//
// One CTA (1024 threads) per window; the matrix lives in shared memory, column-major.
//   1. R' = R + delta I, delta = 3e-5 max_i R_ii (a shift moves eigenvalues, not eigenvectors; it
//      makes the fp32 matrix numerically positive definite and gives rank-deficient windows a
//      complete orthonormal basis).
//   2. Pivoted Cholesky R' = G G^H, right-looking on the full Hermitian storage, no row/column
//      swaps: at step j the largest remaining diagonal entry picks column pi_j, which is scaled in
//      place into the Cholesky column (zero in the rows already eliminated); the rows keep their
//      original order, so G G^H = R' with no permutation to undo.
//   3. One-sided (Hestenes) Jacobi on the columns of G with the round-robin ordering: a plane
//      rotation J of columns (p, q) chosen from the 2x2 Gram [[|g_p|^2, g_p^H g_q], [., |g_q|^2]]
//      makes them orthogonal; G <- G J.  At convergence G W = U Sigma, so R' = U Sigma^2 U^H: the
//      normalised columns ARE the eigenvectors (no separate accumulation of V) and
//      lambda_u = |g_u|^2 - delta.  After the pivoted Cholesky G^H G is strongly diagonally
//      dominant for the graded spectra of clutter-dominated windows (Veselic/Hari, Drmac), so 3-5
//      sweeps replace the 9-10 of two-sided Jacobi on R, and each sweep touches one matrix, not two.
//      16 threads own one column pair per step: 3 dot products reduced by shuffles, one rotation,
//      one barrier per step.  Like two-sided Jacobi this resolves the small (blood / noise)
//      eigen-directions to high relative accuracy: the singular values of G span only the square
//      root of the eigenvalue range.
//   4. Rank the eigenvalues (descending), cut-off rule, eigen-weights, then write V_k and
//      B_k = V_k diag(wt) straight from shared memory.
#include <cfloat>

#include "lcf_internal.h"

namespace lcf {

struct EcArgs {
    int N, NP, Ns, LD;            // Ns = 2 NP column slots (one inert zero column if N is odd); LD = column stride
    int max_sweeps;
    const float2* R;              // [K][N][N] full Hermitian
    double* lam;                  // [K][N] descending
    int* order;                   // [K][N] slot of the i-th largest eigenvalue
    int* cut;                     // [K]
    int* sweeps;                  // [K]
    int* conv;                    // [K]
    float* wslot;                 // [K][Ns]
    double* wslot_dd;             // [K][Ns]
    double* wt;                   // [K][N]
    float2* V;                    // [K][N][Ns]
    float2* B;                    // [K][N][Ns]
    int mode, k_fixed;
    double energy_frac, beta;
};

__device__ __forceinline__ void ec_pair_pq(int m, int s, int M, int& p, int& q) {
    if (m == 0) {
        p = (s == 0) ? 0 : M - s;
        q = M;
    } else {
        p = m - s; if (p < 0) p += M;
        q = M - m - s; if (q < 0) q += M;
    }
}

__global__ void __launch_bounds__(1024, 1) evd_chol_kernel(EcArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = a.N, NP = a.NP, Ns = a.Ns, LD = a.LD, M = Ns - 1;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int k = blockIdx.x;
    float2* G = reinterpret_cast<float2*>(smem_raw);                 // [Ns][LD], element (row i, col u) at u*LD + i
    float2* lj = G + (size_t)Ns * LD;                                // [LD] current Cholesky column
    float* lam_s = reinterpret_cast<float*>(lj + LD);                // [Ns] eigenvalue of slot u
    float* inv_s = lam_s + Ns;                                       // [Ns] 1 / |g_u|
    float* wsl = inv_s + Ns;                                         // [Ns] eigen-weight of slot u
    double* lsort = reinterpret_cast<double*>(wsl + Ns);             // [N] sorted eigenvalues
    int* act = reinterpret_cast<int*>(lsort + Ns);                   // [Ns] row/column still in the trailing matrix
    float* red = reinterpret_cast<float*>(act + Ns);                 // [32]
    int* ish = reinterpret_cast<int*>(red + 32);                     // [4] pivot, flags
    float* fsh = reinterpret_cast<float*>(ish + 4);                  // [4] pivot value, scale

    // ---- load R (row-major [i][j]) into column-major G; zero the padding
    const float2* Rk = a.R + (size_t)k * N * N;
    for (int e = tid; e < Ns * LD; e += 1024) G[e] = make_float2(0.f, 0.f);
    __syncthreads();
    for (int e = tid; e < N * N; e += 1024) {
        const int i = e / N, j = e - i * N;                          // coalesced read of row i
        G[(size_t)j * LD + i] = Rk[e];
    }
    if (tid < Ns) act[tid] = tid < N ? 1 : 0;
    __syncthreads();
    float md = 0.f;
    if (tid < N) md = G[(size_t)tid * LD + tid].x;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) md = fmaxf(md, __shfl_xor_sync(0xffffffffu, md, o));
    if (lane == 0) red[warp] = md;
    __syncthreads();
    float maxdiag = 0.f;
    for (int w = 0; w < 32; ++w) maxdiag = fmaxf(maxdiag, red[w]);
    const float delta = 3e-5f * maxdiag;
    int sweep = 0, converged = 1;

    if (maxdiag > 0.f) {
        if (tid < N) { G[(size_t)tid * LD + tid].x += delta; G[(size_t)tid * LD + tid].y = 0.f; }
        __syncthreads();
        // ---- 2. pivoted Cholesky, in place
        for (int j = 0; j < N; ++j) {
            if (warp == 0) {
                float best = -FLT_MAX; int bi = N;
                for (int i = lane; i < N; i += 32)
                    if (act[i]) { const float d = G[(size_t)i * LD + i].x; if (d > best) { best = d; bi = i; } }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    const float ob = __shfl_xor_sync(0xffffffffu, best, o);
                    const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                    if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
                }
                if (lane == 0) {
                    // a non-positive pivot can only come from rounding: clamp (the column is then ~0)
                    const float piv = fmaxf(best, 1e-30f * maxdiag + 1e-37f);
                    ish[0] = bi; fsh[0] = sqrtf(piv); fsh[1] = rsqrtf(piv);
                }
            }
            __syncthreads();
            const int pv = ish[0];
            const float dsq = fsh[0], sc = fsh[1];
            if (tid < LD) {
                float2 v = make_float2(0.f, 0.f);
                if (tid == pv) v.x = dsq;
                else if (tid < N && act[tid]) { const float2 x = G[(size_t)pv * LD + tid]; v = make_float2(x.x * sc, x.y * sc); }
                G[(size_t)pv * LD + tid] = v;                         // Cholesky column pi_j, zero in eliminated rows
                lj[tid] = (tid == pv) ? make_float2(0.f, 0.f) : v;    // multiplier for the trailing update
            }
            __syncthreads();
            if (tid == 0) act[pv] = 0;
            // trailing update A[i][l] -= L[i] conj(L[l]) on the still-active columns l (8 threads per column)
            {
                const int l = tid >> 3, rr = tid & 7;
                if (l < N && l != pv && act[l]) {
                    const float2 ll = lj[l];
                    float2* col = G + (size_t)l * LD;
                    for (int i0 = 2 * rr; i0 < N; i0 += 16) {
                        float4 x = *reinterpret_cast<float4*>(&col[i0]);
                        const float4 m2 = *reinterpret_cast<const float4*>(&lj[i0]);
                        // x -= m * conj(ll)
                        x.x -= m2.x * ll.x + m2.y * ll.y;  x.y -= m2.y * ll.x - m2.x * ll.y;
                        x.z -= m2.z * ll.x + m2.w * ll.y;  x.w -= m2.w * ll.x - m2.z * ll.y;
                        *reinterpret_cast<float4*>(&col[i0]) = x;
                    }
                }
            }
            __syncthreads();
        }
        // ---- 3. one-sided Jacobi on the columns of G
        const float tol = 4.f * sqrtf((float)N) * FLT_EPSILON;
        const float tol2 = tol * tol;
        const int m = tid >> 4, r = tid & 15;
        const unsigned hmask = (lane < 16) ? 0x0000ffffu : 0xffff0000u;   // m < NP is uniform per half warp
        converged = 0;
        for (;;) {
            int any = 0;
            for (int s = 0; s < M; ++s) {
                int rot = 0;
                if (m < NP) {
                    int p, q; ec_pair_pq(m, s, M, p, q);
                    float2* gp = G + (size_t)p * LD;
                    float2* gq = G + (size_t)q * LD;
                    float4 xp[4], xq[4];
                    float app = 0.f, aqq = 0.f, xr = 0.f, xi = 0.f;
#pragma unroll
                    for (int c = 0; c < 4; ++c) {
                        const int i0 = 2 * r + 32 * c;
                        if (i0 < N) {
                            xp[c] = *reinterpret_cast<const float4*>(&gp[i0]);
                            xq[c] = *reinterpret_cast<const float4*>(&gq[i0]);
                            app = fmaf(xp[c].x, xp[c].x, fmaf(xp[c].y, xp[c].y, fmaf(xp[c].z, xp[c].z, fmaf(xp[c].w, xp[c].w, app))));
                            aqq = fmaf(xq[c].x, xq[c].x, fmaf(xq[c].y, xq[c].y, fmaf(xq[c].z, xq[c].z, fmaf(xq[c].w, xq[c].w, aqq))));
                            // conj(g_p) g_q
                            xr = fmaf(xp[c].x, xq[c].x, fmaf(xp[c].y, xq[c].y, fmaf(xp[c].z, xq[c].z, fmaf(xp[c].w, xq[c].w, xr))));
                            xi = fmaf(xp[c].x, xq[c].y, fmaf(-xp[c].y, xq[c].x, fmaf(xp[c].z, xq[c].w, fmaf(-xp[c].w, xq[c].z, xi))));
                        }
                    }
#pragma unroll
                    for (int o = 8; o > 0; o >>= 1) {                 // within the pair's 16 lanes
                        app += __shfl_xor_sync(hmask, app, o);
                        aqq += __shfl_xor_sync(hmask, aqq, o);
                        xr += __shfl_xor_sync(hmask, xr, o);
                        xi += __shfl_xor_sync(hmask, xi, o);
                    }
                    const float absa2 = xr * xr + xi * xi;
                    if (absa2 > tol2 * app * aqq && absa2 > 0.f) {
                        rot = 1;
                        const float inv = rsqrtf(absa2);
                        const float absa = absa2 * inv;
                        const float tau = (aqq - app) * (0.5f * inv);
                        const float at = fabsf(tau);
                        float t = (at > 1e8f) ? 0.5f / at : 1.f / (at + sqrtf(1.f + tau * tau));
                        if (tau < 0.f) t = -t;
                        const float cs = rsqrtf(1.f + t * t);
                        const float sn = t * cs;
                        const float gr = sn * xr * inv, gi = sn * xi * inv;
                        (void)absa;
#pragma unroll
                        for (int c = 0; c < 4; ++c) {
                            const int i0 = 2 * r + 32 * c;
                            if (i0 < N) {
                                float4 np_, nq_;
                                // g_p' = c g_p - conj(g) g_q,   g_q' = g g_p + c g_q
                                np_.x = cs * xp[c].x - (gr * xq[c].x + gi * xq[c].y);
                                np_.y = cs * xp[c].y - (gr * xq[c].y - gi * xq[c].x);
                                np_.z = cs * xp[c].z - (gr * xq[c].z + gi * xq[c].w);
                                np_.w = cs * xp[c].w - (gr * xq[c].w - gi * xq[c].z);
                                nq_.x = (gr * xp[c].x - gi * xp[c].y) + cs * xq[c].x;
                                nq_.y = (gr * xp[c].y + gi * xp[c].x) + cs * xq[c].y;
                                nq_.z = (gr * xp[c].z - gi * xp[c].w) + cs * xq[c].z;
                                nq_.w = (gr * xp[c].w + gi * xp[c].z) + cs * xq[c].w;
                                *reinterpret_cast<float4*>(&gp[i0]) = np_;
                                *reinterpret_cast<float4*>(&gq[i0]) = nq_;
                            }
                        }
                    }
                }
                any |= __syncthreads_or(rot);
            }
            ++sweep;
            if (!any) { converged = 1; break; }
            if (sweep == a.max_sweeps) break;
        }
    } else {
        // zero matrix (empty window): V = I, all eigenvalues 0
        if (tid < N) G[(size_t)tid * LD + tid] = make_float2(1.f, 0.f);
        __syncthreads();
    }

    // ---- 4. eigenvalues = squared column norms - delta, eigenvectors = normalised columns
    {
        const int u = tid >> 3, rr = tid & 7;                        // 8 threads per column
        float nn = 0.f;
        if (u < Ns) {
            const float2* col = G + (size_t)u * LD;
            for (int i0 = 2 * rr; i0 < N; i0 += 16) {
                const float4 x = *reinterpret_cast<const float4*>(&col[i0]);
                nn = fmaf(x.x, x.x, fmaf(x.y, x.y, fmaf(x.z, x.z, fmaf(x.w, x.w, nn))));
            }
        }
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) nn += __shfl_xor_sync(0xffffffffu, nn, o);
        if (u < Ns && rr == 0) {
            lam_s[u] = (maxdiag > 0.f && u < N) ? nn - delta : 0.f;
            inv_s[u] = nn > 0.f ? rsqrtf(nn) : 0.f;
        }
    }
    __syncthreads();
    // rank (descending, ties by slot index), cut-off, eigen-weights: same rules as jacobi_kernel
    float myl = 0.f;
    int rank = 0;
    if (tid < N) {
        myl = lam_s[tid];
        for (int j = 0; j < N; ++j) {
            const float ljv = lam_s[j];
            rank += (ljv > myl) || (ljv == myl && j < tid);
        }
        lsort[rank] = (double)myl;
        a.lam[(size_t)k * N + rank] = (double)myl;
        a.order[(size_t)k * N + rank] = tid;
    }
    __syncthreads();
    if (tid == 0) {
        int c = a.k_fixed;
        if (a.mode == LCF_HARD_ENERGY || a.mode == LCF_SOFT_ENERGY) {
            double tot = 0.0;
            for (int i = 0; i < N; ++i) tot += lsort[i] > 0.0 ? lsort[i] : 0.0;
            double cum = 0.0;
            c = N;
            for (int mm = 1; mm <= N; ++mm) {
                cum += lsort[mm - 1] > 0.0 ? lsort[mm - 1] : 0.0;
                if (cum > a.energy_frac * tot) { c = mm; break; }
            }
        }
        ish[1] = c;
        a.cut[k] = c;
        a.sweeps[k] = sweep;
        a.conv[k] = converged;
    }
    __syncthreads();
    {
        const int c = ish[1];
        const bool soft = (a.mode == LCF_SOFT_FIXED || a.mode == LCF_SOFT_ENERGY);
        if (tid < Ns) {
            double w = 0.0;
            if (tid < N) {
                const int i1 = rank + 1;                             // 1-based order of the eigenvalue in slot tid
                if (soft) w = 1.0 / (1.0 + exp(-a.beta * (double)(i1 - c)));
                else w = (i1 <= c) ? 0.0 : 1.0;
                a.wt[(size_t)k * N + rank] = w;
            }
            wsl[tid] = (float)w;
            a.wslot[(size_t)k * Ns + tid] = (float)w;
            a.wslot_dd[(size_t)k * Ns + tid] = w;
        }
    }
    __syncthreads();
    // V[a][u] = G[a][u] / |g_u|,  B = V diag(wt): lanes run over the slot u (coalesced global writes)
    float2* Vk = a.V + (size_t)k * N * Ns;
    float2* Bk = a.B + (size_t)k * N * Ns;
    for (int e = tid; e < N * Ns; e += 1024) {
        const int row = e / Ns, u = e - row * Ns;
        const float2 x = G[(size_t)u * LD + row];
        const float s1 = inv_s[u], w = wsl[u];
        const float2 v = make_float2(x.x * s1, x.y * s1);
        Vk[e] = v;
        Bk[e] = make_float2(v.x * w, v.y * w);
    }
}

static size_t ec_smem_bytes(int Ns, int LD) {
    return (size_t)Ns * LD * 8 + (size_t)LD * 8 + 3 * (size_t)Ns * 4 + (size_t)Ns * 8 + (size_t)Ns * 4 + 32 * 4 + 16 + 16 + 64;
}

bool evd_chol_eligible(const lcf_plan* p) { return p->prec == 0 && p->N <= 128 && p->N >= 2; }

cudaError_t configure_evd_chol(lcf_plan* p) {
    p->ec_LD = ((p->N + 1) & ~1) + 2;
    p->ec_smem = ec_smem_bytes(p->Ns, p->ec_LD);
    if (p->ec_smem > (size_t)p->smem_optin) return cudaErrorInvalidConfiguration;
    return cudaFuncSetAttribute(evd_chol_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->ec_smem);
}

cudaError_t launch_evd_chol(lcf_plan* p, cudaStream_t st) {
    EcArgs a;
    a.N = p->N; a.NP = p->NP; a.Ns = p->Ns; a.LD = p->ec_LD; a.max_sweeps = 30;
    a.R = reinterpret_cast<const float2*>(p->R_d);
    a.lam = p->lam_d; a.order = p->order_d; a.cut = p->cut_d; a.sweeps = p->sweeps_d; a.conv = p->conv_d;
    a.wslot = p->wslot_d; a.wslot_dd = p->wslot_dd_d; a.wt = p->wt_d;
    a.V = reinterpret_cast<float2*>(p->V_d); a.B = p->B_d;
    a.mode = p->thr.mode; a.k_fixed = p->thr.k_fixed; a.energy_frac = p->thr.energy_frac; a.beta = p->thr.beta;
    evd_chol_kernel<<<p->K, 1024, p->ec_smem, st>>>(a);
    return cudaGetLastError();
}

}  // namespace lcf
