// lcf_evd_chol.cu -- kernel 2+3, fast path (precision 0, N <= 128): batched Hermitian EVD (Eq. 2,
// PAPER.md:48-50) by pivoted Cholesky + one-sided Jacobi, fused with the eigen-weights and the
// projector factor B_k = V_k diag(wt) (Eq. 9).
//
// One CTA (512 threads) per window; the matrix lives in shared memory, column-major, real and
// imaginary planes apart so that two rows make one f32x2 operand (packed FP32 pipe).
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
//      lambda_u = |g_u|^2 - delta.  The singular values of G span only the square root of the
//      eigenvalue range, so the small (blood / noise) eigen-directions keep the relative accuracy
//      that makes Jacobi the right fp32 solver here (a tridiagonal QR in fp32 would lose them
//      under the 50-60 dB of clutter).  Measured: 8-10 sweeps, as many as two-sided Jacobi on R
//      needs -- the flat noise floor, not the graded clutter part, sets the sweep count -- but each
//      sweep touches one matrix instead of two (no V accumulation) with unit-stride columns.
//      8 threads own one column pair per step: 3 dot products reduced by shuffles, one rotation,
//      one barrier per step.  (With even N >= 32 only steps 1-2 run here, `chol_only`, and the
//      sweeps run on 2-CTA clusters: lcf_evd_cluster.cu.)
//   4. Rank the eigenvalues (descending), cut-off rule, eigen-weights, then write V_k and
//      B_k = V_k diag(wt) straight from shared memory.
#include <cfloat>

#include "lcf_internal.h"
#include "lcf_sm100.cuh"
#include "lcf_thresh.cuh"

namespace lcf {

struct EcArgs {
    int N, NP, Ns, LD;            // Ns = 2 NP column slots (one inert zero column if N is odd); LD = column stride
    int max_sweeps;
    const float2* R;              // [K][N][N] full Hermitian
    const uint32_t* amax;         // non-null: R carries the power-of-two data scale of the tensor-core Gram (squared); eigenvalues are unscaled here
    double* lam;                  // [K][N] descending
    int* order;                   // [K][N] slot of the i-th largest eigenvalue
    int* cut;                     // [K]
    int* sweeps;                  // [K]
    int* conv;                    // [K]
    int* nunconv;                 // [1] count of window EVDs that hit the sweep cap
    float* wslot;                 // [K][Ns]
    double* wslot_dd;             // [K][Ns]
    double* wt;                   // [K][N]
    float2* V;                    // [K][N][Ns]
    float2* B;                    // [K][N][Ns]
    int mode, k_fixed;
    double energy_frac, beta, cut_scale;
    int chol_only;                // 1: stop after the Cholesky factor and write it to gfac / shift (cluster Jacobi follows)
    float* gfac;                  // [K][2][Ns][LD] real plane, imaginary plane of G, column-major
    float* shift;                 // [K] delta, or -1 for an all-zero matrix
    int* nexp;                    // [K] power-of-two exponent this kernel scaled R_k by (0 when R carries the tensor-core data scale)
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

constexpr int EC_THREADS = 512;   // 8 threads per column pair (NP <= 64 pairs)
constexpr int EC_NB = 8;                   // Cholesky steps per block

__device__ __forceinline__ unsigned long long ec_fma2(unsigned long long a, unsigned long long b, unsigned long long c) {
    unsigned long long d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ unsigned long long ec_mul2(unsigned long long a, unsigned long long b) {
    unsigned long long d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ unsigned long long ec_pack(float x, float y) {
    unsigned long long d;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(x), "f"(y));
    return d;
}
__device__ __forceinline__ float ec_hsum(unsigned long long v) {
    float x, y;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(v));
    return x + y;
}

template <int NC, bool FULL, bool GLOB>
__global__ void __launch_bounds__(EC_THREADS, 1) evd_chol_kernel(EcArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double wnorm_sh;                                      // normalisation of the adaptive weights (method 6)
    const int N = a.N, NP = a.NP, Ns = a.Ns, LD = a.LD, M = Ns - 1;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int k = blockIdx.x;
    // planar storage: real and imaginary parts of column u at Gr/Gi + u*LD (LD floats, multiple of 4)
    // (GLOB: the factor does not fit shared memory -- N > 128 -- and is built in place in gfac, global memory, L2-resident;
    // a template parameter, so that the shared-memory variant keeps shared-space loads and stores)
    float* Gr = GLOB ? a.gfac + (size_t)k * 2 * Ns * LD : reinterpret_cast<float*>(smem_raw);   // [Ns][LD]
    float* Gi = Gr + (size_t)Ns * LD;                                // [Ns][LD]
    float* lam_s = GLOB ? reinterpret_cast<float*>(smem_raw) : Gi + (size_t)Ns * LD;            // [Ns] eigenvalue of slot u
    float* inv_s = lam_s + Ns;                                       // [Ns] 1 / |g_u|
    float* wsl = inv_s + Ns;                                         // [Ns] eigen-weight of slot u
    float* red = wsl + Ns;                                           // [32]
    double* lsort = reinterpret_cast<double*>(red + 32);             // [Ns] sorted eigenvalues
    int* ish = reinterpret_cast<int*>(lsort + Ns);                                             // [4] pivot, cut-off
    int* alist = ish + 4;                                            // [Ns] pivot order of the Cholesky steps

    // ---- load R (row-major [i][j]) into the column-major planes (conflict-free: row i lands in column i); zero the padding
    const float2* Rk = a.R + (size_t)k * N * N;
    for (int e = tid; e < 2 * Ns * LD; e += EC_THREADS) Gr[e] = 0.f;
    __syncthreads();
    for (int e = tid; e < N * N; e += EC_THREADS) {
        const int i = e / N, j = e - i * N;                          // coalesced read of row i = conj of column i (R is Hermitian)
        const float2 x = Rk[e];
        Gr[(size_t)i * LD + j] = x.x;
        Gi[(size_t)i * LD + j] = -x.y;
    }
    __syncthreads();
    float md = 0.f;
    if (tid < N) md = Gr[(size_t)tid * LD + tid];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) md = fmaxf(md, __shfl_xor_sync(0xffffffffu, md, o));
    if (lane == 0) red[warp] = md;
    __syncthreads();
    float maxdiag = 0.f;
    for (int w = 0; w < EC_THREADS / 32; ++w) maxdiag = fmaxf(maxdiag, red[w]);
    // R from the CUDA-core Gram is in raw units (amplitude^2 P): bring it to a fixed magnitude (largest diagonal entry
    // in [1, 2)) by an exact power of two, so that the squared norms and their products in the Cholesky and Jacobi
    // tests stay in range whatever the units; undone when the eigenvalues leave (the tensor-core Gram's R already
    // has a fixed scale)
    int nexp = 0;
    if (!a.amax && maxdiag > 0.f && maxdiag < 3.0e38f) {
        int ex;
        frexpf(maxdiag, &ex);
        nexp = 1 - ex;
        nexp = nexp < -120 ? -120 : (nexp > 120 ? 120 : nexp);
        const float sc = ldexpf(1.f, nexp);
        __syncthreads();
        for (int e = tid; e < 2 * Ns * LD; e += EC_THREADS) Gr[e] *= sc;
        maxdiag *= sc;
        __syncthreads();
    }
    if (tid == 0) a.nexp[k] = nexp;
    const float delta = 3e-5f * maxdiag;
    int sweep = 0, converged = 1;

    if (maxdiag > 0.f) {
        if (tid < N) { Gr[(size_t)tid * LD + tid] += delta; Gi[(size_t)tid * LD + tid] = 0.f; }
        __syncthreads();
        // ---- 2. pivoted Cholesky in blocks of EC_NB steps.  Inside a block the chosen column is
        // brought up to date against the block's finished columns only (left-looking over at most
        // EC_NB - 1 columns: one thread per row); at the end of a block every column still to be
        // eliminated takes the block's rank-EC_NB update at once (right-looking: one warp per column,
        // the block's columns held in registers), so the trailing matrix crosses shared memory once per
        // EC_NB steps.  The pivot search is a warp-wide integer maximum (redux) over keys that hold the
        // diagonal entry's top 25 bits above 127 - row (ties, and near-ties within 2^-16, go to the
        // lowest row): each warp reduces its rows when it downdates them, and after the step's barrier
        // every warp reduces the 16 warp keys.
        const int nchc = (N + 3) >> 2;                               // 4-row chunks per column
        const unsigned KM = N > 128 ? 255u : 127u;                   // row index bits of a pivot key
        // Between two barriers a warp both reads what the step needs from the others (the 16 warp keys, the pivot's
        // diagonal entry) and writes what the next step needs; a warp that runs a whole step ahead of a slow one must
        // not change what the slow one still has to read.  So the warp keys alternate between two sets by step
        // parity, and the diagonal of an eliminated row is left in place (its flag elim[] is what marks it).
        float* dgs = lam_s;                                          // [N] current diagonal of the Schur complement
        int* elim = reinterpret_cast<int*>(wsl);                     // [N] 1 once the row is a pivot (wsl is free until the epilogue)
        unsigned* wkey = reinterpret_cast<unsigned*>(red);           // [2][16] per-warp pivot keys, set (j & 1) read at step j
        int* elist = alist;                                          // [N] pivot of step t = slot of Cholesky column t
        {
            unsigned key = 0u;
            if (tid < N) {
                const float d = fmaxf(Gr[(size_t)tid * LD + tid], 0.f);
                dgs[tid] = d;
                elim[tid] = 0;
                key = (__float_as_uint(d) & ~KM) | (KM - (unsigned)tid);
            }
            key = __reduce_max_sync(0xffffffffu, key);
            if (lane == 0) wkey[warp] = key;
        }
        __syncthreads();
        bool exhausted = false;                                      // (every thread decides it from the same dgs[pv]: uniform)
        for (int jb = 0; jb < N; jb += EC_NB) {
            const int je = jb + EC_NB < N ? jb + EC_NB : N;
            for (int j = jb; j < je; ++j) {
                unsigned kk = lane < EC_THREADS / 32 ? wkey[(j & 1) * 16 + lane] : 0u;
                kk = __reduce_max_sync(0xffffffffu, kk);
                const int pv = (int)(KM - (kk & KM));
                unsigned key = 0u;
                if (tid < N) {
                    // R + delta I >= delta I, so every Schur complement has its diagonal >= delta.  R comes out of fp32-grade
                    // arithmetic, though: its smallest eigenvalues are off by a few ulp of the LARGEST one (a rank-deficient
                    // window of 208 coherent frames: down to -3.7e-5 maxdiag, beyond the shift), the matrix is then indefinite
                    // and going on would amplify rounding noise step by step (1e20 and NaN, found by random shapes).  A pivot
                    // below delta / 2 says what is left is that noise: from there on the remaining columns keep their
                    // diagonal only (G G^H then differs from R + delta I by off-diagonal noise of the order of delta).
                    const float praw = dgs[pv];
                    if (praw < 0.5f * delta) exhausted = true;
                    const float piv = fmaxf(praw, 0.25f * delta);
                    const float sc = rsqrtf(piv), dsq = piv * sc;
                    const int i = tid;
                    float sr = 0.f, si = 0.f;
                    for (int t = jb; t < j; ++t) {                   // G[i, e_t] conj(G[pv, e_t]) over the block's finished columns
                        const float* cr = Gr + (size_t)elist[t] * LD;
                        const float* ci = Gi + (size_t)elist[t] * LD;
                        const float gr = cr[i], gi = ci[i], lr = cr[pv], li = ci[pv];
                        sr = fmaf(gr, lr, fmaf(gi, li, sr));
                        si = fmaf(gi, lr, fmaf(-gr, li, si));
                    }
                    const float d = dgs[i];
                    float vr = 0.f, vi = 0.f;                        // Cholesky column pi_j is zero in eliminated rows
                    if (i == pv) { vr = dsq; elim[i] = 1; }
                    else if (!elim[i]) {
                        if (!exhausted) {
                            vr = (Gr[(size_t)pv * LD + i] - sr) * sc;
                            vi = (Gi[(size_t)pv * LD + i] - si) * sc;
                        }
                        const float nd = fmaxf(d - (vr * vr + vi * vi), 0.f);
                        dgs[i] = nd;
                        key = (__float_as_uint(nd) & ~KM) | (KM - (unsigned)i);
                    }
                    Gr[(size_t)pv * LD + i] = vr;
                    Gi[(size_t)pv * LD + i] = vi;
                    if (tid == 0) elist[j] = pv;
                }
                key = __reduce_max_sync(0xffffffffu, key);
                if (lane == 0) wkey[((j + 1) & 1) * 16 + warp] = key;
                __syncthreads();
            }
            if (je < N) {
                // rank-(je - jb) update of the columns still to be eliminated (row chunks lane, lane + 32, ...)
                const float* gcol[EC_NB];
#pragma unroll
                for (int t = 0; t < EC_NB; ++t) gcol[t] = Gr + (size_t)elist[jb + t < je ? jb + t : jb] * LD;
                for (int c0 = 0; c0 < nchc; c0 += 32) {
                    const int ch = c0 + lane;
                    float4 gbr[EC_NB], gbi[EC_NB];
#pragma unroll
                    for (int t = 0; t < EC_NB; ++t) {
                        gbr[t] = gbi[t] = make_float4(0.f, 0.f, 0.f, 0.f);
                        if (jb + t < je && ch < nchc) {
                            gbr[t] = *reinterpret_cast<const float4*>(&gcol[t][4 * ch]);
                            gbi[t] = *reinterpret_cast<const float4*>(&gcol[t][(size_t)Ns * LD + 4 * ch]);
                        }
                    }
                    for (int l = warp; l < N; l += EC_THREADS / 32) {
                        if (elim[l]) continue;                       // already a Cholesky column
                        if (ch < nchc) {
                            float* cr = Gr + (size_t)l * LD + 4 * ch;
                            float* ci = Gi + (size_t)l * LD + 4 * ch;
                            float4 xr = *reinterpret_cast<float4*>(cr), xi = *reinterpret_cast<float4*>(ci);
#pragma unroll
                            for (int t = 0; t < EC_NB; ++t) {
                                // x -= g_t conj(G[l, e_t]):  re -= gr lr + gi li,  im -= gi lr - gr li  (zero columns for t >= je - jb)
                                const float lr = gcol[t][l], li = gcol[t][(size_t)Ns * LD + l];
                                xr.x -= gbr[t].x * lr + gbi[t].x * li;  xi.x -= gbi[t].x * lr - gbr[t].x * li;
                                xr.y -= gbr[t].y * lr + gbi[t].y * li;  xi.y -= gbi[t].y * lr - gbr[t].y * li;
                                xr.z -= gbr[t].z * lr + gbi[t].z * li;  xi.z -= gbi[t].z * lr - gbr[t].z * li;
                                xr.w -= gbr[t].w * lr + gbi[t].w * li;  xi.w -= gbi[t].w * lr - gbr[t].w * li;
                            }
                            *reinterpret_cast<float4*>(cr) = xr;
                            *reinterpret_cast<float4*>(ci) = xi;
                        }
                    }
                }
                __syncthreads();
            }
        }
        if (a.chol_only) {
            float* gout = a.gfac + (size_t)k * 2 * Ns * LD;
            if (!GLOB) for (int e = tid; e < 2 * Ns * LD; e += EC_THREADS) gout[e] = Gr[e];
            if (tid == 0) a.shift[k] = delta;
            return;
        }
        // ---- 3. one-sided Jacobi on the columns of G: 8 threads per pair, 4-row chunks t + 8c
        const float tol = 4.f * sqrtf((float)N) * FLT_EPSILON;
        const float tol2 = tol * tol;
        const int m = tid >> 3, r = tid & 7;
        const unsigned qmask = 0xffu << (lane & 24);                 // the pair's 8 lanes (m < NP is uniform over them)
        const int nch = (N + 3) >> 2;                                // 4-row chunks per column
        converged = 0;
        for (;;) {
            int any = 0;
            for (int s = 0; s < M; ++s) {
                if (m < NP) {
                    int p, q; ec_pair_pq(m, s, M, p, q);
                    float* pr_ = Gr + (size_t)p * LD; float* pi_ = Gi + (size_t)p * LD;
                    float* qr_ = Gr + (size_t)q * LD; float* qi_ = Gi + (size_t)q * LD;
                    ulonglong2 PR[NC], PI[NC], QR[NC], QI[NC];
                    unsigned long long app2 = 0ull, aqq2 = 0ull, re2 = 0ull, ima2 = 0ull, imb2 = 0ull;
#pragma unroll
                    for (int c = 0; c < NC; ++c) {
                        const int ch = r + 8 * c;
                        if (FULL || ch < nch) {
                            PR[c] = *reinterpret_cast<const ulonglong2*>(&pr_[4 * ch]);
                            PI[c] = *reinterpret_cast<const ulonglong2*>(&pi_[4 * ch]);
                            QR[c] = *reinterpret_cast<const ulonglong2*>(&qr_[4 * ch]);
                            QI[c] = *reinterpret_cast<const ulonglong2*>(&qi_[4 * ch]);
                            app2 = ec_fma2(PR[c].x, PR[c].x, app2); app2 = ec_fma2(PI[c].x, PI[c].x, app2);
                            app2 = ec_fma2(PR[c].y, PR[c].y, app2); app2 = ec_fma2(PI[c].y, PI[c].y, app2);
                            aqq2 = ec_fma2(QR[c].x, QR[c].x, aqq2); aqq2 = ec_fma2(QI[c].x, QI[c].x, aqq2);
                            aqq2 = ec_fma2(QR[c].y, QR[c].y, aqq2); aqq2 = ec_fma2(QI[c].y, QI[c].y, aqq2);
                            // conj(g_p) g_q = (pr qr + pi qi) + i (pr qi - pi qr)
                            re2 = ec_fma2(PR[c].x, QR[c].x, re2);   re2 = ec_fma2(PI[c].x, QI[c].x, re2);
                            re2 = ec_fma2(PR[c].y, QR[c].y, re2);   re2 = ec_fma2(PI[c].y, QI[c].y, re2);
                            ima2 = ec_fma2(PR[c].x, QI[c].x, ima2); imb2 = ec_fma2(PI[c].x, QR[c].x, imb2);
                            ima2 = ec_fma2(PR[c].y, QI[c].y, ima2); imb2 = ec_fma2(PI[c].y, QR[c].y, imb2);
                        }
                    }
                    float app = ec_hsum(app2), aqq = ec_hsum(aqq2), xr = ec_hsum(re2), xi = ec_hsum(ima2) - ec_hsum(imb2);
#pragma unroll
                    for (int o = 4; o > 0; o >>= 1) {
                        app += __shfl_xor_sync(qmask, app, o);
                        aqq += __shfl_xor_sync(qmask, aqq, o);
                        xr += __shfl_xor_sync(qmask, xr, o);
                        xi += __shfl_xor_sync(qmask, xi, o);
                    }
                    const float absa2 = xr * xr + xi * xi;
                    if (absa2 > tol2 * app * aqq && absa2 > 0.f) {
                        any = 1;
                        // rotation parameters as in lcf_evd_cluster.cu (ecb_round_tracked): unitary to rounding without bias
                        const float alpha = 0.5f * (aqq - app);
                        const float rinv = rsqrtf(fmaxf(fmaf(alpha, alpha, absa2), 1e-37f));
                        const float c2h = fmaf(0.5f * fabsf(alpha), rinv, 0.5f);
                        const float rc = rsqrtf(c2h);
                        const float cs0 = c2h * rc;
                        const float kk = copysignf(0.5f * rinv * rc, alpha);
                        const float gr = kk * xr, gi = kk * xi;
                        const float resid = fmaf(-cs0, cs0, 1.f) - fmaf(gr, gr, gi * gi);
                        const float cs = fmaf(0.5f * rc, resid, cs0);
                        const unsigned long long c2 = ec_pack(cs, cs), gr2 = ec_pack(gr, gr), gi2 = ec_pack(gi, gi);
                        const unsigned long long ngr2 = ec_pack(-gr, -gr), ngi2 = ec_pack(-gi, -gi);
#pragma unroll
                        for (int c = 0; c < NC; ++c) {
                            const int ch = r + 8 * c;
                            if (FULL || ch < nch) {
                                ulonglong2 npr, npi, nqr, nqi;
                                // g_p' = c g_p - conj(g) g_q,   g_q' = g g_p + c g_q
                                npr.x = ec_fma2(ngi2, QI[c].x, ec_fma2(ngr2, QR[c].x, ec_mul2(c2, PR[c].x)));
                                npr.y = ec_fma2(ngi2, QI[c].y, ec_fma2(ngr2, QR[c].y, ec_mul2(c2, PR[c].y)));
                                npi.x = ec_fma2(gi2, QR[c].x, ec_fma2(ngr2, QI[c].x, ec_mul2(c2, PI[c].x)));
                                npi.y = ec_fma2(gi2, QR[c].y, ec_fma2(ngr2, QI[c].y, ec_mul2(c2, PI[c].y)));
                                nqr.x = ec_fma2(c2, QR[c].x, ec_fma2(ngi2, PI[c].x, ec_mul2(gr2, PR[c].x)));
                                nqr.y = ec_fma2(c2, QR[c].y, ec_fma2(ngi2, PI[c].y, ec_mul2(gr2, PR[c].y)));
                                nqi.x = ec_fma2(c2, QI[c].x, ec_fma2(gi2, PR[c].x, ec_mul2(gr2, PI[c].x)));
                                nqi.y = ec_fma2(c2, QI[c].y, ec_fma2(gi2, PR[c].y, ec_mul2(gr2, PI[c].y)));
                                *reinterpret_cast<ulonglong2*>(&pr_[4 * ch]) = npr;
                                *reinterpret_cast<ulonglong2*>(&pi_[4 * ch]) = npi;
                                *reinterpret_cast<ulonglong2*>(&qr_[4 * ch]) = nqr;
                                *reinterpret_cast<ulonglong2*>(&qi_[4 * ch]) = nqi;
                            }
                        }
                    }
                }
                __syncthreads();
            }
            ++sweep;
            if (!__syncthreads_or(any)) { converged = 1; break; }
            if (sweep == a.max_sweeps) break;
        }
    } else {
        // zero matrix (empty window): V = I, all eigenvalues 0
        if (tid < N) Gr[(size_t)tid * LD + tid] = 1.f;
        __syncthreads();
        if (a.chol_only) {
            float* gout = a.gfac + (size_t)k * 2 * Ns * LD;
            if (!GLOB) for (int e = tid; e < 2 * Ns * LD; e += EC_THREADS) gout[e] = Gr[e];
            if (tid == 0) a.shift[k] = -1.f;
            return;
        }
    }

    // ---- 4. eigenvalues = squared column norms - delta, eigenvectors = normalised columns
    {
        const int u = tid >> 2, rr = tid & 3;                        // 4 threads per column
        float nn = 0.f;
        if (u < Ns) {
            const float* cr = Gr + (size_t)u * LD;
            const float* ci = Gi + (size_t)u * LD;
            for (int i0 = 4 * rr; i0 < N; i0 += 16) {
                const float4 x = *reinterpret_cast<const float4*>(&cr[i0]);
                const float4 y = *reinterpret_cast<const float4*>(&ci[i0]);
                nn = fmaf(x.x, x.x, fmaf(x.y, x.y, fmaf(x.z, x.z, fmaf(x.w, x.w, nn))));
                nn = fmaf(y.x, y.x, fmaf(y.y, y.y, fmaf(y.z, y.z, fmaf(y.w, y.w, nn))));
            }
        }
#pragma unroll
        for (int o = 2; o > 0; o >>= 1) nn += __shfl_xor_sync(0xffffffffu, nn, o);
        if (u < Ns && rr == 0) {
            lam_s[u] = (maxdiag > 0.f && u < N) ? nn - delta : 0.f;
            inv_s[u] = nn > 0.f ? rsqrtf(nn) : 0.f;
        }
    }
    __syncthreads();
    // rank (descending, ties by slot index), cut-off, eigen-weights: same rules as jacobi_kernel
    const double un = a.amax ? ldexp(1.0, -2 * sm100::pow2_scale_exp(*a.amax)) : ldexp(1.0, -nexp);
    float myl = 0.f;
    int rank = 0;
    if (tid < N) {
        myl = lam_s[tid];
        for (int j = 0; j < N; ++j) {
            const float ljv = lam_s[j];
            rank += (ljv > myl) || (ljv == myl && j < tid);
        }
        lsort[rank] = (double)myl * un;
        a.lam[(size_t)k * N + rank] = (double)myl * un;
        a.order[(size_t)k * N + rank] = tid;
    }
    __syncthreads();
    if (tid == 0) {
        const int c = thresh_is_adaptive(a.mode) ? 0 : thresh_cutoff(a.mode, a.k_fixed, a.energy_frac, a.cut_scale, lsort, N);
        if (thresh_is_adaptive(a.mode)) wnorm_sh = thresh_adaptive_norm(lsort, N, a.beta);
        ish[1] = c;
        bool finite = true;                                          // a NaN or Inf anywhere in the spectrum is reported, not passed on as a result
        for (int i = 0; i < N; ++i) finite = finite && isfinite(lsort[i]);
        if (!finite) converged = 0;
        a.cut[k] = c;
        a.sweeps[k] = sweep;
        a.conv[k] = converged;
        if (!converged) atomicAdd(a.nunconv, 1);
    }
    __syncthreads();
    {
        const int c = ish[1];
        const bool soft = thresh_is_soft(a.mode);
        if (tid < Ns) {
            double w = 0.0;
            if (tid < N) {
                const int i1 = rank + 1;                             // 1-based order of the eigenvalue in slot tid
                w = thresh_is_adaptive(a.mode) ? thresh_adaptive_raw((double)myl * un, lsort[0], i1, N, a.beta) / wnorm_sh
                                             : thresh_weight(soft, a.beta, i1, c);
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
    for (int e = tid; e < N * Ns; e += EC_THREADS) {
        const int row = e / Ns, u = e - row * Ns;
        const float s1 = inv_s[u], w = wsl[u];
        const float2 v = make_float2(Gr[(size_t)u * LD + row] * s1, Gi[(size_t)u * LD + row] * s1);
        Vk[e] = v;
        Bk[e] = make_float2(v.x * w, v.y * w);
    }
}

static size_t ec_smem_bytes(int Ns, int LD, bool glob) {
    return (glob ? 0 : (size_t)Ns * LD * 8) + 3 * (size_t)Ns * 4 + 32 * 4 + (size_t)Ns * 8 + 3 * (size_t)Ns * 4 + 16 + 16 + 64;
}

// N <= 128: the matrix lives in shared memory.  128 < N <= ECL8_MAXN (even): only the Cholesky factor is taken here,
// in place in global memory, and the Jacobi sweeps run on 8-CTA clusters (lcf_evd_cluster.cu).
bool evd_chol_eligible(const lcf_plan* p) {
    return p->prec == 0 && p->N >= 2 && (p->N <= 128 || (p->N <= ECL8_MAXN && p->N % 2 == 0));
}

cudaError_t configure_evd_chol(lcf_plan* p) {
    p->ec_LD = ((p->N + 3) & ~3) + 4;   // floats per column plane: whole float4 chunks, +4 shifts the banks column to column
    p->ec_smem = ec_smem_bytes(p->Ns, p->ec_LD, p->N > 128);
    if (p->ec_smem > (size_t)p->smem_optin) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaSuccess;
#define EC_SET(NC, FULL) if (e == cudaSuccess) e = set_max_dyn_smem(evd_chol_kernel<NC, FULL, false>, p->smem_optin)
    EC_SET(1, false); EC_SET(2, false); EC_SET(3, false); EC_SET(4, false);
    EC_SET(1, true); EC_SET(2, true); EC_SET(3, true); EC_SET(4, true);
#undef EC_SET
    return e;
}

cudaError_t launch_evd_chol(lcf_plan* p, cudaStream_t st, bool chol_only) {
    EcArgs a;
    a.chol_only = chol_only ? 1 : 0; a.gfac = p->ec_gfac_d; a.shift = p->ec_shift_d; a.nexp = p->ec_nexp_d;
    a.N = p->N; a.NP = p->NP; a.Ns = p->Ns; a.LD = p->ec_LD; a.max_sweeps = p->sweep_cap > 0 ? p->sweep_cap : 30;
    a.R = reinterpret_cast<const float2*>(p->R_d); a.amax = p->gram_tc ? p->amax_d : nullptr;
    a.lam = p->lam_d; a.order = p->order_d; a.cut = p->cut_d; a.sweeps = p->sweeps_d; a.conv = p->conv_d; a.nunconv = p->nunconv_d;
    a.wslot = p->wslot_d; a.wslot_dd = p->wslot_dd_d; a.wt = p->wt_d;
    a.V = reinterpret_cast<float2*>(p->V_d); a.B = p->B_d;
    a.mode = evd_mode(p); a.k_fixed = evd_kfixed(p); a.energy_frac = p->thr.energy_frac; a.beta = p->thr.beta; a.cut_scale = p->thr.cut_scale;
    if (p->N > 128) {                                                // factor only (chol_only is implied: see evd_chol_eligible)
        if (!chol_only) return cudaErrorInvalidConfiguration;
        evd_chol_kernel<1, false, true><<<p->K, EC_THREADS, p->ec_smem, st>>>(a);
        return cudaGetLastError();
    }
    const int nch = (p->N + 3) / 4, nc = (nch + 7) / 8;
    const bool full = (p->N % 32) == 0;
#define EC_RUN(NC) do { if (full) evd_chol_kernel<NC, true, false><<<p->K, EC_THREADS, p->ec_smem, st>>>(a); \
                        else evd_chol_kernel<NC, false, false><<<p->K, EC_THREADS, p->ec_smem, st>>>(a); } while (0)
    switch (nc) { case 1: EC_RUN(1); break; case 2: EC_RUN(2); break; case 3: EC_RUN(3); break; default: EC_RUN(4); break; }
#undef EC_RUN
    return cudaGetLastError();
}

}  // namespace lcf
