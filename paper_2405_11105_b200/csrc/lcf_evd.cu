// lcf_evd.cu -- kernel 2 (batched Hermitian EVD, Eq. 2) and kernel 3 (eigen-weights
// and projector factor, PAPER.md:57-59 and Eq. 9).
//
// Kernel 2, jacobi_kernel: one CTA per window.  Two-sided Jacobi on the Hermitian R_k with the
// round-robin ("circle method") parallel ordering: at step s the NP = ceil(N/2) disjoint pivots are
//     pair 0:  (p, q) = ((-s) mod M, M)            M = 2 NP - 1
//     pair m:  (p, q) = ((m - s) mod M, (-m - s) mod M),  m = 1 .. NP-1
// so M steps visit every index pair once (one sweep).  Only the strict upper triangle (packed) and
// the real diagonal live in shared memory; A <- J^H A J is applied 2x2 block by 2x2 block,
// block (m, n), m < n, being J_m^H A[{p_m,q_m},{p_n,q_n}] J_n -- every thread updates its blocks in
// place, so a step needs two barriers (rotation parameters, block updates).  The rotation
// J = [[c, g], [-conj(g), c]], g = s e^{i phi}, is the standard one: phi = arg A_pq,
// tau = (A_qq - A_pp) / (2 |A_pq|), t = sign(tau) / (|tau| + sqrt(1 + tau^2)), c = 1/sqrt(1+t^2),
// s = t c.  Eigenvectors are NOT accumulated here: every (c, g) is appended to a rotation log.
// The CTA ends by ranking the eigenvalues (descending), applying the cut-off rule and writing the
// eigen-weights.  Odd N is padded with one inert index (zero row/column, never rotated).
//
// Kernel 3, vbuild_kernel: replays the rotation log on the rows of the identity -- one warp per
// VB_ROWS rows, all (window, row) pairs in parallel over the whole GPU -- which yields V_k, and
// scales column u by its eigen-weight: B_k = V_k diag(wt) is the operand of the projection
// kernel (|s_p V diag(wt) V^H|^2 = |s_p V diag(wt)|^2 because V is unitary).
#include <cfloat>

#include "lcf_internal.h"
#include "lcf_thresh.cuh"

namespace lcf {

template <typename T> struct Cx2;
template <> struct Cx2<float> { using type = float2; };
template <> struct Cx2<double> { using type = double2; };

// pivot pair m of step s (0 <= s < M)
__device__ __forceinline__ void pair_pq(int m, int s, int M, int& p, int& q) {
    if (m == 0) {
        p = (s == 0) ? 0 : M - s;
        q = M;
    } else {
        p = m - s; if (p < 0) p += M;
        q = M - m - s; if (q < 0) q += M;
    }
}

struct JacArgs {
    int N, NP, M, Ns;       // Ns = 2 NP slots, M = Ns - 1
    int max_sweeps;
    const void* R;          // [K][N][N] complex T, full Hermitian
    void* rotlog;           // [K][max_sweeps*M][3][NP] T
    double* lam;            // [K][N] descending
    int* order;             // [K][N]
    int* cut;               // [K]
    int* sweeps;            // [K]
    int* conv;              // [K]
    int* nunconv;           // [1] count of window EVDs that hit the sweep cap
    float* wslot;           // [K][Ns]
    double* wslot_dd;       // [K][Ns]
    double* wt;             // [K][N]
    int mode, k_fixed;
    double energy_frac, beta, cut_scale;
};

template <typename T> __device__ __forceinline__ T eps_of();
template <> __device__ __forceinline__ float eps_of<float>() { return FLT_EPSILON; }
template <> __device__ __forceinline__ double eps_of<double>() { return DBL_EPSILON; }
template <typename T> __device__ __forceinline__ T tiny_of();
template <> __device__ __forceinline__ float tiny_of<float>() { return 1e-36f; }
template <> __device__ __forceinline__ double tiny_of<double>() { return 1e-290; }

template <typename T>
__device__ __forceinline__ T block_sum(T v, T* red /* [32] */, int tid, int nthr) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __syncthreads();
    if ((tid & 31) == 0) red[tid >> 5] = v;
    __syncthreads();
    T tot = T(0);
    int nw = (nthr + 31) >> 5;
    for (int w = 0; w < nw; ++w) tot += red[w];  // fixed order: deterministic, identical in all threads
    return tot;
}

template <typename T>
__global__ void __launch_bounds__(1024, 1) jacobi_kernel(JacArgs a) {
    using C = typename Cx2<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = a.N, NP = a.NP, M = a.M, Ns = a.Ns;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int k = blockIdx.x;
    const int npk = Ns * (Ns - 1) / 2;  // packed strict upper triangle
    C* S = reinterpret_cast<C*>(smem_raw);                 // [npk], element (u,v), u<v, at rowoff(u)+v
    T* d = reinterpret_cast<T*>(S + npk);                  // [Ns] diagonal
    T* pc = d + Ns;                                        // [NP] c of this step
    T* pgr = pc + NP;                                      // [NP] Re g
    T* pgi = pgr + NP;                                     // [NP] Im g
    T* red = pgi + NP;                                     // [32]
    auto rowoff = [Ns](int u) { return (u * (2 * Ns - u - 1)) / 2 - u - 1; };

    // ---- load the upper triangle of R_k (reduced by the Gram stage) ----
    {
        const C* Rk = reinterpret_cast<const C*>(a.R) + (size_t)k * N * N;
        const int nup = Ns * (Ns + 1) / 2;
        for (int e = tid; e < nup; e += nthr) {
            // e -> (u, v), u <= v, row-major over the upper triangle of Ns x Ns
            int u = (int)((2.0f * Ns + 1.0f - sqrtf((2.0f * Ns + 1.0f) * (2.0f * Ns + 1.0f) - 8.0f * (float)e)) * 0.5f);
            if (u < 0) u = 0;
            while (u > 0 && u * (2 * Ns - u + 1) / 2 > e) --u;
            while ((u + 1) * (2 * Ns - u) / 2 <= e) ++u;
            int v = u + (e - u * (2 * Ns - u + 1) / 2);
            T re = T(0), im = T(0);
            if (v < N) {
                const C x = Rk[(size_t)u * N + v];
                re = x.x; im = (u == v) ? T(0) : x.y;
            }
            if (u == v) d[u] = re;
            else { C o; o.x = re; o.y = im; S[rowoff(u) + v] = o; }
        }
    }
    __syncthreads();

    // fp32 only: bring the matrix to a fixed magnitude (largest diagonal entry in [1, 2)) by an exact power of
    // two, so that the squares in the rotation and convergence tests neither underflow nor overflow whatever
    // the units of the data (R ~ amplitude^2 P); the eigenvalues are unscaled in double at the end
    int lam_exp = 0;
    if (sizeof(T) == 4) {
        T mx = T(0);
        for (int u = tid; u < Ns; u += nthr) mx = fmaxf((float)mx, fabsf((float)d[u]));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mx = fmaxf((float)mx, __shfl_xor_sync(0xffffffffu, (float)mx, o));
        __syncthreads();
        if ((tid & 31) == 0) red[tid >> 5] = mx;
        __syncthreads();
        float m = 0.f;
        for (int w = 0; w < (nthr + 31) >> 5; ++w) m = fmaxf(m, (float)red[w]);
        if (m > 0.f && m < 3.0e38f) {
            int ex;
            frexpf(m, &ex);                                   // m = f 2^ex, f in [0.5, 1)
            lam_exp = 1 - ex;                                 // m 2^lam_exp in [1, 2)
            const T sc = (T)ldexpf(1.f, lam_exp < -120 ? -120 : (lam_exp > 120 ? 120 : lam_exp));
            lam_exp = lam_exp < -120 ? -120 : (lam_exp > 120 ? 120 : lam_exp);
            for (int e = tid; e < npk; e += nthr) { C x = S[e]; x.x *= sc; x.y *= sc; S[e] = x; }
            for (int u = tid; u < Ns; u += nthr) d[u] *= sc;
        }
        __syncthreads();
    }
    const double lam_un = ldexp(1.0, -lam_exp);

    T fro2;
    {
        T acc = T(0);
        for (int e = tid; e < npk; e += nthr) { C x = S[e]; acc += x.x * x.x + x.y * x.y; }
        acc *= T(2);
        for (int u = tid; u < Ns; u += nthr) acc += d[u] * d[u];
        fro2 = block_sum<T>(acc, red, tid, nthr);
    }
    const T tol = T(4) * eps_of<T>();
    const T tol2 = tol * tol * fro2;

    // off-diagonal block list of this thread: blocks (m, n), m < n, folded into an
    // R x (NP-1) rectangle (row a holds pairs of row a, then pairs of row NP-1-a)
    const int Wd = NP - 1;                       // rectangle width
    const int Rr = (NP + 1) / 2;                 // rows
    const int nblk = (Wd > 0) ? Rr * Wd : 0;
    const int qa = (Wd > 0) ? nthr / Wd : 0, qj = (Wd > 0) ? nthr % Wd : 0;
    const int a0 = (Wd > 0) ? tid / Wd : 0, j0 = (Wd > 0) ? tid % Wd : 0;

    T* logk = reinterpret_cast<T*>(a.rotlog) + (size_t)k * a.max_sweeps * M * 3 * NP;
    int sweep = 0, converged = 0;
    for (;;) {
        // convergence test at sweep boundaries: off(A)_F^2 <= tol^2 ||A||_F^2
        T acc = T(0);
        for (int e = tid; e < npk; e += nthr) { C x = S[e]; acc += x.x * x.x + x.y * x.y; }
        T off2 = T(2) * block_sum<T>(acc, red, tid, nthr);
        if (off2 <= tol2) { converged = 1; break; }
        if (sweep == a.max_sweeps) { converged = (off2 <= T(1e4) * tol2) ? 1 : 0; break; }
        for (int s = 0; s < M; ++s) {
            // ---- phase P: rotation parameters of the NP pivots ----
            if (tid < NP) {
                int p, q; pair_pq(tid, s, M, p, q);
                const bool swp = p > q;
                const int u = swp ? q : p, v = swp ? p : q;
                C x = S[rowoff(u) + v];
                if (swp) x.y = -x.y;           // x = A[p][q]
                const T app = d[p], aqq = d[q];
                const T absa2 = x.x * x.x + x.y * x.y;
                T c = T(1), gr = T(0), gi = T(0);
                if (absa2 > tiny_of<T>()) {
                    const T absa = sqrt(absa2);
                    const T inv = T(1) / absa;
                    const T tau = (aqq - app) * (T(0.5) * inv);
                    T t;
                    const T at = fabs(tau);
                    if (at > T(1e8)) t = T(0.5) / tau;
                    else { t = T(1) / (at + sqrt(T(1) + tau * tau)); if (tau < T(0)) t = -t; }
                    c = T(1) / sqrt(T(1) + t * t);
                    const T sn = t * c;
                    gr = sn * x.x * inv; gi = sn * x.y * inv;
                    d[p] = app - t * absa;
                    d[q] = aqq + t * absa;
                    C z; z.x = T(0); z.y = T(0);
                    S[rowoff(u) + v] = z;
                }
                pc[tid] = c; pgr[tid] = gr; pgi[tid] = gi;
                T* lg = logk + ((size_t)sweep * M + s) * 3 * NP;
                lg[tid] = c; lg[NP + tid] = gr; lg[2 * NP + tid] = gi;
            }
            __syncthreads();
            // ---- phase U: B <- J_m^H B J_n on every off-diagonal 2x2 block, in place ----
            {
                int ra = a0, rj = j0;
                for (int b = tid; b < nblk; b += nthr) {
                    int m, n;
                    if (rj < Wd - ra) { m = ra; n = ra + 1 + rj; }
                    else { m = NP - 1 - ra; n = NP - ra + (rj - (Wd - ra)); }
                    const bool ok = (m < n) && (n < NP) && !(2 * ra == NP - 1 && rj >= Wd - ra);
                    if (ok) {
                        int pm, qm, pn, qn;
                        pair_pq(m, s, M, pm, qm);
                        pair_pq(n, s, M, pn, qn);
                        const T cm = pc[m], gmr = pgr[m], gmi = pgi[m];
                        const T cn = pc[n], gnr = pgr[n], gni = pgi[n];
                        // addresses + conjugation flags of A[pm][pn], A[pm][qn], A[qm][pn], A[qm][qn]
                        int i00, i01, i10, i11; bool f00, f01, f10, f11;
                        f00 = pm > pn; i00 = f00 ? rowoff(pn) + pm : rowoff(pm) + pn;
                        f01 = pm > qn; i01 = f01 ? rowoff(qn) + pm : rowoff(pm) + qn;
                        f10 = qm > pn; i10 = f10 ? rowoff(pn) + qm : rowoff(qm) + pn;
                        f11 = qm > qn; i11 = f11 ? rowoff(qn) + qm : rowoff(qm) + qn;
                        C b00 = S[i00], b01 = S[i01], b10 = S[i10], b11 = S[i11];
                        if (f00) b00.y = -b00.y;
                        if (f01) b01.y = -b01.y;
                        if (f10) b10.y = -b10.y;
                        if (f11) b11.y = -b11.y;
                        // T = J_m^H B,  J_m^H = [[cm, -gm], [conj(gm), cm]]
                        C t00, t01, t10, t11;
                        t00.x = cm * b00.x - (gmr * b10.x - gmi * b10.y);
                        t00.y = cm * b00.y - (gmr * b10.y + gmi * b10.x);
                        t01.x = cm * b01.x - (gmr * b11.x - gmi * b11.y);
                        t01.y = cm * b01.y - (gmr * b11.y + gmi * b11.x);
                        t10.x = (gmr * b00.x + gmi * b00.y) + cm * b10.x;
                        t10.y = (gmr * b00.y - gmi * b00.x) + cm * b10.y;
                        t11.x = (gmr * b01.x + gmi * b01.y) + cm * b11.x;
                        t11.y = (gmr * b01.y - gmi * b01.x) + cm * b11.y;
                        // B' = T J_n,  J_n = [[cn, gn], [-conj(gn), cn]]
                        b00.x = cn * t00.x - (gnr * t01.x + gni * t01.y);
                        b00.y = cn * t00.y - (gnr * t01.y - gni * t01.x);
                        b01.x = (gnr * t00.x - gni * t00.y) + cn * t01.x;
                        b01.y = (gnr * t00.y + gni * t00.x) + cn * t01.y;
                        b10.x = cn * t10.x - (gnr * t11.x + gni * t11.y);
                        b10.y = cn * t10.y - (gnr * t11.y - gni * t11.x);
                        b11.x = (gnr * t10.x - gni * t10.y) + cn * t11.x;
                        b11.y = (gnr * t10.y + gni * t10.x) + cn * t11.y;
                        if (f00) b00.y = -b00.y;
                        if (f01) b01.y = -b01.y;
                        if (f10) b10.y = -b10.y;
                        if (f11) b11.y = -b11.y;
                        S[i00] = b00; S[i01] = b01; S[i10] = b10; S[i11] = b11;
                    }
                    ra += qa; rj += qj;
                    if (rj >= Wd) { rj -= Wd; ra += 1; }
                }
            }
            __syncthreads();
        }
        ++sweep;
    }

    // ---- epilogue: rank eigenvalues (descending, ties by index), cut-off, eigen-weights ----
    __shared__ double wnorm_sh;                            // normalisation of the adaptive weights (method 6)
    double* lsort = reinterpret_cast<double*>(smem_raw);  // reuse the matrix storage: [N] sorted
    int* csh = reinterpret_cast<int*>(lsort + Ns);
    T myl = T(0);
    int rank = 0;
    if (tid < N) {
        myl = d[tid];
        for (int j = 0; j < N; ++j) {
            T lj = d[j];
            rank += (lj > myl) || (lj == myl && j < tid);
        }
    }
    __syncthreads();  // all reads of d/S done before lsort overwrites S
    if (tid < N) {
        lsort[rank] = (double)myl * lam_un;
        a.lam[(size_t)k * N + rank] = (double)myl * lam_un;
        a.order[(size_t)k * N + rank] = tid;
    }
    __syncthreads();
    if (tid == 0) {
        const int c = thresh_is_adaptive(a.mode) ? 0 : thresh_cutoff(a.mode, a.k_fixed, a.energy_frac, a.cut_scale, lsort, N);
        if (thresh_is_adaptive(a.mode)) wnorm_sh = thresh_adaptive_norm(lsort, N, a.beta);
        *csh = c;
        bool finite = true;                                // a NaN or Inf anywhere in the spectrum is reported, not passed on as a result
        for (int i = 0; i < N; ++i) finite = finite && isfinite(lsort[i]);
        if (!finite) converged = 0;
        a.cut[k] = c;
        a.sweeps[k] = sweep;
        a.conv[k] = converged;
        if (!converged) atomicAdd(a.nunconv, 1);
    }
    __syncthreads();
    const int c = *csh;
    const bool soft = thresh_is_soft(a.mode);
    if (tid < Ns) {   // blockDim.x >= Ns (configure_evd)
        double w = 0.0;
        if (tid < N) {
            const int i1 = rank + 1;  // 1-based order of the eigenvalue held by index tid
            w = thresh_is_adaptive(a.mode) ? thresh_adaptive_raw((double)myl * lam_un, lsort[0], i1, N, a.beta) / wnorm_sh
                                             : thresh_weight(soft, a.beta, i1, c);
            a.wt[(size_t)k * N + rank] = w;
        }
        a.wslot[(size_t)k * Ns + tid] = (float)w;
        a.wslot_dd[(size_t)k * Ns + tid] = w;
    }
}

// ------------------------------------------------------------------------------------------------
struct VbArgs {
    int N, NP, M, Ns, max_sweeps;
    const void* rotlog;
    const int* sweeps;
    const float* wslot;
    void* V;     // [K][N][Ns] complex T
    float2* B;   // [K][N][Ns]
};

template <typename T, int PPL>
__global__ void __launch_bounds__(VB_WARPS * 32) vbuild_kernel(VbArgs a) {
    using C = typename Cx2<T>::type;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = a.N, NP = a.NP, M = a.M, Ns = a.Ns;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int k = blockIdx.y;
    const int row0 = (blockIdx.x * VB_WARPS + warp) * VB_ROWS;
    C* v = reinterpret_cast<C*>(smem_raw) + (size_t)warp * VB_ROWS * Ns;  // [VB_ROWS][Ns]
    if (row0 >= N) return;  // whole warp
    for (int r = 0; r < VB_ROWS; ++r)
        for (int u = lane; u < Ns; u += 32) {
            C z; z.x = (u == row0 + r && row0 + r < N) ? T(1) : T(0); z.y = T(0);
            v[r * Ns + u] = z;
        }
    __syncwarp();
    const T* logk = reinterpret_cast<const T*>(a.rotlog) + (size_t)k * a.max_sweeps * M * 3 * NP;
    const int nsteps = a.sweeps[k] * M;
    T pc[PPL], pr[PPL], pi[PPL];
    auto fetch = [&](int g) {
        const T* lg = logk + (size_t)g * 3 * NP;
#pragma unroll
        for (int j = 0; j < PPL; ++j) {
            int m = lane + 32 * j;
            if (m < NP) { pc[j] = lg[m]; pr[j] = lg[NP + m]; pi[j] = lg[2 * NP + m]; }
            else { pc[j] = T(1); pr[j] = T(0); pi[j] = T(0); }
        }
    };
    if (nsteps > 0) fetch(0);
    int s = 0;
    for (int g = 0; g < nsteps; ++g) {
        T c[PPL], gr[PPL], gi[PPL];
#pragma unroll
        for (int j = 0; j < PPL; ++j) { c[j] = pc[j]; gr[j] = pr[j]; gi[j] = pi[j]; }
        if (g + 1 < nsteps) fetch(g + 1);
#pragma unroll
        for (int j = 0; j < PPL; ++j) {
            int m = lane + 32 * j;
            if (m < NP) {
                int p, q; pair_pq(m, s, M, p, q);
#pragma unroll
                for (int r = 0; r < VB_ROWS; ++r) {
                    C vp = v[r * Ns + p], vq = v[r * Ns + q];
                    C np_, nq_;
                    // v <- v J:  v_p' = c v_p - conj(g) v_q,  v_q' = g v_p + c v_q
                    np_.x = c[j] * vp.x - (gr[j] * vq.x + gi[j] * vq.y);
                    np_.y = c[j] * vp.y - (gr[j] * vq.y - gi[j] * vq.x);
                    nq_.x = (gr[j] * vp.x - gi[j] * vp.y) + c[j] * vq.x;
                    nq_.y = (gr[j] * vp.y + gi[j] * vp.x) + c[j] * vq.y;
                    v[r * Ns + p] = np_; v[r * Ns + q] = nq_;
                }
            }
        }
        __syncwarp();
        if (++s == M) s = 0;
    }
    // write V (slot order) and B = V diag(wslot)
    C* Vk = reinterpret_cast<C*>(a.V) + (size_t)k * N * Ns;
    float2* Bk = a.B + (size_t)k * N * Ns;
    const float* wk = a.wslot + (size_t)k * Ns;
    for (int r = 0; r < VB_ROWS; ++r) {
        int row = row0 + r;
        if (row >= N) break;
        for (int u = lane; u < Ns; u += 32) {
            C x = v[r * Ns + u];
            Vk[(size_t)row * Ns + u] = x;
            float w = wk[u];
            Bk[(size_t)row * Ns + u] = make_float2((float)x.x * w, (float)x.y * w);
        }
    }
}

// diagnostic: F_k = V diag(wt) V^H (Eq. 4), double accumulation.  complement: the same filter written as
// I - V diag(1 - wt) V^H, for the plans whose V holds only the leading eigenvectors (lcf_evd_top.cu: the others have wt = 1)
template <typename T>
__global__ void build_filters_kernel(const void* Vv, const double* wdd, double* F, int N, int Ns, int complement) {
    using C = typename Cx2<T>::type;
    const int k = blockIdx.z;
    const C* V = reinterpret_cast<const C*>(Vv) + (size_t)k * N * Ns;
    const double* w = wdd + (size_t)k * Ns;
    int a_ = blockIdx.y * blockDim.y + threadIdx.y, b_ = blockIdx.x * blockDim.x + threadIdx.x;
    if (a_ >= N || b_ >= N) return;
    double fr = 0.0, fi = 0.0;
    for (int u = 0; u < N; ++u) {
        C va = V[(size_t)a_ * Ns + u], vb = V[(size_t)b_ * Ns + u];
        double ar = va.x, ai = va.y, br = vb.x, bi = vb.y;
        const double wu = complement ? 1.0 - w[u] : w[u];
        fr += wu * (ar * br + ai * bi);
        fi += wu * (ai * br - ar * bi);
    }
    if (complement) { fr = (a_ == b_ ? 1.0 : 0.0) - fr; fi = -fi; }
    double* o = F + ((size_t)k * N * N + (size_t)a_ * N + b_) * 2;
    o[0] = fr; o[1] = fi;
}

static size_t jac_smem_bytes(int Ns, int NP, size_t esz) {
    size_t npk = (size_t)Ns * (Ns - 1) / 2;
    size_t b = npk * 2 * esz + (size_t)Ns * esz + 3 * (size_t)NP * esz + 32 * esz;
    size_t epi = (size_t)Ns * sizeof(double) + 16;   // lsort + csh reuse the front of the buffer
    return (b > epi ? b : epi) + 16;
}

cudaError_t configure_evd(lcf_plan* p) {
    p->jac_smem = jac_smem_bytes(p->Ns, p->NP, p->esz);
    if (p->jac_smem > (size_t)p->smem_optin) return cudaErrorInvalidConfiguration;
    int nblk = ((p->NP + 1) / 2) * (p->NP - 1);
    int thr = ((nblk + 31) / 32) * 32;
    // a whole number of block rounds per step, at least N threads for the epilogue
    int rounds = (thr + 1023) / 1024;
    if (rounds < 1) rounds = 1;
    thr = (((nblk + rounds - 1) / rounds) + 31) / 32 * 32;
    int need = ((p->Ns + 31) / 32) * 32;
    if (thr < need) thr = need;
    if (thr > 1024) thr = 1024;
    if (thr < 32) thr = 32;
    p->jac_threads = thr;
    cudaError_t e;
    if (p->prec == 1) e = set_max_dyn_smem(jacobi_kernel<double>, p->smem_optin);
    else e = set_max_dyn_smem(jacobi_kernel<float>, p->smem_optin);
    return e;
}

cudaError_t launch_jacobi(lcf_plan* p, cudaStream_t st) {
    JacArgs a;
    a.N = p->N; a.NP = p->NP; a.M = p->Ns - 1; a.Ns = p->Ns; a.max_sweeps = (p->sweep_cap > 0 && p->sweep_cap < p->max_sweeps) ? p->sweep_cap : p->max_sweeps;   // the rotation log holds p->max_sweeps
    a.R = p->R_d; a.rotlog = p->rotlog_d;
    a.lam = p->lam_d; a.order = p->order_d; a.cut = p->cut_d; a.sweeps = p->sweeps_d; a.conv = p->conv_d; a.nunconv = p->nunconv_d;
    a.wslot = p->wslot_d; a.wslot_dd = p->wslot_dd_d; a.wt = p->wt_d;
    a.mode = evd_mode(p); a.k_fixed = evd_kfixed(p); a.energy_frac = p->thr.energy_frac; a.beta = p->thr.beta; a.cut_scale = p->thr.cut_scale;
    if (p->prec == 1) jacobi_kernel<double><<<p->K, p->jac_threads, p->jac_smem, st>>>(a);
    else jacobi_kernel<float><<<p->K, p->jac_threads, p->jac_smem, st>>>(a);
    return cudaGetLastError();
}

template <typename T>
static cudaError_t launch_vbuild_t(lcf_plan* p, cudaStream_t st) {
    VbArgs a;
    a.N = p->N; a.NP = p->NP; a.M = p->Ns - 1; a.Ns = p->Ns; a.max_sweeps = (p->sweep_cap > 0 && p->sweep_cap < p->max_sweeps) ? p->sweep_cap : p->max_sweeps;   // the rotation log holds p->max_sweeps
    a.rotlog = p->rotlog_d; a.sweeps = p->sweeps_d; a.wslot = p->wslot_d; a.V = p->V_d; a.B = p->B_d;
    dim3 grid((p->N + VB_WARPS * VB_ROWS - 1) / (VB_WARPS * VB_ROWS), p->K);
    size_t smem = (size_t)VB_WARPS * VB_ROWS * p->Ns * 2 * sizeof(T);
    int ppl = (p->NP + 31) / 32;
    switch (ppl) {
        case 1: vbuild_kernel<T, 1><<<grid, VB_WARPS * 32, smem, st>>>(a); break;
        case 2: vbuild_kernel<T, 2><<<grid, VB_WARPS * 32, smem, st>>>(a); break;
        case 3: vbuild_kernel<T, 3><<<grid, VB_WARPS * 32, smem, st>>>(a); break;
        case 4: vbuild_kernel<T, 4><<<grid, VB_WARPS * 32, smem, st>>>(a); break;
        default: return cudaErrorInvalidConfiguration;
    }
    return cudaGetLastError();
}

cudaError_t launch_vbuild(lcf_plan* p, cudaStream_t st) {
    return p->prec == 1 ? launch_vbuild_t<double>(p, st) : launch_vbuild_t<float>(p, st);
}

cudaError_t launch_build_filters(lcf_plan* p, cudaStream_t st) {
    dim3 blk(16, 16), grid((p->N + 15) / 16, (p->N + 15) / 16, p->K);
    if (p->prec == 1) build_filters_kernel<double><<<grid, blk, 0, st>>>(p->V_d, p->wslot_dd_d, p->F_d, p->N, p->Ns, p->evd_top ? 1 : 0);
    else build_filters_kernel<float><<<grid, blk, 0, st>>>(p->V_d, p->wslot_dd_d, p->F_d, p->N, p->Ns, p->evd_top ? 1 : 0);
    return cudaGetLastError();
}

}  // namespace lcf
