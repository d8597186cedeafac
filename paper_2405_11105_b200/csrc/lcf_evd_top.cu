// lcf_evd_top.cu -- SURVEY.md 8(f) rank 4, "partial EVD": the hard cut-offs by a fixed count and by the
// energy rule need only the c leading eigenpairs of R_k and trace(R_k) = sum_i lambda_i, because the filter is
//     F_k = I - sum_{i<=c} v_i v_i^H          (Eq. 4 with wt_i = 0 for i <= c, 1 above, V unitary)
// so the N - c eigenvectors of the blood / noise part never have to be resolved.  Modes LCF_HARD_FIXED_TOP /
// LCF_HARD_ENERGY_TOP compute exactly that filter by block subspace iteration with Rayleigh-Ritz (a departure from the
// paper's full-spectrum EVD; the full-spectrum modes stay the default):
//     Q <- orth(Y);  Y <- R Q;  H = Q^H Y;  H = J Theta J^H;  Q <- Q J, Y <- Y J        (one round)
// on a block of M = 16 vectors (cuts up to 10), or 32 (cuts up to 26) for the windows the small block cannot settle.
// Tissue dominates R_k by 20-60 dB, so lambda_{M+1} / lambda_c is tiny and the block converges in 2-3 rounds whatever N
// is: O(N^2 M) per round instead of the O(N^3) per sweep of a Jacobi EVD (config 3, 192 windows of 200 frames: 1.1 ms
// against 17 ms of cluster Jacobi).
//
// One CTA (256 threads) per window.  Q lives in shared memory in double, Y in float; every inner product and the
// products with R accumulate in double (R_k itself is the fp32 Gram).  Steps of a round:
//   orth    classical Gram-Schmidt, twice per column (column j against the j columns before it);
//   Y = RQ  thread = (row, block of CPT columns), R read through L2 by columns (R is Hermitian: coalesced);
//   H       M x M inner products, symmetrised; its EVD by one-sided Jacobi on the columns of H (parallel ordering,
//           one warp per pair, the rotations accumulated in J), Ritz values theta_j = Re(J_j^H H J_j), sorted;
//   check   the cut c from theta and trace(R) (same rule as lcf_thresh.cuh); rho_j = |y_j - Q_c Q_c^H y_j|, the part of
//           R q_j outside the span of the leading c Ritz vectors; converged when every rho_j, j <= c, is below
//           2e-6 (theta_j - theta_{c+1}) (the sine of the angle by which it tilts that span), or at the rounding floor
//           of the fp32 column it is computed from.
// Outputs: lambda (the M Ritz values, a rounding-negative one as 0; the N - M others are reported as their mean,
// (trace - sum theta) / (N - M), capped by the last Ritz value so that the array stays descending), c_k, weights, V_k = [q_1 .. q_M, 0 ...], and
// B_k = F_k itself (Hermitian, idempotent: |F^T s|^2 = |F conj(s)|^2 is the filtered power, so the projection kernels
// take it unchanged).
#include <cfloat>

#include "lcf_internal.h"
#include "lcf_sm100.cuh"
#include "lcf_thresh.cuh"

namespace lcf {

constexpr int ET_THREADS = 256;
constexpr int ET_M = 32;                       // block size (large)
constexpr int ET_MS = 16;                      // block size (small)
constexpr int ET_GUARD = 6;                    // Ritz pairs carried beyond the largest admissible cut
constexpr int ET_MAXN = 224;                   // Q (double) + Y (float) + H, J fit one SM's shared memory up to here
constexpr int ET_ROUNDS = 12;                  // default cap on the rounds

struct EtArgs {
    int N, Ns, max_rounds;
    const float2* R;                           // [K][N][N] row-major, Hermitian
    const uint32_t* amax;                      // non-null: R carries the data scale of the tensor-core Gram
    double* lam; int* order; int* cut; int* sweeps; int* conv; int* nunconv;
    float* wslot; double* wslot_dd; double* wt;
    float2* V; float2* B;                      // [K][N][Ns]
    int energy;                                // 0: c = k_fixed, 1: energy rule
    int may_retry;                             // 1: first pass with the small block; a window it cannot settle gets conv = -1 and no output
    int retry;                                 // 1: second pass, only the windows marked conv = -1
    int k_fixed;
    double energy_frac;
};

__device__ __forceinline__ double et_warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
// sum over the CTA, same value in every thread, fixed order (warp partials added 0..7)
__device__ __forceinline__ double et_block_sum(double v, double* red) {
    v = et_warp_sum(v);
    __syncthreads();
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
#pragma unroll
    for (int w = 0; w < ET_THREADS / 32; ++w) s += red[w];
    return s;
}
// start block: a fixed pseudo-random complex matrix (integer hash of (row, column))
__device__ __forceinline__ float2 et_hash(int row, int col) {
    uint32_t h = (uint32_t)row * 2654435761u ^ ((uint32_t)col * 40503u + 0x9e3779b9u);
    h ^= h >> 16; h *= 0x7feb352du; h ^= h >> 15; h *= 0x846ca68bu; h ^= h >> 16;
    const float a = (float)(h & 0xffffu) * (1.f / 32768.f) - 1.f, b = (float)(h >> 16) * (1.f / 32768.f) - 1.f;
    return make_float2(a, b);
}

template <int M, int CPT>
__global__ void __launch_bounds__(ET_THREADS, 1) evd_top_kernel(EtArgs a) {
    extern __shared__ __align__(16) unsigned char et_smem[];
    const int N = a.N, Ns = a.Ns;
    const int LQ = N | 1;                                            // column stride of Q (odd: lanes that read one row of 32 columns hit 32 banks)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int k = blockIdx.x;
    if (a.retry && a.conv[k] != -1) return;                          // second pass: only the windows the small block gave up on
    double2* Q = reinterpret_cast<double2*>(et_smem);                // [M][LQ] orthonormal block (column j at Q + j LQ)
    float2* Y = reinterpret_cast<float2*>(Q + (size_t)M * LQ);      // [M][N] R Q
    double2* H = reinterpret_cast<double2*>(Y + (size_t)M * N);     // [M][M] column-major: Rayleigh quotient, then H J
    double2* J = H + M * M;                                          // [M][M] accumulated rotations
    double2* yb = J + M * M;                                         // [N]   the column being orthogonalised
    double2* hh = yb + N;                                            // [M]   its inner products with the earlier columns
    double* theta = reinterpret_cast<double*>(hh + M);               // [M]
    double* res = theta + M;                                         // [M]   residual norms
    double* red = res + M;                                           // [8]
    int* perm = reinterpret_cast<int*>(red + 8);                     // [M]   rank -> column of J
    int* ish = perm + M;                                             // [4]   cut, converged, rotated
    const float2* Rk = a.R + (size_t)k * N * N;

    // ---- trace(R) and the start block
    double tr = 0.0;
    for (int i = tid; i < N; i += ET_THREADS) tr += (double)Rk[(size_t)i * N + i].x;
    const double trace = et_block_sum(tr, red);
    for (int e = tid; e < M * N; e += ET_THREADS) Y[e] = et_hash(e % N, e / N);
    __syncthreads();

    int c = 0, converged = 0, rounds = 0;
    const int max_rounds = a.max_rounds > 0 ? a.max_rounds : ET_ROUNDS;
    const bool zero = !(trace > 0.0);                                // empty window: nothing to iterate on
    while (!zero) {
        // ---- Q <- orth(Y): column j against columns 0..j-1, classical Gram-Schmidt applied twice
        for (int j = 0; j < M; ++j) {
            double nn = 0.0;
            for (int attempt = 0;; ++attempt) {
                double n0 = 0.0;
                for (int i = tid; i < N; i += ET_THREADS) {
                    const float2 y = Y[(size_t)j * N + i];
                    yb[i] = make_double2(y.x, y.y);
                    n0 += (double)y.x * y.x + (double)y.y * y.y;
                }
                n0 = et_block_sum(n0, red);                          // (its barriers also publish yb)
                for (int pass = 0; pass < 2; ++pass) {
                    for (int i = warp; i < j; i += ET_THREADS / 32) {   // h_i = q_i^H y
                        double hr = 0.0, hi = 0.0;
                        for (int r = lane; r < N; r += 32) {
                            const double2 q = Q[(size_t)i * LQ + r], y = yb[r];
                            hr += q.x * y.x + q.y * y.y; hi += q.x * y.y - q.y * y.x;
                        }
                        hr = et_warp_sum(hr); hi = et_warp_sum(hi);
                        if (lane == 0) hh[i] = make_double2(hr, hi);
                    }
                    __syncthreads();
                    for (int r = tid; r < N; r += ET_THREADS) {     // y -= sum_i h_i q_i
                        double2 y = yb[r];
                        for (int i = 0; i < j; ++i) {
                            const double2 q = Q[(size_t)i * LQ + r], h = hh[i];
                            y.x -= h.x * q.x - h.y * q.y; y.y -= h.x * q.y + h.y * q.x;
                        }
                        yb[r] = y;
                    }
                    __syncthreads();
                }
                nn = 0.0;
                for (int r = tid; r < N; r += ET_THREADS) { const double2 y = yb[r]; nn += y.x * y.x + y.y * y.y; }
                nn = et_block_sum(nn, red);
                // what is left after the projection must stand clear of the rounding of the fp32 column it came from
                // (2^-24 per entry); otherwise -- R of rank <= j, or a column inside the span of the earlier ones -- the
                // column restarts from a fresh pseudo-random vector (its Ritz value will be ~0).  A random vector keeps
                // ~(1 - j/N) of its norm, so the second attempt passes; the third is accepted as it is.
                if ((nn > 1e-13 * n0 && nn > 0.0) || attempt == 2) break;
                for (int i = tid; i < N; i += ET_THREADS) Y[(size_t)j * N + i] = et_hash(i, 1000 + 97 * (attempt + 1) + 31 * rounds + j);
                __syncthreads();
            }
            const double inv = nn > 0.0 ? 1.0 / sqrt(nn) : 0.0;
            for (int r = tid; r < N; r += ET_THREADS) { const double2 y = yb[r]; Q[(size_t)j * LQ + r] = make_double2(y.x * inv, y.y * inv); }
            __syncthreads();
        }
        // ---- Y <- R Q (thread = row, CPT columns; R[row][j] = conj(R[j][row]) is read down column `row`: coalesced)
        {
            constexpr int CS = M / CPT;
            const int NR = (N + 31) & ~31;
            const int row = tid % NR, cs = tid / NR;
            if (row < N && cs < CS) {
                double ar[CPT], ai[CPT];
#pragma unroll
                for (int cc = 0; cc < CPT; ++cc) ar[cc] = ai[cc] = 0.0;
                const double2* q0 = Q + (size_t)(cs * CPT) * LQ;
                constexpr int PF = 8;                                // loads of R in flight per thread (L2 latency, 8 warps per SM)
                for (int j0 = 0; j0 < N; j0 += PF) {
                    float2 rf[PF];
#pragma unroll
                    for (int u = 0; u < PF; ++u) rf[u] = j0 + u < N ? Rk[(size_t)(j0 + u) * N + row] : make_float2(0.f, 0.f);
#pragma unroll
                    for (int u = 0; u < PF; ++u) {
                        const int j = j0 + u < N ? j0 + u : N - 1;   // (a zero R entry past the end adds nothing)
                        const double rr = rf[u].x, ri = -(double)rf[u].y;
#pragma unroll
                        for (int cc = 0; cc < CPT; ++cc) {
                            const double2 q = q0[(size_t)cc * LQ + j];
                            ar[cc] += rr * q.x - ri * q.y; ai[cc] += rr * q.y + ri * q.x;
                        }
                    }
                }
#pragma unroll
                for (int cc = 0; cc < CPT; ++cc) Y[(size_t)(cs * CPT + cc) * N + row] = make_float2((float)ar[cc], (float)ai[cc]);
            }
        }
        __syncthreads();
        ++rounds;
        if (rounds == 1 && max_rounds > 1) continue;                 // the first product only turns the start block towards the leading subspace
        // ---- H = Q^H Y, symmetrised
        for (int e = tid; e < M * M; e += ET_THREADS) {
            const int i = e % M, j = e / M;                          // H[i][j] = q_i^H y_j
            double hr = 0.0, hi = 0.0;
            for (int r = 0; r < N; ++r) {
                const double2 q = Q[(size_t)i * LQ + r]; const float2 y = Y[(size_t)j * N + r];
                hr += q.x * (double)y.x + q.y * (double)y.y; hi += q.x * (double)y.y - q.y * (double)y.x;
            }
            J[e] = make_double2(hr, hi);                             // staged in J
        }
        __syncthreads();
        for (int e = tid; e < M * M; e += ET_THREADS) {
            const int i = e % M, j = e / M;
            const double2 x = J[j * M + i], y = J[i * M + j];        // H[i][j], H[j][i]
            H[j * M + i] = make_double2(0.5 * (x.x + y.x), 0.5 * (x.y - y.y));
        }
        __syncthreads();
        for (int e = tid; e < M * M; e += ET_THREADS) J[e] = make_double2((e % M) == (e / M) ? 1.0 : 0.0, 0.0);
        __syncthreads();
        // ---- EVD of H: one-sided Jacobi on its columns X = H J (lane = row), rotations accumulated in J.  A warp owns
        // PPW pairs of a step and runs them side by side (independent chains).  Rotations stop at cos <= 1e-10: the
        // Ritz vectors only have to be good to the fp32 level of the data.
        {
            constexpr int PPW = (M / 2 + ET_THREADS / 32 - 1) / (ET_THREADS / 32);
            const bool rowok = lane < M;
            for (int sw = 0; sw < 20; ++sw) {
                int rotated = 0;
                for (int s = 0; s < M - 1; ++s) {
                    int pp[PPW], qq[PPW];
                    double2 xp[PPW], xq[PPW];
                    double app[PPW], aqq[PPW], xr[PPW], xi[PPW];
#pragma unroll
                    for (int u = 0; u < PPW; ++u) {
                        const int w = warp + u * (ET_THREADS / 32);
                        const bool on = w < M / 2;
                        pp[u] = !on ? 0 : (w == 0 ? M - 1 : (s + w) % (M - 1));
                        qq[u] = !on ? 0 : (w == 0 ? s : (s - w + (M - 1)) % (M - 1));
                        xp[u] = rowok ? H[pp[u] * M + lane] : make_double2(0.0, 0.0);
                        xq[u] = rowok ? H[qq[u] * M + lane] : make_double2(0.0, 0.0);
                        app[u] = xp[u].x * xp[u].x + xp[u].y * xp[u].y; aqq[u] = xq[u].x * xq[u].x + xq[u].y * xq[u].y;
                        xr[u] = xp[u].x * xq[u].x + xp[u].y * xq[u].y;  xi[u] = xp[u].x * xq[u].y - xp[u].y * xq[u].x;
                    }
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
                        for (int u = 0; u < PPW; ++u) {
                            app[u] += __shfl_xor_sync(0xffffffffu, app[u], o); aqq[u] += __shfl_xor_sync(0xffffffffu, aqq[u], o);
                            xr[u] += __shfl_xor_sync(0xffffffffu, xr[u], o);   xi[u] += __shfl_xor_sync(0xffffffffu, xi[u], o);
                        }
                    }
#pragma unroll
                    for (int u = 0; u < PPW; ++u) {
                        const int w = warp + u * (ET_THREADS / 32);
                        const double absa2 = xr[u] * xr[u] + xi[u] * xi[u];
                        if (w < M / 2 && absa2 > 1e-20 * app[u] * aqq[u] && absa2 > 0.0) {
                            rotated = 1;
                            const double ia = rsqrt(absa2);
                            const double tau = (aqq[u] - app[u]) * (0.5 * ia);
                            const double t = (tau >= 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau));
                            const double cs = rsqrt(1.0 + t * t), sn = t * cs;
                            const double gr = sn * xr[u] * ia, gi = sn * xi[u] * ia;
                            if (rowok) {
                                const int p = pp[u], q = qq[u];
                                // x_p' = c x_p - conj(g) x_q,   x_q' = g x_p + c x_q
                                H[p * M + lane] = make_double2(cs * xp[u].x - (gr * xq[u].x + gi * xq[u].y), cs * xp[u].y - (gr * xq[u].y - gi * xq[u].x));
                                H[q * M + lane] = make_double2(gr * xp[u].x - gi * xp[u].y + cs * xq[u].x, gr * xp[u].y + gi * xp[u].x + cs * xq[u].y);
                                const double2 jp = J[p * M + lane], jq = J[q * M + lane];
                                J[p * M + lane] = make_double2(cs * jp.x - (gr * jq.x + gi * jq.y), cs * jp.y - (gr * jq.y - gi * jq.x));
                                J[q * M + lane] = make_double2(gr * jp.x - gi * jp.y + cs * jq.x, gr * jp.y + gi * jp.x + cs * jq.y);
                            }
                        }
                    }
                    __syncthreads();
                }
                if (!__syncthreads_or(rotated)) break;
            }
        }
        // Ritz values theta_j = Re(J_j^H (H J)_j), ranked (descending, ties by column)
        if (tid < M) {
            double t = 0.0;
            for (int r = 0; r < M; ++r) { const double2 jv = J[tid * M + r], x = H[tid * M + r]; t += jv.x * x.x + jv.y * x.y; }
            res[tid] = t;                                            // staged
        }
        __syncthreads();
        if (tid < M) {
            const double my = res[tid];
            int rk = 0;
            for (int j = 0; j < M; ++j) { const double v = res[j]; rk += (v > my) || (v == my && j < tid); }
            theta[rk] = my; perm[rk] = tid;
        }
        __syncthreads();
        // ---- Q <- Q J[:, perm], Y <- Y J[:, perm] (thread = row; the row's M inputs in registers, outputs written in place)
        for (int r = tid; r < N; r += ET_THREADS) {
            double2 qi[M];
#pragma unroll
            for (int u = 0; u < M; ++u) qi[u] = Q[(size_t)u * LQ + r];
            for (int jj = 0; jj < M; ++jj) {
                const double2* jc = J + perm[jj] * M;
                double orr = 0.0, oi = 0.0;
#pragma unroll
                for (int u = 0; u < M; ++u) { const double2 g = jc[u]; orr += qi[u].x * g.x - qi[u].y * g.y; oi += qi[u].x * g.y + qi[u].y * g.x; }
                Q[(size_t)jj * LQ + r] = make_double2(orr, oi);
            }
            float2 yi[M];
#pragma unroll
            for (int u = 0; u < M; ++u) yi[u] = Y[(size_t)u * N + r];
            for (int jj = 0; jj < M; ++jj) {
                const double2* jc = J + perm[jj] * M;
                double orr = 0.0, oi = 0.0;
#pragma unroll
                for (int u = 0; u < M; ++u) { const double2 g = jc[u]; orr += (double)yi[u].x * g.x - (double)yi[u].y * g.y; oi += (double)yi[u].x * g.y + (double)yi[u].y * g.x; }
                Y[(size_t)jj * N + r] = make_float2((float)orr, (float)oi);
            }
        }
        __syncthreads();
        // ---- the cut, then the convergence test.  What has to converge is the SPAN of the leading c Ritz vectors (mixing
        // among them leaves F alone): rho_j = |y_j - Q_c Q_c^H y_j| is the part of R q_j outside it, and
        // rho_j / (theta_j - theta_{c+1}) the sine of the angle it tilts the span by.  Pair j is done when that is below
        // 2e-6, or when rho_j is at the rounding floor of the fp32 column y_j.
        if (tid == 0) {
            int cc = -1;
            if (!a.energy) cc = a.k_fixed;
            else {
                double cum = 0.0;
                for (int m = 1; m <= M - ET_GUARD; ++m) {                    // the cut has to lie ET_GUARD pairs inside the block
                    cum += theta[m - 1] > 0.0 ? theta[m - 1] : 0.0;
                    if (cum > a.energy_frac * trace) { cc = m; break; }
                }
            }
            ish[0] = cc;
        }
        __syncthreads();
        c = ish[0];
        for (int j = warp; j < c && j < M; j += ET_THREADS / 32) {
            double yy = 0.0, inb = 0.0;
            for (int r = lane; r < N; r += 32) { const float2 y = Y[(size_t)j * N + r]; yy += (double)y.x * y.x + (double)y.y * y.y; }
            yy = et_warp_sum(yy);
            for (int i = 0; i < c && i < M; ++i) {
                double gr = 0.0, gi = 0.0;
                for (int r = lane; r < N; r += 32) {
                    const double2 q = Q[(size_t)i * LQ + r]; const float2 y = Y[(size_t)j * N + r];
                    gr += q.x * (double)y.x + q.y * (double)y.y; gi += q.x * (double)y.y - q.y * (double)y.x;
                }
                gr = et_warp_sum(gr); gi = et_warp_sum(gi);
                inb += gr * gr + gi * gi;
            }
            if (lane == 0) res[j] = yy - inb > 0.0 ? yy - inb : 0.0;     // rho_j^2
        }
        __syncthreads();
        if (tid == 0) {
            int ok = 0;
            if (c >= 0) {
                ok = 1;
                for (int j = 0; j < c && j < M; ++j) {
                    const double rj = sqrt(res[j]), gap = theta[j] - (c < M ? theta[c] : 0.0);
                    if (!(rj <= 2e-6 * gap || rj <= 4e-7 * theta[j])) ok = 0;
                }
            }
            ish[1] = ok;
        }
        __syncthreads();
        converged = ish[1];
        if (converged || rounds >= max_rounds) break;
    }
    if (zero) {                                                      // all-zero window: any basis; the rules of lcf_thresh.cuh on a zero spectrum
        c = a.energy ? N : a.k_fixed;
        converged = 1;
        for (int e = tid; e < M; e += ET_THREADS) theta[e] = 0.0;
        for (int e = tid; e < M * N; e += ET_THREADS) Q[(size_t)(e / N) * LQ + (e % N)] = make_double2((e % N) == (e / N) ? 1.0 : 0.0, 0.0);
        __syncthreads();
    }
    if (a.may_retry && !zero && !(converged && c >= 0)) {            // the small block did not settle it: leave the window to the second pass
        if (tid == 0) a.conv[k] = -1;
        return;
    }
    const bool found = c >= 0;                                       // energy rule: the cut lies inside the block
    const int cu = found ? (c < M ? c : M) : 0;                      // vectors that make up the filter

    // ---- outputs
    const double un = a.amax ? ldexp(1.0, -2 * sm100::pow2_scale_exp(*a.amax)) : 1.0;
    double tsum = 0.0;
    for (int j = 0; j < M && j < N; ++j) tsum += theta[j] > 0.0 ? theta[j] : 0.0;
    const int Mn = M < N ? M : N;
    // reported spectrum: Ritz values (R is positive semi-definite: a value below zero is rounding and is reported as 0),
    // then the mean of what the trace leaves for the others, never above the last Ritz value
    double fill = N > Mn ? (trace - tsum) / (double)(N - Mn) : 0.0;
    fill = fill > 0.0 ? fill : 0.0;
    const double lastv = Mn > 0 && theta[Mn - 1] > 0.0 ? theta[Mn - 1] : 0.0;
    if (fill > lastv) fill = lastv;
    for (int i = tid; i < N; i += ET_THREADS) {
        const double l = i < Mn ? (theta[i] > 0.0 ? theta[i] : 0.0) : fill;
        a.lam[(size_t)k * N + i] = l * un;
        a.order[(size_t)k * N + i] = i;
        const double w = (found && i < c) || (zero && a.energy) ? 0.0 : 1.0;
        a.wt[(size_t)k * N + i] = w;
    }
    for (int u = tid; u < Ns; u += ET_THREADS) {
        const double w = (u < N && !((found && u < c) || (zero && a.energy))) ? 1.0 : 0.0;
        a.wslot[(size_t)k * Ns + u] = (float)w;
        a.wslot_dd[(size_t)k * Ns + u] = w;
    }
    if (tid == 0) {
        a.cut[k] = found ? c : 0;
        a.sweeps[k] = rounds;
        bool finite = isfinite(trace);
        for (int i = 0; i < M; ++i) finite = finite && isfinite(theta[i]);
        const int cv = converged && found && finite;
        a.conv[k] = cv;
        if (!cv) atomicAdd(a.nunconv, 1);
    }
    float2* Vk = a.V + (size_t)k * N * Ns;
    float2* Bk = a.B + (size_t)k * N * Ns;
    const bool allstop = zero && a.energy;                           // zero spectrum under the energy rule: c = N, F = 0
    for (int e = tid; e < N * Ns; e += ET_THREADS) {
        const int row = e / Ns, u = e - row * Ns;
        float2 v = make_float2(0.f, 0.f);
        if (u < Mn) { const double2 q = Q[(size_t)u * LQ + row]; v = make_float2((float)q.x, (float)q.y); }
        Vk[e] = v;
        double fr = 0.0, fi = 0.0;
        if (u < N && !allstop) {
            fr = row == u ? 1.0 : 0.0;
            for (int j = 0; j < cu; ++j) {                           // F[row][u] = delta - sum_j q_j[row] conj(q_j[u])
                const double2 x = Q[(size_t)j * LQ + row], y = Q[(size_t)j * LQ + u];
                fr -= x.x * y.x + x.y * y.y; fi -= x.y * y.x - x.x * y.y;
            }
        }
        Bk[e] = make_float2((float)fr, (float)fi);
    }
}

bool evd_top_mode(int mode) { return mode == LCF_HARD_FIXED_TOP || mode == LCF_HARD_ENERGY_TOP; }

// The subspace iteration runs when the plan asks for it, R is the fp32 Gram and the block can hold the cut; any
// other plan in these modes computes the same filter with the full-spectrum kernels.
bool evd_top_eligible(const lcf_plan* p) {
    if (!evd_top_mode(p->thr.mode) || p->prec != 0 || p->N < ET_M + 8 || p->N > ET_MAXN) return false;
    if (p->thr.mode == LCF_HARD_FIXED_TOP && p->thr.k_fixed > ET_M - ET_GUARD) return false;
    return true;
}

static size_t et_smem_bytes(int N, int M) {
    return (size_t)M * (N | 1) * 16 + (size_t)M * N * 8 + 2 * (size_t)M * M * 16 + (size_t)N * 16 + M * 16 + 2 * M * 8 + 8 * 8 + M * 4 + 16 + 64;
}

cudaError_t configure_evd_top(lcf_plan* p) {
    p->et_smem = et_smem_bytes(p->N, ET_M);
    p->et_smem_small = et_smem_bytes(p->N, ET_MS);
    if (p->et_smem > (size_t)p->smem_optin) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaSuccess;
#define ET_SET(M, CPT) if (e == cudaSuccess) e = set_max_dyn_smem(evd_top_kernel<M, CPT>, p->smem_optin)
    ET_SET(32, 32); ET_SET(32, 16); ET_SET(32, 8); ET_SET(16, 16); ET_SET(16, 8); ET_SET(16, 4);
#undef ET_SET
    return e;
}

template <int M>
static void et_launch(lcf_plan* p, const EtArgs& a, size_t smem, cudaStream_t st) {
    const int NR = (p->N + 31) & ~31;
    const int cs = ET_THREADS / NR;                                  // column blocks that fit beside the rows
    if (cs >= 4) evd_top_kernel<M, M / 4><<<p->K, ET_THREADS, smem, st>>>(a);
    else if (cs >= 2) evd_top_kernel<M, M / 2><<<p->K, ET_THREADS, smem, st>>>(a);
    else evd_top_kernel<M, M><<<p->K, ET_THREADS, smem, st>>>(a);
}

// A block of ET_MS = 16 vectors settles cuts up to 10 and is four times cheaper than the block of 32 (cuts up to 26).
// Fixed count: the block that holds it.  Energy rule: the small block first; the windows it cannot settle (cut beyond
// 10, or a slow tail) are marked and redone by a second launch with the large block, which returns at once elsewhere.
cudaError_t launch_evd_top(lcf_plan* p, cudaStream_t st) {
    EtArgs a;
    a.N = p->N; a.Ns = p->Ns; a.max_rounds = p->sweep_cap;
    a.R = reinterpret_cast<const float2*>(p->R_d); a.amax = p->gram_tc ? p->amax_d : nullptr;
    a.lam = p->lam_d; a.order = p->order_d; a.cut = p->cut_d; a.sweeps = p->sweeps_d; a.conv = p->conv_d; a.nunconv = p->nunconv_d;
    a.wslot = p->wslot_d; a.wslot_dd = p->wslot_dd_d; a.wt = p->wt_d;
    a.V = reinterpret_cast<float2*>(p->V_d); a.B = p->B_d;
    a.energy = p->thr.mode == LCF_HARD_ENERGY_TOP ? 1 : 0; a.k_fixed = p->thr.k_fixed; a.energy_frac = p->thr.energy_frac;
    a.may_retry = 0; a.retry = 0;
    if (!a.energy) {
        if (a.k_fixed <= ET_MS - ET_GUARD) et_launch<ET_MS>(p, a, p->et_smem_small, st);
        else et_launch<ET_M>(p, a, p->et_smem, st);
        return cudaGetLastError();
    }
    a.may_retry = p->sweep_cap > 0 ? 0 : 1;                          // a caller's round cap applies to the first pass alone
    et_launch<ET_MS>(p, a, p->et_smem_small, st);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess || !a.may_retry) return e;
    a.may_retry = 0; a.retry = 1;
    et_launch<ET_M>(p, a, p->et_smem, st);
    return cudaGetLastError();
}

}  // namespace lcf
