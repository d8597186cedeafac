/*
 * lcf_oracle.c -- float64 CPU ORACLE for the localized spatiotemporal EVD clutter filter.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  The product (paper_2405_11105_b200,
 * csrc/, liblcf.so) shares no code with it and never calls it.
 *
 * It is the paper's definition written out with plain loops in double precision
 * (arXiv 2405.11105, /root/reference/PAPER.md; line numbers below are PAPER.md lines):
 *
 *   windows        Eq. 11, PAPER.md:138-147 (2D Gaussian spatial windows, W = diag(w))
 *   gram           Eq. 12, PAPER.md:149-152 (R = sum_p w_p^2 s_p^H s_p); Eq. 1
 *   jacobi         Eq. 2,  PAPER.md:48-50   (R = V Lambda V^H, eigenvalues sorted descending)
 *   weights        PAPER.md:57-59 (hard: first k components zeroed), Eq. 9 PAPER.md:111-118 (sigmoid)
 *   cutoff_median  Eq. 7,  PAPER.md:90-96   (method 3: threshold = scale * median eigenvalue)
 *   cutoff_curvature Eq. 6, PAPER.md:77-83  (method 1: maximum curvature of the log-eigenvalue curve)
 *   weights_adaptive Eq. 10, PAPER.md:120-126 (method 6: Gaussian window over inverse eigenvalue power)
 *   cutoff_slope   PAPER.md:85-89          (method 2: slope of the eigenvalue curve y(n) = lambda_n against a threshold)
 *   cutoff_slope_db  same passage           (named variant: the same rule on the curve in dB)
 *   left_singular  PAPER.md:107            (U from C V = U D, lambda_i = sigma_i^2: spatial singular vectors)
 *   cutoff_ncc     Eq. 8, PAPER.md:98-109   (method 4: cut-off that minimises the spatial NCC of tissue and blood images)
 *   filter         Eq. 4,  PAPER.md:57-59   (F = V Lambda^ V^H)
 *   project_pd     Eq. 4 + PAPER.md:63      (C^ = C_w F; PD = sum over slow time of |C^|^2)
 *   combine        Eq. 13, PAPER.md:154-156 (PD_final = sum_k alpha_k PD_k, alpha_k = 1/mean(PD_k))
 *
 * Readings of silent / ambiguous passages: ^T on complex data is the
 * conjugate transpose; window centres at cell centres, peak 1, separable box truncation
 * |d| <= trunc*sigma; PD is the slow-time SUM; alpha_k uses the mean over the full field of view;
 * 1-based eigen index; the 99.5 % energy rule is BASELINE.json's, not the paper's.
 *
 * Pins (tests/test_oracle_pins.py): numpy eigh/svd/matmul in float64, 2x2 closed form, trace
 * identities, idempotence, rank-r clutter removal, DC removal, a literal windowed-copy brute force.
 * Parity unpinned: nothing (no value printed in the paper is reproducible without its data).
 *
 * Layouts (C order, complex = interleaved re,im):
 *   iq   float  [N][Nx][Nz][2]   frame, lateral x, axial z (z fastest); Casorati row p = z + Nz*x
 *   R,F  double [N][N][2]        R[i][j] = sum_p w^2 conj(S[i][p]) S[j][p]
 *   V    double [N][N][2]        V[a][i] = component a of eigenvector i (columns = eigenvectors)
 *   PD   double [Nx][Nz]
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define RE(A, i, j, n) ((A)[2 * ((size_t)(i) * (n) + (j))])
#define IM(A, i, j, n) ((A)[2 * ((size_t)(i) * (n) + (j)) + 1])

enum { LCFO_HARD_FIXED = 0, LCFO_HARD_ENERGY = 1, LCFO_SOFT_FIXED = 2, LCFO_SOFT_ENERGY = 3,
       LCFO_HARD_MEDIAN = 4, LCFO_SOFT_MEDIAN = 5, LCFO_HARD_CURVATURE = 6, LCFO_SOFT_CURVATURE = 7,
       LCFO_SOFT_ADAPTIVE = 8, LCFO_HARD_SLOPE = 9, LCFO_SOFT_SLOPE = 10, LCFO_HARD_SLOPE_DB = 11, LCFO_SOFT_SLOPE_DB = 12,
       LCFO_HARD_NCC = 13, LCFO_SOFT_NCC = 14,
       /* include/lcf.h's *_TOP modes name a way of computing (leading eigenpairs only), not another filter: here they
        * ARE the definition, F = V diag(wt) V^H from the full decomposition with the hard weights of mode 0 / 1 */
       LCFO_HARD_FIXED_TOP = 15, LCFO_HARD_ENERGY_TOP = 16 };

int lcf_oracle_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* Eq. 11.  One axis of the separable Gaussian window grid.
 * centre c_k = (k + 1/2) * n / K - 1/2 (cell centres); g = exp(-(i-c)^2 / (2 sigma^2)) inside the
 * support |i - c| <= trunc * sigma, 0 outside.  sigma <= 0: all-ones; trunc <= 0: no truncation. */
void lcf_oracle_axis_windows(int n, int K, double sigma, double trunc, double *g /* [K][n] */) {
    for (int k = 0; k < K; ++k) {
        double c = (k + 0.5) * (double)n / (double)K - 0.5;
        for (int i = 0; i < n; ++i) {
            double v;
            if (sigma <= 0.0) {
                v = 1.0;
            } else {
                double d = (double)i - c;
                if (trunc > 0.0 && fabs(d) > trunc * sigma) v = 0.0;
                else v = exp(-(d * d) / (2.0 * sigma * sigma));
            }
            g[(size_t)k * n + i] = v;
        }
    }
}

/* Eq. 12: R[i][j] = sum_p w_p^2 conj(S[i][p]) S[j][p], w_p = gz[z] * gx[x].
 * No 1/P or 1/N normalisation (Eq. 1 is a plain sum). */
void lcf_oracle_gram(const float *iq, int N, int Nx, int Nz, const double *gz, const double *gx,
                     double *R /* [N][N][2] */) {
    size_t P = (size_t)Nx * Nz;
    double *sr = (double *)malloc(sizeof(double) * N), *si = (double *)malloc(sizeof(double) * N);
    memset(R, 0, sizeof(double) * 2 * (size_t)N * N);
    for (int x = 0; x < Nx; ++x) {
        for (int z = 0; z < Nz; ++z) {
            double w = gz[z] * gx[x];
            double w2 = w * w;
            if (w2 == 0.0) continue;
            size_t p = (size_t)x * Nz + z;
            for (int i = 0; i < N; ++i) {
                sr[i] = (double)iq[2 * ((size_t)i * P + p)];
                si[i] = (double)iq[2 * ((size_t)i * P + p) + 1];
            }
            for (int i = 0; i < N; ++i) {
                for (int j = i; j < N; ++j) {
                    /* conj(s_i) * s_j */
                    RE(R, i, j, N) += w2 * (sr[i] * sr[j] + si[i] * si[j]);
                    IM(R, i, j, N) += w2 * (sr[i] * si[j] - si[i] * sr[j]);
                }
            }
        }
    }
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < i; ++j) {
            RE(R, i, j, N) = RE(R, j, i, N);
            IM(R, i, j, N) = -IM(R, j, i, N);
        }
    free(sr);
    free(si);
}

static double offdiag_fro2(const double *A, int N) {
    double s = 0.0;
    for (int i = 0; i < N; ++i)
        for (int j = 0; j < N; ++j)
            if (i != j) s += RE(A, i, j, N) * RE(A, i, j, N) + IM(A, i, j, N) * IM(A, i, j, N);
    return s;
}

/* Eq. 2: R = V Lambda V^H by the cyclic-by-row complex Jacobi method.
 * For p < q with a = A_pq != 0: phi = arg a, tau = (A_qq - A_pp) / (2|a|),
 * t = sign(tau) / (|tau| + sqrt(1 + tau^2)) (t = 1 if tau = 0), c = 1/sqrt(1+t^2), s = t c,
 * J = [[c, s e^{i phi}], [-s e^{-i phi}, c]] on (p, q);  A <- J^H A J,  V <- V J.
 * (J = D G D^H with D = diag(1, e^{-i phi}) and G the real Jacobi rotation of the real-symmetric
 * 2x2 block of D^H A D.)  Stops when off(A)_F <= 1e-14 ||R||_F; eigenvalues = real diag(A), sorted
 * descending (stable on index), V permuted alike.  Returns sweeps used, or -1 if not converged. */
int lcf_oracle_jacobi(const double *R, int N, double *lam /* [N] */, double *V /* [N][N][2] */) {
    size_t nn = (size_t)N * N;
    double *A = (double *)malloc(sizeof(double) * 2 * nn);
    memcpy(A, R, sizeof(double) * 2 * nn);
    memset(V, 0, sizeof(double) * 2 * nn);
    for (int i = 0; i < N; ++i) RE(V, i, i, N) = 1.0;
    double fro2 = 0.0;
    for (size_t e = 0; e < 2 * nn; ++e) fro2 += A[e] * A[e];
    const double tol2 = 1e-28 * fro2;
    int sweep = 0, converged = 0;
    for (sweep = 0; sweep <= 60; ++sweep) {
        if (offdiag_fro2(A, N) <= tol2) { converged = 1; break; }
        if (sweep == 60) break;
        for (int p = 0; p < N - 1; ++p) {
            for (int q = p + 1; q < N; ++q) {
                double ar = RE(A, p, q, N), ai = IM(A, p, q, N);
                double absa = hypot(ar, ai);
                if (absa == 0.0) continue;
                double er = ar / absa, ei = ai / absa;            /* e^{i phi} */
                double tau = (RE(A, q, q, N) - RE(A, p, p, N)) / (2.0 * absa);
                double t = (tau == 0.0) ? 1.0 : ((tau > 0.0 ? 1.0 : -1.0) / (fabs(tau) + sqrt(1.0 + tau * tau)));
                double c = 1.0 / sqrt(1.0 + t * t), s = t * c;
                double gr = s * er, gi = s * ei;                  /* s e^{i phi} */
                /* A <- A J : columns p, q.  (AJ)[k][p] = c A[k][p] - s e^{-i phi} A[k][q];
                 *                          (AJ)[k][q] = s e^{i phi} A[k][p] + c A[k][q] */
                for (int k = 0; k < N; ++k) {
                    double pr = RE(A, k, p, N), pi = IM(A, k, p, N);
                    double qr = RE(A, k, q, N), qi = IM(A, k, q, N);
                    RE(A, k, p, N) = c * pr - (gr * qr + gi * qi);
                    IM(A, k, p, N) = c * pi - (gr * qi - gi * qr);
                    RE(A, k, q, N) = (gr * pr - gi * pi) + c * qr;
                    IM(A, k, q, N) = (gr * pi + gi * pr) + c * qi;
                }
                /* A <- J^H A : rows p, q.  (J^H A)[p][k] = c A[p][k] - s e^{i phi} A[q][k];
                 *                          (J^H A)[q][k] = s e^{-i phi} A[p][k] + c A[q][k] */
                for (int k = 0; k < N; ++k) {
                    double pr = RE(A, p, k, N), pi = IM(A, p, k, N);
                    double qr = RE(A, q, k, N), qi = IM(A, q, k, N);
                    RE(A, p, k, N) = c * pr - (gr * qr - gi * qi);
                    IM(A, p, k, N) = c * pi - (gr * qi + gi * qr);
                    RE(A, q, k, N) = (gr * pr + gi * pi) + c * qr;
                    IM(A, q, k, N) = (gr * pi - gi * pr) + c * qi;
                }
                /* V <- V J */
                for (int k = 0; k < N; ++k) {
                    double pr = RE(V, k, p, N), pi = IM(V, k, p, N);
                    double qr = RE(V, k, q, N), qi = IM(V, k, q, N);
                    RE(V, k, p, N) = c * pr - (gr * qr + gi * qi);
                    IM(V, k, p, N) = c * pi - (gr * qi - gi * qr);
                    RE(V, k, q, N) = (gr * pr - gi * pi) + c * qr;
                    IM(V, k, q, N) = (gr * pi + gi * pr) + c * qi;
                }
            }
        }
    }
    /* sort descending, stable on index (insertion sort on an index array) */
    int *idx = (int *)malloc(sizeof(int) * N);
    for (int i = 0; i < N; ++i) idx[i] = i;
    for (int i = 1; i < N; ++i) {
        int v = idx[i], j = i - 1;
        while (j >= 0 && RE(A, idx[j], idx[j], N) < RE(A, v, v, N)) { idx[j + 1] = idx[j]; --j; }
        idx[j + 1] = v;
    }
    double *Vs = (double *)malloc(sizeof(double) * 2 * nn);
    for (int i = 0; i < N; ++i) {
        lam[i] = RE(A, idx[i], idx[i], N);
        for (int k = 0; k < N; ++k) {
            RE(Vs, k, i, N) = RE(V, k, idx[i], N);
            IM(Vs, k, i, N) = IM(V, k, idx[i], N);
        }
    }
    memcpy(V, Vs, sizeof(double) * 2 * nn);
    free(Vs); free(idx); free(A);
    return converged ? sweep : -1;
}

/* BASELINE.json energy rule (not in the paper): c = smallest 1-based m with
 * sum_{i<=m} max(lam_i, 0) > frac * sum_i max(lam_i, 0);  N if no such m. */
int lcf_oracle_cutoff_energy(const double *lam, int N, double frac) {
    double tot = 0.0;
    for (int i = 0; i < N; ++i) tot += lam[i] > 0.0 ? lam[i] : 0.0;
    double cum = 0.0;
    for (int m = 1; m <= N; ++m) {
        cum += lam[m - 1] > 0.0 ? lam[m - 1] : 0.0;
        if (cum > frac * tot) return m;
    }
    return N;
}

/* Method 3, Eq. 7: threshold T = scale * lambda_median; "the eigen components with
 * eigenvalues larger than this threshold ... can thus be removed": c = #{i : lam_i > T}.
 * lam is sorted descending.  Median of an even count = mean of the two middle values (MATLAB's
 * median; the paper does not say -- DESIGN.md "Readings"). */
int lcf_oracle_cutoff_median(const double *lam, int N, double scale) {
    double med = (N % 2) ? lam[(N - 1) / 2] : 0.5 * (lam[N / 2 - 1] + lam[N / 2]);
    double T = scale * med;
    int c = 0;
    for (int i = 0; i < N; ++i)
        if (lam[i] > T) ++c;
    return c;
}

/* Method 1, Eq. 6: "considering the eigenvalue as a function of eigenvalue order n
 * in logarithmic scale, y(n) = log10 lambda_n ... the curve is normalized as beta y(n)/y(1) Nt before
 * computing the curvature" K = |y''| / (1 + y'^2)^(3/2); "the maximum curvature gives the estimate of
 * threshold cutoff (denoted as k), which is used as the number of eigen components to be rejected".
 * Not in the paper: derivatives are central differences
 * y'(n) = (y(n+1) - y(n-1))/2, y''(n) = y(n+1) - 2 y(n) + y(n-1) on n = 2..N-1; eigenvalues are
 * floored at 1e-12 lambda_1 so that the logarithm exists; the lowest n wins a tie; N < 3,
 * lambda_1 <= 0 or log10 lambda_1 = 0 (normalisation undefined) give k = 0. */
int lcf_oracle_cutoff_curvature(const double *lam, int N, double scale) {
    if (N < 3 || !(lam[0] > 0.0)) return 0;
    double y1 = log10(lam[0]);
    if (y1 == 0.0) return 0;
    double *y = (double *)malloc(sizeof(double) * (size_t)N);
    for (int n = 0; n < N; ++n) {
        double l = lam[n] > 1e-12 * lam[0] ? lam[n] : 1e-12 * lam[0];
        y[n] = scale * (log10(l) / y1) * (double)N;
    }
    int k = 0;
    double best = -1.0;
    for (int n = 2; n <= N - 1; ++n) { /* 1-based order n, y[n-1] */
        double d1 = (y[n] - y[n - 2]) / 2.0;
        double d2 = y[n] - 2.0 * y[n - 1] + y[n - 2];
        double kap = fabs(d2) / pow(1.0 + d1 * d1, 1.5);
        if (kap > best) { best = kap; k = n; }
    }
    free(y);
    return k;
}

/* Method 2: "calculates the slope, or the first derivative of the singular value
 * curve and requires a properly predefined slope threshold above which the singular values are
 * removed ... the slope estimation of the eigenvalue curve y(n) = lambda_n and the identified
 * eigenvalue cutoff based [on] a predefined slope threshold of -1.1."
 * As printed: the curve is the eigenvalues themselves (linear, unlike method 1's log10).  The
 * descending curve has slope y(n+1) - y(n) <= 0 (forward difference); the steep leading part
 * (slope below -T, i.e. "above" the threshold in magnitude) is tissue and is removed; the cut is
 * where the curve first flattens:  k = (first n in 1..N-1 with y(n) - y(n+1) < T) - 1.
 * Reading (DESIGN.md "Readings" 18): the paper's -1.1 is in the units of the authors' data, so the
 * curve is taken relative to its first point, y(n) = lambda_n / lambda_1, and `thresh` = T > 0 is
 * the magnitude of the slope per eigenvalue index on that curve.  A curve that never flattens keeps
 * only its last component (k = N-1); N < 2 or lambda_1 <= 0 give k = 0. */
int lcf_oracle_cutoff_slope(const double *lam, int N, double thresh) {
    if (N < 2 || !(lam[0] > 0.0)) return 0;
    for (int n = 1; n <= N - 1; ++n) { /* 1-based order n: lam[n-1] -> lam[n] */
        double drop = lam[n - 1] / lam[0] - lam[n] / lam[0];
        if (drop < thresh) return n - 1;
    }
    return N - 1;
}

/* Named variant of method 2 (not the printed form): the same rule on the curve in dB,
 * y(n) = 10 log10(lambda_n) -- independent of the units of the data without a normalisation, and
 * the scale on which eigenvalue curves are usually drawn.  `thresh` = drop in dB per eigenvalue
 * index; eigenvalues floored at 1e-12 lambda_1 so that the logarithm exists. */
int lcf_oracle_cutoff_slope_db(const double *lam, int N, double thresh) {
    if (N < 2 || !(lam[0] > 0.0)) return 0;
    for (int n = 1; n <= N - 1; ++n) {
        double a = lam[n - 1] > 1e-12 * lam[0] ? lam[n - 1] : 1e-12 * lam[0];
        double b = lam[n] > 1e-12 * lam[0] ? lam[n] : 1e-12 * lam[0];
        if (10.0 * log10(a) - 10.0 * log10(b) < thresh) return n - 1;
    }
    return N - 1;
}

/* Eigen weights, 1-based order i (stored at wt[i-1]).
 * hard: wt_i = 0 for i <= c, 1 for i > c.
 * soft (Eq. 9): wt_i = 1 / (1 + exp(-beta (i - c))). */
void lcf_oracle_weights(int N, int soft, int c, double beta, double *wt) {
    for (int i = 1; i <= N; ++i) {
        if (soft) wt[i - 1] = 1.0 / (1.0 + exp(-beta * (double)(i - c)));
        else wt[i - 1] = (i <= c) ? 0.0 : 1.0;
    }
}

/* Method 6, Eq. 10: wt_i = win(i) / lambda_i^beta, "win(i) represents the Gaussian
 * window center at i=0 (generated by 'gausswin' function in Matlab). The weighting function wt_i is
 * normalized before assigning to eigenvalues".  Not in the paper: win is the
 * right half of gausswin(2N-1) with MATLAB's default alpha = 2.5, i.e.
 * win(i) = exp(-(alpha (i-1)/(N-1))^2 / 2), i = 1..N (1 at the largest eigenvalue); "normalized" =
 * divided by the largest weight; eigenvalues are floored at 1e-12 lambda_1. */
void lcf_oracle_weights_adaptive(const double *lam, int N, double beta, double *wt) {
    double mx = 0.0;
    for (int i = 1; i <= N; ++i) {
        double l = lam[i - 1] > 1e-12 * lam[0] ? lam[i - 1] : 1e-12 * lam[0];
        double x = 2.5 * (double)(i - 1) / (double)(N - 1);
        double w = (lam[0] > 0.0) ? exp(-0.5 * x * x) / pow(l, beta) : 0.0;
        wt[i - 1] = w;
        if (w > mx) mx = w;
    }
    if (mx > 0.0)
        for (int i = 0; i < N; ++i) wt[i] /= mx;
}

/* Eq. 4, PAPER.md:57-59 with Lambda^ = diag(wt):  F = V diag(wt) V^H. */
void lcf_oracle_filter(const double *V, const double *wt, int N, double *F) {
    for (int a = 0; a < N; ++a)
        for (int b = 0; b < N; ++b) {
            double fr = 0.0, fi = 0.0;
            for (int i = 0; i < N; ++i) {
                double ar = RE(V, a, i, N), ai = IM(V, a, i, N);
                double br = RE(V, b, i, N), bi = IM(V, b, i, N);
                /* V[a][i] * conj(V[b][i]) */
                fr += wt[i] * (ar * br + ai * bi);
                fi += wt[i] * (ai * br - ar * bi);
            }
            RE(F, a, b, N) = fr;
            IM(F, a, b, N) = fi;
        }
}

/* Eq. 4 on the windowed data (Eq. 11) + PAPER.md:63: y_p = (w_p s_p) F;  PD_k(p) = sum_j |y_p[j]|^2.
 * PDk is the full field of view [Nx][Nz] (0 where w = 0). */
void lcf_oracle_project_pd(const float *iq, int N, int Nx, int Nz, const double *gz, const double *gx,
                           const double *F, double *PDk) {
    size_t P = (size_t)Nx * Nz;
    double *sr = (double *)malloc(sizeof(double) * N), *si = (double *)malloc(sizeof(double) * N);
    for (int x = 0; x < Nx; ++x) {
        for (int z = 0; z < Nz; ++z) {
            size_t p = (size_t)x * Nz + z;
            double w = gz[z] * gx[x];
            if (w == 0.0) { PDk[p] = 0.0; continue; }
            for (int i = 0; i < N; ++i) {
                sr[i] = w * (double)iq[2 * ((size_t)i * P + p)];
                si[i] = w * (double)iq[2 * ((size_t)i * P + p) + 1];
            }
            double pw = 0.0;
            for (int j = 0; j < N; ++j) {
                double yr = 0.0, yi = 0.0;
                for (int i = 0; i < N; ++i) {
                    double fr = RE(F, i, j, N), fi = IM(F, i, j, N);
                    yr += sr[i] * fr - si[i] * fi;
                    yi += sr[i] * fi + si[i] * fr;
                }
                pw += yr * yr + yi * yi;
            }
            PDk[p] = pw;
        }
    }
    free(sr);
    free(si);
}

/* "U can be calculated from the eigenvectors according to CV = UD and lambda_i = sigma_i^2":
 * u_i = C_w v_i / sigma_i on the windowed data C_w = W C (Eq. 11), sigma_i = sqrt(lambda_i); only the
 * magnitudes |u_i(p)| are used by method 4 and only they are returned:  Umag [P][N] (pixel p = z + Nz x,
 * component i in the order of lam / V).  A component with lambda_i <= 1e-12 lambda_1 (sigma = 0 up to
 * round-off: u undefined) gets |u_i| = 0. */
void lcf_oracle_left_singular_mag(const float *iq, int N, int Nx, int Nz, const double *gz, const double *gx,
                                  const double *lam, const double *V, double *Umag /* [P][N] */) {
    size_t P = (size_t)Nx * Nz;
    double *sr = (double *)malloc(sizeof(double) * N), *si = (double *)malloc(sizeof(double) * N);
    for (int x = 0; x < Nx; ++x)
        for (int z = 0; z < Nz; ++z) {
            size_t p = (size_t)x * Nz + z;
            double w = gz[z] * gx[x];
            for (int t = 0; t < N; ++t) {
                sr[t] = w * (double)iq[2 * ((size_t)t * P + p)];
                si[t] = w * (double)iq[2 * ((size_t)t * P + p) + 1];
            }
            for (int i = 0; i < N; ++i) {
                double ur = 0.0, ui = 0.0;                 /* (C_w V)[p][i] = sum_t s_t V[t][i] */
                for (int t = 0; t < N; ++t) {
                    double vr = RE(V, t, i, N), vi = IM(V, t, i, N);
                    ur += sr[t] * vr - si[t] * vi;
                    ui += sr[t] * vi + si[t] * vr;
                }
                double sig = (lam[i] > 1e-12 * lam[0] && lam[i] > 0.0) ? sqrt(lam[i]) : 0.0;
                Umag[p * N + i] = sig > 0.0 ? hypot(ur, ui) / sig : 0.0;
            }
        }
    free(sr);
    free(si);
}

/* Method 4, Eq. 8: k = argmin_k NCC(k),
 *   NCC(k) = sum_p I_T I_B / (sqrt(sum_p I_T^2) sqrt(sum_p I_B^2)),
 * with the simplified images of PAPER.md:107 ("a given number fn of left singular vectors next to the
 * cutoff k ... fn = 5, and w_i = 1"; the printed index ranges are garbled -- DESIGN.md "Readings" 19):
 *   I_T(k) = sum_{i=k-fn+1}^{k} |u_i|      I_B(k) = sum_{i=k+1}^{k+fn} |u_i|       (1-based i, clipped to 1..N).
 * k runs over 1..N-1 (at k = N there is no blood image); the lowest k wins a tie; a k whose I_T or I_B
 * vanishes everywhere gets NCC = +inf (never chosen unless all do, then k = 1).  ncc [N] receives the
 * curve (ncc[k-1] = NCC(k), ncc[N-1] = +inf) if not NULL.  Umag [P][N]. */
int lcf_oracle_cutoff_ncc(const double *Umag, size_t P, int N, int fn, double *ncc) {
    int best_k = 1;
    double best = HUGE_VAL;
    for (int k = 1; k <= N; ++k) {
        double v = HUGE_VAL;
        if (k <= N - 1) {
            int t0 = k - fn + 1 < 1 ? 1 : k - fn + 1, b1 = k + fn > N ? N : k + fn;
            double stb = 0.0, stt = 0.0, sbb = 0.0;
            for (size_t p = 0; p < P; ++p) {
                double it = 0.0, ib = 0.0;
                for (int i = t0; i <= k; ++i) it += Umag[p * N + (i - 1)];
                for (int i = k + 1; i <= b1; ++i) ib += Umag[p * N + (i - 1)];
                stb += it * ib; stt += it * it; sbb += ib * ib;
            }
            if (stt > 0.0 && sbb > 0.0) v = stb / (sqrt(stt) * sqrt(sbb));
        }
        if (ncc) ncc[k - 1] = v;
        if (v < best) { best = v; best_k = k; }
    }
    return best_k;
}

/* One window k = (kz, kx) end to end.  Any output pointer may be NULL except lam.
 * Returns Jacobi sweeps (or -1).  c_out = number of rejected components. */
int lcf_oracle_window(const float *iq, int N, int Nx, int Nz, const double *gz, const double *gx,
                      int mode, int k_fixed, double frac, double beta, double cut_scale,
                      double *R_out, double *lam, double *V_out, int *c_out, double *wt_out,
                      double *F_out, double *PDk_out, double *mean_out) {
    size_t nn = (size_t)N * N, P = (size_t)Nx * Nz;
    double *R = (double *)malloc(sizeof(double) * 2 * nn);
    double *V = (double *)malloc(sizeof(double) * 2 * nn);
    double *F = (double *)malloc(sizeof(double) * 2 * nn);
    double *wt = (double *)malloc(sizeof(double) * N);
    double *PDk = (double *)malloc(sizeof(double) * P);
    lcf_oracle_gram(iq, N, Nx, Nz, gz, gx, R);
    int sweeps = lcf_oracle_jacobi(R, N, lam, V);
    int c = k_fixed;
    if (mode == LCFO_HARD_ENERGY || mode == LCFO_SOFT_ENERGY || mode == LCFO_HARD_ENERGY_TOP) c = lcf_oracle_cutoff_energy(lam, N, frac);
    if (mode == LCFO_HARD_MEDIAN || mode == LCFO_SOFT_MEDIAN) c = lcf_oracle_cutoff_median(lam, N, cut_scale);
    if (mode == LCFO_HARD_CURVATURE || mode == LCFO_SOFT_CURVATURE) c = lcf_oracle_cutoff_curvature(lam, N, cut_scale);
    if (mode == LCFO_HARD_SLOPE || mode == LCFO_SOFT_SLOPE) c = lcf_oracle_cutoff_slope(lam, N, cut_scale);
    if (mode == LCFO_HARD_SLOPE_DB || mode == LCFO_SOFT_SLOPE_DB) c = lcf_oracle_cutoff_slope_db(lam, N, cut_scale);
    if (mode == LCFO_HARD_NCC || mode == LCFO_SOFT_NCC) {            /* method 4; method 5 on top of it as the paper pairs them */
        double *Um = (double *)malloc(sizeof(double) * P * (size_t)N);
        lcf_oracle_left_singular_mag(iq, N, Nx, Nz, gz, gx, lam, V, Um);
        c = lcf_oracle_cutoff_ncc(Um, P, N, 5, NULL);
        free(Um);
    }
    int soft = (mode == LCFO_SOFT_FIXED || mode == LCFO_SOFT_ENERGY || mode == LCFO_SOFT_MEDIAN || mode == LCFO_SOFT_CURVATURE ||
                mode == LCFO_SOFT_SLOPE || mode == LCFO_SOFT_SLOPE_DB || mode == LCFO_SOFT_NCC);
    if (mode == LCFO_SOFT_ADAPTIVE) { c = 0; lcf_oracle_weights_adaptive(lam, N, beta, wt); }
    else lcf_oracle_weights(N, soft, c, beta, wt);
    lcf_oracle_filter(V, wt, N, F);
    lcf_oracle_project_pd(iq, N, Nx, Nz, gz, gx, F, PDk);
    double m = 0.0;
    for (size_t p = 0; p < P; ++p) m += PDk[p];
    m /= (double)P;
    if (R_out) memcpy(R_out, R, sizeof(double) * 2 * nn);
    if (V_out) memcpy(V_out, V, sizeof(double) * 2 * nn);
    if (F_out) memcpy(F_out, F, sizeof(double) * 2 * nn);
    if (wt_out) memcpy(wt_out, wt, sizeof(double) * N);
    if (PDk_out) memcpy(PDk_out, PDk, sizeof(double) * P);
    if (c_out) *c_out = c;
    if (mean_out) *mean_out = m;
    free(R); free(V); free(F); free(wt); free(PDk);
    return sweeps;
}

/* Eq. 13: PD = sum_k alpha_k PD_k, alpha_k = 1 / mean_p PD_k(p) (0 if the mean is 0). */
void lcf_oracle_combine(const double *PDk_all /* [K][P] */, int K, size_t P, double *alpha, double *PD) {
    for (size_t p = 0; p < P; ++p) PD[p] = 0.0;
    for (int k = 0; k < K; ++k) {
        const double *pk = PDk_all + (size_t)k * P;
        double m = 0.0;
        for (size_t p = 0; p < P; ++p) m += pk[p];
        m /= (double)P;
        alpha[k] = (m > 0.0) ? 1.0 / m : 0.0;
        for (size_t p = 0; p < P; ++p) PD[p] += alpha[k] * pk[p];
    }
}

/* Whole path for one ensemble: all K = Kz*Kx windows (k = kx*Kz + kz), then Eq. 13.
 * Windows are independent, so they run under OpenMP when compiled with it; the combination is
 * serial in k order.  Optional outputs (NULL to skip): R_all/F_all/V_all [K][N][N][2] (V: columns =
 * eigenvectors, descending eigenvalue order), mean_all [K].
 * Returns 0, or -(k+1) for the first window whose Jacobi iteration did not converge. */
int lcf_oracle_run(const float *iq, int N, int Nx, int Nz, int Kz, int Kx,
                   double sigma_z, double sigma_x, double trunc,
                   int mode, int k_fixed, double frac, double beta, double cut_scale,
                   double *PD /* [Nx][Nz] */, double *lam_all /* [K][N] */, int *c_all /* [K] */,
                   double *mean_all, double *R_all, double *F_all, double *V_all) {
    int K = Kz * Kx;
    size_t P = (size_t)Nx * Nz, nn = (size_t)N * N;
    double *gz = (double *)malloc(sizeof(double) * (size_t)Kz * Nz);
    double *gx = (double *)malloc(sizeof(double) * (size_t)Kx * Nx);
    lcf_oracle_axis_windows(Nz, Kz, sigma_z, trunc, gz);
    lcf_oracle_axis_windows(Nx, Kx, sigma_x, trunc, gx);
    double *means = (double *)malloc(sizeof(double) * K);
    int *status = (int *)malloc(sizeof(int) * K);
    /* PD_k kept only on each window's bounding box so large configs fit in memory */
    double **tiles = (double **)malloc(sizeof(double *) * K);
    int *bx0 = (int *)malloc(sizeof(int) * K), *bx1 = (int *)malloc(sizeof(int) * K);
    int *bz0 = (int *)malloc(sizeof(int) * K), *bz1 = (int *)malloc(sizeof(int) * K);
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (int k = 0; k < K; ++k) {
        int kz = k % Kz, kx = k / Kz;
        const double *gzk = gz + (size_t)kz * Nz, *gxk = gx + (size_t)kx * Nx;
        double *PDk = (double *)malloc(sizeof(double) * P);
        status[k] = lcf_oracle_window(iq, N, Nx, Nz, gzk, gxk, mode, k_fixed, frac, beta, cut_scale,
                                      R_all ? R_all + 2 * nn * k : NULL, lam_all + (size_t)N * k,
                                      V_all ? V_all + 2 * nn * k : NULL, c_all + k, NULL, F_all ? F_all + 2 * nn * k : NULL, PDk, means + k);
        int z0 = Nz, z1 = -1, x0 = Nx, x1 = -1;
        for (int z = 0; z < Nz; ++z) if (gzk[z] != 0.0) { if (z < z0) z0 = z; if (z > z1) z1 = z; }
        for (int x = 0; x < Nx; ++x) if (gxk[x] != 0.0) { if (x < x0) x0 = x; if (x > x1) x1 = x; }
        bz0[k] = z0; bz1[k] = z1; bx0[k] = x0; bx1[k] = x1;
        size_t nz = (z1 >= z0) ? (size_t)(z1 - z0 + 1) : 0, nx = (x1 >= x0) ? (size_t)(x1 - x0 + 1) : 0;
        tiles[k] = (double *)malloc(sizeof(double) * (nz * nx + 1));
        for (size_t x = 0; x < nx; ++x)
            for (size_t z = 0; z < nz; ++z)
                tiles[k][x * nz + z] = PDk[(x0 + x) * (size_t)Nz + (z0 + z)];
        free(PDk);
    }
    for (size_t p = 0; p < P; ++p) PD[p] = 0.0;
    int rc = 0;
    for (int k = 0; k < K; ++k) {
        if (status[k] < 0 && rc == 0) rc = -(k + 1);
        double alpha = (means[k] > 0.0) ? 1.0 / means[k] : 0.0;
        if (mean_all) mean_all[k] = means[k];
        if (bz1[k] >= bz0[k] && bx1[k] >= bx0[k]) {
            size_t nz = (size_t)(bz1[k] - bz0[k] + 1);
            for (int x = bx0[k]; x <= bx1[k]; ++x)
                for (int z = bz0[k]; z <= bz1[k]; ++z)
                    PD[(size_t)x * Nz + z] += alpha * tiles[k][(size_t)(x - bx0[k]) * nz + (z - bz0[k])];
        }
        free(tiles[k]);
    }
    free(tiles); free(bx0); free(bx1); free(bz0); free(bz1);
    free(means); free(status); free(gz); free(gx);
    return rc;
}
