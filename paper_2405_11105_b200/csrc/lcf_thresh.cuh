// lcf_thresh.cuh -- cut-off rules and eigen-weights shared by the three EVD kernels (step a3).
//   fixed      c = k_fixed
//   energy     c = min{m : sum_{i<=m} max(l_i,0) > frac * sum_i max(l_i,0)}    BASELINE.json configs 2-4
//   median     c = #{i : l_i > cut_scale * median(l)}       method 3, Eq. 7
//              (median of an even count = mean of the two middle values, as MATLAB's median)
//   curvature  c = argmax_n K(n), K = |y''| / (1 + y'^2)^(3/2) of the normalised log-eigenvalue curve
//              y(n) = cut_scale * N * log10(l_n) / log10(l_1)         method 1, Eq. 6
//              (central differences on n = 2..N-1, eigenvalues floored at 1e-12 l_1, lowest n on ties:
//              DESIGN.md "Readings")
//   slope      c = min{n in 1..N-1 : y(n) - y(n+1) < cut_scale} - 1 on the curve as printed, y(n) = l_n,
//              taken relative to l_1 (N - 1 if the curve never flattens)           method 2
//   slope_db   the same rule on y(n) = 10 log10(l_n) (dB per index; eigenvalues floored at 1e-12 l_1):
//              a named variant, not the printed form (DESIGN.md "Readings" 18)
//   ncc        c = argmin_k NCC(I_T(k), I_B(k))                 method 4, Eq. 8: lcf_ncc.cu (needs the data)
//   hard       wt_i = 0 for i <= c, 1 above
//   soft       wt_i = 1 / (1 + exp(-beta (i - c)))          method 5, Eq. 9
//   adaptive   wt_i = win(i) / l_i^beta, normalised to max 1     method 6, Eq. 10
//              win = right half of MATLAB's gausswin(2N-1): exp(-(2.5 (i-1)/(N-1))^2 / 2); eigenvalues
//              floored at 1e-12 l_1; no cut-off (c = 0)
// i is the 1-based order of the eigenvalue (descending).  Everything in double on the sorted
// eigenvalues, one thread per window: O(N).
#pragma once
#include "../../include/lcf.h"

namespace lcf {

__host__ __device__ inline bool thresh_is_soft(int mode) {
    return mode == LCF_SOFT_FIXED || mode == LCF_SOFT_ENERGY || mode == LCF_SOFT_MEDIAN || mode == LCF_SOFT_CURVATURE ||
           mode == LCF_SOFT_ADAPTIVE || mode == LCF_SOFT_SLOPE || mode == LCF_SOFT_SLOPE_DB || mode == LCF_SOFT_NCC;
}

__device__ inline int thresh_cutoff(int mode, int k_fixed, double energy_frac, double cut_scale, const double* lsort, int N) {
    if (mode == LCF_HARD_ENERGY || mode == LCF_SOFT_ENERGY) {
        double tot = 0.0;
        for (int i = 0; i < N; ++i) tot += lsort[i] > 0.0 ? lsort[i] : 0.0;
        double cum = 0.0;
        for (int m = 1; m <= N; ++m) {
            cum += lsort[m - 1] > 0.0 ? lsort[m - 1] : 0.0;
            if (cum > energy_frac * tot) return m;
        }
        return N;
    }
    if (mode == LCF_HARD_MEDIAN || mode == LCF_SOFT_MEDIAN) {
        const double med = (N & 1) ? lsort[(N - 1) / 2] : 0.5 * (lsort[N / 2 - 1] + lsort[N / 2]);
        const double T = cut_scale * med;
        int c = 0;
        while (c < N && lsort[c] > T) ++c;      // sorted descending
        return c;
    }
    if (mode == LCF_HARD_CURVATURE || mode == LCF_SOFT_CURVATURE) {
        if (N < 3 || !(lsort[0] > 0.0)) return 0;
        const double y1 = log10(lsort[0]);
        if (y1 == 0.0) return 0;
        const double sc = cut_scale * (double)N / y1, fl = 1e-12 * lsort[0];
        double ym = sc * y1;                                              // y(n-1)
        double y0 = sc * log10(lsort[1] > fl ? lsort[1] : fl);            // y(n)
        double best = -1.0;
        int c = 0;
        for (int n = 2; n <= N - 1; ++n) {                                // 1-based n
            const double yp = sc * log10(lsort[n] > fl ? lsort[n] : fl);  // y(n+1)
            const double d1 = 0.5 * (yp - ym), d2 = yp - 2.0 * y0 + ym;
            const double q = 1.0 + d1 * d1;
            const double kap = fabs(d2) / (q * sqrt(q));
            if (kap > best) { best = kap; c = n; }
            ym = y0; y0 = yp;
        }
        return c;
    }
    if (mode == LCF_HARD_SLOPE || mode == LCF_SOFT_SLOPE) {
        if (N < 2 || !(lsort[0] > 0.0)) return 0;
        for (int n = 1; n <= N - 1; ++n)                                  // 1-based n: drop from l_n to l_{n+1}, as a fraction of l_1
            if (lsort[n - 1] / lsort[0] - lsort[n] / lsort[0] < cut_scale) return n - 1;
        return N - 1;
    }
    if (mode == LCF_HARD_SLOPE_DB || mode == LCF_SOFT_SLOPE_DB) {
        if (N < 2 || !(lsort[0] > 0.0)) return 0;
        const double fl = 1e-12 * lsort[0];
        double y0 = 10.0 * log10(lsort[0]);
        for (int n = 1; n <= N - 1; ++n) {                                // 1-based n: drop from l_n to l_{n+1}
            const double yp = 10.0 * log10(lsort[n] > fl ? lsort[n] : fl);
            if (y0 - yp < cut_scale) return n - 1;
            y0 = yp;
        }
        return N - 1;
    }
    return k_fixed;
}

__host__ __device__ inline bool thresh_is_adaptive(int mode) { return mode == LCF_SOFT_ADAPTIVE; }

// un-normalised adaptive weight of the i1-th largest eigenvalue lam (relative to lam1 = largest: the
// constant lam1^beta cancels in the normalisation and keeps the powers in range)
__device__ inline double thresh_adaptive_raw(double lam, double lam1, int i1, int N, double beta) {
    if (!(lam1 > 0.0)) return 0.0;
    const double r = lam > 1e-12 * lam1 ? lam / lam1 : 1e-12;
    const double x = 2.5 * (double)(i1 - 1) / (double)(N - 1);
    return exp(-0.5 * x * x) * pow(r, -beta);
}
// max_i of the above over the sorted spectrum (one thread)
__device__ inline double thresh_adaptive_norm(const double* lsort, int N, double beta) {
    double m = 0.0;
    for (int i = 1; i <= N; ++i) {
        const double w = thresh_adaptive_raw(lsort[i - 1], lsort[0], i, N, beta);
        if (w > m) m = w;
    }
    return m > 0.0 ? m : 1.0;
}

__device__ inline double thresh_weight(bool soft, double beta, int i1, int c) {
    if (soft) return 1.0 / (1.0 + exp(-beta * (double)(i1 - c)));
    return (i1 <= c) ? 0.0 : 1.0;
}

}  // namespace lcf
