// lcf_thresh.cuh -- cut-off rules and eigen-weights shared by the three EVD kernels (step a3).
//   fixed      c = k_fixed
//   energy     c = min{m : sum_{i<=m} max(l_i,0) > frac * sum_i max(l_i,0)}    BASELINE.json configs 2-4
//   median     c = #{i : l_i > cut_scale * median(l)}       method 3, Eq. 7
//              (median of an even count = mean of the two middle values, as MATLAB's median)
//   hard       wt_i = 0 for i <= c, 1 above
//   soft       wt_i = 1 / (1 + exp(-beta (i - c)))          method 5, Eq. 9
// i is the 1-based order of the eigenvalue (descending).  Everything in double on the sorted
// eigenvalues, one thread per window: O(N).
#pragma once
#include "../../include/lcf.h"

namespace lcf {

__host__ __device__ inline bool thresh_is_soft(int mode) {
    return mode == LCF_SOFT_FIXED || mode == LCF_SOFT_ENERGY || mode == LCF_SOFT_MEDIAN;
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
    return k_fixed;
}

__device__ inline double thresh_weight(bool soft, double beta, int i1, int c) {
    if (soft) return 1.0 / (1.0 + exp(-beta * (double)(i1 - c)));
    return (i1 <= c) ? 0.0 : 1.0;
}

}  // namespace lcf
