/*
 * lcf.h -- C ABI of liblcf.so: the B200 (sm_100a) localized spatiotemporal EVD clutter filter.
 *
 * One call of lcf_filter() runs, for one slow-time ensemble, the whole hot path of
 * arXiv 2405.11105 (Huang et al.), cited below as PAPER.md:<line> of the extracted text:
 *
 *   a1  window-weighted temporal covariances   R_k = S^H diag(w_k^2) S        Eqs. 1, 11, 12
 *                                                                              PAPER.md:41-46, 138-152
 *   a2  batched Hermitian eigendecomposition   R_k = V_k Lambda_k V_k^H       Eq. 2
 *   a3  eigen-weights and projector factor     wt (hard cut / sigmoid), B_k = V_k diag(wt)
 *                                                                              PAPER.md:57-59, Eq. 9 :111-118
 *   a4  projection + power Doppler             PD_k(p) = w_k(p)^2 sum_t |(s_p V_k diag(wt) V_k^H)_t|^2
 *                                                                              Eq. 4
 *   a5  recombination                          PD = sum_k PD_k / mean_p(PD_k)  Eq. 13
 *
 * Every step runs in hand-written CUDA kernels; there is no CPU fallback.  All functions return an
 * lcf_status; none throws, aborts or prints.  Pointers are marked HOST or DEVICE.
 *
 * Data layout (the Casorati matrix of an Ny x Nx x Nt MATLAB cube, z fastest):
 *   iq  DEVICE, complex64 interleaved (re, im), C order [N][Nx][Nz]: frame t, lateral x, axial z.
 *       Casorati row p = z + Nz*x, column = frame.  16-byte aligned.  Read only.
 *   pd  DEVICE, float32 [Nx][Nz].  Overwritten.
 *   Window index k = kx*Kz + kz.
 */
#ifndef LCF_H_
#define LCF_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lcf_plan lcf_plan; /* opaque; owns window tables and all device workspace */

typedef enum {
    LCF_OK = 0,
    LCF_ERR_INVALID_ARG = 1,   /* NULL pointer, non-positive size, bad mode/parameter            */
    LCF_ERR_UNSUPPORTED = 2,   /* N beyond what the EVD kernel holds in shared memory            */
    LCF_ERR_ALLOC = 3,         /* device or host allocation failed                                */
    LCF_ERR_CUDA = 4,          /* a CUDA call or launch failed (sticky per plan)                  */
    LCF_ERR_NOT_CONVERGED = 5  /* some window's Jacobi iteration hit the sweep cap unconverged    */
} lcf_status;

/* Gaussian window grid (Eq. 11; centre/SD formulas are not given in the paper,
 * DESIGN.md "Readings"): per axis, centre c_k = (k + 1/2) n / K - 1/2 (0-based
 * pixels), g(i) = exp(-(i - c_k)^2 / (2 sigma^2)) for |i - c_k| <= trunc_sigmas * sigma, else 0;
 * w_k(z, x) = g_z(z) g_x(x).  sigma <= 0 on an axis: g = 1 on that axis (all-ones window).
 * trunc_sigmas <= 0: no truncation.  Evaluated in double precision. */
typedef struct {
    int Kz, Kx;
    float sigma_z, sigma_x;
    float trunc_sigmas;
} lcf_windows;

typedef enum {
    LCF_HARD_FIXED = 0,  /* wt_i = 0 for i <= k_fixed, 1 above (i is 1-based)          */
    LCF_HARD_ENERGY = 1, /* hard, c = min{m : sum_{i<=m} max(l_i,0) > energy_frac * sum_i max(l_i,0)}*/
    LCF_SOFT_FIXED = 2,  /* wt_i = 1 / (1 + exp(-beta (i - k_fixed)))  (Eq. 9)     */
    LCF_SOFT_ENERGY = 3, /* sigmoid centred on the energy-rule c                                     */
    LCF_HARD_MEDIAN = 4, /* hard, c = #{i : l_i > cut_scale * median(l)}  (method 3, Eq. 7,
                            PAPER.md:90-96; even count: mean of the two middle eigenvalues)         */
    LCF_SOFT_MEDIAN = 5, /* sigmoid (Eq. 9) centred on the median-rule c                             */
    LCF_HARD_CURVATURE = 6, /* hard, c = index of the maximum curvature of the normalised log-eigenvalue
                            curve cut_scale * N * log10(l_n) / log10(l_1)  (method 1, Eq. 6,
                            PAPER.md:77-83; finite differences as in DESIGN.md "Readings")          */
    LCF_SOFT_CURVATURE = 7, /* sigmoid (Eq. 9) centred on the curvature-rule c                       */
    LCF_SOFT_ADAPTIVE = 8,  /* wt_i = win(i) / l_i^beta normalised to max 1, win = right half of a
                            Gaussian window (method 6, Eq. 10); no cut-off: c = 0;
                            the weights follow the small eigenvalues, so use precision = 1          */
    LCF_HARD_SLOPE = 9,     /* hard, method 2 as printed: slope of the eigenvalue curve
                            y(n) = l_n / l_1 (linear; relative to its first point so that the threshold
                            has no units: DESIGN.md "Readings" 18); c = (first n in 1..N-1 with
                            y(n) - y(n+1) < cut_scale) - 1: the steep leading components go            */
    LCF_SOFT_SLOPE = 10,    /* sigmoid (Eq. 9) centred on the slope-rule c                          */
    LCF_HARD_SLOPE_DB = 11, /* named variant of method 2: the same rule on y(n) = 10 log10(l_n), cut_scale
                            in dB per eigenvalue index (eigenvalues floored at 1e-12 l_1)           */
    LCF_SOFT_SLOPE_DB = 12, /* sigmoid (Eq. 9) centred on the dB-slope c                            */
    LCF_HARD_NCC = 13,      /* hard, method 4 (Eq. 8): c = argmin over k = 1..N-1 of the spatial
                            normalised cross-correlation of I_T(k) = sum_{i=k-4..k} |u_i| and I_B(k) =
                            sum_{i=k+1..k+5} |u_i| (clipped to 1..N), u_i = C_w v_i / sigma_i the left singular
                            vectors of the windowed data (fn = 5, w_i = 1; lowest k on ties;
                            DESIGN.md "Readings" 19).  Costs a third pass over the data                 */
    LCF_SOFT_NCC = 14,      /* sigmoid (Eq. 9) centred on the NCC c: methods 4 + 5 as the paper pairs them
                                                                                       */
    LCF_HARD_FIXED_TOP = 15,  /* the filter of LCF_HARD_FIXED, F = I - sum_{i<=k_fixed} v_i v_i^H, from the leading
                            eigenpairs only (block subspace iteration on M = 16 vectors, or 32 where the cut needs
                            them: DESIGN.md section 10, "partial EVD"; a departure from the paper's full-spectrum
                            EVD).  Getters: the first M eigenvalues / eigenvectors are Ritz pairs,
                            the other eigenvalues are reported as their mean (trace(R) - sum of the M) / (N - M),
                            the other eigenvectors as zero columns; lcf_get_sweeps counts rounds of the iteration.
                            Only the k_fixed (or c_k) leading pairs are iterated to the accuracy of the full EVD;
                            the Ritz values behind them are lower bounds of their eigenvalues, as converged as the
                            cut needed (typically within 1e-4 of the largest; with k_fixed = 0 nothing is iterated).
                            Runs for precision 0, 40 <= N <= 224, k_fixed <= 26; other plans in this mode compute
                            the same filter with the full EVD (lcf_get_work: evd_chol = 2 when it runs)   */
    LCF_HARD_ENERGY_TOP = 16  /* the same for LCF_HARD_ENERGY: c from the leading eigenvalues and trace(R_k).  A
                            window whose cut is not reached within 26 eigenvalues is reported like an
                            unconverged EVD (LCF_ERR_NOT_CONVERGED: use LCF_HARD_ENERGY)                  */
} lcf_thresh_mode;

typedef struct {
    lcf_thresh_mode mode;
    int k_fixed;        /* 0 <= k_fixed <= N (FIXED modes, FIXED_TOP)                           */
    double energy_frac; /* in (0, 1) (ENERGY modes, ENERGY_TOP)                                 */
    double beta;        /* > 0 (SOFT modes: sigmoid sharpness; ADAPTIVE: the exponent of Eq. 10)  */
    int precision;      /* 0: fp32-grade Gram, EVD and projection.  1: double precision throughout -- exact-product
                           fp64 Gram, fp64 EVD, fp64 projection (single precision can hamper the
                           EVD of long packets; "a double precision may be essential"); the image is still
                           returned as float.  "fp32-grade": on the tensor-core kernels
                           (even Nz) each fp32 operand, scaled by a power of two taken
                           from the ensemble's largest sample, is the sum of two fp16 numbers (22
                           significant bits) and products accumulate in fp32 (DESIGN.md section
                           6); the CUDA-core kernels that cover the other shapes use fp32.      */
    double cut_scale;   /* > 0 (MEDIAN, CURVATURE modes): the scaling factor beta of Eq. 7 / Eq. 6;
                           (SLOPE modes): the slope threshold per eigenvalue index, as a fraction of
                           l_1 (SLOPE) or in dB (SLOPE_DB)                                        */
} lcf_thresh;

/* the CUDA runtime's stream handle, so that this header stays plain C without cuda_runtime.h */
#ifndef __CUDA_RUNTIME_H__
#ifndef __DRIVER_TYPES_H__
typedef struct CUstream_st* cudaStream_t;
#endif
#endif

/* Builds window tables, the work decomposition and all device workspace on the current CUDA device.
 * Nz, Nx, N >= 1 (N >= 2).  *out is set to NULL on failure.  Synchronous (allocates, copies). */
lcf_status lcf_plan_create(lcf_plan** out, int Nz, int Nx, int N, const lcf_windows* win,
                           const lcf_thresh* thr);

/* Enqueues the whole path on `stream` (NULL = default stream) and returns without synchronising; no
 * allocation, no host<->device copy.  One call in flight per plan (the workspace is shared): use
 * one plan per stream to pipeline.  iq_dev and pd_dev must not alias.  Returns LCF_ERR_CUDA if a
 * launch failed.  Because it does not synchronise it cannot know whether the EVD of THIS call
 * converged: that is reported by lcf_get_converged, by every getter, and by the host entry points. */
lcf_status lcf_filter(lcf_plan* plan, const void* iq_dev, float* pd_dev, cudaStream_t stream);

/* Sliding-window form of lcf_filter (packets in a sliding temporal window).  The caller promises
 * that frames [0, N - stride) of this ensemble are frames [stride, N) of the ensemble of the previous
 * lcf_filter_stream call on this plan: the covariance entries of those frames are taken from the previous
 * call (shifted; rescaled by the exact power of two between the two data scales) and only the columns of the
 * `stride` new frames are computed.  The first call, a call after lcf_filter, and stride = 0 or N compute
 * everything.  Everything after the Gram is lcf_filter's.  Needs the tensor-core Gram path (precision 0,
 * 32 <= N <= 128, even Nz): LCF_ERR_UNSUPPORTED otherwise.  Workspace is allocated on first use.  Asynchronous. */
lcf_status lcf_filter_stream(lcf_plan* plan, const void* iq_dev, float* pd_dev, int stride, cudaStream_t stream);

/* `count` device-resident ensembles, pipelined on three lanes: two twins of the plan (same parameters, their own
 * workspace, created on first use -- they triple the plan's device memory) take the ensembles in turn on internal
 * streams, so the kernels of consecutive ensembles overlap (what the latency-bound EVD of one leaves idle, the
 * contractions of the next use).  iq_devs / pd_devs: HOST arrays of `count` DEVICE pointers; any three consecutive
 * ensembles are in flight together and need distinct pd buffers.  Asynchronous and stream-ordered like
 * lcf_filter: the lanes start after the work already enqueued on `stream`, and `stream` continues after all lanes
 * are done.  Results are bit-identical to `count` lcf_filter calls.  The getters afterwards describe the last
 * ensemble of lane 0 (index a multiple of 3); lcf_get_converged counts all lanes. */
lcf_status lcf_filter_batch(lcf_plan* plan, const void* const* iq_devs, float* const* pd_devs, int count, cudaStream_t stream);

/* Same path with HOST buffers (pinned or pageable): copies iq_host -> plan-owned device staging,
 * filters, copies the image back and synchronises `stream`.  The staging buffers are allocated on
 * first use (LCF_ERR_ALLOC on failure).  Returns LCF_ERR_NOT_CONVERGED (image written) if a
 * window's EVD hit the sweep cap. */
lcf_status lcf_filter_host(lcf_plan* plan, const void* iq_host, float* pd_host, cudaStream_t stream);

/* `count` ensembles from HOST buffers, pipelined: the host->device copy of ensemble i+1 (on a
 * plan-owned copy stream, three staging buffers) overlaps the kernels of ensembles i and i-1, which run on the
 * lanes of lcf_filter_batch; each image is copied back as soon as it is done.  `stream` is synchronised
 * at entry.  iq_hosts / pd_hosts: HOST arrays of `count` HOST
 * pointers (pinned memory for the copies to be asynchronous).  Returns after everything has
 * completed (synchronises both streams).  Results are identical to `count` lcf_filter_host calls.
 * Returns LCF_ERR_NOT_CONVERGED (all images written) if any window of any ensemble hit the sweep cap. */
lcf_status lcf_filter_host_batch(lcf_plan* plan, const void* const* iq_hosts, float* const* pd_hosts, int count, cudaStream_t stream);

/* Frees everything.  lcf_plan_destroy(NULL) is a no-op returning LCF_OK. */
lcf_status lcf_plan_destroy(lcf_plan* plan);

/* ---- diagnostics for the parity harness.  Each synchronises the plan's last stream, copies
 * device -> HOST and describes the most recent lcf_filter call.  They return
 * LCF_ERR_NOT_CONVERGED (after filling the output) if any window's EVD did not converge. ---- */
int lcf_num_windows(const lcf_plan* plan);                         /* K = Kz*Kx (0 if plan NULL) */
/* Synchronises the plan's last stream and reads one device counter: LCF_OK if every window's EVD
 * of every lcf_filter call since the last lcf_get_converged (or plan creation) converged, else
 * LCF_ERR_NOT_CONVERGED; *windows (HOST, may be NULL) = number of unconverged window EVDs. */
lcf_status lcf_get_converged(lcf_plan* plan, int* windows);
/* Caps the Jacobi sweeps of the following lcf_filter calls (0 = the kernels' defaults: 30 in the
 * fp32 kernels, 40 in fp64).  For latency-bounded use and for testing the non-convergence report. */
lcf_status lcf_set_max_sweeps(lcf_plan* plan, int max_sweeps);
lcf_status lcf_get_eigenvalues(lcf_plan* plan, double* lam /* HOST [K][N], descending */);
lcf_status lcf_get_cutoffs(lcf_plan* plan, int* c /* HOST [K]: rejected components per window */);
lcf_status lcf_get_sweeps(lcf_plan* plan, int* sweeps /* HOST [K]: Jacobi sweeps used */);
lcf_status lcf_get_gram(lcf_plan* plan, double* R /* HOST [K][N][N][2], R[i][j] as in Eq. 12 */);
/* V[a][i] = component a of the eigenvector of the i-th largest eigenvalue */
lcf_status lcf_get_eigenvectors(lcf_plan* plan, double* V /* HOST [K][N][N][2] */);
/* NCC modes only (LCF_ERR_INVALID_ARG otherwise): ncc[k-1] = NCC(k) of Eq. 8 for k = 1..N-1, ncc[N-1] = +inf */
lcf_status lcf_get_ncc(lcf_plan* plan, double* ncc /* HOST [K][N] */);
/* wt[i] = weight of the i-th largest eigenvalue (0-based storage of the paper's 1-based i) */
lcf_status lcf_get_weights(lcf_plan* plan, double* wt /* HOST [K][N] */);
/* F_k = V diag(wt) V^H (Eq. 4), built on the device from V and wt */
lcf_status lcf_get_filters(lcf_plan* plan, double* F /* HOST [K][N][N][2] */);
/* m_k = mean over the full field of view of PD_k (Eq. 13's 1/alpha_k) */
lcf_status lcf_get_window_means(lcf_plan* plan, double* m /* HOST [K] */);

/* ---- measurement helpers ---- */
/* Mean device time in ms of each stage -- [gram, evd, weights_projector, projection, combine] --
 * over the lcf_filter calls made since timing was last enabled (at most the last 64).  With timing
 * enabled lcf_filter records CUDA events on the caller's stream between its launches; it still
 * does not synchronise.  lcf_get_stage_ms synchronises the stream. */
lcf_status lcf_set_timing(lcf_plan* plan, int enabled);
lcf_status lcf_get_stage_ms(lcf_plan* plan, float ms[5] /* HOST */);
/* Algorithmic work of one lcf_filter call: Hermitian-half Gram flops,
 * projection flops, compulsory HBM bytes, sum_k P_k, kernel launches per call; which kernels the
 * plan selected (1 = tcgen05 Gram / Cholesky + one-sided Jacobi EVD / tcgen05 projection, 0 = the
 * FP32/FP64 CUDA-core kernels) and, for the tensor-core kernels, the flops the MMAs execute
 * (three fp16 products of hi/lo splits per fp32 product, padded tiles) -- the algorithmic flops are what the rooflines are quoted on. */
typedef struct {
    double gram_flops, proj_flops, hbm_bytes, sum_Pk;
    int launches;
    int gram_tc, evd_chol, proj_tc;   /* kernels chosen: evd_chol 0 two-sided Jacobi, 1 Cholesky + one-sided Jacobi, 2 leading eigenpairs (the *_TOP modes) */
    double gram_tensor_flops, proj_tensor_flops;
} lcf_work;
lcf_status lcf_get_work(const lcf_plan* plan, lcf_work* out /* HOST */);
/* Arithmetic-pipe microbenchmark on the current device: kind 0 = FP32 FFMA, 1 = FP32 packed
 * FFMA2 (fma.rn.f32x2), 2 = FP64 DFMA, 3 = tcgen05.mma.kind::f16 (128 x 256 x 16, operands resident
 * in shared memory, fp32 accumulate in tensor memory).  Writes achieved TFLOP/s (2 flops per FMA). */
lcf_status lcf_measure_peak(int kind, double* tflops /* HOST */);
/* Host logic of the tensor-core path's power-of-two operand scaling: the
 * exponent k with amax * 2^k in [256, 512) for a finite amax > 0 (clamped to [-100, 100]); 0 for
 * amax = 0, denormal, infinite or NaN.  Host function, no device work. */
int lcf_scale_exponent(float amax);

const char* lcf_status_string(lcf_status s);
/* After LCF_ERR_CUDA from lcf_filter: "<stage>: <CUDA error string>" of the first failed launch
 * (stages: gram, evd, weights/projector, projection, combine); "" if none.  HOST string owned by
 * the plan.  Launch failures are sticky; asynchronous execution faults surface at the next call
 * that synchronises (run with CUDA_LAUNCH_BLOCKING=1 to attribute them to a stage). */
const char* lcf_last_error(const lcf_plan* plan);

#ifdef __cplusplus
}
#endif
#endif /* LCF_H_ */
