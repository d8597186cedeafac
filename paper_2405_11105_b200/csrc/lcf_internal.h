// lcf_internal.h -- plan layout and kernel launchers shared by the liblcf.so translation units.
// Product code: shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <cstddef>
#include <cstdint>
#include <vector>

#include "../../include/lcf.h"

namespace lcf {

// ---- window geometry (Eq. 11; truncation/centres: DESIGN.md "Readings") ----
struct WinBox {      // support box of window k = kx*Kz + kz, and where its PD tile lives
    int z0, Lz;      // axial support [z0, z0+Lz)
    int x0, Lx;      // lateral support [x0, x0+Lx)
    int kz, kx;
    int Pk;          // Lz*Lx
    int pad_;
    long long tile_off;  // offset (floats) of this window's PD_k tile [Lx][Lz] in the tile buffer
};

// One Gram CTA: window k, flattened box pixels q in [q0, q1) (q = (x-x0)*Lz + (z-z0)), tile batch.
struct GramItem {
    int k, q0, q1, batch, pslot;
};
// One projection CTA: window k, box pixels [q0, q1) with q1-q0 <= PROJ_TPIX.
struct ProjItem {
    int k, q0, q1;
};
// One segment of the tensor-core Gram: `ntile` consecutive 16-pixel tiles of window k from tile0.
struct GtcSeg {
    int k, tile0, ntile, pad_;
};
// One segment of the tensor-core projection: `ntile` consecutive 64-pixel tiles of window k,
// eigen-column block b.
struct PtcSeg {
    int k, b, tile0, ntile;
};

// Block-form tensor-core Gram (128 < N <= 256, lcf_gram_tc2.cu): a block of R_k (rows m0.., nc columns from c0,
// frames f0 .. f0 + nbox loaded) and a segment of one (window, block) job.
struct G2Block {
    int m0, c0, nc, f0, nbox;
};
struct G2Seg {
    int k, blk, tile0, ntile, cta;
};

constexpr int GRAM_TP = 32;        // pixels per shared-memory tile of the Gram kernel
constexpr int GRAM_FLUSH_TILES = 16; // fp32 accumulators are folded into the fp64 partial every 16 tiles (512 px)
constexpr int GRAM_THREADS = 160;  // max thread tiles per Gram CTA (136 upper tiles at N=128)
constexpr int PROJ_TPIX = 64;      // pixels per projection CTA
constexpr int PROJ_KT = 16;        // frames per pipeline stage of the projection kernel
constexpr int PROJ_STAGES = 3;
constexpr int VB_WARPS = 8;        // warps per CTA of the weights/projector kernel
constexpr int VB_ROWS = 2;         // rows of V per warp

// CUtensorMaps of the IQ pointers a plan has seen (a streaming caller cycles through a few fixed
// offsets into one resident sequence): encoded once per pointer, round-robin replacement.
struct TmapCache {
    static constexpr int CAP = 32;
    const void* key[CAP] = {};
    alignas(64) unsigned char map[CAP][128];
    int n = 0, next = 0;
    const unsigned char* find(const void* iq) const {
        for (int i = 0; i < n; ++i)
            if (key[i] == iq) return map[i];
        return nullptr;
    }
    unsigned char* slot(const void* iq) {       // where to encode the map of a new pointer
        const int i = n < CAP ? n++ : (next = (next + 1) % CAP);
        key[i] = iq;
        return map[i];
    }
    void drop_last(const void* iq) {            // encoding failed: forget the key
        for (int i = 0; i < n; ++i)
            if (key[i] == iq) key[i] = nullptr;
    }
};

struct TmapCache3 {                             // same, three maps per pointer
    static constexpr int CAP = 16;
    const void* key[CAP] = {};
    alignas(64) unsigned char map[CAP][384];
    int n = 0, next = 0;
    const unsigned char* find(const void* iq) const {
        for (int i = 0; i < n; ++i)
            if (key[i] == iq) return map[i];
        return nullptr;
    }
    unsigned char* slot(const void* iq) {
        const int i = n < CAP ? n++ : (next = (next + 1) % CAP);
        key[i] = iq;
        return map[i];
    }
    void drop_last(const void* iq) {
        for (int i = 0; i < n; ++i)
            if (key[i] == iq) key[i] = nullptr;
    }
};

constexpr int TIMER_RING = 64;     // lcf_filter calls whose stage events are kept
struct StageTimer {
    cudaEvent_t ev[TIMER_RING][6];
    bool have = false;
    long long calls = 0;           // calls recorded since timing was (re)enabled
};

}  // namespace lcf

struct lcf_plan {
    int Nz = 0, Nx = 0, N = 0, Kz = 0, Kx = 0, K = 0;
    long long P = 0;
    lcf_windows win{};
    lcf_thresh thr{};
    int prec = 0;            // 0 fp32, 1 fp64 (Gram, Jacobi, V)
    int NP = 0, Ns = 0;      // rotation pairs per Jacobi step, slots (= 2*NP >= N)
    int max_sweeps = 0;
    int sweep_cap = 0;       // lcf_set_max_sweeps: 0 = each EVD kernel's default
    size_t esz = 4;          // sizeof(real) of the Gram/EVD precision

    // host copies
    std::vector<double> gz_h, gx_h;      // [Kz][Nz], [Kx][Nx]
    std::vector<lcf::WinBox> box_h;      // [K]
    std::vector<int> pfirst_h;           // [K+1] first projection item of window k
    std::vector<int> gfirst_h;           // [K+1] first Gram partial slot of window k
    long long sumPk = 0;

    // device: tables
    double *gz_d = nullptr, *gx_d = nullptr;
    lcf::WinBox* box_d = nullptr;
    int *kzlo_d = nullptr, *kzhi_d = nullptr, *kxlo_d = nullptr, *kxhi_d = nullptr;  // per pixel coord
    // Gram
    lcf::GramItem* gitems_d = nullptr;
    int n_gitems = 0, n_gslots = 0, gram_Tn = 0, gram_TM = 0, gram_tiles_per_batch = 0, gram_batches = 0;
    int* gfirst_d = nullptr;
    double2* gpart_d = nullptr; // [n_gslots][N][N] complex double (canonical half written)
    void* R_d = nullptr;       // [K][N][N] complex real (full Hermitian)
    // tensor-core Gram (precision 0, N <= 128): lcf_gram_tc.cu
    bool gram_tc = false;
    int gtc_grid = 0, gtc_nseg = 0, gtc_group = 8;
    uint32_t gtc_raw_stride = 0;
    size_t gtc_smem = 0;
    lcf::GtcSeg* gtc_segs_d = nullptr;
    int *gtc_cta_first_d = nullptr, *gtc_seg_first_d = nullptr;
    float* gtc_part_d = nullptr;            // [nseg][4][128][128]
    lcf::TmapCache gtc_tmaps;
    // block-form tensor-core Gram (precision 0, 128 < N <= 256): lcf_gram_tc2.cu
    bool gram_tc2 = false;
    int g2_grid = 0, g2_nseg = 0, g2_c1 = 0;
    uint32_t g2_raw_stride = 0, g2_mat_bytes = 0;
    size_t g2_smem = 0;
    lcf::G2Block g2_blk[3] = {};
    lcf::G2Seg* g2_segs_d = nullptr;
    int *g2_cta_first_d = nullptr, *g2_seg_first_d = nullptr;
    float* g2_part_d = nullptr;             // [nseg][2][128][128]
    lcf::TmapCache3 g2_tmaps;
    // sliding-window reuse (lcf_filter_stream, N <= 128): the block-form kernel computes the new frames' columns only
    bool strm_ready = false, strm_valid = false;
    float2* Rprev_d = nullptr;              // [K][N][N] R of the previous lcf_filter_stream call (data scale of that call)
    uint32_t* amax_prev_d = nullptr;
    // Cholesky + one-sided Jacobi EVD (precision 0, N <= 128): lcf_evd_chol.cu
    bool evd_chol = false, evd_cluster = false;   // cluster: Cholesky kernel, then one-sided Jacobi on 2-CTA clusters
    int ec_LD = 0;
    size_t ec_smem = 0, ecl_smem = 0;
    bool evd_top = false;                         // LCF_HARD_*_TOP: block subspace iteration instead of a full EVD (lcf_evd_top.cu)
    size_t et_smem = 0, et_smem_small = 0;
    float* ec_gfac_d = nullptr;             // [K][2][Ns][LD] Cholesky factor planes
    float* ec_shift_d = nullptr;            // [K]
    int* ec_nexp_d = nullptr;               // [K]
    // tensor-core projection (N <= 128): lcf_project_tc.cu
    bool proj_tc = false;
    int ptc_grid = 0, ptc_nseg = 0, ptc_NB = 0, ptc_Kp = 0, ptc_nstg = 0, ptc_G = 1;
    size_t ptc_smem = 0;
    lcf::PtcSeg* ptc_segs_d = nullptr;
    int* ptc_cta_first_d = nullptr;
    float* ptc_bpack_d = nullptr;           // [K][NB][Kp/4][256][4]
    float* ptc_part_d = nullptr;            // [NB][sum_k P_k]
    bool ptc_pre = false, ptc_premaps_ready = false;   // pre-split fp16 planes of the ensemble (lcf_project_tc.cu, PRE variant)
    void *ptc_sh_d = nullptr, *ptc_sl_d = nullptr;     // [Kp/8][Nx][Nz][2][8] fp16 hi / lo
    alignas(64) unsigned char ptc_premaps[256];
    uint32_t* amax_d = nullptr;             // bits of max |re|, |im| over the ensemble (tensor-core paths scale by a power of two)
    // EVD
    void* rotlog_d = nullptr;  // [K][max_sweeps*(Ns-1)][3][NP] real
    double* lam_d = nullptr;   // [K][N] descending
    int* order_d = nullptr;    // [K][N] slot of the i-th largest eigenvalue
    int* cut_d = nullptr;      // [K]
    int* sweeps_d = nullptr;   // [K]
    int* conv_d = nullptr;     // [K] 1 = converged
    int* nunconv_d = nullptr;  // [1] window EVDs that hit the sweep cap since the counter was last read
    float* wslot_d = nullptr;  // [K][Ns] weight of the eigenvector sitting in slot s
    double* wslot_dd_d = nullptr;  // [K][Ns] same, double (diagnostic filter build)
    double* wt_d = nullptr;    // [K][N] weight by rank
    void* V_d = nullptr;       // [K][N][Ns] complex real, slot order
    float2* B_d = nullptr;     // [K][N][Ns] complex float: V diag(wslot)
    // method 4 (spatial NCC cut-off, lcf_ncc.cu): allocated for the NCC modes only
    float* ncc_mag_d = nullptr;        // [sum_k P_k][ncc_magN]  |u_i(p)| by rank
    int ncc_magN = 0;
    float* ncc_isig_d = nullptr;       // [K][ncc_magN]
    float* ncc_part_d = nullptr;       // [K][32 chunks][3][N]
    double* ncc_curve_d = nullptr;     // [K][N]  NCC(k), k = 1..N (last = +inf)
    // projection / combine
    lcf::ProjItem* pitems_d = nullptr;
    int n_pitems = 0;
    int* pfirst_d = nullptr;
    float* tiles_d = nullptr;  // [sumPk]
    float* tsum_d = nullptr;   // [n_pitems]
    double* mean_d = nullptr;  // [K]
    float* alpha_d = nullptr;  // [K]
    double* F_d = nullptr;     // [K][N][N][2] (diagnostic, allocated on demand)
    // host staging for lcf_filter_host
    void* iq_stage_d = nullptr;
    float* pd_stage_d = nullptr;
    // second staging set, copy stream and events of lcf_filter_host_batch
    void *iq_stage2_d = nullptr, *iq_stage3_d = nullptr;
    float *pd_stage2_d = nullptr, *pd_stage3_d = nullptr;
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t ev_copied[3] = {nullptr, nullptr, nullptr}, ev_done[3] = {nullptr, nullptr, nullptr};

    // lane pipelining of lcf_filter_batch (three lanes) / lcf_filter_host_batch (two): twin plans (same parameters,
    // their own workspace) and one internal stream per lane, created on first use
    lcf_plan* twin = nullptr;               // chain: plan -> twin -> twin's twin (lane 0, 1, 2)
    cudaStream_t lane_st[3] = {nullptr, nullptr, nullptr};
    cudaEvent_t ev_fork = nullptr, ev_join[3] = {nullptr, nullptr, nullptr};

    cudaStream_t last_stream = nullptr;
    bool ran = false;
    bool cuda_failed = false;
    char last_error[160] = "";   // stage and CUDA error string of the first failed launch
    bool timing = false;
    lcf::StageTimer timer;
    int smem_optin = 0;
    int num_sms = 0;
    // launch geometry decided at create
    int jac_threads = 0, jac_bpt = 0;
    size_t jac_smem = 0, gram_smem = 0, proj_smem = 0;
    int proj_threads = 0, proj_nct = 0;
};

namespace lcf {
// The dynamic shared-memory limit of a kernel is a per-function, process-wide attribute: every
// kernel gets the device's opt-in maximum (minus its static shared memory) once, so plans of
// different sizes that are alive at the same time cannot lower each other's limit.
template <class F>
inline cudaError_t set_max_dyn_smem(F* fn, int optin) {
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, reinterpret_cast<const void*>(fn));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(reinterpret_cast<const void*>(fn), cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes);
}
// each returns the cudaError_t of configuring/launching; kernels are asynchronous on `st`
cudaError_t launch_gram(lcf_plan* p, const float2* iq, cudaStream_t st);
cudaError_t launch_jacobi(lcf_plan* p, cudaStream_t st);
cudaError_t launch_vbuild(lcf_plan* p, cudaStream_t st);
cudaError_t launch_project(lcf_plan* p, const float2* iq, cudaStream_t st);
cudaError_t launch_combine(lcf_plan* p, float* pd, cudaStream_t st);
cudaError_t launch_build_filters(lcf_plan* p, cudaStream_t st);
cudaError_t launch_project_dd(lcf_plan* p, const float2* iq, cudaStream_t st);
cudaError_t configure_gram(lcf_plan* p);     // each: opt-in shared memory size, launch geometry
cudaError_t configure_evd(lcf_plan* p);
cudaError_t configure_project(lcf_plan* p);
bool gram_tc_eligible(const lcf_plan* p);
cudaError_t configure_gram_tc(lcf_plan* p, std::vector<GtcSeg>& segs, std::vector<int>& cta_first, std::vector<int>& seg_first);
cudaError_t launch_gram_tc(lcf_plan* p, const float2* iq, cudaStream_t st);
bool gram_tc2_eligible(const lcf_plan* p);
cudaError_t configure_gram_tc2(lcf_plan* p, std::vector<G2Seg>& segs, std::vector<int>& cta_first, std::vector<int>& seg_first);
cudaError_t launch_gram_tc2(lcf_plan* p, const float2* iq, cudaStream_t st);
bool gram_stream_eligible(const lcf_plan* p);
cudaError_t configure_gram_stream(lcf_plan* p, std::vector<G2Seg>& segs, std::vector<int>& cta_first, std::vector<int>& seg_first);
cudaError_t launch_gram_stream(lcf_plan* p, const float2* iq, int stride, cudaStream_t st);
bool evd_chol_eligible(const lcf_plan* p);
cudaError_t configure_evd_chol(lcf_plan* p);
cudaError_t launch_evd_chol(lcf_plan* p, cudaStream_t st, bool chol_only);
bool evd_top_mode(int mode);
bool evd_top_eligible(const lcf_plan* p);
cudaError_t configure_evd_top(lcf_plan* p);
cudaError_t launch_evd_top(lcf_plan* p, cudaStream_t st);
constexpr int ECL8_MAXN = 208;                // most frames of the 8-CTA cluster EVD (13 column pairs per CTA)
bool evd_cluster_eligible(const lcf_plan* p);
cudaError_t configure_evd_cluster(lcf_plan* p);
cudaError_t launch_evd_cluster(lcf_plan* p, cudaStream_t st);
bool project_tc_eligible(const lcf_plan* p);
cudaError_t configure_project_tc(lcf_plan* p, std::vector<PtcSeg>& segs, std::vector<int>& cta_first);
cudaError_t launch_project_tc(lcf_plan* p, const float2* iq, cudaStream_t st);
cudaError_t launch_absmax(lcf_plan* p, const float2* iq, cudaStream_t st);
cudaError_t launch_presplit(lcf_plan* p, const float2* iq, cudaStream_t st);
bool ncc_mode(int mode);
cudaError_t launch_ncc(lcf_plan* p, const float2* iq, cudaStream_t st);
// what the EVD kernels are told: under the NCC modes they run with every eigen-weight 1 (hard cut at 0), so that
// B_k = V_k for the left singular vectors; lcf_ncc.cu then sets the cut-off, the weights and B_k
inline int evd_mode(const lcf_plan* p) {   // the rule the full-spectrum EVD kernels apply
    if (p->thr.mode == LCF_HARD_NCC || p->thr.mode == LCF_SOFT_NCC || p->thr.mode == LCF_HARD_FIXED_TOP) return (int)LCF_HARD_FIXED;
    if (p->thr.mode == LCF_HARD_ENERGY_TOP) return (int)LCF_HARD_ENERGY;
    return (int)p->thr.mode;
}
inline int evd_kfixed(const lcf_plan* p) { return (p->thr.mode == LCF_HARD_NCC || p->thr.mode == LCF_SOFT_NCC) ? 0 : p->thr.k_fixed; }
}  // namespace lcf
