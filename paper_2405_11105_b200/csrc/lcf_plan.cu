// lcf_plan.cu -- the C ABI of liblcf.so (include/lcf.h): plan construction (window tables of
// Eq. 11, work decomposition, workspace), lcf_filter (enqueues the kernels of
// steps a1..a5), diagnostics getters.  Host code only builds tables and moves bytes; every step of
// the path runs in the kernels of lcf_gram.cu / lcf_evd.cu / lcf_project.cu.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "lcf_internal.h"
#include "lcf_sm100.cuh"
#include "lcf_thresh.cuh"

using namespace lcf;

namespace {

template <typename T>
bool dev_alloc(T** p, size_t count) {
    *p = nullptr;
    if (count == 0) count = 1;
    return cudaMalloc(reinterpret_cast<void**>(p), count * sizeof(T)) == cudaSuccess;
}
template <typename T>
bool dev_upload(T** p, const std::vector<T>& h) {
    if (!dev_alloc(p, h.size())) return false;
    if (h.empty()) return true;
    return cudaMemcpy(*p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice) == cudaSuccess;
}

// One axis of the window grid (Eq. 11; centres at cell centres, inclusive box truncation).
void axis_windows(int n, int K, double sigma, double trunc, std::vector<double>& g, std::vector<int>& lo,
                  std::vector<int>& hi) {
    g.assign((size_t)K * n, 0.0);
    lo.assign(K, 0);
    hi.assign(K, -1);
    for (int k = 0; k < K; ++k) {
        const double c = (k + 0.5) * (double)n / (double)K - 0.5;
        int l = n, h = -1;
        for (int i = 0; i < n; ++i) {
            double v;
            if (sigma <= 0.0) v = 1.0;
            else {
                const double d = (double)i - c;
                if (trunc > 0.0 && std::fabs(d) > trunc * sigma) v = 0.0;
                else v = std::exp(-(d * d) / (2.0 * sigma * sigma));
            }
            g[(size_t)k * n + i] = v;
            if (v != 0.0) { if (i < l) l = i; if (i > h) h = i; }
        }
        // a Gaussian that underflows to 0 inside its box leaves holes; the box [l, h] still covers it
        lo[k] = l; hi[k] = h;
    }
}

void free_plan_device(lcf_plan* p) {
    cudaFree(p->gz_d); cudaFree(p->gx_d); cudaFree(p->box_d);
    cudaFree(p->kzlo_d); cudaFree(p->kzhi_d); cudaFree(p->kxlo_d); cudaFree(p->kxhi_d);
    cudaFree(p->gitems_d); cudaFree(p->gfirst_d); cudaFree(p->gpart_d); cudaFree(p->R_d);
    cudaFree(p->rotlog_d); cudaFree(p->lam_d); cudaFree(p->order_d); cudaFree(p->cut_d);
    cudaFree(p->sweeps_d); cudaFree(p->conv_d); cudaFree(p->nunconv_d); cudaFree(p->wslot_d); cudaFree(p->wslot_dd_d); cudaFree(p->wt_d);
    cudaFree(p->V_d); cudaFree(p->B_d); cudaFree(p->pitems_d); cudaFree(p->pfirst_d);
    cudaFree(p->tiles_d); cudaFree(p->tsum_d); cudaFree(p->mean_d); cudaFree(p->alpha_d);
    cudaFree(p->F_d); cudaFree(p->iq_stage_d); cudaFree(p->pd_stage_d);
    cudaFree(p->iq_stage2_d); cudaFree(p->pd_stage2_d); cudaFree(p->iq_stage3_d); cudaFree(p->pd_stage3_d);
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    for (int i = 0; i < 3; ++i) { if (p->lane_st[i]) cudaStreamDestroy(p->lane_st[i]); if (p->ev_join[i]) cudaEventDestroy(p->ev_join[i]); }
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    for (int i = 0; i < 3; ++i) { if (p->ev_copied[i]) cudaEventDestroy(p->ev_copied[i]); if (p->ev_done[i]) cudaEventDestroy(p->ev_done[i]); }
    cudaFree(p->ec_gfac_d); cudaFree(p->ec_shift_d); cudaFree(p->ec_nexp_d);
    cudaFree(p->ptc_segs_d); cudaFree(p->ptc_cta_first_d); cudaFree(p->ptc_bpack_d); cudaFree(p->ptc_part_d); cudaFree(p->amax_d);
    cudaFree(p->gtc_segs_d); cudaFree(p->gtc_cta_first_d); cudaFree(p->gtc_seg_first_d); cudaFree(p->gtc_part_d);
    cudaFree(p->ptc_sh_d); cudaFree(p->ptc_sl_d); cudaFree(p->Rprev_d); cudaFree(p->amax_prev_d);
    cudaFree(p->ncc_mag_d); cudaFree(p->ncc_isig_d); cudaFree(p->ncc_part_d); cudaFree(p->ncc_curve_d);
    cudaFree(p->g2_segs_d); cudaFree(p->g2_cta_first_d); cudaFree(p->g2_seg_first_d); cudaFree(p->g2_part_d);
    if (p->timer.have)
        for (auto& set : p->timer.ev)
            for (auto& e : set) cudaEventDestroy(e);
}

lcf_status sync_plan(lcf_plan* p) {
    if (!p) return LCF_ERR_INVALID_ARG;
    if (!p->ran) return LCF_ERR_INVALID_ARG;
    if (cudaStreamSynchronize(p->last_stream) != cudaSuccess) { p->cuda_failed = true; return LCF_ERR_CUDA; }
    return LCF_OK;
}

lcf_status conv_status(lcf_plan* p) {
    std::vector<int> cv(p->K);
    if (cudaMemcpy(cv.data(), p->conv_d, sizeof(int) * p->K, cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
    for (int v : cv)
        if (!v) return LCF_ERR_NOT_CONVERGED;
    return LCF_OK;
}

// reads and clears the count of window EVDs that hit the sweep cap (the caller has synchronised)
lcf_status take_unconverged(lcf_plan* p, int* count) {
    int n = 0;
    for (lcf_plan* q = p; q; q = q->twin) {
        int m = 0;
        if (q != p && q->ran && cudaStreamSynchronize(q->last_stream) != cudaSuccess) return LCF_ERR_CUDA;
        if (cudaMemcpy(&m, q->nunconv_d, sizeof(int), cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
        if (m != 0 && cudaMemset(q->nunconv_d, 0, sizeof(int)) != cudaSuccess) return LCF_ERR_CUDA;
        n += m;
    }
    if (count) *count = n;
    return n ? LCF_ERR_NOT_CONVERGED : LCF_OK;
}

// twin plan, lane streams and events of the two-lane batch entry points (first use)
constexpr int LCF_LANES = 3;     // measured at config 2: 626 / 769 / 798 / 802 ensembles/s with 1 / 2 / 3 / 4 lanes

lcf_status ensure_lanes(lcf_plan* p, int lanes) {
    lcf_plan* q = p;
    for (int l = 1; l < lanes; ++l) {
        if (!q->twin) {
            lcf_status s = lcf_plan_create(&q->twin, p->Nz, p->Nx, p->N, &p->win, &p->thr);
            if (s != LCF_OK) { q->twin = nullptr; return s; }
        }
        q = q->twin;
        q->sweep_cap = p->sweep_cap;
    }
    for (int i = 0; i < lanes; ++i) {
        if (!p->lane_st[i] && cudaStreamCreateWithFlags(&p->lane_st[i], cudaStreamNonBlocking) != cudaSuccess) return LCF_ERR_CUDA;
        if (!p->ev_join[i] && cudaEventCreateWithFlags(&p->ev_join[i], cudaEventDisableTiming) != cudaSuccess) return LCF_ERR_CUDA;
    }
    if (!p->ev_fork && cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming) != cudaSuccess) return LCF_ERR_CUDA;
    return LCF_OK;
}

lcf_plan* lane_plan(lcf_plan* p, int lane) {
    for (int l = 0; l < lane; ++l) p = p->twin;
    return p;
}

}  // namespace

extern "C" const char* lcf_status_string(lcf_status s) {
    switch (s) {
        case LCF_OK: return "ok";
        case LCF_ERR_INVALID_ARG: return "invalid argument";
        case LCF_ERR_UNSUPPORTED: return "unsupported size or configuration (plan: the EVD matrix does not fit shared memory; other calls: lcf_last_error)";
        case LCF_ERR_ALLOC: return "allocation failed";
        case LCF_ERR_CUDA: return "CUDA error";
        case LCF_ERR_NOT_CONVERGED: return "EVD did not converge";
    }
    return "unknown status";
}

extern "C" lcf_status lcf_plan_create(lcf_plan** out, int Nz, int Nx, int N, const lcf_windows* win,
                                      const lcf_thresh* thr) {
    if (!out) return LCF_ERR_INVALID_ARG;
    *out = nullptr;
    if (!win || !thr) return LCF_ERR_INVALID_ARG;
    if (Nz < 1 || Nx < 1 || N < 2 || win->Kz < 1 || win->Kx < 1) return LCF_ERR_INVALID_ARG;
    if ((long long)Nz * Nx > (1LL << 30) || (long long)win->Kz * win->Kx > 65535) return LCF_ERR_INVALID_ARG;
    if ((int)thr->mode < 0 || (int)thr->mode > 16 || (thr->precision != 0 && thr->precision != 1)) return LCF_ERR_INVALID_ARG;
    const bool fixed = thr->mode == LCF_HARD_FIXED || thr->mode == LCF_SOFT_FIXED || thr->mode == LCF_HARD_FIXED_TOP;
    const bool soft = thresh_is_soft(thr->mode);
    if (fixed && (thr->k_fixed < 0 || thr->k_fixed > N)) return LCF_ERR_INVALID_ARG;
    const bool energy = thr->mode == LCF_HARD_ENERGY || thr->mode == LCF_SOFT_ENERGY || thr->mode == LCF_HARD_ENERGY_TOP;
    const bool median = thr->mode == LCF_HARD_MEDIAN || thr->mode == LCF_SOFT_MEDIAN ||
                        thr->mode == LCF_HARD_CURVATURE || thr->mode == LCF_SOFT_CURVATURE ||
                        thr->mode == LCF_HARD_SLOPE || thr->mode == LCF_SOFT_SLOPE ||
                        thr->mode == LCF_HARD_SLOPE_DB || thr->mode == LCF_SOFT_SLOPE_DB;     // modes that read cut_scale
    if (energy && !(thr->energy_frac > 0.0 && thr->energy_frac < 1.0)) return LCF_ERR_INVALID_ARG;
    if (median && !(thr->cut_scale > 0.0) ) return LCF_ERR_INVALID_ARG;
    if (soft && !(thr->beta > 0.0)) return LCF_ERR_INVALID_ARG;
    if (!std::isfinite(win->sigma_z) || !std::isfinite(win->sigma_x) || !std::isfinite(win->trunc_sigmas))
        return LCF_ERR_INVALID_ARG;

    lcf_plan* p = new (std::nothrow) lcf_plan();
    if (!p) return LCF_ERR_ALLOC;
    p->Nz = Nz; p->Nx = Nx; p->N = N; p->Kz = win->Kz; p->Kx = win->Kx; p->K = win->Kz * win->Kx;
    p->P = (long long)Nz * Nx;
    p->win = *win; p->thr = *thr; p->prec = thr->precision;
    p->esz = p->prec ? 8 : 4;
    p->NP = (N + 1) / 2; p->Ns = 2 * p->NP;
    p->max_sweeps = p->prec ? 40 : 24;

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&p->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess ||
        cudaDeviceGetAttribute(&p->num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
        delete p;
        return LCF_ERR_CUDA;
    }

    // ---- windows ----
    std::vector<int> zlo, zhi, xlo, xhi;
    axis_windows(Nz, p->Kz, (double)win->sigma_z, (double)win->trunc_sigmas, p->gz_h, zlo, zhi);
    axis_windows(Nx, p->Kx, (double)win->sigma_x, (double)win->trunc_sigmas, p->gx_h, xlo, xhi);
    p->box_h.resize(p->K);
    long long off = 0;
    for (int kx = 0; kx < p->Kx; ++kx)
        for (int kz = 0; kz < p->Kz; ++kz) {
            WinBox& b = p->box_h[kx * p->Kz + kz];
            b.kz = kz; b.kx = kx; b.pad_ = 0;
            b.z0 = zlo[kz]; b.Lz = zhi[kz] >= zlo[kz] ? zhi[kz] - zlo[kz] + 1 : 0;
            b.x0 = xlo[kx]; b.Lx = xhi[kx] >= xlo[kx] ? xhi[kx] - xlo[kx] + 1 : 0;
            if (b.Lz == 0 || b.Lx == 0) { b.Lz = 0; b.Lx = 0; b.z0 = 0; b.x0 = 0; }
            b.Pk = b.Lz * b.Lx;
            b.tile_off = off;
            off += b.Pk;
        }
    p->sumPk = off;
    // windows covering each pixel coordinate (supports are intervals with monotone ends)
    auto cover = [](int n, int K, const std::vector<int>& lo, const std::vector<int>& hi, std::vector<int>& klo,
                    std::vector<int>& khi) {
        klo.assign(n, 0); khi.assign(n, -1);
        for (int i = 0; i < n; ++i) {
            int a = K, b = -1;
            for (int k = 0; k < K; ++k)
                if (hi[k] >= lo[k] && i >= lo[k] && i <= hi[k]) { if (k < a) a = k; if (k > b) b = k; }
            klo[i] = a; khi[i] = b;
        }
    };
    std::vector<int> kzlo, kzhi, kxlo, kxhi;
    cover(Nz, p->Kz, zlo, zhi, kzlo, kzhi);
    cover(Nx, p->Kx, xlo, xhi, kxlo, kxhi);

    // ---- kernel geometry ----
    if (configure_gram(p) != cudaSuccess || configure_evd(p) != cudaSuccess || configure_project(p) != cudaSuccess ||
        p->NP > 128) {
        cudaGetLastError();
        delete p;
        return LCF_ERR_UNSUPPORTED;
    }

    // ---- tensor-core Gram decomposition (precision 0, N <= 128, even Nz) ----
    std::vector<GtcSeg> gtc_segs;
    std::vector<int> gtc_cta_first, gtc_seg_first;
    p->gram_tc = gram_tc_eligible(p);
    if (p->gram_tc && configure_gram_tc(p, gtc_segs, gtc_cta_first, gtc_seg_first) != cudaSuccess) {
        cudaGetLastError();
        p->gram_tc = false;
    }
    p->evd_chol = evd_chol_eligible(p);
    if (p->evd_chol && configure_evd_chol(p) != cudaSuccess) {
        cudaGetLastError();
        p->evd_chol = false;
    }
    p->evd_top = evd_top_eligible(p);
    if (p->evd_top && configure_evd_top(p) != cudaSuccess) {
        cudaGetLastError();
        p->evd_top = false;
    }
    if (!p->evd_chol && !p->evd_top) p->gram_tc = false;   // the tensor-core Gram leaves R in its data scale, which only these EVD kernels undo
    std::vector<G2Seg> g2_segs;
    std::vector<int> g2_cta_first, g2_seg_first;
    p->gram_tc2 = gram_tc2_eligible(p);     // block form above 128 frames; its reduction undoes the data scale itself
    if (p->gram_tc2 && configure_gram_tc2(p, g2_segs, g2_cta_first, g2_seg_first) != cudaSuccess) {
        cudaGetLastError();
        p->gram_tc2 = false;
    }
    p->evd_cluster = p->evd_chol && evd_cluster_eligible(p);
    if (p->evd_cluster && configure_evd_cluster(p) != cudaSuccess) {
        cudaGetLastError();
        p->evd_cluster = false;
    }
    if (p->N > 128 && !p->evd_cluster) p->evd_chol = false;   // above 128 frames the Cholesky kernel only factors (the cluster kernel sweeps)
    std::vector<PtcSeg> ptc_segs;
    std::vector<int> ptc_cta_first;
    p->proj_tc = project_tc_eligible(p);
    if (p->proj_tc && configure_project_tc(p, ptc_segs, ptc_cta_first) != cudaSuccess) {
        cudaGetLastError();
        p->proj_tc = false;
    }
    // ---- Gram work items: each window's box split into pixel chunks (multiples of GRAM_TP) ----
    std::vector<GramItem> gitems;
    p->gfirst_h.assign(p->K + 1, 0);
    if (!p->gram_tc && !p->gram_tc2) {
        long long target = p->sumPk / ((long long)p->num_sms * 6) + 1;
        long long ch = ((target + GRAM_TP - 1) / GRAM_TP) * GRAM_TP;
        if (ch < 4 * GRAM_TP) ch = 4 * GRAM_TP;
        int slot = 0;
        for (int k = 0; k < p->K; ++k) {
            p->gfirst_h[k] = slot;
            const int Pk = p->box_h[k].Pk;
            if (Pk > 0) {
                int nch = (int)((Pk + ch / 2) / ch);
                if (nch < 1) nch = 1;
                int per = (Pk + nch - 1) / nch;
                per = ((per + GRAM_TP - 1) / GRAM_TP) * GRAM_TP;
                for (int q0 = 0; q0 < Pk; q0 += per) {
                    int q1 = q0 + per < Pk ? q0 + per : Pk;
                    for (int b = 0; b < p->gram_batches; ++b) gitems.push_back({k, q0, q1, b, slot});
                    ++slot;
                }
            }
        }
        p->gfirst_h[p->K] = slot;
        p->n_gslots = slot;
        p->n_gitems = (int)gitems.size();
    }
    // ---- projection work items ----
    std::vector<ProjItem> pitems;
    p->pfirst_h.assign(p->K + 1, 0);
    for (int k = 0; k < p->K; ++k) {
        p->pfirst_h[k] = (int)pitems.size();
        for (int q0 = 0; q0 < p->box_h[k].Pk; q0 += PROJ_TPIX)
            pitems.push_back({k, q0, q0 + PROJ_TPIX < p->box_h[k].Pk ? q0 + PROJ_TPIX : p->box_h[k].Pk});
    }
    p->pfirst_h[p->K] = (int)pitems.size();
    p->n_pitems = (int)pitems.size();

    // ---- device memory ----
    const size_t N2 = (size_t)N * N, K = (size_t)p->K, Ns = (size_t)p->Ns, M = Ns - 1;
    bool ok = true;
    ok = ok && dev_upload(&p->gz_d, p->gz_h) && dev_upload(&p->gx_d, p->gx_h) && dev_upload(&p->box_d, p->box_h);
    ok = ok && dev_upload(&p->kzlo_d, kzlo) && dev_upload(&p->kzhi_d, kzhi) && dev_upload(&p->kxlo_d, kxlo) &&
         dev_upload(&p->kxhi_d, kxhi);
    ok = ok && dev_upload(&p->gitems_d, gitems) && dev_upload(&p->gfirst_d, p->gfirst_h);
    ok = ok && dev_upload(&p->pitems_d, pitems) && dev_upload(&p->pfirst_d, p->pfirst_h);
    ok = ok && dev_alloc(&p->gpart_d, (size_t)p->n_gslots * N2);
    if (p->gram_tc) {
        ok = ok && dev_upload(&p->gtc_segs_d, gtc_segs) && dev_upload(&p->gtc_cta_first_d, gtc_cta_first) &&
             dev_upload(&p->gtc_seg_first_d, gtc_seg_first) &&
             dev_alloc(&p->gtc_part_d, (size_t)(p->gtc_nseg ? p->gtc_nseg : 1) * 2 * 128 * 128);
    }
    if (p->gram_tc2) {
        ok = ok && dev_upload(&p->g2_segs_d, g2_segs) && dev_upload(&p->g2_cta_first_d, g2_cta_first) &&
             dev_upload(&p->g2_seg_first_d, g2_seg_first) &&
             dev_alloc(&p->g2_part_d, (size_t)(p->g2_nseg ? p->g2_nseg : 1) * 2 * 128 * 128);
    }
    if (p->evd_cluster) ok = ok && dev_alloc(&p->ec_gfac_d, K * 2 * Ns * (size_t)p->ec_LD) && dev_alloc(&p->ec_shift_d, K);
    if (p->evd_chol) ok = ok && dev_alloc(&p->ec_nexp_d, K);
    if (p->proj_tc) {
        ok = ok && dev_upload(&p->ptc_segs_d, ptc_segs) && dev_upload(&p->ptc_cta_first_d, ptc_cta_first) &&
             dev_alloc(&p->ptc_bpack_d, K * (size_t)(p->ptc_NB + 1) * (size_t)(p->ptc_Kp / 8) * 1024) &&
             dev_alloc(&p->ptc_part_d, (size_t)p->ptc_NB * (size_t)(p->sumPk ? p->sumPk : 1));
    }
    if (p->gram_tc || p->gram_tc2 || p->proj_tc) ok = ok && dev_alloc(&p->amax_d, 1);
    if (p->proj_tc && p->ptc_pre) {
        const size_t plane = (size_t)(p->ptc_Kp / 8) * (size_t)p->P * 32;
        ok = ok && dev_alloc(reinterpret_cast<unsigned char**>(&p->ptc_sh_d), plane) && dev_alloc(reinterpret_cast<unsigned char**>(&p->ptc_sl_d), plane);
    }
    if (ncc_mode(thr->mode)) {
        p->ncc_magN = p->proj_tc ? p->ptc_NB * 64 : N;
        ok = ok && dev_alloc(&p->ncc_mag_d, (size_t)(p->sumPk ? p->sumPk : 1) * p->ncc_magN) && dev_alloc(&p->ncc_isig_d, K * p->ncc_magN) &&
             dev_alloc(&p->ncc_part_d, K * 32 * 3 * N) && dev_alloc(&p->ncc_curve_d, K * N);
    }
    ok = ok && dev_alloc(reinterpret_cast<unsigned char**>(&p->R_d), K * N2 * 2 * p->esz);
    // the rotation log is replayed by vbuild_kernel, which only follows the two-sided jacobi_kernel
    if (!p->evd_chol) ok = ok && dev_alloc(reinterpret_cast<unsigned char**>(&p->rotlog_d), K * p->max_sweeps * M * 3 * p->NP * p->esz);
    ok = ok && dev_alloc(&p->lam_d, K * N) && dev_alloc(&p->order_d, K * N) && dev_alloc(&p->cut_d, K) &&
         dev_alloc(&p->sweeps_d, K) && dev_alloc(&p->conv_d, K) && dev_alloc(&p->nunconv_d, 1) && dev_alloc(&p->wslot_d, K * Ns) &&
         dev_alloc(&p->wslot_dd_d, K * Ns) && dev_alloc(&p->wt_d, K * N);
    ok = ok && dev_alloc(reinterpret_cast<unsigned char**>(&p->V_d), K * N * Ns * 2 * p->esz);
    ok = ok && dev_alloc(&p->B_d, K * N * Ns);
    ok = ok && dev_alloc(&p->tiles_d, (size_t)p->sumPk) && dev_alloc(&p->tsum_d, (size_t)p->n_pitems) &&
         dev_alloc(&p->mean_d, K) && dev_alloc(&p->alpha_d, K);
    if (!ok) {
        cudaGetLastError();
        free_plan_device(p);
        delete p;
        return LCF_ERR_ALLOC;
    }
    // the Gram kernel leaves the non-canonical half of each partial unwritten; clear once so no
    // uninitialised memory is ever read by tools (the loader never reads that half)
    cudaMemset(p->gpart_d, 0, (size_t)p->n_gslots * N2 * sizeof(double2));
    cudaMemset(p->nunconv_d, 0, sizeof(int));
    if (cudaDeviceSynchronize() != cudaSuccess) {
        free_plan_device(p);
        delete p;
        return LCF_ERR_CUDA;
    }
    *out = p;
    return LCF_OK;
}

extern "C" lcf_status lcf_plan_destroy(lcf_plan* p) {
    if (!p) return LCF_OK;
    if (p->twin) { lcf_plan_destroy(p->twin); p->twin = nullptr; }
    if (p->ran) cudaStreamSynchronize(p->last_stream);
    free_plan_device(p);
    cudaGetLastError();
    delete p;
    return LCF_OK;
}

// stride > 0: the Gram comes from the previous call's R and the new frames' columns (lcf_filter_stream)
static lcf_status filter_impl(lcf_plan* p, const void* iq_dev, float* pd_dev, cudaStream_t stream, int stride) {
    if (!p || !iq_dev || !pd_dev) return LCF_ERR_INVALID_ARG;
    if (p->cuda_failed) return LCF_ERR_CUDA;
    cudaStream_t st = stream;
    const float2* iq = reinterpret_cast<const float2*>(iq_dev);
    const bool tm = p->timing && p->timer.have;
    cudaError_t e = cudaSuccess;
    cudaEvent_t* evs = p->timer.ev[p->timer.calls % TIMER_RING];
    auto mark = [&](int i) { if (tm && e == cudaSuccess) e = cudaEventRecord(evs[i], st); };
    int stage = 0;
    auto run = [&](int id, cudaError_t r) { if (e == cudaSuccess && r != cudaSuccess) { e = r; stage = id; } };
    mark(0);
    if (e == cudaSuccess && (p->gram_tc || p->gram_tc2 || p->proj_tc)) run(1, launch_absmax(p, iq, st));
    if (e == cudaSuccess && p->proj_tc) run(1, launch_presplit(p, iq, st));
    if (e == cudaSuccess) {
        if (stride > 0) run(1, launch_gram_stream(p, iq, stride, st));
        else run(1, p->gram_tc ? launch_gram_tc(p, iq, st) : (p->gram_tc2 ? launch_gram_tc2(p, iq, st) : launch_gram(p, iq, st)));
    }
    if (e == cudaSuccess && stride >= 0 && p->strm_ready) {       // keep R and its data scale for the next streamed call
        run(1, cudaMemcpyAsync(p->Rprev_d, p->R_d, (size_t)p->K * p->N * p->N * sizeof(float2), cudaMemcpyDeviceToDevice, st));
        if (e == cudaSuccess) run(1, cudaMemcpyAsync(p->amax_prev_d, p->amax_d, sizeof(uint32_t), cudaMemcpyDeviceToDevice, st));
    }
    mark(1);
    if (p->evd_top) {
        if (e == cudaSuccess) run(2, launch_evd_top(p, st));
    } else {
        if (e == cudaSuccess) run(2, p->evd_chol ? launch_evd_chol(p, st, p->evd_cluster) : launch_jacobi(p, st));
        if (e == cudaSuccess && p->evd_cluster) run(2, launch_evd_cluster(p, st));
    }
    mark(2);
    if (e == cudaSuccess && !p->evd_chol && !p->evd_top) run(3, launch_vbuild(p, st));
    if (e == cudaSuccess && ncc_mode(p->thr.mode)) run(3, launch_ncc(p, iq, st));
    mark(3);
    if (e == cudaSuccess) run(4, p->prec == 1 ? launch_project_dd(p, iq, st) : (p->proj_tc ? launch_project_tc(p, iq, st) : launch_project(p, iq, st)));
    mark(4);
    if (e == cudaSuccess) run(5, launch_combine(p, pd_dev, st));
    mark(5);
    if (e != cudaSuccess) {
        static const char* names[] = {"event record", "gram", "evd", "weights/projector", "projection", "combine"};
        snprintf(p->last_error, sizeof(p->last_error), "%s: %s", names[stage], cudaGetErrorString(e));
    }
    if (tm) ++p->timer.calls;
    p->last_stream = st;
    p->ran = true;
    if (e != cudaSuccess) { p->cuda_failed = true; return LCF_ERR_CUDA; }
    return LCF_OK;
}

extern "C" lcf_status lcf_filter(lcf_plan* p, const void* iq_dev, float* pd_dev, cudaStream_t stream) {
    if (p) p->strm_valid = false;                       // a plain call breaks the chain of streamed ensembles
    return filter_impl(p, iq_dev, pd_dev, stream, -1);
}

extern "C" lcf_status lcf_filter_stream(lcf_plan* p, const void* iq_dev, float* pd_dev, int stride, cudaStream_t stream) {
    if (!p || !iq_dev || !pd_dev || stride < 0 || stride > p->N) return LCF_ERR_INVALID_ARG;
    if (!gram_stream_eligible(p)) {
        snprintf(p->last_error, sizeof(p->last_error), "lcf_filter_stream needs the tensor-core Gram of 32 .. 128 frames (precision 0, even Nz); use lcf_filter with this plan");
        return LCF_ERR_UNSUPPORTED;
    }
    if (!p->strm_ready) {                               // first use: segments, partials, the kept R
        std::vector<G2Seg> segs;
        std::vector<int> cta_first, seg_first;
        if (configure_gram_stream(p, segs, cta_first, seg_first) != cudaSuccess) { cudaGetLastError(); return LCF_ERR_UNSUPPORTED; }
        bool ok = dev_upload(&p->g2_segs_d, segs) && dev_upload(&p->g2_cta_first_d, cta_first) && dev_upload(&p->g2_seg_first_d, seg_first) &&
                  dev_alloc(&p->g2_part_d, (size_t)(p->g2_nseg ? p->g2_nseg : 1) * 2 * 128 * 128) &&
                  dev_alloc(&p->Rprev_d, (size_t)p->K * p->N * p->N) && dev_alloc(&p->amax_prev_d, 1);
        if (!ok) { cudaGetLastError(); return LCF_ERR_ALLOC; }
        p->strm_ready = true;
    }
    // stride = 0 or no previous streamed call: the whole Gram; otherwise only the new frames' columns
    const bool reuse = p->strm_valid && stride > 0 && stride < p->N;
    lcf_status s = filter_impl(p, iq_dev, pd_dev, stream, reuse ? stride : 0);
    p->strm_valid = (s == LCF_OK);
    return s;
}

extern "C" lcf_status lcf_filter_batch(lcf_plan* p, const void* const* iq_devs, float* const* pd_devs, int count, cudaStream_t stream) {
    if (!p || !iq_devs || !pd_devs || count < 0) return LCF_ERR_INVALID_ARG;
    for (int i = 0; i < count; ++i)
        if (!iq_devs[i] || !pd_devs[i]) return LCF_ERR_INVALID_ARG;
    if (p->cuda_failed) return LCF_ERR_CUDA;
    if (count == 0) return LCF_OK;
    const int lanes = count < LCF_LANES ? (count < 1 ? 1 : count) : LCF_LANES;
    lcf_status ls = ensure_lanes(p, lanes);
    if (ls != LCF_OK) return ls;
    // fork: the lanes start after everything already enqueued on the caller's stream
    cudaError_t e = cudaEventRecord(p->ev_fork, stream);
    for (int l = 0; l < lanes && e == cudaSuccess; ++l) e = cudaStreamWaitEvent(p->lane_st[l], p->ev_fork, 0);
    for (int i = 0; i < count && e == cudaSuccess && ls == LCF_OK; ++i)
        ls = lcf_filter(lane_plan(p, i % lanes), iq_devs[i], pd_devs[i], p->lane_st[i % lanes]);
    // join: the caller's stream continues when every lane is done
    for (int l = 0; l < lanes && e == cudaSuccess; ++l) {
        e = cudaEventRecord(p->ev_join[l], p->lane_st[l]);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(stream, p->ev_join[l], 0);
    }
    if (ls != LCF_OK) return ls;
    if (e != cudaSuccess) { p->cuda_failed = true; return LCF_ERR_CUDA; }
    return LCF_OK;
}

extern "C" lcf_status lcf_filter_host(lcf_plan* p, const void* iq_host, float* pd_host, cudaStream_t stream) {
    if (!p || !iq_host || !pd_host) return LCF_ERR_INVALID_ARG;
    if (p->cuda_failed) return LCF_ERR_CUDA;
    const size_t iq_bytes = (size_t)p->N * p->P * sizeof(float2), pd_bytes = (size_t)p->P * sizeof(float);
    if (!p->iq_stage_d) {
        if (cudaMalloc(&p->iq_stage_d, iq_bytes) != cudaSuccess ||
            cudaMalloc(reinterpret_cast<void**>(&p->pd_stage_d), pd_bytes) != cudaSuccess) {
            cudaGetLastError();
            cudaFree(p->iq_stage_d); p->iq_stage_d = nullptr;
            return LCF_ERR_ALLOC;
        }
    }
    cudaStream_t st = stream;
    if (cudaMemcpyAsync(p->iq_stage_d, iq_host, iq_bytes, cudaMemcpyHostToDevice, st) != cudaSuccess) {
        p->cuda_failed = true;
        return LCF_ERR_CUDA;
    }
    lcf_status s = lcf_filter(p, p->iq_stage_d, p->pd_stage_d, stream);
    if (s != LCF_OK) return s;
    if (cudaMemcpyAsync(pd_host, p->pd_stage_d, pd_bytes, cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaStreamSynchronize(st) != cudaSuccess) {
        p->cuda_failed = true;
        return LCF_ERR_CUDA;
    }
    return take_unconverged(p, nullptr);
}

extern "C" const char* lcf_last_error(const lcf_plan* p) { return p ? p->last_error : "null plan"; }

extern "C" lcf_status lcf_filter_host_batch(lcf_plan* p, const void* const* iq_hosts, float* const* pd_hosts, int count, cudaStream_t stream) {
    if (!p || !iq_hosts || !pd_hosts || count < 0) return LCF_ERR_INVALID_ARG;
    for (int i = 0; i < count; ++i)
        if (!iq_hosts[i] || !pd_hosts[i]) return LCF_ERR_INVALID_ARG;
    if (p->cuda_failed) return LCF_ERR_CUDA;
    if (count == 0) return LCF_OK;
    const size_t iq_bytes = (size_t)p->N * p->P * sizeof(float2), pd_bytes = (size_t)p->P * sizeof(float);
    // staging buffers, copy stream and events are created on first use
    constexpr int NS = LCF_LANES;                       // staging sets = lanes: ensemble i uses set and lane i % NS
    void** iqs[NS] = {&p->iq_stage_d, &p->iq_stage2_d, &p->iq_stage3_d};
    float** pds[NS] = {&p->pd_stage_d, &p->pd_stage2_d, &p->pd_stage3_d};
    for (int b = 0; b < NS; ++b) {
        if (!*iqs[b] && cudaMalloc(iqs[b], iq_bytes) != cudaSuccess) { cudaGetLastError(); *iqs[b] = nullptr; return LCF_ERR_ALLOC; }
        if (!*pds[b] && cudaMalloc(reinterpret_cast<void**>(pds[b]), pd_bytes) != cudaSuccess) { cudaGetLastError(); *pds[b] = nullptr; return LCF_ERR_ALLOC; }
        if (!p->ev_copied[b] && cudaEventCreateWithFlags(&p->ev_copied[b], cudaEventDisableTiming) != cudaSuccess) return LCF_ERR_CUDA;
        if (!p->ev_done[b] && cudaEventCreateWithFlags(&p->ev_done[b], cudaEventDisableTiming) != cudaSuccess) return LCF_ERR_CUDA;
    }
    if (!p->copy_stream && cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking) != cudaSuccess) return LCF_ERR_CUDA;
    lcf_status ls = ensure_lanes(p, NS);
    if (ls != LCF_OK) return ls;
    // ensemble i: copy on the copy stream into staging set i % NS, kernels of lane i % NS (plan or a twin) on that lane's
    // stream, image copied back on the lane's stream.  The copy of ensemble i + NS waits for the kernels of ensemble i;
    // with three sets the copy engine does not idle behind them (two sets: 667 ensembles/s at config 2).
    cudaStream_t cs = p->copy_stream;
    cudaError_t e = cudaStreamSynchronize(stream);      // everything the caller enqueued before is done
    for (int i = 0; i < count && e == cudaSuccess && ls == LCF_OK; ++i) {
        const int b = i % NS;
        cudaStream_t st = p->lane_st[b];
        if (i >= NS) e = cudaStreamWaitEvent(cs, p->ev_done[b], 0);      // the staging buffer is free once the kernels of ensemble i - NS have read it
        if (e == cudaSuccess) e = cudaMemcpyAsync(*iqs[b], iq_hosts[i], iq_bytes, cudaMemcpyHostToDevice, cs);
        if (e == cudaSuccess) e = cudaEventRecord(p->ev_copied[b], cs);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(st, p->ev_copied[b], 0);
        if (e != cudaSuccess) break;
        ls = lcf_filter(lane_plan(p, b), *iqs[b], *pds[b], st);
        if (ls != LCF_OK) break;
        e = cudaEventRecord(p->ev_done[b], st);          // input consumed (and image ready)
        if (e == cudaSuccess) e = cudaMemcpyAsync(pd_hosts[i], *pds[b], pd_bytes, cudaMemcpyDeviceToHost, st);
    }
    cudaError_t e2 = cudaStreamSynchronize(cs);
    for (int l = 0; l < NS; ++l) { cudaError_t e3 = cudaStreamSynchronize(p->lane_st[l]); if (e2 == cudaSuccess) e2 = e3; }
    if (ls != LCF_OK) return ls;
    if (e != cudaSuccess || e2 != cudaSuccess) { p->cuda_failed = true; return LCF_ERR_CUDA; }
    return take_unconverged(p, nullptr);
}

extern "C" int lcf_num_windows(const lcf_plan* p) { return p ? p->K : 0; }

extern "C" lcf_status lcf_set_max_sweeps(lcf_plan* p, int max_sweeps) {
    if (!p || max_sweeps < 0) return LCF_ERR_INVALID_ARG;
    p->sweep_cap = max_sweeps;
    return LCF_OK;
}

extern "C" lcf_status lcf_get_converged(lcf_plan* p, int* windows) {
    if (windows) *windows = 0;
    lcf_status s = sync_plan(p);
    if (s != LCF_OK) return s;
    return take_unconverged(p, windows);
}

extern "C" lcf_status lcf_get_eigenvalues(lcf_plan* p, double* lam) {
    lcf_status s = sync_plan(p);
    if (s != LCF_OK || !lam) return s != LCF_OK ? s : LCF_ERR_INVALID_ARG;
    if (cudaMemcpy(lam, p->lam_d, sizeof(double) * p->K * p->N, cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
    return conv_status(p);
}

extern "C" lcf_status lcf_get_cutoffs(lcf_plan* p, int* c) {
    lcf_status s = sync_plan(p);
    if (s != LCF_OK || !c) return s != LCF_OK ? s : LCF_ERR_INVALID_ARG;
    if (cudaMemcpy(c, p->cut_d, sizeof(int) * p->K, cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
    return conv_status(p);
}

extern "C" lcf_status lcf_get_sweeps(lcf_plan* p, int* sw) {
    lcf_status s = sync_plan(p);
    if (s != LCF_OK || !sw) return s != LCF_OK ? s : LCF_ERR_INVALID_ARG;
    if (cudaMemcpy(sw, p->sweeps_d, sizeof(int) * p->K, cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
    return conv_status(p);
}

extern "C" lcf_status lcf_get_ncc(lcf_plan* p, double* ncc) {
    lcf_status s = sync_plan(p);
    if (s != LCF_OK || !ncc) return s != LCF_OK ? s : LCF_ERR_INVALID_ARG;
    if (!p->ncc_curve_d) return LCF_ERR_INVALID_ARG;           // not an NCC-mode plan
    if (cudaMemcpy(ncc, p->ncc_curve_d, sizeof(double) * p->K * p->N, cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
    return conv_status(p);
}

extern "C" lcf_status lcf_get_weights(lcf_plan* p, double* wt) {
    lcf_status s = sync_plan(p);
    if (s != LCF_OK || !wt) return s != LCF_OK ? s : LCF_ERR_INVALID_ARG;
    if (cudaMemcpy(wt, p->wt_d, sizeof(double) * p->K * p->N, cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
    return conv_status(p);
}

extern "C" lcf_status lcf_get_window_means(lcf_plan* p, double* m) {
    lcf_status s = sync_plan(p);
    if (s != LCF_OK || !m) return s != LCF_OK ? s : LCF_ERR_INVALID_ARG;
    if (cudaMemcpy(m, p->mean_d, sizeof(double) * p->K, cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
    return conv_status(p);
}

extern "C" lcf_status lcf_get_gram(lcf_plan* p, double* R) {
    lcf_status s = sync_plan(p);
    if (s != LCF_OK || !R) return s != LCF_OK ? s : LCF_ERR_INVALID_ARG;
    const size_t n = (size_t)p->K * p->N * p->N * 2;
    if (p->prec == 1) {
        if (cudaMemcpy(R, p->R_d, n * sizeof(double), cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
    } else {
        std::vector<float> tmp(n);
        if (cudaMemcpy(tmp.data(), p->R_d, n * sizeof(float), cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
        double un = 1.0;
        if (p->gram_tc) {   // the tensor-core Gram leaves R in its power-of-two data scale
            uint32_t bits = 0;
            if (cudaMemcpy(&bits, p->amax_d, sizeof(bits), cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
            un = std::ldexp(1.0, -2 * sm100::pow2_scale_exp(bits));
        }
        for (size_t i = 0; i < n; ++i) R[i] = (double)tmp[i] * un;
    }
    return conv_status(p);
}

extern "C" lcf_status lcf_get_eigenvectors(lcf_plan* p, double* V) {
    lcf_status s = sync_plan(p);
    if (s != LCF_OK || !V) return s != LCF_OK ? s : LCF_ERR_INVALID_ARG;
    const size_t K = p->K, N = p->N, Ns = p->Ns, n = K * N * Ns * 2;
    std::vector<double> tmp(n);
    if (p->prec == 1) {
        if (cudaMemcpy(tmp.data(), p->V_d, n * sizeof(double), cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
    } else {
        std::vector<float> t32(n);
        if (cudaMemcpy(t32.data(), p->V_d, n * sizeof(float), cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
        for (size_t i = 0; i < n; ++i) tmp[i] = (double)t32[i];
    }
    std::vector<int> order(K * N);
    if (cudaMemcpy(order.data(), p->order_d, sizeof(int) * K * N, cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
    for (size_t k = 0; k < K; ++k)
        for (size_t a = 0; a < N; ++a)
            for (size_t i = 0; i < N; ++i) {
                const size_t u = (size_t)order[k * N + i];
                const double* src = &tmp[((k * N + a) * Ns + u) * 2];
                double* dst = &V[((k * N + a) * N + i) * 2];
                dst[0] = src[0]; dst[1] = src[1];
            }
    return conv_status(p);
}

extern "C" lcf_status lcf_get_filters(lcf_plan* p, double* F) {
    lcf_status s = sync_plan(p);
    if (s != LCF_OK || !F) return s != LCF_OK ? s : LCF_ERR_INVALID_ARG;
    const size_t n = (size_t)p->K * p->N * p->N * 2;
    if (!p->F_d && cudaMalloc(reinterpret_cast<void**>(&p->F_d), n * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        p->F_d = nullptr;
        return LCF_ERR_ALLOC;
    }
    if (launch_build_filters(p, p->last_stream) != cudaSuccess || cudaStreamSynchronize(p->last_stream) != cudaSuccess)
        return LCF_ERR_CUDA;
    if (cudaMemcpy(F, p->F_d, n * sizeof(double), cudaMemcpyDeviceToHost) != cudaSuccess) return LCF_ERR_CUDA;
    return conv_status(p);
}

extern "C" lcf_status lcf_set_timing(lcf_plan* p, int enabled) {
    if (!p) return LCF_ERR_INVALID_ARG;
    if (enabled && !p->timer.have) {
        for (auto& set : p->timer.ev)
            for (auto& e : set)
                if (cudaEventCreate(&e) != cudaSuccess) return LCF_ERR_CUDA;
        p->timer.have = true;
    }
    p->timing = enabled != 0;
    p->timer.calls = 0;
    return LCF_OK;
}

extern "C" lcf_status lcf_get_stage_ms(lcf_plan* p, float ms[5]) {
    if (!p || !ms || !p->timing || !p->timer.have || p->timer.calls == 0) return LCF_ERR_INVALID_ARG;
    lcf_status s = sync_plan(p);
    if (s != LCF_OK) return s;
    const long long n = p->timer.calls < TIMER_RING ? p->timer.calls : TIMER_RING;
    double acc[5] = {0, 0, 0, 0, 0};
    for (long long c = 0; c < n; ++c)
        for (int i = 0; i < 5; ++i) {
            float t = 0.f;
            if (cudaEventElapsedTime(&t, p->timer.ev[c][i], p->timer.ev[c][i + 1]) != cudaSuccess) return LCF_ERR_CUDA;
            acc[i] += t;
        }
    for (int i = 0; i < 5; ++i) ms[i] = (float)(acc[i] / (double)n);
    return LCF_OK;
}

extern "C" lcf_status lcf_get_work(const lcf_plan* p, lcf_work* w) {
    if (!p || !w) return LCF_ERR_INVALID_ARG;
    const double N = p->N, S = (double)p->sumPk;
    w->sum_Pk = S;
    w->gram_flops = 8.0 * S * N * (N + 1.0) / 2.0;   // Hermitian half, 8 real flops per complex MAC
    w->proj_flops = 8.0 * S * N * N;                 // dense N x N projector factor
    w->hbm_bytes = 8.0 * N * (double)p->P + 4.0 * (double)p->P;
    w->launches = ((p->gram_tc || p->gram_tc2 || p->proj_tc) ? 1 : 0) + ((p->proj_tc && p->ptc_pre) ? 1 : 0) + 2 + (p->evd_chol ? (p->evd_cluster ? 2 : 1) : 2) + (p->proj_tc ? 3 : 1) + 2;   // absmax, gram+reduce, evd(+V build), projection(+pack, finish), alpha, combine
    w->gram_tc = (p->gram_tc || p->gram_tc2) ? 1 : 0; w->evd_chol = p->evd_top ? 2 : (p->evd_chol ? 1 : 0); w->proj_tc = (p->proj_tc && p->prec == 0) ? 1 : 0;
    w->gram_tensor_flops = 0.0; w->proj_tensor_flops = 0.0;
    for (int k = 0; k < p->K; ++k) {
        const WinBox& b = p->box_h[k];
        if (b.Pk == 0) continue;
        const double ntz = (double)((b.z0 + b.Lz - (b.z0 & ~1) + 15) / 16);
        const double Np = (double)((p->N + 15) / 16 * 16);
        // Gram: 16-pixel tiles, per tile three 128 x 2Np x 16 MMAs and one 128 x Np x 16 (= seven 128 x Np x 16 products)
        if (p->gram_tc) w->gram_tensor_flops += ntz * b.Lx * 2.0 * 7.0 * 2.0 * 128.0 * Np * 8.0;
        // block form: per tile and block twelve 128 x nc x 16 MMAs
        if (p->gram_tc2)
            for (int j = 0; j < 3; ++j) w->gram_tensor_flops += ntz * b.Lx * 12.0 * 2.0 * 128.0 * p->g2_blk[j].nc * 16.0;
        // projection: 64-pixel tiles x column blocks, per 16 frames one 128x256x16 and one 128x128x16 MMA
        if (p->proj_tc)
            w->proj_tensor_flops += ntz * (double)((b.Lx + 3) / 4) * p->ptc_NB * (p->ptc_Kp / 8) * 2.0 * 128.0 * (256.0 + 128.0) * 8.0;
    }
    return LCF_OK;
}

extern "C" int lcf_scale_exponent(float amax) {
    uint32_t bits;
    std::memcpy(&bits, &amax, sizeof(bits));
    return lcf::sm100::pow2_scale_exp(bits & 0x7fffffffu);
}
