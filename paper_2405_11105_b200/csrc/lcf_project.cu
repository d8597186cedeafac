// lcf_project.cu -- kernel 4: fused projection, |.|^2 slow-time sum and weighted overlap-add.
//
//   4a  project_kernel:  U[p][u] = sum_t S[t][p] B_k[t][u]   (Eq. 4, with
//       B_k = V_k diag(wt); V_k unitary, so sum_t |(s_p V diag(wt) V^H)_t|^2 = sum_u |U[p][u]|^2)
//       PD_k(p) = w_k(p)^2 sum_u |U[p][u]|^2                 (Eq. 11)
//       One CTA = PROJ_TPIX pixels of one window x all columns; the filtered cube is never formed:
//       the CTA keeps an 8x8 complex register tile per thread, reduces |.|^2 over columns on chip
//       and writes one float per (window, pixel) plus one partial sum per CTA.
//   4b  alpha_kernel:    m_k = (1/P) sum_p PD_k(p), alpha_k = 1/m_k (0 if m_k = 0)   (Eq. 13)
//   4c  combine_kernel:  PD(p) = sum_k alpha_k PD_k(p) gathered over the windows covering p
//       (Eq. 13) -- a gather, so the image is written once, no atomics.
#include "lcf_internal.h"

namespace lcf {

struct ProjArgs {
    const float2* iq;
    int N, Ns, Nz, Nx;
    long long P;
    const float2* B;  // [K][N][Ns]
    const WinBox* box;
    const ProjItem* items;
    const double* gz;
    const double* gx;
    float* tiles;
    float* tsum;
    int nct;   // column tiles of 8
};

__device__ __forceinline__ void cp_async8_zfill(void* smem_dst, const void* gsrc, int src_bytes) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(d), "l"(gsrc), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async16_zfill(void* smem_dst, const void* gsrc, int src_bytes) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(d), "l"(gsrc), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int NLEFT> __device__ __forceinline__ void cp_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(NLEFT) : "memory"); }

__global__ void __launch_bounds__(256, 1) project_kernel(ProjArgs a) {
    constexpr int TPIX = PROJ_TPIX, KT = PROJ_KT, ST = PROJ_STAGES;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = a.N, Ns = a.Ns, NCT = a.nct, NCP = NCT * 8;
    float2* Ss = reinterpret_cast<float2*>(smem_raw);            // [ST][KT][TPIX]
    float2* Bs = Ss + ST * KT * TPIX;                            // [ST][KT][NCP]
    long long* poff = reinterpret_cast<long long*>(Bs + (size_t)ST * KT * NCP);  // [TPIX], -1 = invalid
    const int tid = threadIdx.x, nthr = blockDim.x;
    const ProjItem it = a.items[blockIdx.x];
    const WinBox bx = a.box[it.k];
    const int pg = tid & 7, ct = tid >> 3;
    const bool active = ct < NCT;

    if (tid < TPIX) {
        int q = it.q0 + tid;
        long long off = -1;
        if (q < it.q1) {
            int xr = q / bx.Lz, zr = q - xr * bx.Lz;
            off = (long long)(bx.x0 + xr) * a.Nz + (bx.z0 + zr);
        }
        poff[tid] = off;
    }
    // zero the padding columns of every B stage once (columns Ns..NCP-1 are never staged)
    if (NCP > Ns)
        for (int e = tid; e < ST * KT * (NCP - Ns); e += nthr) {
            int row = e / (NCP - Ns), cc = Ns + e % (NCP - Ns);
            Bs[(size_t)row * NCP + cc] = make_float2(0.f, 0.f);
        }
    __syncthreads();

    const float2* Bk = a.B + (size_t)it.k * N * Ns;
    const int nchunk = (N + KT - 1) / KT;
    const int halfNs = Ns >> 1;
    auto issue = [&](int kc) {
        if (kc < nchunk) {
            const int slot = kc % ST;
            float2* sdst = Ss + (size_t)slot * KT * TPIX;
            for (int e = tid; e < KT * TPIX; e += nthr) {
                int tt = e / TPIX, px = e - tt * TPIX;
                int t = kc * KT + tt;
                long long off = poff[px];
                bool ok = (off >= 0) && (t < N);
                const float2* src = a.iq + (ok ? (long long)t * a.P + off : 0);
                cp_async8_zfill(&sdst[e], src, ok ? 8 : 0);
            }
            float2* bdst = Bs + (size_t)slot * KT * NCP;
            for (int e = tid; e < KT * halfNs; e += nthr) {
                int tt = e / halfNs, cc = e - tt * halfNs;
                int t = kc * KT + tt;
                bool ok = t < N;
                const float2* src = Bk + (ok ? (size_t)t * Ns + 2 * cc : 0);
                cp_async16_zfill(&bdst[(size_t)tt * NCP + 2 * cc], src, ok ? 16 : 0);
            }
        }
        cp_commit();
    };

    float acc_re[8][8], acc_im[8][8];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) { acc_re[i][j] = 0.f; acc_im[i][j] = 0.f; }

#pragma unroll
    for (int s = 0; s < ST - 1; ++s) issue(s);
    for (int kc = 0; kc < nchunk; ++kc) {
        cp_wait<ST - 2>();
        __syncthreads();
        issue(kc + ST - 1);
        if (active) {
            const float2* sS = Ss + (size_t)(kc % ST) * KT * TPIX;
            const float2* sB = Bs + (size_t)(kc % ST) * KT * NCP;
#pragma unroll 1
            for (int tt = 0; tt < KT; ++tt) {
                float4 sv[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) sv[i] = *reinterpret_cast<const float4*>(&sS[tt * TPIX + 2 * pg + 16 * i]);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const float4 bv = *reinterpret_cast<const float4*>(&sB[(size_t)tt * NCP + 2 * ct + 2 * NCT * j]);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        // s * b for pixels (2i, 2i+1) x columns (2j, 2j+1)
                        acc_re[2 * i][2 * j] = fmaf(sv[i].x, bv.x, acc_re[2 * i][2 * j]);
                        acc_re[2 * i][2 * j] = fmaf(-sv[i].y, bv.y, acc_re[2 * i][2 * j]);
                        acc_im[2 * i][2 * j] = fmaf(sv[i].x, bv.y, acc_im[2 * i][2 * j]);
                        acc_im[2 * i][2 * j] = fmaf(sv[i].y, bv.x, acc_im[2 * i][2 * j]);
                        acc_re[2 * i][2 * j + 1] = fmaf(sv[i].x, bv.z, acc_re[2 * i][2 * j + 1]);
                        acc_re[2 * i][2 * j + 1] = fmaf(-sv[i].y, bv.w, acc_re[2 * i][2 * j + 1]);
                        acc_im[2 * i][2 * j + 1] = fmaf(sv[i].x, bv.w, acc_im[2 * i][2 * j + 1]);
                        acc_im[2 * i][2 * j + 1] = fmaf(sv[i].y, bv.z, acc_im[2 * i][2 * j + 1]);
                        acc_re[2 * i + 1][2 * j] = fmaf(sv[i].z, bv.x, acc_re[2 * i + 1][2 * j]);
                        acc_re[2 * i + 1][2 * j] = fmaf(-sv[i].w, bv.y, acc_re[2 * i + 1][2 * j]);
                        acc_im[2 * i + 1][2 * j] = fmaf(sv[i].z, bv.y, acc_im[2 * i + 1][2 * j]);
                        acc_im[2 * i + 1][2 * j] = fmaf(sv[i].w, bv.x, acc_im[2 * i + 1][2 * j]);
                        acc_re[2 * i + 1][2 * j + 1] = fmaf(sv[i].z, bv.z, acc_re[2 * i + 1][2 * j + 1]);
                        acc_re[2 * i + 1][2 * j + 1] = fmaf(-sv[i].w, bv.w, acc_re[2 * i + 1][2 * j + 1]);
                        acc_im[2 * i + 1][2 * j + 1] = fmaf(sv[i].z, bv.w, acc_im[2 * i + 1][2 * j + 1]);
                        acc_im[2 * i + 1][2 * j + 1] = fmaf(sv[i].w, bv.z, acc_im[2 * i + 1][2 * j + 1]);
                    }
                }
            }
        }
    }
    cp_wait<0>();
    __syncthreads();   // all stages consumed: the staging memory is reused for the column reduction
    float* red = reinterpret_cast<float*>(smem_raw);   // [NCT][TPIX]
    if (active) {
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            float s = 0.f;
#pragma unroll
            for (int j = 0; j < 8; ++j) s += acc_re[i][j] * acc_re[i][j] + acc_im[i][j] * acc_im[i][j];
            int px = 2 * pg + 16 * (i >> 1) + (i & 1);
            red[ct * TPIX + px] = s;
        }
    }
    __syncthreads();
    if (tid < TPIX) {
        float s = 0.f;
        for (int c = 0; c < NCT; ++c) s += red[c * TPIX + tid];
        int q = it.q0 + tid;
        float val = 0.f;
        if (q < it.q1) {
            int xr = q / bx.Lz, zr = q - xr * bx.Lz;
            double w = a.gz[(size_t)bx.kz * a.Nz + bx.z0 + zr] * a.gx[(size_t)bx.kx * a.Nx + bx.x0 + xr];
            val = (float)(w * w) * s;
            a.tiles[bx.tile_off + q] = val;
        }
        // deterministic CTA sum of the TPIX values (2 warps)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) val += __shfl_xor_sync(0xffffffffu, val, o);
        __shared__ float wsum[TPIX / 32];
        if ((tid & 31) == 0) wsum[tid >> 5] = val;
        __syncwarp();
        asm volatile("bar.sync 1, %0;\n" ::"n"(TPIX) : "memory");
        if (tid == 0) {
            float t = 0.f;
            for (int w2 = 0; w2 < TPIX / 32; ++w2) t += wsum[w2];
            a.tsum[blockIdx.x] = t;
        }
    }
}

// 4a in double (precision = 1: "a double precision may be essential"): the same contraction on the FP64
// pipe, B_k = V_k diag(wt) formed on the fly from the fp64 eigenvectors and weights.  CTA = one ProjItem (<= 64 pixels);
// thread (tp, tc) of a 16 x 16 grid keeps pixels tp + 16 i and columns tc + 16 j (i, j < 4) of a 64-column tile in
// registers; frames stream through shared memory PDD_KT at a time (converted to double on the way in); the squared
// magnitudes are summed over the columns of a tile in the thread, over tiles in the thread, over tc in shared memory.
constexpr int PDD_KT = 8;
__global__ void __launch_bounds__(256) project_dd_kernel(const float2* iq, int N, int Ns, int Nz, int Nx, long long P, const double2* V,
                                                        const double* wdd, const WinBox* box, const ProjItem* items, const double* gz,
                                                        const double* gx, float* tiles, float* tsum) {
    __shared__ double2 Ss[PDD_KT][64], Bs[PDD_KT][64];
    __shared__ double red[16][64];
    __shared__ long long poff[64];
    const int tid = threadIdx.x, tp = tid & 15, tc = tid >> 4;
    const ProjItem it = items[blockIdx.x];
    const WinBox bx = box[it.k];
    if (tid < 64) {
        const int q = it.q0 + tid;
        long long off = -1;
        if (q < it.q1) { const int xr = q / bx.Lz, zr = q - xr * bx.Lz; off = (long long)(bx.x0 + xr) * Nz + (bx.z0 + zr); }
        poff[tid] = off;
    }
    __syncthreads();
    const double2* Vk = V + (size_t)it.k * N * Ns;
    const double* wk = wdd + (size_t)it.k * Ns;
    double psum[4] = {0.0, 0.0, 0.0, 0.0};
    for (int c0 = 0; c0 < Ns; c0 += 64) {
        double ar[4][4], ai[4][4];
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) ar[i][j] = ai[i][j] = 0.0;
        for (int t0 = 0; t0 < N; t0 += PDD_KT) {
            for (int e = tid; e < PDD_KT * 64; e += 256) {
                const int tt = e >> 6, x = e & 63, t = t0 + tt;
                double2 sv = make_double2(0.0, 0.0), bv = make_double2(0.0, 0.0);
                if (t < N) {
                    if (poff[x] >= 0) { const float2 f = iq[(size_t)t * P + poff[x]]; sv = make_double2(f.x, f.y); }
                    const int u = c0 + x;
                    if (u < Ns) { const double2 v = Vk[(size_t)t * Ns + u]; const double w = wk[u]; bv = make_double2(v.x * w, v.y * w); }
                }
                Ss[tt][x] = sv; Bs[tt][x] = bv;
            }
            __syncthreads();
#pragma unroll
            for (int tt = 0; tt < PDD_KT; ++tt) {
                double2 s[4], b[4];
#pragma unroll
                for (int i = 0; i < 4; ++i) { s[i] = Ss[tt][tp + 16 * i]; b[i] = Bs[tt][tc + 16 * i]; }
#pragma unroll
                for (int i = 0; i < 4; ++i)
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        ar[i][j] = fma(s[i].x, b[j].x, fma(-s[i].y, b[j].y, ar[i][j]));
                        ai[i][j] = fma(s[i].x, b[j].y, fma(s[i].y, b[j].x, ai[i][j]));
                    }
            }
            __syncthreads();
        }
#pragma unroll
        for (int i = 0; i < 4; ++i)
#pragma unroll
            for (int j = 0; j < 4; ++j) psum[i] += ar[i][j] * ar[i][j] + ai[i][j] * ai[i][j];
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) red[tc][tp + 16 * i] = psum[i];
    __syncthreads();
    if (tid < 64) {
        double s = 0.0;
        for (int c = 0; c < 16; ++c) s += red[c][tid];
        const int q = it.q0 + tid;
        float val = 0.f;
        if (q < it.q1) {
            const int xr = q / bx.Lz, zr = q - xr * bx.Lz;
            const double w = gz[(size_t)bx.kz * Nz + bx.z0 + zr] * gx[(size_t)bx.kx * Nx + bx.x0 + xr];
            val = (float)(w * w * s);
            tiles[bx.tile_off + q] = val;
        }
        // the CTA's sum of its (rounded) pixel values, fixed order, as project_kernel forms it
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) val += __shfl_xor_sync(0xffffffffu, val, o);
        __shared__ float wsum[2];
        if ((tid & 31) == 0) wsum[tid >> 5] = val;
        asm volatile("bar.sync 1, 64;\n" ::: "memory");
        if (tid == 0) tsum[blockIdx.x] = wsum[0] + wsum[1];
    }
}

__global__ void alpha_kernel(const float* tsum, const int* pfirst, long long P, double* mean, float* alpha) {
    const int k = blockIdx.x, tid = threadIdx.x;
    __shared__ double sh[128];
    double acc = 0.0;
    for (int i = pfirst[k] + tid; i < pfirst[k + 1]; i += 128) acc += (double)tsum[i];
    sh[tid] = acc;
    __syncthreads();
    for (int o = 64; o > 0; o >>= 1) {
        if (tid < o) sh[tid] += sh[tid + o];
        __syncthreads();
    }
    if (tid == 0) {
        double m = sh[0] / (double)P;
        mean[k] = m;
        alpha[k] = (m > 0.0) ? (float)(1.0 / m) : 0.f;
    }
}

struct CombArgs {
    int Nz, Nx, Kz;
    const int *kzlo, *kzhi, *kxlo, *kxhi;
    const WinBox* box;
    const float* tiles;
    const float* alpha;
    float* pd;
};

__global__ void combine_kernel(CombArgs a) {
    const int z = blockIdx.x * blockDim.x + threadIdx.x, x = blockIdx.y;
    if (z >= a.Nz) return;
    float s = 0.f;
    const int z0 = a.kzlo[z], z1 = a.kzhi[z], x0 = a.kxlo[x], x1 = a.kxhi[x];
    for (int kx = x0; kx <= x1; ++kx)
        for (int kz = z0; kz <= z1; ++kz) {
            const int k = kx * a.Kz + kz;
            const WinBox b = a.box[k];
            const float v = a.tiles[b.tile_off + (long long)(x - b.x0) * b.Lz + (z - b.z0)];
            s = fmaf(a.alpha[k], v, s);
        }
    a.pd[(size_t)x * a.Nz + z] = s;
}

static size_t proj_smem_bytes(int nct) {
    size_t st = (size_t)PROJ_STAGES * PROJ_KT * (PROJ_TPIX + nct * 8) * sizeof(float2) + PROJ_TPIX * sizeof(long long);
    size_t red = (size_t)nct * PROJ_TPIX * sizeof(float);
    return st > red ? st : red;
}

cudaError_t configure_project(lcf_plan* p) {
    p->proj_nct = (p->Ns + 7) / 8;
    p->proj_threads = ((p->proj_nct * 8 + 31) / 32) * 32;
    if (p->proj_threads < PROJ_TPIX) p->proj_threads = PROJ_TPIX;
    if (p->proj_threads > 256) return cudaErrorInvalidConfiguration;
    p->proj_smem = proj_smem_bytes(p->proj_nct);
    if (p->proj_smem > (size_t)p->smem_optin) return cudaErrorInvalidConfiguration;
    return set_max_dyn_smem(project_kernel, p->smem_optin);
}

cudaError_t launch_project(lcf_plan* p, const float2* iq, cudaStream_t st) {
    if (p->n_pitems == 0) return cudaSuccess;
    ProjArgs a;
    a.iq = iq; a.N = p->N; a.Ns = p->Ns; a.Nz = p->Nz; a.Nx = p->Nx; a.P = p->P; a.B = p->B_d; a.box = p->box_d;
    a.items = p->pitems_d; a.gz = p->gz_d; a.gx = p->gx_d; a.tiles = p->tiles_d; a.tsum = p->tsum_d; a.nct = p->proj_nct;
    project_kernel<<<p->n_pitems, p->proj_threads, p->proj_smem, st>>>(a);
    return cudaGetLastError();
}

cudaError_t launch_project_dd(lcf_plan* p, const float2* iq, cudaStream_t st) {
    if (p->n_pitems == 0) return cudaSuccess;
    project_dd_kernel<<<p->n_pitems, 256, 0, st>>>(iq, p->N, p->Ns, p->Nz, p->Nx, p->P, reinterpret_cast<const double2*>(p->V_d), p->wslot_dd_d,
                                                   p->box_d, p->pitems_d, p->gz_d, p->gx_d, p->tiles_d, p->tsum_d);
    return cudaGetLastError();
}

cudaError_t launch_combine(lcf_plan* p, float* pd, cudaStream_t st) {
    alpha_kernel<<<p->K, 128, 0, st>>>(p->tsum_d, p->pfirst_d, p->P, p->mean_d, p->alpha_d);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    CombArgs a;
    a.Nz = p->Nz; a.Nx = p->Nx; a.Kz = p->Kz; a.kzlo = p->kzlo_d; a.kzhi = p->kzhi_d; a.kxlo = p->kxlo_d; a.kxhi = p->kxhi_d;
    a.box = p->box_d; a.tiles = p->tiles_d; a.alpha = p->alpha_d; a.pd = pd;
    dim3 grid((p->Nz + 127) / 128, p->Nx);
    combine_kernel<<<grid, 128, 0, st>>>(a);
    return cudaGetLastError();
}

}  // namespace lcf
