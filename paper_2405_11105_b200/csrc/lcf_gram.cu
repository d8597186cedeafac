// lcf_gram.cu -- kernel 1: batched window-weighted complex Gram (Eq. 12)
//
//   R_k[i][j] = sum_{p in supp k} w_k(p)^2 conj(S[i][p]) S[j][p],   w_k(p) = g_z(z) g_x(x)  (Eq. 11)
//
// One CTA = (window k, a chunk of the window's support box, a batch of thread tiles).  The CTA walks
// its chunk in tiles of GRAM_TP pixels: cp.async stages the raw complex64 samples of all N frames,
// each thread rescales the samples it staged by w (so the tile holds W_k S, Eq. 11) into a padded
// operand tile, and every thread accumulates a TM x TM complex register tile of A^H A.  Thread tile
// (ti, tj) owns rows {ti + Tn*ii} and columns {tj + Tn*jj} (strided, so a warp's operand reads are
// bank-conflict free); only tiles with ti <= tj are computed (Hermitian symmetry) -- entry (i, j) is
// canonical iff (i mod Tn) <= (j mod Tn), the other half is its conjugate.  Partial sums go to a
// per-chunk fp64 buffer that the EVD kernel's loader reduces in a fixed order (deterministic, no
// atomics).  T = float: FP32 FMA (products exact inside the FMA), but an fp32 accumulator only ever
// sums GRAM_FLUSH_TILES * GRAM_TP pixels: it is then added into the CTA's fp64 partial and cleared.
// A plain fp32 running sum over a whole chunk (thousands of pixels) loses ~1e-5 of |R|, which the
// 60-70 dB clutter-to-blood ratio amplifies into >1e-3 power-Doppler errors.
// T = double: the fp32 samples are widened, products are exact in fp64, one store at the end.
#include "lcf_internal.h"

namespace lcf {

struct GramArgs {
    const float2* iq;
    int N, Nz, Kz;
    long long P;
    int Tn, ntiles, tiles_per_batch;
    const double* gz;  // [Kz][Nz]
    const double* gx;  // [Kx][Nx]
    int Nx;
    const WinBox* box;
    const GramItem* items;
    double2* part;  // [slot][N][N] complex double
};

template <typename T> struct Cx;
template <> struct Cx<float> { using type = float2; };
template <> struct Cx<double> { using type = double2; };

__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc) {
    unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;\n" ::: "memory"); }

template <typename T> struct GramCfg;
template <> struct GramCfg<float> { static constexpr int TM = 8, TPS = GRAM_TP + 2; };   // 272 B rows
template <> struct GramCfg<double> { static constexpr int TM = 4, TPS = GRAM_TP + 1; };  // 528 B rows

template <typename T>
__global__ void __launch_bounds__(GRAM_THREADS, (sizeof(T) == 4 ? 2 : 1)) gram_kernel(GramArgs a) {
    using C = typename Cx<T>::type;
    constexpr int TM = GramCfg<T>::TM, TPS = GramCfg<T>::TPS, TP = GRAM_TP;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = a.N, Tn = a.Tn, Nr = Tn * TM;
    float2* stage = reinterpret_cast<float2*>(smem_raw);                       // [N][TP]
    C* As = reinterpret_cast<C*>(smem_raw + (size_t)N * TP * sizeof(float2));  // [Nr][TPS]

    const int tid = threadIdx.x, nthr = blockDim.x;
    const GramItem it = a.items[blockIdx.x];
    const WinBox bx = a.box[it.k];
    const double* gz = a.gz + (size_t)bx.kz * a.Nz;
    const double* gx = a.gx + (size_t)bx.kx * a.Nx;

    // thread tile (ti, tj), ti <= tj, enumerated row-major over the upper triangle
    int e = it.batch * a.tiles_per_batch + tid;
    const bool active = (tid < a.tiles_per_batch) && (e < a.ntiles);
    int ti = 0, tj = 0;
    if (active) {
        int rowlen = Tn;
        while (e >= rowlen) { e -= rowlen; --rowlen; ++ti; }
        tj = ti + e;
    }

    T acc_re[TM][TM], acc_im[TM][TM];
#pragma unroll
    for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TM; ++j) { acc_re[i][j] = T(0); acc_im[i][j] = T(0); }

    // zero the padding rows (frames >= N) once
    for (int idx = tid; idx < (Nr - N) * TPS; idx += nthr) {
        C z; z.x = T(0); z.y = T(0);
        As[(size_t)N * TPS + idx] = z;
    }

    const int pp = tid & (TP - 1);   // this thread always stages pixel column pp of the tile
    const int t0 = tid >> 5, tstep = nthr >> 5;
    const int ntile = (it.q1 - it.q0 + TP - 1) / TP;

    // pixel of tile `tile` handled by this thread: offset into a frame, weight, validity
    auto pixel = [&](int tile, long long& off, T& w) -> bool {
        int q = it.q0 + tile * TP + pp;
        if (q >= it.q1) { off = 0; w = T(0); return false; }
        int xr = q / bx.Lz, zr = q - xr * bx.Lz;
        int x = bx.x0 + xr, z = bx.z0 + zr;
        off = (long long)x * a.Nz + z;
        w = (T)(gz[z] * gx[x]);
        return true;
    };
    auto issue = [&](long long off, bool valid) {
        if (valid) {
            const float2* src = a.iq + off;
            for (int t = t0; t < N; t += tstep) cp_async8(&stage[t * TP + pp], src + (long long)t * a.P);
        }
        cp_async_commit();
    };

    // add the register tile into this CTA's fp64 partial (first flush overwrites: no memset needed)
    int nflushed = 0;
    auto flush = [&](bool first) {
        if (active) {
            double2* out = a.part + (size_t)it.pslot * N * N + (size_t)ti * N + tj;
#pragma unroll
            for (int i = 0; i < TM; ++i) {
                if (ti + Tn * i < N) {
#pragma unroll
                    for (int j = 0; j < TM; ++j) {
                        if (tj + Tn * j < N) {
                            double2* o = out + Tn * j;
                            double2 v = make_double2(0.0, 0.0);
                            if (!first) v = *o;
                            v.x += (double)acc_re[i][j]; v.y += (double)acc_im[i][j];
                            *o = v;
                        }
                    }
                }
                out += (size_t)Tn * N;
                asm volatile("" ::: "memory");   // one row of the tile at a time: bounds the live loads
#pragma unroll
                for (int j = 0; j < TM; ++j) { acc_re[i][j] = T(0); acc_im[i][j] = T(0); }
            }
        }
        ++nflushed;
    };

    long long off; T w;
    bool valid = pixel(0, off, w);
    issue(off, valid);
    for (int tile = 0; tile < ntile; ++tile) {
        cp_async_wait_all();
        __syncthreads();  // everyone finished computing on the previous operand tile
        for (int t = t0; t < N; t += tstep) {
            C v; v.x = T(0); v.y = T(0);
            if (valid) { float2 s = stage[t * TP + pp]; v.x = w * (T)s.x; v.y = w * (T)s.y; }
            As[t * TPS + pp] = v;
        }
        if (tile + 1 < ntile) { valid = pixel(tile + 1, off, w); issue(off, valid); }
        __syncthreads();  // operand tile complete
        if (active) {
            if constexpr (sizeof(T) == 4) {
                const float2* Af = reinterpret_cast<const float2*>(As);
#pragma unroll 1
                for (int p2 = 0; p2 < TP; p2 += 2) {
                    float4 av[TM];
#pragma unroll
                    for (int i = 0; i < TM; ++i) av[i] = *reinterpret_cast<const float4*>(&Af[(ti + Tn * i) * TPS + p2]);
#pragma unroll
                    for (int j = 0; j < TM; ++j) {
                        const float4 bv = *reinterpret_cast<const float4*>(&Af[(tj + Tn * j) * TPS + p2]);
#pragma unroll
                        for (int i = 0; i < TM; ++i) {
                            // conj(a) * b, two pixels
                            acc_re[i][j] = fmaf(av[i].x, bv.x, acc_re[i][j]);
                            acc_re[i][j] = fmaf(av[i].y, bv.y, acc_re[i][j]);
                            acc_im[i][j] = fmaf(av[i].x, bv.y, acc_im[i][j]);
                            acc_im[i][j] = fmaf(-av[i].y, bv.x, acc_im[i][j]);
                            acc_re[i][j] = fmaf(av[i].z, bv.z, acc_re[i][j]);
                            acc_re[i][j] = fmaf(av[i].w, bv.w, acc_re[i][j]);
                            acc_im[i][j] = fmaf(av[i].z, bv.w, acc_im[i][j]);
                            acc_im[i][j] = fmaf(-av[i].w, bv.z, acc_im[i][j]);
                        }
                    }
                }
            } else {
                const double2* Ad = reinterpret_cast<const double2*>(As);
#pragma unroll 2
                for (int p1 = 0; p1 < TP; ++p1) {
                    double2 av[TM], bv[TM];
#pragma unroll
                    for (int i = 0; i < TM; ++i) av[i] = Ad[(ti + Tn * i) * TPS + p1];
#pragma unroll
                    for (int j = 0; j < TM; ++j) bv[j] = Ad[(tj + Tn * j) * TPS + p1];
#pragma unroll
                    for (int i = 0; i < TM; ++i)
#pragma unroll
                        for (int j = 0; j < TM; ++j) {
                            acc_re[i][j] = fma(av[i].x, bv[j].x, acc_re[i][j]);
                            acc_re[i][j] = fma(av[i].y, bv[j].y, acc_re[i][j]);
                            acc_im[i][j] = fma(av[i].x, bv[j].y, acc_im[i][j]);
                            acc_im[i][j] = fma(-av[i].y, bv[j].x, acc_im[i][j]);
                        }
                }
            }
        }
        // single flush site (keeps the accumulators out of local memory)
        if (tile + 1 == ntile || (sizeof(T) == 4 && (tile + 1) % GRAM_FLUSH_TILES == 0)) flush(nflushed == 0);
    }
}

static size_t gram_smem_bytes(int N, int Tn, bool dbl) {
    int TM = dbl ? GramCfg<double>::TM : GramCfg<float>::TM;
    int TPS = dbl ? GramCfg<double>::TPS : GramCfg<float>::TPS;
    return (size_t)N * GRAM_TP * sizeof(float2) + (size_t)Tn * TM * TPS * (dbl ? 16 : 8);
}

cudaError_t configure_gram(lcf_plan* p) {
    const bool dbl = p->prec == 1;
    p->gram_TM = dbl ? GramCfg<double>::TM : GramCfg<float>::TM;
    p->gram_Tn = (p->N + p->gram_TM - 1) / p->gram_TM;
    int ntiles = p->gram_Tn * (p->gram_Tn + 1) / 2;
    p->gram_batches = (ntiles + GRAM_THREADS - 1) / GRAM_THREADS;
    p->gram_tiles_per_batch = (ntiles + p->gram_batches - 1) / p->gram_batches;
    p->gram_smem = gram_smem_bytes(p->N, p->gram_Tn, dbl);
    if (p->gram_smem > (size_t)p->smem_optin) return cudaErrorInvalidConfiguration;
    if (dbl) return set_max_dyn_smem(gram_kernel<double>, p->smem_optin);
    return set_max_dyn_smem(gram_kernel<float>, p->smem_optin);
}

// R_k = sum of the window's per-chunk fp64 partials in a fixed order (deterministic, no atomics);
// entry (u, v) is canonical in the partial iff (u mod Tn) <= (v mod Tn), otherwise its conjugate is.
template <typename T>
__global__ void gram_reduce_kernel(const double2* part, const int* gfirst, int N, int Tn, void* Rv) {
    using C = typename Cx<T>::type;
    const int k = blockIdx.z;
    const int u = blockIdx.y * 16 + threadIdx.y, v = blockIdx.x * 16 + threadIdx.x;
    if (u >= N || v >= N) return;
    const bool direct = (u % Tn) <= (v % Tn);
    const size_t idx = direct ? (size_t)u * N + v : (size_t)v * N + u;
    double re = 0.0, im = 0.0;
    for (int s = gfirst[k]; s < gfirst[k + 1]; ++s) {
        const double2 x = part[(size_t)s * N * N + idx];
        re += x.x; im += x.y;
    }
    if (!direct) im = -im;
    if (u == v) im = 0.0;
    C o; o.x = (T)re; o.y = (T)im;
    reinterpret_cast<C*>(Rv)[(size_t)k * N * N + (size_t)u * N + v] = o;
}

cudaError_t launch_gram(lcf_plan* p, const float2* iq, cudaStream_t st) {
    GramArgs a;
    a.iq = iq; a.N = p->N; a.Nz = p->Nz; a.Kz = p->Kz; a.P = p->P; a.Nx = p->Nx;
    a.Tn = p->gram_Tn; a.ntiles = p->gram_Tn * (p->gram_Tn + 1) / 2; a.tiles_per_batch = p->gram_tiles_per_batch;
    a.gz = p->gz_d; a.gx = p->gx_d; a.box = p->box_d; a.items = p->gitems_d; a.part = p->gpart_d;
    int threads = ((p->gram_tiles_per_batch + 31) / 32) * 32;
    if (p->n_gitems > 0) {
        if (p->prec == 1) gram_kernel<double><<<p->n_gitems, threads, p->gram_smem, st>>>(a);
        else gram_kernel<float><<<p->n_gitems, threads, p->gram_smem, st>>>(a);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    dim3 blk(16, 16), grid((p->N + 15) / 16, (p->N + 15) / 16, p->K);
    if (p->prec == 1) gram_reduce_kernel<double><<<grid, blk, 0, st>>>(p->gpart_d, p->gfirst_d, p->N, p->gram_Tn, p->R_d);
    else gram_reduce_kernel<float><<<grid, blk, 0, st>>>(p->gpart_d, p->gfirst_d, p->N, p->gram_Tn, p->R_d);
    return cudaGetLastError();
}

}  // namespace lcf
