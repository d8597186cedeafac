// lcf_gram_tc2.cu -- kernel 1, tensor-core path for 128 < N <= 256 frames: the window-weighted complex
// Gram (Eq. 12) as BLOCKS of R on tcgen05, fp16 split precision.
//
// lcf_gram_tc.cu holds the whole 128 x Np result of a window in one SM's tensor memory and gets the
// lo.hi products from the hi.lo ones by transposition; neither works above 128 frames (two row
// tiles, 4 Np > 512 TMEM columns).  Here R_k is cut into blocks of 128 rows x at most 128 columns,
//     J0: rows [0,128)  x cols [0,c1)      J1: rows [0,128)  x cols [c1,Np)      J2: rows [128,Np) x cols [128,Np)
// (c1 = 16 ceil(Np / 32); the block below the diagonal is the conjugate transpose of J1's upper part),
// and a (window, block) pair is an independent job: its CTA loads and converts only the frames the
// block touches, and accumulates the block directly,
//     Re R[i][j] += xr_i xr_j + xi_i xi_j          Im R[i][j] += xr_i xi_j - xi_i xr_j       (x = w s, Eq. 11)
// with every fp32 x = hi + lo (fp16 each, 22 bits together; the data scaled by a power of two as in
// lcf_gram_tc.cu):  a b ~ ah bh + ah bl + al bh  ->  12 tcgen05.mma.kind::f16 128 x nc x 16 per
// 16-pixel tile into two TMEM accumulators (Re at column 0, Im at column 256), the three negative
// products through the instruction descriptor's negate-A bit.
// The fp32 accumulation of the tensor core truncates, so both accumulators are drained into registers
// of the drain warps every `group` tiles (128 pixels) and restarted with the accumulate flag.
// Roles, pipeline and operand layout (K-major core matrices, no swizzle) as in lcf_gram_tc.cu; the
// four operand matrices Rh, Rl, Ih, Il of a stage are apart and hold the frames at their absolute
// row, so a block's A and B operands are the same tiles at row offsets m0 and c0.
// gram_tc2_reduce_kernel sums a (window, block)'s segments in fp64, undoes the data scale and writes
// the full Hermitian R_k (the lower triangle is the mirrored upper one, exactly).
#include <cuda.h>
#include <cmath>

#include "lcf_internal.h"
#include "lcf_sm100.cuh"

namespace lcf {

using namespace sm100;

constexpr int G2_PX = 16;                  // pixels per tile
constexpr int G2_STAGES = 4;               // raw and operand stages
constexpr int G2_CONV_WARPS = 8, G2_DRAIN_WARPS = 8, G2_FIRST_CONV = 4;
constexpr int G2_FIRST_DRAIN = G2_FIRST_CONV + G2_CONV_WARPS;
constexpr int G2_THREADS = 32 * (G2_FIRST_DRAIN + G2_DRAIN_WARPS);
constexpr int G2_CONV_GROUPS = 2, G2_WPG = G2_CONV_WARPS / G2_CONV_GROUPS;
static_assert(G2_STAGES % G2_CONV_GROUPS == 0, "a converter group must see every use of its stages");

struct G2Args {
    int N, Np, Nz, Nx;
    int group;                 // tiles per drain
    const double* gz;          // [Kz][Nz]
    const double* gx;          // [Kx][Nx]
    const WinBox* box;
    const G2Seg* segs;
    const int* cta_first;      // [grid+1]
    float* part;               // [nseg][2][128][128]
    uint32_t raw_stride;       // bytes between raw stages (multiple of 1024)
    uint32_t mat_bytes;        // one operand matrix: 2 chunks x Np rows x 16 bytes
    const uint32_t* amax;
    G2Block blk[3];
};

struct G2Bars {
    uint64_t full[G2_STAGES], empty[G2_STAGES];
    uint64_t opfull[G2_STAGES], opempty[G2_STAGES];
    uint64_t accfull, accempty;
    uint32_t tmem_base;
    alignas(16) float wts[G2_STAGES][2 * G2_PX];
};

static __device__ __forceinline__ void g2_sts128u(uint32_t addr, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
static __device__ __forceinline__ ulonglong2 g2_lds128u(uint32_t addr) {
    ulonglong2 v;
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "r"(addr));
    return v;
}
static __device__ __forceinline__ float2 g2_mul2(unsigned long long a, unsigned long long b) {
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    float2 f;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(f.x), "=f"(f.y) : "l"(r));
    return f;
}

struct G2Maps { CUtensorMap m[3]; };

__global__ void __launch_bounds__(G2_THREADS, 1) gram_tc2_kernel(const __grid_constant__ G2Maps maps, G2Args a) {
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    unsigned char* sbase = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
    unsigned char* raw = sbase;                                               // [STAGES][raw_stride]
    unsigned char* ops = sbase + (size_t)G2_STAGES * a.raw_stride;            // [STAGES][Rh | Rl | Ih | Il]
    const uint32_t op_bytes = 4u * a.mat_bytes;
    // an M = 128 operand that starts at row m0 = 128 of an Np < 256 row matrix reads past its end: one
    // more matrix of slack keeps those (unused) reads inside the allocation
    G2Bars* bars = reinterpret_cast<G2Bars*>(ops + (size_t)G2_STAGES * op_bytes + a.mat_bytes);
    double* gzs = reinterpret_cast<double*>(bars + 1);
    double* gxs = gzs + a.Nz;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int N = a.N;
    const int seg0 = a.cta_first[blockIdx.x], seg1 = a.cta_first[blockIdx.x + 1];

    // rows >= N of the operand matrices are never written: zero everything once
    for (uint32_t i = tid * 16; i < G2_STAGES * op_bytes + a.mat_bytes; i += G2_THREADS * 16) *reinterpret_cast<uint4*>(ops + i) = make_uint4(0, 0, 0, 0);
    fence_proxy_async_smem();
    if (tid == 0) {
        for (int s = 0; s < G2_STAGES; ++s) {
            mbar_init(&bars->full[s], 1); mbar_init(&bars->empty[s], G2_WPG);
            mbar_init(&bars->opfull[s], G2_WPG); mbar_init(&bars->opempty[s], 1);
        }
        mbar_init(&bars->accfull, 1);
        mbar_init(&bars->accempty, G2_DRAIN_WARPS);
        mbar_fence_init();
    }
    if (warp == 1) tmem_alloc<512>(&bars->tmem_base);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = bars->tmem_base;

    if (warp < G2_FIRST_CONV) asm volatile("setmaxnreg.dec.sync.aligned.u32 32;");
    if (warp == 0) {
        // =========================== TMA producer ===========================
        if (lane < 3) tma_prefetch_desc(&maps.m[lane]);
        const double scale = (double)pow2f(pow2_scale_exp(*a.amax));
        uint32_t it = 0;
        for (int sg = seg0; sg < seg1; ++sg) {
            const G2Seg seg = a.segs[sg];
            const G2Block bk = a.blk[seg.blk];
            const WinBox bx = a.box[seg.k];
            const int ze = bx.z0 & ~1;
            const int ntz = (bx.z0 + bx.Lz - ze + G2_PX - 1) / G2_PX;
            const uint32_t bytes = (uint32_t)bk.nbox * 128u;
            __syncwarp();
            for (int i = lane; i < a.Nz; i += 32) gzs[i] = a.gz[(size_t)bx.kz * a.Nz + i];
            for (int i = lane; i < a.Nx; i += 32) gxs[i] = a.gx[(size_t)bx.kx * a.Nx + i];
            __syncwarp();
            for (int t = 0; t < seg.ntile; ++t, ++it) {
                const int s = it % G2_STAGES;
                const uint32_t ph = (it / G2_STAGES) & 1;
                const int tau = seg.tile0 + t;
                const int txi = tau / ntz, tzi = tau - txi * ntz;
                const int z = ze + tzi * G2_PX, x = bx.x0 + txi;
                mbar_wait(&bars->empty[s], ph ^ 1);
                if (lane < G2_PX) {
                    const int zz = z + lane;
                    float w = 0.f;
                    if (zz < a.Nz && x < a.Nx) w = (float)(gzs[zz] * gxs[x] * scale);
                    bars->wts[s][2 * lane] = w; bars->wts[s][2 * lane + 1] = w;
                }
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive_expect_tx(&bars->full[s], bytes);
                    tma_load_3d(raw + (size_t)s * a.raw_stride, &maps.m[seg.blk], 2 * z, x, bk.f0, &bars->full[s]);
                }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer ===========================
        const uint32_t tRe = tmem, tIm = tmem + 256;
        const uint32_t lbo = (uint32_t)a.Np * 16u;
        const uint64_t desc0 = make_smem_desc(smem_u32(ops), lbo, 128, SWZ_NONE);
        const uint64_t mb = (uint64_t)(a.mat_bytes >> 4);
        uint32_t it = 0, gc = 0;
        for (int sg = seg0; sg < seg1; ++sg) {
            const G2Seg seg = a.segs[sg];
            const G2Block bk = a.blk[seg.blk];
            const uint32_t idp = make_idesc_f16(128, bk.nc, false, false), idn = make_idesc_f16(128, bk.nc, true, false);
            const uint64_t aoff = (uint64_t)((bk.m0 * 16) >> 4), boff = (uint64_t)((bk.c0 * 16) >> 4);
            for (int t = 0; t < seg.ntile; ++t, ++it) {
                const int o = it % G2_STAGES;
                const uint32_t pho = (it / G2_STAGES) & 1;
                const bool group_first = (t % a.group) == 0;
                const bool group_last = ((t + 1) % a.group) == 0 || t + 1 == seg.ntile;
                mbar_wait(&bars->opfull[o], pho);
                if (group_first) mbar_wait(&bars->accempty, (gc & 1) ^ 1);
                tc_fence_after_sync();
                if (elect_one()) {
                    const uint64_t d = desc0 + (uint64_t)((o * op_bytes) >> 4);
                    const uint64_t aRh = d + aoff, aRl = d + mb + aoff, aIh = d + 2 * mb + aoff, aIl = d + 3 * mb + aoff;
                    const uint64_t bRh = d + boff, bRl = d + mb + boff, bIh = d + 2 * mb + boff, bIl = d + 3 * mb + boff;
                    const uint32_t acc0 = group_first ? 0u : 1u;          // the drained accumulators restart from this tile
                    mma_f16(tRe, aRh, bRh, idp, acc0);
                    mma_f16(tRe, aRh, bRl, idp, 1u);
                    mma_f16(tRe, aRl, bRh, idp, 1u);
                    mma_f16(tRe, aIh, bIh, idp, 1u);
                    mma_f16(tRe, aIh, bIl, idp, 1u);
                    mma_f16(tRe, aIl, bIh, idp, 1u);
                    mma_f16(tIm, aRh, bIh, idp, acc0);
                    mma_f16(tIm, aRh, bIl, idp, 1u);
                    mma_f16(tIm, aRl, bIh, idp, 1u);
                    mma_f16(tIm, aIh, bRh, idn, 1u);
                    mma_f16(tIm, aIh, bRl, idn, 1u);
                    mma_f16(tIm, aIl, bRh, idn, 1u);
                    mma_commit(&bars->opempty[o]);
                    if (group_last) mma_commit(&bars->accfull);
                }
                __syncwarp();
                if (group_last) ++gc;
            }
        }
    } else if (warp >= G2_FIRST_CONV && warp < G2_FIRST_DRAIN) {
        // =========================== converters ===========================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 72;");
        const int cw = warp - G2_FIRST_CONV;
        const uint32_t raw_u32 = smem_u32(raw), ops_u32 = smem_u32(ops), wts_u32 = smem_u32(&bars->wts[0][0]);
        const uint32_t lbo = (uint32_t)a.Np * 16u, mbb = a.mat_bytes;
        const int grp = cw / G2_WPG, gw = cw % G2_WPG;
        uint32_t it = 0;
        for (int sg = seg0; sg < seg1; ++sg) {
            const G2Seg seg = a.segs[sg];
            const G2Block bk = a.blk[seg.blk];
            const int nfr = (N - bk.f0) < bk.nbox ? (N - bk.f0) : bk.nbox;      // real frames in the stage
            const int nwt = 2 * ((nfr + 31) / 32);
            for (int t = 0; t < seg.ntile; ++t, ++it) {
                if ((int)(it % G2_CONV_GROUPS) != grp) continue;
                const int s = it % G2_STAGES;
                const uint32_t ph = (it / G2_STAGES) & 1;
                const uint32_t rs = raw_u32 + (uint32_t)s * a.raw_stride;
                const uint32_t os = ops_u32 + (uint32_t)s * op_bytes;
                const uint32_t ws = wts_u32 + (uint32_t)s * (G2_PX * 8);
                mbar_wait(&bars->full[s], ph);
                mbar_wait(&bars->opempty[s], ph ^ 1);
#pragma unroll 1
                for (int wt = gw; wt < nwt; wt += G2_WPG) {
                    const int c8 = wt & 1, fr = (wt >> 1) * 32 + lane;
                    if (fr < nfr) {
                        const uint32_t sw = (uint32_t)(fr & 7);
                        ulonglong2 wq[4], pq[4];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            wq[u] = g2_lds128u(ws + (uint32_t)c8 * 64u + 16 * u);
                            pq[u] = g2_lds128u(rs + (uint32_t)fr * 128u + ((((uint32_t)(4 * c8 + u)) ^ sw) << 4));
                        }
                        uint32_t rh[4], rl[4], ih[4], il[4];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const float2 v0 = g2_mul2(pq[u].x, wq[u].x), v1 = g2_mul2(pq[u].y, wq[u].y);
                            f16_split2(v0.x, v1.x, rh[u], rl[u]);
                            f16_split2(v0.y, v1.y, ih[u], il[u]);
                        }
                        const uint32_t dst = os + (uint32_t)c8 * lbo + (uint32_t)(bk.f0 + fr) * 16u;
                        g2_sts128u(dst, rh[0], rh[1], rh[2], rh[3]);
                        g2_sts128u(dst + mbb, rl[0], rl[1], rl[2], rl[3]);
                        g2_sts128u(dst + 2 * mbb, ih[0], ih[1], ih[2], ih[3]);
                        g2_sts128u(dst + 3 * mbb, il[0], il[1], il[2], il[3]);
                    }
                }
                fence_proxy_async_smem();
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive(&bars->empty[s]);
                    mbar_arrive(&bars->opfull[s]);
                }
            }
        }
    } else if (warp >= G2_FIRST_DRAIN) {
        // =========================== accumulator drain ===========================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 152;");
        const int dw = warp - G2_FIRST_DRAIN;
        const int quad = warp & 3;
        const int half = dw >> 2;                     // which 64 columns of Re / Im this warp keeps
        const uint32_t tlane = tmem + ((uint32_t)(quad * 32) << 16);
        const int row = quad * 32 + lane;
        float acc[128];
#pragma unroll
        for (int i = 0; i < 128; ++i) acc[i] = 0.f;
        uint32_t gc = 0;
        for (int sg = seg0; sg < seg1; ++sg) {
            const G2Seg seg = a.segs[sg];
            const int nc = a.blk[seg.blk].nc;
            const int ngroups = (seg.ntile + a.group - 1) / a.group;
            for (int g = 0; g < ngroups; ++g) {
                mbar_wait(&bars->accfull, gc & 1);
                tc_fence_after_sync();
#pragma unroll
                for (int blk = 0; blk < 8; ++blk) {
                    const int cj = half * 64 + (blk & 3) * 16;
                    if (cj < nc) {
                        uint32_t v[16];
                        tmem_ld16(tlane + (blk < 4 ? 0u : 256u) + (uint32_t)cj, v);
                        tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 16; ++j) acc[blk * 16 + j] += __uint_as_float(v[j]);
                    }
                }
                tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars->accempty);
                ++gc;
            }
            // segment end: this segment's partial block (Re, Im), rows = TMEM lanes
            float* out = a.part + (size_t)sg * 2 * 128 * 128 + (size_t)row * 128 + half * 64;
#pragma unroll
            for (int blk = 0; blk < 8; ++blk) {
                const int cj = half * 64 + (blk & 3) * 16;
                if (cj < nc) {
                    float* o2 = out + (size_t)(blk >> 2) * 128 * 128 + (blk & 3) * 16;
#pragma unroll
                    for (int j = 0; j < 16; j += 4)
                        *reinterpret_cast<float4*>(o2 + j) = make_float4(acc[blk * 16 + j], acc[blk * 16 + j + 1], acc[blk * 16 + j + 2], acc[blk * 16 + j + 3]);
                }
            }
#pragma unroll
            for (int i = 0; i < 128; ++i) acc[i] = 0.f;
        }
    }
    tc_fence_before_sync();
    __syncthreads();
    if (warp == 1) tmem_dealloc<512>(tmem);
}

// R_k[i][j], i <= j, = sum over the segments of the block that holds (i, j), in fp64, times 2^(-2k) (the
// data scale of the fp16 operands); the lower triangle is its exact mirror.  seg_first is indexed
// by k * 3 + block.
__global__ void gram_tc2_reduce_kernel(const float* part, const int* seg_first, int N, int c1, const uint32_t* amax, float2* R) {
    const int k = blockIdx.z;
    const int i = blockIdx.y * 16 + threadIdx.y, j = blockIdx.x * 16 + threadIdx.x;
    if (i >= N || j >= N) return;
    const int a = i <= j ? i : j, b = i <= j ? j : i;          // the upper-triangle entry (a, b)
    int blk, r, c;
    if (a < 128) { blk = b < c1 ? 0 : 1; r = a; c = b - (blk ? c1 : 0); }
    else { blk = 2; r = a - 128; c = b - 128; }
    double re = 0.0, im = 0.0;
    for (int s = seg_first[k * 3 + blk]; s < seg_first[k * 3 + blk + 1]; ++s) {
        const float* p = part + (size_t)s * 2 * 128 * 128 + (size_t)r * 128 + c;
        re += (double)p[0];
        im += (double)p[16384];
    }
    const double un = ldexp(1.0, -2 * sm100::pow2_scale_exp(*amax));
    if (i == j) im = 0.0;
    if (i > j) im = -im;
    R[((size_t)k * N + i) * N + j] = make_float2((float)(re * un), (float)(im * un));
}

// ---------------------------------------------------------------- host side
typedef CUresult (*G2EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static G2EncodeFn g2_encode_fn() {
    static G2EncodeFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<G2EncodeFn>(p);
    }
    return fn;
}

// one map per block: box = 16 pixels x 1 x nbox frames (whole 8-frame swizzle atoms), 128B swizzle
static const G2Maps* g2_encode_maps(lcf_plan* p, const void* iq) {
    if (const unsigned char* m = p->g2_tmaps.find(iq)) return reinterpret_cast<const G2Maps*>(m);
    G2EncodeFn fn = g2_encode_fn();
    if (!fn) return nullptr;
    unsigned char* slot = p->g2_tmaps.slot(iq);
    for (int b = 0; b < 3; ++b) {
        cuuint64_t dims[3] = {(cuuint64_t)2 * p->Nz, (cuuint64_t)p->Nx, (cuuint64_t)p->N};
        cuuint64_t strides[2] = {(cuuint64_t)p->Nz * 8, (cuuint64_t)p->P * 8};
        cuuint32_t box[3] = {2 * G2_PX, 1, (cuuint32_t)p->g2_blk[b].nbox};
        cuuint32_t es[3] = {1, 1, 1};
        CUresult r = fn(reinterpret_cast<CUtensorMap*>(slot) + b, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(iq), dims, strides, box,
                        es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) { p->g2_tmaps.drop_last(iq); return nullptr; }
    }
    return reinterpret_cast<const G2Maps*>(slot);
}

bool gram_tc2_eligible(const lcf_plan* p) {
    return p->prec == 0 && p->N > 128 && p->N <= 256 && (p->Nz % 2) == 0 && g2_encode_fn() != nullptr;
}

// jobs = (window, block, tile) in that order; contiguous slices of equal estimated cost, cut at (window, block)
cudaError_t configure_gram_tc2(lcf_plan* p, std::vector<G2Seg>& segs, std::vector<int>& cta_first, std::vector<int>& seg_first) {
    const int K = p->K, N = p->N, Np = (N + 15) / 16 * 16;
    const int c1 = 16 * ((Np + 31) / 32);
    auto box8 = [&](int f0, int f1) { int n = (f1 < N ? f1 : N) - f0; return (n + 7) / 8 * 8; };
    p->g2_c1 = c1;
    p->g2_blk[0] = {0, 0, c1, 0, box8(0, 128)};
    p->g2_blk[1] = {0, c1, Np - c1, 0, box8(0, Np)};
    p->g2_blk[2] = {128, 128, Np - 128, 128, box8(128, Np)};
    double wgt[3];
    for (int b = 0; b < 3; ++b) wgt[b] = 6.0 * p->g2_blk[b].nc + 2.0 * p->g2_blk[b].nbox;   // MMA cycles + conversion, per tile
    std::vector<double> pre((size_t)K * 3 + 1, 0.0);
    std::vector<long long> ntl(K);
    for (int k = 0; k < K; ++k) {
        const WinBox& b = p->box_h[k];
        ntl[k] = b.Pk > 0 ? (long long)((b.z0 + b.Lz - (b.z0 & ~1) + G2_PX - 1) / G2_PX) * b.Lx : 0;
        for (int j = 0; j < 3; ++j) pre[(size_t)k * 3 + j + 1] = pre[(size_t)k * 3 + j] + wgt[j] * (double)ntl[k];
    }
    const double T = pre[(size_t)K * 3];
    long long total_tiles = 0;
    for (int k = 0; k < K; ++k) total_tiles += 3 * ntl[k];
    int grid = (int)(total_tiles < p->num_sms ? total_tiles : p->num_sms);
    if (grid < 1) grid = 1;
    p->g2_grid = grid;
    segs.clear();
    cta_first.assign(grid + 1, 0);
    seg_first.assign((size_t)K * 3 + 1, 0);
    // tile t of job j starts at cost pre[j] + w t and belongs to the CTA whose equal share of the total cost holds that point
    const double per = T / grid;
    std::vector<std::vector<G2Seg>> per_job((size_t)K * 3);
    for (size_t j = 0; j < (size_t)K * 3; ++j) {
        const int k = (int)(j / 3), b = (int)(j % 3);
        const long long nt = ntl[k];
        long long t0 = 0;
        while (t0 < nt) {
            int c = (int)((pre[j] + wgt[b] * (double)t0) / per);
            if (c > grid - 1) c = grid - 1;
            long long t1 = nt;
            if (c < grid - 1) {
                t1 = (long long)std::ceil(((double)(c + 1) * per - pre[j]) / wgt[b]);
                if (t1 <= t0) t1 = t0 + 1;
                if (t1 > nt) t1 = nt;
            }
            per_job[j].push_back({k, b, (int)t0, (int)(t1 - t0), c});
            t0 = t1;
        }
    }
    // segments in job order (so a (window, block)'s segments are contiguous); CTA lists follow the same order
    std::vector<int> cta_of;
    for (size_t j = 0; j < (size_t)K * 3; ++j) {
        seg_first[j] = (int)segs.size();
        for (auto& s : per_job[j]) { cta_of.push_back(s.cta); segs.push_back(s); }
    }
    seg_first[(size_t)K * 3] = (int)segs.size();
    // cta ids are non-decreasing along the list
    int si = 0;
    for (int cc = 0; cc < grid; ++cc) {
        cta_first[cc] = si;
        while (si < (int)segs.size() && cta_of[si] == cc) ++si;
    }
    cta_first[grid] = (int)segs.size();
    p->g2_nseg = (int)segs.size();
    p->g2_raw_stride = (uint32_t)(((size_t)p->g2_blk[1].nbox * 128 + 1023) / 1024 * 1024);
    p->g2_mat_bytes = (uint32_t)(2 * Np * 16);
    p->g2_smem = 1024 + (size_t)G2_STAGES * p->g2_raw_stride + (size_t)(4 * G2_STAGES + 1) * p->g2_mat_bytes + sizeof(G2Bars) + 16 +
                 (size_t)(p->Nz + p->Nx) * sizeof(double);
    if (p->g2_smem > (size_t)p->smem_optin) return cudaErrorInvalidConfiguration;
    return set_max_dyn_smem(gram_tc2_kernel, p->smem_optin);
}

cudaError_t launch_gram_tc2(lcf_plan* p, const float2* iq, cudaStream_t st) {
    if (p->g2_nseg == 0) return cudaSuccess;
    const G2Maps* maps = g2_encode_maps(p, iq);
    if (!maps) return cudaErrorInvalidValue;
    G2Args a;
    a.N = p->N; a.Np = (p->N + 15) / 16 * 16; a.Nz = p->Nz; a.Nx = p->Nx;
    a.group = p->gtc_group;
    a.gz = p->gz_d; a.gx = p->gx_d; a.box = p->box_d; a.segs = p->g2_segs_d; a.cta_first = p->g2_cta_first_d;
    a.part = p->g2_part_d; a.raw_stride = p->g2_raw_stride; a.mat_bytes = p->g2_mat_bytes; a.amax = p->amax_d;
    for (int b = 0; b < 3; ++b) a.blk[b] = p->g2_blk[b];
    gram_tc2_kernel<<<p->g2_grid, G2_THREADS, p->g2_smem, st>>>(*maps, a);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    dim3 blk(16, 16), grid((p->N + 15) / 16, (p->N + 15) / 16, p->K);
    gram_tc2_reduce_kernel<<<grid, blk, 0, st>>>(p->g2_part_d, p->g2_seg_first_d, p->N, p->g2_c1, p->amax_d, reinterpret_cast<float2*>(p->R_d));
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Sliding-window reuse (packets in a sliding temporal window), N <= 128.
// If ensemble e+1 is ensemble e advanced by `s` frames, R_{e+1}[i][j] = R_e[i+s][j+s] for i, j < N - s: only the
// columns of the s new frames are computed -- one block job per window, rows [0,128) x columns [c0, Np),
// c0 = 16 floor((N - s) / 16), with the block-form kernel above -- and the rest is the previous R shifted (and
// rescaled by the exact power of two between the two ensembles' data scales).  R stays in the data scale of the
// tensor-core path (the Cholesky / cluster EVD kernels undo it).
__global__ void gram_stream_assemble_kernel(const float* part, const int* seg_first, int N, int s, int c0, const float2* Rprev,
                                            const uint32_t* amax_prev, const uint32_t* amax, float2* R) {
    const int k = blockIdx.z;
    const int i = blockIdx.y * 16 + threadIdx.y, j = blockIdx.x * 16 + threadIdx.x;
    if (i >= N || j >= N) return;
    const int a = i <= j ? i : j, b = i <= j ? j : i;          // the upper-triangle entry (a, b)
    float re, im;
    if (b < N - s) {
        const float2 v = Rprev[((size_t)k * N + (a + s)) * N + (b + s)];
        const float f = sm100::pow2f(2 * (sm100::pow2_scale_exp(*amax) - sm100::pow2_scale_exp(*amax_prev)));
        re = v.x * f; im = v.y * f;
    } else {
        double sr = 0.0, si = 0.0;
        for (int sg = seg_first[k]; sg < seg_first[k + 1]; ++sg) {
            const float* p = part + (size_t)sg * 2 * 128 * 128 + (size_t)a * 128 + (b - c0);
            sr += (double)p[0];
            si += (double)p[16384];
        }
        re = (float)sr; im = (float)si;
    }
    if (i == j) im = 0.f;
    if (i > j) im = -im;
    R[((size_t)k * N + i) * N + j] = make_float2(re, im);
}

bool gram_stream_eligible(const lcf_plan* p) { return p->gram_tc && p->N <= 128 && p->N >= 32 && g2_encode_fn() != nullptr; }

// one job per window, equal tile counts per CTA (the block is the same for every window)
cudaError_t configure_gram_stream(lcf_plan* p, std::vector<G2Seg>& segs, std::vector<int>& cta_first, std::vector<int>& seg_first) {
    const int K = p->K, N = p->N, Np = (N + 15) / 16 * 16;
    std::vector<long long> pre(K + 1, 0);
    for (int k = 0; k < K; ++k) {
        const WinBox& b = p->box_h[k];
        pre[k + 1] = pre[k] + (b.Pk > 0 ? (long long)((b.z0 + b.Lz - (b.z0 & ~1) + G2_PX - 1) / G2_PX) * b.Lx : 0);
    }
    const long long T = pre[K];
    int grid = (int)(T < p->num_sms ? T : p->num_sms);
    if (grid < 1) grid = 1;
    p->g2_grid = grid;
    segs.clear();
    cta_first.assign(grid + 1, 0);
    seg_first.assign(K + 1, 0);
    std::vector<int> cta_of;
    int k = 0;
    for (int c = 0; c < grid; ++c) {
        long long g0 = T * c / grid, g1 = T * (c + 1) / grid;
        while (g0 < g1) {
            while (k < K && pre[k + 1] <= g0) ++k;
            const long long e = pre[k + 1] < g1 ? pre[k + 1] : g1;
            segs.push_back({k, 0, (int)(g0 - pre[k]), (int)(e - g0), c});
            g0 = e;
        }
    }
    int si = 0;
    for (int c = 0; c < grid; ++c) { cta_first[c] = si; while (si < (int)segs.size() && segs[si].cta == c) ++si; }
    cta_first[grid] = (int)segs.size();
    si = 0;
    for (int kk = 0; kk < K; ++kk) { seg_first[kk] = si; while (si < (int)segs.size() && segs[si].k == kk) ++si; }
    seg_first[K] = si;
    p->g2_nseg = (int)segs.size();
    const int nbox = (N + 7) / 8 * 8;
    for (int b = 0; b < 3; ++b) p->g2_blk[b] = {0, 0, Np, 0, nbox};
    p->g2_raw_stride = (uint32_t)(((size_t)nbox * 128 + 1023) / 1024 * 1024);
    p->g2_mat_bytes = (uint32_t)(2 * Np * 16);
    p->g2_smem = 1024 + (size_t)G2_STAGES * p->g2_raw_stride + (size_t)(4 * G2_STAGES + 1) * p->g2_mat_bytes + sizeof(G2Bars) + 16 +
                 (size_t)(p->Nz + p->Nx) * sizeof(double);
    if (p->g2_smem > (size_t)p->smem_optin) return cudaErrorInvalidConfiguration;
    return set_max_dyn_smem(gram_tc2_kernel, p->smem_optin);
}

// R_d <- Gram of the ensemble at iq, given that the previous call's ensemble (whose R is in Rprev_d) was this one
// shifted back by `stride` frames
cudaError_t launch_gram_stream(lcf_plan* p, const float2* iq, int stride, cudaStream_t st) {
    const int N = p->N, Np = (N + 15) / 16 * 16;
    const G2Maps* maps = g2_encode_maps(p, iq);
    if (!maps) return cudaErrorInvalidValue;
    const int c0 = (N - stride) / 16 * 16;
    G2Args a;
    a.N = N; a.Np = Np; a.Nz = p->Nz; a.Nx = p->Nx;
    a.group = p->gtc_group;
    a.gz = p->gz_d; a.gx = p->gx_d; a.box = p->box_d; a.segs = p->g2_segs_d; a.cta_first = p->g2_cta_first_d;
    a.part = p->g2_part_d; a.raw_stride = p->g2_raw_stride; a.mat_bytes = p->g2_mat_bytes; a.amax = p->amax_d;
    for (int b = 0; b < 3; ++b) a.blk[b] = {0, c0, Np - c0, 0, p->g2_blk[0].nbox};
    if (p->g2_nseg > 0) {
        gram_tc2_kernel<<<p->g2_grid, G2_THREADS, p->g2_smem, st>>>(*maps, a);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
    }
    dim3 blk(16, 16), grid((N + 15) / 16, (N + 15) / 16, p->K);
    gram_stream_assemble_kernel<<<grid, blk, 0, st>>>(p->g2_part_d, p->g2_seg_first_d, N, stride, c0, p->Rprev_d, p->amax_prev_d, p->amax_d,
                                                       reinterpret_cast<float2*>(p->R_d));
    return cudaGetLastError();
}

}  // namespace lcf
