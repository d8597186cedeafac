// lcf_project_tc.cu -- kernel 4a, tensor-core path: fused projection + |.|^2 slow-time sum (Eq. 4,
// PAPER.md:57-63) on tcgen05 in fp16 split precision (three fp16 products per fp32 product), for N <= 256
// (above 128 frames the resident B block grows past 64 KB and the pipeline runs with 4 stages instead of 8).
//
//   U[p][u] = sum_t S[t][p] B_k[t][u],  B_k = V_k diag(wt)     PD_k(p) = w_k(p)^2 sum_u |U[p][u]|^2
//
// Real formulation.  Rows m of the A operand are the interleaved re/im samples of 64 pixels
// (m = 2p: Re S, m = 2p+1: Im S), K = frames, and one CTA works on a block of 64 eigen-columns u
// whose operand tile stays resident in shared memory for a whole segment:
//   B tile rows  [0,64) Re B hi   [64,128) Im B hi   [128,192) Re B lo   [192,256) Im B lo        (project_tc_kernel)
//   D[:, 0:256] += A_hi * B[0:256]^T        D[:, 0:128] += A_lo * B[0:128]^T        (two MMAs / 16 frames)
//   P_r[m][u] = D[m][u] + D[m][128+u] = X_m . Re B_u      P_i[m][u] = D[m][64+u] + D[m][192+u]
//   U_r = P_r[2p] - P_i[2p+1]      U_i = P_i[2p] + P_r[2p+1]
// Split precision on the FP16 tensor path (.kind::f16, twice the TF32 rate and half the operand
// bytes): every fp32 value x, scaled by a power of two, is hi + lo with hi = fp16(x) and
// lo = fp16(x - hi), 22 significant bits together; the products hi.hi + hi.lo + lo.hi are
// accumulated in fp32 and the lo.lo term (2^-22 of a term) is dropped.  The data are scaled so that
// max |S| lands in [256, 512) (absmax_kernel), B (entries <= 1 in modulus) by 256: lo then stays a
// normal fp16 number down to 2^-9 of the maximum and an absolute 2^-25 of it below.  Stacking B hi
// over B lo makes one N = 256 MMA do two of the three products.
//
// The ensemble is split ONCE per call into fp16 hi / lo planes (presplit_kernel) laid out so that a TMA box is a
// K-major A operand tile: the projection has no window weight inside its contraction, so the conversion is not
// repeated for each of the ~15 windows and 2-4 column blocks that read a pixel, and no converter warps exist.
//
// Persistent CTAs walk a static slice of the list of (window, column block group, 64-pixel tile) jobs,
// cut into segments at (window, group) changes.  Roles:
//   warp 0      producer: the segment's packed B tile (one bulk copy), then per 16 frames two TMA boxes
//               {16 z x 16 halves, 4 x, 2 chunks} of the hi and lo planes -> A_hi / A_lo of an operand stage;
//   warp 1      MMA issuer (uniform control flow, one elected lane);
//   epilogue    TMEM -> registers, pair exchange by shuffle, |U|^2 summed over the 64 columns, times w^2, one float
//               per (block, pixel); two accumulator buffers so the epilogue of a tile overlaps the MMAs of the next.
// project_tc2_kernel (two resident column blocks as one N = 256 operand, N <= 152) and project_tc_kernel (one block, its hi
// and lo rows as one N = 256 operand) differ in the resident tile and the TMEM layout only.  proj_tc_pack_kernel builds the
// B tiles from B_k; proj_tc_finish_kernel adds the column blocks into the per-window PD tiles and the per-chunk sums that
// the alpha / combine kernels use.
#include <cuda.h>
#include <cuda_fp16.h>
#include <cstring>

#include "lcf_internal.h"
#include "lcf_sm100.cuh"

namespace lcf {

using namespace sm100;

constexpr int PTC_TZ = 16, PTC_TX = 4;                     // pixel tile: 16 z x 4 x = 64 pixels = 128 rows
constexpr int PTC_ROWS = 128;
constexpr int PTC_KC = 16;                                 // frames per A stage
constexpr int PTC_UB = 64;                                 // eigen-columns per block
constexpr int PTC_OP_STAGES = 8;
constexpr int PTC_A_BYTES = PTC_KC * PTC_ROWS * 2;         // one of A_hi / A_lo per stage: 4 KB of fp16
constexpr int PTC_OP_BYTES = 2 * PTC_A_BYTES;
constexpr int PTC_A_LBO = PTC_ROWS * 16;                   // 2048: next 8-frame chunk of A
constexpr int PTC_B_LBO = 256 * 16;                        // 4096: next 8-frame chunk of B
constexpr int PTC_SBO = 128;
constexpr float PTC_B_SCALE = 256.f;
constexpr int PTC_EPI_WARPS = 4;
constexpr int PTC_FIRST_EPI = 12;                           // project_tc_kernel: warps 12-15 (warps 2-11 idle)
constexpr int PTC_THREADS = 32 * (PTC_FIRST_EPI + PTC_EPI_WARPS);

struct PtcArgs {
    int N, Kp, Nz, Nx;             // Kp = N rounded up to 16 frames
    const double* gz;              // [Kz][Nz]
    const double* gx;              // [Kx][Nx]
    const WinBox* box;
    const PtcSeg* segs;
    const int* cta_first;          // [grid+1]
    const float* bpack;            // [K][NB][Kp/8][256][8] fp16 (pointer in float units: 1024 floats per chunk)
    const uint32_t* amax;          // bits of max |S|
    int NB;
    float* part;                   // [NB][sum_k P_k]
    long long sumPk;
    int nstg;                      // operand stages in use
    // MAG variant (method 4, lcf_ncc.cu): B = V in rank order; instead of the power sum the epilogue writes
    // |u_i(p)| = w(p) |U[p][i]| / sigma_i  to  mag[(tile_off + q) * magN + rank]
    float* mag;
    int magN;
    const float* isig;             // [K][NB * 64]  1 / sigma by rank (0 beyond N or where sigma = 0)
};

struct PtcBars {
    uint64_t opfull[PTC_OP_STAGES], opempty[PTC_OP_STAGES];
    uint64_t accfull[2], accempty[2];
    uint64_t bfull, bfree;
    uint32_t tmem_base;
};

__device__ __forceinline__ float ptc_lds32(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void ptc_sts128(uint32_t addr, float x, float y, float z, float w) {
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}
__device__ __forceinline__ void ptc_sts128u(uint32_t addr, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
struct PtcMaps { CUtensorMap m[2]; };    // hi plane, lo plane

// MAG epilogue helper: val = Re U (even lane) / Im U (odd lane) of the pair's pixel for 16 eigen-columns.  The even lane
// returns |U| isig w of columns 0-7, the odd lane of columns 8-15 (each squares what it has, hands the partner the half it
// needs: 8 shuffles and 8 square roots per lane instead of 16 and 16); sqrt as v * rsqrt(v), 2 ulp.
__device__ __forceinline__ void ptc_mag8(const float (&val)[16], bool odd, const float* isg, float wpix, float (&s8)[8]) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const float lo2 = val[i] * val[i], hi2 = val[8 + i] * val[8 + i];
        const float v = (odd ? hi2 : lo2) + __shfl_xor_sync(0xffffffffu, odd ? lo2 : hi2, 1);
        s8[i] = (v > 1e-36f ? v * rsqrtf(v) : 0.f) * isg[(odd ? 8 : 0) + i] * wpix;
    }
}

template <bool MAG>
__global__ void __launch_bounds__(PTC_THREADS, 1) project_tc_kernel(const __grid_constant__ PtcMaps maps, PtcArgs a) {
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    unsigned char* sbase = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
    const uint32_t SMSK = (uint32_t)a.nstg - 1u, SSH = a.nstg == 8 ? 3u : 2u;           // operand stages in use: 8 (or 4)
    unsigned char* bsm = sbase;                                               // resident B block: Kp / 8 chunks of 4 KB
    unsigned char* ops = sbase + (size_t)(a.Kp / 8) * PTC_B_LBO;              // [stages][A_hi 4 KB | A_lo 4 KB]
    PtcBars* bars = reinterpret_cast<PtcBars*>(ops + a.nstg * PTC_OP_BYTES);
    double* gzs = reinterpret_cast<double*>(bars + 1);                        // [Nz] window table rows (epilogue only)
    double* gxs = gzs + a.Nz;                                                 // [Nx]
    float* isig_s = reinterpret_cast<float*>(gxs + a.Nx);                     // [64] (MAG) 1 / sigma of the segment's column block

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int seg0 = a.cta_first[blockIdx.x], seg1 = a.cta_first[blockIdx.x + 1];
    const int nst = (a.Kp + PTC_KC - 1) / PTC_KC;          // A stages per tile
    const uint32_t bbytes = (uint32_t)(a.Kp / 8) * 4096u;

    if (tid == 0) {
        for (int s = 0; s < PTC_OP_STAGES; ++s) { mbar_init(&bars->opfull[s], 1); mbar_init(&bars->opempty[s], 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(&bars->accfull[b], 1); mbar_init(&bars->accempty[b], PTC_EPI_WARPS); }
        mbar_init(&bars->bfull, 1);
        mbar_init(&bars->bfree, 1);
        mbar_fence_init();
    }
    if (warp == 1) tmem_alloc<512>(&bars->tmem_base);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = bars->tmem_base;

    if (warp == 0) {
        // =========================== producer ===========================
        if (lane == 0) { tma_prefetch_desc(&maps.m[0]); tma_prefetch_desc(&maps.m[1]); }
        uint32_t it = 0;
        for (int sg = seg0; sg < seg1; ++sg) {
            const PtcSeg seg = a.segs[sg];
            const WinBox bx = a.box[seg.k];
            const int ze = bx.z0 & ~1;                     // 16-byte aligned start of the TMA inner dimension
            const int ntz = (bx.z0 + bx.Lz - ze + PTC_TZ - 1) / PTC_TZ;
            if (sg > seg0) mbar_wait(&bars->bfree, (uint32_t)(sg - seg0 - 1) & 1);   // MMAs of the old block done
            if (lane == 0) {
                mbar_arrive_expect_tx(&bars->bfull, bbytes);
                bulk_load(bsm, a.bpack + ((size_t)seg.k * a.NB + seg.b) * (size_t)(a.Kp / 8) * 1024, bbytes, &bars->bfull);
            }
            for (int t = 0; t < seg.ntile; ++t) {
                const int tau = seg.tile0 + t;
                const int txi = tau / ntz, tzi = tau - txi * ntz;
                const int z = ze + tzi * PTC_TZ, x = bx.x0 + txi * PTC_TX;
                for (int st = 0; st < nst; ++st, ++it) {
                    const int s = (it & SMSK);
                    mbar_wait(&bars->opempty[s], ((it >> SSH) & 1) ^ 1);     // operand tiles straight from the pre-split planes
                    if (lane == 0) {
                        mbar_arrive_expect_tx(&bars->opfull[s], PTC_OP_BYTES);
                        tma_load_3d(ops + (size_t)s * PTC_OP_BYTES, &maps.m[0], 16 * z, x, 2 * st, &bars->opfull[s]);
                        tma_load_3d(ops + (size_t)s * PTC_OP_BYTES + PTC_A_BYTES, &maps.m[1], 16 * z, x, 2 * st, &bars->opfull[s]);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer ===========================
        const uint32_t idesc256 = make_idesc_f16(PTC_ROWS, 256, false, false);
        const uint32_t idesc128 = make_idesc_f16(PTC_ROWS, 128, false, false);
        const uint64_t descA0 = make_smem_desc(smem_u32(ops), PTC_A_LBO, PTC_SBO, SWZ_NONE);
        const uint64_t descB0 = make_smem_desc(smem_u32(bsm), PTC_B_LBO, PTC_SBO, SWZ_NONE);
        uint32_t it = 0, tl = 0;
        for (int sg = seg0; sg < seg1; ++sg) {
            const int nt = a.segs[sg].ntile;
            mbar_wait(&bars->bfull, (uint32_t)(sg - seg0) & 1);
            for (int t = 0; t < nt; ++t, ++tl) {
                const uint32_t buf = tl & 1;
                mbar_wait(&bars->accempty[buf], ((tl >> 1) & 1) ^ 1);
                const uint32_t tD = tmem + buf * 256;
                for (int st = 0; st < nst; ++st, ++it) {
                    const int o = (it & SMSK);
                    mbar_wait(&bars->opfull[o], (it >> SSH) & 1);
                    tc_fence_after_sync();
                    if (elect_one()) {
                        const uint64_t dAh = descA0 + (uint64_t)((o * PTC_OP_BYTES) >> 4);
                        const uint64_t dAl = dAh + (uint64_t)(PTC_A_BYTES >> 4);
                        const uint64_t dB = descB0 + (uint64_t)((st * 2 * PTC_B_LBO) >> 4);
                        mma_f16(tD, dAh, dB, idesc256, st == 0 ? 0u : 1u);
                        mma_f16(tD, dAl, dB, idesc128, 1u);
                        mma_commit(&bars->opempty[o]);
                        if (st + 1 == nst) mma_commit(&bars->accfull[buf]);
                    }
                    __syncwarp();
                }
            }
            if (elect_one()) mma_commit(&bars->bfree);     // every MMA that reads this B block has completed
            __syncwarp();
        }
    } else if (warp >= PTC_FIRST_EPI) {
        // =========================== epilogue ===========================
        const int quad = warp & 3;
        const uint32_t tlane = tmem + ((uint32_t)(quad * 32) << 16);
        const int m = quad * 32 + lane;
        const int pix = m >> 1, xi = pix >> 4, zi = pix & 15;
        // 1 / (data scale x B scale): exact power of two, applied to U before squaring
        const float unscale = pow2f(-8 - pow2_scale_exp(*a.amax));
        uint32_t tl = 0;
        int curk = -1;
        for (int sg = seg0; sg < seg1; ++sg) {
            const PtcSeg seg = a.segs[sg];
            const WinBox bx = a.box[seg.k];
            const int ze = bx.z0 & ~1;
            const int ntz = (bx.z0 + bx.Lz - ze + PTC_TZ - 1) / PTC_TZ;
            if (seg.k != curk) {
                asm volatile("bar.sync 1, 128;" ::: "memory");
                const int et = tid - PTC_FIRST_EPI * 32;
                for (int i = et; i < a.Nz; i += 128) gzs[i] = a.gz[(size_t)bx.kz * a.Nz + i];
                for (int i = et; i < a.Nx; i += 128) gxs[i] = a.gx[(size_t)bx.kx * a.Nx + i];
                asm volatile("bar.sync 1, 128;" ::: "memory");
                curk = seg.k;
            }
            if (MAG) {
                asm volatile("bar.sync 1, 128;" ::: "memory");
                const int et = tid - PTC_FIRST_EPI * 32;
                if (et < 64) isig_s[et] = a.isig[((size_t)seg.k * a.NB + seg.b) * 64 + et];
                asm volatile("bar.sync 1, 128;" ::: "memory");
            }
            float* out = a.part + (size_t)seg.b * a.sumPk + bx.tile_off;
            for (int t = 0; t < seg.ntile; ++t, ++tl) {
                const uint32_t buf = tl & 1;
                const int tau = seg.tile0 + t;
                const int txi = tau / ntz, tzi = tau - txi * ntz;
                const int zz = ze + tzi * PTC_TZ + zi, xx = bx.x0 + txi * PTC_TX + xi;
                mbar_wait(&bars->accfull[buf], (tl >> 1) & 1);
                tc_fence_after_sync();
                const bool valid = zz >= bx.z0 && zz < bx.z0 + bx.Lz && xx < bx.x0 + bx.Lx;
                float acc = 0.f;
                float wpix = 0.f;
                float* mrow = nullptr;
                if (MAG && valid) {
                    wpix = (float)(gzs[zz] * gxs[xx]);
                    mrow = a.mag + ((size_t)bx.tile_off + (size_t)(xx - bx.x0) * bx.Lz + (zz - bx.z0)) * a.magN + seg.b * PTC_UB;
                }
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    uint32_t va[16], vb[16], vc[16], vd[16];
                    const uint32_t col = buf * 256 + j * 16;
                    tmem_ld16(tlane + col, va);
                    tmem_ld16(tlane + col + 64, vb);
                    tmem_ld16(tlane + col + 128, vc);
                    tmem_ld16(tlane + col + 192, vd);
                    tmem_ld_wait();
                    float val[16];
#pragma unroll
                    for (int i = 0; i < 16; ++i) {
                        const float pr = __uint_as_float(va[i]) + __uint_as_float(vc[i]);
                        const float pi = __uint_as_float(vb[i]) + __uint_as_float(vd[i]);
                        const float po = __shfl_xor_sync(0xffffffffu, pi, 1);
                        val[i] = ((lane & 1) ? pr + po : pr - po) * unscale;   // odd row: Im U, even row: Re U
                        if (!MAG) acc = fmaf(val[i], val[i], acc);
                    }
                    if (MAG) {                               // the pair's even lane stores ranks 0-7 of the 16, the odd lane 8-15
                        const bool odd = (lane & 1) != 0;
                        float s8[8];
                        ptc_mag8(val, odd, isig_s + j * 16, wpix, s8);
                        if (valid) {
                            float4* o4 = reinterpret_cast<float4*>(mrow + j * 16 + (odd ? 8 : 0));
                            o4[0] = make_float4(s8[0], s8[1], s8[2], s8[3]);
                            o4[1] = make_float4(s8[4], s8[5], s8[6], s8[7]);
                        }
                    }
                }
                tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars->accempty[buf]);
                if (!MAG) {
                    acc += __shfl_xor_sync(0xffffffffu, acc, 1);
                    if (!(lane & 1) && valid) {
                        const double w = gzs[zz] * gxs[xx];
                        out[(size_t)(xx - bx.x0) * bx.Lz + (zz - bx.z0)] = (float)(w * w) * acc;
                    }
                }
            }
        }
    }
    tc_fence_before_sync();
    __syncthreads();
    if (warp == 1) tmem_dealloc<512>(tmem);
}

// ------------------------------------------------------------------------------------------------
// project_tc2_kernel: the pre-split projection with up to TWO 64-column blocks of B resident, both fed by the same
// A tiles.  project_tc_kernel re-reads every pixel once per (window, column block): 2.1 GB of L2 traffic per
// ensemble at config 2 (5 TB/s, ~60 % of what a plain read loop gets from L2 on this part) next to a
// shared-memory port that is already the bound.  Here a segment is a (window, block group) and per 16 frames
//   D_j[:, 0:128] += A_hi Bh_j^T       D_j += A_hi Bl_j^T       D_j += A_lo Bh_j^T          (j = 0, 1: three N = 128 MMAs each)
// with Bh_j / Bl_j the hi / lo halves (rows 0-127 / 128-255) of block j's resident tile: the lo products accumulate
// into the hi product's columns, so a block needs 128 TMEM columns instead of 256 and two blocks are double-buffered
// in the 512.  D_j[:, 0:64] = X . Re B, D_j[:, 64:128] = X . Im B.  Eight epilogue warps: two per TMEM lane quadrant,
// one per block.  Groups hold one block when two do not fit in shared memory next to the stages (N > 152).
constexpr int PT2_STAGES = 8;
constexpr int PT2_EPI0 = 8;                                    // warps 8-15: epilogue; 0: producer; 1: MMA issuer
struct Pt2Bars {
    uint64_t opfull[PT2_STAGES], opempty[PT2_STAGES];
    uint64_t accfull[2], accempty[2];
    uint64_t bfull, bfree;
    uint32_t tmem_base;
};

template <bool MAG>
__global__ void __launch_bounds__(PTC_THREADS, 1) project_tc2_kernel(const __grid_constant__ PtcMaps maps, PtcArgs a, int G) {
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    unsigned char* sbase = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
    const uint32_t bbytes = (uint32_t)(a.Kp / 8) * 2 * PTC_B_LBO;             // the resident group tile: 512 rows per chunk
    unsigned char* bsm = sbase;
    unsigned char* ops = sbase + bbytes;                                      // [STAGES][A_hi 4 KB | A_lo 4 KB]
    Pt2Bars* bars = reinterpret_cast<Pt2Bars*>(ops + PT2_STAGES * PTC_OP_BYTES);
    double* gzs = reinterpret_cast<double*>(bars + 1);
    double* gxs = gzs + a.Nz;
    float* isig_s = reinterpret_cast<float*>(gxs + a.Nx);                     // [2][64] (MAG)

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int seg0 = a.cta_first[blockIdx.x], seg1 = a.cta_first[blockIdx.x + 1];
    const int nst = (a.Kp + PTC_KC - 1) / PTC_KC;

    if (tid == 0) {
        for (int s = 0; s < PT2_STAGES; ++s) { mbar_init(&bars->opfull[s], 1); mbar_init(&bars->opempty[s], 1); }
        for (int b = 0; b < 2; ++b) { mbar_init(&bars->accfull[b], 1); mbar_init(&bars->accempty[b], 8); }
        mbar_init(&bars->bfull, 1);
        mbar_init(&bars->bfree, 1);
        mbar_fence_init();
    }
    if (warp == 1) tmem_alloc<512>(&bars->tmem_base);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = bars->tmem_base;

    if (warp == 0) {
        // =========================== producer ===========================
        if (lane == 0) { tma_prefetch_desc(&maps.m[0]); tma_prefetch_desc(&maps.m[1]); }
        uint32_t it = 0;
        for (int sg = seg0; sg < seg1; ++sg) {
            const PtcSeg seg = a.segs[sg];                 // seg.b = block group
            const WinBox bx = a.box[seg.k];
            const int nb = a.NB - seg.b * G < G ? a.NB - seg.b * G : G;
            const int ze = bx.z0 & ~1;
            const int ntz = (bx.z0 + bx.Lz - ze + PTC_TZ - 1) / PTC_TZ;
            if (sg > seg0) mbar_wait(&bars->bfree, (uint32_t)(sg - seg0 - 1) & 1);
            if (lane == 0) {
                mbar_arrive_expect_tx(&bars->bfull, bbytes);
                bulk_load(bsm, a.bpack + ((size_t)seg.k * ((a.NB + 1) / 2) + seg.b) * (size_t)(a.Kp / 8) * 2048, bbytes, &bars->bfull);
            }
            for (int t = 0; t < seg.ntile; ++t) {
                const int tau = seg.tile0 + t;
                const int txi = tau / ntz, tzi = tau - txi * ntz;
                const int z = ze + tzi * PTC_TZ, x = bx.x0 + txi * PTC_TX;
                for (int st = 0; st < nst; ++st, ++it) {
                    const int s = it % PT2_STAGES;
                    mbar_wait(&bars->opempty[s], ((it / PT2_STAGES) & 1) ^ 1);
                    if (lane == 0) {
                        mbar_arrive_expect_tx(&bars->opfull[s], PTC_OP_BYTES);
                        tma_load_3d(ops + (size_t)s * PTC_OP_BYTES, &maps.m[0], 16 * z, x, 2 * st, &bars->opfull[s]);
                        tma_load_3d(ops + (size_t)s * PTC_OP_BYTES + PTC_A_BYTES, &maps.m[1], 16 * z, x, 2 * st, &bars->opfull[s]);
                    }
                }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer ===========================
        const uint32_t idesc256 = make_idesc_f16(PTC_ROWS, 256, false, false), idesc128 = make_idesc_f16(PTC_ROWS, 128, false, false);
        const uint64_t descA0 = make_smem_desc(smem_u32(ops), PTC_A_LBO, PTC_SBO, SWZ_NONE);
        const uint64_t descB0 = make_smem_desc(smem_u32(bsm), 2 * PTC_B_LBO, PTC_SBO, SWZ_NONE);
        uint32_t it = 0, tl = 0;
        for (int sg = seg0; sg < seg1; ++sg) {
            const PtcSeg seg = a.segs[sg];
            const int nb = a.NB - seg.b * G < G ? a.NB - seg.b * G : G;
            mbar_wait(&bars->bfull, (uint32_t)(sg - seg0) & 1);
            for (int t = 0; t < seg.ntile; ++t, ++tl) {
                const uint32_t buf = tl & 1;
                mbar_wait(&bars->accempty[buf], ((tl >> 1) & 1) ^ 1);
                for (int st = 0; st < nst; ++st, ++it) {
                    const int o = it % PT2_STAGES;
                    mbar_wait(&bars->opfull[o], (it / PT2_STAGES) & 1);
                    tc_fence_after_sync();
                    if (elect_one()) {
                        const uint64_t dAh = descA0 + (uint64_t)((o * PTC_OP_BYTES) >> 4);
                        const uint64_t dAl = dAh + (uint64_t)(PTC_A_BYTES >> 4);
                        // both blocks at once: B rows [0,256) = hi of block 0 | hi of block 1, rows [256,512) = their lo halves
                        const uint32_t tD = tmem + buf * 256;
                        const uint32_t idesc = nb == 2 ? idesc256 : idesc128;
                        const uint64_t dBh = descB0 + (uint64_t)((st * 2 * 2 * PTC_B_LBO) >> 4);
                        const uint64_t dBl = dBh + (uint64_t)((256 * 16) >> 4);
                        mma_f16(tD, dAh, dBh, idesc, st == 0 ? 0u : 1u);
                        mma_f16(tD, dAh, dBl, idesc, 1u);
                        mma_f16(tD, dAl, dBh, idesc, 1u);
                        mma_commit(&bars->opempty[o]);
                        if (st + 1 == nst) mma_commit(&bars->accfull[buf]);
                    }
                    __syncwarp();
                }
            }
            if (elect_one()) mma_commit(&bars->bfree);
            __syncwarp();
        }
    } else if (warp >= PT2_EPI0) {
        // =========================== epilogue: warp (quadrant, block j of the group) ===========================
        const int quad = warp & 3, jb = (warp - PT2_EPI0) >> 2;
        const uint32_t tlane = tmem + ((uint32_t)(quad * 32) << 16);
        const int m = quad * 32 + lane;
        const int pix = m >> 1, xi = pix >> 4, zi = pix & 15;
        const float unscale = pow2f(-8 - pow2_scale_exp(*a.amax));
        uint32_t tl = 0;
        int curk = -1;
        for (int sg = seg0; sg < seg1; ++sg) {
            const PtcSeg seg = a.segs[sg];
            const WinBox bx = a.box[seg.k];
            const int nb = a.NB - seg.b * G < G ? a.NB - seg.b * G : G;
            const bool mine = jb < nb;
            const int blk = seg.b * G + jb;
            const int ze = bx.z0 & ~1;
            const int ntz = (bx.z0 + bx.Lz - ze + PTC_TZ - 1) / PTC_TZ;
            if (seg.k != curk || MAG) {
                asm volatile("bar.sync 1, 256;" ::: "memory");
                const int et = tid - PT2_EPI0 * 32;
                if (seg.k != curk) {
                    for (int i = et; i < a.Nz; i += 256) gzs[i] = a.gz[(size_t)bx.kz * a.Nz + i];
                    for (int i = et; i < a.Nx; i += 256) gxs[i] = a.gx[(size_t)bx.kx * a.Nx + i];
                }
                if (MAG && et < 128) isig_s[et] = (et >> 6) < nb ? a.isig[((size_t)seg.k * a.NB + seg.b * G + (et >> 6)) * 64 + (et & 63)] : 0.f;
                asm volatile("bar.sync 1, 256;" ::: "memory");
                curk = seg.k;
            }
            float* out = a.part + (size_t)(mine ? blk : 0) * a.sumPk + bx.tile_off;
            for (int t = 0; t < seg.ntile; ++t, ++tl) {
                const uint32_t buf = tl & 1;
                const int tau = seg.tile0 + t;
                const int txi = tau / ntz, tzi = tau - txi * ntz;
                const int zz = ze + tzi * PTC_TZ + zi, xx = bx.x0 + txi * PTC_TX + xi;
                mbar_wait(&bars->accfull[buf], (tl >> 1) & 1);
                tc_fence_after_sync();
                const bool valid = mine && zz >= bx.z0 && zz < bx.z0 + bx.Lz && xx < bx.x0 + bx.Lx;
                float acc = 0.f, wpix = 0.f;
                float* mrow = nullptr;
                if (MAG && valid) {
                    wpix = (float)(gzs[zz] * gxs[xx]);
                    mrow = a.mag + ((size_t)bx.tile_off + (size_t)(xx - bx.x0) * bx.Lz + (zz - bx.z0)) * a.magN + blk * PTC_UB;
                }
                if (mine) {
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        uint32_t va[16], vb[16];
                        const uint32_t col = buf * 256 + (uint32_t)jb * 128 + j * 16;
                        tmem_ld16(tlane + col, va);
                        tmem_ld16(tlane + col + 64, vb);
                        tmem_ld_wait();
                        float val[16];
#pragma unroll
                        for (int i = 0; i < 16; ++i) {
                            const float pr = __uint_as_float(va[i]), pi = __uint_as_float(vb[i]);
                            const float po = __shfl_xor_sync(0xffffffffu, pi, 1);
                            val[i] = ((lane & 1) ? pr + po : pr - po) * unscale;   // odd row: Im U, even row: Re U
                            if (!MAG) acc = fmaf(val[i], val[i], acc);
                        }
                        if (MAG) {
                            const bool odd = (lane & 1) != 0;
                            float s8[8];
                            ptc_mag8(val, odd, isig_s + jb * 64 + j * 16, wpix, s8);
                            if (valid) {
                                float4* o4 = reinterpret_cast<float4*>(mrow + j * 16 + (odd ? 8 : 0));
                                o4[0] = make_float4(s8[0], s8[1], s8[2], s8[3]);
                                o4[1] = make_float4(s8[4], s8[5], s8[6], s8[7]);
                            }
                        }
                    }
                }
                tc_fence_before_sync();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bars->accempty[buf]);
                if (!MAG && mine) {
                    acc += __shfl_xor_sync(0xffffffffu, acc, 1);
                    if (!(lane & 1) && valid) {
                        const double w = gzs[zz] * gxs[xx];
                        out[(size_t)(xx - bx.x0) * bx.Lz + (zz - bx.z0)] = (float)(w * w) * acc;
                    }
                }
            }
        }
    }
    tc_fence_before_sync();
    __syncthreads();
    if (warp == 1) tmem_dealloc<512>(tmem);
}

// B_k [N][Ns] complex (row = frame, column = eigen slot) -> per (window, 64-column block) the
// resident fp16 operand tile [Kp/8 chunks][256 rows][8 frames]: rows = Re hi | Im hi | Re lo | Im lo of 256 B
// GROUP2: two blocks share one tile of 512 rows per chunk, [hi b0 | hi b1 | lo b0 | lo b1] (128 rows each: Re 64, Im 64), so
// that project_tc2_kernel's MMAs take both blocks' hi (or lo) rows as one N = 256 operand.  `order` (rank -> slot)
// non-null: columns in rank order (method 4).
template <bool GROUP2>
__global__ void proj_tc_pack_kernel(const float2* B, const int* order, int N, int Ns, int Kp, int NB, float* bpack) {
    constexpr int ROWS = GROUP2 ? 512 : 256;
    const int NJ = GROUP2 ? (NB + 1) / 2 : NB;                                // tiles per window
    const int kb = blockIdx.x / (Kp / 8), c8 = blockIdx.x - kb * (Kp / 8);   // kb = k * NJ + tile; one 8-frame chunk per CTA
    const int k = kb / NJ, jt = kb - k * NJ;
    const float2* Bk = B + (size_t)k * N * Ns;
    uint4* out = reinterpret_cast<uint4*>(bpack + (size_t)kb * (Kp / 8) * (ROWS * 4)) + (size_t)c8 * ROWS;
    for (int r = threadIdx.x; r < ROWS; r += blockDim.x) {
        int b, col;
        bool im, lo;
        if (GROUP2) { const int part = r >> 7; b = jt * 2 + (part & 1); lo = part >= 2; im = (r >> 6) & 1; col = r & 63; }
        else { b = jt; lo = r >= 128; im = (r >> 6) & 1; col = r & 63; }
        const int cidx = b * PTC_UB + col;                                    // eigen slot, or rank
        int u = -1;
        if (b < NB) u = order ? (cidx < N ? order[(size_t)k * N + cidx] : -1) : (cidx < Ns ? cidx : -1);
        float x[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) {
            const int t = 8 * c8 + i;
            x[i] = 0.f;
            if (t < N && u >= 0) { const float2 c = Bk[(size_t)t * Ns + u]; x[i] = (im ? c.y : c.x) * PTC_B_SCALE; }
        }
        uint32_t h[4], l[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) f16_split2(x[2 * i], x[2 * i + 1], h[i], l[i]);
        out[r] = lo ? make_uint4(l[0], l[1], l[2], l[3]) : make_uint4(h[0], h[1], h[2], h[3]);
    }
}

// S -> fp16 hi / lo planes, scaled by the power of two of absmax_kernel, in the layout
//   [t8 = frame / 8][x][z][re, im][frame % 8]      (32 bytes per pixel and 8-frame chunk)
// so that the TMA box {16 z x 16 halves, 4 x, 2 chunks} lands in shared memory as the K-major A operand
// [chunk][row m = (x, z, re/im)][8 frames] of project_tc_kernel.  Frames >= N are zero.
__global__ void __launch_bounds__(256) presplit_kernel(const float2* iq, int N, int T8, long long P, const uint32_t* amax, uint4* sh, uint4* sl) {
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;        // (t8, pixel)
    if (e >= (long long)T8 * P) return;
    const long long pix = e % P;
    const int t8 = (int)(e / P);
    const float scale = pow2f(pow2_scale_exp(*amax));
    float re[8], im[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int t = 8 * t8 + i;
        float2 v = make_float2(0.f, 0.f);
        if (t < N) v = iq[(size_t)t * P + pix];
        re[i] = v.x * scale; im[i] = v.y * scale;
    }
    uint32_t h[8], l[8];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        f16_split2(re[2 * i], re[2 * i + 1], h[i], l[i]);
        f16_split2(im[2 * i], im[2 * i + 1], h[4 + i], l[4 + i]);
    }
    sh[2 * e] = make_uint4(h[0], h[1], h[2], h[3]); sh[2 * e + 1] = make_uint4(h[4], h[5], h[6], h[7]);
    sl[2 * e] = make_uint4(l[0], l[1], l[2], l[3]); sl[2 * e + 1] = make_uint4(l[4], l[5], l[6], l[7]);
}

// bits of max(|re|, |im|) over the ensemble (non-negative floats order like their bit patterns)
__global__ void absmax_kernel(const float4* x, size_t n4, const float* tail, int ntail, uint32_t* out) {
    float m = 0.f;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        const float4 v = __ldg(&x[i]);
        m = fmaxf(fmaxf(m, fmaxf(fabsf(v.x), fabsf(v.y))), fmaxf(fabsf(v.z), fabsf(v.w)));
    }
    if (blockIdx.x == 0 && (int)threadIdx.x < ntail) m = fmaxf(m, fabsf(tail[threadIdx.x]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
    __shared__ float ws[32];
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = m;
    __syncthreads();
    if (threadIdx.x < 32) {
        m = threadIdx.x < (blockDim.x >> 5) ? ws[threadIdx.x] : 0.f;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
        if (threadIdx.x == 0 && m == m) atomicMax(out, __float_as_uint(m));
    }
}

// PD_k tile = sum over the column blocks; per-chunk sums for alpha_kernel (same items as project_kernel)
__global__ void proj_tc_finish_kernel(const float* part, long long sumPk, int NB, const WinBox* box, const ProjItem* items,
                                      float* tiles, float* tsum) {
    const ProjItem it = items[blockIdx.x];
    const long long off = box[it.k].tile_off;
    const int q = it.q0 + threadIdx.x;
    float v = 0.f;
    if (q < it.q1) {
        for (int b = 0; b < NB; ++b) v += part[(size_t)b * sumPk + off + q];
        tiles[off + q] = v;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    __shared__ float ws[PROJ_TPIX / 32];
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        float t = 0.f;
        for (int w = 0; w < PROJ_TPIX / 32; ++w) t += ws[w];
        tsum[blockIdx.x] = t;
    }
}

// ---------------------------------------------------------------- host side
typedef CUresult (*PtcEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static PtcEncodeFn ptc_encode_fn() {
    static PtcEncodeFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<PtcEncodeFn>(p);
    }
    return fn;
}

// fp16 planes [T8][Nx][Nz * 16 halves]; box = {256 halves (16 z), 4 x, 2 chunks}, no swizzle
static bool ptc_encode_premaps(lcf_plan* p) {
    if (p->ptc_premaps_ready) return true;
    PtcEncodeFn fn = ptc_encode_fn();
    if (!fn || !p->ptc_sh_d || !p->ptc_sl_d) return false;
    void* planes[2] = {p->ptc_sh_d, p->ptc_sl_d};
    for (int i = 0; i < 2; ++i) {
        cuuint64_t dims[3] = {(cuuint64_t)p->Nz * 16, (cuuint64_t)p->Nx, (cuuint64_t)(p->ptc_Kp / 8)};
        cuuint64_t strides[2] = {(cuuint64_t)p->Nz * 32, (cuuint64_t)p->P * 32};
        cuuint32_t box[3] = {16 * PTC_TZ, PTC_TX, 2};
        cuuint32_t es[3] = {1, 1, 1};
        CUresult r = fn(reinterpret_cast<CUtensorMap*>(p->ptc_premaps) + i, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, planes[i], dims, strides, box, es,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return false;
    }
    p->ptc_premaps_ready = true;
    return true;
}

// the ensemble's fp16 hi / lo planes for the PRE variant (after absmax, before the projection)
cudaError_t launch_presplit(lcf_plan* p, const float2* iq, cudaStream_t st) {
    if (!p->ptc_pre) return cudaSuccess;
    const long long n = (long long)(p->ptc_Kp / 8) * p->P;
    presplit_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(iq, p->N, p->ptc_Kp / 8, p->P, p->amax_d, reinterpret_cast<uint4*>(p->ptc_sh_d),
                                                                  reinterpret_cast<uint4*>(p->ptc_sl_d));
    return cudaGetLastError();
}

// precision 1 projects in double (project_dd_kernel); its NCC modes still take the magnitude pass of method 4 from here
bool project_tc_eligible(const lcf_plan* p) {
    if (p->prec == 1 && !ncc_mode(p->thr.mode)) return false;
    return p->N <= 256 && p->N >= PTC_KC && (p->Nz % 2) == 0 && p->Nz >= PTC_TZ && p->Nx >= PTC_TX && ptc_encode_fn() != nullptr;
}

// jobs = (window, column block, tile) in that order; static contiguous slices, cut at (window, block)
cudaError_t configure_project_tc(lcf_plan* p, std::vector<PtcSeg>& segs, std::vector<int>& cta_first) {
    const int K = p->K;
    p->ptc_NB = (p->Ns + PTC_UB - 1) / PTC_UB;
    p->ptc_Kp = (p->N + 15) / 16 * 16;
    const int NB = p->ptc_NB;
    // block groups of the two-block kernel: two resident B blocks when they fit next to the stages
    const size_t bbytes = (size_t)(p->ptc_Kp / 8) * PTC_B_LBO;
    auto smem2 = [&](int G) {
        return (size_t)1024 + G * bbytes + (size_t)PT2_STAGES * PTC_OP_BYTES + sizeof(Pt2Bars) + 16 + (size_t)(p->Nz + p->Nx) * sizeof(double) +
               128 * sizeof(float);
    };
    int G = (NB >= 2 && smem2(2) <= (size_t)p->smem_optin) ? 2 : 1;
    if (smem2(G) > (size_t)p->smem_optin) return cudaErrorInvalidConfiguration;
    p->ptc_pre = true;
    p->ptc_G = G;
    p->ptc_nstg = PT2_STAGES;
    // one block per group (N > 152): project_tc_kernel's wide form (one N = 256 and one N = 128 MMA per 16 frames) reads
    // fewer operand bytes per flop than three N = 128 MMAs (measured at config 3: 4.0 against 4.95 ms)
    p->ptc_smem = G == 2 ? smem2(2)
                         : 1024 + bbytes + (size_t)p->ptc_nstg * PTC_OP_BYTES + sizeof(PtcBars) + 16 + (size_t)(p->Nz + p->Nx) * sizeof(double) + 64 * sizeof(float);
    if (p->ptc_smem > (size_t)p->smem_optin) return cudaErrorInvalidConfiguration;
    const int NG = (NB + G - 1) / G;
    // jobs = (window, block group, tile); a tile of a group costs as many units as the group has blocks
    std::vector<long long> pre((size_t)K * NG + 1, 0), ntile((size_t)K, 0);
    std::vector<int> wg((size_t)NG);
    for (int g = 0; g < NG; ++g) wg[g] = NB - g * G < G ? NB - g * G : G;
    for (int k = 0; k < K; ++k) {
        const WinBox& b = p->box_h[k];
        ntile[k] = b.Pk > 0 ? (long long)((b.z0 + b.Lz - (b.z0 & ~1) + PTC_TZ - 1) / PTC_TZ) * ((b.Lx + PTC_TX - 1) / PTC_TX) : 0;
        for (int g = 0; g < NG; ++g) pre[(size_t)k * NG + g + 1] = pre[(size_t)k * NG + g] + ntile[k] * wg[g];
    }
    const long long T = pre[(size_t)K * NG];
    long long total_tiles = 0;
    for (int k = 0; k < K; ++k) total_tiles += ntile[k] * NG;
    int grid = (int)(total_tiles < p->num_sms ? total_tiles : p->num_sms);
    if (grid < 1) grid = 1;
    p->ptc_grid = grid;
    segs.clear();
    cta_first.assign(grid + 1, 0);
    std::vector<int> cta_of;
    for (size_t j = 0; j < (size_t)K * NG; ++j) {
        const int k = (int)(j / NG), g = (int)(j % NG);
        const long long nt = ntile[k], w = wg[g];
        long long t0 = 0;
        while (t0 < nt) {                      // tile t starts at cost pre[j] + w t: it goes to the CTA whose equal share holds that point
            long long c = (pre[j] + w * t0) * grid / (T > 0 ? T : 1);
            if (c > grid - 1) c = grid - 1;
            long long t1 = nt;
            if (c < grid - 1) {
                const long long bound = (T * (c + 1) + grid - 1) / grid;          // first cost not in share c
                t1 = (bound - pre[j] + w - 1) / w;
                if (t1 <= t0) t1 = t0 + 1;
                if (t1 > nt) t1 = nt;
            }
            segs.push_back({k, g, (int)t0, (int)(t1 - t0)});
            cta_of.push_back((int)c);
            t0 = t1;
        }
    }
    int si = 0;
    for (int c = 0; c < grid; ++c) { cta_first[c] = si; while (si < (int)segs.size() && cta_of[si] <= c) ++si; }
    cta_first[grid] = (int)segs.size();
    p->ptc_nseg = (int)segs.size();
    cudaError_t e = set_max_dyn_smem(project_tc2_kernel<false>, p->smem_optin);
    if (e == cudaSuccess) e = set_max_dyn_smem(project_tc2_kernel<true>, p->smem_optin);
    if (e == cudaSuccess) e = set_max_dyn_smem(project_tc_kernel<false>, p->smem_optin);
    if (e == cudaSuccess) e = set_max_dyn_smem(project_tc_kernel<true>, p->smem_optin);
    return e;
}

static bool ptc_fill_maps(lcf_plan* p, const void*, PtcMaps& maps) {
    if (!ptc_encode_premaps(p)) return false;
    memcpy(&maps, p->ptc_premaps, sizeof(maps));
    return true;
}

static void ptc_launch_pack(lcf_plan* p, const int* order, cudaStream_t st) {
    if (p->ptc_G == 2)
        proj_tc_pack_kernel<true><<<p->K * ((p->ptc_NB + 1) / 2) * (p->ptc_Kp / 8), 256, 0, st>>>(p->B_d, order, p->N, p->Ns, p->ptc_Kp, p->ptc_NB, p->ptc_bpack_d);
    else
        proj_tc_pack_kernel<false><<<p->K * p->ptc_NB * (p->ptc_Kp / 8), 256, 0, st>>>(p->B_d, order, p->N, p->Ns, p->ptc_Kp, p->ptc_NB, p->ptc_bpack_d);
}

static void ptc_fill_args(lcf_plan* p, PtcArgs& a) {
    a.N = p->N; a.Kp = p->ptc_Kp; a.Nz = p->Nz; a.Nx = p->Nx;
    a.gz = p->gz_d; a.gx = p->gx_d; a.box = p->box_d; a.segs = p->ptc_segs_d; a.cta_first = p->ptc_cta_first_d;
    a.bpack = p->ptc_bpack_d; a.amax = p->amax_d; a.NB = p->ptc_NB; a.part = p->ptc_part_d; a.sumPk = p->sumPk; a.nstg = p->ptc_nstg;
    a.mag = nullptr; a.magN = 0; a.isig = nullptr;
}

cudaError_t launch_project_tc(lcf_plan* p, const float2* iq, cudaStream_t st) {
    if (p->ptc_nseg == 0 || p->n_pitems == 0) return cudaSuccess;
    PtcMaps maps;
    if (!ptc_fill_maps(p, iq, maps)) return cudaErrorInvalidValue;
    ptc_launch_pack(p, nullptr, st);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    PtcArgs a;
    ptc_fill_args(p, a);
    if (p->ptc_G == 2) project_tc2_kernel<false><<<p->ptc_grid, PTC_THREADS, p->ptc_smem, st>>>(maps, a, 2);
    else project_tc_kernel<false><<<p->ptc_grid, PTC_THREADS, p->ptc_smem, st>>>(maps, a);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    proj_tc_finish_kernel<<<p->n_pitems, PROJ_TPIX, 0, st>>>(p->ptc_part_d, p->sumPk, p->ptc_NB, p->box_d, p->pitems_d, p->tiles_d, p->tsum_d);
    return cudaGetLastError();
}

// Method 4 (lcf_ncc.cu): |u_i(p)| = w(p) |(s_p V)_i| / sigma_i for every pixel of every window, components in rank
// order, through the same tcgen05 pipeline (B_d must hold V, i.e. all eigen-weights 1).
cudaError_t launch_project_tc_mag(lcf_plan* p, const float2* iq, cudaStream_t st) {
    if (p->ptc_nseg == 0 || p->n_pitems == 0) return cudaSuccess;
    PtcMaps maps;
    if (!ptc_fill_maps(p, iq, maps)) return cudaErrorInvalidValue;
    ptc_launch_pack(p, p->order_d, st);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    PtcArgs a;
    ptc_fill_args(p, a);
    a.mag = p->ncc_mag_d; a.magN = p->ncc_magN; a.isig = p->ncc_isig_d;
    if (p->ptc_G == 2) project_tc2_kernel<true><<<p->ptc_grid, PTC_THREADS, p->ptc_smem, st>>>(maps, a, 2);
    else project_tc_kernel<true><<<p->ptc_grid, PTC_THREADS, p->ptc_smem, st>>>(maps, a);
    return cudaGetLastError();
}

// amax_d <- bits of the largest |re|, |im| of the ensemble (the tensor-core kernels scale by a power of two)
cudaError_t launch_absmax(lcf_plan* p, const float2* iq, cudaStream_t st) {
    cudaError_t e = cudaMemsetAsync(p->amax_d, 0, sizeof(uint32_t), st);
    if (e != cudaSuccess) return e;
    const size_t nf = (size_t)p->N * p->P * 2, n4 = nf / 4;
    absmax_kernel<<<p->num_sms * 4, 512, 0, st>>>(reinterpret_cast<const float4*>(iq), n4, reinterpret_cast<const float*>(iq) + n4 * 4,
                                                   (int)(nf - n4 * 4), p->amax_d);
    return cudaGetLastError();
}

}  // namespace lcf
