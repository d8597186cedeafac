// lcf_gram_tc.cu -- kernel 1, tensor-core path: batched window-weighted complex Gram (Eq. 12,
// PAPER.md:149-152) on tcgen05 in fp16 split precision (three fp16 products per fp32 product), for precision 0 and N <= 128.
//
//   R_k[i][j] = sum_p w_k(p)^2 conj(S[i][p]) S[j][p]            X = W_k S (Eq. 11), X = Xr + i Xi
//   Re R = Xr Xr^T + Xi Xi^T          Im R = G - G^T,  G = Xr Xi^T          (frames x frames, K = pixels)
//
// Every fp32 sample of X, scaled by a power of two so that max |S| lands in [256, 512)
// (absmax_kernel), is split x = hi + lo with hi = fp16(x), lo = fp16(x - hi) (22 significant bits
// together) for the FP16 tensor path (.kind::f16, K = 16 pixels = one tile per MMA), so
//   Re R = D0 + H + H^T      D0 = Rh Rh^T + Ih Ih^T        H = Rh Rl^T + Ih Il^T
//   Im R = (G0 + L) - (G0 + L)^T     G0 = Rh Ih^T          L = Rh Il^T - Ih Rl^T
// (the lo.lo products, 2^-22 of a term, are dropped).  The operand tiles are stacked, [Rh | Rl] and
// [Ih | Il] (hi rows, then the lo rows from row Np), so that three 128 x 2Np x 16 tcgen05.mma
// and one 128 x Np x 16 per 16 pixels do the seven products:
//   [D0 | H] += Rh^T [Rh | Rl]     [D0 | H] += Ih^T [Ih | Il]     [G0 | L] += Rh^T [Ih | Il]     L -= Ih^T Rl
// (an MMA with N = 2Np reads its A tile once for two products, and shared-memory bandwidth is what
// bounds this kernel).  Two TMEM accumulators of
// 2Np columns at columns 0 and 256.
//
// Persistent CTAs (one per SM) walk a static, contiguous slice of the global list of 16-pixel
// tiles (16 z-contiguous pixels of one window: one 128-byte row per frame), cut into segments at
// window boundaries.  Roles (640 threads, register file re-split with setmaxnreg):
//   warp 0       TMA producer: [N frames][16 px] complex64 box -> 128B-swizzled raw stage, plus the
//                16 window weights of the tile (window table rows staged in shared memory);
//   warp 1       MMA issuer: uniform control flow, one elected lane issues and commits;
//   warps 4-11   converters: raw stage -> w * s (f32x2) -> hi/lo -> four K-major operand tiles
//                (canonical no-swizzle core-matrix layout) -> fence.proxy.async -> mbarrier;
//   warps 12-19  accumulator drain (152 registers each): see below.
// tcgen05 accumulates in fp32 with truncation (measured: 2^24 + 1.5 -> 2^24), a bias that grows
// with the number of adds into a large running sum; D0 and G0 are therefore drained every
// `group` tiles (128 pixels = 32 adds) into fp32 registers of the drain warps (round to nearest)
// and zeroed there with tcgen05.st (the fused MMAs have one accumulate flag for D0 and H together),
// H and L (2^-11 of the main terms) stay in TMEM for the whole segment.  Each segment ends by
// writing two 128 x 128 fp32 partials (D0 / 2 + H and G0 + L); gram_tc_reduce_kernel sums a window's segments in fp64,
// applies the (anti)symmetrisation above and writes the full Hermitian R_k.
// Measured bound (clock64 per role, B200): the 128x128x8 MMA reads 8 KB of operands per 64 cycles,
// i.e. the whole 128 B/clk of shared-memory bandwidth, so the converter's and TMA's shared-memory
// traffic (64 KB per tile next to 112 KB of operand reads) stretches an MMA from 64 to ~105 cycles.
#include <cuda.h>

#include "lcf_internal.h"
#include "lcf_sm100.cuh"

namespace lcf {

using namespace sm100;

constexpr int GTC_PX = 16;                 // pixels per tile
constexpr int GTC_RT = 128;                // operand tile rows (frames, zero padded)
constexpr int GTC_RAW_STAGES = 6;
constexpr int GTC_OP_STAGES = 6;
constexpr int GTC_CONV_WARPS = 8;
constexpr int GTC_DRAIN_WARPS = 8;
constexpr int GTC_FIRST_CONV = 4;            // warps 0-3: TMA producer, MMA issuer, two idle (one warpgroup)
constexpr int GTC_FIRST_DRAIN = GTC_FIRST_CONV + GTC_CONV_WARPS;
constexpr int GTC_THREADS = 32 * (GTC_FIRST_DRAIN + GTC_DRAIN_WARPS);
constexpr int GTC_PAIR_BYTES = 2 * GTC_RT * GTC_PX * 2;  // one stacked fp16 operand (hi rows, then lo rows from row Np): 8 KB
constexpr int GTC_OP_BYTES = 2 * GTC_PAIR_BYTES;         // [Rh | Rl], [Ih | Il]
constexpr int GTC_LBO = 2 * GTC_RT * 16;                 // next 8-pixel K chunk (256 rows of 16 bytes)
constexpr int GTC_SBO = 128;                             // next 8-frame row group
constexpr int GTC_CONV_GROUPS = 2;           // converter groups working on alternate tiles
constexpr int GTC_WPG = GTC_CONV_WARPS / GTC_CONV_GROUPS;
// a group must see every use of the stages it touches (an mbarrier waiter may not skip a phase)
static_assert(GTC_RAW_STAGES % GTC_CONV_GROUPS == 0 && GTC_OP_STAGES % GTC_CONV_GROUPS == 0, "stages per group");

struct GtcArgs {
    int N, Np, Nz, Nx, Kz;
    int group;                 // tiles per D0/G0 drain
    const double* gz;          // [Kz][Nz]
    const double* gx;          // [Kx][Nx]
    const WinBox* box;
    const GtcSeg* segs;
    const int* cta_first;      // [grid+1]
    float* part;               // [nseg][2][128][128]
    uint32_t raw_stride;       // bytes between raw stages (multiple of 1024)
    const uint32_t* amax;      // bits of max |S| (power-of-two scaling of the fp16 operands)
};

struct GtcBars {
    uint64_t full[GTC_RAW_STAGES], empty[GTC_RAW_STAGES];
    uint64_t opfull[GTC_OP_STAGES], opempty[GTC_OP_STAGES];
    uint64_t accfull, accempty;
    uint32_t tmem_base;
    alignas(16) float wts[GTC_RAW_STAGES][2 * GTC_PX];   // each pixel weight twice: (w, w) pairs for f32x2
};

__device__ __forceinline__ void sts128(uint32_t addr, const float4& v) {
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w) : "memory");
}

__device__ __forceinline__ void sts128u(uint32_t addr, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(addr), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}

__device__ __forceinline__ ulonglong2 lds128u(uint32_t addr) {
    ulonglong2 v;
    asm volatile("ld.shared.v2.b64 {%0, %1}, [%2];" : "=l"(v.x), "=l"(v.y) : "r"(addr));
    return v;
}
// packed fp32 pair arithmetic (sm_100 f32x2 pipe): (a.x*b.x, a.y*b.y) and (a.x-b.x, a.y-b.y)
__device__ __forceinline__ float2 mul2(unsigned long long a, unsigned long long b) {
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    float2 f;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(f.x), "=f"(f.y) : "l"(r));
    return f;
}
__device__ __forceinline__ float2 sub2(float2 a, float2 b) {
    unsigned long long ua, ub, r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(ua) : "f"(a.x), "f"(a.y));
    asm("mov.b64 %0, {%1, %2};" : "=l"(ub) : "f"(b.x), "f"(b.y));
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(ua), "l"(ub));
    float2 f;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(f.x), "=f"(f.y) : "l"(r));
    return f;
}
__global__ void __launch_bounds__(GTC_THREADS, 1) gram_tc_kernel(const __grid_constant__ CUtensorMap tmap, GtcArgs a) {
    extern __shared__ __align__(1024) unsigned char smem_dyn[];
    unsigned char* sbase = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_dyn) + 1023) & ~(uintptr_t)1023);
    unsigned char* raw = sbase;                                               // [RAW_STAGES][raw_stride]
    unsigned char* ops = sbase + (size_t)GTC_RAW_STAGES * a.raw_stride;       // [OP_STAGES][GTC_OP_BYTES]
    GtcBars* bars = reinterpret_cast<GtcBars*>(ops + (size_t)GTC_OP_STAGES * GTC_OP_BYTES);
    double* gzs = reinterpret_cast<double*>(bars + 1);                        // [Nz] window table rows (producer only)
    double* gxs = gzs + a.Nz;                                                 // [Nx]

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int N = a.N;
    const int seg0 = a.cta_first[blockIdx.x], seg1 = a.cta_first[blockIdx.x + 1];

    // ---- one-time setup: zero the operand stages (rows >= N are never written), barriers, TMEM
    for (int i = tid * 16; i < GTC_OP_STAGES * GTC_OP_BYTES; i += GTC_THREADS * 16) *reinterpret_cast<uint4*>(ops + i) = make_uint4(0, 0, 0, 0);
    fence_proxy_async_smem();
    if (tid == 0) {
        for (int s = 0; s < GTC_RAW_STAGES; ++s) { mbar_init(&bars->full[s], 1); mbar_init(&bars->empty[s], GTC_WPG); }
        for (int s = 0; s < GTC_OP_STAGES; ++s) { mbar_init(&bars->opfull[s], GTC_WPG); mbar_init(&bars->opempty[s], 1); }
        mbar_init(&bars->accfull, 1);
        mbar_init(&bars->accempty, GTC_DRAIN_WARPS);
        mbar_fence_init();
    }
    if (warp == 1) tmem_alloc<512>(&bars->tmem_base);
    tc_fence_before_sync();
    __syncthreads();
    tc_fence_after_sync();
    const uint32_t tmem = bars->tmem_base;

    if (warp < GTC_FIRST_CONV) asm volatile("setmaxnreg.dec.sync.aligned.u32 32;");
    if (warp == 0) {
        // =========================== TMA producer ===========================
        if (lane == 0) tma_prefetch_desc(&tmap);
        const double scale = (double)pow2f(pow2_scale_exp(*a.amax));   // folded into the window weights
        uint32_t it = 0;
        for (int sg = seg0; sg < seg1; ++sg) {
            const GtcSeg seg = a.segs[sg];
            const WinBox bx = a.box[seg.k];
            const int ze = bx.z0 & ~1;    // TMA needs a 16-byte aligned start in the swizzled inner dimension
            const int ntz = (bx.z0 + bx.Lz - ze + GTC_PX - 1) / GTC_PX;
            // this window's separable table rows -> shared memory (one global round trip per segment,
            // not per tile: the producer's per-tile latency bounds the whole pipeline)
            __syncwarp();
            for (int i = lane; i < a.Nz; i += 32) gzs[i] = a.gz[(size_t)bx.kz * a.Nz + i];
            for (int i = lane; i < a.Nx; i += 32) gxs[i] = a.gx[(size_t)bx.kx * a.Nx + i];
            __syncwarp();
            for (int t = 0; t < seg.ntile; ++t, ++it) {
                const int s = it % GTC_RAW_STAGES;
                const uint32_t ph = (it / GTC_RAW_STAGES) & 1;
                const int tau = seg.tile0 + t;
                const int txi = tau / ntz, tzi = tau - txi * ntz;
                const int z = ze + tzi * GTC_PX, x = bx.x0 + txi;
                mbar_wait(&bars->empty[s], ph ^ 1);
                if (lane < GTC_PX) {
                    const int zz = z + lane;
                    float w = 0.f;
                    if (zz < a.Nz && x < a.Nx) w = (float)(gzs[zz] * gxs[x] * scale);
                    bars->wts[s][2 * lane] = w; bars->wts[s][2 * lane + 1] = w;
                }
                __syncwarp();
                if (lane == 0) {
                    mbar_arrive_expect_tx(&bars->full[s], (uint32_t)((N + 7) / 8 * 8) * 128u);
                    tma_load_3d(raw + (size_t)s * a.raw_stride, &tmap, 2 * z, x, 0, &bars->full[s]);
                }
            }
        }
    } else if (warp == 1) {
        // =========================== MMA issuer ===========================
        // the whole warp runs the loop (uniform control flow); one elected lane issues
        {
            const uint32_t idesc2 = make_idesc_f16(GTC_RT, 2 * a.Np, false, false);
            const uint32_t idesc_na = make_idesc_f16(GTC_RT, a.Np, true, false);
            const uint32_t tDH = tmem, tGL = tmem + 256;   // [D0 | H] and [G0 | L], each Np + Np columns
            // descriptor of the stacked operand [Rh | Rl], k-step 0 of stage 0; the others differ in the address field only
            const uint64_t desc0 = make_smem_desc(smem_u32(ops), GTC_LBO, GTC_SBO, SWZ_NONE);
            const uint64_t lo_off = (uint64_t)((a.Np * 16) >> 4);
            uint32_t it = 0, gc = 0;
            for (int sg = seg0; sg < seg1; ++sg) {
                const int nt = a.segs[sg].ntile;
                for (int t = 0; t < nt; ++t, ++it) {
                    const int o = it % GTC_OP_STAGES;
                    const uint32_t pho = (it / GTC_OP_STAGES) & 1;
                    const bool group_first = (t % a.group) == 0;
                    const bool group_last = ((t + 1) % a.group) == 0 || t + 1 == nt;
                    mbar_wait(&bars->opfull[o], pho);
                    if (group_first) mbar_wait(&bars->accempty, (gc & 1) ^ 1);
                    tc_fence_after_sync();
                    if (elect_one()) {
                        const uint64_t dst = desc0 + (uint64_t)((o * GTC_OP_BYTES) >> 4);
                        const uint64_t dR = dst;                                           // [Rh | Rl], K = the tile's 16 pixels
                        const uint64_t dI = dst + (uint64_t)(GTC_PAIR_BYTES >> 4);         // [Ih | Il]
                        const uint32_t accs = (t == 0) ? 0u : 1u;   // everything restarts per segment;
                        // D0 and G0 are zeroed by the drain warps at group ends (a fused MMA has one flag)
                        mma_f16(tDH, dR, dR, idesc2, accs);                   // Rh^T [Rh | Rl]
                        mma_f16(tDH, dI, dI, idesc2, 1u);                     // Ih^T [Ih | Il]
                        mma_f16(tGL, dR, dI, idesc2, accs);                   // Rh^T [Ih | Il]
                        mma_f16(tGL + (uint32_t)a.Np, dI, dR + lo_off, idesc_na, 1u);   // L -= Ih^T Rl
                        mma_commit(&bars->opempty[o]);
                        if (group_last) mma_commit(&bars->accfull);
                    }
                    __syncwarp();
                    if (group_last) ++gc;
                }
            }
        }
    } else if (warp >= GTC_FIRST_CONV && warp < GTC_FIRST_DRAIN) {
        // =========================== converters ===========================
        asm volatile("setmaxnreg.dec.sync.aligned.u32 72;");
        const int cw = warp - GTC_FIRST_CONV;         // 0..7
        // this thread's tasks per tile: (4-pixel chunk c4, frame fr); offsets are the same for every tile
        const int nwt = 2 * ((N + 31) / 32);          // warp tasks per tile: (8-pixel chunk, 32-frame block)
        const uint32_t lo_bytes = (uint32_t)a.Np * 16u;
        const uint32_t raw_u32 = smem_u32(raw), ops_u32 = smem_u32(ops), wts_u32 = smem_u32(&bars->wts[0][0]);
        // The converter warps form GTC_CONV_GROUPS groups that take alternate tiles, so that one
        // group's load -> convert -> store -> fence latency overlaps the other's; a warp walks its
        // tasks of a tile one after the other (same registers as one task).
        const int grp = cw / GTC_WPG, gw = cw % GTC_WPG;
        uint32_t it = 0;
        for (int sg = seg0; sg < seg1; ++sg) {
            const int nt = a.segs[sg].ntile;
            for (int t = 0; t < nt; ++t, ++it) {
                if ((int)(it % GTC_CONV_GROUPS) != grp) continue;
                const int s = it % GTC_RAW_STAGES, o = it % GTC_OP_STAGES;
                const uint32_t ph = (it / GTC_RAW_STAGES) & 1, pho = (it / GTC_OP_STAGES) & 1;
                const uint32_t rs = raw_u32 + (uint32_t)s * a.raw_stride;
                const uint32_t os = ops_u32 + (uint32_t)o * GTC_OP_BYTES;
                const uint32_t ws = wts_u32 + (uint32_t)s * (GTC_PX * 8);
                mbar_wait(&bars->full[s], ph);
                mbar_wait(&bars->opempty[o], pho ^ 1);
#pragma unroll 1
                for (int wt = gw; wt < nwt; wt += GTC_WPG) {
                    const int c8 = wt & 1, fr = (wt >> 1) * 32 + lane;
                    if (fr < N) {
                        const uint32_t sw = (uint32_t)(fr & 7);
                        ulonglong2 wq[4], pq[4];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            wq[u] = lds128u(ws + (uint32_t)c8 * 64u + 16 * u);                                        // (w0, w0), (w1, w1) of pixels 2u, 2u+1 of the chunk
                            pq[u] = lds128u(rs + (uint32_t)fr * 128u + ((((uint32_t)(4 * c8 + u)) ^ sw) << 4));      // (re0, im0), (re1, im1)
                        }
                        uint32_t rh[4], rl[4], ih[4], il[4];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            const float2 v0 = mul2(pq[u].x, wq[u].x), v1 = mul2(pq[u].y, wq[u].y);
                            f16_split2(v0.x, v1.x, rh[u], rl[u]);
                            f16_split2(v0.y, v1.y, ih[u], il[u]);
                        }
                        const uint32_t dst = os + (uint32_t)c8 * GTC_LBO + (uint32_t)fr * 16u;      // hi row; the lo row is Np rows further
                        sts128u(dst, rh[0], rh[1], rh[2], rh[3]);
                        sts128u(dst + GTC_PAIR_BYTES, ih[0], ih[1], ih[2], ih[3]);
                        sts128u(dst + lo_bytes, rl[0], rl[1], rl[2], rl[3]);
                        sts128u(dst + GTC_PAIR_BYTES + lo_bytes, il[0], il[1], il[2], il[3]);
                    }
                }
                fence_proxy_async_smem();             // this lane's operand writes -> async proxy
                __syncwarp();
                if (lane == 0) {                      // one arrival per converter warp of the group on each barrier
                    mbar_arrive(&bars->empty[s]);     // raw stage (and its weights) consumed
                    mbar_arrive(&bars->opfull[o]);
                }
            }
        }
    } else if (warp >= GTC_FIRST_DRAIN) {
        // =========================== accumulator drain ===========================
        asm volatile("setmaxnreg.inc.sync.aligned.u32 152;");
        const int dw = warp - GTC_FIRST_DRAIN;        // 0..7
        const int quad = warp & 3;                    // TMEM lane quadrant this warp may touch
        const int half = dw >> 2;                     // which 64 columns of D0 / G0 this warp keeps
        const uint32_t tlane = tmem + ((uint32_t)(quad * 32) << 16);
        const int row = quad * 32 + lane;
        float acc[128];
#pragma unroll
        for (int i = 0; i < 128; ++i) acc[i] = 0.f;
        uint32_t gc = 0;
        for (int sg = seg0; sg < seg1; ++sg) {
            const int nt = a.segs[sg].ntile;
            const int ngroups = (nt + a.group - 1) / a.group;
            for (int g = 0; g < ngroups; ++g) {
                // D0, G0 of the finished group -> registers (round-to-nearest adds)
                mbar_wait(&bars->accfull, gc & 1);
                tc_fence_after_sync();
#pragma unroll
                for (int blk = 0; blk < 8; ++blk) {
                    const int cj = half * 64 + (blk & 3) * 16;             // column inside D0 (blk < 4) / G0
                    if (cj < a.Np) {
                        uint32_t v[16];
                        tmem_ld16(tlane + (blk < 4 ? 0u : 256u) + (uint32_t)cj, v);
                        tmem_ld_wait();
#pragma unroll
                        for (int j = 0; j < 16; ++j) acc[blk * 16 + j] += __uint_as_float(v[j]);
                    }
                }
                if (g + 1 < ngroups) {
                    // the next group accumulates onto zeros again (H and L next to them keep running)
#pragma unroll
                    for (int blk = 0; blk < 8; ++blk) {
                        const int cj = half * 64 + (blk & 3) * 16;
                        if (cj < a.Np) tmem_st16_zero(tlane + (blk < 4 ? 0u : 256u) + (uint32_t)cj);
                    }
                    tmem_st_wait();
                    tc_fence_before_sync();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&bars->accempty);   // one arrival per drain warp
                    ++gc;
                }
            }
            // ---- segment end: the two partials of this segment, P0 = D0 / 2 + H and P1 = G0 + L
            // (Re R = P0 + P0^T since D0 is symmetric, Im R = P1 - P1^T)
            float* out = a.part + (size_t)sg * 2 * 128 * 128 + (size_t)row * 128 + half * 64;
#pragma unroll
            for (int blk = 0; blk < 8; ++blk) {
                const int m = blk >> 2;                                    // 0: D0 with H, 1: G0 with L
                const int cj = half * 64 + (blk & 3) * 16;
                if (cj < a.Np) {
                    uint32_t v[16];
                    tmem_ld16(tlane + (blk < 4 ? 0u : 256u) + (uint32_t)(a.Np + cj), v);
                    tmem_ld_wait();
                    const float sc = m == 0 ? 0.5f : 1.f;
                    float* o2 = out + (size_t)m * 128 * 128 + (blk & 3) * 16;
#pragma unroll
                    for (int j = 0; j < 16; j += 4)
                        *reinterpret_cast<float4*>(o2 + j) = make_float4(fmaf(sc, acc[blk * 16 + j], __uint_as_float(v[j])),
                                                                         fmaf(sc, acc[blk * 16 + j + 1], __uint_as_float(v[j + 1])),
                                                                         fmaf(sc, acc[blk * 16 + j + 2], __uint_as_float(v[j + 2])),
                                                                         fmaf(sc, acc[blk * 16 + j + 3], __uint_as_float(v[j + 3])));
                }
            }
#pragma unroll
            for (int i = 0; i < 128; ++i) acc[i] = 0.f;
            tc_fence_before_sync();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bars->accempty);
            ++gc;
        }
    }
    tc_fence_before_sync();
    __syncthreads();
    if (warp == 1) tmem_dealloc<512>(tmem);
}

// R_k = sum over the window's segments, in fp64:  Re R = P0 + P0^T,  Im R = P1 - P1^T  (P0 = D0 / 2 + H, P1 = G0 + L).
// R_k stays in the power-of-two data scale (squared): the fp32 EVD then works on numbers of a fixed
// magnitude whatever the units of the input; the EVD kernels unscale the eigenvalues, lcf_get_gram R.
// One 16 x 16 tile of R per CTA; the transposed tile comes through shared memory so that both reads
// of the partials are coalesced.
template <typename T>
__global__ void gram_tc_reduce_kernel(const float* part, const int* seg_first, int N, void* Rv) {
    __shared__ float t0[16][17], t1[16][17];
    const int k = blockIdx.z, tx = threadIdx.x, ty = threadIdx.y;
    const int i0 = blockIdx.y * 16, j0 = blockIdx.x * 16;
    const int i = i0 + ty, j = j0 + tx;
    double re = 0.0, im = 0.0;
    for (int s = seg_first[k]; s < seg_first[k + 1]; ++s) {
        const float* p = part + (size_t)s * 2 * 128 * 128;
        const size_t ij = (size_t)i * 128 + j, tr = (size_t)(j0 + ty) * 128 + (i0 + tx);   // rows < 128 always exist
        const float a0 = p[ij], a1 = p[16384 + ij];
        __syncthreads();
        t0[ty][tx] = p[tr];
        t1[ty][tx] = p[16384 + tr];
        __syncthreads();
        re += (double)a0 + (double)t0[tx][ty];          // P0[i][j] + P0[j][i]
        im += (double)a1 - (double)t1[tx][ty];
    }
    if (i >= N || j >= N) return;
    if (i == j) im = 0.0;
    if (sizeof(T) == 4) {
        float2* R = reinterpret_cast<float2*>(Rv) + (size_t)k * N * N;
        R[(size_t)i * N + j] = make_float2((float)re, (float)im);
    } else {
        double2* R = reinterpret_cast<double2*>(Rv) + (size_t)k * N * N;
        R[(size_t)i * N + j] = make_double2(re, im);
    }
}

// ---------------------------------------------------------------- host side
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// [N][Nx][Nz] complex64 seen as float [N][Nx][2 Nz]; box = 16 pixels x 1 x N frames, 128B swizzle
static const CUtensorMap* encode_iq_map(lcf_plan* p, const void* iq) {
    if (const unsigned char* m = p->gtc_tmaps.find(iq)) return reinterpret_cast<const CUtensorMap*>(m);
    EncodeTiledFn fn = encode_fn();
    if (!fn) return nullptr;
    unsigned char* slot = p->gtc_tmaps.slot(iq);
    cuuint64_t dims[3] = {(cuuint64_t)2 * p->Nz, (cuuint64_t)p->Nx, (cuuint64_t)p->N};
    cuuint64_t strides[2] = {(cuuint64_t)p->Nz * 8, (cuuint64_t)p->P * 8};
    cuuint32_t box[3] = {2 * GTC_PX, 1, (cuuint32_t)((p->N + 7) / 8 * 8)};   // whole 1024-byte swizzle atoms; frames >= N are zero-filled
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = fn(reinterpret_cast<CUtensorMap*>(slot), CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<void*>(iq), dims,
                    strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { p->gtc_tmaps.drop_last(iq); return nullptr; }
    return reinterpret_cast<const CUtensorMap*>(slot);
}

bool gram_tc_eligible(const lcf_plan* p) {
    return p->prec == 0 && p->N <= 128 && p->N >= 2 && (p->Nz % 2) == 0 && encode_fn() != nullptr;
}

// work decomposition: static contiguous slices of the global tile list, cut at window boundaries
cudaError_t configure_gram_tc(lcf_plan* p, std::vector<GtcSeg>& segs, std::vector<int>& cta_first, std::vector<int>& seg_first) {
    const int K = p->K;
    std::vector<long long> nt(K);
    long long T = 0;
    for (int k = 0; k < K; ++k) {
        const WinBox& b = p->box_h[k];
        nt[k] = b.Pk > 0 ? (long long)((b.z0 + b.Lz - (b.z0 & ~1) + GTC_PX - 1) / GTC_PX) * b.Lx : 0;
        T += nt[k];
    }
    int grid = (int)(T < p->num_sms ? T : p->num_sms);
    if (grid < 1) grid = 1;
    p->gtc_grid = grid;
    segs.clear();
    cta_first.assign(grid + 1, 0);
    seg_first.assign(K + 1, 0);
    // global tile g in [0,T): window by prefix sums
    std::vector<long long> pre(K + 1, 0);
    for (int k = 0; k < K; ++k) pre[k + 1] = pre[k] + nt[k];
    std::vector<std::vector<GtcSeg>> per_cta(grid);
    for (int b = 0; b < grid; ++b) {
        long long g0 = T * b / grid, g1 = T * (b + 1) / grid;
        int k = 0;
        while (g0 < g1) {
            while (k < K && pre[k + 1] <= g0) ++k;
            long long e = pre[k + 1] < g1 ? pre[k + 1] : g1;
            per_cta[b].push_back({k, (int)(g0 - pre[k]), (int)(e - g0), 0});
            g0 = e;
        }
    }
    for (int b = 0; b < grid; ++b) {
        cta_first[b] = (int)segs.size();
        for (auto& s : per_cta[b]) segs.push_back(s);
    }
    cta_first[grid] = (int)segs.size();
    // segments are in global tile order, so each window's segments are contiguous
    int si = 0;
    for (int k = 0; k < K; ++k) {
        seg_first[k] = si;
        while (si < (int)segs.size() && segs[si].k == k) ++si;
    }
    seg_first[K] = si;
    p->gtc_nseg = (int)segs.size();
    p->gtc_raw_stride = (uint32_t)(((size_t)p->N * 128 + 1023) / 1024 * 1024);
    p->gtc_smem = 1024 + (size_t)GTC_RAW_STAGES * p->gtc_raw_stride + (size_t)GTC_OP_STAGES * GTC_OP_BYTES + sizeof(GtcBars) +
                  (size_t)(p->Nz + p->Nx) * sizeof(double);
    if (p->gtc_smem > (size_t)p->smem_optin) return cudaErrorInvalidConfiguration;
    return set_max_dyn_smem(gram_tc_kernel, p->smem_optin);
}

cudaError_t launch_gram_tc(lcf_plan* p, const float2* iq, cudaStream_t st) {
    if (p->gtc_nseg == 0) return cudaSuccess;
    const CUtensorMap* tmap = encode_iq_map(p, iq);
    if (!tmap) return cudaErrorInvalidValue;
    GtcArgs a;
    a.N = p->N; a.Np = (p->N + 15) / 16 * 16; a.Nz = p->Nz; a.Nx = p->Nx; a.Kz = p->Kz;
    a.group = p->gtc_group;
    a.gz = p->gz_d; a.gx = p->gx_d; a.box = p->box_d; a.segs = p->gtc_segs_d; a.cta_first = p->gtc_cta_first_d;
    a.part = p->gtc_part_d; a.raw_stride = p->gtc_raw_stride; a.amax = p->amax_d;
    gram_tc_kernel<<<p->gtc_grid, GTC_THREADS, p->gtc_smem, st>>>(*tmap, a);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    dim3 blk(16, 16), grid((p->N + 15) / 16, (p->N + 15) / 16, p->K);
    gram_tc_reduce_kernel<float><<<grid, blk, 0, st>>>(p->gtc_part_d, p->gtc_seg_first_d, p->N, p->R_d);
    return cudaGetLastError();
}

}  // namespace lcf
