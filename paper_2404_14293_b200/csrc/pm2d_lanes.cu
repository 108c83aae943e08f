// pm2d_lanes.cu -- the LANE storage order and its fused gather + push + deposit kernel (sm_100a).
//
// Why.  A thread-per-particle stage kernel issues, per particle and stage, 9 LDS.64 (gather, Eq. 15) and 9 x 3
// shared atomics (deposit, Eq. 14).  A warp-wide shared access costs as many wavefronts as lanes collide on a bank,
// and with one copy of the windows the bank of a node is its column: lanes whose particles sit in neighbouring cells
// collide as soon as one rounds up to its nearest node and the next one down -- 2.3 wavefronts per atomic measured on
// the layered order (profiles/r01i), which made the shared-memory pipe the limiter.
//
// The lane order removes the collisions by construction.  Inside a sub-tile (32 columns x 16 or 32 cell rows) the
// particles are ranked by y and cut into 32 slabs of equal population; slab i is what lane i works on.  Slot =
// 32 * w + i for the w-th particle (in x order) of slab i, so a warp holds one particle of every slab, and with the
// uniform loading of the paper's set-ups slab i is cell column i to within a fraction of a cell.  Lane i always
// uses bank i + b (b = 0..2 the footprint column): the windows are kept in NCOPY copies, copy m holding node column
// c at index t = c - m + 1, and a particle whose nearest node column is cy takes copy m = cy - i.  With four copies
// (m = -1..2) a particle may sit up to 1.5 cells outside its slab before it leaves the fast path -- a 3 keV electron
// needs more than a rebin period of 16 steps for that (0.5 % of the visits, measured by pm2d_stray_count).  Such
// strays, and particles hotter than the range of the float -> int trick below, are listed and served after the
// main loop on the same windows with a copy chosen per node (conflicts allowed), or by k_stage_overflow on the
// global grids when they left the window.  Every route adds the same integers, so the grids do not depend on it.
//
// float -> int without the XU pipe: the windows count in units of 2^sn (density) resp. 2^sp (momentum) global
// units, chosen so that a single contribution stays below 2^22; then fma(weight, q, 1.5 * 2^23) has the rounded
// integer in its mantissa (one FFMA + one integer subtract instead of FMUL + F2I; F2I issues at 16 lanes per clock
// and SM, measured 2.0 cycles per warp instruction against 0.27 for FFMA).
#include <algorithm>
#include <cmath>

#include <cuda.h>

#include "pm2d_particle_dev.cuh"

namespace {

constexpr int LT = 34;                      // window columns per copy: t = lane + b, lane < 32, b < 3
constexpr int LFP = 48;                     // force-window pitch in float2: a multiple of 16 (LDS.64 runs in half-warps)
#ifndef LANES_NT_HOT
#define LANES_NT_HOT 384
#endif
#ifndef LANES_NT_COLD
#define LANES_NT_COLD 256
#endif
#ifndef LANES_MINB_HOT
#define LANES_MINB_HOT 3
#endif
#ifndef LANES_MINB_COLD
#define LANES_MINB_COLD 3
#endif
// Flush of interior windows by cp.reduce.async.bulk (one bulk integer reduction per window row and quantity) instead of
// one RED per node.  Measured on c3 (r02h): stage kernels 5.16 ms per step against 4.94 with plain REDs -- a CTA has to
// wait for its bulk reductions to have read shared memory before it may exit, while REDs are fire and forget; off.
constexpr bool LANES_BULK_FLUSH = false;
// Where the listed strays are served: by the CTA itself on its shared windows (one particle per thread after the main
// loop: the whole CTA waits a full particle latency for a handful of strays), or by k_lanes_overflow on the global grids.
constexpr bool LANES_STRAYS_IN_CTA = true;     // the global route measured 5.19 against 4.85 ms of stage kernels on c3 (r02n)
// A box load must start on a 16-byte boundary of the global row, i.e. on an even column of float2: with the odd-shift
// copies as box loads of their own the kernel dies with "an illegal instruction was encountered" (tried, r02p).  The even
// copies are box loads, the odd ones shifted duplicates made in shared memory.
// A CTA asks L2 for the particle records and the force window of the CTA that will run LANES_PF_DIST blocks later (about
// one generation of resident CTAs: 3 per SM), three bulk prefetches and one box prefetch by one thread: r02b had 26 % of the
// warp samples waiting on the particle loads (long scoreboard) with the records of one round loaded one round ahead.
#ifndef LANES_PF_DIST
#define LANES_PF_DIST 444
#endif
// The deposit windows are zeroed by one bulk-async copy from a block of zeros in the workspace (L2-resident) instead of
// STS.128 by the threads: the copy engine's writes do not pass the LSU data pipe, which bounds this kernel.
#ifndef LANES_TMA_ZERO
#define LANES_TMA_ZERO 1
#endif
constexpr int LSTRAY = 256;                 // stray list of a CTA (a full list spills to the global overflow list)
constexpr uint32_t LSTRAY_DEP = 0x80000000u;
constexpr float MAGIC = 12582912.0f;        // 1.5 * 2^23
constexpr int MAGIC_BITS = 0x4B400000;

// ---- bulk-async copies (TMA): the force window of an interior sub-tile is NCOPY box loads of one tensor map ------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@!p bra WAIT_%=;\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void bulk_load(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)), "l"(src),
                 "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void tma_load_2d(void *dst, const CUtensorMap *tm, int c0, int c1, uint64_t *bar)
{
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(smem_u32(dst)),
                 "l"(tm), "r"(c0), "r"(c1), "r"(smem_u32(bar))
                 : "memory");
}

// shared -> global bulk reduction (integer add) of `bytes` contiguous bytes, 16-byte aligned on both sides
__device__ __forceinline__ void bulk_reduce_add_s32(int32_t *gdst, const int32_t *ssrc, uint32_t bytes)
{
    asm volatile("cp.reduce.async.bulk.global.shared::cta.bulk_group.add.s32 [%0], [%1], %2;" ::"l"(gdst), "r"(smem_u32(ssrc)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_commit_wait_read()
{
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}
// L2 prefetches of the bulk-async family: `bytes` contiguous bytes (16-byte granules) resp. one box of a tensor map
__device__ __forceinline__ void l2_prefetch_bulk(const void *p, uint32_t bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
__device__ __forceinline__ void l2_prefetch_box(const CUtensorMap *tm, int c0, int c1)
{
    asm volatile("cp.async.bulk.prefetch.tensor.2d.L2.global.tile [%0, {%1, %2}];" ::"l"(tm), "r"(c0), "r"(c1) : "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

template <int QMASK>
struct LaneQ {
    static constexpr int NQ = (QMASK & 1) + ((QMASK & 2) ? 2 : 0);
    static constexpr int DP = ((NQ * LT + 31) / 32) * 32;     // deposit-window pitch in words: rows are bank-neutral
    static constexpr int OFF_N = 0, OFF_PX = (QMASK & 1) * LT, OFF_PY = OFF_PX + LT;
};

template <int STAGE, int QMASK, int NCOPY, int SUBROWS>
constexpr size_t lanes_smem_bytes()
{
    constexpr int WR = SUBROWS + 2 * HALO + 1;
    return (size_t)NCOPY * WR * LaneQ<QMASK>::DP * 4 + (STAGE < 2 ? (size_t)NCOPY * WR * LFP * 8 : 0);
}

__device__ __forceinline__ int magic_int(float v_plus_magic) { return __float_as_int(v_plus_magic) - MAGIC_BITS; }
__device__ __forceinline__ float pow2i(int k) { return __int_as_float((127 + k) << 23); }      // 2^k, |k| < 127

// nearest node (+ POS_BIAS, tile-relative) and the signed offset from it in units of 2^-24 cell, all in integers
__device__ __forceinline__ void lane_decode(uint32_t f, int &cb, int &di)
{
    const uint32_t g = f + (1u << (POS_FRAC_BITS - 1));
    cb = (int)(g >> POS_FRAC_BITS);
    di = (int)(g & POS_FRAC_MASK) - (1 << (POS_FRAC_BITS - 1));
}

// O1 / Eq. 13: LaneW<SHAPE>::scale times the weights of the nodes c-1, c, c+1 around the nearest node c.  SINE:
// G = (1 - cos)/2 without its 1/2 (folded into dt and the deposit scales): with b = (DD/2 - 1/2 - d) pi/DD the
// control-volume faces sit at the cosine arguments b (> -pi/2DD, < pi/2: only the lower clamp can act) and b + pi/DD
// (> 0: only the upper one).
template <int SHAPE>
struct LaneW {
    static constexpr float scale = SHAPE == PM2D_SINE ? 2.f : 1.f;
    static constexpr float inv2 = 1.f / (scale * scale);
};

template <int SHAPE>
__device__ __forceinline__ void lane_weights(int di, const PartParams &P, float W[3])
{
    if (SHAPE == PM2D_SINE) {
        const float b = fmaf((float)di, P.w4_slope, P.w4_off);
        const float c0 = __cosf(fmaxf(b, 0.f)), c1 = __cosf(fminf(b + P.k_rad, 3.14159265358979f));
        W[0] = 1.f - c0;
        W[1] = c0 - c1;
        W[2] = 1.f + c1;
    } else
        weights3<SHAPE>((float)di * (1.0f / 16777216.0f), P, W);
}

// both axes at once: the packed FFMA2 / FADD2 of sm_100a work on the (x, y) pairs; same values as lane_weights
template <int SHAPE>
__device__ __forceinline__ void lane_weights_xy(int dix, int diy, const PartParams &P, float Wx[3], float Wy[3])
{
    if (SHAPE == PM2D_SINE) {
        const float2 d = make_float2((float)dix, (float)diy);
        const float2 b = __ffma2_rn(d, make_float2(P.w4_slope, P.w4_slope), make_float2(P.w4_off, P.w4_off));
        const float2 t1 = __fadd2_rn(b, make_float2(P.k_rad, P.k_rad));
        const float2 c0 = make_float2(__cosf(fmaxf(b.x, 0.f)), __cosf(fmaxf(b.y, 0.f)));
        const float2 c1 = make_float2(__cosf(fminf(t1.x, 3.14159265358979f)), __cosf(fminf(t1.y, 3.14159265358979f)));
        const float2 one = make_float2(1.f, 1.f), neg = make_float2(-1.f, -1.f);
        const float2 w0 = __ffma2_rn(c0, neg, one), w1 = __ffma2_rn(c1, neg, c0), w2 = __fadd2_rn(c1, one);
        Wx[0] = w0.x; Wy[0] = w0.y;
        Wx[1] = w1.x; Wy[1] = w1.y;
        Wx[2] = w2.x; Wy[2] = w2.y;
    } else {
        lane_weights<SHAPE>(dix, P, Wx);
        lane_weights<SHAPE>(diy, P, Wy);
    }
}

// Eq. 14 in fixed point, the same on every route (fast path, listed strays, global overflow) so that the grids do not
// depend on the route a particle takes:
//   density   rint((Wx[a] * qn) * Wy[b]), qn = w * nscale                      [global units, F2I: exact range]
//   momentum  rint((Wx[a] * qx) * Wy[b]), qx = (w * pscale 2^-sp) * u_x        [window units of 2^sp global units]
//             by one FFMA with 1.5 * 2^23 while |u| <= ucap (the product stays below 2^22), by F2I beyond.
__device__ __forceinline__ int lane_pfix(float ww, float q, bool wide)
{
    return wide ? __float2int_rn(ww * q) : magic_int(fmaf(ww, q, MAGIC));
}

// 3 x 3 nodes on the global grids (a particle whose footprint left the windows), same integers as the windows
template <int SHAPE, int QMASK>
__device__ __forceinline__ void lane_deposit_global(const PartParams &P, int gx0, int gy0, uint32_t xf, uint32_t yf, float ux, float uy,
                                                    float w, int sp)
{
    int cxb, cyb, dix, diy;
    float Wx[3], Wy[3];
    lane_decode(xf, cxb, dix);
    lane_decode(yf, cyb, diy);
    lane_weights<SHAPE>(dix, P, Wx);
    lane_weights<SHAPE>(diy, P, Wy);
    const bool wide = fmaxf(fabsf(ux), fabsf(uy)) > P.ucap;
    const float qn = w * (P.nscale * LaneW<SHAPE>::inv2), qp = w * (P.pscale * LaneW<SHAPE>::inv2 * pow2i(-sp)), qx = qp * ux, qy = qp * uy;
#pragma unroll 1
    for (int a = 0; a < 3; a++) {
        const int gi = fold_x(gx0 + cxb - POS_BIAS - 1 + a, P.nx);
        const int fac = (gi == 0 || gi == P.nx) ? 2 : 1;
#pragma unroll 1
        const float an = Wx[a] * qn, ax = Wx[a] * qx, ay = Wx[a] * qy;
        for (int b = 0; b < 3; b++) {
            const int gj = (gy0 + cyb - POS_BIAS - 1 + b) & (P.ny - 1);
            const size_t k = (size_t)gi * P.ny + gj;
            if (QMASK & 1) atomicAdd(&P.nfix[k], fac * __float2int_rn(an * Wy[b]));
            if (QMASK & 2) {
                atomicAdd(&P.pxfix[k], (fac << sp) * lane_pfix(Wy[b], ax, wide));
                atomicAdd(&P.pyfix[k], (fac << sp) * lane_pfix(Wy[b], ay, wide));
            }
        }
    }
}

// ---- one particle outside the fast path: copy chosen per node column ------------------------------------------------
// Returns nothing; a particle whose footprint left the windows goes to the global overflow list (gather) or
// straight to the global grids (deposit), exactly like process_direct.
template <int SHAPE, int STAGE, int QMASK, int NCOPY, int SUBROWS>
__device__ __forceinline__ void lane_stray(const PartParams &P, int64_t p, bool dep_only, int gx0, int gy0, int row0, int tile,
                                           int sp, const float2 *Fs, int32_t *dep)
{
    constexpr int WR = SUBROWS + 2 * HALO + 1, MLO = NCOPY == 4 ? -1 : 0, DP = LaneQ<QMASK>::DP, TS = NCOPY == 2 ? 1 : 0;
    constexpr float GS = LaneW<SHAPE>::inv2;
    PV me = P.pv[p];
    uint32_t xf = me.x, yf = me.y;
    float ux = me.ux, uy = me.uy;
    auto gather = [&](uint32_t xg, uint32_t yg, float2 &f) -> bool {
        int cxb, cyb, dix, diy;
        float Wx[3], Wy[3];
        lane_decode(xg, cxb, dix);
        lane_decode(yg, cyb, diy);
        const int rb = cxb - POS_BIAS - 1 - row0, z0 = cyb - POS_BIAS - MLO;      // z = c - MLO + 1 of the first footprint column c = cy - 1
        if ((unsigned)rb > (unsigned)(WR - 3) || (unsigned)z0 > (unsigned)(NCOPY + 30)) return false;
        lane_weights<SHAPE>(dix, P, Wx);
        lane_weights<SHAPE>(diy, P, Wy);
        float fx = 0.f, fy = 0.f;
#pragma unroll
        for (int b = 0; b < 3; b++) {
            const int z = z0 + b, ci = min(max(z - 16, 0), NCOPY - 1), t = z - ci;
            float rx = 0.f, ry = 0.f;
#pragma unroll
            for (int a = 0; a < 3; a++) {
                const float2 v = Fs[(ci * WR + rb + a) * LFP + t + TS];
                rx += Wx[a] * v.x;
                ry += Wx[a] * v.y;
            }
            fx += Wy[b] * rx;
            fy += Wy[b] * ry;
        }
        f = make_float2(fx, fy);
        return true;
    };
    if (STAGE == 0) {
        float uhx, uhy;
        if (dep_only) {
            const float2 uh = P.uh[p];
            uhx = uh.x;
            uhy = uh.y;
        } else {
            float2 f;
            if (!gather(xf, yf, f)) { push_overflow(P, p, tile, false); return; }
            uhx = __fmaf_rn(GS * P.dt, f.x, ux);                                   // Eq. 17
            uhy = __fmaf_rn(GS * P.dt, f.y, uy);
            P.uh[p] = make_float2(uhx, uhy);
        }
        xf = advance(xf, P.hx, __fadd_rn(uhx, ux));
        yf = advance(yf, P.hy, __fadd_rn(uhy, uy));
        ux = uhx;
        uy = uhy;
    } else if (STAGE == 1 && !dep_only) {
        const float2 uh = P.uh[p];
        const uint32_t xh = advance(xf, P.hx, __fadd_rn(uh.x, ux));                // x^ of Eq. 17 again
        const uint32_t yh = advance(yf, P.hy, __fadd_rn(uh.y, uy));
        float2 f;
        if (!gather(xh, yh, f)) { push_overflow(P, p, tile, false); return; }
        float unx = __fmaf_rn(0.5f * GS * P.dt, f.x, 0.5f * __fadd_rn(uh.x, ux));  // Eq. 19
        const float uny = __fmaf_rn(0.5f * GS * P.dt, f.y, 0.5f * __fadd_rn(uh.y, uy));
        xf = advance(xf, P.hx, __fadd_rn(unx, ux));
        yf = advance(yf, P.hy, __fadd_rn(uny, uy));
        reflect_x(xf, unx, gx0, P.nx);
        me.x = xf; me.y = yf; me.ux = unx; me.uy = uny;
        P.pv[p] = me;
        ux = unx;
        uy = uny;
    }
    const float w = P.w[p];
    int cxb, cyb, dix, diy;
    float Wx[3], Wy[3];
    lane_decode(xf, cxb, dix);
    lane_decode(yf, cyb, diy);
    const int rb = cxb - POS_BIAS - 1 - row0, z0 = cyb - POS_BIAS - MLO;
    if ((unsigned)rb > (unsigned)(WR - 3) || (unsigned)z0 > (unsigned)(NCOPY + 30)) {
        lane_deposit_global<SHAPE, QMASK>(P, gx0, gy0, xf, yf, ux, uy, w, sp);
        return;
    }
    lane_weights<SHAPE>(dix, P, Wx);
    lane_weights<SHAPE>(diy, P, Wy);
    const bool wide = fmaxf(fabsf(ux), fabsf(uy)) > P.ucap;
    const float qn = w * (P.nscale * GS), qp = w * (P.pscale * GS * pow2i(-sp)), qx = qp * ux, qy = qp * uy;
#pragma unroll
    for (int b = 0; b < 3; b++) {
        const int z = z0 + b, ci = min(max(z - 16, 0), NCOPY - 1), t = z - ci;
#pragma unroll
        for (int a = 0; a < 3; a++) {
            int32_t *d = dep + (ci * WR + rb + a) * DP + t;
            if (QMASK & 1) atomicAdd(d + LaneQ<QMASK>::OFF_N, __float2int_rn((Wx[a] * qn) * Wy[b]));
            if (QMASK & 2) {
                atomicAdd(d + LaneQ<QMASK>::OFF_PX, lane_pfix(Wy[b], Wx[a] * qx, wide));
                atomicAdd(d + LaneQ<QMASK>::OFF_PY, lane_pfix(Wy[b], Wx[a] * qy, wide));
            }
        }
    }
}

// ---- the fused stage kernel of the lane order ------------------------------------------------------------------------
// One CTA per sub-tile.  STAGE 0: gather at x^n, Eq. 17, deposit (x^, u^); STAGE 1: gather at x^, Eq. 19 + walls,
// deposit (x^{n+1}, u^{n+1}); STAGE 2: deposit only.  QMASK bit 0: density, bit 1: momentum.
template <int SHAPE, int STAGE, int QMASK, int NCOPY, int SUBROWS, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) k_stage_lanes(const PartParams P, const __grid_constant__ CUtensorMap tmF)
{
    constexpr int WR = SUBROWS + 2 * HALO + 1, SUBS = TILE / SUBROWS, MLO = NCOPY == 4 ? -1 : 0;
    constexpr int DP = LaneQ<QMASK>::DP, NDEP = NCOPY * WR * DP;
    // force-window copy ci holds node column c at index c - (gy0 + ci + MLO - 1) + TS; TS makes copy 0 start on the even
    // column gy0 - 2 (box loads start on 16-byte boundaries)
    constexpr int TS = NCOPY == 2 ? 1 : 0, LTS = LT + TS;
    extern __shared__ __align__(128) int32_t lanes_smem[];
    int32_t *dep = lanes_smem;                                             // [NCOPY][WR][DP]
    float2 *Fs = reinterpret_cast<float2 *>(lanes_smem + NDEP);           // [NCOPY][WR][LFP]
    __shared__ uint32_t slist[LSTRAY];
    __shared__ int scount;
    __shared__ __align__(8) uint64_t fbar;
    const int tile = blockIdx.x / SUBS, sub = blockIdx.x % SUBS, lane_ = threadIdx.x & 31;
    const int gx0 = (tile / P.nty) * TILE, gy0 = (tile % P.nty) * TILE;
    const int row0 = sub * SUBROWS - HALO;                                  // tile-relative node row of window row 0
    // A sub-tile whose window lies inside the grid takes the even copies as box loads of WR rows x LFP columns (bulk-async,
    // one mbarrier) and derives the odd ones in shared memory; windows that fold at an x wall or wrap in y are copied by
    // the threads from the global grid.  The deposit windows are zeroed by a bulk copy on the same barrier.  Both depend on
    // the block index alone and are issued before anything is read from global memory (r02c: 7 % of the warp samples sat
    // in the wait for them when they followed the loads of the sub-tile's particle range).
    const bool bulk = STAGE < 2 && gy0 - 2 >= 0 && gy0 + 36 <= P.ny && gx0 + row0 >= 0 && gx0 + row0 + WR - 1 < P.nx;
    static_assert(NDEP * 4 <= PM2D_ZEROS_BYTES && (NDEP * 4) % 16 == 0, "bulk zero fill");
    constexpr bool USE_BAR = LANES_TMA_ZERO || STAGE < 2;
    if (USE_BAR && threadIdx.x == 0 && (LANES_TMA_ZERO || bulk)) {
        mbar_init(&fbar, 1);
        mbar_expect_tx(&fbar, (uint32_t)((LANES_TMA_ZERO ? NDEP * 4 : 0) + (bulk ? (NCOPY / 2) * WR * LFP * sizeof(float2) : 0)));
        if (bulk) {
#pragma unroll
            for (int ci = 0; ci < NCOPY; ci += 2) tma_load_2d(Fs + ci * WR * LFP, &tmF, gy0 + ci - 2, gx0 + row0, &fbar);
        }
        if (LANES_TMA_ZERO) bulk_load(dep, P.zeros, NDEP * 4, &fbar);
    }
    const int64_t t0 = P.tile_off[tile], t1 = P.tile_off[tile + 1];
    int64_t s0 = t0, s1 = t1;
    if (SUBS == 2) {
        const int64_t mid = t0 + P.sub0[tile];
        if (sub == 0) s1 = mid; else s0 = mid;
    }
    if (LANES_PF_DIST > 0 && threadIdx.x == NT - 32) {
        auto prefetch_block = [&](int b) {
            if (b >= (int)gridDim.x) return;
            const int tl = b / SUBS, sb = b % SUBS;
            int64_t a0 = P.tile_off[tl], a1 = P.tile_off[tl + 1];
            if (SUBS == 2) {
                const int64_t mid = a0 + P.sub0[tl];
                if (sb == 0) a1 = mid; else a0 = mid;
            }
            if (a1 <= a0) return;
            l2_prefetch_bulk(P.pv + a0, (uint32_t)(a1 - a0) * 16u);
            const int64_t wl = a0 & ~(int64_t)3;                               // 16-byte granules; a short tail is left out
            l2_prefetch_bulk(P.w + wl, ((uint32_t)(a1 - wl) * 4u) & ~15u);
            if (STAGE == 1) {
                const int64_t ul = a0 & ~(int64_t)1;
                l2_prefetch_bulk(P.uh + ul, ((uint32_t)(a1 - ul) * 8u) & ~15u);
            }
            if (STAGE < 2) {
                const int bx0 = (tl / P.nty) * TILE + sb * SUBROWS - HALO, by0 = (tl % P.nty) * TILE;
                if (by0 - 2 >= 0 && by0 + 36 <= P.ny && bx0 >= 0 && bx0 + WR - 1 < P.nx) {
#pragma unroll
                    for (int ci = 0; ci < NCOPY; ci += 2) l2_prefetch_box(&tmF, by0 + ci - 2, bx0);
                }
            }
        };
        prefetch_block((int)blockIdx.x + LANES_PF_DIST);
        if ((int)blockIdx.x < LANES_PF_DIST) prefetch_block((int)blockIdx.x);
    }
    if (s1 == s0) {          // nothing to do, but the bulk copies write this CTA's shared memory: wait them out
        if (USE_BAR && threadIdx.x == 0 && (LANES_TMA_ZERO || bulk)) mbar_wait(&fbar, 0);
        return;
    }
    // the records of the first two rounds are asked for before the windows are set up
    PV *const pvs = P.pv + s0;
    const float *const ws = P.w + s0;
    float2 *const uhs = P.uh + s0;
    const int np_sub = (int)(s1 - s0);
    auto load = [&](int i, PV &me, float &w, float2 &uh) {
        if (i < np_sub) {
            me = pvs[i];
            w = ws[i];
            if (STAGE == 1) uh = uhs[i];
        }
    };
    PV me0 = PV{0u, 0u, 0.f, 0.f}, me1 = me0;
    float w0 = 0.f, w1 = 0.f;
    float2 uh0 = make_float2(0.f, 0.f), uh1 = uh0;
    load((int)threadIdx.x, me0, w0, uh0);
    load((int)threadIdx.x + NT, me1, w1, uh1);
    // momentum windows count in units of 2^sp global units (from the tile's largest weight, k_lanesort)
    const int sp = P.lane_exp[tile];
    const float pst = P.pscale * pow2i(-sp);

    if (STAGE < 2 && !bulk) {
        constexpr int NE = NCOPY * WR * LTS, IT = (NE + NT - 1) / NT;
        float2 v[IT];
#pragma unroll
        for (int k = 0; k < IT; k++) {
            const int e = threadIdx.x + k * NT;
            const int ci = e / (WR * LTS), rem = e - ci * (WR * LTS), r = rem / LTS, t = rem - r * LTS;
            const int gi = fold_x(gx0 + row0 + r, P.nx);
            const int gj = (gy0 + t - TS + ci + MLO - 1) & (P.ny - 1);
            v[k] = e < NE ? P.F[(size_t)gi * P.ny + gj] : make_float2(0.f, 0.f);
        }
#pragma unroll
        for (int k = 0; k < IT; k++) {
            const int e = threadIdx.x + k * NT;
            const int ci = e / (WR * LTS), rem = e - ci * (WR * LTS), r = rem / LTS, t = rem - r * LTS;
            if (e < NE) Fs[(ci * WR + r) * LFP + t] = v[k];
        }
    }
    if (!LANES_TMA_ZERO) {
        int4 *d4 = reinterpret_cast<int4 *>(dep);
        for (int e = threadIdx.x; e < NDEP / 4; e += NT) d4[e] = make_int4(0, 0, 0, 0);
    }
    if (threadIdx.x == 0) scount = 0;
    __syncthreads();
    if (LANES_TMA_ZERO && !(STAGE < 2 && bulk)) mbar_wait(&fbar, 0);
    if (STAGE < 2 && bulk) {
        mbar_wait(&fbar, 0);
        // odd copy ci = even copy ci - 1 moved by one column: a warp takes a window row at a time (lane = column), the
        // LTS - 32 columns beyond ride on the first lanes
        for (int rr = threadIdx.x >> 5; rr < (NCOPY / 2) * WR; rr += NT / 32) {
            const int h = rr / WR, r = rr - h * WR;                       // warp-uniform
            const float2 *src = Fs + (2 * h * WR + r) * LFP + 1;
            float2 *dst = Fs + ((2 * h + 1) * WR + r) * LFP;
            const float2 v0 = src[lane_], v1 = lane_ < LTS - 32 ? src[32 + lane_] : make_float2(0.f, 0.f);
            dst[lane_] = v0;
            if (lane_ < LTS - 32) dst[32 + lane_] = v1;
        }
        __syncthreads();
    }

    const int lane = threadIdx.x & 31;
    constexpr float GS = LaneW<SHAPE>::inv2;
    // launch constants that only scale by powers of two come ready from the host (lane_dt = GS dt, lane_qns = GS nscale):
    // the kernel runs at 56 registers and re-derived them every round of the loop
    const float dtg = STAGE == 1 ? P.lane_dt_half : P.lane_dt;
    const float qns = P.lane_qns, qps = pst * GS;
    const bool wall_tile = gx0 == 0 || gx0 + TILE >= P.nx;             // only these tiles can see a particle cross a wall
    const int rofs = POS_BIAS + 1 + row0, cofs = POS_BIAS + lane + MLO;
    // advance() with the factor 2^24 folded into h on the host (a power of two: the same bits)
    const float hx24 = P.hx24, hy24 = P.hy24;
    auto adv24 = [](uint32_t f, float h24, float usum) { return f + (uint32_t)__float2int_rn(__fmul_rn(h24, usum)); };
    // one particle: gather, push, deposit (or hand it to the stray list)
    auto particle = [&](PV me, const float w, const float2 uh, const int i) {
        float ux = me.ux, uy = me.uy;
        uint32_t xd = me.x, yd = me.y;
        float Wx[3], Wy[3];
        if (STAGE < 2) {
            uint32_t xg = me.x, yg = me.y;
            if (STAGE == 1) {
                xg = adv24(me.x, hx24, __fadd_rn(uh.x, ux));
                yg = adv24(me.y, hy24, __fadd_rn(uh.y, uy));
            }
            int cxb, cyb, dix, diy;
            lane_decode(xg, cxb, dix);
            lane_decode(yg, cyb, diy);
            const int ci = cyb - cofs, rb = cxb - rofs;
            if ((unsigned)ci >= (unsigned)NCOPY || (unsigned)rb > (unsigned)(WR - 3)) {
                const int slot = atomicAdd(&scount, 1);
                if (slot < LSTRAY) slist[slot] = (uint32_t)i;
                else push_overflow(P, s0 + i, tile, false);
                return;
            }
            lane_weights_xy<SHAPE>(dix, diy, P, Wx, Wy);
            const float2 *fw = Fs + (ci * WR + rb) * LFP + lane + TS;
            // Eq. 15, both components of F at once (FFMA2 on the (Fx, Fy) pairs as LDS.64 delivers them)
            float2 f2 = make_float2(0.f, 0.f);
            {
                const float2 wy0 = make_float2(Wy[0], Wy[0]), wy1 = make_float2(Wy[1], Wy[1]), wy2 = make_float2(Wy[2], Wy[2]);
#pragma unroll
                for (int a = 0; a < 3; a++) {
                    float2 r = __fmul2_rn(wy0, fw[a * LFP]);
                    r = __ffma2_rn(wy1, fw[a * LFP + 1], r);
                    r = __ffma2_rn(wy2, fw[a * LFP + 2], r);
                    f2 = __ffma2_rn(make_float2(Wx[a], Wx[a]), r, f2);
                }
            }
            const float fx = f2.x, fy = f2.y;
            if (STAGE == 0) {
                const float uhx = __fmaf_rn(dtg, fx, ux), uhy = __fmaf_rn(dtg, fy, uy);             // Eq. 17
                uhs[i] = make_float2(uhx, uhy);
                xd = adv24(me.x, hx24, __fadd_rn(uhx, ux));
                yd = adv24(me.y, hy24, __fadd_rn(uhy, uy));
                ux = uhx;
                uy = uhy;
            } else {
                float unx = __fmaf_rn(dtg, fx, 0.5f * __fadd_rn(uh.x, ux));                         // Eq. 19
                const float uny = __fmaf_rn(dtg, fy, 0.5f * __fadd_rn(uh.y, uy));
                xd = adv24(me.x, hx24, __fadd_rn(unx, ux));
                yd = adv24(me.y, hy24, __fadd_rn(uny, uy));
                if (wall_tile) reflect_x(xd, unx, gx0, P.nx);
                me.x = xd; me.y = yd; me.ux = unx; me.uy = uny;
                pvs[i] = me;
                ux = unx;
                uy = uny;
            }
        }
        int cxb, cyb, dix, diy;
        lane_decode(xd, cxb, dix);
        lane_decode(yd, cyb, diy);
        const int ci = cyb - cofs, rb = cxb - rofs;
        const bool wide = (QMASK & 2) && fmaxf(fabsf(ux), fabsf(uy)) > P.ucap;    // beyond the range of the FFMA trick
        if ((unsigned)ci >= (unsigned)NCOPY || (unsigned)rb > (unsigned)(WR - 3) || wide) {
            const int slot = atomicAdd(&scount, 1);
            if (slot < LSTRAY) slist[slot] = (uint32_t)i | LSTRAY_DEP;
            else push_overflow(P, s0 + i, tile, true);
            return;
        }
        lane_weights_xy<SHAPE>(dix, diy, P, Wx, Wy);
        const float qn = w * qns, qp = w * qps, qx = qp * ux, qy = qp * uy;
        int32_t *dw = dep + (ci * WR + rb) * DP + lane;
        const float2 q2 = make_float2(qx, qy), magic2 = make_float2(MAGIC, MAGIC);
#pragma unroll
        for (int a = 0; a < 3; a++) {
            const float an = Wx[a] * qn;
            const float2 a2 = __fmul2_rn(make_float2(Wx[a], Wx[a]), q2);          // (Wx[a] qx, Wx[a] qy)
#pragma unroll
            for (int b = 0; b < 3; b++) {
                if (QMASK & 1) atomicAdd(dw + a * DP + LaneQ<QMASK>::OFF_N + b, __float2int_rn(an * Wy[b]));
                if (QMASK & 2) {
                    const float2 v2 = __ffma2_rn(make_float2(Wy[b], Wy[b]), a2, magic2);
                    atomicAdd(dw + a * DP + LaneQ<QMASK>::OFF_PX + b, magic_int(v2.x));
                    atomicAdd(dw + a * DP + LaneQ<QMASK>::OFF_PY + b, magic_int(v2.y));
                }
            }
        }
    };
    // Two particles per round of the loop; a register set is refilled with the record of the round after next as soon as
    // its particle is done (36 resident warps do not hide the loads), the two sets swap roles instead of being copied.
    for (int i = threadIdx.x; i < np_sub; i += 2 * NT) {
        particle(me0, w0, uh0, i);
        if (i + NT >= np_sub) break;
        load(i + 2 * NT, me0, w0, uh0);
        particle(me1, w1, uh1, i + NT);
        load(i + 3 * NT, me1, w1, uh1);
    }
    __syncthreads();
    {   // strays
        const int ns = min(scount, LSTRAY);
        if (threadIdx.x == 0 && scount > 0) atomicAdd(P.stray_total, (unsigned long long)scount);
        if (LANES_STRAYS_IN_CTA) {
            for (int e = threadIdx.x; e < ns; e += NT) {
                const uint32_t ent = slist[e];
                lane_stray<SHAPE, STAGE, QMASK, NCOPY, SUBROWS>(P, s0 + (int64_t)(ent & ~LSTRAY_DEP), (ent & LSTRAY_DEP) != 0, gx0, gy0, row0,
                                                                tile, sp, Fs, dep);
            }
            if (ns > 0) __syncthreads();
        } else if (ns > 0) {
            // the CTA's list moves to the global overflow list in one block (one atomic per CTA): k_lanes_overflow serves
            // the strays on the global grids while this CTA goes on to its flush
            __shared__ int sbase;
            if (threadIdx.x == 0) sbase = atomicAdd(P.ovf_count, ns);
            __syncthreads();
            for (int e = threadIdx.x; e < ns; e += NT) {
                const uint32_t ent = slist[e];
                const int slot = sbase + e;
                if (slot < P.ovf_cap) {
                    P.ovf_p[slot] = (s0 + (int64_t)(ent & ~LSTRAY_DEP)) | ((ent & LSTRAY_DEP) ? OVF_DEP : 0);
                    P.ovf_tile[slot] = tile;
                } else
                    P.flags[2] = 1;
            }
        }
    }
    // flush: node (row r, z) with z = c - MLO + 1 is the sum of the copies that hold it.
    constexpr int NCOL = NCOPY + 33;
    const int mp = 1 << sp;
    if (LANES_BULK_FLUSH && STAGE < 2 && bulk) {
        // Interior window (no wall, no wrap): the sums go to a dense staging array [quantity][row][FW] in the space of
        // the force window (its last reader is behind the barrier above), columns gy0 - 4 .. gy0 + FW - 5 so that every
        // row starts on a 16-byte boundary of the global grid, and one bulk reduction per row and quantity
        // (cp.reduce.async.bulk, integer add) replaces one RED per node.
        constexpr int FW = 44, NQ = LaneQ<QMASK>::NQ, Z0 = 4 + MLO - 1;      // staging column of z = 0
        int32_t *stg = reinterpret_cast<int32_t *>(Fs);
        static_assert(NQ * WR * FW * 4 <= NCOPY * WR * LFP * 8, "staging fits in the force window");
        for (int e = threadIdx.x; e < WR * FW; e += NT) {
            const int r = e / FW, zc = e - r * FW, z = zc - Z0;
            int v = 0, vx = 0, vy = 0;
#pragma unroll
            for (int ci = 0; ci < NCOPY; ci++) {
                const int t = z - ci;
                if ((unsigned)t < (unsigned)LT) {
                    const int32_t *d = dep + (ci * WR + r) * DP + t;
                    if (QMASK & 1) v += d[LaneQ<QMASK>::OFF_N];
                    if (QMASK & 2) {
                        vx += d[LaneQ<QMASK>::OFF_PX];
                        vy += d[LaneQ<QMASK>::OFF_PY];
                    }
                }
            }
            if (QMASK & 1) stg[r * FW + zc] = v;
            if (QMASK & 2) {
                stg[((QMASK & 1) * WR + r) * FW + zc] = mp * vx;
                stg[(((QMASK & 1) + 1) * WR + r) * FW + zc] = mp * vy;
            }
        }
        fence_proxy_async_smem();
        __syncthreads();
        if (threadIdx.x < NQ * WR) {
            const int q = threadIdx.x / WR, r = threadIdx.x - q * WR;
            int32_t *g = (QMASK == 3 ? (q == 0 ? P.nfix : (q == 1 ? P.pxfix : P.pyfix)) : (QMASK == 1 ? P.nfix : (q == 0 ? P.pxfix : P.pyfix)));
            bulk_reduce_add_s32(g + (size_t)(gx0 + row0 + r) * P.ny + (gy0 - 4), stg + (q * WR + r) * FW, FW * 4);
            bulk_commit_wait_read();
        }
        return;
    }
    // one global integer reduction per touched node; wall columns hold half a control volume and count twice (Q9); rows
    // beyond a wall fold back.  A warp takes a window row at a time (lane = z < 32: no index arithmetic per node, the row's
    // fold, wall factor and base address are warp-uniform); the NCOL - 32 columns beyond are spread over the CTA afterwards.
    auto flush_node = [&](int r, int z) {
        int v = 0, vx = 0, vy = 0;
#pragma unroll
        for (int ci = 0; ci < NCOPY; ci++) {
            const int t = z - ci;
            if ((unsigned)t < (unsigned)LT) {
                const int32_t *d = dep + (ci * WR + r) * DP + t;
                if (QMASK & 1) v += d[LaneQ<QMASK>::OFF_N];
                if (QMASK & 2) {
                    vx += d[LaneQ<QMASK>::OFF_PX];
                    vy += d[LaneQ<QMASK>::OFF_PY];
                }
            }
        }
        if ((v | vx | vy) == 0) return;
        const int gi = fold_x(gx0 + row0 + r, P.nx);
        const int gj = (gy0 + z + MLO - 1) & (P.ny - 1);
        const int wall = (gi == 0 || gi == P.nx) ? 1 : 0;
        const size_t k = (size_t)gi * P.ny + gj;
        // the integer sums wrap: report it instead of handing wrapped moments to the solvers.  Density (all terms of one
        // sign): one window alone beyond half the int32 range, n > n_cap / 2 = 4 n_max of the profile.  Momentum (terms of
        // either sign, a hot species reaches a large fraction of the range by noise alone): this window's sum itself is
        // outside int32, |n u| > n_cap / 16 = n_max / 2
        if (abs(v) > ((1 << 30) >> wall) || max(abs(vx), abs(vy)) > (0x7fffffff >> (sp + wall))) P.flags[3] = 2;
        const int mpw = 1 << (sp + wall);
        if (v) atomicAdd(&P.nfix[k], v * (1 + wall));
        if (vx) atomicAdd(&P.pxfix[k], vx * mpw);
        if (vy) atomicAdd(&P.pyfix[k], vy * mpw);
    };
    for (int r = threadIdx.x >> 5; r < WR; r += NT / 32) flush_node(r, lane);
    constexpr int NTAIL = NCOL - 32;
    for (int e = threadIdx.x; e < WR * NTAIL; e += NT) flush_node(e / NTAIL, 32 + e % NTAIL);
}

// the deferred particles of k_stage_lanes: same arithmetic, gather from the global force grid, deposit on the global grids
template <int SHAPE, int STAGE, int QMASK>
__global__ void __launch_bounds__(128) k_lanes_overflow(const PartParams P)
{
    const int n = min(*P.ovf_count, P.ovf_cap);
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n; k += gridDim.x * blockDim.x) {
        const int tile = P.ovf_tile[k];
        const int64_t ent = P.ovf_p[k], p = ent & ~OVF_DEP;
        const bool dep_only = (ent & OVF_DEP) != 0;
        const int gx0 = (tile / P.nty) * TILE, gy0 = (tile % P.nty) * TILE;
        PV me = P.pv[p];
        uint32_t xf = me.x, yf = me.y;
        float ux = me.ux, uy = me.uy;
        bool ok;
        if (STAGE == 0) {
            float uhx, uhy;
            if (dep_only) {
                const float2 uh = P.uh[p];
                uhx = uh.x;
                uhy = uh.y;
            } else {
                const float2 f = gather_direct<SHAPE, false>(P, gx0, gy0, xf, yf, nullptr, ok);
                uhx = __fmaf_rn(P.dt, f.x, ux);                                        // Eq. 17
                uhy = __fmaf_rn(P.dt, f.y, uy);
                P.uh[p] = make_float2(uhx, uhy);
            }
            xf = advance(xf, P.hx, __fadd_rn(uhx, ux));
            yf = advance(yf, P.hy, __fadd_rn(uhy, uy));
            ux = uhx;
            uy = uhy;
        } else if (STAGE == 1 && !dep_only) {
            const float2 uh = P.uh[p];
            const uint32_t xh = advance(xf, P.hx, __fadd_rn(uh.x, ux));
            const uint32_t yh = advance(yf, P.hy, __fadd_rn(uh.y, uy));
            const float2 f = gather_direct<SHAPE, false>(P, gx0, gy0, xh, yh, nullptr, ok);
            float unx = __fmaf_rn(0.5f * P.dt, f.x, 0.5f * __fadd_rn(uh.x, ux));       // Eq. 19
            const float uny = __fmaf_rn(0.5f * P.dt, f.y, 0.5f * __fadd_rn(uh.y, uy));
            xf = advance(xf, P.hx, __fadd_rn(unx, ux));
            yf = advance(yf, P.hy, __fadd_rn(uny, uy));
            reflect_x(xf, unx, gx0, P.nx);
            me.x = xf; me.y = yf; me.ux = unx; me.uy = uny;
            P.pv[p] = me;
            ux = unx;
            uy = uny;
        }
        lane_deposit_global<SHAPE, QMASK>(P, gx0, gy0, xf, yf, ux, uy, P.w[p], P.lane_exp[tile]);
    }
}

// ---- the lane order: rebin pass 2 ---------------------------------------------------------------------------------------
// One CTA per tile, after the tile pass (k_rebin_scatter) has brought every particle into its tile.  Two stable
// counting sorts over the tile's list:
//   (every position below is the SORT position of lane_sort_pos: where the particle will be half a rebin period from now)
//   A  by key_A = (h, column, y sub-bin of 1/32 cell)            -> rank rho in (h, y); h = sub-tile (cell row >= 16)
//      slab = the rho-th of N_h particles cut into 32 slabs whose sizes differ by at most one (the first N_h mod 32
//      slabs hold one more)
//   B  by key_B = (h, slab, x bin)                                -> w = rank inside the slab, in x order
//   slot = first slot of h + 32 w + slab.
// Ties keep the order of the list (that of the tile pass), so the result is a pure function of the input order.
struct LaneSortParams {
    const PV *src;
    const float *wsrc;
    const int64_t *idsrc;
    PV *dst;
    float *wdst;
    int64_t *iddst;
    const int64_t *tile_off;
    int32_t *sub0;
    int32_t *lane_exp;          // [ntiles] out: sp of the tile (momentum unit of the windows of k_stage_lanes)
    float pscale_ucap;          // global fixed-point scale of the momentum times the velocity cap
    float predx, predy;         // see lane_sort_pos
    int nx, ny, nty;
    uint32_t *scratch;          // [np] keys between the sweeps
    const int64_t *perm1;       // optional (tests): slot before the tile pass of every slot after it
    int32_t *keys_out;
    int64_t *perm_out;
    int32_t *flags;
    int subs;
};

constexpr int LS_WARPS = 8, LS_BINS = 2048;

// The position a particle is sorted by: where free flight puts it half a rebin period from now, x + u * pred with pred =
// rebin_every * dt_p / (2 dx) * 2^24 (tile-relative, 2^-24 cells), clamped to the tile.  A particle then strays from its
// lane by the drift of half a period in either direction instead of a whole period in one: 3 keV electrons at a period
// of 16 steps leave the four-copy range in 0.005 % of the visits instead of 0.4 %.
__device__ __forceinline__ uint32_t lane_sort_pos(uint32_t f, float u, float pred, int cells)
{
    const int64_t v = (int64_t)f - ((int64_t)POS_BIAS << POS_FRAC_BITS) + (int64_t)__float2int_rn(__fmul_rn(u, pred));
    return (uint32_t)min(max(v, (int64_t)0), ((int64_t)cells << POS_FRAC_BITS) - 1);
}

__device__ __forceinline__ int lane_slab(int rho, int n)
{
    const int base = n >> 5, rem = n & 31, cut = rem * (base + 1);
    return rho < cut ? rho / (base + 1) : rem + (rho - cut) / max(base, 1);
}

// first rank of slab i among n particles
__device__ __forceinline__ int lane_slab_start(int i, int n)
{
    const int base = n >> 5, rem = n & 31;
    return i * base + min(i, rem);
}

// stable rank of every particle of this warp's part [beg, end) in its bin: hist[bin] holds the first rank of the bin
// for this warp (16-bit, updated as the batches go by); fn(i, rank, key) is called once per particle
// load(i) fetches what the particle needs (its key among it) -- the loads of LS_AHEAD batches are issued before the first
// of them is ranked, so the serial chain match -> histogram update of a warp does not wait for memory batch by batch
constexpr int LS_AHEAD = 4;
template <class T, class LoadFn, class KeyFn, class OutFn>
__device__ __forceinline__ void lane_rank_sweep(int64_t beg, int64_t end, int lane, uint16_t *myhist, LoadFn load, KeyFn key, OutFn out)
{
    for (int64_t base0 = beg; base0 < end; base0 += 32 * LS_AHEAD) {
        T v[LS_AHEAD];
#pragma unroll
        for (int u = 0; u < LS_AHEAD; u++) {
            const int64_t i = base0 + 32 * u + lane;
            if (i < end) v[u] = load(i);
        }
#pragma unroll
        for (int u = 0; u < LS_AHEAD; u++) {
            if (base0 + 32 * u >= end) break;        // warp-uniform
            const int64_t i = base0 + 32 * u + lane;
            const bool live = i < end;
            int k = LS_BINS + lane;                  // dead lanes: unique keys
            if (live) k = key(v[u]);
            const unsigned peers = __match_any_sync(0xffffffffu, k);
            const int rank = __popc(peers & ((1u << lane) - 1u));
            const int leader = __ffs(peers) - 1;
            int b = 0;
            if (live && lane == leader) {
                b = myhist[k];
                myhist[k] = (uint16_t)(b + __popc(peers));
            }
            b = __shfl_sync(0xffffffffu, b, leader);
            __syncwarp();
            if (live) out(i, b + rank, k, v[u]);
        }
    }
}

// exclusive scan of hist[warp][bin] over (bin, warp): hist becomes the first rank per (warp, bin).  Thread t takes the
// bins t, t + 256, ... so that a warp reads consecutive 16-bit counters (one wavefront; with bins 8t .. 8t+7 per thread
// the scans were 73 % of the kernel's shared wavefronts, all of them 4-way conflicts: 4.8 ms for c3's electrons, r02k).
__device__ __forceinline__ void lane_scan(uint16_t *hist, int32_t *wsum)
{
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int carry = 0;
    for (int c = threadIdx.x; c < LS_BINS; c += LS_WARPS * 32) {
        int v[LS_WARPS], s = 0;
#pragma unroll
        for (int w = 0; w < LS_WARPS; w++) {
            v[w] = hist[w * LS_BINS + c];
            s += v[w];
        }
        int incl = s;
        for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) wsum[wid] = incl;
        __syncthreads();
        int run = carry + incl - s, total = 0;
#pragma unroll
        for (int w = 0; w < LS_WARPS; w++) {
            const int ws = wsum[w];
            if (w < wid) run += ws;
            total += ws;
        }
#pragma unroll
        for (int w = 0; w < LS_WARPS; w++) {
            hist[w * LS_BINS + c] = (uint16_t)run;
            run += v[w];
        }
        carry += total;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(LS_WARPS * 32) k_lanesort(const LaneSortParams C)
{
    __shared__ uint16_t hist[LS_WARPS * LS_BINS];      // 32 KB
    __shared__ int32_t wsum[LS_WARPS];
    __shared__ int wmax_bits;
    const int tile = blockIdx.x;
    const int64_t t0 = C.tile_off[tile];
    const int64_t n = C.tile_off[tile + 1] - t0;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (n == 0) {
        if (threadIdx.x == 0) { C.sub0[tile] = 0; C.lane_exp[tile] = 0; }
        return;
    }
    if (threadIdx.x == 0) wmax_bits = 0;
    if (n > 65535) {                                   // 16-bit ranks: the lane order is for species below 16 per cell
        if (threadIdx.x == 0) { C.flags[3] = 1; C.sub0[tile] = 0; }
        return;
    }
    uint32_t *hist32 = reinterpret_cast<uint32_t *>(hist);
    for (int e = threadIdx.x; e < LS_WARPS * LS_BINS / 2; e += LS_WARPS * 32) hist32[e] = 0u;
    __syncthreads();
    int64_t per = (n + LS_WARPS - 1) / LS_WARPS;
    per = (per + 31) & ~(int64_t)31;
    const int64_t beg = min(n, wid * per), end = min(n, beg + per);
    uint16_t *myhist = hist + wid * LS_BINS;
    uint32_t *scr = C.scratch + t0;
    const bool two = C.subs == 2;
    const int tw = min(TILE, C.nx - (tile / C.nty) * TILE), th = min(TILE, C.ny - (tile % C.nty) * TILE);     // cells of this tile
    // sweep 1: key_A | x bin << 16 of every particle, counts of key_A
    for (int64_t base0 = beg; base0 < end; base0 += 32 * LS_AHEAD) {
        PV mv[LS_AHEAD];
#pragma unroll
        for (int u = 0; u < LS_AHEAD; u++) {
            const int64_t i = base0 + 32 * u + lane;
            if (i < end) mv[u] = C.src[t0 + i];
        }
#pragma unroll
        for (int u = 0; u < LS_AHEAD; u++) {
            if (base0 + 32 * u >= end) break;
            const int64_t i = base0 + 32 * u + lane;
            const bool live = i < end;
            int k = LS_BINS + lane;
            if (live) {
                const PV me = mv[u];
                const uint32_t xk = lane_sort_pos(me.x, me.ux, C.predx, tw), yk = lane_sort_pos(me.y, me.uy, C.predy, th);
                const int cx = (int)(xk >> POS_FRAC_BITS), cy = (int)(yk >> POS_FRAC_BITS);
                const int h = two ? cx >> 4 : 0;
                k = (h << 10) | (cy << 5) | (int)((yk >> (POS_FRAC_BITS - 5)) & 31u);
                const int xb = two ? ((cx & 15) << 1) | (int)((xk >> (POS_FRAC_BITS - 1)) & 1u) : cx;
                scr[i] = (uint32_t)k | ((uint32_t)xb << 16);
            }
            const unsigned peers = __match_any_sync(0xffffffffu, k);
            if (live && lane == __ffs(peers) - 1) myhist[k] = (uint16_t)(myhist[k] + __popc(peers));
            __syncwarp();
        }
    }
    __syncthreads();
    lane_scan(hist, wsum);
    const int n0 = two ? (int)hist[LS_BINS / 2] : (int)n, n1 = (int)n - n0;     // first rank of bin (h = 1, 0, 0) = particles of sub-tile 0
    if (threadIdx.x == 0) C.sub0[tile] = n0;
    // sweep 2: rank in (h, y) -> slab -> key_B
    lane_rank_sweep<uint32_t>(
        beg, end, lane, myhist, [&](int64_t i) { return scr[i]; }, [](uint32_t v) { return (int)(v & 0xffffu); },
        [&](int64_t i, int rho, int k, uint32_t v) {
            const int h = k >> 10, xb = (int)(v >> 16);
            const int slab = h ? lane_slab(rho - n0, n1) : lane_slab(rho, n0);
            scr[i] = (uint32_t)((h << 10) | (slab << 5) | xb);
        });
    __syncthreads();
    for (int e = threadIdx.x; e < LS_WARPS * LS_BINS / 2; e += LS_WARPS * 32) hist32[e] = 0u;
    __syncthreads();
    // sweep 3: counts of key_B
    for (int64_t base0 = beg; base0 < end; base0 += 32 * LS_AHEAD) {
        int kk[LS_AHEAD];
#pragma unroll
        for (int u = 0; u < LS_AHEAD; u++) {
            const int64_t i = base0 + 32 * u + lane;
            kk[u] = i < end ? (int)scr[i] : LS_BINS + lane;
        }
#pragma unroll
        for (int u = 0; u < LS_AHEAD; u++) {
            if (base0 + 32 * u >= end) break;
            const bool live = base0 + 32 * u + lane < end;
            const unsigned peers = __match_any_sync(0xffffffffu, kk[u]);
            if (live && lane == __ffs(peers) - 1) myhist[kk[u]] = (uint16_t)(myhist[kk[u]] + __popc(peers));
            __syncwarp();
        }
    }
    __syncthreads();
    lane_scan(hist, wsum);
    // sweep 4: rank in (h, slab, x) -> slot; move the records
    float wmax = 0.f;
    struct Rec {
        PV me;
        float w;
        int key;
    };
    lane_rank_sweep<Rec>(
        beg, end, lane, myhist, [&](int64_t i) { return Rec{C.src[t0 + i], C.wsrc[t0 + i], (int)scr[i]}; }, [](const Rec &r) { return r.key; },
        [&](int64_t i, int rb, int k, const Rec &r) {
            const int h = k >> 10, slab = (k >> 5) & 31;
            const int nn = h ? n1 : n0, hb = h ? n0 : 0;
            const int w = rb - hb - lane_slab_start(slab, nn);      // rank inside the slab
            const int64_t q = t0 + hb + 32 * w + slab;
            const PV me = r.me;
            const float wi = r.w;
            wmax = fmaxf(wmax, wi);
            C.dst[q] = me;
            C.wdst[q] = wi;
            if (C.idsrc) C.iddst[q] = C.idsrc[t0 + i];
            if (C.perm1) {
                const int64_t old = C.perm1[t0 + i];
                if (C.keys_out)
                    C.keys_out[old] = tile * TCELLS + (int)(lane_sort_pos(me.x, me.ux, C.predx, tw) >> POS_FRAC_BITS) * TILE +
                                      (int)(lane_sort_pos(me.y, me.uy, C.predy, th) >> POS_FRAC_BITS);
                if (C.perm_out) C.perm_out[q] = old;
            }
        });
    // the tile's largest weight fixes the units of its shared windows: one contribution stays below 2^22
    for (int o = 16; o > 0; o >>= 1) wmax = fmaxf(wmax, __shfl_xor_sync(0xffffffffu, wmax, o));
    if (lane == 0) atomicMax(&wmax_bits, __float_as_int(wmax));       // weights are >= 0: their bit patterns order like integers
    __syncthreads();
    if (threadIdx.x == 0) {
        const float wm = __int_as_float(wmax_bits);
        C.lane_exp[tile] = wm > 0.f ? max(0, ilogbf(wm * C.pscale_ucap) + 1 - 22) : 0;
    }
}

__global__ void k_iota64(int64_t *p, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = i;
}

}  // namespace

// free flight of half a rebin period, in 2^-24 cells per unit velocity (axis 0 = x, 1 = y)
float lane_pred(const pm2d_ctx *c, int axis)
{
    return (float)((double)c->g.rebin_every * c->dtp / (2.0 * (axis ? c->g.dy : c->g.dx)) * 16777216.0);
}

// velocity cap of the FFMA float -> int path of the momentum deposit: four thermal velocities; faster particles take the
// exact path (a listed stray).  The smaller the cap, the finer the momentum unit of the windows.
double lane_ucap(const SpeciesDev &S) { return std::max(4.0 * sqrt(S.vth2), 0.004); }

// =================================================================================================
// Sort every tile of species s into the lane order.  from_primary: the unsorted arrays are the current ones (loader,
// pm2d_set_particles) -- they become the second buffers first; else they already sit in the second buffers (after
// the tile pass of the rebin).  perm1_dev (tests): slot before the tile pass of every slot of the source arrays.
int launch_lanesort(pm2d_ctx *c, int s, bool from_primary, int32_t *keys_dev, int64_t *perm_dev, const int64_t *perm1_dev)
{
    SpeciesDev &S = c->sp[s];
    if (S.np == 0) {
        PM2D_CUDA_CHECK(cudaMemsetAsync(S.sub0, 0, (size_t)c->ntiles * sizeof(int32_t), c->stream));
        PM2D_CUDA_CHECK(cudaMemsetAsync(S.lane_exp, 0, (size_t)c->ntiles * sizeof(int32_t), c->stream));
        return PM2D_OK;
    }
    if (from_primary) {
        std::swap(S.pv, S.pv2);
        std::swap(S.w, S.w2);
        std::swap(S.id, S.id2);
    }
    LaneSortParams C;
    C.src = S.pv2; C.wsrc = S.w2; C.idsrc = S.id ? S.id2 : nullptr;
    C.dst = S.pv; C.wdst = S.w; C.iddst = S.id;
    C.tile_off = from_primary ? S.tile_off : S.tile_off2;
    C.sub0 = S.sub0;
    C.lane_exp = S.lane_exp;
    C.pscale_ucap = c->pscale * (float)lane_ucap(S);
    C.nx = c->g.nx; C.ny = c->g.ny; C.nty = c->nty;
    C.predx = lane_pred(c, 0);
    C.predy = lane_pred(c, 1);
    C.scratch = reinterpret_cast<uint32_t *>(S.uh);          // u^ is scratch outside a step
    C.perm1 = perm1_dev; C.keys_out = keys_dev; C.perm_out = perm_dev;
    C.flags = c->flags;
    C.subs = S.lane_subs;
    k_lanesort<<<c->ntiles, LS_WARPS * 32, 0, c->stream>>>(C);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}

// hot species (thermal drift of a cell or more per rebin period): four window copies on half tiles; cold ones: two on
// whole tiles
template <int SHAPE, int STAGE, int QMASK>
static int launch_lanes_variant(const PartParams &P, const CUtensorMap &tm, int ntiles, int hot, cudaStream_t st)
{
#define PM2D_LANES_LAUNCH(NCOPY, SUBROWS, NT, MINB)                                                                          \
    do {                                                                                                                     \
        constexpr size_t bytes = lanes_smem_bytes<STAGE, QMASK, NCOPY, SUBROWS>();                                          \
        auto kern = k_stage_lanes<SHAPE, STAGE, QMASK, NCOPY, SUBROWS, NT, MINB>;                                            \
        static bool once = false;                                                                                            \
        if (!once) {                                                                                                         \
            PM2D_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));            \
            PM2D_CUDA_CHECK(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100));                \
            once = true;                                                                                                     \
        }                                                                                                                    \
        kern<<<ntiles * (TILE / SUBROWS), NT, bytes, st>>>(P, tm);                                                           \
    } while (0)
    if (hot) PM2D_LANES_LAUNCH(4, 16, LANES_NT_HOT, LANES_MINB_HOT);
    else PM2D_LANES_LAUNCH(2, 32, LANES_NT_COLD, LANES_MINB_COLD);     // half tiles for the cold species: 4.83 instead of 4.74 ms on c3 (r02j)
#undef PM2D_LANES_LAUNCH
    k_lanes_overflow<SHAPE, STAGE, QMASK><<<148 * 8, 128, 0, st>>>(P);
    return PM2D_OK;
}

template <int SHAPE>
static int launch_lanes_shape(const PartParams &P, const CUtensorMap &tm, int stage, int qmask, int ntiles, int hot, cudaStream_t st)
{
    if (stage == 0) return qmask == 3 ? launch_lanes_variant<SHAPE, 0, 3>(P, tm, ntiles, hot, st) : launch_lanes_variant<SHAPE, 0, 1>(P, tm, ntiles, hot, st);
    if (stage == 1) return qmask == 3 ? launch_lanes_variant<SHAPE, 1, 3>(P, tm, ntiles, hot, st) : launch_lanes_variant<SHAPE, 1, 1>(P, tm, ntiles, hot, st);
    if (qmask == 3) return launch_lanes_variant<SHAPE, 2, 3>(P, tm, ntiles, hot, st);
    if (qmask == 2) return launch_lanes_variant<SHAPE, 2, 2>(P, tm, ntiles, hot, st);
    return launch_lanes_variant<SHAPE, 2, 1>(P, tm, ntiles, hot, st);
}

// tensor map of the nodal force grid of species s: [(nx+1)][ny] elements of 8 bytes (float2), box = LFP columns x the
// window rows of the species' sub-tiles
int lanes_make_tensor_map(pm2d_ctx *c, int s)
{
    SpeciesDev &S = c->sp[s];
    static_assert(sizeof(CUtensorMap) == sizeof(S.tmapF), "tensor map storage");
    typedef CUresult (*EncodeFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                 const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static EncodeFn encode = nullptr;
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        PM2D_CUDA_CHECK(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
        if (!fn || q != cudaDriverEntryPointSuccess) {
            pm2d_set_error("cuTensorMapEncodeTiled is not available in this driver");
            return PM2D_ECUDA;
        }
        encode = (EncodeFn)fn;
    }
    const int wr = (S.lane_subs == 2 ? 16 : 32) + 2 * HALO + 1;
    const cuuint64_t dims[2] = {(cuuint64_t)c->g.ny, (cuuint64_t)c->g.nx + 1};
    const cuuint64_t strides[1] = {(cuuint64_t)c->g.ny * sizeof(float2)};
    const cuuint32_t box[2] = {(cuuint32_t)std::min(LFP, c->g.ny), (cuuint32_t)std::min(wr, c->g.nx + 1)};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = encode(reinterpret_cast<CUtensorMap *>(S.tmapF), CU_TENSOR_MAP_DATA_TYPE_UINT64, 2, S.F, dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        pm2d_set_error("cuTensorMapEncodeTiled failed");
        return PM2D_ECUDA;
    }
    return PM2D_OK;
}

int launch_stage_lanes(pm2d_ctx *c, int s, int stage, int qmask)
{
    SpeciesDev &S = c->sp[s];
    if (S.np == 0) return PM2D_OK;
    PartParams P = make_part_params(c, s);
    PM2D_CUDA_CHECK(cudaMemsetAsync(c->ovf_count, 0, sizeof(int32_t), c->stream));
    if (stage == 0) {          // stage A deposits (x^, u^) into the second set
        P.nfix = S.nhat; P.pxfix = S.pxhat; P.pyfix = S.pyhat;
    }
    const int hot = S.lane_copies == 4;
    int rc;
    const CUtensorMap &tm = *reinterpret_cast<const CUtensorMap *>(S.tmapF);
    if (S.cfg.shape == PM2D_CIC) rc = launch_lanes_shape<PM2D_CIC>(P, tm, stage, qmask, c->ntiles, hot, c->stream);
    else if (S.cfg.shape == PM2D_TSC) rc = launch_lanes_shape<PM2D_TSC>(P, tm, stage, qmask, c->ntiles, hot, c->stream);
    else rc = launch_lanes_shape<PM2D_SINE>(P, tm, stage, qmask, c->ntiles, hot, c->stream);
    if (rc) return rc;
    count_launch(c, 2);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}
