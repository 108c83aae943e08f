// pm2d_particles.cu -- particle kernels of libpm2d.so (sm_100a):
//   * fused gather + push + deposit, stage A (Eq. 17) and stage B (Eq. 19)      [P:L191-221]
//   * deposit-only pass (initial item (1) of the flow, lazy momentum grids)       [Eq. 14, P:L187]
//   * counter-based particle loader (Philox-4x32-10)         [P:L154-162]
//   * deterministic stable rebin: tile pass specialised to neighbour moves, then a sort inside
//     every tile by (layer, cell) or by cell                                      [DESIGN.md 6.4]
//
// Data layout.  A particle is a 16-byte record PV {x, y, ux, uy} plus a weight w
// and, between the two stages of a step, the predictor velocity u^ (float2).  Particles are stored
// tile by tile (PM2D_TILE x PM2D_TILE cells); inside a tile, as of the last rebin, either LAYERED
// (by rank in the cell, then by the cell's rank in its column, then by column: 32 consecutive particles lie in 32
// different cells of 32 different columns) or
// CELL-MAJOR (cell_off gives every cell's run).  A position is a pair of 32-bit fixed-point numbers
// relative to the tile's origin,
//     xfix = (cell_rel + POS_BIAS) << 24 | frac24,
// so the in-cell offset carries 24 bits whatever the size of the box, the push is an exact integer
// add of a rounded displacement, and the canonical (ix, fx) of include/pm2d.h is read off exactly.
//
// Fused stage kernels.  A CTA owns one tile: it copies the nodal force of the tile +
// halo into shared memory, its particles gather from that window, are pushed, and deposit into a
// shared int32 fixed-point window that is flushed once with global integer reductions.  Integer
// accumulation makes the grids independent of the order of the atomics (bit-reproducible) and
// n_i - n_e exact.
//   k_stage_direct (layered species): one particle per thread, shared atomics per particle;
//   k_stage        (cell-major species): every thread owns a strip of S cells of one cell column and
//                  keeps, in registers, the force on and the deposit to the 4 x 4 nodes around its
//                  current cell; sliding to the next cell row adds the finished node row to the
//                  window with 4 x 3 conflict-free ATOMS.  Particles outside the patch ("strays")
//                  are listed and served with the per-particle code after the strips;
//   k_stage_overflow: particles whose footprint left the tile's window, on the global grids.
#include <algorithm>
#include <cmath>
#include <cstdlib>

#include "pm2d_particle_dev.cuh"

namespace {

// particles a strip thread cannot serve from its register patch are listed per CTA and processed by all
// threads after the strips (no divergence inside the strip loops); a full list spills to the global one
constexpr int STRAY_CAP = 1024;
constexpr int STRIP_SPLIT = 64;             // CTAs that may share one tile in k_stage
constexpr int SPLIT_PARTICLES = 16384;      // ... one per so many particles of the tile
constexpr int PF_ROWS = 2;            // L2 prefetch distance of the strips, in cell rows
constexpr bool SHIFT_PATCH = true;   // one copy of the particle loop (instruction cache) at the price of register moves per cell
constexpr uint32_t STRAY_DEP = 0x80000000u;            // flag: deposit only

__device__ __forceinline__ void defer_stray(const PartParams &P, uint32_t *slist, int *scount, int64_t p, int64_t t0, int tile,
                                            bool dep_only)
{
    int slot = atomicAdd(scount, 1);
    if (slot < STRAY_CAP) slist[slot] = (uint32_t)(p - t0) | (dep_only ? STRAY_DEP : 0u);
    else push_overflow(P, p, tile, dep_only);
}

// The nodal force of Eq. 16 / 18 (k_force, pm2d_fields.cu) for the nodes of the tile window -> shared
// memory.  Window rows beyond a wall hold F of the mirror node (Q9: the gather folds indices), window
// columns wrap (y periodic).  All loads of a thread are issued before the first store.
template <int NT, int PITCH = WPITCH>
__device__ __forceinline__ void load_force_window(const PartParams &P, int gx0, int gy0, float2 *Fs)
{
    constexpr int IT = (WIN * WIN + NT - 1) / NT;
    float2 v[IT];
#pragma unroll
    for (int k = 0; k < IT; k++) {
        const int e = threadIdx.x + k * NT;
        const int r = e / WIN, cidx = e - r * WIN;
        const int gi = fold_x(gx0 + r - HALO, P.nx);
        const int gj = (gy0 + cidx - HALO) & (P.ny - 1);
        v[k] = (e < WIN * WIN) ? P.F[(size_t)gi * P.ny + gj] : make_float2(0.f, 0.f);
    }
#pragma unroll
    for (int k = 0; k < IT; k++) {
        const int e = threadIdx.x + k * NT;
        const int r = e / WIN, cidx = e - r * WIN;
        if (e < WIN * WIN) Fs[r * PITCH + cidx] = v[k];
    }
}

// ---- register patch of a strip thread: force on, and deposit to, the 4 x 4 nodes around its current cell.
// A strip runs along x (rows of cells); the 32 lanes of a warp hold the 32 cell columns of the tile, so at
// every row the warp reads one contiguous piece of the cell-sorted particle arrays and its shared-memory
// accesses fall into consecutive banks.  Logical patch row a (node row i-1+a of cell row i) lives in
// physical row (a + ROT) & 3, so sliding to the next cell row renames rows instead of moving registers.
struct Patch {
    float2 F[4][4];      // (Fx, Fy)
    float2 dn[4][2];     // density deposit, columns (0,1) and (2,3)
    float2 dp[4][4];     // momentum deposit (Px, Py)
};

__device__ __forceinline__ float2 dup2(float v) { return make_float2(v, v); }

__device__ __forceinline__ bool in_patch(int rel) { return (uint32_t)(rel + (1 << 23)) < (1u << 25); }   // offset in [-1/2, 3/2)

// walking state of a strip thread
struct StripCtx {
    int64_t t0;                  // first slot of the tile
    int32_t n_tile;              // particles in the tile
    const int32_t *coff;         // shared: coff[c] = first slot (tile-relative) of cell c = row * TILE + column
    const int32_t *cend;         // shared: one past the last slot of cell c that this CTA serves (tile split)
    uint32_t ay_fix;
    int j, wc0, tile, gx0;
    const float2 *Fs;
    int32_t *dep;
    uint32_t *slist;             // shared stray list of the CTA
    int *scount;
    int cell_cap;                // particles per cell served from the patch
    int32_t q;                   // tile-relative slot of the prefetched particle
    PV cur;                      // prefetched particle q
    float wcur;
    float2 uhcur;
};

template <int SHAPE, int STAGE, int QMASK, int ROT>
__device__ __forceinline__ void strip_particle(const PartParams &P, Patch &pt, const StripCtx &c, const PV me, const float wme,
                                               const float2 uhme, const int64_t p, const uint32_t ax_fix)
{
    constexpr float GS = 1.f / (W4Scale<SHAPE>::value * W4Scale<SHAPE>::value);   // undoes the scale of weights4
    float ux = me.ux, uy = me.uy;
    uint32_t xd = me.x, yd = me.y;                        // deposit position
    float Wx[4], Wy[4];
    if (STAGE < 2) {
        uint32_t xg = me.x, yg = me.y;                    // gather position: x^n (stage A), x^ (stage B, Q4)
        if (STAGE == 1) {
            xg = advance(me.x, P.hx, __fadd_rn(uhme.x, ux));
            yg = advance(me.y, P.hy, __fadd_rn(uhme.y, uy));
        }
        const int rx = (int)(xg - ax_fix), ry = (int)(yg - c.ay_fix);
        if (!in_patch(rx) || !in_patch(ry)) {
            defer_stray(P, c.slist, c.scount, p, c.t0, c.tile, false);
            return;
        }
        weights4<SHAPE>(rx, P, Wx);
        weights4<SHAPE>(ry, P, Wy);
        float2 f = make_float2(0.f, 0.f);                 // Eq. 15, both components at once (FFMA2)
        const float2 wy0 = dup2(Wy[0]), wy1 = dup2(Wy[1]), wy2 = dup2(Wy[2]), wy3 = dup2(Wy[3]);
#pragma unroll
        for (int a = 0; a < 4; a++) {
            const int pa = (a + ROT) & 3;
            float2 sa = __fmul2_rn(wy0, pt.F[pa][0]);
            sa = __ffma2_rn(wy1, pt.F[pa][1], sa);
            sa = __ffma2_rn(wy2, pt.F[pa][2], sa);
            sa = __ffma2_rn(wy3, pt.F[pa][3], sa);
            f = __ffma2_rn(dup2(Wx[a]), sa, f);
        }
        if (STAGE == 0) {
            const float uhx = __fmaf_rn(GS * P.dt, f.x, ux), uhy = __fmaf_rn(GS * P.dt, f.y, uy);   // Eq. 17
            P.uh[p] = make_float2(uhx, uhy);
            xd = advance(me.x, P.hx, __fadd_rn(uhx, ux));
            yd = advance(me.y, P.hy, __fadd_rn(uhy, uy));
            ux = uhx;
            uy = uhy;
        } else {
            float unx = __fmaf_rn(0.5f * GS * P.dt, f.x, 0.5f * __fadd_rn(uhme.x, ux));             // Eq. 19
            float uny = __fmaf_rn(0.5f * GS * P.dt, f.y, 0.5f * __fadd_rn(uhme.y, uy));
            xd = advance(me.x, P.hx, __fadd_rn(unx, ux));
            yd = advance(me.y, P.hy, __fadd_rn(uny, uy));
            reflect_x(xd, unx, c.gx0, P.nx);
            PV out;
            out.x = xd; out.y = yd; out.ux = unx; out.uy = uny;
            P.pv[p] = out;
            ux = unx;
            uy = uny;
        }
    }
    const int rx = (int)(xd - ax_fix), ry = (int)(yd - c.ay_fix);
    if (!in_patch(rx) || !in_patch(ry)) {
        defer_stray(P, c.slist, c.scount, p, c.t0, c.tile, true);
        return;
    }
    weights4<SHAPE>(rx, P, Wx);
    weights4<SHAPE>(ry, P, Wy);
    const float q = wme * (GS * P.nscale);                // Eq. 14 in fixed-point units
    const float2 qu = make_float2(ux * P.pratio, uy * P.pratio);
    const float2 wy01 = make_float2(Wy[0], Wy[1]), wy23 = make_float2(Wy[2], Wy[3]);
    const float2 wy0 = dup2(Wy[0]), wy1 = dup2(Wy[1]), wy2 = dup2(Wy[2]), wy3 = dup2(Wy[3]);
#pragma unroll
    for (int a = 0; a < 4; a++) {
        const int pa = (a + ROT) & 3;
        const float2 qa = dup2(Wx[a] * q);
        if (QMASK & 1) {
            pt.dn[pa][0] = __ffma2_rn(qa, wy01, pt.dn[pa][0]);
            pt.dn[pa][1] = __ffma2_rn(qa, wy23, pt.dn[pa][1]);
        }
        if (QMASK & 2) {
            const float2 qp = __fmul2_rn(qa, qu);
            pt.dp[pa][0] = __ffma2_rn(qp, wy0, pt.dp[pa][0]);
            pt.dp[pa][1] = __ffma2_rn(qp, wy1, pt.dp[pa][1]);
            pt.dp[pa][2] = __ffma2_rn(qp, wy2, pt.dp[pa][2]);
            pt.dp[pa][3] = __ffma2_rn(qp, wy3, pt.dp[pa][3]);
        }
    }
}

// flush physical row PR of the deposit patch into window row wr, columns wc0 .. wc0+3, and clear it
template <int QMASK, int PR>
__device__ __forceinline__ void flush_row(Patch &pt, int32_t *dep, int wr, int wc0)
{
    const int e = wr * WPITCH + wc0;
    if (QMASK & 1) {
        atomicAdd(&dep[e], __float2int_rn(pt.dn[PR][0].x));
        atomicAdd(&dep[e + 1], __float2int_rn(pt.dn[PR][0].y));
        atomicAdd(&dep[e + 2], __float2int_rn(pt.dn[PR][1].x));
        atomicAdd(&dep[e + 3], __float2int_rn(pt.dn[PR][1].y));
        pt.dn[PR][0] = pt.dn[PR][1] = make_float2(0.f, 0.f);
    }
    if (QMASK & 2) {
#pragma unroll
        for (int b = 0; b < 4; b++) {
            atomicAdd(&dep[WIN * WPITCH + e + b], __float2int_rn(pt.dp[PR][b].x));
            atomicAdd(&dep[2 * WIN * WPITCH + e + b], __float2int_rn(pt.dp[PR][b].y));
            pt.dp[PR][b] = make_float2(0.f, 0.f);
        }
    }
}

template <int PR>
__device__ __forceinline__ void load_force_row(Patch &pt, const float2 *Fs, int wr, int wc0)
{
#pragma unroll
    for (int b = 0; b < 4; b++) pt.F[PR][b] = Fs[wr * WPITCH + wc0 + b];
}

__device__ __forceinline__ void prefetch_l2(const void *ptr) { asm volatile("prefetch.global.L2 [%0];" ::"l"(ptr)); }

// DRAM -> L2 ahead of the strip: the particles of cell c of this thread's column
template <int STAGE>
__device__ __forceinline__ void prefetch_cell(const PartParams &P, const StripCtx &c, int cell)
{
    const int32_t q = c.coff[min(cell, TCELLS - 1)];
    if (q < c.n_tile) {
        prefetch_l2(P.pv + c.t0 + q);
        prefetch_l2(P.w + c.t0 + q);
        if (STAGE == 1) prefetch_l2(P.uh + c.t0 + q);
    }
}

// all particles of cell (i, j), then slide the patch to cell row i+1: physical row ROT is renamed (4 unrolled
// copies, ROT = 0..3), or, with SHIFT, the registers move and one copy serves every row (ROT = 0)
template <int SHAPE, int STAGE, int QMASK, int ROT, bool SHIFT>
__device__ __forceinline__ void strip_cell(const PartParams &P, Patch &pt, StripCtx &c, const int i)
{
    const int cell = i * TILE + c.j;
    const int32_t beg = c.coff[cell], end = c.cend[cell];
    const int32_t next_beg = c.coff[min(cell + TILE, TCELLS)];          // where this thread reads next
    const uint32_t ax_fix = (uint32_t)(i + POS_BIAS) << POS_FRAC_BITS;
    // the lanes of a warp walk their cells in lockstep: a cell much fuller than the tile's mean would stall
    // the other 31 lanes, so only its first cell_cap particles go through the patch, the rest to the stray list
    const int32_t fast_end = min(end, beg + c.cell_cap);
    int32_t q = beg;
    prefetch_cell<STAGE>(P, c, cell + PF_ROWS * TILE);
    if (beg < fast_end && c.q != beg) {                                  // no prefetch in flight (strip start, after empty cells)
        c.cur = P.pv[c.t0 + beg];
        c.wcur = P.w[c.t0 + beg];
        if (STAGE == 1) c.uhcur = P.uh[c.t0 + beg];
        c.q = beg;
    }
    // warp-uniform loop: the lanes reconverge at every particle (vote) instead of drifting apart in the
    // unrolled copies of this function
    for (;;) {
        const bool act = q < fast_end;
        if (!__any_sync(0xffffffffu, act)) break;
        if (act) {
            const PV me = c.cur;
            const float wme = c.wcur;
            const float2 uhme = c.uhcur;
            const int32_t nxt = (q + 1 < fast_end) ? q + 1 : next_beg;
            if (nxt < c.n_tile) {
                c.cur = P.pv[c.t0 + nxt];
                c.wcur = P.w[c.t0 + nxt];
                if (STAGE == 1) c.uhcur = P.uh[c.t0 + nxt];
            }
            c.q = nxt;
            strip_particle<SHAPE, STAGE, QMASK, ROT>(P, pt, c, me, wme, uhme, c.t0 + q, ax_fix);
            q++;
        }
    }
    for (; q < end; q++) defer_stray(P, c.slist, c.scount, c.t0 + q, c.t0, c.tile, false);
    __syncwarp();
    flush_row<QMASK, ROT>(pt, c.dep, i - 1 + HALO, c.wc0);                // node row i-1 is complete for this strip
    if (SHIFT) {                                                          // one copy of the loop body: move the patch up one row
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int b = 0; b < 4; b++) {
                if ((QMASK & 1) && b < 2) pt.dn[a][b] = pt.dn[a + 1][b];
                if (QMASK & 2) pt.dp[a][b] = pt.dp[a + 1][b];
                if (STAGE < 2) pt.F[a][b] = pt.F[a + 1][b];
            }
#pragma unroll
        for (int b = 0; b < 4; b++) {
            if (b < 2) pt.dn[3][b] = make_float2(0.f, 0.f);
            pt.dp[3][b] = make_float2(0.f, 0.f);
        }
        if (STAGE < 2) load_force_row<3>(pt, c.Fs, i + 3 + HALO, c.wc0);
    } else if (STAGE < 2)
        load_force_row<ROT>(pt, c.Fs, i + 3 + HALO, c.wc0);
}

template <int SHAPE, int STAGE, int QMASK, int S>
__global__ void __launch_bounds__(TCELLS / S, S >= 8 ? 4 : 2) k_stage(const PartParams P)
{
    static_assert(S % 4 == 0 && TILE % S == 0, "strip length");
    constexpr int NT = TCELLS / S;
    constexpr int NQ = (QMASK & 2) ? 3 : 1;
    __shared__ int32_t dep[NQ * WIN * WPITCH];
    __shared__ float2 Fs[(STAGE < 2) ? WIN * WPITCH : 1];
    __shared__ int32_t coff[TCELLS + 1];
    __shared__ int32_t cend[TCELLS];
    __shared__ uint32_t slist[STRAY_CAP];
    __shared__ int scount;
    // a tile is served by up to STRIP_SPLIT CTAs (blockIdx = tile * STRIP_SPLIT + part), one per SPLIT_PARTICLES
    // particles: part k of n takes the k-th n-th of every cell's run.  A filament tile of BJ config 5 holds 1.2 M
    // particles; as one CTA's work it would set the tail of the launch and overrun the CTA's stray list.
    const int tile = blockIdx.x / STRIP_SPLIT, part = blockIdx.x % STRIP_SPLIT;
    const int64_t t0 = P.tile_off[tile];
    const int64_t tile_n = P.tile_off[tile + 1] - t0;
    if (tile_n == 0) return;
    const int nsplit = (int)min((int64_t)STRIP_SPLIT, (tile_n + SPLIT_PARTICLES - 1) / SPLIT_PARTICLES);
    if (part >= nsplit) return;
    const int gx0 = (tile / P.nty) * TILE, gy0 = (tile % P.nty) * TILE;

    {
        const int32_t *co = P.cell_off + (size_t)tile * CPITCH;
        constexpr int IT = (TCELLS + NT) / NT;
        int32_t v[IT];
#pragma unroll
        for (int k = 0; k < IT; k++) {
            const int e = threadIdx.x + k * NT;
            v[k] = e <= TCELLS ? co[e] : 0;
        }
        if (STAGE < 2) load_force_window<NT>(P, gx0, gy0, Fs);
#pragma unroll
        for (int k = 0; k < IT; k++) {
            const int e = threadIdx.x + k * NT;
            if (e <= TCELLS) coff[e] = v[k];
        }
    }
    if (nsplit > 1) {   // this CTA's share of every cell's run: [beg + len * part / nsplit, beg + len * (part + 1) / nsplit)
        __syncthreads();
        constexpr int IT = (TCELLS + NT - 1) / NT;
        int32_t b[IT], e2[IT];
#pragma unroll
        for (int k = 0; k < IT; k++) {
            const int e = threadIdx.x + k * NT;
            if (e < TCELLS) {
                const int64_t lo = coff[e], len = coff[e + 1] - lo;
                b[k] = (int32_t)(lo + len * part / nsplit);
                e2[k] = (int32_t)(lo + len * (part + 1) / nsplit);
            }
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < IT; k++) {
            const int e = threadIdx.x + k * NT;
            if (e < TCELLS) { coff[e] = b[k]; cend[e] = e2[k]; }
        }
    } else {
        __syncthreads();
        for (int e = threadIdx.x; e < TCELLS; e += NT) cend[e] = coff[e + 1];
    }
    for (int e = threadIdx.x; e < NQ * WIN * WPITCH; e += NT) dep[e] = 0;
    if (threadIdx.x == 0) scount = 0;
    __syncthreads();

    const int j = threadIdx.x & 31, i0 = (threadIdx.x >> 5) * S;          // cell column, first cell row of the strip
    StripCtx ctx;
    ctx.t0 = t0;
    ctx.n_tile = coff[TCELLS];
    ctx.coff = coff;
    ctx.cend = cend;
    ctx.ay_fix = (uint32_t)(j + POS_BIAS) << POS_FRAC_BITS;
    ctx.j = j; ctx.wc0 = j - 1 + HALO; ctx.tile = tile; ctx.gx0 = gx0;
    ctx.Fs = Fs; ctx.dep = dep; ctx.slist = slist; ctx.scount = &scount;
    // ceil(mean particles per cell); sparse tiles (mean <= 1.5) get one more, or a third of them would stray;
    // dense tiles (mean >= 16: relative fluctuations are small, gradients across the tile are not) take no cap
    ctx.cell_cap = ctx.n_tile >= 16 * TCELLS
                       ? 0x3fffffff
                       : (2 * ctx.n_tile <= 3 * TCELLS ? P.sparse_cap : min(0x3fffffff, (ctx.n_tile + TCELLS - 1) / TCELLS + P.cap_extra));
    ctx.q = -1;
    ctx.cur = PV{0u, 0u, 0.f, 0.f};
    ctx.wcur = 0.f;
    ctx.uhcur = make_float2(0.f, 0.f);
    Patch pt;
#pragma unroll
    for (int a = 0; a < 4; a++)
#pragma unroll
        for (int b = 0; b < 4; b++) {
            pt.F[a][b] = pt.dp[a][b] = make_float2(0.f, 0.f);
            if (b < 2) pt.dn[a][b] = make_float2(0.f, 0.f);
        }
#pragma unroll
    for (int k = 0; k < PF_ROWS; k++) prefetch_cell<STAGE>(P, ctx, (i0 + k) * TILE + j);
    if (STAGE < 2) {
        load_force_row<0>(pt, Fs, i0 - 1 + HALO, ctx.wc0);
        load_force_row<1>(pt, Fs, i0 + HALO, ctx.wc0);
        load_force_row<2>(pt, Fs, i0 + 1 + HALO, ctx.wc0);
        load_force_row<3>(pt, Fs, i0 + 2 + HALO, ctx.wc0);
    }
    if (SHIFT_PATCH) {
#pragma unroll 1
        for (int k = 0; k < S; k++) strip_cell<SHAPE, STAGE, QMASK, 0, true>(P, pt, ctx, i0 + k);
    } else {
#pragma unroll 1
        for (int kk = 0; kk < S; kk += 4) {
            strip_cell<SHAPE, STAGE, QMASK, 0, false>(P, pt, ctx, i0 + kk);
            strip_cell<SHAPE, STAGE, QMASK, 1, false>(P, pt, ctx, i0 + kk + 1);
            strip_cell<SHAPE, STAGE, QMASK, 2, false>(P, pt, ctx, i0 + kk + 2);
            strip_cell<SHAPE, STAGE, QMASK, 3, false>(P, pt, ctx, i0 + kk + 3);
        }
    }
    {   // node rows i0+S-1 .. i0+S+1 (logical rows 0..2 of the cell row after the strip)
        flush_row<QMASK, 0>(pt, dep, i0 + S - 1 + HALO, ctx.wc0);
        flush_row<QMASK, 1>(pt, dep, i0 + S + HALO, ctx.wc0);
        flush_row<QMASK, 2>(pt, dep, i0 + S + 1 + HALO, ctx.wc0);
    }
    __syncthreads();
    {   // strays: 3 x 3 nodes around the nearest node, straight on the shared windows
        const int ns = min(scount, STRAY_CAP);
        if (threadIdx.x == 0 && scount > 0) atomicAdd(P.stray_total, (unsigned long long)scount);
        for (int e = threadIdx.x; e < ns; e += NT) {
            const uint32_t ent = slist[e];
            const int64_t p = t0 + (int64_t)(ent & ~STRAY_DEP);
            const bool dep_only = (ent & STRAY_DEP) != 0;
            if (!process_direct<SHAPE, STAGE, QMASK, true>(P, p, dep_only, gx0, gy0, Fs, dep)) push_overflow(P, p, tile, dep_only);
        }
        if (ns > 0) __syncthreads();
    }

    // flush: one global integer reduction per touched window node; wall columns hold half a
    // control volume and count twice (Q9); rows beyond a wall fold back (mirror particles)
    for (int e = threadIdx.x; e < WIN * WIN; e += NT) {
        const int rr = e / WIN, cidx = e - rr * WIN;
        const int se = rr * WPITCH + cidx;
        const int v = (QMASK & 1) ? dep[se] : 0;
        const int vx = (QMASK & 2) ? dep[WIN * WPITCH + se] : 0, vy = (QMASK & 2) ? dep[2 * WIN * WPITCH + se] : 0;
        if ((v | vx | vy) == 0) continue;
        const int gi = fold_x(gx0 + rr - HALO, P.nx);
        const int gj = (gy0 + cidx - HALO) & (P.ny - 1);
        const int fac = (gi == 0 || gi == P.nx) ? 2 : 1;
        const size_t k = (size_t)gi * P.ny + gj;
        if (v) atomicAdd(&P.nfix[k], fac * v);
        if (vx) atomicAdd(&P.pxfix[k], fac * vx);
        if (vy) atomicAdd(&P.pyfix[k], fac * vy);
    }
}

// ---- thread-per-particle stage kernel for layered species ------------------------------------------------------
// In the layered order the 32 lanes of a warp hold particles of 32 different, consecutive cells of (mostly) one
// cell row.  To make their shared accesses conflict-free the footprint is taken as 3 nodes around the nearest node
// in x and the 4 nodes around the CELL in y (the lane direction): the window column then depends on the cell only,
// and with a window pitch that is a multiple of 32 words the bank is the column, whatever the row.  12 nodes: 12
// LDS.64 for the gather, 12 x 3 ATOMS for the deposit, one wavefront each.
constexpr int DPITCH = 64;
constexpr int DFPITCH = 48;   // force window of the anchored variant: 48 float2 = 96 words, a multiple of 32 as well
constexpr int NNPITCH = 64;   // deposit-window pitch of the nearest-node variant
// its force-window pitch: 48 float2 = 96 words (the 16 lanes of an LDS.64 half-warp fall on 16 different bank pairs
// when they hold 16 consecutive columns); 42.6 KB per CTA with the deposit windows: five resident CTAs
template <int STAGE>
struct NNFPitch { static constexpr int value = 48; };

template <int SHAPE, int STAGE, int QMASK>
__device__ __forceinline__ bool direct_particle(const PartParams &P, int64_t p, int gx0, int gy0, const float2 *Fs, int32_t *dep)
{
    constexpr float GY = 1.f / W4Scale<SHAPE>::value;             // undoes the scale of weights4 (y only)
    PV me = P.pv[p];
    const float w = P.w[p];
    float ux = me.ux, uy = me.uy;
    uint32_t xd = me.x, yd = me.y;
    float Wx[3], Wy[4];
    if (STAGE < 2) {
        float2 uh = make_float2(0.f, 0.f);
        uint32_t xg = me.x, yg = me.y;
        if (STAGE == 1) {
            uh = P.uh[p];
            xg = advance(me.x, P.hx, __fadd_rn(uh.x, ux));
            yg = advance(me.y, P.hy, __fadd_rn(uh.y, uy));
        }
        int cx;
        float dx_;
        decode(xg, cx, dx_);
        const int cyc = (int)(yg >> POS_FRAC_BITS) - POS_BIAS;    // cell, not nearest node
        if (cx - 1 < -HALO || cx + 1 > TILE + HALO || cyc - 1 < -HALO || cyc + 2 > TILE + HALO) return false;
        weights3<SHAPE>(dx_, P, Wx);
        weights4<SHAPE>((int)(yg & POS_FRAC_MASK), P, Wy);
        const float2 *fw = Fs + (cx - 1 + HALO) * DFPITCH + (cyc - 1 + HALO);
        float2 f = make_float2(0.f, 0.f);
        const float2 wy0 = dup2(Wy[0]), wy1 = dup2(Wy[1]), wy2 = dup2(Wy[2]), wy3 = dup2(Wy[3]);
#pragma unroll
        for (int a = 0; a < 3; a++) {
            float2 sa = __fmul2_rn(wy0, fw[a * DFPITCH]);
            sa = __ffma2_rn(wy1, fw[a * DFPITCH + 1], sa);
            sa = __ffma2_rn(wy2, fw[a * DFPITCH + 2], sa);
            sa = __ffma2_rn(wy3, fw[a * DFPITCH + 3], sa);
            f = __ffma2_rn(dup2(Wx[a]), sa, f);
        }
        if (STAGE == 0) {
            const float uhx = __fmaf_rn(GY * P.dt, f.x, ux), uhy = __fmaf_rn(GY * P.dt, f.y, uy);       // Eq. 17
            P.uh[p] = make_float2(uhx, uhy);
            xd = advance(me.x, P.hx, __fadd_rn(uhx, ux));
            yd = advance(me.y, P.hy, __fadd_rn(uhy, uy));
            ux = uhx;
            uy = uhy;
        } else {
            float unx = __fmaf_rn(0.5f * GY * P.dt, f.x, 0.5f * __fadd_rn(uh.x, ux));                   // Eq. 19
            const float uny = __fmaf_rn(0.5f * GY * P.dt, f.y, 0.5f * __fadd_rn(uh.y, uy));
            xd = advance(me.x, P.hx, __fadd_rn(unx, ux));
            yd = advance(me.y, P.hy, __fadd_rn(uny, uy));
            reflect_x(xd, unx, gx0, P.nx);
            me.x = xd; me.y = yd; me.ux = unx; me.uy = uny;
            P.pv[p] = me;
            ux = unx;
            uy = uny;
        }
    }
    int cx;
    float dx_;
    decode(xd, cx, dx_);
    const int cyc = (int)(yd >> POS_FRAC_BITS) - POS_BIAS;
    if (cx - 1 < -HALO || cx + 1 > TILE + HALO || cyc - 1 < -HALO || cyc + 2 > TILE + HALO) {
        // off the window (far from its tile): 3 x 3 nodes on the global grids, like the overflow pass
        deposit_direct<SHAPE, QMASK, false>(P, gx0, gy0, xd, yd, ux, uy, w, nullptr);
        return true;
    }
    weights3<SHAPE>(dx_, P, Wx);
    weights4<SHAPE>((int)(yd & POS_FRAC_MASK), P, Wy);
    const float q = w * (GY * P.nscale);
    const float2 qu = make_float2(ux * P.pratio, uy * P.pratio);
    int32_t *dw = dep + (cx - 1 + HALO) * DPITCH + (cyc - 1 + HALO);
#pragma unroll
    for (int a = 0; a < 3; a++) {
        const float qa = Wx[a] * q;
#pragma unroll
        for (int b = 0; b < 4; b++) {
            const float qn = qa * Wy[b];
            if (QMASK & 1) atomicAdd(&dw[a * DPITCH + b], __float2int_rn(qn));
            if (QMASK & 2) {
                const float2 qp = __fmul2_rn(dup2(qn), qu);
                atomicAdd(&dw[WIN * DPITCH + a * DPITCH + b], __float2int_rn(qp.x));
                atomicAdd(&dw[2 * WIN * DPITCH + a * DPITCH + b], __float2int_rn(qp.y));
            }
        }
    }
    return true;
}

// ANCH: the cell-anchored 3 x 4 footprint above (conflict-free as long as the particles sit in the cells they were
// sorted into: species that hardly move between rebins, e.g. ions); else the 3 x 3 nodes around the nearest node
// on the odd-pitch windows (process_direct), whose conflicts do not depend on the drift.
template <int SHAPE, int STAGE, int QMASK, bool ANCH>
__global__ void __launch_bounds__(256, 5) k_stage_direct(const PartParams P)
{
    constexpr int NT = 256;
    constexpr int NQ = (QMASK & 2) ? 3 : 1;
    constexpr int PITCH = ANCH ? DPITCH : NNPITCH;
    constexpr int FPITCH = ANCH ? DFPITCH : NNFPitch<STAGE>::value;
    extern __shared__ int32_t direct_smem[];
    int32_t *dep = direct_smem;                                                      // [NQ][WIN][PITCH]
    float2 *Fs = reinterpret_cast<float2 *>(direct_smem + ((NQ * WIN * PITCH + 1) & ~1));   // [WIN][PITCH]
    const int tile = blockIdx.x;
    const int64_t t0 = P.tile_off[tile], t1 = P.tile_off[tile + 1];
    if (t1 == t0) return;
    const int gx0 = (tile / P.nty) * TILE, gy0 = (tile % P.nty) * TILE;
    if (STAGE < 2) load_force_window<NT, FPITCH>(P, gx0, gy0, Fs);
    for (int e = threadIdx.x; e < NQ * WIN * PITCH; e += NT) dep[e] = 0;
    __syncthreads();
    for (int64_t p = t0 + threadIdx.x; p < t1; p += NT) {
        const bool ok = ANCH ? direct_particle<SHAPE, STAGE, QMASK>(P, p, gx0, gy0, Fs, dep)
                             : process_direct<SHAPE, STAGE, QMASK, true, NNPITCH, NNFPitch<STAGE>::value>(P, p, false, gx0, gy0, Fs, dep);
        if (!ok) push_overflow(P, p, tile, false);
    }
    __syncthreads();
    for (int e = threadIdx.x; e < WIN * WIN; e += NT) {
        const int rr = e / WIN, cidx = e - rr * WIN;
        const int se = rr * PITCH + cidx;
        const int v = (QMASK & 1) ? dep[se] : 0;
        const int vx = (QMASK & 2) ? dep[WIN * PITCH + se] : 0, vy = (QMASK & 2) ? dep[2 * WIN * PITCH + se] : 0;
        if ((v | vx | vy) == 0) continue;
        const int gi = fold_x(gx0 + rr - HALO, P.nx);
        const int gj = (gy0 + cidx - HALO) & (P.ny - 1);
        const int fac = (gi == 0 || gi == P.nx) ? 2 : 1;
        const size_t k = (size_t)gi * P.ny + gj;
        if (v) atomicAdd(&P.nfix[k], fac * v);
        if (vx) atomicAdd(&P.pxfix[k], fac * vx);
        if (vy) atomicAdd(&P.pyfix[k], fac * vy);
    }
}

template <int STAGE, int QMASK, bool ANCH>
constexpr size_t direct_smem_bytes()
{
    return (size_t)(((((QMASK & 2) ? 3 : 1) * WIN * (ANCH ? DPITCH : NNPITCH)) + 1) & ~1) * 4 +
           (STAGE < 2 ? (size_t)WIN * (ANCH ? DFPITCH : NNFPitch<STAGE>::value) * 8 : 0);
}

// the deferred particles of k_stage: same arithmetic, global grids only
template <int SHAPE, int STAGE, int QMASK>
__global__ void __launch_bounds__(128) k_stage_overflow(const PartParams P)
{
    const int n = min(*P.ovf_count, P.ovf_cap);
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n; k += gridDim.x * blockDim.x) {
        const int tile = P.ovf_tile[k];
        const int64_t ent = P.ovf_p[k];
        process_direct<SHAPE, STAGE, QMASK, false>(P, ent & ~OVF_DEP, (ent & OVF_DEP) != 0, (tile / P.nty) * TILE, (tile % P.nty) * TILE, nullptr,
                                                   nullptr);
    }
}

// ---- PM2D_ORDER_RANDOM: no tile staging at all (BASELINE config 5, run A) -------------------------------------------
// one particle per thread in storage order; gather from the global force grid, integer atomics on the global grids
template <int SHAPE, int STAGE, int QMASK>
__global__ void __launch_bounds__(256) k_stage_random(const PartParams P, const int32_t *__restrict__ ptile, int64_t np)
{
    for (int64_t p = (int64_t)blockIdx.x * 256 + threadIdx.x; p < np; p += (int64_t)gridDim.x * 256) {
        const int tile = ptile[p];
        process_direct<SHAPE, STAGE, QMASK, false>(P, p, false, (tile / P.nty) * TILE, (tile % P.nty) * TILE, nullptr, nullptr);
        if (STAGE == 1) {     // the tile-relative fixed point covers cells -64 .. 191 of the loading tile
            const uint32_t cx = P.pv[p].x >> POS_FRAC_BITS, cy = P.pv[p].y >> POS_FRAC_BITS;
            if (cx < 4u || cx > 250u || cy < 4u || cy > 250u) P.flags[2] = 1;
        }
    }
}

}  // namespace

// =================================================================================================
// loader, binning, rebin
namespace {

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; r++) {
        uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

struct LoadParams {
    PV *pv;
    float *w;
    int64_t *id;
    const int32_t *chunk_tile;
    const int64_t *chunk_beg;
    const int64_t *tile_off;
    const int32_t *nchunks;
    int nx, ny, nty;
    int ppc_x, ppc_y, load, species;
    uint32_t seed_lo, seed_hi;
    double vth;
    int prof_kind, taper_cells, taper_cells_y;
    double p0, p1, p2;
    const int32_t *cell_off;     // NUMBER_WEIGHTED: the tile's cell runs give (cell, k) of a slot
    int layered;                 // storage order inside a tile: (rank in cell, cell) instead of (cell, rank)
    int sx0, sx1, sy0, sy1;      // pm2d_profile.slab resolved: cells with sx0 <= i < sx1, sy0 <= j < sy1 are loaded
};

// the loaded cells of a tile: rows [ri0, ri1) x columns [rj0, rj1), tile-relative (empty: ri1 <= ri0 or rj1 <= rj0)
struct TileRect {
    int ri0, ri1, rj0, rj1;
    __host__ __device__ int rows() const { return ri1 > ri0 ? ri1 - ri0 : 0; }
    __host__ __device__ int cols() const { return rj1 > rj0 ? rj1 - rj0 : 0; }
};
__host__ __device__ inline TileRect tile_rect(int gx0, int gy0, int nx, int ny, int sx0, int sx1, int sy0, int sy1)
{
    const int wx = min(TILE, nx - gx0), wy = min(TILE, ny - gy0);
    TileRect r;
    r.ri0 = min(max(sx0 - gx0, 0), wx); r.ri1 = min(max(sx1 - gx0, 0), wx);
    r.rj0 = min(max(sy0 - gy0, 0), wy); r.rj1 = min(max(sy1 - gy0, 0), wy);
    return r;
}

__device__ double profile_density(const LoadParams &L, int i)
{
    const double PI = 3.14159265358979323846;
    double xc = ((double)i + 0.5) / (double)L.nx, n;
    if (L.prof_kind == PM2D_PROFILE_UNIFORM) n = L.p0;
    else if (L.prof_kind == PM2D_PROFILE_LINEAR) n = L.p0 + (L.p1 - L.p0) * xc;
    else n = fmin(L.p0 * exp(xc * L.p1), L.p2);
    if (L.taper_cells > 0) {
        double d = fmin((double)i + 0.5, (double)L.nx - 0.5 - (double)i);
        if (d < (double)L.taper_cells) {
            double s = sin(0.5 * PI * d / (double)L.taper_cells);
            n = n * (PM2D_TAPER_FLOOR + (1.0 - PM2D_TAPER_FLOOR) * (s * s));
        }
    }
    return n;
}

// the same taper at the y walls (pm2d_profile.taper_cells_y)
__device__ double taper_y(const LoadParams &L, int j)
{
    const double PI = 3.14159265358979323846;
    if (L.taper_cells_y <= 0) return 1.0;
    const double d = fmin((double)j + 0.5, (double)L.ny - 0.5 - (double)j);
    if (d >= (double)L.taper_cells_y) return 1.0;
    const double s = sin(0.5 * PI * d / (double)L.taper_cells_y);
    return PM2D_TAPER_FLOOR + (1.0 - PM2D_TAPER_FLOOR) * (s * s);
}

// one CTA per chunk; a tile with wx*wy cells stores its cells row-major, ppc particles each:
// slot s holds particle k = s % ppc of the (s / ppc)-th cell
__global__ void __launch_bounds__(PTHREADS) k_load(const LoadParams L)
{
    const double PI = 3.14159265358979323846;
    const int chunk = blockIdx.x;
    if (chunk >= *L.nchunks) return;
    const int tile = L.chunk_tile[chunk];
    const int64_t t0 = L.tile_off[tile];
    const int64_t beg = L.chunk_beg[chunk];
    int64_t end = beg + CHUNK;
    if (L.tile_off[tile + 1] < end) end = L.tile_off[tile + 1];
    const int gx0 = (tile / L.nty) * TILE, gy0 = (tile % L.nty) * TILE;
    const TileRect tr = tile_rect(gx0, gy0, L.nx, L.ny, L.sx0, L.sx1, L.sy0, L.sy1);
    const int wy = max(tr.cols(), 1);                  // loaded columns per row of this tile
    const int ppc = L.ppc_x * L.ppc_y;
    for (int64_t p = beg + threadIdx.x; p < end; p += PTHREADS) {
        int s = (int)(p - t0);
        int li, lj, k;
        if (L.load == PM2D_NUMBER_WEIGHTED) {      // last cell whose run starts at or before slot s
            const int32_t *co = L.cell_off + (size_t)tile * CPITCH;
            int lo = 0, hi = TCELLS - 1;
            while (lo < hi) {
                int mid = (lo + hi + 1) >> 1;
                if (co[mid] <= s) lo = mid; else hi = mid - 1;
            }
            li = lo >> 5; lj = lo & 31; k = s - co[lo];
        } else if (L.layered) {                    // layer-major: the k-th particles of all cells are contiguous
            const int cells = tr.rows() * wy;
            k = s / cells;
            int lc = s - k * cells;
            li = lc / wy; lj = lc - li * wy;
            li += tr.ri0; lj += tr.rj0;
        } else {
            int lc = s / ppc;
            k = s - lc * ppc;
            li = lc / wy; lj = lc - li * wy;
            li += tr.ri0; lj += tr.rj0;
        }
        int64_t cell = (int64_t)(gx0 + li) * L.ny + (gy0 + lj);
        int64_t pid = (int64_t)k * ((int64_t)L.nx * L.ny) + cell;
        uint32_t r[4];
        philox4x32_10((uint32_t)(pid & 0xFFFFFFFF), (uint32_t)(pid >> 32), (uint32_t)L.species, 0u, L.seed_lo, L.seed_hi, r);
        uint32_t fx24, fy24;
        float ux = 0.f, uy = 0.f;
        if (L.load == PM2D_LATTICE_COLD) {
            fx24 = (uint32_t)floor((((double)(k / L.ppc_y)) + 0.5) / (double)L.ppc_x * 16777216.0);
            fy24 = (uint32_t)floor((((double)(k % L.ppc_y)) + 0.5) / (double)L.ppc_y * 16777216.0);
        } else {
            fx24 = r[0] >> 8;
            fy24 = r[1] >> 8;
            double U1 = ((double)r[2] + 1.0) * (1.0 / 4294967296.0), U2 = (double)r[3] * (1.0 / 4294967296.0);
            double R = L.vth * sqrt(-2.0 * log(U1));
            ux = (float)(R * cos(2.0 * PI * U2));
            uy = (float)(R * sin(2.0 * PI * U2));
        }
        PV out;
        out.x = ((uint32_t)(li + POS_BIAS) << POS_FRAC_BITS) | fx24;
        out.y = ((uint32_t)(lj + POS_BIAS) << POS_FRAC_BITS) | fy24;
        out.ux = ux;
        out.uy = uy;
        L.pv[p] = out;
        L.w[p] = L.load == PM2D_NUMBER_WEIGHTED ? (float)(L.p0 / (double)ppc) : (float)(profile_density(L, gx0 + li) * taper_y(L, gy0 + lj) / (double)ppc);
        if (L.id) L.id[p] = pid;
    }
}

// cell offsets of the loader's order: ppc particles in every cell of the slab (the whole box without one)
__global__ void k_uniform_cell_off(int32_t *cell_off, int ntiles, int nty, int nx, int ny, int ppc, int sx0, int sx1, int sy0, int sy1)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= (int64_t)ntiles * CPITCH) return;
    const int t = (int)(e / CPITCH), c = (int)(e - (int64_t)t * CPITCH);
    const int gx0 = (t / nty) * TILE, gy0 = (t % nty) * TILE;
    const TileRect tr = tile_rect(gx0, gy0, nx, ny, sx0, sx1, sy0, sy1);
    const int li = c >> 5, lj = c & 31;                 // c == TCELLS: li = 32
    // loaded cells before (li, lj) in row-major order
    const int full = min(max(li - tr.ri0, 0), tr.rows());
    const int part = (li >= tr.ri0 && li < tr.ri1) ? min(max(lj - tr.rj0, 0), tr.cols()) : 0;
    cell_off[e] = ppc * (full * tr.cols() + part);
}

// NUMBER_WEIGHTED: particles per cell = floor(ppc * taper(i) * filament(j) + U), U a Philox uniform of the cell
// (dithered rounding); one CTA per tile writes the tile's cell_off and its total
__global__ void __launch_bounds__(256) k_weighted_cell_off(int32_t *cell_off, int32_t *tile_cnt, const double *shape_y,
                                                           const double *taper_x, int nty, int nx, int ny, double ppc, int species,
                                                           uint32_t seed_lo, uint32_t seed_hi)
{
    __shared__ int32_t wsum[8];
    const int t = blockIdx.x, lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int gx0 = (t / nty) * TILE, gy0 = (t % nty) * TILE;
    int cnt[4], s = 0;
#pragma unroll
    for (int u = 0; u < 4; u++) {
        const int c = threadIdx.x * 4 + u, gi = gx0 + (c >> 5), gj = gy0 + (c & 31);
        cnt[u] = 0;
        if (gi < nx && gj < ny) {
            const int64_t cell = (int64_t)gi * ny + gj;
            uint32_t r[4];
            philox4x32_10((uint32_t)(cell & 0xFFFFFFFF), (uint32_t)(cell >> 32), (uint32_t)species, 1u, seed_lo, seed_hi, r);
            const double lam = __dmul_rn(__dmul_rn(ppc, taper_x[gi]), shape_y[gj]);
            cnt[u] = (int)floor(__dadd_rn(lam, (double)r[0] * (1.0 / 4294967296.0)));
        }
        s += cnt[u];
    }
    int incl = s;
    for (int o = 1; o < 32; o <<= 1) {
        int v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) wsum[wid] = incl;
    __syncthreads();
    int run = incl - s;
    for (int w = 0; w < wid; w++) run += wsum[w];
    int32_t *co = cell_off + (size_t)t * CPITCH;
#pragma unroll
    for (int u = 0; u < 4; u++) {
        co[threadIdx.x * 4 + u] = run;
        run += cnt[u];
    }
    if (threadIdx.x == 255) {
        co[TCELLS] = run;
        tile_cnt[t] = run;
    }
}

// ---- single-CTA scans over tiles ----------------------------------------------------------------
constexpr int SCAN_THREADS = 1024;

__device__ int64_t block_exclusive_scan(int64_t v, int64_t *total)
{
    __shared__ int64_t warp_sums[32];
    __shared__ int64_t grand;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int64_t incl = v;
    for (int o = 1; o < 32; o <<= 1) {
        int64_t t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    __syncthreads();
    if (lane == 31) warp_sums[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        int64_t s = warp_sums[lane], si = s;
        for (int o = 1; o < 32; o <<= 1) {
            int64_t t = __shfl_up_sync(0xffffffffu, si, o);
            if (lane >= o) si += t;
        }
        warp_sums[lane] = si - s;
        if (lane == 31) grand = si;
    }
    __syncthreads();
    *total = grand;
    return warp_sums[wid] + incl - v;
}

// tile_off[t] = exclusive scan of cnt[t]; tile_off[ntiles] = total
__global__ void __launch_bounds__(SCAN_THREADS) k_scan_tiles(const int32_t *cnt, int ntiles, int64_t *tile_off)
{
    const int per = (ntiles + SCAN_THREADS - 1) / SCAN_THREADS;
    const int t0 = threadIdx.x * per, t1 = min(ntiles, t0 + per);
    int64_t s = 0;
    for (int t = t0; t < t1; t++) s += cnt[t];
    int64_t total;
    int64_t run = block_exclusive_scan(s, &total);
    for (int t = t0; t < t1; t++) {
        tile_off[t] = run;
        run += cnt[t];
    }
    if (threadIdx.x == 0) tile_off[ntiles] = total;
}

// chunk list from tile offsets: tile t gets ceil(count/CHUNK) chunks
__global__ void __launch_bounds__(SCAN_THREADS) k_build_chunks(const int64_t *tile_off, int ntiles, int32_t *tile_first_chunk,
                                                               int32_t *chunk_tile, int64_t *chunk_beg, int32_t *nchunks,
                                                               int max_chunks, int32_t *flags)
{
    const int per = (ntiles + SCAN_THREADS - 1) / SCAN_THREADS;
    const int t0 = threadIdx.x * per, t1 = min(ntiles, t0 + per);
    int64_t s = 0;
    for (int t = t0; t < t1; t++) s += (tile_off[t + 1] - tile_off[t] + CHUNK - 1) / CHUNK;
    int64_t total;
    int64_t run = block_exclusive_scan(s, &total);
    if (total > max_chunks) {
        if (threadIdx.x == 0) { flags[1] = 1; *nchunks = 0; }
        return;
    }
    for (int t = t0; t < t1; t++) {
        int64_t b = tile_off[t], e = tile_off[t + 1];
        tile_first_chunk[t] = (int32_t)run;
        for (; b < e; b += CHUNK) {
            chunk_tile[run] = t;
            chunk_beg[run] = b;
            run++;
        }
    }
    if (threadIdx.x == 0) {
        tile_first_chunk[ntiles] = (int32_t)total;
        *nchunks = (int32_t)total;
    }
}

__global__ void k_uniform_tile_counts(int32_t *cnt, int ntx, int nty, int nx, int ny, int ppc, int sx0, int sx1, int sy0, int sy1)
{
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntx * nty) return;
    int gx0 = (t / nty) * TILE, gy0 = (t % nty) * TILE;
    const TileRect tr = tile_rect(gx0, gy0, nx, ny, sx0, sx1, sy0, sy1);
    cnt[t] = ppc * tr.rows() * tr.cols();
}

// ---- rebin, pass 1: stable move between neighbouring tiles ------------------------------------------
struct RebinParams {
    const PV *pv;
    const float *w;
    const int64_t *id;
    PV *pv2;
    float *w2;
    int64_t *id2;
    const int32_t *chunk_tile;
    const int64_t *chunk_beg;
    const int64_t *tile_off;
    const int64_t *tile_off2;
    const int32_t *nchunks;
    const int32_t *tile_first_chunk;
    int32_t *cnt9;
    int64_t *rel9;
    int32_t *newcount;
    int32_t *flags;
    int64_t *perm1;        // optional: for every slot after pass 1, the slot before it
    int nx, ny, ntx, nty;
    float predx, predy;    // lane order: free flight of half a rebin period in 2^-24 cells per unit velocity, else 0
};

// destination of a particle: tile displacement (dti, dtj) in {-1,0,1}^2 and the canonical slot
// (dti+1)*3 + c, where c folds y-displacements that reach the same tile when nty < 3
// Lane-order species (predx, predy != 0) are listed in the tile of their SORT position -- where free flight puts them half
// a rebin period from now (lane_sort_pos, pm2d_lanes.cu) -- so that over the period they stay within half a period's
// drift of their tile in either direction instead of a whole period's in one: 0.04 % of c3's electrons left the 2-cell
// halo of their window per stage at a period of 16 steps and went the slow way over the global grids.  A sort position
// beyond an x wall keeps the particle where it is (it will reflect).
__device__ __forceinline__ int rebin_slot(const RebinParams &R, int gx0, int gy0, const PV &me, int &dti, int &dtj, bool &bad)
{
    const int tw = min(TILE, R.nx - gx0), th = min(TILE, R.ny - gy0);
    const int cx = (int)(me.x >> POS_FRAC_BITS) - POS_BIAS, cy = (int)(me.y >> POS_FRAC_BITS) - POS_BIAS;
    const bool pred = R.predx != 0.f || R.predy != 0.f;
    int pcx = cx, pcy = cy;
    if (pred) {
        pcx = (int)(((int64_t)me.x + (int64_t)__float2int_rn(__fmul_rn(me.ux, R.predx))) >> POS_FRAC_BITS) - POS_BIAS;
        pcy = (int)(((int64_t)me.y + (int64_t)__float2int_rn(__fmul_rn(me.uy, R.predy))) >> POS_FRAC_BITS) - POS_BIAS;
    }
    dti = pcx < 0 ? -1 : (pcx >= tw ? 1 : 0);
    dtj = pcy < 0 ? -1 : (pcy >= th ? 1 : 0);
    int ti = gx0 / TILE + dti;
    if (pred && (ti < 0 || ti >= R.ntx)) {
        dti = 0;
        ti = gx0 / TILE;
    }
    const int nxr = cx - dti * TILE, nyr = cy - dtj * th;      // tile-relative cell after the move
    if (pred) bad = ti < 0 || ti >= R.ntx || nxr < -24 || nxr >= TILE + 24 || nyr < -24 || nyr >= TILE + 24;
    else bad = ti < 0 || ti >= R.ntx || nxr < 0 || nxr >= min(TILE, R.nx - ti * TILE) || nyr < 0 || nyr >= th;
    int c = R.nty == 1 ? 1 : (R.nty == 2 ? (dtj != 0 ? 2 : 1) : dtj + 1);
    return (dti + 1) * 3 + c;
}

__global__ void __launch_bounds__(PTHREADS) k_rebin_count(const RebinParams R)
{
    __shared__ int32_t cnt[9];
    const int chunk = blockIdx.x;
    if (chunk >= *R.nchunks) return;
    const int tile = R.chunk_tile[chunk];
    const int64_t beg = R.chunk_beg[chunk];
    int64_t end = beg + CHUNK;
    if (R.tile_off[tile + 1] < end) end = R.tile_off[tile + 1];
    const int gx0 = (tile / R.nty) * TILE, gy0 = (tile % R.nty) * TILE;
    if (threadIdx.x < 9) cnt[threadIdx.x] = 0;
    __syncthreads();
    int local[9] = {0, 0, 0, 0, 0, 0, 0, 0, 0};
    bool anybad = false;
    for (int64_t p = beg + threadIdx.x; p < end; p += PTHREADS) {
        int dti, dtj;
        bool bad;
        PV me = PV{0u, 0u, 0.f, 0.f};
        if (R.predx != 0.f || R.predy != 0.f) me = R.pv[p];
        else {
            const uint2 xy = *reinterpret_cast<const uint2 *>(&R.pv[p]);
            me.x = xy.x;
            me.y = xy.y;
        }
        int slot = rebin_slot(R, gx0, gy0, me, dti, dtj, bad);
        anybad |= bad;
#pragma unroll
        for (int s = 0; s < 9; s++) local[s] += (slot == s);
    }
#pragma unroll
    for (int s = 0; s < 9; s++) {
        int v = local[s];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0 && v) atomicAdd(&cnt[s], v);
    }
    if (anybad) R.flags[0] = 1;
    __syncthreads();
    if (threadIdx.x < 9) R.cnt9[(size_t)chunk * 9 + threadIdx.x] = cnt[threadIdx.x];
}

// one thread per destination tile: walk its (<= 9) source tiles in ascending key order, chunk by
// chunk, handing out offsets -> the new order is the stable counting sort of the old array by tile
__global__ void k_rebin_offsets(const RebinParams R)
{
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= R.ntx * R.nty) return;
    const int ti = t / R.nty, tj = t % R.nty;
    int skey[9], sslot[9], ns = 0;
    for (int dti = -1; dti <= 1; dti++) {
        int si = ti - dti;
        if (si < 0 || si >= R.ntx) continue;
        for (int c = 0; c < 3; c++) {
            int dtj;
            if (R.nty == 1) { if (c != 1) continue; dtj = 0; }
            else if (R.nty == 2) { if (c == 0) continue; dtj = c - 1; }
            else dtj = c - 1;
            int sj = ((tj - dtj) % R.nty + R.nty) % R.nty;
            int key = si * R.nty + sj, slot = (dti + 1) * 3 + c;
            int k = ns++;
            while (k > 0 && skey[k - 1] > key) { skey[k] = skey[k - 1]; sslot[k] = sslot[k - 1]; k--; }
            skey[k] = key; sslot[k] = slot;
        }
    }
    int64_t run = 0;
    for (int k = 0; k < ns; k++) {
        int c0 = R.tile_first_chunk[skey[k]], c1 = R.tile_first_chunk[skey[k] + 1];
        for (int c = c0; c < c1; c++) {
            R.rel9[(size_t)c * 9 + sslot[k]] = run;
            run += R.cnt9[(size_t)c * 9 + sslot[k]];
        }
    }
    R.newcount[t] = (int32_t)run;
}

__global__ void __launch_bounds__(PTHREADS) k_rebin_scatter(const RebinParams R)
{
    __shared__ int32_t wcnt[PTHREADS / 32][10];
    __shared__ int64_t run[10];
    const int chunk = blockIdx.x;
    if (chunk >= *R.nchunks) return;
    const int tile = R.chunk_tile[chunk];
    const int64_t beg = R.chunk_beg[chunk];
    int64_t end = beg + CHUNK;
    if (R.tile_off[tile + 1] < end) end = R.tile_off[tile + 1];
    const int gx0 = (tile / R.nty) * TILE, gy0 = (tile % R.nty) * TILE;
    const int th = min(TILE, R.ny - gy0);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (threadIdx.x < 10) run[threadIdx.x] = threadIdx.x < 9 ? R.rel9[(size_t)chunk * 9 + threadIdx.x] : 0;
    for (int64_t base = beg; base < end; base += PTHREADS) {
        const int64_t p = base + threadIdx.x;
        const bool live = p < end;
        int slot = 9, dti = 0, dtj = 0;
        PV me = {0u, 0u, 0.f, 0.f};
        bool bad = false;
        if (live) {
            me = R.pv[p];
            slot = rebin_slot(R, gx0, gy0, me, dti, dtj, bad);
        }
        if (lane < 10) wcnt[wid][lane] = 0;
        __syncthreads();
        unsigned peers = __match_any_sync(0xffffffffu, slot);
        int rank = __popc(peers & ((1u << lane) - 1u));
        if (rank == 0) wcnt[wid][slot] = __popc(peers);
        __syncthreads();
        if (live) {
            int64_t off = run[slot] + rank;
            for (int w2 = 0; w2 < wid; w2++) off += wcnt[w2][slot];
            int ti = gx0 / TILE + dti;
            ti = max(0, min(R.ntx - 1, ti));
            int tj = ((gy0 / TILE + dtj) % R.nty + R.nty) % R.nty;
            int dest = ti * R.nty + tj;
            int64_t q = R.tile_off2[dest] + off;
            if (bad) q = p;   // flagged by k_rebin_count; keep memory safe
            me.x -= (uint32_t)(dti * TILE) << POS_FRAC_BITS;
            me.y -= (uint32_t)(dtj * th) << POS_FRAC_BITS;
            R.pv2[q] = me;
            R.w2[q] = R.w[p];
            if (R.id) R.id2[q] = R.id[p];
            if (R.perm1) R.perm1[q] = p;
        }
        __syncthreads();
        if (threadIdx.x < 9) {
            int64_t s = 0;
            for (int w2 = 0; w2 < PTHREADS / 32; w2++) s += wcnt[w2][threadIdx.x];
            run[threadIdx.x] += s;
        }
        __syncthreads();
    }
}

// ---- rebin, pass 2: stable counting sort by cell inside every tile -----------------------------------
// One CTA per tile.  Each warp owns a contiguous part of the tile's list; per-warp histograms, one scan
// over (cell, warp), then every warp ranks its particles batch by batch with match_any -- the result is
// the stable sort by cell of the pass-1 order, hence (with pass 1) the stable sort by (tile, cell).
struct CellSortParams {
    const PV *src;
    const float *wsrc;
    const int64_t *idsrc;
    PV *dst;
    float *wdst;
    int64_t *iddst;
    const int64_t *tile_off;   // offsets of the pass-1 order (= of the result)
    int32_t *cell_off;
    const int64_t *perm1;      // optional (tests)
    int32_t *keys_out;         // optional: destination key of every particle, in the order before pass 1
    int64_t *perm_out;         // optional: for every final slot the slot before pass 1
};

constexpr int CS_WARPS = 8;

__device__ __forceinline__ int cell_of(uint32_t xf, uint32_t yf)
{
    int cx = (int)(xf >> POS_FRAC_BITS) - POS_BIAS, cy = (int)(yf >> POS_FRAC_BITS) - POS_BIAS;
    cx = max(0, min(TILE - 1, cx));
    cy = max(0, min(TILE - 1, cy));
    return cx * TILE + cy;
}

// LAYERED: inside the tile the particles are ordered by (rank in their cell; rank of the cell among the cells of its
// column that reach this rank; column) instead of (cell, rank): 32 consecutive particles then lie in 32 different
// cells of 32 different columns, which is what the thread-per-particle stage kernel wants (with the deposit windows
// on pitch 64 the bank of a node is its column: the shared atomics of a warp spread over the banks).  Ranks
// >= LAYERS form a cell-major tail.  Shared memory: hist | cr[LAYERS][TCELLS] (uint8) | cellbeg | tb | lay | T | M.
constexpr int LAYERS = PM2D_LAYERS;
constexpr size_t CELLSORT_LAYERED_SMEM = (size_t)CS_WARPS * TCELLS * 4 + (size_t)LAYERS * TCELLS + (size_t)(TCELLS + 1) * 4 +
                                         (size_t)TCELLS * 4 + (LAYERS + 2) * 4 + (size_t)LAYERS * (TILE + 1) * 4 + (size_t)LAYERS * TILE * 4 + 64;

template <bool LAYERED>
__global__ void __launch_bounds__(CS_WARPS * 32) k_cellsort(const CellSortParams C)
{
    extern __shared__ int32_t cs_smem[];
    int32_t *hist = cs_smem;                                                  // [CS_WARPS][TCELLS]
    uint8_t *cr = reinterpret_cast<uint8_t *>(hist + CS_WARPS * TCELLS);      // [LAYERS][TCELLS] (LAYERED)
    int32_t *cellbeg = LAYERED ? reinterpret_cast<int32_t *>(cr + LAYERS * TCELLS) : hist + CS_WARPS * TCELLS;   // [TCELLS+1]
    int32_t *tb = cellbeg + TCELLS + 1;                                       // [TCELLS] (LAYERED)
    int32_t *lay = LAYERED ? tb + TCELLS : cellbeg + TCELLS + 1;              // [LAYERS+2] layer offsets, tail offset
    int32_t *Tt = lay + LAYERS + 2;                                           // [LAYERS][TILE+1] (LAYERED)
    uint32_t *Mm = reinterpret_cast<uint32_t *>(Tt + LAYERS * (TILE + 1));    // [LAYERS][TILE] (LAYERED)
    __shared__ int32_t wsum[CS_WARPS];
    const int tile = blockIdx.x;
    const int64_t t0 = C.tile_off[tile];
    const int64_t n = C.tile_off[tile + 1] - t0;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    int32_t *co = C.cell_off + (size_t)tile * CPITCH;
    for (int e = threadIdx.x; e < CS_WARPS * TCELLS; e += CS_WARPS * 32) hist[e] = 0;
    __syncthreads();
    int64_t per = (n + CS_WARPS - 1) / CS_WARPS;
    per = (per + 31) & ~(int64_t)31;
    const int64_t beg = min(n, wid * per), end = min(n, beg + per);
    int32_t *myhist = hist + wid * TCELLS;
    for (int64_t i0 = beg + lane; i0 < end; i0 += 4 * 32) {      // four loads in flight per lane
        uint2 xy[4];
#pragma unroll
        for (int u = 0; u < 4; u++)
            if (i0 + 32 * u < end) xy[u] = *reinterpret_cast<const uint2 *>(&C.src[t0 + i0 + 32 * u]);
#pragma unroll
        for (int u = 0; u < 4; u++)
            if (i0 + 32 * u < end) atomicAdd(&myhist[cell_of(xy[u].x, xy[u].y)], 1);
    }
    __syncthreads();
    {   // exclusive scan over (cell, warp): thread t owns cells 4t .. 4t+3
        const int c0 = threadIdx.x * (TCELLS / (CS_WARPS * 32));
        int s = 0;
        for (int c = c0; c < c0 + TCELLS / (CS_WARPS * 32); c++)
            for (int w = 0; w < CS_WARPS; w++) s += hist[w * TCELLS + c];
        int incl = s;
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) wsum[wid] = incl;
        __syncthreads();
        int run = incl - s;
        for (int w = 0; w < wid; w++) run += wsum[w];
        for (int c = c0; c < c0 + TCELLS / (CS_WARPS * 32); c++) {
            co[c] = run;
            cellbeg[c] = run;
            for (int w = 0; w < CS_WARPS; w++) {
                int v = hist[w * TCELLS + c];
                hist[w * TCELLS + c] = run;
                run += v;
            }
        }
        if (threadIdx.x == CS_WARPS * 32 - 1) {
            co[TCELLS] = run;
            cellbeg[TCELLS] = run;
        }
    }
    __syncthreads();
    if (LAYERED) {
        // Layer r (r < LAYERS) holds one particle of every cell with more than r particles, ordered by (k, j): j the
        // cell's column (the lane direction of the stage kernel), k the rank of the cell among the occupied cells of
        // its column.  Any 32 consecutive slots of a layer then lie in (almost always) 32 different columns, also in
        // the sparse upper layers; a full layer is simply row-major.  Tables:
        //   cr[r][c]  = k of cell c in layer r          occ (implicit)  = occupied cells of column j in layer r
        //   T[r][k]   = slots of layer r with rank < k = sum_j min(occ_j, k)
        //   M[r][k]   = bit j set: column j has more than k occupied cells
        //   lay[r]    = first slot of layer r; lay[LAYERS] = first slot of the cell-major tail, tb[c] its cell offsets
        static_assert(LAYERS == 16 && TILE == 32 && CS_WARPS * 32 * 2 == LAYERS * TILE, "two (layer, column) tasks per thread");
        __shared__ uint8_t occ[LAYERS][TILE];
        __shared__ int32_t wsumt[CS_WARPS];
#pragma unroll
        for (int t = 0; t < 2; t++) {
            const int task = threadIdx.x + t * CS_WARPS * 32, r = task >> 5, j = task & 31;
            int run = 0;
            for (int i = 0; i < TILE; i++) {
                const int c = i * TILE + j;
                if (cellbeg[c + 1] - cellbeg[c] > r) cr[r * TCELLS + c] = (uint8_t)run++;
            }
            occ[r][j] = (uint8_t)run;
        }
        constexpr int PER = TCELLS / (CS_WARPS * 32);
        const int c0 = threadIdx.x * PER;
        int loct = 0;
#pragma unroll
        for (int u = 0; u < PER; u++) loct += max(cellbeg[c0 + u + 1] - cellbeg[c0 + u] - LAYERS, 0);
        int inct = loct;
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, inct, o);
            if (lane >= o) inct += t;
        }
        if (lane == 31) wsumt[wid] = inct;
        __syncthreads();
        for (int task = threadIdx.x; task < LAYERS * (TILE + 1); task += CS_WARPS * 32) {
            const int r = task / (TILE + 1), k = task - r * (TILE + 1);
            int sum = 0;
            uint32_t mask = 0u;
            for (int j = 0; j < TILE; j++) {
                const int o = occ[r][j];
                sum += min(o, k);
                if (o > k) mask |= 1u << j;
            }
            Tt[r * (TILE + 1) + k] = sum;
            if (k < TILE) Mm[r * TILE + k] = mask;
        }
        {
            int runt = inct - loct;
            for (int w = 0; w < wid; w++) runt += wsumt[w];
#pragma unroll
            for (int u = 0; u < PER; u++) {
                tb[c0 + u] = runt;
                runt += max(cellbeg[c0 + u + 1] - cellbeg[c0 + u] - LAYERS, 0);
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            int slot = 0;
            for (int r = 0; r < LAYERS; r++) {
                lay[r] = slot;
                slot += Tt[r * (TILE + 1) + TILE];
            }
            lay[LAYERS] = slot;
        }
        __syncthreads();
    }
    for (int64_t base0 = beg; base0 < end; base0 += 4 * 32) {    // the records of four batches are loaded ahead of their ranking
        PV mv[4];
        float wv[4];
#pragma unroll
        for (int u = 0; u < 4; u++) {
            const int64_t i = base0 + 32 * u + lane;
            mv[u] = PV{0u, 0u, 0.f, 0.f};
            wv[u] = 0.f;
            if (i < end) {
                mv[u] = C.src[t0 + i];
                wv[u] = C.wsrc[t0 + i];
            }
        }
#pragma unroll
        for (int u = 0; u < 4; u++) {
            const int64_t base = base0 + 32 * u;
            if (base >= end) break;                      // warp-uniform
            const int64_t i = base + lane;
            const bool live = i < end;
            const PV me = mv[u];
            int c = TCELLS + lane;                       // dead lanes: unique keys
            if (live) c = cell_of(me.x, me.y);
            const unsigned peers = __match_any_sync(0xffffffffu, c);
            const int rank = __popc(peers & ((1u << lane) - 1u));
            const int leader = __ffs(peers) - 1;
            int b = 0;
            if (live && lane == leader) {
                b = myhist[c];
                myhist[c] = b + __popc(peers);
            }
            b = __shfl_sync(0xffffffffu, b, leader);
            __syncwarp();
            if (live) {
                int64_t q = t0 + b + rank;                 // cell-major slot
                if (LAYERED) {
                    const int r = b + rank - cellbeg[c];   // stable rank of the particle in its cell
                    if (r < LAYERS) {
                        const int k = cr[r * TCELLS + c], j = c & (TILE - 1);
                        q = t0 + lay[r] + Tt[r * (TILE + 1) + k] + __popc(Mm[r * TILE + k] & ((1u << j) - 1u));
                    } else
                        q = t0 + lay[LAYERS] + tb[c] + (r - LAYERS);
                }
                C.dst[q] = me;
                C.wdst[q] = wv[u];
                if (C.idsrc) C.iddst[q] = C.idsrc[t0 + i];
                if (C.perm1) {
                    const int64_t old = C.perm1[t0 + i];
                    if (C.keys_out) C.keys_out[old] = tile * TCELLS + c;
                    if (C.perm_out) C.perm_out[q] = old;
                }
            }
        }
    }
}

// A pseudo-random bijection of [0, n): four Feistel rounds on 2 * hb bits, walked until the image is < n.
__device__ __forceinline__ uint32_t mix32(uint32_t x)
{
    x ^= x >> 16; x *= 0x7feb352du;
    x ^= x >> 15; x *= 0x846ca68bu;
    x ^= x >> 16;
    return x;
}
__device__ __forceinline__ int64_t feistel_perm(int64_t q, int64_t n, int hb, uint32_t key)
{
    const uint32_t mask = (1u << hb) - 1u;
    do {
        uint32_t L = (uint32_t)(q >> hb) & mask, R = (uint32_t)q & mask;
#pragma unroll
        for (int r = 0; r < 4; r++) {
            const uint32_t t = L ^ (mix32(R * 0x9E3779B1u + key + 0x632BE5ABu * (uint32_t)r) & mask);
            L = R;
            R = t;
        }
        q = ((int64_t)L << hb) | R;
    } while (q >= n);
    return q;
}

// slot q takes the particle of slot perm(q) of the tile-ordered arrays, and remembers its tile
__global__ void __launch_bounds__(256) k_shuffle_random(const PV *pv, const float *w, const int64_t *id, PV *pv2, float *w2, int64_t *id2,
                                                        int32_t *ptile, const int64_t *tile_off, int ntiles, int64_t np, int hb, uint32_t key)
{
    for (int64_t q = (int64_t)blockIdx.x * 256 + threadIdx.x; q < np; q += (int64_t)gridDim.x * 256) {
        const int64_t src = feistel_perm(q, np, hb, key);
        int lo = 0, hi = ntiles;                 // last tile with tile_off[tile] <= src
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (tile_off[mid] <= src) lo = mid; else hi = mid;
        }
        pv2[q] = pv[src];
        w2[q] = w[src];
        if (id) id2[q] = id[src];
        ptile[q] = lo;
    }
}

// canonical (ix, iy, fx, fy) and velocity of the particles of each chunk, as separate arrays
__global__ void __launch_bounds__(PTHREADS) k_unpack(const PV *pv, const int32_t *chunk_tile, const int64_t *chunk_beg,
                                                     const int64_t *tile_off, const int32_t *nchunks, int nty, int ny, int32_t *ix,
                                                     int32_t *iy, float *fx, float *fy, float *ux, float *uy, const int32_t *ptile)
{
    const int chunk = blockIdx.x;
    if (chunk >= *nchunks) return;
    const int ctile = chunk_tile[chunk];
    const int64_t beg = chunk_beg[chunk];
    int64_t end = beg + CHUNK;
    if (tile_off[ctile + 1] < end) end = tile_off[ctile + 1];
    for (int64_t p = beg + threadIdx.x; p < end; p += PTHREADS) {
        const int tile = ptile ? ptile[p] : ctile;      // random order: the slots of a chunk hold particles of any tile
        const int gx0 = (tile / nty) * TILE, gy0 = (tile % nty) * TILE;
        const PV me = pv[p];
        ix[p] = gx0 + (int)(me.x >> POS_FRAC_BITS) - POS_BIAS;
        iy[p] = (gy0 + (int)(me.y >> POS_FRAC_BITS) - POS_BIAS) & (ny - 1);
        fx[p] = (float)(me.x & POS_FRAC_MASK) * (1.0f / 16777216.0f);
        fy[p] = (float)(me.y & POS_FRAC_MASK) * (1.0f / 16777216.0f);
        ux[p] = me.ux;
        uy[p] = me.uy;
    }
}

}  // namespace

// =================================================================================================
// host launchers
PartParams make_part_params(pm2d_ctx *c, int s)
{
    SpeciesDev &S = c->sp[s];
    PartParams P;
    P.pv = S.pv; P.uh = S.uh; P.w = S.w;
    P.tile_off = S.tile_off; P.cell_off = S.cell_off;
    P.F = S.F;
    P.nfix = S.nfix; P.pxfix = S.pxfix; P.pyfix = S.pyfix; P.flags = c->flags;
    P.stray_total = c->stray_total;
    P.zeros = c->zeros;
    P.ovf_p = c->ovf_p; P.ovf_tile = c->ovf_tile; P.ovf_count = c->ovf_count; P.ovf_cap = c->ovf_cap;
    P.nx = c->g.nx; P.ny = c->g.ny; P.nty = c->nty;
    P.dt = (float)c->dtp;                                   // particle step: S wave steps (Q21)
    P.hx = (float)(c->dtp / (2.0 * c->g.dx));
    P.hy = (float)(c->dtp / (2.0 * c->g.dy));
    P.nscale = c->nscale; P.pscale = c->pscale;
    P.pratio = c->pscale / c->nscale;
    P.half_dd = (float)(0.5 * S.cfg.DD);
    P.dd = (float)S.cfg.DD;
    P.k_rad = (float)(3.14159265358979323846 / S.cfg.DD);
    P.cap_extra = c->cap_extra;
    P.sparse_cap = 2;
    P.w4_slope = (float)(-3.14159265358979323846 / S.cfg.DD / 16777216.0);
    P.w4_off = (float)((0.5 * S.cfg.DD - 0.5) * 3.14159265358979323846 / S.cfg.DD);
    P.sub0 = S.sub0;
    P.lane_exp = S.lane_exp;
    P.ucap = (float)lane_ucap(S);
    const float gs = S.cfg.shape == PM2D_SINE ? 0.25f : 1.f;
    P.hx24 = P.hx * 16777216.0f;
    P.hy24 = P.hy * 16777216.0f;
    P.lane_dt = gs * P.dt;
    P.lane_dt_half = 0.5f * gs * P.dt;
    P.lane_qns = gs * P.nscale;
    return P;
}

constexpr int STRIP = 8;   // cells per strip thread: 128 threads per tile

template <int SHAPE>
static void launch_stage_shape(const PartParams &P, int stage, int qmask, int grid, bool sparse, bool anch, cudaStream_t st)
{
#define PM2D_LAUNCH(ST, Q)                                                         \
    do {                                                                           \
        if (sparse && anch) {                                                      \
            static bool once_ = false;                                             \
            if (!once_) {                                                          \
                cudaFuncSetAttribute(k_stage_direct<SHAPE, ST, Q, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)direct_smem_bytes<ST, Q, true>()); \
                once_ = true;                                                      \
            }                                                                      \
            k_stage_direct<SHAPE, ST, Q, true><<<grid, 256, direct_smem_bytes<ST, Q, true>(), st>>>(P); \
        } else if (sparse)                                                         \
            k_stage_direct<SHAPE, ST, Q, false><<<grid, 256, direct_smem_bytes<ST, Q, false>(), st>>>(P); \
        else k_stage<SHAPE, ST, Q, STRIP><<<grid * STRIP_SPLIT, TCELLS / STRIP, 0, st>>>(P); \
        k_stage_overflow<SHAPE, ST, Q><<<148 * 8, 128, 0, st>>>(P);                    \
    } while (0)
    if (stage == 0) { if (qmask == 3) PM2D_LAUNCH(0, 3); else PM2D_LAUNCH(0, 1); }
    else if (stage == 1) { if (qmask == 3) PM2D_LAUNCH(1, 3); else PM2D_LAUNCH(1, 1); }
    else { if (qmask == 3) PM2D_LAUNCH(2, 3); else if (qmask == 2) PM2D_LAUNCH(2, 2); else PM2D_LAUNCH(2, 1); }
#undef PM2D_LAUNCH
}

// stage 0 / 1: the caller has put the nodal force of the stage into S.F and zeroed the target deposit set
static int launch_stage_any(pm2d_ctx *c, int s, int stage, int qmask)
{
    SpeciesDev &S = c->sp[s];
    if (S.np == 0) return PM2D_OK;
    if (S.lanes) return launch_stage_lanes(c, s, stage, qmask);
    PartParams P = make_part_params(c, s);
    PM2D_CUDA_CHECK(cudaMemsetAsync(c->ovf_count, 0, sizeof(int32_t), c->stream));
    if (stage == 0) {          // stage A deposits (x^, u^) into the second set (zeroed by the caller's side stream)
        P.nfix = S.nhat; P.pxfix = S.pxhat; P.pyfix = S.pyhat;
    }
    if (S.random) {
        const int grid = (int)std::min<int64_t>((S.np + 255) / 256, (int64_t)148 * 64);
#define PM2D_LAUNCH_R(SH)                                                                                              \
        do {                                                                                                           \
            if (stage == 0) { if (qmask == 3) k_stage_random<SH, 0, 3><<<grid, 256, 0, c->stream>>>(P, S.ptile, S.np); \
                              else k_stage_random<SH, 0, 1><<<grid, 256, 0, c->stream>>>(P, S.ptile, S.np); }          \
            else if (stage == 1) { if (qmask == 3) k_stage_random<SH, 1, 3><<<grid, 256, 0, c->stream>>>(P, S.ptile, S.np); \
                                   else k_stage_random<SH, 1, 1><<<grid, 256, 0, c->stream>>>(P, S.ptile, S.np); }     \
            else if (qmask == 3) k_stage_random<SH, 2, 3><<<grid, 256, 0, c->stream>>>(P, S.ptile, S.np);              \
            else if (qmask == 2) k_stage_random<SH, 2, 2><<<grid, 256, 0, c->stream>>>(P, S.ptile, S.np);              \
            else k_stage_random<SH, 2, 1><<<grid, 256, 0, c->stream>>>(P, S.ptile, S.np);                              \
        } while (0)
        if (S.cfg.shape == PM2D_CIC) PM2D_LAUNCH_R(PM2D_CIC);
        else if (S.cfg.shape == PM2D_TSC) PM2D_LAUNCH_R(PM2D_TSC);
        else PM2D_LAUNCH_R(PM2D_SINE);
#undef PM2D_LAUNCH_R
        count_launch(c, 1);
        PM2D_CUDA_CHECK(cudaGetLastError());
        return PM2D_OK;
    }
    // layered species take the thread-per-particle kernel, cell-major ones the strip kernel
    const bool sparse = S.layered;
    // thermal drift between two rebins, in cells: below a tenth of a cell the particles are (almost all) still in the
    // cells they were sorted into
    const bool anch = sqrt(S.vth2) * c->dtp / fmin(c->g.dx, c->g.dy) * (double)(c->g.rebin_every > 0 ? c->g.rebin_every : 32) < 0.1;
    if (S.cfg.shape == PM2D_CIC) launch_stage_shape<PM2D_CIC>(P, stage, qmask, c->ntiles, sparse, anch, c->stream);
    else if (S.cfg.shape == PM2D_TSC) launch_stage_shape<PM2D_TSC>(P, stage, qmask, c->ntiles, sparse, anch, c->stream);
    else launch_stage_shape<PM2D_SINE>(P, stage, qmask, c->ntiles, sparse, anch, c->stream);
    count_launch(c, 2);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}


void launch_stage_overflow(const PartParams &P, int shape, int stage, int qmask, cudaStream_t st)
{
#define PM2D_OVF(SH, ST, Q) k_stage_overflow<SH, ST, Q><<<148 * 8, 128, 0, st>>>(P)
#define PM2D_OVF_SHAPE(SH)                                                                   \
    do {                                                                                     \
        if (stage == 0) { if (qmask == 3) PM2D_OVF(SH, 0, 3); else PM2D_OVF(SH, 0, 1); }       \
        else if (stage == 1) { if (qmask == 3) PM2D_OVF(SH, 1, 3); else PM2D_OVF(SH, 1, 1); }  \
        else if (qmask == 3) PM2D_OVF(SH, 2, 3);                                             \
        else if (qmask == 2) PM2D_OVF(SH, 2, 2);                                             \
        else PM2D_OVF(SH, 2, 1);                                                             \
    } while (0)
    if (shape == PM2D_CIC) PM2D_OVF_SHAPE(PM2D_CIC);
    else if (shape == PM2D_TSC) PM2D_OVF_SHAPE(PM2D_TSC);
    else PM2D_OVF_SHAPE(PM2D_SINE);
#undef PM2D_OVF_SHAPE
#undef PM2D_OVF
}

int launch_stage(pm2d_ctx *c, int s, int stage)
{
    return launch_stage_any(c, s, stage, c->g.eager_moments ? 3 : 1);
}

int launch_deposit_only(pm2d_ctx *c, int s, bool density, bool momentum)
{
    int q = (density ? 1 : 0) | (momentum ? 2 : 0);
    if (!q) return PM2D_OK;
    return launch_stage_any(c, s, 2, q);
}

int launch_build_chunks(pm2d_ctx *c, int s)
{
    SpeciesDev &S = c->sp[s];
    k_build_chunks<<<1, SCAN_THREADS, 0, c->stream>>>(S.tile_off, c->ntiles, S.tile_first_chunk, S.chunk_tile, S.chunk_beg,
                                                       S.nchunks_dev, S.max_chunks, c->flags);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}

int launch_load_particles(pm2d_ctx *c, int s)
{
    SpeciesDev &S = c->sp[s];
    const int ppc = S.cfg.ppc_x * S.cfg.ppc_y;
    const int32_t *sl = c->profile.slab;
    const bool whole = !(sl[0] | sl[1] | sl[2] | sl[3]);
    const int sx0 = whole ? 0 : sl[0], sx1 = whole ? c->g.nx : sl[1], sy0 = whole ? 0 : sl[2], sy1 = whole ? c->g.ny : sl[3];
    if (S.cfg.load == PM2D_NUMBER_WEIGHTED) {
        k_weighted_cell_off<<<c->ntiles, 256, 0, c->stream>>>(S.cell_off, S.tile_cnt, c->shape_y, c->taper_x, c->nty, c->g.nx, c->g.ny,
                                                              (double)ppc, s, (uint32_t)(c->seed & 0xFFFFFFFFu), (uint32_t)(c->seed >> 32));
        k_scan_tiles<<<1, SCAN_THREADS, 0, c->stream>>>(S.tile_cnt, c->ntiles, S.tile_off);
        count_launch(c, 2);
        int64_t total = 0;
        PM2D_CUDA_CHECK(cudaMemcpyAsync(&total, S.tile_off + c->ntiles, sizeof(total), cudaMemcpyDeviceToHost, c->stream));
        PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
        if (total > S.cap) {
            pm2d_set_error("NUMBER_WEIGHTED: capacity is smaller than the number of particles the profile asks for");
            return PM2D_ENOMEM;
        }
        S.np = total;
    } else {
        k_uniform_tile_counts<<<(c->ntiles + 255) / 256, 256, 0, c->stream>>>(S.tile_cnt, c->ntx, c->nty, c->g.nx, c->g.ny, ppc, sx0, sx1, sy0, sy1);
        k_scan_tiles<<<1, SCAN_THREADS, 0, c->stream>>>(S.tile_cnt, c->ntiles, S.tile_off);
        const int64_t ncell = (int64_t)c->ntiles * CPITCH;
        k_uniform_cell_off<<<(unsigned)((ncell + 255) / 256), 256, 0, c->stream>>>(S.cell_off, c->ntiles, c->nty, c->g.nx, c->g.ny, ppc, sx0, sx1,
                                                                                   sy0, sy1);
        count_launch(c, 3);
        S.np = (int64_t)(sx1 - sx0) * (sy1 - sy0) * ppc;          // the slab's cells; capacity stays that of the whole box
    }
    int rc = launch_build_chunks(c, s);
    if (rc) return rc;
    LoadParams L;
    L.pv = S.pv; L.w = S.w; L.id = S.id;
    L.chunk_tile = S.chunk_tile; L.chunk_beg = S.chunk_beg; L.tile_off = S.tile_off; L.nchunks = S.nchunks_dev;
    L.nx = c->g.nx; L.ny = c->g.ny; L.nty = c->nty;
    L.ppc_x = S.cfg.ppc_x; L.ppc_y = S.cfg.ppc_y; L.load = S.cfg.load; L.species = s;
    L.seed_lo = (uint32_t)(c->seed & 0xFFFFFFFFu); L.seed_hi = (uint32_t)(c->seed >> 32);
    L.vth = sqrt(S.cfg.T_keV / 511.0 / S.cfg.mass);
    L.prof_kind = c->profile.kind; L.taper_cells = c->profile.taper_cells; L.taper_cells_y = c->profile.taper_cells_y;
    L.p0 = c->profile.p[0]; L.p1 = c->profile.p[1]; L.p2 = c->profile.p[2];
    L.cell_off = S.cell_off;
    L.layered = S.layered ? 1 : 0;
    L.sx0 = sx0; L.sx1 = sx1; L.sy0 = sy0; L.sy1 = sy1;
    k_load<<<S.max_chunks, PTHREADS, 0, c->stream>>>(L);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}

// PM2D_ORDER_RANDOM: permute the freshly loaded (tile-ordered) arrays into the second buffers and make those current
int launch_shuffle_random(pm2d_ctx *c, int s)
{
    SpeciesDev &S = c->sp[s];
    if (S.np == 0) return PM2D_OK;
    int bits = 1;
    while (((int64_t)1 << bits) < S.np) bits++;
    const int hb = (bits + 1) / 2;
    const int grid = (int)std::min<int64_t>((S.np + 255) / 256, (int64_t)148 * 64);
    k_shuffle_random<<<grid, 256, 0, c->stream>>>(S.pv, S.w, S.id, S.pv2, S.w2, S.id2, S.ptile, S.tile_off, c->ntiles, S.np, hb,
                                                  (uint32_t)(c->seed * 0x9E3779B97F4A7C15ull >> 32) + (uint32_t)s);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    std::swap(S.pv, S.pv2);
    std::swap(S.w, S.w2);
    std::swap(S.id, S.id2);
    return PM2D_OK;
}

// keys_dev / perm_dev: optional outputs of the test entry point pm2d_rebin; perm_tmp_dev: scratch of np
// int64, required when either is given
int launch_rebin(pm2d_ctx *c, int s, int32_t *keys_dev, int64_t *perm_dev, int64_t *perm_tmp_dev)
{
    SpeciesDev &S = c->sp[s];
    if (S.np == 0) return PM2D_OK;
    RebinParams R;
    R.pv = S.pv; R.w = S.w; R.id = S.id;
    R.pv2 = S.pv2; R.w2 = S.w2; R.id2 = S.id2;
    R.chunk_tile = S.chunk_tile; R.chunk_beg = S.chunk_beg; R.tile_off = S.tile_off; R.tile_off2 = S.tile_off2;
    R.nchunks = S.nchunks_dev; R.tile_first_chunk = S.tile_first_chunk;
    R.cnt9 = S.chunk_cnt9; R.rel9 = S.chunk_rel9; R.newcount = S.tile_cnt; R.flags = c->flags;
    R.perm1 = (keys_dev || perm_dev) ? perm_tmp_dev : nullptr;
    R.nx = c->g.nx; R.ny = c->g.ny; R.ntx = c->ntx; R.nty = c->nty;
    R.predx = S.lanes ? lane_pred(c, 0) : 0.f;
    R.predy = S.lanes ? lane_pred(c, 1) : 0.f;
    k_rebin_count<<<S.max_chunks, PTHREADS, 0, c->stream>>>(R);
    k_rebin_offsets<<<(c->ntiles + 127) / 128, 128, 0, c->stream>>>(R);
    k_scan_tiles<<<1, SCAN_THREADS, 0, c->stream>>>(S.tile_cnt, c->ntiles, S.tile_off2);
    k_rebin_scatter<<<S.max_chunks, PTHREADS, 0, c->stream>>>(R);
    if (S.lanes) {
        int rc = launch_lanesort(c, s, false, keys_dev, perm_dev, R.perm1);
        if (rc) return rc;
        count_launch(c, 4);
        std::swap(S.tile_off, S.tile_off2);
        return launch_build_chunks(c, s);
    }
    CellSortParams C;
    C.src = S.pv2; C.wsrc = S.w2; C.idsrc = S.id ? S.id2 : nullptr;
    C.dst = S.pv; C.wdst = S.w; C.iddst = S.id;
    C.tile_off = S.tile_off2; C.cell_off = S.cell_off;
    C.perm1 = R.perm1; C.keys_out = keys_dev; C.perm_out = perm_dev;
    if (S.layered) PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_cellsort<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)CELLSORT_LAYERED_SMEM));
    if (S.layered) k_cellsort<true><<<c->ntiles, CS_WARPS * 32, CELLSORT_LAYERED_SMEM, c->stream>>>(C);
    else k_cellsort<false><<<c->ntiles, CS_WARPS * 32, (size_t)CS_WARPS * TCELLS * 4 + (TCELLS + 1) * 4 + 64 * 4, c->stream>>>(C);
    count_launch(c, 5);
    PM2D_CUDA_CHECK(cudaGetLastError());
    std::swap(S.tile_off, S.tile_off2);
    return launch_build_chunks(c, s);
}

int launch_unpack_particles(pm2d_ctx *c, int s, int32_t *ix, int32_t *iy, float *fx, float *fy, float *ux, float *uy)
{
    SpeciesDev &S = c->sp[s];
    if (S.np == 0) return PM2D_OK;
    k_unpack<<<S.max_chunks, PTHREADS, 0, c->stream>>>(S.pv, S.chunk_tile, S.chunk_beg, S.tile_off, S.nchunks_dev, c->nty, c->g.ny,
                                                        ix, iy, fx, fy, ux, uy, S.random ? S.ptile : nullptr);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}
