// pm2d_particle_dev.cuh -- device helpers shared by the particle kernels (pm2d_particles.cu, pm2d_lanes.cu):
// kernel parameters, shape weights (Eqs. 12-13), fixed-point position helpers, and the per-particle stage
// code on 3 x 3 nodes (shared windows or global grids).  Each translation unit gets its own copy.
#pragma once
#include "pm2d_internal.h"

struct PartParams {
    // particles
    PV *pv;
    float2 *uh;
    const float *w;
    const int64_t *tile_off;
    const int32_t *cell_off;
    // grids
    const float2 *F;          // nodal force of this species, Eq. 16 (stage A) / Eq. 18 (stage B)
    int32_t *nfix, *pxfix, *pyfix;
    int32_t *flags;
    unsigned long long *stray_total;   // statistics: particles served outside the register patch
    const int32_t *zeros;              // PM2D_ZEROS_BYTES of zeros (bulk zero fill of the lanes windows)
    int64_t *ovf_p;           // overflow list: particles whose gather footprint left the tile window
    int32_t *ovf_tile, *ovf_count;
    int ovf_cap;
    int nx, ny, nty;
    float dt, hx, hy;        // hx = dt / (2 dx): cells per unit (u' + u)
    float nscale, pscale;
    float pratio;            // pscale / nscale
    float half_dd;           // DD / 2
    float dd;                // DD
    float k_rad;             // pi / DD  (sine: G(t) = 1/2 - 1/2 cos(k_rad t))
    float w4_slope, w4_off;  // sine weights4: cosine argument = rel * w4_slope + w4_off
    int sparse_cap;          // cell_cap of sparse tiles (mean <= 1.5 per cell)
    int cap_extra;           // cell_cap = ceil(mean particles per cell of the tile) + cap_extra
    // lane order (pm2d_lanes.cu): the shared windows count in units of 2^sn (density) / 2^sp (momentum) global units so
    // that one contribution stays below 2^22 and float -> int is one FFMA with the constant 1.5 * 2^23
    const int32_t *sub0;     // [ntiles] particles of sub-tile 0
    const int32_t *lane_exp; // [ntiles] sn | sp << 8
    float ucap;              // |u| beyond this takes the exact (F2I) path
    // constants of k_stage_lanes that differ from the above by powers of two only (exact on the host): GS = 1/4 for the
    // sine cloud (the 1/2 of each axis' G = (1 - cos)/2), 1 otherwise
    float hx24, hy24;        // hx 2^24, hy 2^24: displacement in units of 2^-24 cell per unit (u' + u)
    float lane_dt;           // GS dt
    float lane_dt_half;      // GS dt / 2
    float lane_qns;          // GS nscale
};

// host side: fill the parameters of species s (pm2d_particles.cu)
PartParams make_part_params(pm2d_ctx *c, int s);
// the deferred particles of a stage kernel, on the global grids (pm2d_particles.cu); shape = PM2D_CIC/TSC/SINE
void launch_stage_overflow(const PartParams &P, int shape, int stage, int qmask, cudaStream_t st);

namespace {



__device__ __forceinline__ int fold_x(int i, int nx)
{
    if (i < 0) i = -i;
    if (i > nx) i = 2 * nx - i;
    if (i < 0) i = 0;          // rows more than nx beyond a wall (tiny boxes) are never touched by a particle
    return i;
}

// O1 / Eq. 13: cumulative shape G(t), t already clamped to [0, DD].  SINE: G = 1/2 - 1/2 cos(pi t/DD)
// (Q1) through MUFU.COS (abs. error < 5e-7); TSC, CIC: textbook (ref. [42]).
template <int SHAPE>
__device__ __forceinline__ float shape_G(float t, float k_rad)
{
    if (SHAPE == PM2D_SINE) return fmaf(-0.5f, __cosf(t * k_rad), 0.5f);
    if (SHAPE == PM2D_TSC) {
        float u = fminf(t, 2.f - t), h = 0.5f * u * u;
        return t < 1.f ? h : 1.f - h;
    }
    return t;   // CIC, DD = 1
}

// weights of the three nodes c-1, c, c+1 around the nearest node c for a particle at offset d in
// [-1/2, 1/2) from it: control-volume faces c-1/2, c+1/2 at t0 = DD/2 - 1/2 - d, t1 = t0 + 1 from the
// particle's left edge;  W[c-1] = G(t0), W[c] = G(t1) - G(t0), W[c+1] = 1 - G(t1).
template <int SHAPE>
__device__ __forceinline__ void weights3(float d, const PartParams &P, float W[3])
{
    float t0 = fminf(fmaxf(P.half_dd - 0.5f - d, 0.f), P.dd);
    float t1 = fminf(fmaxf(P.half_dd + 0.5f - d, 0.f), P.dd);
    float g0 = shape_G<SHAPE>(t0, P.k_rad), g1 = shape_G<SHAPE>(t1, P.k_rad);
    W[0] = g0;
    W[1] = g1 - g0;
    W[2] = 1.f - g1;
}

// weights of the four nodes c-1 .. c+2 around cell c for a particle whose offset from the cell's origin is
// rel * 2^-24 in [-1/2, 3/2): faces c-1/2, c+1/2, c+3/2 at t_k = DD/2 + k - 1/2 - f; the outer faces c-3/2
// and c+5/2 lie outside the cloud (G = 0, 1) because DD <= 2.  Returns W4_SCALE<SHAPE> * weight: for the sine
// cloud the factor 1/2 of G = (1 - cos)/2 is left to the caller (folded into dt and the deposit scale).
template <int SHAPE>
struct W4Scale { static constexpr float value = SHAPE == PM2D_SINE ? 2.f : 1.f; };

template <int SHAPE>
__device__ __forceinline__ void weights4(int rel, const PartParams &P, float W[4])
{
    if (SHAPE == PM2D_SINE) {
        // everything in radians of the cosine argument: b = (DD/2 - 1/2 - f) pi/DD, clamped to [0, pi]
        const float b = fmaf((float)rel, P.w4_slope, P.w4_off);
        const float t0 = fminf(fmaxf(b, 0.f), 3.14159265358979f);
        const float t1 = fminf(fmaxf(b + P.k_rad, 0.f), 3.14159265358979f);
        const float t2 = fminf(fmaxf(b + 2.f * P.k_rad, 0.f), 3.14159265358979f);
        const float c0 = __cosf(t0), c1 = __cosf(t1), c2 = __cosf(t2);
        W[0] = 1.f - c0;
        W[1] = c0 - c1;
        W[2] = c1 - c2;
        W[3] = 1.f + c2;
    } else {
        const float b = P.half_dd - 0.5f - (float)rel * (1.0f / 16777216.0f);
        float t0 = fminf(fmaxf(b, 0.f), P.dd);
        float t1 = fminf(fmaxf(b + 1.f, 0.f), P.dd);
        float t2 = fminf(fmaxf(b + 2.f, 0.f), P.dd);
        float g0 = shape_G<SHAPE>(t0, P.k_rad), g1 = shape_G<SHAPE>(t1, P.k_rad), g2 = shape_G<SHAPE>(t2, P.k_rad);
        W[0] = g0;
        W[1] = g1 - g0;
        W[2] = g2 - g1;
        W[3] = 1.f - g2;
    }
}

// nearest node (tile-relative) and offset from it, exact
__device__ __forceinline__ void decode(uint32_t f, int &c, float &d)
{
    int cell = (int)(f >> POS_FRAC_BITS) - POS_BIAS;
    float fr = (float)(f & POS_FRAC_MASK) * (1.0f / 16777216.0f);
    int up = fr >= 0.5f;
    c = cell + up;
    d = fr - (float)up;
}

__device__ __forceinline__ uint32_t advance(uint32_t f, float h, float usum)
{
    // displacement in cells = h * (u' + u), rounded once to 2^-24 cell
    float disp = __fmul_rn(__fmul_rn(h, usum), 16777216.0f);
    return f + (uint32_t)__float2int_rn(disp);
}

// x walls reflect (Q9); y is periodic and needs nothing until the rebin
__device__ __forceinline__ void reflect_x(uint32_t &xf, float &ux, int gx0, int nx)
{
    const int64_t org = ((int64_t)gx0 - POS_BIAS) << POS_FRAC_BITS;
    int64_t gx = org + (int64_t)xf;
    const int64_t wall = (int64_t)nx << POS_FRAC_BITS;
    if (gx < 0) {
        gx = -gx;
        ux = -ux;
    } else if (gx >= wall) {
        gx = 2 * wall - gx;
        if (gx >= wall) gx = wall - 1;
        ux = -ux;
    } else
        return;
    xf = (uint32_t)(gx - org);
}

__device__ __forceinline__ bool in_window(int cx, int cy)
{
    return cx - 1 >= -HALO && cx + 1 <= TILE + HALO && cy - 1 >= -HALO && cy + 1 <= TILE + HALO;
}

// ---- deposit of one particle outside the register patch: 3 x 3 nodes around the nearest node, into the
// shared window when it covers them, else straight to the global grids (particle far from its tile)
template <int SHAPE, int QMASK, bool WINDOWED, int PITCH = WPITCH>
__device__ __forceinline__ void deposit_direct(const PartParams &P, int gx0, int gy0, uint32_t xf, uint32_t yf, float ux, float uy,
                                               float w, int32_t *dep)
{
    int cx, cy;
    float dx_, dy_, Wx[3], Wy[3];
    decode(xf, cx, dx_);
    decode(yf, cy, dy_);
    weights3<SHAPE>(dx_, P, Wx);
    weights3<SHAPE>(dy_, P, Wy);
    const float qn = w * P.nscale, qx = w * ux * P.pscale, qy = w * uy * P.pscale;
    if (WINDOWED && in_window(cx, cy)) {
        const int base = (cx - 1 + HALO) * PITCH + (cy - 1 + HALO);
#pragma unroll
        for (int a = 0; a < 3; a++)
#pragma unroll
            for (int b = 0; b < 3; b++) {
                float ww = Wx[a] * Wy[b];
                if (ww == 0.f) continue;
                int e = base + a * PITCH + b;
                if (QMASK & 1) atomicAdd(&dep[e], __float2int_rn(ww * qn));
                if (QMASK & 2) {
                    atomicAdd(&dep[WIN * PITCH + e], __float2int_rn(ww * qx));
                    atomicAdd(&dep[2 * WIN * PITCH + e], __float2int_rn(ww * qy));
                }
            }
        return;
    }
#pragma unroll 1
    for (int a = 0; a < 3; a++) {
        int gi = fold_x(gx0 + cx - 1 + a, P.nx);
        int fac = (gi == 0 || gi == P.nx) ? 2 : 1;
#pragma unroll 1
        for (int b = 0; b < 3; b++) {
            int gj = (gy0 + cy - 1 + b) & (P.ny - 1);
            float ww = Wx[a] * Wy[b];
            size_t k = (size_t)gi * P.ny + gj;
            if (QMASK & 1) atomicAdd(&P.nfix[k], fac * __float2int_rn(ww * qn));
            if (QMASK & 2) {
                atomicAdd(&P.pxfix[k], fac * __float2int_rn(ww * qx));
                atomicAdd(&P.pyfix[k], fac * __float2int_rn(ww * qy));
            }
        }
    }
}

// Eq. 15 on 3 x 3 nodes around the nearest node: from the shared force window, or (overflow path)
// from forces evaluated on the global grids
template <int SHAPE, bool WINDOWED, int PITCH = WPITCH>
__device__ __forceinline__ float2 gather_direct(const PartParams &P, int gx0, int gy0, uint32_t xf, uint32_t yf, const float2 *Fs, bool &ok)
{
    int cx, cy;
    float dx_, dy_, Wx[3], Wy[3];
    decode(xf, cx, dx_);
    decode(yf, cy, dy_);
    ok = !WINDOWED || in_window(cx, cy);
    if (!ok) return make_float2(0.f, 0.f);
    weights3<SHAPE>(dx_, P, Wx);
    weights3<SHAPE>(dy_, P, Wy);
    float fx = 0.f, fy = 0.f;
    if (WINDOWED) {
        const int base = (cx - 1 + HALO) * PITCH + (cy - 1 + HALO);
#pragma unroll
        for (int a = 0; a < 3; a++) {
            float rx = 0.f, ry = 0.f;
#pragma unroll
            for (int b = 0; b < 3; b++) {
                float2 f = Fs[base + a * PITCH + b];
                rx += Wy[b] * f.x;
                ry += Wy[b] * f.y;
            }
            fx += Wx[a] * rx;
            fy += Wx[a] * ry;
        }
    } else {
#pragma unroll 1
        for (int a = 0; a < 3; a++) {
            int gi = fold_x(gx0 + cx - 1 + a, P.nx);
#pragma unroll 1
            for (int b = 0; b < 3; b++) {
                int gj = (gy0 + cy - 1 + b) & (P.ny - 1);
                float2 f = P.F[(size_t)gi * P.ny + gj];
                float ww = Wx[a] * Wy[b];
                fx += ww * f.x;
                fy += ww * f.y;
            }
        }
    }
    return make_float2(fx, fy);
}

// One particle through one stage outside the register patch.  STAGE 0: predictor (Eq. 17); STAGE 1:
// corrector (Eq. 19) + particle boundaries; STAGE 2: deposit only.  QMASK bit 0: density, bit 1: momentum.
// dep_only: the strip thread already gathered and pushed this particle (u^ resp. the new state is stored);
// only its deposit is left.  WINDOWED: shared windows; returns false (nothing done) when the gather
// footprint lies outside the window -- the caller defers the particle to k_stage_overflow (WINDOWED =
// false, global grids).  The force window is a copy of the global force grid and the deposits are integer
// sums, so all three routes (register patch, window, global) give identical grids.
template <int SHAPE, int STAGE, int QMASK, bool WINDOWED, int PITCH = WPITCH, int FPITCH = PITCH>
__device__ __forceinline__ bool process_direct(const PartParams &P, int64_t p, bool dep_only, int gx0, int gy0, const float2 *Fs,
                                               int32_t *dep)
{
    PV me = P.pv[p];
    uint32_t xf = me.x, yf = me.y;
    float ux = me.ux, uy = me.uy;
    if (STAGE == 0) {
        float uhx, uhy;
        if (dep_only) {
            const float2 uh = P.uh[p];
            uhx = uh.x;
            uhy = uh.y;
        } else {
            bool ok;
            float2 f = gather_direct<SHAPE, WINDOWED, FPITCH>(P, gx0, gy0, xf, yf, Fs, ok);
            if (!ok) return false;
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
        uint32_t xh = advance(xf, P.hx, __fadd_rn(uh.x, ux));                      // x^ of Eq. 17 again
        uint32_t yh = advance(yf, P.hy, __fadd_rn(uh.y, uy));
        bool ok;
        float2 f = gather_direct<SHAPE, WINDOWED, FPITCH>(P, gx0, gy0, xh, yh, Fs, ok);
        if (!ok) return false;
        float unx = __fmaf_rn(0.5f * P.dt, f.x, 0.5f * __fadd_rn(uh.x, ux));       // Eq. 19
        float uny = __fmaf_rn(0.5f * P.dt, f.y, 0.5f * __fadd_rn(uh.y, uy));
        xf = advance(xf, P.hx, __fadd_rn(unx, ux));
        yf = advance(yf, P.hy, __fadd_rn(uny, uy));
        reflect_x(xf, unx, gx0, P.nx);
        me.x = xf; me.y = yf; me.ux = unx; me.uy = uny;
        P.pv[p] = me;
        ux = unx;
        uy = uny;
    }
    deposit_direct<SHAPE, QMASK, WINDOWED, PITCH>(P, gx0, gy0, xf, yf, ux, uy, P.w[p], dep);
    return true;
}

constexpr int64_t OVF_DEP = (int64_t)1 << 62;          // overflow-list flag: deposit only

__device__ __forceinline__ void push_overflow(const PartParams &P, int64_t p, int tile, bool dep_only)
{
    int slot = atomicAdd(P.ovf_count, 1);
    if (slot < P.ovf_cap) {
        P.ovf_p[slot] = p | (dep_only ? OVF_DEP : 0);
        P.ovf_tile[slot] = tile;
    } else
        P.flags[2] = 1;
}

}  // namespace
