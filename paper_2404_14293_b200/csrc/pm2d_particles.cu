// pm2d_particles.cu -- particle kernels of libpm2d.so (sm_100a):
//   * fused gather + push + deposit, stage A (Eq. 17) and stage B (Eq. 19)      [P:L191-221]
//   * deposit-only pass (initial item (1) of the flow, lazy momentum grids)       [Eq. 14, P:L187]
//   * counter-based particle loader (Philox-4x32-10)         [P:L154-162]
//   * stable tile rebin (counting sort specialised to neighbour moves)            [DESIGN.md 6.4]
//
// Data layout.  Particles are SoA, stored tile by tile (PM2D_TILE x PM2D_TILE cells); a particle's
// position is a pair of 32-bit fixed-point numbers relative to its tile's origin,
//     xfix = (cell_rel + POS_BIAS) << 24 | frac24,
// so the in-cell offset carries 24 bits whatever the size of the box, the push is an exact integer
// add of a rounded displacement, and the canonical (ix, fx) of include/pm2d.h is read off exactly.
// A CTA owns one chunk (<= CHUNK particles of one tile): it stages the force of the tile + halo in
// shared memory, accumulates the deposit of its particles in a shared int32 fixed-point window
// (native ATOMS.ADD; float atomics in shared memory are CAS loops on sm_100a) and flushes the
// window once with global integer reductions.  Integer accumulation makes the deposited grids
// independent of the order of the atomics (bit-reproducible) and n_i - n_e exact.
#include "pm2d_internal.h"

namespace {

struct PartParams {
    // particles
    uint32_t *x, *y;
    float *ux, *uy, *uhx, *uhy;
    const float *w;
    const int32_t *chunk_tile;
    const int64_t *chunk_beg;
    const int64_t *tile_off;
    const int32_t *nchunks;
    // grids
    const float2 *F;          // materialised force grid (slow path / diagnostics); may be NULL
    const float2 *Enode;      // nodal E of the last Poisson solve
    const float *a;           // [ncomp][nn], level n (stage A) or n+1 (stage B)
    int ncomp;
    float qE, pond, cv2;      // -sign 4 pi^2 / m ; 1 for electrons ; C v_th^2
    float inv_2dx, inv_2dy;
    const int32_t *nfix_in;   // density the force is built from (n^n or n^); the deposit goes to nfix
    int32_t *nfix, *pxfix, *pyfix;
    int32_t *flags;
    int64_t *ovf_p;           // overflow list: particles whose gather footprint left the tile window
    int32_t *ovf_tile, *ovf_count;
    int ovf_cap;
    int nx, ny, nty;
    float dt, hx, hy;        // hx = dt / (2 dx): cells per unit (u' + u)
    float nscale, pscale;
    float half_dd;           // DD / 2
    float shape_k;           // 0.5 / DD  (sine: G(s) = sinpi(s * shape_k)^2)
};

__device__ __forceinline__ int fold_x(int i, int nx)
{
    if (i < 0) i = -i;
    if (i > nx) i = 2 * nx - i;
    if (i < 0) i = 0;          // rows more than nx beyond a wall (tiny boxes) are never touched by a particle
    return i;
}

// O1 / Eq. 13: weights of the three nodes c-1, c, c+1 around the nearest node c for a particle at
// offset d in [-1/2, 1/2) from it.  With s measured from the particle's left edge, the control-
// volume faces c-1/2 and c+1/2 sit at s0 = DD/2 - 1/2 - d and s1 = s0 + 1, and
//   W[c-1] = G(s0), W[c] = G(s1) - G(s0), W[c+1] = 1 - G(s1),  G clamped to [0, DD].
template <int SHAPE>
__device__ __forceinline__ void weights3(float d, float half_dd, float shape_k, float W[3])
{
    if (SHAPE == PM2D_TSC) {
        float a = 0.5f - d, b = 0.5f + d;
        W[0] = 0.5f * a * a;
        W[2] = 0.5f * b * b;
        W[1] = 0.75f - d * d;
    } else if (SHAPE == PM2D_CIC) {
        W[0] = fmaxf(-d, 0.f);
        W[2] = fmaxf(d, 0.f);
        W[1] = 1.f - fabsf(d);
    } else {
        float dd = 2.f * half_dd;
        float s0 = fminf(fmaxf(half_dd - 0.5f - d, 0.f), dd);
        float s1 = fminf(fmaxf(half_dd + 0.5f - d, 0.f), dd);
        float g0 = sinpif(s0 * shape_k), g1 = sinpif(s1 * shape_k);
        g0 *= g0;
        g1 *= g1;
        W[0] = g0;
        W[1] = g1 - g0;
        W[2] = 1.f - g1;
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

template <int QMASK>
__device__ __forceinline__ void deposit_window(int32_t *dep, int cx, int cy, const float Wx[3], const float Wy[3],
                                               float qn, float qx, float qy, bool skip_zero)
{
    const int base = (cx - 1 + HALO) * WPITCH + (cy - 1 + HALO);
#pragma unroll
    for (int a = 0; a < 3; a++) {
#pragma unroll
        for (int b = 0; b < 3; b++) {
            float ww = Wx[a] * Wy[b];
            if (skip_zero && ww == 0.f) continue;
            int e = base + a * WPITCH + b;
            if (QMASK & 1) atomicAdd(&dep[e], __float2int_rn(ww * qn));
            if (QMASK & 2) {
                atomicAdd(&dep[WIN * WPITCH + e], __float2int_rn(ww * qx));
                atomicAdd(&dep[2 * WIN * WPITCH + e], __float2int_rn(ww * qy));
            }
        }
    }
}

// slow path: footprint outside the shared window (a particle that drifted more than HALO - 1/2
// cells from its tile since the last rebin) -> straight to the global grids
template <int QMASK>
__device__ __noinline__ void deposit_global(const PartParams &P, int gx0, int gy0, int cx, int cy, const float Wx[3],
                                            const float Wy[3], float qn, float qx, float qy)
{
    for (int a = 0; a < 3; a++) {
        int gi = fold_x(gx0 + cx - 1 + a, P.nx);
        int fac = (gi == 0 || gi == P.nx) ? 2 : 1;
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

// Eq. 16 at one global node (slow path only)
__device__ __forceinline__ float2 force_at_node(const PartParams &P, int gi, int gj)
{
    const size_t nn = (size_t)(P.nx + 1) * P.ny;
    const int il = gi > 0 ? gi - 1 : 0, ih = gi < P.nx ? gi + 1 : P.nx;
    const float sx = (il == gi || ih == gi) ? 2.f * P.inv_2dx : P.inv_2dx;
    const int jm = (gj - 1) & (P.ny - 1), jp = (gj + 1) & (P.ny - 1);
    const size_t k = (size_t)gi * P.ny + gj, kl = (size_t)il * P.ny + gj, kh = (size_t)ih * P.ny + gj;
    const size_t kd = (size_t)gi * P.ny + jm, ku = (size_t)gi * P.ny + jp;
    float2 E = P.Enode[k];
    float fx = P.qE * E.x, fy = P.qE * E.y;
    if (P.pond != 0.f) {
        float ah = 0.f, al = 0.f, au = 0.f, ad = 0.f;
        for (int c = 0; c < P.ncomp; c++) {
            float v;
            v = P.a[c * nn + kh]; ah += v * v;
            v = P.a[c * nn + kl]; al += v * v;
            v = P.a[c * nn + ku]; au += v * v;
            v = P.a[c * nn + kd]; ad += v * v;
        }
        fx -= 0.5f * sx * (ah - al);
        fy -= 0.5f * P.inv_2dy * (au - ad);
    }
    const int n0 = P.nfix_in[k];
    if (n0 > 0 && P.cv2 != 0.f) {
        const float inv_n = 1.f / (float)n0;
        fx -= P.cv2 * sx * (float)(P.nfix_in[kh] - P.nfix_in[kl]) * inv_n;
        fy -= P.cv2 * P.inv_2dy * (float)(P.nfix_in[ku] - P.nfix_in[kd]) * inv_n;
    }
    return make_float2(fx, fy);
}

__device__ __noinline__ float2 gather_global(const PartParams &P, int gx0, int gy0, int cx, int cy, const float Wx[3],
                                             const float Wy[3])
{
    float fx = 0.f, fy = 0.f;
#pragma unroll 1
    for (int a = 0; a < 3; a++) {
        int gi = fold_x(gx0 + cx - 1 + a, P.nx);
#pragma unroll 1
        for (int b = 0; b < 3; b++) {
            int gj = (gy0 + cy - 1 + b) & (P.ny - 1);
            float2 f = force_at_node(P, gi, gj);
            float ww = Wx[a] * Wy[b];
            fx += ww * f.x;
            fy += ww * f.y;
        }
    }
    return make_float2(fx, fy);
}

__device__ __forceinline__ bool in_window(int cx, int cy)
{
    return cx - 1 >= -HALO && cx + 1 <= TILE + HALO && cy - 1 >= -HALO && cy + 1 <= TILE + HALO;
}

__device__ __forceinline__ float2 gather_window(const float2 *Fs, int cx, int cy, const float Wx[3], const float Wy[3])
{
    const int base = (cx - 1 + HALO) * WPITCH + (cy - 1 + HALO);
    float fx = 0.f, fy = 0.f;
#pragma unroll
    for (int a = 0; a < 3; a++) {
        float rx = 0.f, ry = 0.f;
#pragma unroll
        for (int b = 0; b < 3; b++) {
            float2 f = Fs[base + a * WPITCH + b];
            rx += Wy[b] * f.x;
            ry += Wy[b] * f.y;
        }
        fx += Wx[a] * rx;
        fy += Wx[a] * ry;
    }
    return make_float2(fx, fy);
}


// Eq. 16 / 18 evaluated for the nodes of the tile window, straight into shared memory:
//   F = qE E_node - (1/2) grad(sum_c a_c^2) [electrons] - C v_th^2 grad(n)/n
// central differences, one-sided on the wall rows, pressure term 0 where n = 0 (Q10).  Window rows
// beyond a wall hold F of the mirror node (Q9: the gather folds indices), whose x-difference runs
// the other way in window coordinates.  a2s / ns: scratch of (WIN+2)^2 values (window + 1 ring).
constexpr int WF = WIN + 2;
__device__ __forceinline__ void build_force_window(const PartParams &P, int gx0, int gy0, float *a2s, int32_t *ns, float2 *Fs)
{
    const size_t nn = (size_t)(P.nx + 1) * P.ny;
#pragma unroll 2
    for (int e = threadIdx.x; e < WF * WF; e += PTHREADS) {
        int r = e / WF, cidx = e - r * WF;
        int gi = fold_x(gx0 + r - HALO - 1, P.nx);
        int gj = (gy0 + cidx - HALO - 1) & (P.ny - 1);
        size_t k = (size_t)gi * P.ny + gj;
        float s2 = 0.f;
        if (P.pond != 0.f)
            for (int c = 0; c < P.ncomp; c++) {
                float v = P.a[c * nn + k];
                s2 += v * v;
            }
        a2s[e] = s2;
        ns[e] = P.nfix_in[k];
    }
    __syncthreads();
#pragma unroll 1
    for (int e = threadIdx.x; e < WIN * WIN; e += PTHREADS) {
        int r = e / WIN, cidx = e - r * WIN;
        int raw = gx0 + r - HALO;
        int gi = fold_x(raw, P.nx);
        int gj = (gy0 + cidx - HALO) & (P.ny - 1);
        const int c0 = (r + 1) * WF + (cidx + 1);
        // x-difference in window coordinates -> difference at the (possibly mirrored) node
        int lo = c0 - WF, hi = c0 + WF;
        float sx = P.inv_2dx;
        if (raw < 0 || raw > P.nx) sx = -sx;
        if (gi == 0) { lo = c0; hi = (raw == 0) ? c0 + WF : c0 - WF; sx = 2.f * P.inv_2dx; }
        else if (gi == P.nx) { hi = c0; lo = (raw == P.nx) ? c0 - WF : c0 + WF; sx = 2.f * P.inv_2dx; }
        float2 E = P.Enode[(size_t)gi * P.ny + gj];
        float fx = P.qE * E.x, fy = P.qE * E.y;
        if (P.pond != 0.f) {
            fx -= 0.5f * sx * (a2s[hi] - a2s[lo]);
            fy -= 0.5f * P.inv_2dy * (a2s[c0 + 1] - a2s[c0 - 1]);
        }
        const int n0 = ns[c0];
        if (n0 > 0 && P.cv2 != 0.f) {
            const float inv_n = 1.f / (float)n0;
            fx -= P.cv2 * sx * (float)(ns[hi] - ns[lo]) * inv_n;
            fy -= P.cv2 * P.inv_2dy * (float)(ns[c0 + 1] - ns[c0 - 1]) * inv_n;
        }
        Fs[r * WPITCH + cidx] = make_float2(fx, fy);
    }
    __syncthreads();
}

// One particle through one stage.  STAGE 0: predictor (Eq. 17); STAGE 1: corrector (Eq. 19) + particle
// boundaries; STAGE 2: deposit only.  QMASK bit 0: density, bit 1: momentum.
// WINDOWED: gather from / deposit into the CTA's shared windows; returns false (nothing done) when the
// gather footprint lies outside the window -- the caller defers the particle to k_stage_overflow, which
// runs the same code with WINDOWED = false straight on the global grids.
template <int SHAPE, int STAGE, int QMASK, bool WINDOWED>
__device__ __forceinline__ bool process_particle(const PartParams &P, int64_t p, int gx0, int gy0, const float2 *Fs, int32_t *dep)
{
    uint32_t xf = P.x[p], yf = P.y[p];
    float ux = P.ux[p], uy = P.uy[p];
    float Wx[3], Wy[3];
    int cx, cy;
    float dx_, dy_;
    if (STAGE == 0) {
        decode(xf, cx, dx_);
        decode(yf, cy, dy_);
        if (WINDOWED && !in_window(cx, cy)) return false;
        weights3<SHAPE>(dx_, P.half_dd, P.shape_k, Wx);
        weights3<SHAPE>(dy_, P.half_dd, P.shape_k, Wy);
        float2 f = WINDOWED ? gather_window(Fs, cx, cy, Wx, Wy) : gather_global(P, gx0, gy0, cx, cy, Wx, Wy);
        float uhx = __fmaf_rn(P.dt, f.x, ux), uhy = __fmaf_rn(P.dt, f.y, uy);     // Eq. 17
        P.uhx[p] = uhx;
        P.uhy[p] = uhy;
        xf = advance(xf, P.hx, __fadd_rn(uhx, ux));
        yf = advance(yf, P.hy, __fadd_rn(uhy, uy));
        ux = uhx;
        uy = uhy;
    } else if (STAGE == 1) {
        const float uhx = P.uhx[p], uhy = P.uhy[p];
        uint32_t xh = advance(xf, P.hx, __fadd_rn(uhx, ux));                      // x^ of Eq. 17 again
        uint32_t yh = advance(yf, P.hy, __fadd_rn(uhy, uy));
        decode(xh, cx, dx_);
        decode(yh, cy, dy_);
        if (WINDOWED && !in_window(cx, cy)) return false;
        weights3<SHAPE>(dx_, P.half_dd, P.shape_k, Wx);
        weights3<SHAPE>(dy_, P.half_dd, P.shape_k, Wy);
        float2 f = WINDOWED ? gather_window(Fs, cx, cy, Wx, Wy) : gather_global(P, gx0, gy0, cx, cy, Wx, Wy);
        float unx = __fmaf_rn(0.5f * P.dt, f.x, 0.5f * __fadd_rn(uhx, ux));       // Eq. 19
        float uny = __fmaf_rn(0.5f * P.dt, f.y, 0.5f * __fadd_rn(uhy, uy));
        xf = advance(xf, P.hx, __fadd_rn(unx, ux));
        yf = advance(yf, P.hy, __fadd_rn(uny, uy));
        // x walls reflect (Q9); y is periodic and needs nothing until the rebin
        int64_t gx = (((int64_t)gx0 - POS_BIAS) << POS_FRAC_BITS) + (int64_t)xf;
        const int64_t wall = (int64_t)P.nx << POS_FRAC_BITS;
        if (gx < 0) {
            gx = -gx;
            unx = -unx;
        } else if (gx >= wall) {
            gx = 2 * wall - gx;
            if (gx >= wall) gx = wall - 1;
            unx = -unx;
        }
        xf = (uint32_t)(gx - (((int64_t)gx0 - POS_BIAS) << POS_FRAC_BITS));
        P.x[p] = xf;
        P.y[p] = yf;
        P.ux[p] = unx;
        P.uy[p] = uny;
        ux = unx;
        uy = uny;
    }
    decode(xf, cx, dx_);
    decode(yf, cy, dy_);
    weights3<SHAPE>(dx_, P.half_dd, P.shape_k, Wx);
    weights3<SHAPE>(dy_, P.half_dd, P.shape_k, Wy);
    const float w = P.w[p];
    const float qn = w * P.nscale, qx = w * ux * P.pscale, qy = w * uy * P.pscale;
    if (WINDOWED && in_window(cx, cy))
        deposit_window<QMASK>(dep, cx, cy, Wx, Wy, qn, qx, qy, SHAPE == PM2D_CIC);
    else
        deposit_global<QMASK>(P, gx0, gy0, cx, cy, Wx, Wy, qn, qx, qy);
    return true;
}

template <int SHAPE, int STAGE, int QMASK>
__global__ void __launch_bounds__(PTHREADS, 4) k_stage(const PartParams P)
{
    constexpr int NQ = (QMASK & 2) ? 3 : 1;
    // dep doubles as the scratch of build_force_window (2 (WIN+2)^2 words) before it is zeroed
    constexpr int DEPW = (STAGE < 2 && NQ * WIN * WPITCH < 2 * WF * WF) ? 2 * WF * WF : NQ * WIN * WPITCH;
    __shared__ int32_t dep[DEPW];
    __shared__ float2 Fs[(STAGE < 2) ? WIN * WPITCH : 1];
    const int chunk = blockIdx.x;
    if (chunk >= *P.nchunks) return;
    const int tile = P.chunk_tile[chunk];
    const int64_t beg = P.chunk_beg[chunk];
    int64_t end = beg + CHUNK;
    {
        int64_t te = P.tile_off[tile + 1];
        if (te < end) end = te;
    }
    const int gx0 = (tile / P.nty) * TILE, gy0 = (tile % P.nty) * TILE;

    if (STAGE < 2) build_force_window(P, gx0, gy0, reinterpret_cast<float *>(dep), dep + WF * WF, Fs);
    for (int e = threadIdx.x; e < NQ * WIN * WPITCH; e += PTHREADS) dep[e] = 0;
    __syncthreads();

    for (int64_t p = beg + threadIdx.x; p < end; p += PTHREADS) {
        if (!process_particle<SHAPE, STAGE, QMASK, true>(P, p, gx0, gy0, Fs, dep)) {
            // drifted more than HALO - 1/2 cells out of its tile since the last rebin: rare; deferred
            int slot = atomicAdd(P.ovf_count, 1);
            if (slot < P.ovf_cap) {
                P.ovf_p[slot] = p;
                P.ovf_tile[slot] = tile;
            } else
                P.flags[2] = 1;
        }
    }
    __syncthreads();

    // flush: one global integer reduction per touched window node; wall columns hold half a
    // control volume and count twice (Q9); rows beyond a wall fold back (mirror particles)
    for (int e = threadIdx.x; e < WIN * WIN; e += PTHREADS) {
        int r = e / WIN, cidx = e - r * WIN;
        int se = r * WPITCH + cidx;
        int gi = fold_x(gx0 + r - HALO, P.nx);
        int gj = (gy0 + cidx - HALO) & (P.ny - 1);
        int fac = (gi == 0 || gi == P.nx) ? 2 : 1;
        size_t k = (size_t)gi * P.ny + gj;
        if (QMASK & 1) {
            int v = dep[se];
            if (v) atomicAdd(&P.nfix[k], fac * v);
        }
        if (QMASK & 2) {
            int vx = dep[WIN * WPITCH + se], vy = dep[2 * WIN * WPITCH + se];
            if (vx) atomicAdd(&P.pxfix[k], fac * vx);
            if (vy) atomicAdd(&P.pyfix[k], fac * vy);
        }
    }
}

// the deferred particles of k_stage: same arithmetic, global grids only
template <int SHAPE, int STAGE, int QMASK>
__global__ void __launch_bounds__(128) k_stage_overflow(const PartParams P)
{
    const int n = min(*P.ovf_count, P.ovf_cap);
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n; k += gridDim.x * blockDim.x) {
        const int tile = P.ovf_tile[k];
        process_particle<SHAPE, STAGE, QMASK, false>(P, P.ovf_p[k], (tile / P.nty) * TILE, (tile % P.nty) * TILE, nullptr, nullptr);
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
    uint32_t *x, *y;
    float *ux, *uy, *w;
    int64_t *id;
    const int32_t *chunk_tile;
    const int64_t *chunk_beg;
    const int64_t *tile_off;
    const int32_t *nchunks;
    int nx, ny, nty;
    int ppc_x, ppc_y, load, species;
    uint32_t seed_lo, seed_hi;
    double vth;
    int prof_kind, taper_cells;
    double p0, p1, p2;
};

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
            n = n * (s * s);
        }
    }
    return n;
}

// one CTA per chunk; slot s of a tile with wx*wy cells holds particle k = s / cells of cell s % cells
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
    const int wx = min(TILE, L.nx - gx0), wy = min(TILE, L.ny - gy0);
    const int cells = wx * wy, ppc = L.ppc_x * L.ppc_y;
    for (int64_t p = beg + threadIdx.x; p < end; p += PTHREADS) {
        int s = (int)(p - t0);
        int k = s / cells, lc = s - k * cells;
        int li = lc / wy, lj = lc - li * wy;
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
        L.x[p] = ((uint32_t)(li + POS_BIAS) << POS_FRAC_BITS) | fx24;
        L.y[p] = ((uint32_t)(lj + POS_BIAS) << POS_FRAC_BITS) | fy24;
        L.ux[p] = ux;
        L.uy[p] = uy;
        L.w[p] = (float)(profile_density(L, gx0 + li) / (double)ppc);
        if (L.id) L.id[p] = pid;
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

__global__ void k_uniform_tile_counts(int32_t *cnt, int ntx, int nty, int nx, int ny, int ppc)
{
    int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntx * nty) return;
    int gx0 = (t / nty) * TILE, gy0 = (t % nty) * TILE;
    cnt[t] = ppc * min(TILE, nx - gx0) * min(TILE, ny - gy0);
}

// ---- rebin ---------------------------------------------------------------------------------------
struct RebinParams {
    const uint32_t *x, *y;
    const float *ux, *uy, *w;
    const int64_t *id;
    uint32_t *x2, *y2;
    float *ux2, *uy2, *w2;
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
    int32_t *keys_out;
    int64_t *perm_out;
    int nx, ny, ntx, nty;
};

// destination of a particle: tile displacement (dti, dtj) in {-1,0,1}^2 and the canonical slot
// (dti+1)*3 + c, where c folds y-displacements that reach the same tile when nty < 3
__device__ __forceinline__ int rebin_slot(const RebinParams &R, int gx0, int gy0, uint32_t xf, uint32_t yf, int &dti,
                                          int &dtj, bool &bad)
{
    const int tw = min(TILE, R.nx - gx0), th = min(TILE, R.ny - gy0);
    int cx = (int)(xf >> POS_FRAC_BITS) - POS_BIAS, cy = (int)(yf >> POS_FRAC_BITS) - POS_BIAS;
    dti = cx < 0 ? -1 : (cx >= tw ? 1 : 0);
    dtj = cy < 0 ? -1 : (cy >= th ? 1 : 0);
    int nxr = cx - dti * TILE, nyr = cy - dtj * th;      // tile-relative cell after the move
    int ti = gx0 / TILE + dti;
    bad = ti < 0 || ti >= R.ntx || nxr < 0 || nxr >= min(TILE, R.nx - ti * TILE) || nyr < 0 || nyr >= th;
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
        int slot = rebin_slot(R, gx0, gy0, R.x[p], R.y[p], dti, dtj, bad);
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
// chunk, handing out offsets -> the new order is the stable counting sort of the old array by key
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
        uint32_t xf = 0, yf = 0;
        bool bad = false;
        if (live) {
            xf = R.x[p];
            yf = R.y[p];
            slot = rebin_slot(R, gx0, gy0, xf, yf, dti, dtj, bad);
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
            R.x2[q] = xf - ((uint32_t)(dti * TILE) << POS_FRAC_BITS);
            R.y2[q] = yf - ((uint32_t)(dtj * th) << POS_FRAC_BITS);
            R.ux2[q] = R.ux[p];
            R.uy2[q] = R.uy[p];
            R.w2[q] = R.w[p];
            if (R.id) R.id2[q] = R.id[p];
            if (R.keys_out) R.keys_out[p] = dest;
            if (R.perm_out) R.perm_out[q] = p;
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

// canonical (ix, iy, fx, fy) of the particles of each chunk
__global__ void __launch_bounds__(PTHREADS) k_unpack(const uint32_t *x, const uint32_t *y, const int32_t *chunk_tile,
                                                     const int64_t *chunk_beg, const int64_t *tile_off,
                                                     const int32_t *nchunks, int nty, int ny, int32_t *ix, int32_t *iy,
                                                     float *fx, float *fy)
{
    const int chunk = blockIdx.x;
    if (chunk >= *nchunks) return;
    const int tile = chunk_tile[chunk];
    const int64_t beg = chunk_beg[chunk];
    int64_t end = beg + CHUNK;
    if (tile_off[tile + 1] < end) end = tile_off[tile + 1];
    const int gx0 = (tile / nty) * TILE, gy0 = (tile % nty) * TILE;
    for (int64_t p = beg + threadIdx.x; p < end; p += PTHREADS) {
        uint32_t xf = x[p], yf = y[p];
        ix[p] = gx0 + (int)(xf >> POS_FRAC_BITS) - POS_BIAS;
        iy[p] = (gy0 + (int)(yf >> POS_FRAC_BITS) - POS_BIAS) & (ny - 1);
        fx[p] = (float)(xf & POS_FRAC_MASK) * (1.0f / 16777216.0f);
        fy[p] = (float)(yf & POS_FRAC_MASK) * (1.0f / 16777216.0f);
    }
}

}  // namespace

// =================================================================================================
// host launchers
static PartParams make_part_params(pm2d_ctx *c, int s, const float *a_level)
{
    SpeciesDev &S = c->sp[s];
    PartParams P;
    P.x = S.x; P.y = S.y; P.ux = S.ux; P.uy = S.uy; P.uhx = S.uhx; P.uhy = S.uhy; P.w = S.w;
    P.chunk_tile = S.chunk_tile; P.chunk_beg = S.chunk_beg; P.tile_off = S.tile_off; P.nchunks = S.nchunks_dev;
    P.F = S.F; P.Enode = c->Enode; P.a = a_level; P.ncomp = c->g.ncomp;
    P.qE = (float)(-(double)S.cfg.sign * 4.0 * 3.14159265358979323846 * 3.14159265358979323846 / S.cfg.mass);
    P.pond = S.cfg.sign < 0 ? 1.f : 0.f;
    P.cv2 = (float)(S.cfg.pressure_coeff * S.vth2);
    P.inv_2dx = (float)(1.0 / (2.0 * c->g.dx));
    P.inv_2dy = (float)(1.0 / (2.0 * c->g.dy));
    P.nfix_in = S.nfix; P.nfix = S.nfix; P.pxfix = S.pxfix; P.pyfix = S.pyfix; P.flags = c->flags;
    P.ovf_p = c->ovf_p; P.ovf_tile = c->ovf_tile; P.ovf_count = c->ovf_count; P.ovf_cap = c->ovf_cap;
    P.nx = c->g.nx; P.ny = c->g.ny; P.nty = c->nty;
    P.dt = (float)c->g.dt;
    P.hx = (float)(c->g.dt / (2.0 * c->g.dx));
    P.hy = (float)(c->g.dt / (2.0 * c->g.dy));
    P.nscale = c->nscale; P.pscale = c->pscale;
    P.half_dd = (float)(0.5 * S.cfg.DD);
    P.shape_k = (float)(0.5 / S.cfg.DD);
    return P;
}

template <int SHAPE>
static void launch_stage_shape(const PartParams &P, int stage, int qmask, int grid, cudaStream_t st)
{
#define PM2D_LAUNCH(ST, Q)                                        \
    do {                                                          \
        k_stage<SHAPE, ST, Q><<<grid, PTHREADS, 0, st>>>(P);      \
        if (ST < 2) k_stage_overflow<SHAPE, ST, Q><<<148, 128, 0, st>>>(P); \
    } while (0)
    if (stage == 0) { if (qmask == 3) PM2D_LAUNCH(0, 3); else PM2D_LAUNCH(0, 1); }
    else if (stage == 1) { if (qmask == 3) PM2D_LAUNCH(1, 3); else PM2D_LAUNCH(1, 1); }
    else { if (qmask == 3) PM2D_LAUNCH(2, 3); else if (qmask == 2) PM2D_LAUNCH(2, 2); else PM2D_LAUNCH(2, 1); }
#undef PM2D_LAUNCH
}

static int launch_stage_any(pm2d_ctx *c, int s, int stage, int qmask)
{
    SpeciesDev &S = c->sp[s];
    if (S.np == 0) return PM2D_OK;
    PartParams P = make_part_params(c, s, stage == 0 ? c->a[1] : c->a[0]);
    const int grid = S.max_chunks;
    if (stage < 2) {
        // the force window reads n_s while other CTAs already deposit: ping-pong the density grid
        const size_t bytes = (size_t)c->nn * sizeof(int32_t);
        P.nfix = S.nfix2;
        PM2D_CUDA_CHECK(cudaMemsetAsync(c->ovf_count, 0, sizeof(int32_t), c->stream));
        PM2D_CUDA_CHECK(cudaMemsetAsync(S.nfix2, 0, bytes, c->stream));
        if (qmask & 2) {
            PM2D_CUDA_CHECK(cudaMemsetAsync(S.pxfix, 0, bytes, c->stream));
            PM2D_CUDA_CHECK(cudaMemsetAsync(S.pyfix, 0, bytes, c->stream));
        }
    }
    if (S.cfg.shape == PM2D_CIC) launch_stage_shape<PM2D_CIC>(P, stage, qmask, grid, c->stream);
    else if (S.cfg.shape == PM2D_TSC) launch_stage_shape<PM2D_TSC>(P, stage, qmask, grid, c->stream);
    else launch_stage_shape<PM2D_SINE>(P, stage, qmask, grid, c->stream);
    count_launch(c, stage < 2 ? 2 : 1);
    PM2D_CUDA_CHECK(cudaGetLastError());
    if (stage < 2) std::swap(S.nfix, S.nfix2);
    return PM2D_OK;
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
    k_uniform_tile_counts<<<(c->ntiles + 255) / 256, 256, 0, c->stream>>>(S.tile_cnt, c->ntx, c->nty, c->g.nx, c->g.ny, ppc);
    k_scan_tiles<<<1, SCAN_THREADS, 0, c->stream>>>(S.tile_cnt, c->ntiles, S.tile_off);
    count_launch(c, 2);
    int rc = launch_build_chunks(c, s);
    if (rc) return rc;
    LoadParams L;
    L.x = S.x; L.y = S.y; L.ux = S.ux; L.uy = S.uy; L.w = S.w; L.id = S.id;
    L.chunk_tile = S.chunk_tile; L.chunk_beg = S.chunk_beg; L.tile_off = S.tile_off; L.nchunks = S.nchunks_dev;
    L.nx = c->g.nx; L.ny = c->g.ny; L.nty = c->nty;
    L.ppc_x = S.cfg.ppc_x; L.ppc_y = S.cfg.ppc_y; L.load = S.cfg.load; L.species = s;
    L.seed_lo = (uint32_t)(c->seed & 0xFFFFFFFFu); L.seed_hi = (uint32_t)(c->seed >> 32);
    L.vth = sqrt(S.cfg.T_keV / 511.0 / S.cfg.mass);
    L.prof_kind = c->profile.kind; L.taper_cells = c->profile.taper_cells;
    L.p0 = c->profile.p[0]; L.p1 = c->profile.p[1]; L.p2 = c->profile.p[2];
    k_load<<<S.max_chunks, PTHREADS, 0, c->stream>>>(L);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}

int launch_rebin(pm2d_ctx *c, int s, int32_t *keys_dev, int64_t *perm_dev)
{
    SpeciesDev &S = c->sp[s];
    if (S.np == 0) return PM2D_OK;
    RebinParams R;
    R.x = S.x; R.y = S.y; R.ux = S.ux; R.uy = S.uy; R.w = S.w; R.id = S.id;
    R.x2 = S.x2; R.y2 = S.y2; R.ux2 = S.uhx; R.uy2 = S.uhy; R.w2 = S.w2; R.id2 = S.id2;
    R.chunk_tile = S.chunk_tile; R.chunk_beg = S.chunk_beg; R.tile_off = S.tile_off; R.tile_off2 = S.tile_off2;
    R.nchunks = S.nchunks_dev; R.tile_first_chunk = S.tile_first_chunk;
    R.cnt9 = S.chunk_cnt9; R.rel9 = S.chunk_rel9; R.newcount = S.tile_cnt; R.flags = c->flags;
    R.keys_out = keys_dev; R.perm_out = perm_dev;
    R.nx = c->g.nx; R.ny = c->g.ny; R.ntx = c->ntx; R.nty = c->nty;
    k_rebin_count<<<S.max_chunks, PTHREADS, 0, c->stream>>>(R);
    k_rebin_offsets<<<(c->ntiles + 127) / 128, 128, 0, c->stream>>>(R);
    k_scan_tiles<<<1, SCAN_THREADS, 0, c->stream>>>(S.tile_cnt, c->ntiles, S.tile_off2);
    k_rebin_scatter<<<S.max_chunks, PTHREADS, 0, c->stream>>>(R);
    count_launch(c, 4);
    PM2D_CUDA_CHECK(cudaGetLastError());
    std::swap(S.x, S.x2);
    std::swap(S.y, S.y2);
    std::swap(S.w, S.w2);
    std::swap(S.ux, S.uhx);
    std::swap(S.uy, S.uhy);
    std::swap(S.id, S.id2);
    std::swap(S.tile_off, S.tile_off2);
    return launch_build_chunks(c, s);
}

int launch_unpack_particles(pm2d_ctx *c, int s, int64_t, int64_t, int32_t *ix, int32_t *iy, float *fx, float *fy)
{
    SpeciesDev &S = c->sp[s];
    if (S.np == 0) return PM2D_OK;
    k_unpack<<<S.max_chunks, PTHREADS, 0, c->stream>>>(S.x, S.y, S.chunk_tile, S.chunk_beg, S.tile_off, S.nchunks_dev, c->nty,
                                                        c->g.ny, ix, iy, fx, fy);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}
