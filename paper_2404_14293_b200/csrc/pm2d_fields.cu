// pm2d_fields.cu -- mesh kernels of libpm2d.so (sm_100a):
//   * wave equation, Eq. 6: x-marching register stencil, one thread per column j
//   * x-boundary absorbing condition Eq. 8 with laser injection (Eq. 4)
//   * optional absorbing y walls and corners (Q23)
//   * nodal fluid force, Eq. 16 / 18
//   * small conversions between the fixed-point deposit grids and float
#include "pm2d_internal.h"

namespace {

constexpr float FOUR_PI2 = 39.47841760435743f;

struct NeSrc {
    const int32_t *n[PM2D_MAX_SPECIES];   // density grids of the negative species
    int count;
    float inv_nscale;
};

// Eq. 6.  CTA = 128 threads x 4 columns x FROWS rows; each thread marches along x keeping a[i-1], a[i], a[i+1] of its
// four columns in registers (128-bit loads and stores); the two outer y neighbours come from the same cache lines
// through L1.  ny is a power of two >= 8, so a thread's four columns never wrap.
constexpr int FCOLS = 128, FVEC = 4, FROWS = 32, FBATCH = 2;

__device__ __forceinline__ float4 ne_at4(const NeSrc &S, size_t k)
{
    int4 v = make_int4(0, 0, 0, 0);
    for (int s = 0; s < S.count; s++) {
        const int4 t = *reinterpret_cast<const int4 *>(S.n[s] + k);
        v.x += t.x; v.y += t.y; v.z += t.z; v.w += t.w;
    }
    return make_float4((float)v.x * S.inv_nscale, (float)v.y * S.inv_nscale, (float)v.z * S.inv_nscale, (float)v.w * S.inv_nscale);
}

__device__ __forceinline__ float wave_node(float hi, float mid, float lo, float l, float r, float old, float den, float cx, float cy,
                                           float dt2)
{
    const float lap = cx * (hi - 2.f * mid + lo) + cy * (r - 2.f * mid + l);
    const float src = FOUR_PI2 * den * mid;
    return 2.f * mid - old + dt2 * (lap - src);
}

__global__ void __launch_bounds__(FCOLS) k_wave(const float *__restrict__ a, const float *__restrict__ am, float *__restrict__ ap,
                                                NeSrc ne, int nx, int ny, float cx, float cy, float dt2)
{
    const int j = (blockIdx.x * FCOLS + threadIdx.x) * FVEC;
    if (j >= ny) return;
    const int i0 = 1 + blockIdx.y * FROWS, i1 = min(nx, i0 + FROWS);   // interior rows i0 .. i1-1
    if (i0 >= i1) return;
    const int jm = (j - 1) & (ny - 1), jp = (j + FVEC) & (ny - 1);
    float4 lo = *reinterpret_cast<const float4 *>(a + (size_t)(i0 - 1) * ny + j);
    float4 mid = *reinterpret_cast<const float4 *>(a + (size_t)i0 * ny + j);
    for (int ib = i0; ib < i1; ib += FBATCH) {
        // the loads of FBATCH rows are issued together: the march itself is a chain of dependent rows
        float4 hi[FBATCH], old[FBATCH], den[FBATCH];
        float l[FBATCH], r[FBATCH];
#pragma unroll
        for (int u = 0; u < FBATCH; u++) {
            const size_t row = (size_t)min(ib + u, i1 - 1) * ny;
            hi[u] = *reinterpret_cast<const float4 *>(a + row + ny + j);
            l[u] = a[row + jm];
            r[u] = a[row + jp];
            old[u] = *reinterpret_cast<const float4 *>(am + row + j);
            den[u] = ne_at4(ne, row + j);
        }
#pragma unroll
        for (int u = 0; u < FBATCH; u++) {
            if (ib + u < i1) {
                const size_t row = (size_t)(ib + u) * ny;
                float4 o;
                o.x = wave_node(hi[u].x, mid.x, lo.x, l[u], mid.y, old[u].x, den[u].x, cx, cy, dt2);
                o.y = wave_node(hi[u].y, mid.y, lo.y, mid.x, mid.z, old[u].y, den[u].y, cx, cy, dt2);
                o.z = wave_node(hi[u].z, mid.z, lo.z, mid.y, mid.w, old[u].z, den[u].z, cx, cy, dt2);
                o.w = wave_node(hi[u].w, mid.w, lo.w, mid.z, r[u], old[u].w, den[u].w, cx, cy, dt2);
                *reinterpret_cast<float4 *>(ap + row + j) = o;
                lo = mid;
                mid = hi[u];
            }
        }
    }
}

struct BcParams {
    float g[PM2D_MAX_LASERS][6];   // carrier*ramp at (x=0: t-dt, t, t+dt), (x=dx: t-dt, t, t+dt)
    float y0[PM2D_MAX_LASERS], inv_w0[PM2D_MAX_LASERS];   // inv_w0 = 0: plane wave
    int comp[PM2D_MAX_LASERS];
    int nlaser;
    float alpha, beta, gam, dy;
};

__device__ __forceinline__ float beam_env(const BcParams &B, int l, float y)
{
    float r = (y - B.y0[l]) * B.inv_w0[l];
    return __expf(-r * r);
}

// Oblique incidence (Eq. 5; Q22): envelope and carrier no longer separate, so the incident wave
// is evaluated per boundary node and time level, in double (the phase 2 pi omega (t - xb) grows without bound).
struct ObLaser {
    double a0, omega2, y0, inv_w0, inv_2rise, sa, ca, lead;   // omega2 = 2 omega; inv_2rise = 1 / (2 t_rise) or 0
    int comp, oblique;
};
struct ObParams {
    ObLaser L[PM2D_MAX_LASERS];
    double t_now, dt, dx, Ly, inv_Ly;
};

// Eq. 4 in the beam's coordinates; (x, y) are box coordinates, y' = y - y0 at the nearest periodic image
__device__ double oblique_inc(const ObLaser &L, double x, double y, double t, double Ly, double inv_Ly)
{
    double xb = x, yb = y - L.y0, lead = 0.0;
    if (L.oblique) {
        double d = y - L.y0;
        d -= Ly * floor(d * inv_Ly + 0.5);
        xb = x * L.ca - d * L.sa;                 // Eq. 5
        yb = x * L.sa + d * L.ca;
        lead = L.lead;
    }
    const double phase = t - xb, tau = phase - lead;
    if (tau <= 0.0) return 0.0;
    double v = L.a0 * cospi(L.omega2 * phase);
    if (L.inv_w0 > 0.0) {
        const double r = yb * L.inv_w0;
        v *= exp(-r * r);
    }
    if (L.inv_2rise > 0.0 && tau * L.inv_2rise < 0.5) {
        const double sr = sinpi(tau * L.inv_2rise);
        v *= sr * sr;
    }
    return v;
}

// Eq. 8 solved for the boundary node, both x walls, one thread per j.  Left wall: applied to the
// scattered field s = a - a_inc and a_inc added back.  OBLIQUE: some beam has alpha != 0.
template <bool OBLIQUE>
__global__ void k_boundary(const float *__restrict__ a, const float *__restrict__ am, float *__restrict__ ap, BcParams B,
                           ObParams O, int comp, int nx, int ny, float *__restrict__ probe)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= ny) return;
    const int jm = (j - 1) & (ny - 1), jp = (j + 1) & (ny - 1);
    // incident wave at the 3 columns j-1, j, j+1: inc[col][x][t]
    float inc[3][6];
    const int cols[3] = {jm, j, jp};
    if (OBLIQUE) {
        for (int q = 0; q < 3; q++)
            for (int k = 0; k < 6; k++) {
                double v = 0.0;
                for (int l = 0; l < B.nlaser; l++)
                    if (B.comp[l] == comp)
                        v += oblique_inc(O.L[l], (k / 3) * O.dx, cols[q] * (double)B.dy, O.t_now + (k % 3 - 1) * O.dt, O.Ly, O.inv_Ly);
                inc[q][k] = (float)v;
            }
    } else {
        for (int q = 0; q < 3; q++)
            for (int k = 0; k < 6; k++) inc[q][k] = 0.f;
        for (int l = 0; l < B.nlaser; l++) {
            if (B.comp[l] != comp) continue;
            for (int q = 0; q < 3; q++) {
                float e = beam_env(B, l, cols[q] * B.dy);
                for (int k = 0; k < 6; k++) inc[q][k] += e * B.g[l][k];
            }
        }
    }
    const float ab = 1.f / (B.alpha + B.beta);
    {   // left wall: rows 0, 1
        float s0 = a[j] - inc[1][1], s0m = am[j] - inc[1][0];
        float s1 = a[ny + j] - inc[1][4], s1m = am[ny + j] - inc[1][3], s1p = ap[ny + j] - inc[1][5];
        float D0 = (a[jp] - inc[2][1]) - 2.f * s0 + (a[jm] - inc[0][1]);
        float D1 = (a[ny + jp] - inc[2][4]) - 2.f * s1 + (a[ny + jm] - inc[0][4]);
        float s0p = (B.alpha * (s1p - s1m + s0m) - B.beta * (s1p + s1m + s0m - 2.f * s0 - 2.f * s1) + B.gam * (D0 + D1)) * ab;
        ap[j] = s0p + inc[1][2];
        if (probe) probe[j] = s0p;                 // boundary record, left wall: the scattered field (pm2d_get_probe)
    }
    {   // right wall: rows nx, nx-1, no incident wave
        const size_t r0 = (size_t)nx * ny, r1 = (size_t)(nx - 1) * ny;
        float E0 = a[r0 + jp] - 2.f * a[r0 + j] + a[r0 + jm];
        float E1 = a[r1 + jp] - 2.f * a[r1 + j] + a[r1 + jm];
        const float v = (B.alpha * (ap[r1 + j] - am[r1 + j] + am[r0 + j]) -
                         B.beta * (ap[r1 + j] + am[r1 + j] + am[r0 + j] - 2.f * a[r0 + j] - 2.f * a[r1 + j]) + B.gam * (E0 + E1)) * ab;
        ap[r0 + j] = v;
        if (probe) probe[ny + j] = v;              // right wall: a itself
    }
}

// Absorbing y walls (pm2d_grid.bc_y = PM2D_BC_Y_ABSORB; "on all of four boundaries", Q23): Eq. 8 with
// the roles of x and y exchanged on the wall columns j = 0 and j = ny-1, rows 1..nx-1, no incident wave; then the four
// corners by the first-order outgoing condition along the diagonal.  Runs after k_wave and k_boundary and overwrites
// what their periodic stencils left in the two wall columns.  One thread per (row, wall); the wall columns are ny
// floats apart, so every access is its own sector: 2 (nx-1) nodes x 14 sectors, microseconds at any BJ size.
struct BcYParams {
    float alpha_y, beta, gam_x, kap;   // 1/(2 dt dy), 1/(2 dt^2), 1/(4 dx^2), (dt - hd)/(dt + hd), hd = sqrt(dx^2 + dy^2)
};
__global__ void k_boundary_y(const float *__restrict__ a, const float *__restrict__ am, float *__restrict__ ap, BcYParams B, int nx,
                             int ny, float *__restrict__ probe)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;   // 0..nx
    const int side = blockIdx.y;
    if (i > nx) return;
    const int j0 = side ? ny - 1 : 0, j1 = side ? ny - 2 : 1;
    if (i == 0 || i == nx) {
        // corner c, diagonal neighbour d: a_c^{n+1} = a_d^n + kappa (a_d^{n+1} - a_c^n)
        const size_t kc = (size_t)i * ny + j0, kd = (size_t)(i == 0 ? 1 : nx - 1) * ny + j1;
        const float v = a[kd] + B.kap * (ap[kd] - a[kc]);
        if (probe) {   // the corner's boundary record follows its new value (left: the incident part stays split off)
            if (i == 0) probe[j0] += v - ap[kc];
            else probe[ny + j0] = v;
        }
        ap[kc] = v;
        return;
    }
    const size_t k0 = (size_t)i * ny + j0, k1 = (size_t)i * ny + j1;
    const float D0 = a[k0 + ny] - 2.f * a[k0] + a[k0 - ny];
    const float D1 = a[k1 + ny] - 2.f * a[k1] + a[k1 - ny];
    ap[k0] = (B.alpha_y * (ap[k1] - am[k1] + am[k0]) - B.beta * (ap[k1] + am[k1] + am[k0] - 2.f * a[k0] - 2.f * a[k1]) +
              B.gam_x * (D0 + D1)) / (B.alpha_y + B.beta);
}

// Eq. 16 / 18 on the nodes.  E arrives already averaged to the nodes (Q3; pm2d_poisson.cu).
struct ForceParams {
    const float2 *Enode;
    const float *a;          // [ncomp][nn], the level the stage needs (n or n+1)
    const int32_t *nfix;     // this species' density
    float2 *F;
    int nx, ny, ncomp;
    float qE;                // -sign * 4 pi^2 / mass
    float pond;              // 1 for electrons, 0 otherwise
    float cv2;               // C * v_th^2
    float inv_2dx, inv_2dy;
};

__device__ __forceinline__ float a2_at(const ForceParams &P, size_t k, size_t nn)
{
    float s = 0.f;
    for (int c = 0; c < P.ncomp; c++) {
        float v = P.a[c * nn + k];
        s += v * v;
    }
    return s;
}

// CTA = 128 columns x GROWS rows; each thread marches along x keeping |a|^2 and n of rows i-1, i, i+1 in
// registers (central x-differences, one-sided on the wall rows); the y neighbours come through L1.
constexpr int GCOLS = 128, GROWS = 32;
__global__ void __launch_bounds__(GCOLS) k_force(const ForceParams P)
{
    const int j = blockIdx.x * GCOLS + threadIdx.x;
    if (j >= P.ny) return;
    const int i0 = blockIdx.y * GROWS, i1 = min(P.nx + 1, i0 + GROWS);
    const size_t nn = (size_t)(P.nx + 1) * P.ny;
    const int jm = (j - 1) & (P.ny - 1), jp = (j + 1) & (P.ny - 1);
    const bool pond = P.pond != 0.f, press = P.cv2 != 0.f;
    const size_t rlo = (size_t)(i0 > 0 ? i0 - 1 : 0) * P.ny, r0 = (size_t)i0 * P.ny;
    float a_lo = pond ? a2_at(P, rlo + j, nn) : 0.f, a_mid = pond ? a2_at(P, r0 + j, nn) : 0.f;
    int n_lo = P.nfix[rlo + j], n_mid = P.nfix[r0 + j];
    for (int i = i0; i < i1; i++) {
        const size_t row = (size_t)i * P.ny, rhi = (size_t)(i < P.nx ? i + 1 : P.nx) * P.ny;
        const float a_hi = pond ? a2_at(P, rhi + j, nn) : 0.f;
        const int n_hi = P.nfix[rhi + j];
        const float sx = (i == 0 || i == P.nx) ? 2.f * P.inv_2dx : P.inv_2dx;     // one-sided at the walls
        const float2 E = P.Enode[row + j];
        float fx = P.qE * E.x, fy = P.qE * E.y;
        if (pond) {
            fx -= 0.5f * sx * (a_hi - a_lo);
            fy -= 0.5f * P.inv_2dy * (a2_at(P, row + jp, nn) - a2_at(P, row + jm, nn));
        }
        if (n_mid > 0 && press) {
            const float inv_n = 1.f / (float)n_mid;
            fx -= P.cv2 * sx * (float)(n_hi - n_lo) * inv_n;
            fy -= P.cv2 * P.inv_2dy * (float)(P.nfix[row + jp] - P.nfix[row + jm]) * inv_n;
        }
        P.F[row + j] = make_float2(fx, fy);
        a_lo = a_mid; a_mid = a_hi;
        n_lo = n_mid; n_mid = n_hi;
    }
}

__global__ void k_fix_to_float(const int32_t *src, float scale, float *dst, size_t n)
{
    size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) dst[k] = (float)src[k] * scale;
}
__global__ void k_float_to_fix(const float *src, float scale, int32_t *dst, size_t n)
{
    size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) dst[k] = __float2int_rn(src[k] * scale);
}
__global__ void k_sum_fix(NeSrc S, int32_t *dst, size_t n)
{
    size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    int v = 0;
    for (int s = 0; s < S.count; s++) v += S.n[s][k];
    dst[k] = v;
}

}  // namespace

// carrier * ramp of one laser at retarded time tau (double on the host: the phase 2 pi omega tau
// grows without bound and must not be rounded to float)
static double laser_g(const pm2d_laser &L, double tau)
{
    const double PI = 3.14159265358979323846;
    if (tau <= 0.0) return 0.0;
    double ramp = 1.0;
    if (L.t_rise > 0.0 && tau < L.t_rise) {
        double s = sin(0.5 * PI * tau / L.t_rise);
        ramp = s * s;
    }
    return L.a0 * ramp * cos(2.0 * PI * L.omega * tau);
}

// one step of Eq. 6 + Eq. 8: a[0] <- a[1], a[2]; sub = index of the wave step inside the particle step (Q21)
int launch_field_step(pm2d_ctx *c, int sub)
{
    const int nx = c->g.nx, ny = c->g.ny;
    const double dx = c->g.dx, dy = c->g.dy, dt = c->g.dt, t_now = (double)(c->step * c->nsub + sub) * dt;
    NeSrc ne;
    ne.count = 0;
    ne.inv_nscale = c->inv_nscale;
    for (int s = 0; s < c->nsp; s++)
        if (c->sp[s].cfg.sign < 0) ne.n[ne.count++] = c->sp[s].nfix;
    BcParams B;
    B.nlaser = c->nlaser;
    for (int l = 0; l < c->nlaser; l++) {
        const pm2d_laser &L = c->laser[l];
        for (int xk = 0; xk < 2; xk++)
            for (int tk = 0; tk < 3; tk++) B.g[l][xk * 3 + tk] = (float)laser_g(L, t_now + (tk - 1) * dt - xk * dx);
        B.y0[l] = (float)L.y0;
        B.inv_w0[l] = L.w0 > 0.0 ? (float)(1.0 / L.w0) : 0.f;
        B.comp[l] = L.comp;
    }
    B.alpha = (float)(1.0 / (2.0 * dt * dx));
    B.beta = (float)(1.0 / (2.0 * dt * dt));
    B.gam = (float)(1.0 / (4.0 * dy * dy));
    B.dy = (float)dy;
    ObParams O;
    bool oblique = false;
    for (int l = 0; l < c->nlaser; l++) {
        const pm2d_laser &L = c->laser[l];
        ObLaser &Q = O.L[l];
        Q.a0 = L.a0; Q.omega2 = 2.0 * L.omega; Q.y0 = L.y0;
        Q.inv_w0 = L.w0 > 0.0 ? 1.0 / L.w0 : 0.0;
        Q.inv_2rise = L.t_rise > 0.0 ? 0.5 / L.t_rise : 0.0;
        Q.sa = sin(L.alpha); Q.ca = cos(L.alpha);
        Q.lead = 0.5 * ny * dy * fabs(Q.sa);
        Q.comp = L.comp;
        Q.oblique = L.alpha != 0.0;
        oblique = oblique || Q.oblique;
    }
    O.t_now = t_now; O.dt = dt; O.dx = dx; O.Ly = ny * dy; O.inv_Ly = 1.0 / (ny * dy);
    dim3 grid((ny + FCOLS * FVEC - 1) / (FCOLS * FVEC), (nx - 1 + FROWS - 1) / FROWS);
    for (int comp = 0; comp < c->g.ncomp; comp++) {
        const size_t off = (size_t)comp * c->nn;
        k_wave<<<grid, FCOLS, 0, c->stream>>>(c->a[1] + off, c->a[2] + off, c->a[0] + off, ne, nx, ny, (float)(1.0 / (dx * dx)),
                                              (float)(1.0 / (dy * dy)), (float)(dt * dt));
        // boundary record of particle step q = step + 1, taken from its last wave step: slot (q - 1) % probe_steps
        float *probe = (c->probe && sub == c->nsub - 1)
                           ? c->probe + ((size_t)(c->step % c->g.probe_steps) * c->g.ncomp + comp) * 2 * ny : nullptr;
        if (oblique) k_boundary<true><<<(ny + 127) / 128, 128, 0, c->stream>>>(c->a[1] + off, c->a[2] + off, c->a[0] + off, B, O, comp, nx, ny, probe);
        else k_boundary<false><<<(ny + 127) / 128, 128, 0, c->stream>>>(c->a[1] + off, c->a[2] + off, c->a[0] + off, B, O, comp, nx, ny, probe);
        count_launch(c, 2);
        if (c->g.bc_y == PM2D_BC_Y_ABSORB) {
            BcYParams Y;
            const double hd = sqrt(dx * dx + dy * dy);
            Y.alpha_y = (float)(1.0 / (2.0 * dt * dy));
            Y.beta = B.beta;
            Y.gam_x = (float)(1.0 / (4.0 * dx * dx));
            Y.kap = (float)((dt - hd) / (dt + hd));
            k_boundary_y<<<dim3((nx + 1 + 127) / 128, 2), 128, 0, c->stream>>>(c->a[1] + off, c->a[2] + off, c->a[0] + off, Y, nx, ny, probe);
            count_launch(c, 1);
        }
    }
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}

int launch_force(pm2d_ctx *c, int s, const float *a_level)
{
    SpeciesDev &S = c->sp[s];
    ForceParams P;
    const double PI = 3.14159265358979323846;
    P.Enode = c->Enode; P.a = a_level; P.nfix = S.nfix; P.F = S.F;
    P.nx = c->g.nx; P.ny = c->g.ny; P.ncomp = c->g.ncomp;
    P.qE = (float)(-(double)S.cfg.sign * 4.0 * PI * PI / S.cfg.mass);
    P.pond = S.cfg.sign < 0 ? 1.f : 0.f;
    P.cv2 = (float)(S.cfg.pressure_coeff * S.vth2);
    P.inv_2dx = (float)(1.0 / (2.0 * c->g.dx));
    P.inv_2dy = (float)(1.0 / (2.0 * c->g.dy));
    dim3 grid((c->g.ny + GCOLS - 1) / GCOLS, (c->g.nx + 1 + GROWS - 1) / GROWS);
    k_force<<<grid, GCOLS, 0, c->stream>>>(P);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}

int launch_fix_background(pm2d_ctx *c, int s)
{
    NeSrc src;
    src.count = 0;
    src.inv_nscale = 1.f;
    for (int t = 0; t < c->nsp; t++)
        if (t != s && c->sp[t].cfg.mobile && c->sp[t].cfg.sign == -c->sp[s].cfg.sign) src.n[src.count++] = c->sp[t].nfix;
    k_sum_fix<<<(unsigned)((c->nn + 255) / 256), 256, 0, c->stream>>>(src, c->sp[s].nfix, (size_t)c->nn);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}

int launch_fix_to_float(pm2d_ctx *c, const int32_t *src, float scale, float *dst)
{
    k_fix_to_float<<<(unsigned)((c->nn + 255) / 256), 256, 0, c->stream>>>(src, scale, dst, (size_t)c->nn);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}

int launch_float_to_fix(pm2d_ctx *c, const float *src, float scale, int32_t *dst)
{
    k_float_to_fix<<<(unsigned)((c->nn + 255) / 256), 256, 0, c->stream>>>(src, scale, dst, (size_t)c->nn);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}
