// pm2d_poisson.cu -- the electrostatic module without cuFFT / cuSPARSE:
//   k_fft_rho   : rho = sum_s sign_s n_s (exact integer difference of the fixed-point deposits),
//                 radix-2 FFT along y in shared memory, one CTA per grid row          (Eq. 9-10)
//   k_tridiag   : one thread per k_y: Thomas ("chasing") sweep along x in double with the
//                 right-hand-side independent c' coefficients precomputed at init      (Eq. 11)
//                 the back-substitution emits the spectrum of E already averaged to the nodes
//   k_ifft_pair : one complex inverse FFT per row returns E_x (real part) and E_y (imaginary part)
//
// Why E leaves the solver in spectral form.  The paper differences phi in real space
// and the force needs E on the nodes (Q3).  Both operations are shifts and sums along y and x, so
// by the DFT shift theorem they are exact multipliers of each mode (theta = 2 pi l / ny):
//   E_x,node(i) = -cos^2(theta/2) (phi^_{i+1} - phi^_{i-1}) / (2 dx)
//   E_y,node(i) = -i sin(theta) (phi^_{i-1} + 2 phi^_i + phi^_{i+1}) / (4 dy)
// (walls: one-sided forms below).  Applying them to the double-precision phi^ avoids differencing
// a float32 phi whose long-wavelength part is ~1e4 times larger than the plasma-wave part.
#include "pm2d_internal.h"

namespace {

constexpr int FFT_THREADS = 256;

struct RhoSrc {
    const int32_t *n[PM2D_MAX_SPECIES];
    int sign[PM2D_MAX_SPECIES];
    int count;
    float inv_nscale;
};

// in-place radix-2 decimation-in-time FFT of buf[0..n-1] (already in bit-reversed order);
// tw[k] = exp(-2 pi i k / n); inverse uses the conjugate twiddles.
template <bool INVERSE>
__device__ void fft_shared(float2 *buf, const float2 *__restrict__ tw, int n, int log2n)
{
    for (int s = 1; s <= log2n; s++) {
        const int h = 1 << (s - 1);
        const int tstride = n >> s;
        __syncthreads();
        for (int b = threadIdx.x; b < n / 2; b += blockDim.x) {
            int k = b & (h - 1);
            int p = ((b >> (s - 1)) << s) + k, q = p + h;
            float2 w = tw[k * tstride];
            if (INVERSE) w.y = -w.y;
            float2 u = buf[p], v = buf[q];
            float2 t = make_float2(v.x * w.x - v.y * w.y, v.x * w.y + v.y * w.x);
            buf[p] = make_float2(u.x + t.x, u.y + t.y);
            buf[q] = make_float2(u.x - t.x, u.y - t.y);
        }
    }
    __syncthreads();
}

__global__ void __launch_bounds__(FFT_THREADS) k_fft_rho(RhoSrc S, const float2 *__restrict__ tw, float2 *__restrict__ rho_hat,
                                                         int ny, int log2n, int LP)
{
    extern __shared__ float2 buf[];
    const int i = blockIdx.x + 1;                     // rows 1 .. nx-1 (phi = 0 on the walls, Q5)
    const size_t row = (size_t)i * ny;
    for (int j = threadIdx.x; j < ny; j += blockDim.x) {
        int v = 0;
        for (int s = 0; s < S.count; s++) v += S.sign[s] * S.n[s][row + j];
        buf[__brev((unsigned)j) >> (32 - log2n)] = make_float2((float)v * S.inv_nscale, 0.f);
    }
    fft_shared<false>(buf, tw, ny, log2n);
    for (int l = threadIdx.x; l <= ny / 2; l += blockDim.x) rho_hat[(size_t)i * LP + l] = buf[l];
}

__global__ void k_cp_init(double *cp, int nx, int ny, int LP, double dx, double Ly)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l > ny / 2) return;
    const double PI = 3.14159265358979323846;
    const double ky = 2.0 * PI * (double)l / Ly;
    const double b = -2.0 - ky * ky * dx * dx;
    double c = 0.0;
    for (int i = 1; i < nx; i++) {
        c = 1.0 / (b - c);
        cp[(size_t)i * LP + l] = c;
    }
}

struct TriParams {
    const float2 *rho_hat;
    float2 *phi_hat;      // may alias rho_hat (row i is read before it is written); NULL: not wanted
    const double *cp;
    double2 *d;
    float2 *ehx, *ehy;
    int nx, ny, LP;
    double dx2, inv_dx, inv_dy, inv_ny;
};

__global__ void __launch_bounds__(32) k_tridiag(const TriParams T)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l > T.ny / 2) return;
    const int nx = T.nx, LP = T.LP;
    constexpr int B = 8;
    // forward elimination: d_i = (dx^2 rho^_i - d_{i-1}) c'_i
    double dr = 0.0, di = 0.0;
    for (int i0 = 1; i0 < nx; i0 += B) {
        float2 r[B];
        double c[B];
#pragma unroll
        for (int k = 0; k < B; k++) {
            int i = min(i0 + k, nx - 1);
            r[k] = T.rho_hat[(size_t)i * LP + l];
            c[k] = T.cp[(size_t)i * LP + l];
        }
#pragma unroll
        for (int k = 0; k < B; k++) {
            int i = i0 + k;
            if (i < nx) {
                dr = (T.dx2 * (double)r[k].x - dr) * c[k];
                di = (T.dx2 * (double)r[k].y - di) * c[k];
                T.d[(size_t)i * LP + l] = make_double2(dr, di);
            }
        }
    }
    // back substitution phi_i = d_i - c'_i phi_{i+1}, emitting the nodal-E spectrum of row i+1 as soon
    // as phi_i is known
    const double PI = 3.14159265358979323846;
    const double theta = 2.0 * PI * (double)l / (double)T.ny;
    const double c2 = cos(0.5 * theta) * cos(0.5 * theta), sn = sin(theta);
    const double kx = -c2 * 0.5 * T.inv_dx * T.inv_ny;       // times (phi_{i+1} - phi_{i-1})
    const double kyf = -sn * 0.25 * T.inv_dy * T.inv_ny;     // times i (phi_{i-1} + 2 phi_i + phi_{i+1})
    double p2r = 0.0, p2i = 0.0;     // phi_{i+2}
    double p1r = 0.0, p1i = 0.0;     // phi_{i+1}   (starts as phi_nx = 0)
    for (int i1 = nx - 1; i1 >= 1; i1 -= B) {
        double2 dd[B];
        double c[B];
#pragma unroll
        for (int k = 0; k < B; k++) {
            int i = max(i1 - k, 1);
            dd[k] = T.d[(size_t)i * LP + l];
            c[k] = T.cp[(size_t)i * LP + l];
        }
#pragma unroll
        for (int k = 0; k < B; k++) {
            int i = i1 - k;
            if (i >= 1) {
                double pr = dd[k].x - c[k] * p1r, pi = dd[k].y - c[k] * p1i;     // phi_i
                // row i+1 now has both neighbours
                int e = i + 1;
                double ex_r, ex_i, ey_r, ey_i;
                if (e == nx) {      // right wall: mean of the two cells at nx - 1/2
                    ex_r = 2.0 * kx * (p1r - pr); ex_i = 2.0 * kx * (p1i - pi);
                    ey_r = -2.0 * kyf * (pi + p1i); ey_i = 2.0 * kyf * (pr + p1r);
                } else {
                    ex_r = kx * (p2r - pr); ex_i = kx * (p2i - pi);
                    double sr = pr + 2.0 * p1r + p2r, si = pi + 2.0 * p1i + p2i;
                    ey_r = -kyf * si; ey_i = kyf * sr;                            // i * (sr + i si)
                }
                T.ehx[(size_t)e * LP + l] = make_float2((float)ex_r, (float)ex_i);
                T.ehy[(size_t)e * LP + l] = make_float2((float)ey_r, (float)ey_i);
                if (T.phi_hat) T.phi_hat[(size_t)i * LP + l] = make_float2((float)(pr * T.inv_ny), (float)(pi * T.inv_ny));
                p2r = p1r; p2i = p1i;
                p1r = pr; p1i = pi;
            }
        }
    }
    // rows 1 and 0: phi_0 = 0; p1 = phi_1, p2 = phi_2 (or phi_nx = 0 when nx == 2)
    {
        double ex_r = kx * (p2r - 0.0), ex_i = kx * (p2i - 0.0);
        double sr = 0.0 + 2.0 * p1r + p2r, si = 0.0 + 2.0 * p1i + p2i;
        T.ehx[(size_t)1 * LP + l] = make_float2((float)ex_r, (float)ex_i);
        T.ehy[(size_t)1 * LP + l] = make_float2((float)(-kyf * si), (float)(kyf * sr));
        // left wall: mean of the two cells at 1/2
        T.ehx[l] = make_float2((float)(2.0 * kx * p1r), (float)(2.0 * kx * p1i));
        T.ehy[l] = make_float2((float)(-2.0 * kyf * p1i), (float)(2.0 * kyf * p1r));
        if (T.phi_hat) {
            T.phi_hat[l] = make_float2(0.f, 0.f);
            T.phi_hat[(size_t)nx * LP + l] = make_float2(0.f, 0.f);
        }
    }
}

// MODE 0: Z = ehx + i ehy -> Enode (float2);  MODE 1: Z = phi^ -> phi (float, real part)
template <int MODE>
__global__ void __launch_bounds__(FFT_THREADS) k_ifft(const float2 *__restrict__ hx, const float2 *__restrict__ hy,
                                                      const float2 *__restrict__ tw, float2 *__restrict__ Enode,
                                                      float *__restrict__ phi, int ny, int log2n, int LP)
{
    extern __shared__ float2 buf[];
    const int i = blockIdx.x;
    for (int l = threadIdx.x; l <= ny / 2; l += blockDim.x) {
        float2 a = hx[(size_t)i * LP + l];
        float2 b = MODE == 0 ? hy[(size_t)i * LP + l] : make_float2(0.f, 0.f);
        // Z_l = a + i b ; Z_{ny-l} = conj(a) + i conj(b)
        buf[__brev((unsigned)l) >> (32 - log2n)] = make_float2(a.x - b.y, a.y + b.x);
        if (l > 0 && l < ny / 2) buf[__brev((unsigned)(ny - l)) >> (32 - log2n)] = make_float2(a.x + b.y, -a.y + b.x);
    }
    fft_shared<true>(buf, tw, ny, log2n);
    for (int j = threadIdx.x; j < ny; j += blockDim.x) {
        if (MODE == 0) Enode[(size_t)i * ny + j] = buf[j];
        else phi[(size_t)i * ny + j] = buf[j].x;
    }
}

__global__ void k_twiddle_init(float2 *tw, int ny)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= ny / 2) return;
    double s, c;
    sincospi(-2.0 * (double)k / (double)ny, &s, &c);
    tw[k] = make_float2((float)c, (float)s);
}

}  // namespace

static int ilog2(int n)
{
    int l = 0;
    while ((1 << l) < n) l++;
    return l;
}

int launch_poisson_init(pm2d_ctx *c)
{
    const int ny = c->g.ny;
    k_twiddle_init<<<(ny / 2 + 127) / 128, 128, 0, c->stream>>>(c->twiddle, ny);
    k_cp_init<<<(ny / 2 + 1 + 31) / 32, 32, 0, c->stream>>>(c->cp, c->g.nx, ny, c->LP, c->g.dx, ny * c->g.dy);
    count_launch(c, 2);
    PM2D_CUDA_CHECK(cudaGetLastError());
    if (ny * sizeof(float2) > 48 * 1024) {
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_fft_rho, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(ny * sizeof(float2))));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_ifft<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(ny * sizeof(float2))));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_ifft<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(ny * sizeof(float2))));
    }
    return PM2D_OK;
}

// rho from the current density grids -> nodal E (and phi if wanted, for diagnostics)
int launch_poisson(pm2d_ctx *c, bool want_phi)
{
    const int nx = c->g.nx, ny = c->g.ny, log2n = ilog2(ny);
    const size_t smem = ny * sizeof(float2);
    RhoSrc S;
    S.count = 0;
    S.inv_nscale = c->inv_nscale;
    for (int s = 0; s < c->nsp; s++)
        if (c->sp[s].cfg.sign != 0) {
            S.n[S.count] = c->sp[s].nfix;
            S.sign[S.count] = c->sp[s].cfg.sign;
            S.count++;
        }
    if (nx >= 2) k_fft_rho<<<nx - 1, FFT_THREADS, smem, c->stream>>>(S, c->twiddle, c->rho_hat, ny, log2n, c->LP);
    TriParams T;
    T.rho_hat = c->rho_hat; T.phi_hat = want_phi ? c->rho_hat : nullptr; T.cp = c->cp; T.d = c->dtmp;
    T.ehx = c->ehx; T.ehy = c->ehy; T.nx = nx; T.ny = ny; T.LP = c->LP;
    T.dx2 = c->g.dx * c->g.dx; T.inv_dx = 1.0 / c->g.dx; T.inv_dy = 1.0 / c->g.dy; T.inv_ny = 1.0 / ny;
    k_tridiag<<<(ny / 2 + 1 + 31) / 32, 32, 0, c->stream>>>(T);
    k_ifft<0><<<nx + 1, FFT_THREADS, smem, c->stream>>>(c->ehx, c->ehy, c->twiddle, c->Enode, nullptr, ny, log2n, c->LP);
    count_launch(c, 3);
    if (want_phi) {
        k_ifft<1><<<nx + 1, FFT_THREADS, smem, c->stream>>>(c->rho_hat, nullptr, c->twiddle, nullptr, c->phi, ny, log2n, c->LP);
        count_launch(c);
    }
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}
