// pm2d_poisson.cu -- the electrostatic module without cuFFT / cuSPARSE:
//   k_fft_rho     : rho = sum_s sign_s n_s (exact integer difference of the fixed-point deposits),
//                   Stockham radix-4 FFT along y in shared memory, one CTA per grid row   (Eq. 9-10)
//   k_tri_sums / k_tri_reduced / k_tri_local : the tridiagonal systems of Eq. 11, one per k_y,
//                   solved exactly (to rounding) by the chasing method applied to x-partitions
//                   of TRI_M rows so that (k_y, partition) pairs -- not just k_y -- run in parallel
//   k_ifft        : one complex inverse FFT per row returns E_x (real part) and E_y (imaginary part)
//
// Partitioned chasing method.  Rows kM (k = 1..P-1) are interfaces with unknown values g_k.  Inside a
// partition the solution is  phi = y + g_k V + g_{k+1} W, with y the local solve for zero interface
// values and V, W the two homogeneous solutions (right-hand-side independent, tabulated at init).
// By symmetry of the local matrix, y_1 = -sum_j V_j r_j and y_m = -sum_j W_j r_j, so the reduced
// (P-1)-unknown tridiagonal system for g needs only two weighted column sums per partition
// (k_tri_sums), is solved by one thread per k_y (k_tri_reduced), and then every partition is
// solved ONCE with its true boundary values, entirely in registers, in double (k_tri_local).
//
// Why E leaves the solver in spectral form.  The paper differences phi in real space
// and the force needs E on the nodes (Q3).  Both are shifts and sums along y and x, hence exact
// multipliers of each mode by the DFT shift theorem (theta = 2 pi l / ny):
//   E_x,node(i) = -cos^2(theta/2) (phi^_{i+1} - phi^_{i-1}) / (2 dx)
//   E_y,node(i) = -i sin(theta) (phi^_{i-1} + 2 phi^_i + phi^_{i+1}) / (4 dy)
// (walls: one-sided forms below).  Applying them to the double-precision phi^ avoids differencing
// a float32 phi whose long-wavelength part is ~1e4 times larger than the plasma-wave part.
#include "pm2d_internal.h"

namespace {

constexpr int FFT_THREADS = 256;
constexpr int M = TRI_M;

struct RhoSrc {
    const int32_t *n[PM2D_MAX_SPECIES];
    int sign[PM2D_MAX_SPECIES];
    int count;
    float inv_nscale;
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// Stockham autosort FFT of n points held in shared memory (natural order in, natural order out).
// x, y: ping-pong buffers; tw[t] = exp(-2 pi i t / n), t < n/2.  Returns the buffer with the result.
template <bool INVERSE>
__device__ float2 *fft_stockham(float2 *x, float2 *y, const float2 *__restrict__ tw, int n)
{
    int Ns = 1;
    while (Ns < n) {
        __syncthreads();
        if (n / Ns >= 4) {
            const int q = n >> 2, tstep = n / (4 * Ns);
            for (int j = threadIdx.x; j < q; j += blockDim.x) {
                const int k = j & (Ns - 1);
                float2 v0 = x[j], v1 = x[j + q], v2 = x[j + 2 * q], v3 = x[j + 3 * q];
                if (Ns > 1) {
                    float2 w1 = tw[k * tstep], w2 = tw[2 * k * tstep];
                    if (INVERSE) { w1.y = -w1.y; w2.y = -w2.y; }
                    float2 w3 = cmul(w1, w2);
                    v1 = cmul(v1, w1); v2 = cmul(v2, w2); v3 = cmul(v3, w3);
                }
                float2 a0 = make_float2(v0.x + v2.x, v0.y + v2.y), a1 = make_float2(v0.x - v2.x, v0.y - v2.y);
                float2 a2 = make_float2(v1.x + v3.x, v1.y + v3.y), d = make_float2(v1.x - v3.x, v1.y - v3.y);
                float2 a3 = INVERSE ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x);     // (+/- i) d
                const int j0 = ((j - k) << 2) + k;
                y[j0] = make_float2(a0.x + a2.x, a0.y + a2.y);
                y[j0 + Ns] = make_float2(a1.x + a3.x, a1.y + a3.y);
                y[j0 + 2 * Ns] = make_float2(a0.x - a2.x, a0.y - a2.y);
                y[j0 + 3 * Ns] = make_float2(a1.x - a3.x, a1.y - a3.y);
            }
            Ns <<= 2;
        } else {
            const int h = n >> 1, tstep = n / (2 * Ns);
            for (int j = threadIdx.x; j < h; j += blockDim.x) {
                const int k = j & (Ns - 1);
                float2 w = tw[k * tstep];
                if (INVERSE) w.y = -w.y;
                float2 a = x[j], b = cmul(x[j + h], w);
                const int j0 = ((j - k) << 1) + k;
                y[j0] = make_float2(a.x + b.x, a.y + b.y);
                y[j0 + Ns] = make_float2(a.x - b.x, a.y - b.y);
            }
            Ns <<= 1;
        }
        float2 *t = x; x = y; y = t;
    }
    __syncthreads();
    return x;
}

// ---- register-blocked FFT for n >= 512 ----------------------------------------------------------------
// n/16 threads; every thread holds 16 points.  A pass reads the points of its radix-R butterflies (R = 16,
// last pass 8 / 4 / 2) from shared memory into registers, transforms them there and writes them back in
// Stockham order, so n = 4096 takes three passes and two exchanges through shared memory instead of six.
// The buffer is padded by one element per 16 (index i -> i + i/16) against bank conflicts of the strided
// writes.
__device__ __forceinline__ int pad16(int i) { return i + (i >> 4); }

template <int IDX>
__device__ __forceinline__ constexpr float cos16()
{
    return IDX == 0 ? 1.f : IDX == 1 ? 0.9238795325112867f : IDX == 2 ? 0.7071067811865476f : IDX == 3 ? 0.3826834323650898f
         : IDX == 4 ? 0.f : IDX == 5 ? -0.3826834323650898f : IDX == 6 ? -0.7071067811865476f : -0.9238795325112867f;
}
template <int IDX>
__device__ __forceinline__ constexpr float sin16()
{
    return IDX == 0 ? 0.f : IDX == 1 ? 0.3826834323650898f : IDX == 2 ? 0.7071067811865476f : IDX == 3 ? 0.9238795325112867f
         : IDX == 4 ? 1.f : IDX == 5 ? 0.9238795325112867f : IDX == 6 ? 0.7071067811865476f : 0.3826834323650898f;
}

// o * exp(-/+ 2 pi i IDX / 16)
template <int IDX, bool INV>
__device__ __forceinline__ float2 mul_w16(float2 o)
{
    if (IDX == 0) return o;
    if (IDX == 4) return INV ? make_float2(-o.y, o.x) : make_float2(o.y, -o.x);
    const float c = cos16<IDX>(), sn = INV ? sin16<IDX>() : -sin16<IDX>();
    return make_float2(o.x * c - o.y * sn, o.x * sn + o.y * c);
}

template <int R, bool INV, int K>
struct DftCombine {
    static __device__ __forceinline__ void run(float2 *v, const float2 *e, const float2 *o)
    {
        const float2 t = mul_w16<K * (16 / R), INV>(o[K]);
        v[K] = make_float2(e[K].x + t.x, e[K].y + t.y);
        v[K + R / 2] = make_float2(e[K].x - t.x, e[K].y - t.y);
        if (K + 1 < R / 2) DftCombine<R, INV, (K + 1 < R / 2) ? K + 1 : K>::run(v, e, o);
    }
};

// DFT of R points in registers, natural order in and out (radix-2 decimation in time, fully unrolled)
template <int R, bool INV>
__device__ __forceinline__ void dft_reg(float2 *v)
{
    if (R == 1) return;
    float2 e[R / 2 > 0 ? R / 2 : 1], o[R / 2 > 0 ? R / 2 : 1];
#pragma unroll
    for (int k = 0; k < R / 2; k++) {
        e[k] = v[2 * k];
        o[k] = v[2 * k + 1];
    }
    dft_reg<(R > 1 ? R / 2 : 1), INV>(e);
    dft_reg<(R > 1 ? R / 2 : 1), INV>(o);
    DftCombine<(R > 1 ? R : 2), INV, 0>::run(v, e, o);
}

// plain_out: the pass writes its results unpadded (index i instead of pad16(i)): the last pass of a transform
// whose consumer reads runs of consecutive points (k_ifft's force epilogue)
// NY != 0: the transform length is the compile-time constant NY (n and Ns then fold into immediate offsets)
template <int R, bool INV, int NY = 0>
__device__ __forceinline__ void fft16_pass(float2 *buf, const float2 *__restrict__ tw, int n, int Ns, bool plain_out = false)
{
    if (NY) n = NY;
    const int pad_mask = plain_out ? 0 : -1;
    constexpr int NB = 16 / R;
    const int T = NY ? NY / 16 : (int)blockDim.x, q = n / R;
    float2 v[NB][R];
#pragma unroll
    for (int b = 0; b < NB; b++) {
        const int j = threadIdx.x + b * T;
#pragma unroll
        for (int r = 0; r < R; r++) v[b][r] = buf[pad16(j + r * q)];
    }
    __syncthreads();
#pragma unroll
    for (int b = 0; b < NB; b++) {
        const int j = threadIdx.x + b * T, k = j & (Ns - 1);
        if (Ns > 1) {
            // twiddles w^r, r < R, of w = exp(-/+ 2 pi i k / (Ns R)): one table load (k step < n / R), the powers by
            // a product tree of depth log2 R (w^r = w^p w^(r-p), p the largest power of two <= r) -- R - 1 gathers
            // with up to 32 cache lines per warp each cost far more than R - 2 complex products
            const int step = n / (Ns * R);
            float2 w[R];
            w[1] = tw[k * step];
            if (INV) w[1].y = -w[1].y;
#pragma unroll
            for (int r = 2; r < R; r++) {
                const int p = r >= 8 ? 8 : (r >= 4 ? 4 : 2);
                w[r] = (r == p) ? cmul(w[r / 2], w[r / 2]) : cmul(w[p], w[r - p]);
            }
#pragma unroll
            for (int r = 1; r < R; r++) v[b][r] = cmul(v[b][r], w[r]);
        }
        dft_reg<R, INV>(v[b]);
        const int j0 = (j - k) * R + k;
#pragma unroll
        for (int r = 0; r < R; r++) {
            const int o = j0 + r * Ns;
            buf[o + ((o >> 4) & pad_mask)] = v[b][r];
        }
    }
    __syncthreads();
}

// in place on the padded buffer; blockDim.x == n / 16, n a power of two >= 512; callers synchronise before
template <bool INV, int NY = 0>
__device__ __forceinline__ void fft16_inplace(float2 *buf, const float2 *__restrict__ tw, int n, bool plain_out = false)
{
    if (NY) {       // constant length: every pass is its own, fully folded copy
        constexpr int L16 = NY >= 65536 ? 4 : (NY >= 4096 ? 3 : (NY >= 256 ? 2 : 1));      // radix-16 passes
        constexpr int REM = NY >> (4 * L16);
#pragma unroll
        for (int ps = 0; ps < L16; ps++) fft16_pass<16, INV, NY>(buf, tw, NY, 1 << (4 * ps), plain_out && REM == 1 && ps == L16 - 1);
        if (REM == 8) fft16_pass<8, INV, NY>(buf, tw, NY, 1 << (4 * L16), plain_out);
        else if (REM == 4) fft16_pass<4, INV, NY>(buf, tw, NY, 1 << (4 * L16), plain_out);
        else if (REM == 2) fft16_pass<2, INV, NY>(buf, tw, NY, 1 << (4 * L16), plain_out);
        return;
    }
    int Ns = 1;
    while (n / Ns >= 16) {
        fft16_pass<16, INV>(buf, tw, n, Ns, plain_out && n / Ns == 16);
        Ns <<= 4;
    }
    const int rem = n / Ns;
    if (rem == 8) fft16_pass<8, INV>(buf, tw, n, Ns, plain_out);
    else if (rem == 4) fft16_pass<4, INV>(buf, tw, n, Ns, plain_out);
    else if (rem == 2) fft16_pass<2, INV>(buf, tw, n, Ns, plain_out);
}

// Two real rows per complex transform: z = rho_a + i rho_b, then rho^_a = (Z_l + conj Z_{n-l}) / 2 and
// rho^_b = (Z_l - conj Z_{n-l}) / 2i.  BIG: register-blocked FFT on the padded buffer (ny >= 512).
template <int BIG, int NY = 0>
__global__ void __launch_bounds__(BIG == 2 ? 512 : FFT_THREADS, BIG == 1 ? 4 : 1) k_fft_rho(RhoSrc S, const float2 *__restrict__ tw,
                                                                     float2 *__restrict__ rho_hat, int nx, int ny_, int LP)
{
    extern __shared__ float2 buf[];
    const int ny = NY ? NY : ny_, bdim = NY ? NY / 16 : (int)blockDim.x;
    const int ia = 1 + 2 * blockIdx.x, ib = ia + 1;     // rows 1 .. nx-1 (phi = 0 on the walls, Q5)
    const bool has_b = ib <= nx - 1;
    const size_t rowa = (size_t)ia * ny, rowb = (size_t)ib * ny;
    if (BIG) {
        // bdim == ny / 16: every thread owns 16 columns, taken in two halves of 8 (registers); the loads of a
        // half are issued before their first use
#pragma unroll
        for (int half = 0; half < 2; half++) {
            int va[8], vb[8];
#pragma unroll
            for (int k = 0; k < 8; k++) va[k] = vb[k] = 0;
            for (int s = 0; s < S.count; s++) {
                const int32_t *na = S.n[s] + rowa, *nb = S.n[s] + (has_b ? rowb : rowa);
                int ta[8], tb[8];
#pragma unroll
                for (int k = 0; k < 8; k++) {
                    ta[k] = na[threadIdx.x + (half * 8 + k) * bdim];
                    tb[k] = nb[threadIdx.x + (half * 8 + k) * bdim];
                }
#pragma unroll
                for (int k = 0; k < 8; k++) {
                    va[k] += S.sign[s] * ta[k];
                    vb[k] += S.sign[s] * tb[k];
                }
            }
#pragma unroll
            for (int k = 0; k < 8; k++)
                buf[pad16(threadIdx.x + (half * 8 + k) * bdim)] =
                    make_float2((float)va[k] * S.inv_nscale, has_b ? (float)vb[k] * S.inv_nscale : 0.f);
        }
    } else {
        for (int j = threadIdx.x; j < ny; j += bdim) {
            int va = 0, vb = 0;
            for (int s = 0; s < S.count; s++) {
                va += S.sign[s] * S.n[s][rowa + j];
                if (has_b) vb += S.sign[s] * S.n[s][rowb + j];
            }
            buf[j] = make_float2((float)va * S.inv_nscale, (float)vb * S.inv_nscale);
        }
    }
    float2 *r = buf;
    if (BIG) {
        __syncthreads();
        fft16_inplace<false, NY>(buf, tw, ny);
    } else
        r = fft_stockham<false>(buf, buf + ny, tw, ny);
    for (int l = threadIdx.x; l <= ny / 2; l += bdim) {
        const int lc = (ny - l) & (ny - 1);
        const float2 z = r[BIG ? pad16(l) : l], zc = r[BIG ? pad16(lc) : lc];
        rho_hat[(size_t)ia * LP + l] = make_float2(0.5f * (z.x + zc.x), 0.5f * (z.y - zc.y));
        if (has_b) rho_hat[(size_t)ib * LP + l] = make_float2(0.5f * (z.y + zc.y), 0.5f * (zc.x - z.x));
    }
}

// nodal force of every mobile species, Eq. 16 / 18, evaluated in the epilogue of the inverse
// transform of E (E enters the force only at the node itself):
//   F = qE E_node - (1/2) grad(sum_c a_c^2) [electrons] - C v_th^2 grad(n)/n
// central differences, one-sided on the wall rows, pressure term 0 where n = 0 (Q10)
struct ForceOut {
    const int32_t *nfix[PM2D_MAX_SPECIES];
    float2 *F[PM2D_MAX_SPECIES];
    float qE[PM2D_MAX_SPECIES], pond[PM2D_MAX_SPECIES], cv2[PM2D_MAX_SPECIES];
    int count;
    const float *a;          // [ncomp][nn], the level the stage needs (n or n+1)
    int ncomp, nx;
    float inv_2dx, inv_2dy;
};

// BIG: 0 = radix-4 Stockham (ny < 512), 1 = register-blocked FFT with ny/16 <= 256 threads, 2 = with 512 threads (ny = 8192).
// MODE 0: Z = ehx + i ehy -> Enode (float2);  MODE 1: Z = phi^ -> phi (float, real part);
// MODE 2: Z = ehx + i ehy -> F_s of every mobile species (ForceOut)
// NS: species slots of the force epilogue (2 covers electrons + one ion species with fewer registers)
template <int MODE, int BIG, int NS = PM2D_MAX_SPECIES, int NY = 0>
__global__ void __launch_bounds__(BIG == 2 ? 512 : FFT_THREADS, BIG == 1 ? (NS <= 2 ? 4 : 2) : 1) k_ifft(const float2 *__restrict__ hx, const float2 *__restrict__ hy,
                                                      const float2 *__restrict__ tw, float2 *__restrict__ Enode,
                                                      float *__restrict__ phi, int ny_, int LP, const ForceOut FO)
{
    extern __shared__ float2 buf[];
    const int ny = NY ? NY : ny_, bdim = NY ? NY / 16 : (int)blockDim.x;
    const int i = blockIdx.x;
#pragma unroll 4
    for (int l = threadIdx.x; l <= ny / 2; l += bdim) {
        float2 a = hx[(size_t)i * LP + l];
        float2 b = MODE != 1 ? hy[(size_t)i * LP + l] : make_float2(0.f, 0.f);
        // Z_l = a + i b ; Z_{ny-l} = conj(a) + i conj(b)
        buf[BIG ? pad16(l) : l] = make_float2(a.x - b.y, a.y + b.x);
        if (l > 0 && l < ny / 2) buf[BIG ? pad16(ny - l) : ny - l] = make_float2(a.x + b.y, -a.y + b.x);
    }
    float2 *r = buf;
    if (BIG) {
        __syncthreads();
        fft16_inplace<true, NY>(buf, tw, ny, MODE == 2);
    } else
        r = fft_stockham<true>(buf, buf + ny, tw, ny);
    if (MODE == 2 && BIG) {
        // four consecutive nodes per thread: 128-bit loads of the density and vector-potential rows, E from the
        // unpadded buffer as two LDS.128 (lanes 4..7 of every quarter-warp take the two halves in the other order:
        // no bank conflicts), two 128-bit stores of F per species
        const size_t nn = (size_t)(FO.nx + 1) * ny;
        const int il = i > 0 ? i - 1 : 0, ih = i < FO.nx ? i + 1 : FO.nx;
        const float sx = (il == i || ih == i) ? 2.f * FO.inv_2dx : FO.inv_2dx;     // one-sided at the walls
        const size_t row = (size_t)i * ny, rl = (size_t)il * ny, rh = (size_t)ih * ny;
        bool any_pond = false;
        for (int s = 0; s < FO.count; s++) any_pond |= FO.pond[s] != 0.f;
        const int swz = (threadIdx.x >> 2) & 1;
#pragma unroll 1
        for (int g = threadIdx.x; g < ny / 4; g += bdim) {
            const int j0 = 4 * g, jm = (j0 - 1) & (ny - 1), jp = (j0 + 4) & (ny - 1);
            int4 n0[NS], nh[NS], nl[NS];
            int nd[NS], nu[NS];
#pragma unroll
            for (int s = 0; s < NS; s++)
                if (s < FO.count) {
                    const int32_t *n = FO.nfix[s];
                    n0[s] = *reinterpret_cast<const int4 *>(n + row + j0);
                    nh[s] = *reinterpret_cast<const int4 *>(n + rh + j0);
                    nl[s] = *reinterpret_cast<const int4 *>(n + rl + j0);
                    nd[s] = n[row + jm];
                    nu[s] = n[row + jp];
                }
            float px[4] = {0.f, 0.f, 0.f, 0.f}, py[4] = {0.f, 0.f, 0.f, 0.f};
            if (any_pond) {
                for (int c = 0; c < FO.ncomp; c++) {
                    const float *ac = FO.a + c * nn;
                    const float4 vh = *reinterpret_cast<const float4 *>(ac + rh + j0);
                    const float4 vl = *reinterpret_cast<const float4 *>(ac + rl + j0);
                    const float4 v0 = *reinterpret_cast<const float4 *>(ac + row + j0);
                    const float vd = ac[row + jm], vu = ac[row + jp];
                    const float hx = 0.5f * sx, hy = 0.5f * FO.inv_2dy;
                    px[0] += hx * (vh.x * vh.x - vl.x * vl.x);
                    px[1] += hx * (vh.y * vh.y - vl.y * vl.y);
                    px[2] += hx * (vh.z * vh.z - vl.z * vl.z);
                    px[3] += hx * (vh.w * vh.w - vl.w * vl.w);
                    py[0] += hy * (v0.y * v0.y - vd * vd);
                    py[1] += hy * (v0.z * v0.z - v0.x * v0.x);
                    py[2] += hy * (v0.w * v0.w - v0.y * v0.y);
                    py[3] += hy * (vu * vu - v0.z * v0.z);
                }
            }
            const float4 *rb = reinterpret_cast<const float4 *>(r) + 2 * g;
            const float4 ea = rb[swz], eb = rb[swz ^ 1];
            const float4 e01 = swz ? eb : ea, e23 = swz ? ea : eb;
            const float Ex[4] = {e01.x, e01.z, e23.x, e23.z}, Ey[4] = {e01.y, e01.w, e23.y, e23.w};
#pragma unroll
            for (int s = 0; s < NS; s++)
                if (s < FO.count) {
                    const int c0[4] = {n0[s].x, n0[s].y, n0[s].z, n0[s].w};
                    const int dxn[4] = {nh[s].x - nl[s].x, nh[s].y - nl[s].y, nh[s].z - nl[s].z, nh[s].w - nl[s].w};
                    const int dyn[4] = {n0[s].y - nd[s], n0[s].z - n0[s].x, n0[s].w - n0[s].y, nu[s] - n0[s].z};
                    float fx[4], fy[4];
#pragma unroll
                    for (int u = 0; u < 4; u++) {
                        fx[u] = FO.qE[s] * Ex[u];
                        fy[u] = FO.qE[s] * Ey[u];
                        if (FO.pond[s] != 0.f) { fx[u] -= px[u]; fy[u] -= py[u]; }
                        if (c0[u] > 0 && FO.cv2[s] != 0.f) {
                            const float inv_n = 1.f / (float)c0[u];
                            fx[u] -= FO.cv2[s] * sx * (float)dxn[u] * inv_n;
                            fy[u] -= FO.cv2[s] * FO.inv_2dy * (float)dyn[u] * inv_n;
                        }
                    }
                    float4 *out = reinterpret_cast<float4 *>(FO.F[s] + row + j0);
                    out[0] = make_float4(fx[0], fy[0], fx[1], fy[1]);
                    out[1] = make_float4(fx[2], fy[2], fx[3], fy[3]);
                }
        }
        return;
    }
    if (MODE == 2) {
        const size_t nn = (size_t)(FO.nx + 1) * ny;
        const int il = i > 0 ? i - 1 : 0, ih = i < FO.nx ? i + 1 : FO.nx;
        const float sx = (il == i || ih == i) ? 2.f * FO.inv_2dx : FO.inv_2dx;     // one-sided at the walls
        const size_t row = (size_t)i * ny, rl = (size_t)il * ny, rh = (size_t)ih * ny;
        bool any_pond = false;
        for (int s = 0; s < FO.count; s++) any_pond |= FO.pond[s] != 0.f;
        // four nodes per thread at a time, all loads of a batch issued before the arithmetic
        constexpr int NB = 2;
        for (int jb = threadIdx.x; jb < ny; jb += NB * bdim) {
            int jj[NB], jm[NB], jp[NB];
            float px[NB], py[NB];
#pragma unroll
            for (int u = 0; u < NB; u++) {
                jj[u] = min(jb + u * (int)bdim, ny - 1);           // clamped duplicates are not stored
                jm[u] = (jj[u] - 1) & (ny - 1);
                jp[u] = (jj[u] + 1) & (ny - 1);
                px[u] = py[u] = 0.f;
            }
            int n0[NS][NB], nh[NS][NB], nl[NS][NB], nu[NS][NB], nd[NS][NB];
#pragma unroll
            for (int s = 0; s < NS; s++)
                if (s < FO.count) {
                    const int32_t *n = FO.nfix[s];
#pragma unroll
                    for (int u = 0; u < NB; u++) {
                        n0[s][u] = n[row + jj[u]];
                        nh[s][u] = n[rh + jj[u]];
                        nl[s][u] = n[rl + jj[u]];
                        nu[s][u] = n[row + jp[u]];
                        nd[s][u] = n[row + jm[u]];
                    }
                }
            if (any_pond) {
                for (int c = 0; c < FO.ncomp; c++) {
                    const float *ac = FO.a + c * nn;
                    float vh[NB], vl[NB], vu[NB], vd[NB];
#pragma unroll
                    for (int u = 0; u < NB; u++) {
                        vh[u] = ac[rh + jj[u]];
                        vl[u] = ac[rl + jj[u]];
                        vu[u] = ac[row + jp[u]];
                        vd[u] = ac[row + jm[u]];
                    }
#pragma unroll
                    for (int u = 0; u < NB; u++) {
                        px[u] += 0.5f * sx * (vh[u] * vh[u] - vl[u] * vl[u]);
                        py[u] += 0.5f * FO.inv_2dy * (vu[u] * vu[u] - vd[u] * vd[u]);
                    }
                }
            }
#pragma unroll
            for (int s = 0; s < NS; s++)
                if (s < FO.count) {
#pragma unroll
                    for (int u = 0; u < NB; u++) {
                        const float2 E = r[BIG ? pad16(jj[u]) : jj[u]];
                        float fx = FO.qE[s] * E.x, fy = FO.qE[s] * E.y;
                        if (FO.pond[s] != 0.f) { fx -= px[u]; fy -= py[u]; }
                        if (n0[s][u] > 0 && FO.cv2[s] != 0.f) {
                            const float inv_n = 1.f / (float)n0[s][u];
                            fx -= FO.cv2[s] * sx * (float)(nh[s][u] - nl[s][u]) * inv_n;
                            fy -= FO.cv2[s] * FO.inv_2dy * (float)(nu[s][u] - nd[s][u]) * inv_n;
                        }
                        if (jb + u * (int)bdim < ny) FO.F[s][row + jj[u]] = make_float2(fx, fy);
                    }
                }
        }
        return;
    }
    for (int j = threadIdx.x; j < ny; j += bdim) {
        const float2 z = r[BIG ? pad16(j) : j];
        if (MODE == 0) Enode[(size_t)i * ny + j] = z;
        else phi[(size_t)i * ny + j] = z.x;
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

// ---- partitioned chasing method ---------------------------------------------------------------------
// tables [cls][j][LP], cls 0 = full partition (m = M-1 interior rows), cls 1 = last partition (m_last)
struct TriTables {
    double *cp, *V, *W;     // local c', spikes V (1 at the left interface), W (1 at the right interface)
    double *den;            // [P][LP]: 1 / pivot of row k of the reduced (interface) system, k = 1 .. P-1
};

__global__ void k_tri_tables(TriTables T, int ny, int LP, int m_last, int P, double dx, double Ly)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l > ny / 2) return;
    const double PI = 3.14159265358979323846;
    const double ky = 2.0 * PI * (double)l / Ly;
    const double b = -2.0 - ky * ky * dx * dx;                   // Eq. 11 times dx^2
    for (int cls = 0; cls < 2; cls++) {
        const int m = cls == 0 ? M - 1 : m_last;
        double *cp = T.cp + (size_t)cls * M * LP, *V = T.V + (size_t)cls * M * LP, *W = T.W + (size_t)cls * M * LP;
        double c = 0.0;
        for (int j = 1; j <= m; j++) {
            c = 1.0 / (b - c);
            cp[(size_t)j * LP + l] = c;
        }
        // V: local solve of A V = -e_1 ; W: A W = -e_m
        double d = 0.0;
        for (int j = 1; j <= m; j++) {
            d = ((j == 1 ? -1.0 : 0.0) - d) * cp[(size_t)j * LP + l];
            V[(size_t)j * LP + l] = d;                             // forward result, overwritten below
        }
        double v = 0.0;
        for (int j = m; j >= 1; j--) {
            v = V[(size_t)j * LP + l] - cp[(size_t)j * LP + l] * v;
            V[(size_t)j * LP + l] = v;
        }
        double w = 0.0;
        for (int j = m; j >= 1; j--) {
            w = (j == m ? -cp[(size_t)j * LP + l] : 0.0) - cp[(size_t)j * LP + l] * w;
            W[(size_t)j * LP + l] = w;
        }
    }
    // pivots of the reduced system (right-hand-side independent): row k is
    //   Vm g_{k-1} + (Wm + b + V1(k)) g_k + W1 g_{k+1} = ...
    const double Vm = T.V[(size_t)(M - 1) * LP + l], Wm = T.W[(size_t)(M - 1) * LP + l];
    const double V1 = T.V[(size_t)1 * LP + l], W1 = T.W[(size_t)1 * LP + l];
    const double V1_last = m_last >= 1 ? T.V[((size_t)M + 1) * LP + l] : 0.0;
    double cprev = 0.0;
    for (int k = 1; k <= P - 1; k++) {
        const double den = 1.0 / (Wm + b + (k == P - 1 ? V1_last : V1) - Vm * cprev);
        cprev = W1 * den;
        T.den[(size_t)k * LP + l] = den;
    }
}

struct TriParams {
    const float2 *rho_hat;
    float2 *phi_hat;      // may alias rho_hat; NULL: not wanted
    TriTables tab;
    double2 *sumV, *sumW; // [P][LP]
    double2 *g;           // [P+1][LP] interface values (g_0 = g_P = 0)
    float2 *ehx, *ehy;
    int nx, ny, LP, P, m_last;
    double dx2, inv_dx, inv_dy, inv_ny, Ly;
};

// S_V = sum_j V_j r_j, S_W = sum_j W_j r_j over the interior rows of partition k (r = dx^2 rho^)
__global__ void __launch_bounds__(128) k_tri_sums(const TriParams T)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y;
    if (l > T.ny / 2) return;
    const int cls = (k == T.P - 1) ? 1 : 0, m = cls ? T.m_last : M - 1;
    const double *V = T.tab.V + (size_t)cls * M * T.LP, *W = T.tab.W + (size_t)cls * M * T.LP;
    double svr = 0.0, svi = 0.0, swr = 0.0, swi = 0.0;
#pragma unroll 8
    for (int j = 1; j <= m; j++) {
        float2 r = T.rho_hat[(size_t)(k * M + j) * T.LP + l];
        double v = V[(size_t)j * T.LP + l], w = W[(size_t)j * T.LP + l];
        svr += v * (double)r.x; svi += v * (double)r.y;
        swr += w * (double)r.x; swi += w * (double)r.y;
    }
    T.sumV[(size_t)k * T.LP + l] = make_double2(T.dx2 * svr, T.dx2 * svi);
    T.sumW[(size_t)k * T.LP + l] = make_double2(T.dx2 * swr, T.dx2 * swi);
}

// reduced system for the interface values, one thread per k_y, chasing method in double
__global__ void __launch_bounds__(32) k_tri_reduced(const TriParams T)
{
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l > T.ny / 2) return;
    const int LP = T.LP, P = T.P;
    const double PI = 3.14159265358979323846;
    const double ky = 2.0 * PI * (double)l / T.Ly;
    const double b = -2.0 - ky * ky * T.dx2;
    const double Vm = T.tab.V[(size_t)(M - 1) * LP + l], Wm = T.tab.W[(size_t)(M - 1) * LP + l];
    const double V1 = T.tab.V[(size_t)1 * LP + l], W1 = T.tab.W[(size_t)1 * LP + l];
    const double V1_last = T.m_last >= 1 ? T.tab.V[((size_t)M + 1) * LP + l] : 0.0;
    T.g[l] = make_double2(0.0, 0.0);
    T.g[(size_t)P * LP + l] = make_double2(0.0, 0.0);
    if (P < 2) return;
    // forward: row k: Vm g_{k-1} + (Wm + b + V1(k)) g_k + W1 g_{k+1} = r_{kM} + S_W(k-1) + S_V(k)
    double cprev = 0.0, dr = 0.0, di = 0.0;
    double2 *cd = T.g;                       // store d_k in g[k] and c'_k in sumV[k].x (free after read)
    constexpr int CH = 8;                    // the inputs of CH rows are loaded before their (serial) elimination
    for (int k0 = 1; k0 <= P - 1; k0 += CH) {
        float2 r[CH];
        double2 sw[CH], sv[CH];
#pragma unroll
        for (int u = 0; u < CH; u++) {
            const int k = min(k0 + u, P - 1);
            r[u] = T.rho_hat[(size_t)(k * M) * LP + l];
            sw[u] = T.sumW[(size_t)(k - 1) * LP + l];
            sv[u] = T.sumV[(size_t)k * LP + l];
        }
#pragma unroll
        for (int u = 0; u < CH; u++) {
            const int k = k0 + u;
            if (k <= P - 1) {
                double diag = Wm + b + (k == P - 1 ? V1_last : V1);
                double den = 1.0 / (diag - Vm * cprev);
                double Rr = T.dx2 * (double)r[u].x + sw[u].x + sv[u].x, Ri = T.dx2 * (double)r[u].y + sw[u].y + sv[u].y;
                dr = (Rr - Vm * dr) * den;
                di = (Ri - Vm * di) * den;
                cprev = W1 * den;
                cd[(size_t)k * LP + l] = make_double2(dr, di);
                T.sumV[(size_t)k * LP + l].x = cprev;
            }
        }
    }
    double gr = 0.0, gi = 0.0;
    for (int k0 = P - 1; k0 >= 1; k0 -= CH) {
        double2 d[CH];
        double cc[CH];
#pragma unroll
        for (int u = 0; u < CH; u++) {
            const int k = max(k0 - u, 1);
            d[u] = cd[(size_t)k * LP + l];
            cc[u] = T.sumV[(size_t)k * LP + l].x;
        }
#pragma unroll
        for (int u = 0; u < CH; u++) {
            const int k = k0 - u;
            if (k >= 1) {
                gr = d[u].x - cc[u] * gr;
                gi = d[u].y - cc[u] * gi;
                cd[(size_t)k * LP + l] = make_double2(gr, gi);
            }
        }
    }
}

// The same solve with every input of the thread -- r, S_W, S_V and the tabulated pivots of all P-1 rows -- copied to
// shared memory by cp.async first: the two recurrences then run at arithmetic latency instead of meeting a memory
// round trip per chunk of rows.  Few threads per CTA (the staged column of one k_y is 48 (P-1) bytes).
constexpr int TR_THREADS = 8;
__host__ __device__ constexpr size_t tri_reduced_smem(int P) { return (size_t)(P - 1) * TR_THREADS * 48; }

__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gmem_src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}
__device__ __forceinline__ void cp_async8r(void *smem_dst, const void *gmem_src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}

__global__ void __launch_bounds__(TR_THREADS) k_tri_reduced_staged(const TriParams T)
{
    extern __shared__ __align__(16) unsigned char tr_smem[];
    const int LP = T.LP, P = T.P, nk = P - 1;
    const int l = blockIdx.x * TR_THREADS + threadIdx.x;
    if (l > T.ny / 2) return;
    T.g[l] = make_double2(0.0, 0.0);
    T.g[(size_t)P * LP + l] = make_double2(0.0, 0.0);
    if (P < 2) return;
    double2 *sws = reinterpret_cast<double2 *>(tr_smem) + threadIdx.x;                                   // [nk][TR_THREADS]; later d_k
    double2 *svs = reinterpret_cast<double2 *>(tr_smem) + (size_t)nk * TR_THREADS + threadIdx.x;
    double *dens = reinterpret_cast<double *>(tr_smem + (size_t)nk * TR_THREADS * 32) + threadIdx.x;
    float2 *rs = reinterpret_cast<float2 *>(tr_smem + (size_t)nk * TR_THREADS * 40) + threadIdx.x;
    for (int k = 1; k <= nk; k++) {
        const int e = (k - 1) * TR_THREADS;
        cp_async16(sws + e, T.sumW + (size_t)(k - 1) * LP + l);
        cp_async16(svs + e, T.sumV + (size_t)k * LP + l);
        cp_async8r(dens + e, T.tab.den + (size_t)k * LP + l);
        cp_async8r(rs + e, T.rho_hat + (size_t)(k * M) * LP + l);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    const double Vm = T.tab.V[(size_t)(M - 1) * LP + l], W1 = T.tab.W[(size_t)1 * LP + l];
    asm volatile("cp.async.wait_all;" ::: "memory");
    double dr = 0.0, di = 0.0;
#pragma unroll 4
    for (int k = 1; k <= nk; k++) {
        const int e = (k - 1) * TR_THREADS;
        const double den = dens[e];
        const double2 sw = sws[e], sv = svs[e];
        const float2 r = rs[e];
        const double Rr = T.dx2 * (double)r.x + sw.x + sv.x, Ri = T.dx2 * (double)r.y + sw.y + sv.y;
        dr = (Rr - Vm * dr) * den;
        di = (Ri - Vm * di) * den;
        sws[e] = make_double2(dr, di);
    }
    double gr = 0.0, gi = 0.0;
#pragma unroll 4
    for (int k = nk; k >= 1; k--) {
        const int e = (k - 1) * TR_THREADS;
        const double cc = W1 * dens[e];
        const double2 d = sws[e];
        gr = d.x - cc * gr;
        gi = d.y - cc * gi;
        T.g[(size_t)k * LP + l] = make_double2(gr, gi);
    }
}

// one thread per (k_y, partition): local chasing solve in registers with the true interface values,
// then the nodal-E spectra of rows kM .. kM+m (plus the wall row nx for the last partition)
// The thread's column of rho^ (rows kM .. kM+m) and of the elimination table go to shared memory by
// cp.async first -- 2 M independent copies in flight per thread, no registers held -- because the
// chasing recurrence itself is serial and would otherwise meet one DRAM latency per row.  Every thread
// reads back only what it copied itself: cp.async.wait_all is the only synchronisation needed.
constexpr int TL_THREADS = 128;
constexpr size_t TL_SMEM = (size_t)M * TL_THREADS * (sizeof(float2) + sizeof(double));

__device__ __forceinline__ void cp_async8(void *smem_dst, const void *gmem_src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"((uint32_t)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src) : "memory");
}

__global__ void __launch_bounds__(TL_THREADS) k_tri_local(const TriParams T)
{
    extern __shared__ __align__(16) unsigned char tl_smem[];
    float2 *rs = reinterpret_cast<float2 *>(tl_smem) + threadIdx.x;                                  // [M][TL_THREADS]
    double *cs = reinterpret_cast<double *>(tl_smem + (size_t)M * TL_THREADS * sizeof(float2)) + threadIdx.x;
    const int l = blockIdx.x * blockDim.x + threadIdx.x, k = blockIdx.y;
    if (l > T.ny / 2) return;
    const int LP = T.LP;
    const int cls = (k == T.P - 1) ? 1 : 0, m = cls ? T.m_last : M - 1;
    const size_t row0 = (size_t)k * M;
    {
        const double *cp = T.tab.cp + (size_t)cls * M * LP;
        cp_async8(rs, T.rho_hat + row0 * LP + l);
#pragma unroll
        for (int j = 1; j < M; j++)
            if (j <= m) {
                cp_async8(rs + j * TL_THREADS, T.rho_hat + (row0 + j) * LP + l);
                cp_async8(cs + j * TL_THREADS, cp + (size_t)j * LP + l);
            }
        asm volatile("cp.async.commit_group;" ::: "memory");
    }
    const double2 gl = T.g[(size_t)k * LP + l], gr = T.g[(size_t)(k + 1) * LP + l];
    asm volatile("cp.async.wait_all;" ::: "memory");
    double dr[M], di[M];
    // forward elimination with the interface values folded into rows 1 and m
    {
        double pr = 0.0, pi = 0.0;
#pragma unroll
        for (int j = 1; j < M; j++) {
            if (j <= m) {
                float2 r = rs[j * TL_THREADS];
                double c = cs[j * TL_THREADS];
                double rr = T.dx2 * (double)r.x, ri = T.dx2 * (double)r.y;
                if (j == 1) { rr -= gl.x; ri -= gl.y; }
                if (j == m) { rr -= gr.x; ri -= gr.y; }
                pr = (rr - pr) * c;
                pi = (ri - pi) * c;
            }
            dr[j] = pr; di[j] = pi;
        }
    }
    const double PI = 3.14159265358979323846;
    const double theta = 2.0 * PI * (double)l / (double)T.ny;
    const double ch = cos(0.5 * theta), sn = sin(theta);
    const double kx = -ch * ch * 0.5 * T.inv_dx * T.inv_ny;     // times (phi_{e+1} - phi_{e-1})
    const double kyf = -sn * 0.25 * T.inv_dy * T.inv_ny;        // times i (phi_{e-1} + 2 phi_e + phi_{e+1})
    // back substitution from row m down to 1; p1 = phi_{j+1}, p2 = phi_{j+2}
    double p2r = 0.0, p2i = 0.0, p1r = gr.x, p1i = gr.y;
    const bool right_wall = (k == T.P - 1);    // then gr = g_P = 0 = phi_nx
#pragma unroll
    for (int j = M - 1; j >= 1; j--) {
        if (j <= m) {
            double c = cs[j * TL_THREADS];
            // phi_j; the right boundary value is already folded into d_m
            double pr = dr[j] - (j == m ? 0.0 : c * p1r), pi = di[j] - (j == m ? 0.0 : c * p1i);
            const size_t e = row0 + j + 1;                           // row j+1 now has both neighbours
            if (j == m) {
                if (right_wall) {    // e == nx: mean of the two cells at nx - 1/2
                    T.ehx[e * LP + l] = make_float2((float)(-2.0 * kx * pr), (float)(-2.0 * kx * pi));
                    T.ehy[e * LP + l] = make_float2((float)(-2.0 * kyf * pi), (float)(2.0 * kyf * pr));
                }   // else: row e is the next partition's interface row, emitted there
            } else {
                double sr = pr + 2.0 * p1r + p2r, si = pi + 2.0 * p1i + p2i;
                T.ehx[e * LP + l] = make_float2((float)(kx * (p2r - pr)), (float)(kx * (p2i - pi)));
                T.ehy[e * LP + l] = make_float2((float)(-kyf * si), (float)(kyf * sr));
            }
            if (T.phi_hat) T.phi_hat[(row0 + j) * LP + l] = make_float2((float)(pr * T.inv_ny), (float)(pi * T.inv_ny));
            p2r = p1r; p2i = p1i;
            p1r = pr; p1i = pi;
        }
    }
    // now p1 = phi_1 and p2 = phi_2 (or the right boundary value); m == 0: p1 = right boundary value
    if (m >= 1) {        // row kM+1: left neighbour is the interface value
        double sr = gl.x + 2.0 * p1r + p2r, si = gl.y + 2.0 * p1i + p2i;
        const size_t e = row0 + 1;
        T.ehx[e * LP + l] = make_float2((float)(kx * (p2r - gl.x)), (float)(kx * (p2i - gl.y)));
        T.ehy[e * LP + l] = make_float2((float)(-kyf * si), (float)(kyf * sr));
    } else if (right_wall) {   // empty last partition: the wall row nx is this interface's right neighbour
        const size_t e = row0 + 1;
        T.ehx[e * LP + l] = make_float2((float)(-2.0 * kx * gl.x), (float)(-2.0 * kx * gl.y));
        T.ehy[e * LP + l] = make_float2((float)(-2.0 * kyf * gl.y), (float)(2.0 * kyf * gl.x));
    }
    // interface row kM itself
    if (k == 0) {        // left wall: mean of the two cells at 1/2, phi_0 = 0
        T.ehx[l] = make_float2((float)(2.0 * kx * p1r), (float)(2.0 * kx * p1i));
        T.ehy[l] = make_float2((float)(-2.0 * kyf * p1i), (float)(2.0 * kyf * p1r));
        if (T.phi_hat) {
            T.phi_hat[l] = make_float2(0.f, 0.f);
            T.phi_hat[(size_t)T.nx * LP + l] = make_float2(0.f, 0.f);
        }
    } else {
        // phi_{kM-1} from the interface equation: phi_{kM-1} + b g_k + phi_{kM+1} = dx^2 rho^_{kM}
        const double kyc = 2.0 * PI * (double)l / T.Ly;
        const double b = -2.0 - kyc * kyc * T.dx2;
        float2 r = rs[0];
        double lr = T.dx2 * (double)r.x - b * gl.x - p1r, li = T.dx2 * (double)r.y - b * gl.y - p1i;
        double sr = lr + 2.0 * gl.x + p1r, si = li + 2.0 * gl.y + p1i;
        T.ehx[row0 * LP + l] = make_float2((float)(kx * (p1r - lr)), (float)(kx * (p1i - li)));
        T.ehy[row0 * LP + l] = make_float2((float)(-kyf * si), (float)(kyf * sr));
        if (T.phi_hat) T.phi_hat[row0 * LP + l] = make_float2((float)(gl.x * T.inv_ny), (float)(gl.y * T.inv_ny));
    }
}

}  // namespace

int launch_poisson_init(pm2d_ctx *c)
{
    const int ny = c->g.ny, nx = c->g.nx;
    c->tri_P = (nx + M - 1) / M;
    c->tri_mlast = nx - (c->tri_P - 1) * M - 1;
    k_twiddle_init<<<(ny / 2 + 127) / 128, 128, 0, c->stream>>>(c->twiddle, ny);
    TriTables T{c->tri_cp, c->tri_V, c->tri_W, c->tri_den};
    k_tri_tables<<<(ny / 2 + 1 + 31) / 32, 32, 0, c->stream>>>(T, ny, c->LP, c->tri_mlast, c->tri_P, c->g.dx, ny * c->g.dy);
    if (c->tri_P >= 2 && tri_reduced_smem(c->tri_P) <= 100 * 1024)
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_tri_reduced_staged, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)tri_reduced_smem(c->tri_P)));
    count_launch(c, 2);
    PM2D_CUDA_CHECK(cudaGetLastError());
    const int smem = 2 * ny * (int)sizeof(float2);       // small-n path only (ny < 512): 8 KB at most
    (void)smem;
    {
        const int big_smem = (8192 + 8192 / 16) * (int)sizeof(float2);
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_tri_local, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TL_SMEM));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_fft_rho<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, big_smem));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_ifft<0, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, big_smem));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_ifft<1, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, big_smem));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_ifft<2, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, big_smem));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_ifft<2, 1, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, big_smem));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_fft_rho<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, big_smem));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_fft_rho<2, 8192>, cudaFuncAttributeMaxDynamicSharedMemorySize, big_smem));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_ifft<2, 2, PM2D_MAX_SPECIES, 8192>, cudaFuncAttributeMaxDynamicSharedMemorySize, big_smem));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_ifft<0, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, big_smem));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_ifft<1, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, big_smem));
        PM2D_CUDA_CHECK(cudaFuncSetAttribute(k_ifft<2, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, big_smem));
    }
    return PM2D_OK;
}

// rho from the current density grids -> nodal E (and phi if wanted, for diagnostics); with force_a (a time
// level of the vector potential) the nodal force of every mobile species instead of E
int launch_poisson(pm2d_ctx *c, bool want_phi, const float *force_a, bool use_hat)
{
    const int nx = c->g.nx, ny = c->g.ny;
    const int big = ny >= 8192 ? 2 : (ny >= 512 ? 1 : 0);
    const size_t smem = big ? (size_t)(ny + ny / 16) * sizeof(float2) : 2 * (size_t)ny * sizeof(float2);
    const int fft_threads = big ? ny / 16 : FFT_THREADS;
    RhoSrc S;
    S.count = 0;
    S.inv_nscale = c->inv_nscale;
    for (int s = 0; s < c->nsp; s++)
        if (c->sp[s].cfg.sign != 0) {
            S.n[S.count] = (use_hat && c->sp[s].cfg.mobile) ? c->sp[s].nhat : c->sp[s].nfix;
            S.sign[S.count] = c->sp[s].cfg.sign;
            S.count++;
        }
    if (ny == 8192) k_fft_rho<2, 8192><<<nx / 2, fft_threads, smem, c->stream>>>(S, c->twiddle, c->rho_hat, nx, ny, c->LP);
    else if (ny == 4096) k_fft_rho<1, 4096><<<nx / 2, fft_threads, smem, c->stream>>>(S, c->twiddle, c->rho_hat, nx, ny, c->LP);
    else if (ny == 2048) k_fft_rho<1, 2048><<<nx / 2, fft_threads, smem, c->stream>>>(S, c->twiddle, c->rho_hat, nx, ny, c->LP);
    else if (ny == 1024) k_fft_rho<1, 1024><<<nx / 2, fft_threads, smem, c->stream>>>(S, c->twiddle, c->rho_hat, nx, ny, c->LP);
    else if (big == 2) k_fft_rho<2><<<nx / 2, fft_threads, smem, c->stream>>>(S, c->twiddle, c->rho_hat, nx, ny, c->LP);
    else if (big == 1) k_fft_rho<1><<<nx / 2, fft_threads, smem, c->stream>>>(S, c->twiddle, c->rho_hat, nx, ny, c->LP);
    else k_fft_rho<0><<<nx / 2, fft_threads, smem, c->stream>>>(S, c->twiddle, c->rho_hat, nx, ny, c->LP);
    TriParams T;
    T.rho_hat = c->rho_hat; T.phi_hat = want_phi ? c->rho_hat : nullptr;
    T.tab = TriTables{c->tri_cp, c->tri_V, c->tri_W, c->tri_den};
    T.sumV = c->tri_sumV; T.sumW = c->tri_sumW; T.g = c->tri_g;
    T.ehx = c->ehx; T.ehy = c->ehy; T.nx = nx; T.ny = ny; T.LP = c->LP; T.P = c->tri_P; T.m_last = c->tri_mlast;
    T.dx2 = c->g.dx * c->g.dx; T.inv_dx = 1.0 / c->g.dx; T.inv_dy = 1.0 / c->g.dy; T.inv_ny = 1.0 / ny; T.Ly = ny * c->g.dy;
    dim3 grid((ny / 2 + 1 + 127) / 128, c->tri_P);
    k_tri_sums<<<grid, 128, 0, c->stream>>>(T);
    if (c->tri_P >= 2 && tri_reduced_smem(c->tri_P) <= 100 * 1024)
        k_tri_reduced_staged<<<(ny / 2 + 1 + TR_THREADS - 1) / TR_THREADS, TR_THREADS, tri_reduced_smem(c->tri_P), c->stream>>>(T);
    else
        k_tri_reduced<<<(ny / 2 + 1 + 31) / 32, 32, 0, c->stream>>>(T);
    k_tri_local<<<grid, TL_THREADS, TL_SMEM, c->stream>>>(T);
    ForceOut FO;
    FO.count = 0;
    if (force_a) {
        const double PI = 3.14159265358979323846;
        for (int s = 0; s < c->nsp; s++) {
            SpeciesDev &Q = c->sp[s];
            if (!Q.cfg.mobile || Q.np == 0) continue;
            const int k = FO.count++;
            FO.nfix[k] = use_hat ? Q.nhat : Q.nfix; FO.F[k] = Q.F;
            FO.qE[k] = (float)(-(double)Q.cfg.sign * 4.0 * PI * PI / Q.cfg.mass);
            FO.pond[k] = Q.cfg.sign < 0 ? 1.f : 0.f;
            FO.cv2[k] = (float)(Q.cfg.pressure_coeff * Q.vth2);
        }
        FO.a = force_a; FO.ncomp = c->g.ncomp; FO.nx = nx;
        FO.inv_2dx = (float)(1.0 / (2.0 * c->g.dx)); FO.inv_2dy = (float)(1.0 / (2.0 * c->g.dy));
        if (ny == 8192) k_ifft<2, 2, PM2D_MAX_SPECIES, 8192><<<nx + 1, fft_threads, smem, c->stream>>>(c->ehx, c->ehy, c->twiddle, nullptr, nullptr, ny, c->LP, FO);
        else if (ny == 4096 && FO.count <= 2) k_ifft<2, 1, 2, 4096><<<nx + 1, fft_threads, smem, c->stream>>>(c->ehx, c->ehy, c->twiddle, nullptr, nullptr, ny, c->LP, FO);
        else if (ny == 2048 && FO.count <= 2) k_ifft<2, 1, 2, 2048><<<nx + 1, fft_threads, smem, c->stream>>>(c->ehx, c->ehy, c->twiddle, nullptr, nullptr, ny, c->LP, FO);
        else if (ny == 1024 && FO.count <= 2) k_ifft<2, 1, 2, 1024><<<nx + 1, fft_threads, smem, c->stream>>>(c->ehx, c->ehy, c->twiddle, nullptr, nullptr, ny, c->LP, FO);
        else if (big == 2) k_ifft<2, 2><<<nx + 1, fft_threads, smem, c->stream>>>(c->ehx, c->ehy, c->twiddle, nullptr, nullptr, ny, c->LP, FO);
        else if (big == 1 && FO.count <= 2) k_ifft<2, 1, 2><<<nx + 1, fft_threads, smem, c->stream>>>(c->ehx, c->ehy, c->twiddle, nullptr, nullptr, ny, c->LP, FO);
        else if (big == 1) k_ifft<2, 1><<<nx + 1, fft_threads, smem, c->stream>>>(c->ehx, c->ehy, c->twiddle, nullptr, nullptr, ny, c->LP, FO);
        else k_ifft<2, 0><<<nx + 1, fft_threads, smem, c->stream>>>(c->ehx, c->ehy, c->twiddle, nullptr, nullptr, ny, c->LP, FO);
    } else if (big == 2)
        k_ifft<0, 2><<<nx + 1, fft_threads, smem, c->stream>>>(c->ehx, c->ehy, c->twiddle, c->Enode, nullptr, ny, c->LP, FO);
    else if (big == 1)
        k_ifft<0, 1><<<nx + 1, fft_threads, smem, c->stream>>>(c->ehx, c->ehy, c->twiddle, c->Enode, nullptr, ny, c->LP, FO);
    else
        k_ifft<0, 0><<<nx + 1, fft_threads, smem, c->stream>>>(c->ehx, c->ehy, c->twiddle, c->Enode, nullptr, ny, c->LP, FO);
    count_launch(c, 5);
    if (want_phi) {
        if (big == 2) k_ifft<1, 2><<<nx + 1, fft_threads, smem, c->stream>>>(c->rho_hat, nullptr, c->twiddle, nullptr, c->phi, ny, c->LP, FO);
        else if (big == 1) k_ifft<1, 1><<<nx + 1, fft_threads, smem, c->stream>>>(c->rho_hat, nullptr, c->twiddle, nullptr, c->phi, ny, c->LP, FO);
        else k_ifft<1, 0><<<nx + 1, fft_threads, smem, c->stream>>>(c->rho_hat, nullptr, c->twiddle, nullptr, c->phi, ny, c->LP, FO);
        count_launch(c);
    }
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}
