// pm2d_static.cu -- pm2d_mode_amplitudes_static: the Fourier-mode amplitudes of pm2d_mode_amplitudes (a8) for callers that
// may not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).  No ctx, no workspace: the
// caller passes the density and the result as device pointers, and the scratch is the file-scope array below.
//
// The sum  A(m_x, m_y) = sum_{i, j} vol_i n_{i j} exp(-2 pi i (m_x i / nx + m_y j / ny))  is taken in two passes:
//   k_modes_rows  one CTA per node row i: R_i(m) = vol_i sum_j n_{i j} exp(-2 pi i m_y j / ny)   -> scratch[i][m]
//   k_modes_cols  one CTA per mode m:     A(m)   = sum_i R_i(m) exp(-2 pi i m_x i / nx)          -> out[2 m], out[2 m + 1]
// float32 inputs, float64 sums in a fixed order (unlike the atomics of k_diag_modes the result is reproducible); the
// phases are reduced mod 1 in integers before sincospi, as in k_diag_modes.
#include <mutex>

#include "pm2d_internal.h"

namespace {

constexpr int SM_THREADS = 256;
constexpr int SM_MAX_DEVICES = 64;

// [row][mode] (re, im): 16385 * 16 * 16 B = 4.0 MiB, held by every GPU that loads libpm2d.so until the process exits.
// In host code this name is a host-side stand-in, NOT a device address: only static_scratch() below may touch it.
static __device__ __align__(256) double2 g_modes_scratch[(size_t)PM2D_STATIC_MAX_ROWS * PM2D_MAX_MODES];

struct StaticModes {
    const float *n;
    double2 *rows;
    double *out;
    int nx, ny, nmodes;
    int mx[PM2D_MAX_MODES], my[PM2D_MAX_MODES];
};

// sum over the CTA of a (re, im) pair; the result is valid in thread 0
__device__ __forceinline__ double2 block_sum2(double2 v)
{
    __shared__ double2 ws[SM_THREADS / 32];
    for (int o = 16; o > 0; o >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, o);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, o);
    }
    __syncthreads();                                   // ws of the previous call has been read
    if ((threadIdx.x & 31) == 0) ws[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0)
        for (int k = 1; k < SM_THREADS / 32; k++) {
            v.x += ws[k].x;
            v.y += ws[k].y;
        }
    return v;
}

__global__ void __launch_bounds__(SM_THREADS) k_modes_rows(const StaticModes M)
{
    const int i = blockIdx.x;
    double re[PM2D_MAX_MODES], im[PM2D_MAX_MODES];
#pragma unroll
    for (int m = 0; m < PM2D_MAX_MODES; m++) re[m] = im[m] = 0.0;
    const double inv_ny = 1.0 / M.ny;
    const float *row = M.n + (size_t)i * M.ny;
    for (int j = threadIdx.x; j < M.ny; j += SM_THREADS) {
        const double n = (double)row[j];
        if (n == 0.0) continue;
#pragma unroll
        for (int m = 0; m < PM2D_MAX_MODES; m++) {
            if (m >= M.nmodes) break;
            const int64_t py = ((int64_t)M.my[m] * j) % M.ny;
            double sn, cs;
            sincospi(-2.0 * (double)py * inv_ny, &sn, &cs);
            re[m] += n * cs;
            im[m] += n * sn;
        }
    }
    const double vol = (i == 0 || i == M.nx) ? 0.5 : 1.0;
#pragma unroll
    for (int m = 0; m < PM2D_MAX_MODES; m++) {
        if (m >= M.nmodes) break;
        const double2 s = block_sum2(make_double2(re[m], im[m]));
        if (threadIdx.x == 0) M.rows[(size_t)i * PM2D_MAX_MODES + m] = make_double2(vol * s.x, vol * s.y);
    }
}

__global__ void __launch_bounds__(SM_THREADS) k_modes_cols(const StaticModes M)
{
    const int m = blockIdx.x;
    const double inv_nx = 1.0 / M.nx;
    double2 acc = make_double2(0.0, 0.0);
    for (int i = threadIdx.x; i <= M.nx; i += SM_THREADS) {
        const double2 r = M.rows[(size_t)i * PM2D_MAX_MODES + m];
        const int64_t px = ((int64_t)M.mx[m] * i) % M.nx;
        double sn, cs;
        sincospi(-2.0 * (double)px * inv_nx, &sn, &cs);
        acc.x += r.x * cs - r.y * sn;
        acc.y += r.x * sn + r.y * cs;
    }
    acc = block_sum2(acc);
    if (threadIdx.x == 0) {
        M.out[2 * m] = acc.x;
        M.out[2 * m + 1] = acc.y;
    }
}

// device address of g_modes_scratch on the current device: resolved once per device, with that device current
int static_scratch(double2 **ptr)
{
    static std::mutex mu;
    static double2 *cache[SM_MAX_DEVICES] = {};
    int dev = -1;
    PM2D_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= SM_MAX_DEVICES) {
        pm2d_set_error("pm2d_mode_amplitudes_static: device ordinal out of range");
        return PM2D_EINVAL;
    }
    std::lock_guard<std::mutex> lock(mu);
    if (!cache[dev]) {
        void *p = nullptr;
        PM2D_CUDA_CHECK(cudaGetSymbolAddress(&p, g_modes_scratch));
        if (!p) {
            pm2d_set_error("pm2d_mode_amplitudes_static: cudaGetSymbolAddress returned a null address");
            return PM2D_ECUDA;
        }
        cache[dev] = (double2 *)p;
    }
    *ptr = cache[dev];
    return PM2D_OK;
}

}  // namespace

extern "C" int pm2d_mode_amplitudes_static(const float *n_dev, int nx, int ny, int nmodes, const int32_t *mx, const int32_t *my,
                                           double *out_dev, void *stream)
{
    if (!n_dev || !out_dev || !mx || !my || nx < 1 || ny < 1 || nmodes < 1 || nmodes > PM2D_MAX_MODES) {
        pm2d_set_error("pm2d_mode_amplitudes_static: bad argument (non-null pointers, nx, ny >= 1, 1 <= nmodes <= PM2D_MAX_MODES)");
        return PM2D_EINVAL;
    }
    if (nx + 1 > PM2D_STATIC_MAX_ROWS) {
        pm2d_set_error("pm2d_mode_amplitudes_static: nx + 1 = " + std::to_string(nx + 1) + " node rows exceed PM2D_STATIC_MAX_ROWS = " +
                       std::to_string(PM2D_STATIC_MAX_ROWS) + " (the size of the static scratch array); use pm2d_mode_amplitudes");
        return PM2D_EINVAL;
    }
    StaticModes M;
    int rc = static_scratch(&M.rows);
    if (rc) return rc;
    M.n = n_dev; M.out = out_dev;
    M.nx = nx; M.ny = ny; M.nmodes = nmodes;
    for (int m = 0; m < PM2D_MAX_MODES; m++) {
        M.mx[m] = m < nmodes ? mx[m] : 0;
        M.my[m] = m < nmodes ? my[m] : 0;
    }
    // every scratch entry the second kernel reads is written by the first one of the same call: nothing has to start at zero
    cudaStream_t st = (cudaStream_t)stream;
    k_modes_rows<<<nx + 1, SM_THREADS, 0, st>>>(M);
    k_modes_cols<<<nmodes, SM_THREADS, 0, st>>>(M);
    PM2D_CUDA_CHECK(cudaGetLastError());
    return PM2D_OK;
}
