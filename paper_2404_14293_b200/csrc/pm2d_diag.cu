// pm2d_diag.cu -- energy / charge diagnostics as block reductions (Q11):
//   W = sum_s sum_p (1/2) m_s w_p |u_p|^2 + 2 pi^2 sum |E|^2 + (1/2) sum n_e |a|^2
//       + (1/8 pi^2) sum (|d_t a|^2 + |grad a|^2) + sum_s m_s C_s v_s^2 sum n_s ln n_s
// float32 inputs, float64 accumulation, one atomicAdd(double) per CTA and quantity.
#include "pm2d_internal.h"

namespace {

__device__ __forceinline__ void block_add(double v, double *dst)
{
    __shared__ double ws[32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __syncthreads();
    if (lane == 0) ws[wid] = v;
    __syncthreads();
    if (wid == 0) {
        v = lane < (blockDim.x + 31) / 32 ? ws[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0 && v != 0.0) atomicAdd(dst, v);
    }
}

struct GridDiag {
    const float *phi, *a_now, *a_old;
    const int32_t *ne[PM2D_MAX_SPECIES];
    int ne_count;
    int nx, ny, ncomp;
    float inv_nscale, inv_dx, inv_dy, inv_dt;
    double *red;
};

// one thread per node: cell (i, j) terms for i < nx, node terms for all i
__global__ void __launch_bounds__(256) k_diag_grid(const GridDiag D)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
    double es = 0.0, wint = 0.0, em = 0.0;
    if (j < D.ny) {
        const size_t nn = (size_t)(D.nx + 1) * D.ny;
        const int jp = (j + 1) & (D.ny - 1);
        const size_t k = (size_t)i * D.ny + j, ku = (size_t)i * D.ny + jp;
        const double vol = (i == 0 || i == D.nx) ? 0.5 : 1.0;
        if (i < D.nx) {
            float p00 = D.phi[k], p01 = D.phi[ku], p10 = D.phi[k + D.ny], p11 = D.phi[ku + D.ny];
            float ex = -0.5f * ((p11 - p01) + (p10 - p00)) * D.inv_dx;
            float ey = -0.5f * ((p11 - p10) + (p01 - p00)) * D.inv_dy;
            es = (double)ex * ex + (double)ey * ey;
        }
        int nv = 0;
        for (int s = 0; s < D.ne_count; s++) nv += D.ne[s][k];
        double a2 = 0.0;
        for (int c = 0; c < D.ncomp; c++) {
            float a = D.a_now[c * nn + k];
            float at = (a - D.a_old[c * nn + k]) * D.inv_dt;
            float ay = (D.a_now[c * nn + ku] - a) * D.inv_dy;
            a2 += (double)a * a;
            em += vol * ((double)at * at + (double)ay * ay);
            if (i < D.nx) {
                float ax = (D.a_now[c * nn + k + D.ny] - a) * D.inv_dx;
                em += (double)ax * ax;
            }
        }
        wint = 0.5 * vol * (double)nv * D.inv_nscale * a2;
    }
    block_add(es, &D.red[0]);
    block_add(wint, &D.red[1]);
    block_add(em, &D.red[2]);
}

__global__ void __launch_bounds__(256) k_diag_species_grid(const int32_t *nfix, int nx, int ny, float inv_nscale, double *red_th,
                                                           double *red_charge)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x, i = blockIdx.y;
    double th = 0.0, q = 0.0;
    if (j < ny) {
        const double vol = (i == 0 || i == nx) ? 0.5 : 1.0;
        double n = (double)nfix[(size_t)i * ny + j] * inv_nscale;
        q = vol * n;
        if (n > 0.0) th = vol * n * log(n);
    }
    block_add(th, red_th);
    block_add(q, red_charge);
}

__global__ void __launch_bounds__(256) k_diag_kinetic(const PV *pv, const float *w, int64_t np, double *red)
{
    double s = 0.0;
    for (int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; p < np; p += (int64_t)gridDim.x * blockDim.x) {
        const PV me = pv[p];
        s += (double)w[p] * ((double)me.ux * me.ux + (double)me.uy * me.uy);
    }
    block_add(s, red);
}

// a8: Fourier-mode amplitudes of a nodal density.  Grid-stride over the nodes, every thread keeps the running sums
// of all modes in double; the phase m_x i / nx + m_y j / ny is reduced mod 1 in integers before sincospi.
struct ModeParams {
    const int32_t *nfix;
    int nx, ny, nmodes;
    int mx[PM2D_MAX_MODES], my[PM2D_MAX_MODES];
    double inv_nscale;
    double *red;          // [2 * nmodes]: re, im interleaved
};

__global__ void __launch_bounds__(256) k_diag_modes(const ModeParams M)
{
    double re[PM2D_MAX_MODES], im[PM2D_MAX_MODES];
#pragma unroll
    for (int m = 0; m < PM2D_MAX_MODES; m++) re[m] = im[m] = 0.0;
    const int64_t nn = (int64_t)(M.nx + 1) * M.ny;
    const double inv_nx = 1.0 / M.nx, inv_ny = 1.0 / M.ny;
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < nn; k += (int64_t)gridDim.x * blockDim.x) {
        const int i = (int)(k / M.ny), j = (int)(k - (int64_t)i * M.ny);
        const int v = M.nfix[k];
        if (v == 0) continue;
        const double n = ((i == 0 || i == M.nx) ? 0.5 : 1.0) * (double)v * M.inv_nscale;
#pragma unroll
        for (int m = 0; m < PM2D_MAX_MODES; m++) {
            if (m >= M.nmodes) break;
            const int64_t px = ((int64_t)M.mx[m] * i) % M.nx, py = ((int64_t)M.my[m] * j) % M.ny;
            double sn, cs;
            sincospi(-2.0 * ((double)px * inv_nx + (double)py * inv_ny), &sn, &cs);
            re[m] += n * cs;
            im[m] += n * sn;
        }
    }
#pragma unroll
    for (int m = 0; m < PM2D_MAX_MODES; m++) {
        if (m >= M.nmodes) break;
        block_add(re[m], &M.red[2 * m]);
        block_add(im[m], &M.red[2 * m + 1]);
    }
}

// 8f.4: weighted velocity histogram of the particles of a sub-box; one CTA per chunk of a tile's particle list
struct HistParams {
    const PV *pv;
    const float *w;
    const int32_t *chunk_tile, *nchunks, *ptile;
    const int64_t *chunk_beg, *tile_off;
    int nty, ny, i0, i1, j0, j1, comp, nbins;
    float umin, scale;
    double *hist;
};

__global__ void __launch_bounds__(PTHREADS) k_diag_vhist(const HistParams H)
{
    __shared__ double sh[PM2D_MAX_BINS];
    const int chunk = blockIdx.x;
    if (chunk >= *H.nchunks) return;
    for (int b = threadIdx.x; b < H.nbins; b += PTHREADS) sh[b] = 0.0;
    __syncthreads();
    const int ctile = H.chunk_tile[chunk];
    const int64_t beg = H.chunk_beg[chunk];
    int64_t end = beg + CHUNK;
    if (H.tile_off[ctile + 1] < end) end = H.tile_off[ctile + 1];
    for (int64_t p = beg + threadIdx.x; p < end; p += PTHREADS) {
        const int tile = H.ptile ? H.ptile[p] : ctile;
        const PV me = H.pv[p];
        const int ix = (tile / H.nty) * TILE + (int)(me.x >> POS_FRAC_BITS) - POS_BIAS;
        const int iy = ((tile % H.nty) * TILE + (int)(me.y >> POS_FRAC_BITS) - POS_BIAS) & (H.ny - 1);
        if (ix < H.i0 || ix >= H.i1 || iy < H.j0 || iy >= H.j1) continue;
        const float u = H.comp ? me.uy : me.ux;
        const float t = floorf(__fmul_rn(__fsub_rn(u, H.umin), H.scale));
        if (!(t >= 0.f) || !(t < (float)H.nbins)) continue;
        atomicAdd(&sh[(int)t], (double)H.w[p]);
    }
    __syncthreads();
    for (int b = threadIdx.x; b < H.nbins; b += PTHREADS)
        if (sh[b] != 0.0) atomicAdd(&H.hist[b], sh[b]);
}

// Frequency spectrum of the boundary records (pm2d_probe_spectrum): CTA = 128 columns x one omega.  The phase factors
// of 128 records at a time are computed once per CTA in double (one record per thread) and shared; every thread then
// walks those records of its own column (coalesced rows of the ring), accumulating A_j(w) in double.
struct SpecParams {
    const float *probe;      // ring base of (comp, wall): record q-1 at probe + slot * stride
    size_t stride;           // ncomp * 2 * ny
    int cap, first_slot, nrec;
    int j0, j1;
    double dts;
    double omega[PM2D_MAX_OMEGAS];
    double *red;             // [nomega]
};
__global__ void __launch_bounds__(128) k_probe_spectrum(const SpecParams S)
{
    __shared__ double2 tw[128];
    __shared__ double part[4];
    const int j = S.j0 + blockIdx.x * 128 + threadIdx.x;
    const double w2 = 2.0 * S.omega[blockIdx.y] * S.dts;
    double re = 0.0, im = 0.0;
    for (int m0 = 0; m0 < S.nrec; m0 += 128) {
        double sn, cs;
        sincospi(w2 * (double)(m0 + threadIdx.x), &sn, &cs);
        __syncthreads();
        tw[threadIdx.x] = make_double2(cs, -sn);
        __syncthreads();
        const int mend = min(128, S.nrec - m0);
        if (j < S.j1) {
            int slot = (S.first_slot + m0) % S.cap;
            for (int m = 0; m < mend; m++) {
                const double h = (double)S.probe[(size_t)slot * S.stride + j];
                re += h * tw[m].x;
                im += h * tw[m].y;
                if (++slot == S.cap) slot = 0;
            }
        }
    }
    double p = (j < S.j1) ? (re * re + im * im) * S.dts * S.dts : 0.0;
    for (int o = 16; o > 0; o >>= 1) p += __shfl_down_sync(0xffffffffu, p, o);
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = p;
    __syncthreads();
    if (threadIdx.x == 0) atomicAdd(&S.red[blockIdx.y], part[0] + part[1] + part[2] + part[3]);
}

}  // namespace

// the kept boundary records: n of them, the first one of particle step `first` (1-based), in ring slot `slot`
static int64_t probe_window(const pm2d_ctx *c, int64_t *first, int *slot)
{
    const int64_t R = c->g.probe_steps, n = c->step < R ? c->step : R;
    *first = c->step - n + 1;
    *slot = (int)((*first - 1) % R);
    return n;
}

extern "C" int64_t pm2d_get_probe(pm2d_ctx *c, int wall, int comp, float *host, size_t cap, int64_t *first_step)
{
    if (!c || wall < 0 || wall > 1 || comp < 0 || comp >= c->g.ncomp || !host) {
        pm2d_set_error("pm2d_get_probe: bad argument");
        return PM2D_EINVAL;
    }
    if (!c->probe) {
        pm2d_set_error("pm2d_get_probe: pm2d_grid.probe_steps is 0");
        return PM2D_ESTATE;
    }
    int64_t first;
    int slot;
    const int64_t n = probe_window(c, &first, &slot);
    const size_t ny = (size_t)c->g.ny, stride = (size_t)c->g.ncomp * 2 * ny;
    if ((size_t)n * ny > cap) {
        pm2d_set_error("pm2d_get_probe: host buffer too small");
        return PM2D_EINVAL;
    }
    if (first_step) *first_step = first;
    const float *base = c->probe + ((size_t)comp * 2 + wall) * ny;
    // two pieces of the ring: slots slot .. R-1, then 0 .. slot-1
    const int64_t n1 = n < c->g.probe_steps - slot ? n : c->g.probe_steps - slot;
    if (n1 > 0)
        PM2D_CUDA_CHECK(cudaMemcpy2DAsync(host, ny * sizeof(float), base + (size_t)slot * stride, stride * sizeof(float), ny * sizeof(float),
                                          (size_t)n1, cudaMemcpyDeviceToHost, c->stream));
    if (n > n1)
        PM2D_CUDA_CHECK(cudaMemcpy2DAsync(host + (size_t)n1 * ny, ny * sizeof(float), base, stride * sizeof(float), ny * sizeof(float),
                                          (size_t)(n - n1), cudaMemcpyDeviceToHost, c->stream));
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    return n;
}

extern "C" int64_t pm2d_probe_spectrum(pm2d_ctx *c, int wall, int comp, int j0, int j1, int nomega, const double *omega,
                                       double *power)
{
    if (!c || wall < 0 || wall > 1 || comp < 0 || comp >= c->g.ncomp || j0 < 0 || j1 > c->g.ny || j0 >= j1 || nomega < 1 ||
        nomega > PM2D_MAX_OMEGAS || !omega || !power) {
        pm2d_set_error("pm2d_probe_spectrum: bad argument");
        return PM2D_EINVAL;
    }
    if (!c->probe) {
        pm2d_set_error("pm2d_probe_spectrum: pm2d_grid.probe_steps is 0");
        return PM2D_ESTATE;
    }
    int64_t first;
    int slot;
    const int64_t n = probe_window(c, &first, &slot);
    for (int k = 0; k < nomega; k++) power[k] = 0.0;
    if (n == 0) return 0;
    SpecParams S;
    S.probe = c->probe + ((size_t)comp * 2 + wall) * c->g.ny;
    S.stride = (size_t)c->g.ncomp * 2 * c->g.ny;
    S.cap = c->g.probe_steps; S.first_slot = slot; S.nrec = (int)n;
    S.j0 = j0; S.j1 = j1;
    S.dts = c->dtp;
    for (int k = 0; k < PM2D_MAX_OMEGAS; k++) S.omega[k] = k < nomega ? omega[k] : 0.0;
    S.red = c->red;
    PM2D_CUDA_CHECK(cudaMemsetAsync(c->red, 0, 64 * sizeof(double), c->stream));
    k_probe_spectrum<<<dim3((j1 - j0 + 127) / 128, nomega), 128, 0, c->stream>>>(S);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    PM2D_CUDA_CHECK(cudaMemcpyAsync(power, c->red, (size_t)nomega * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    return n;
}

extern "C" int pm2d_velocity_histogram(pm2d_ctx *c, int species, int i0, int i1, int j0, int j1, int comp, double umin, double umax,
                                       int nbins, double *hist)
{
    if (!c || species < 0 || species >= c->nsp || !hist || nbins < 1 || nbins > PM2D_MAX_BINS || comp < 0 || comp > 1 ||
        !(umax > umin) || i0 < 0 || i1 > c->g.nx || i0 >= i1 || j0 < 0 || j1 > c->g.ny || j0 >= j1) {
        pm2d_set_error("pm2d_velocity_histogram: bad argument");
        return PM2D_EINVAL;
    }
    SpeciesDev &S = c->sp[species];
    for (int b = 0; b < nbins; b++) hist[b] = 0.0;
    if (!S.cfg.mobile || S.np == 0) return PM2D_OK;
    HistParams H;
    H.pv = S.pv; H.w = S.w; H.chunk_tile = S.chunk_tile; H.nchunks = S.nchunks_dev; H.ptile = S.random ? S.ptile : nullptr;
    H.chunk_beg = S.chunk_beg; H.tile_off = S.tile_off;
    H.nty = c->nty; H.ny = c->g.ny; H.i0 = i0; H.i1 = i1; H.j0 = j0; H.j1 = j1; H.comp = comp; H.nbins = nbins;
    H.umin = (float)umin;
    H.scale = (float)((double)nbins / (umax - umin));
    H.hist = c->hist;
    PM2D_CUDA_CHECK(cudaMemsetAsync(c->hist, 0, (size_t)nbins * sizeof(double), c->stream));
    k_diag_vhist<<<S.max_chunks, PTHREADS, 0, c->stream>>>(H);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    PM2D_CUDA_CHECK(cudaMemcpyAsync(hist, c->hist, (size_t)nbins * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    return PM2D_OK;
}

extern "C" int pm2d_mode_amplitudes(pm2d_ctx *c, int species, int nmodes, const int32_t *mx, const int32_t *my, double *re,
                                    double *im)
{
    if (!c || species < 0 || species >= c->nsp || nmodes < 1 || nmodes > PM2D_MAX_MODES || !mx || !my || !re || !im)
    {
        pm2d_set_error("pm2d_mode_amplitudes: bad argument (species, 1 <= nmodes <= PM2D_MAX_MODES, non-null arrays)");
        return PM2D_EINVAL;
    }
    ModeParams M;
    M.nfix = c->sp[species].nfix;
    M.nx = c->g.nx; M.ny = c->g.ny; M.nmodes = nmodes;
    for (int m = 0; m < PM2D_MAX_MODES; m++) {
        M.mx[m] = m < nmodes ? mx[m] : 0;
        M.my[m] = m < nmodes ? my[m] : 0;
    }
    M.inv_nscale = (double)c->inv_nscale;
    M.red = c->red;
    PM2D_CUDA_CHECK(cudaMemsetAsync(c->red, 0, 64 * sizeof(double), c->stream));
    k_diag_modes<<<592, 256, 0, c->stream>>>(M);
    count_launch(c);
    PM2D_CUDA_CHECK(cudaGetLastError());
    double h[2 * PM2D_MAX_MODES];
    PM2D_CUDA_CHECK(cudaMemcpyAsync(h, c->red, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    for (int m = 0; m < nmodes; m++) {
        re[m] = h[2 * m];
        im[m] = h[2 * m + 1];
    }
    return PM2D_OK;
}

// expects c->phi to hold phi of the current densities (caller ran launch_poisson(c, true))
int launch_diagnostics(pm2d_ctx *c, pm2d_diag *out)
{
    const double PI = 3.14159265358979323846;
    PM2D_CUDA_CHECK(cudaMemsetAsync(c->red, 0, 64 * sizeof(double), c->stream));
    GridDiag D;
    D.phi = c->phi; D.a_now = c->a[1]; D.a_old = c->a[2];
    D.ne_count = 0;
    for (int s = 0; s < c->nsp; s++)
        if (c->sp[s].cfg.sign < 0) D.ne[D.ne_count++] = c->sp[s].nfix;
    D.nx = c->g.nx; D.ny = c->g.ny; D.ncomp = c->g.ncomp;
    D.inv_nscale = c->inv_nscale; D.inv_dx = (float)(1.0 / c->g.dx); D.inv_dy = (float)(1.0 / c->g.dy);
    D.inv_dt = (float)(1.0 / c->g.dt);
    D.red = c->red;
    dim3 grid((c->g.ny + 255) / 256, c->g.nx + 1);
    k_diag_grid<<<grid, 256, 0, c->stream>>>(D);
    count_launch(c);
    for (int s = 0; s < c->nsp; s++) {
        SpeciesDev &S = c->sp[s];
        k_diag_species_grid<<<grid, 256, 0, c->stream>>>(S.nfix, c->g.nx, c->g.ny, c->inv_nscale, c->red + 4 + 3 * s, c->red + 5 + 3 * s);
        count_launch(c);
        if (S.cfg.mobile && S.np > 0) {
            k_diag_kinetic<<<592, 256, 0, c->stream>>>(S.pv, S.w, S.np, c->red + 3 + 3 * s);
            count_launch(c);
        }
    }
    PM2D_CUDA_CHECK(cudaGetLastError());
    double h[64];
    PM2D_CUDA_CHECK(cudaMemcpyAsync(h, c->red, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    out->step = c->step;
    out->time = c->step * c->dtp;
    out->W_es = 2.0 * PI * PI * h[0];
    out->W_int = h[1];
    out->W_em = h[2] / (8.0 * PI * PI);
    out->W_total = out->W_es + out->W_int + out->W_em;
    for (int s = 0; s < PM2D_MAX_SPECIES; s++) {
        out->W_kin[s] = out->W_th[s] = out->charge[s] = 0.0;
        out->count[s] = 0;
    }
    for (int s = 0; s < c->nsp; s++) {
        SpeciesDev &S = c->sp[s];
        out->W_kin[s] = 0.5 * S.cfg.mass * h[3 + 3 * s];
        out->W_th[s] = S.cfg.mass * S.cfg.pressure_coeff * S.vth2 * h[4 + 3 * s];
        out->charge[s] = h[5 + 3 * s];
        out->count[s] = S.np;
        out->W_total += out->W_kin[s] + out->W_th[s];
    }
    return PM2D_OK;
}
