// pm2d_api.cu -- the C ABI of include/pm2d.h: argument checks, workspace carving, the host step
// scheduler and the host<->device accessors.  No arithmetic of the method lives here
// except the laser carrier phases handed to the boundary kernel (pm2d_fields.cu).
#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>

#include "pm2d_internal.h"

static thread_local std::string g_err;
void pm2d_set_error(const std::string &s) { g_err = s; }
extern "C" const char *pm2d_last_error(void) { return g_err.c_str(); }
#ifndef PM2D_BUILD_ID
#define PM2D_BUILD_ID "unknown"
#endif
extern "C" const char *pm2d_version(void) { return "pm2d-b200 0.2 (sm_100a, build " PM2D_BUILD_ID ")"; }

extern "C" int pm2d_struct_size(int which)
{
    switch (which) {
    case 0: return (int)sizeof(pm2d_grid);
    case 1: return (int)sizeof(pm2d_species);
    case 2: return (int)sizeof(pm2d_profile);
    case 3: return (int)sizeof(pm2d_laser);
    case 4: return (int)sizeof(pm2d_diag);
    default: return -1;
    }
}

static int fail(int code, const std::string &msg)
{
    g_err = msg;
    return code;
}

static void destroy_ctx(pm2d_ctx *c);

namespace {

__global__ void k_extract_comp(const float2 *src, int comp, float *dst, size_t n)
{
    size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) dst[k] = comp == 0 ? src[k].x : src[k].y;
}

struct Carver {
    char *base;
    size_t off;
    template <class T>
    T *take(size_t count)
    {
        off = (off + 255) & ~(size_t)255;
        T *p = base ? reinterpret_cast<T *>(base + off) : nullptr;
        off += count * sizeof(T);
        return p;
    }
};

bool is_pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

int64_t species_np(const pm2d_grid &g, const pm2d_species &s)
{
    if (!s.mobile) return 0;
    if (s.load == PM2D_LOAD_NONE || s.load == PM2D_NUMBER_WEIGHTED) return s.capacity;
    return (int64_t)g.nx * g.ny * s.ppc_x * s.ppc_y;
}

// Eq. 5 on a y-periodic box (Q22): a plane wave must come back to itself after Ly
int validate_laser_angle(const pm2d_laser &L, double Ly)
{
    if (!(std::fabs(L.alpha) <= 1.0)) return fail(PM2D_EINVAL, "laser alpha must be within [-1, 1] rad");
    if (L.alpha != 0.0 && !(L.w0 > 0.0)) {
        const double m = L.omega * std::sin(L.alpha) * Ly;
        if (std::fabs(m - std::nearbyint(m)) > 1e-6) return fail(PM2D_EINVAL, "oblique plane wave: omega*sin(alpha)*Ly must be an integer (y is periodic)");
    }
    return PM2D_OK;
}

int validate(const pm2d_grid *g, const pm2d_species *sp, int nsp)
{
    if (!g || !sp) return fail(PM2D_EINVAL, "null argument");
    if (nsp < 1 || nsp > PM2D_MAX_SPECIES) return fail(PM2D_EINVAL, "nsp out of range");
    if (g->nx < 8 || g->nx > 32767) return fail(PM2D_EINVAL, "nx must be in [8, 32767]");
    if (!is_pow2(g->ny) || g->ny < 8 || g->ny > 8192) return fail(PM2D_EINVAL, "ny must be a power of two in [8, 8192]");
    if (g->ncomp < 1 || g->ncomp > 3) return fail(PM2D_EINVAL, "ncomp must be 1..3");
    if (g->rebin_every < 0 || g->rebin_every > 32) return fail(PM2D_EINVAL, "rebin_every must be 0..32");
    if (g->particle_order < PM2D_ORDER_AUTO || g->particle_order > PM2D_ORDER_LANES) return fail(PM2D_EINVAL, "unknown particle_order");
    if (!(g->dx > 0) || !(g->dy > 0) || !(g->dt > 0)) return fail(PM2D_EINVAL, "dx, dy, dt must be positive");
    if (g->dt / g->dx > 0.999 || g->dt / g->dy > 0.999)
        return fail(PM2D_EINVAL, "dt/dx must be < 1: a particle may not cross more than one cell per step");
    if (g->subcycle < 0 || g->subcycle > 16) return fail(PM2D_EINVAL, "subcycle must be 0..16");
    if (g->subcycle > 1 && (g->subcycle * g->dt / g->dx > 4.0 || g->subcycle * g->dt / g->dy > 4.0))
        return fail(PM2D_EINVAL, "subcycle*dt/dx must be <= 4");
    if (g->bc_y != PM2D_BC_Y_PERIODIC && g->bc_y != PM2D_BC_Y_ABSORB) return fail(PM2D_EINVAL, "unknown bc_y");
    if (g->probe_steps < 0 || g->probe_steps > 65536) return fail(PM2D_EINVAL, "probe_steps must be 0..65536");
    for (int s = 0; s < nsp; s++) {
        const pm2d_species &q = sp[s];
        if (!(q.mass > 0)) return fail(PM2D_EINVAL, "species mass must be positive");
        if (q.sign < -1 || q.sign > 1) return fail(PM2D_EINVAL, "species sign must be -1, 0, +1");
        if (q.shape == PM2D_CIC) { if (q.DD != 1.0) return fail(PM2D_EINVAL, "CIC needs DD = 1"); }
        else if (q.shape == PM2D_TSC) { if (q.DD != 2.0) return fail(PM2D_EINVAL, "TSC needs DD = 2"); }
        else if (q.shape == PM2D_SINE) { if (!(q.DD > 0.0) || q.DD > 2.0) return fail(PM2D_EINVAL, "SINE needs 0 < DD <= 2 (3-node footprint)"); }
        else return fail(PM2D_EINVAL, "unknown shape");
        if (q.load < PM2D_LOAD_NONE || q.load > PM2D_NUMBER_WEIGHTED) return fail(PM2D_EINVAL, "unknown load");
        if (q.load != PM2D_LOAD_NONE && (q.ppc_x < 1 || q.ppc_y < 1)) return fail(PM2D_EINVAL, "ppc_x, ppc_y must be >= 1");
        if (q.load != PM2D_LOAD_NONE && !q.mobile) return fail(PM2D_EINVAL, "an immobile species is a fixed background: load must be NONE");
        if (species_np(*g, q) < 0 || species_np(*g, q) > ((int64_t)1 << 31) - 1) return fail(PM2D_EINVAL, "particle count out of range");
    }
    return PM2D_OK;
}

// carve (or, with base == nullptr, just size) every device array
size_t layout(pm2d_ctx *c, char *base)
{
    Carver cv{base, 0};
    const pm2d_grid &g = c->g;
    const size_t nn = (size_t)(g.nx + 1) * g.ny;
    const int ntx = (g.nx + TILE - 1) / TILE, nty = (g.ny + TILE - 1) / TILE, ntiles = ntx * nty;
    const int LP = g.ny / 2 + 2;
    c->nn = (int64_t)nn; c->ntx = ntx; c->nty = nty; c->ntiles = ntiles; c->LP = LP;
    const size_t ns = (size_t)(g.nx + 1) * LP;
    for (int k = 0; k < 3; k++) c->a[k] = cv.take<float>(g.ncomp * nn);
    c->rho_hat = cv.take<float2>(ns);
    {
        const size_t P = (size_t)(g.nx + TRI_M - 1) / TRI_M;
        c->tri_cp = cv.take<double>((size_t)2 * TRI_M * LP);
        c->tri_V = cv.take<double>((size_t)2 * TRI_M * LP);
        c->tri_W = cv.take<double>((size_t)2 * TRI_M * LP);
        c->tri_den = cv.take<double>(P * LP);
        c->tri_sumV = cv.take<double2>(P * LP);
        c->tri_sumW = cv.take<double2>(P * LP);
        c->tri_g = cv.take<double2>((P + 1) * LP);
    }
    c->ehx = cv.take<float2>(ns);
    c->ehy = cv.take<float2>(ns);
    c->Enode = cv.take<float2>(nn);
    c->phi = cv.take<float>(nn);
    c->twiddle = cv.take<float2>(g.ny / 2);
    c->red = cv.take<double>(64);
    c->hist = cv.take<double>(PM2D_MAX_BINS);
    c->probe = g.probe_steps > 0 ? cv.take<float>((size_t)g.probe_steps * g.ncomp * 2 * g.ny) : nullptr;
    c->flags = cv.take<int32_t>(4);
    c->shape_y = cv.take<double>(g.ny);
    c->taper_x = cv.take<double>(g.nx);
    c->stray_total = cv.take<unsigned long long>(1);
    c->zeros = cv.take<int32_t>(PM2D_ZEROS_BYTES / 4);
    {   // overflow list of the stage kernels: a quarter of the largest species, at least 2^20 entries
        int64_t most = 0;
        for (int s = 0; s < c->nsp; s++) most = std::max<int64_t>(most, species_np(g, c->sp[s].cfg));
        c->ovf_cap = (int)std::min<int64_t>(std::max<int64_t>((int64_t)1 << 20, most / 4), (int64_t)1 << 30);
    }
    c->ovf_p = cv.take<int64_t>(c->ovf_cap);
    c->ovf_tile = cv.take<int32_t>(c->ovf_cap);
    c->ovf_count = cv.take<int32_t>(4);
    for (int s = 0; s < c->nsp; s++) {
        SpeciesDev &S = c->sp[s];
        S.nfix = cv.take<int32_t>(nn);
        S.pxfix = S.pyfix = nullptr; S.F = nullptr;
        S.np = S.cap = species_np(g, S.cfg);
        S.layered = false;
        S.lanes = false;
        S.lane_subs = 1;
        S.lane_copies = 2;
        S.sub0 = nullptr;
        S.lane_exp = nullptr;
        S.random = false;
        S.ptile = nullptr;
        if (!S.cfg.mobile) continue;
        S.random = g.particle_order == PM2D_ORDER_RANDOM;
        // AUTO, up to 16 particles per cell on average: the lane order + k_stage_lanes, except for species that drift a cell
        // or more per rebin period AND hold fewer than 3 particles per cell -- there the half-tile windows of the
        // four-copy variant serve too few particles each and the layered order + k_stage_direct wins (cbet electrons,
        // 1 per cell: stage kernels 5.5 against 6.5 ms, rebin 1.2 against 2.1 ms per step, r02j).  The number-weighted
        // loader follows a profile in y (the lanes assume a population that is uniform in y) and fills cell runs: cell-major.
        // thermal drift over a rebin period, in cells: below a tenth of a cell two window copies on whole tiles do
        const double drift = std::sqrt(S.cfg.T_keV / 511.0 / S.cfg.mass) * (g.subcycle > 1 ? g.subcycle : 1) * g.dt / std::min(g.dx, g.dy) *
                             (double)(g.rebin_every > 0 ? g.rebin_every : 32);
        if (S.cfg.load != PM2D_NUMBER_WEIGHTED) {
            const bool sparse = g.particle_order == PM2D_ORDER_AUTO && S.cap <= (int64_t)PM2D_LAYERS * g.nx * g.ny;
            const bool thin_hot = drift >= 0.1 && S.cap < (int64_t)3 * g.nx * g.ny;
            S.lanes = g.particle_order == PM2D_ORDER_LANES || (sparse && !thin_hot);
            S.layered = g.particle_order == PM2D_ORDER_LAYERED || (sparse && thin_hot);
        }
        if (S.lanes) {
            S.lane_copies = drift < 0.1 ? 2 : 4;
            S.lane_subs = S.lane_copies == 4 ? 2 : 1;
            S.sub0 = cv.take<int32_t>(ntiles);
            S.lane_exp = cv.take<int32_t>(ntiles);
        }
        S.pxfix = cv.take<int32_t>(nn);
        S.pyfix = cv.take<int32_t>(nn);
        S.nhat = cv.take<int32_t>(nn);
        S.pxhat = cv.take<int32_t>(nn);
        S.pyhat = cv.take<int32_t>(nn);
        S.F = cv.take<float2>(nn);
        const size_t cap = (size_t)std::max<int64_t>(S.cap, 1);
        S.pv = cv.take<PV>(cap); S.pv2 = cv.take<PV>(cap);
        S.uh = cv.take<float2>(cap);
        S.w = cv.take<float>(cap); S.w2 = cv.take<float>(cap);
        S.cell_off = cv.take<int32_t>((size_t)ntiles * CPITCH);
        if (S.random) S.ptile = cv.take<int32_t>(cap);
        S.id = S.id2 = nullptr;
        if (g.track_ids) { S.id = cv.take<int64_t>(cap); S.id2 = cv.take<int64_t>(cap); }
        S.max_chunks = ntiles + (int32_t)(cap / CHUNK) + 1;
        S.tile_off = cv.take<int64_t>(ntiles + 1);
        S.tile_off2 = cv.take<int64_t>(ntiles + 1);
        S.chunk_tile = cv.take<int32_t>(S.max_chunks);
        S.chunk_beg = cv.take<int64_t>(S.max_chunks + 1);
        S.chunk_cnt9 = cv.take<int32_t>((size_t)S.max_chunks * 9);
        S.chunk_rel9 = cv.take<int64_t>((size_t)S.max_chunks * 9);
        S.tile_first_chunk = cv.take<int32_t>(ntiles + 1);
        S.tile_cnt = cv.take<int32_t>(ntiles);
        S.nchunks_dev = cv.take<int32_t>(4);
    }
    return (cv.off + 255) & ~(size_t)255;
}

void phase_begin(pm2d_ctx *c, int ph)
{
    c->cur_phase = ph;
    if (!c->prof_on) return;
    cudaEvent_t e;
    cudaEventCreate(&e);
    cudaEventRecord(e, c->stream);
    c->ev.push_back(e);
    c->ev_phase.push_back(ph);
}
void phase_end(pm2d_ctx *c)
{
    if (c->prof_on) {
        cudaEvent_t e;
        cudaEventCreate(&e);
        cudaEventRecord(e, c->stream);
        c->ev.push_back(e);
        c->ev_phase.push_back(-1);
    }
    c->cur_phase = -1;
}

int check_flags(pm2d_ctx *c)
{
    int32_t h[4];
    PM2D_CUDA_CHECK(cudaMemcpyAsync(h, c->flags, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    if (h[0]) return fail(PM2D_ESTATE, "a particle moved further than one tile between rebins (rebin_every too large)");
    if (h[1]) return fail(PM2D_ESTATE, "chunk table overflow");
    if (h[2]) return fail(PM2D_ESTATE, "too many particles outside their tile window (rebin_every too large)");
    if (h[3] == 2) return fail(PM2D_ESTATE, "a deposit exceeds the fixed-point range of the grids (density above 4 n_max of the profile, or |n u| above n_max / 2)");
    if (h[3]) return fail(PM2D_ESTATE, "lane order: a tile holds more than 65535 particles (use PM2D_ORDER_CELL_MAJOR)");
    return PM2D_OK;
}

int zero_moments(pm2d_ctx *c, int s, bool density, bool momentum)
{
    SpeciesDev &S = c->sp[s];
    const size_t bytes = (size_t)c->nn * sizeof(int32_t);
    if (density) PM2D_CUDA_CHECK(cudaMemsetAsync(S.nfix, 0, bytes, c->stream));
    if (momentum) {
        PM2D_CUDA_CHECK(cudaMemsetAsync(S.pxfix, 0, bytes, c->stream));
        PM2D_CUDA_CHECK(cudaMemsetAsync(S.pyfix, 0, bytes, c->stream));
    }
    return PM2D_OK;
}

// The deposit set `which` (0: n, Px, Py of stage B; 1: those of stage A) has had its last reader enqueued on
// the main stream: zero it on the side stream, concurrently with whatever the main stream does next.
int zero_set_async(pm2d_ctx *c, int which)
{
    PM2D_CUDA_CHECK(cudaEventRecord(c->ev_free[which], c->stream));
    PM2D_CUDA_CHECK(cudaStreamWaitEvent(c->zstream, c->ev_free[which], 0));
    const size_t bytes = (size_t)c->nn * sizeof(int32_t);
    for (int s = 0; s < c->nsp; s++) {
        SpeciesDev &S = c->sp[s];
        if (!S.cfg.mobile || S.np == 0) continue;
        PM2D_CUDA_CHECK(cudaMemsetAsync(which ? S.nhat : S.nfix, 0, bytes, c->zstream));
        if (c->g.eager_moments) {
            PM2D_CUDA_CHECK(cudaMemsetAsync(which ? S.pxhat : S.pxfix, 0, bytes, c->zstream));
            PM2D_CUDA_CHECK(cudaMemsetAsync(which ? S.pyhat : S.pyfix, 0, bytes, c->zstream));
        }
    }
    PM2D_CUDA_CHECK(cudaEventRecord(c->ev_zero[which], c->zstream));
    return PM2D_OK;
}

// deposit every moment of species s from its current particles (item (1) of the flow)
int redeposit(pm2d_ctx *c, int s)
{
    int rc = zero_moments(c, s, true, true);
    if (rc) return rc;
    return launch_deposit_only(c, s, true, c->g.eager_moments != 0);
}

int refix_backgrounds(pm2d_ctx *c)
{
    for (int s = 0; s < c->nsp; s++)
        if (!c->sp[s].cfg.mobile) {
            int rc = launch_fix_background(c, s);
            if (rc) return rc;
        }
    return PM2D_OK;
}

}  // namespace

extern "C" size_t pm2d_query_workspace(const pm2d_grid *grid, const pm2d_species *species, int nsp)
{
    if (validate(grid, species, nsp) != PM2D_OK) return 0;
    pm2d_ctx *c = new (std::nothrow) pm2d_ctx();
    if (!c) return 0;
    c->g = *grid;
    c->nsub = grid->subcycle > 1 ? grid->subcycle : 1;
    c->dtp = c->nsub * grid->dt;
    c->nsp = nsp;
    for (int s = 0; s < nsp; s++) c->sp[s].cfg = species[s];
    size_t bytes = layout(c, nullptr);
    delete c;
    return bytes;
}

extern "C" int pm2d_init(const pm2d_grid *grid, const pm2d_species *species, int nsp, const pm2d_profile *profile,
                         const pm2d_laser *lasers, int nlaser, uint64_t seed, void *dev_workspace, size_t bytes,
                         void *cuda_stream, pm2d_ctx **out)
{
    if (!out) return fail(PM2D_EINVAL, "null out");
    *out = nullptr;
    int rc = validate(grid, species, nsp);
    if (rc) return rc;
    if (!profile) return fail(PM2D_EINVAL, "null profile");
    if (nlaser < 0 || nlaser > PM2D_MAX_LASERS || (nlaser > 0 && !lasers)) return fail(PM2D_EINVAL, "bad laser table");
    for (int l = 0; l < nlaser; l++)
    {
        if (lasers[l].comp < 0 || lasers[l].comp >= grid->ncomp) return fail(PM2D_EINVAL, "laser component out of range");
        if ((rc = validate_laser_angle(lasers[l], grid->ny * grid->dy))) return rc;
    }
    if (profile->kind < PM2D_PROFILE_UNIFORM || profile->kind > PM2D_PROFILE_FILAMENT_Y) return fail(PM2D_EINVAL, "unknown profile");
    if (profile->taper_cells_y < 0 || profile->taper_cells_y > grid->ny / 2) return fail(PM2D_EINVAL, "taper_cells_y must be in [0, ny/2]");
    if (profile->taper_cells_y > 0)
        for (int s = 0; s < nsp; s++)
            if (species[s].load == PM2D_NUMBER_WEIGHTED) return fail(PM2D_EINVAL, "taper_cells_y is not available with PM2D_NUMBER_WEIGHTED");
    if (profile->slab[0] | profile->slab[1] | profile->slab[2] | profile->slab[3]) {
        const int32_t *b = profile->slab;
        if (b[0] < 0 || b[0] >= b[1] || b[1] > grid->nx || b[2] < 0 || b[2] >= b[3] || b[3] > grid->ny)
            return fail(PM2D_EINVAL, "profile slab must satisfy 0 <= x_lo < x_hi <= nx and 0 <= y_lo < y_hi <= ny");
        for (int s = 0; s < nsp; s++)
            if (species[s].load == PM2D_NUMBER_WEIGHTED) return fail(PM2D_EINVAL, "a slab extent is not available with PM2D_NUMBER_WEIGHTED");
    }
    double nmax;
    if (profile->kind == PM2D_PROFILE_UNIFORM) nmax = profile->p[0];
    else if (profile->kind == PM2D_PROFILE_LINEAR) nmax = std::max(profile->p[0], profile->p[1]);
    else if (profile->kind == PM2D_PROFILE_FILAMENT_Y) {
        if (!(profile->p[2] > 0.0) || !(profile->p[1] >= 0.0)) return fail(PM2D_EINVAL, "filament needs sigma > 0, A >= 0");
        nmax = profile->p[0] * (1.0 + profile->p[1]);
    } else nmax = std::min(profile->p[0] * std::exp(std::max(profile->p[1], 0.0)), profile->p[2]);
    if (!(nmax >= 0.0) || nmax > 1e3) return fail(PM2D_EINVAL, "profile density out of range");
    // discrete stability of Eq. 6 with the plasma term (P:L120 and its bound with n_e)
    {
        const double PI = 3.14159265358979323846;
        double s2 = grid->dt * grid->dt * (1.0 / (grid->dx * grid->dx) + 1.0 / (grid->dy * grid->dy) + PI * PI * nmax);
        if (s2 > 1.0) return fail(PM2D_EINVAL, "dt violates the stability bound dt*sqrt(1/dx^2+1/dy^2+pi^2 n_max) <= 1 (P:L120)");
    }
    if (!dev_workspace) return fail(PM2D_EINVAL, "null workspace");
    if (((uintptr_t)dev_workspace & 255) != 0) return fail(PM2D_EINVAL, "workspace must be 256-byte aligned");
    pm2d_ctx *c = new (std::nothrow) pm2d_ctx();
    if (!c) return fail(PM2D_ENOMEM, "host allocation failed");
    c->g = *grid;
    c->nsub = grid->subcycle > 1 ? grid->subcycle : 1;
    c->dtp = c->nsub * grid->dt;
    c->nsp = nsp;
    c->nlaser = nlaser;
    for (int s = 0; s < nsp; s++) {
        c->sp[s].cfg = species[s];
        c->sp[s].vth2 = species[s].T_keV / 511.0 / species[s].mass;
    }
    for (int l = 0; l < nlaser; l++) c->laser[l] = lasers[l];
    c->profile = *profile;
    c->seed = seed;
    c->stream = (cudaStream_t)cuda_stream;
    c->zstream = nullptr;
    for (int k = 0; k < 2; k++) c->ev_free[k] = c->ev_zero[k] = nullptr;
    c->step = 0;
    c->uh_valid = false;
    c->cap_extra = 0;
    c->prof_on = false;
    c->cur_phase = -1;
    c->launches = 0;
    c->prof_steps = 0;
    for (int p = 0; p < PM2D_PH_COUNT; p++) { c->prof_ms[p] = 0; c->prof_launch[p] = 0; }
    const size_t need = layout(c, (char *)dev_workspace);
    if (need > bytes) {
        destroy_ctx(c);
        return fail(PM2D_ENOMEM, "workspace too small");
    }
#define INIT_CHECK(call)           \
    do {                           \
        int rc_ = (call);          \
        if (rc_) {                 \
            destroy_ctx(c);              \
            return rc_;            \
        }                          \
    } while (0)
#define INIT_CUDA(call)                                                          \
    do {                                                                         \
        cudaError_t e_ = (call);                                                 \
        if (e_ != cudaSuccess) {                                                 \
            destroy_ctx(c);                                                            \
            return fail(PM2D_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
        }                                                                        \
    } while (0)
    INIT_CUDA(cudaMemsetAsync(dev_workspace, 0, need, c->stream));
    INIT_CUDA(cudaStreamCreateWithFlags(&c->zstream, cudaStreamNonBlocking));
    for (int k = 0; k < 2; k++) {
        INIT_CUDA(cudaEventCreateWithFlags(&c->ev_free[k], cudaEventDisableTiming));
        INIT_CUDA(cudaEventCreateWithFlags(&c->ev_zero[k], cudaEventDisableTiming));
        INIT_CUDA(cudaEventRecord(c->ev_zero[k], c->stream));     // both deposit sets start zeroed
    }
    INIT_CHECK(launch_poisson_init(c));
    {   // relative density of the cell columns (filament) and the x taper, for the number-weighted loader
        std::vector<double> sy(grid->ny, 1.0), tx(grid->nx, 1.0);
        const double PI = 3.14159265358979323846;
        if (profile->kind == PM2D_PROFILE_FILAMENT_Y) {
            double sum = 0.0;
            for (int j = 0; j < grid->ny; j++) {
                const double r = ((double)j + 0.5 - 0.5 * grid->ny) / profile->p[2];
                sy[j] = 1.0 + profile->p[1] * std::exp(-0.5 * r * r);
                sum += sy[j];
            }
            for (int j = 0; j < grid->ny; j++) sy[j] /= sum / grid->ny;
        }
        if (profile->taper_cells > 0)
            for (int i = 0; i < grid->nx; i++) {
                const double d = std::min((double)i + 0.5, (double)grid->nx - 0.5 - (double)i);
                if (d < (double)profile->taper_cells) {
                    const double sn = std::sin(0.5 * PI * d / (double)profile->taper_cells);
                    tx[i] = PM2D_TAPER_FLOOR + (1.0 - PM2D_TAPER_FLOOR) * (sn * sn);
                }
            }
        if (profile->kind == PM2D_PROFILE_FILAMENT_Y) nmax = profile->p[0] * *std::max_element(sy.begin(), sy.end());
        INIT_CUDA(cudaMemcpyAsync(c->shape_y, sy.data(), sy.size() * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        INIT_CUDA(cudaMemcpyAsync(c->taper_x, tx.data(), tx.size() * sizeof(double), cudaMemcpyHostToDevice, c->stream));
        INIT_CUDA(cudaStreamSynchronize(c->stream));
    }
    // fixed-point scale: n_cap = power of two >= 8 n_max
    {
        double cap = 8.0 * (nmax > 0.0 ? nmax : 1.0);
        int e = (int)std::ceil(std::log2(cap));
        double ncap = std::ldexp(1.0, e);
        c->nscale = (float)(2147483648.0 / ncap);
        c->inv_nscale = (float)(ncap / 2147483648.0);
        c->pscale = c->nscale * 16.0f;            // |n u| <= n_cap / 16 = n_max / 2
        c->inv_pscale = c->inv_nscale / 16.0f;
    }
    for (int s = 0; s < nsp; s++) {
        SpeciesDev &S = c->sp[s];
        if (!S.cfg.mobile) continue;
        if (S.lanes) INIT_CHECK(lanes_make_tensor_map(c, s));
        if (S.cfg.load != PM2D_LOAD_NONE) {
            INIT_CHECK(launch_load_particles(c, s));
            if (S.random) INIT_CHECK(launch_shuffle_random(c, s));
            if (S.lanes) INIT_CHECK(launch_lanesort(c, s, true, nullptr, nullptr, nullptr));
        } else {
            S.np = 0;   // until pm2d_set_particles
            INIT_CHECK(launch_build_chunks(c, s));   // all-zero tile_off -> zero chunks
        }
        INIT_CHECK(redeposit(c, s));
    }
    INIT_CHECK(refix_backgrounds(c));
    INIT_CHECK(check_flags(c));
#undef INIT_CHECK
#undef INIT_CUDA
    *out = c;
    return PM2D_OK;
}

static void destroy_ctx(pm2d_ctx *c)
{
    if (!c) return;
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    if (c->zstream) {
        cudaStreamSynchronize(c->zstream);
        cudaStreamDestroy(c->zstream);
    }
    for (int k = 0; k < 2; k++) {
        if (c->ev_free[k]) cudaEventDestroy(c->ev_free[k]);
        if (c->ev_zero[k]) cudaEventDestroy(c->ev_zero[k]);
    }
    delete c;
}

extern "C" void pm2d_free(pm2d_ctx *c) { destroy_ctx(c); }

// P:L81, Fig. 1(a): a_sz = a cos(theta), a_px = a sin(theta) cos(beta), a_py = a sin(theta) sin(beta); components 0 = z, 1 = x, 2 = y
extern "C" int pm2d_polarised_beam(const pm2d_laser *proto, double theta, double beta, pm2d_laser out[3])
{
    if (!proto || !out) return fail(PM2D_EINVAL, "null argument");
    const double amp[3] = {proto->a0 * std::cos(theta), proto->a0 * std::sin(theta) * std::cos(beta), proto->a0 * std::sin(theta) * std::sin(beta)};
    int n = 0;
    for (int comp = 0; comp < 3; comp++) {
        if (std::fabs(amp[comp]) <= 1e-300 * std::fabs(proto->a0)) continue;
        out[n] = *proto;
        out[n].a0 = amp[comp];
        out[n].comp = comp;
        n++;
    }
    return n;
}

extern "C" int pm2d_set_lasers(pm2d_ctx *c, const pm2d_laser *lasers, int nlaser)
{
    if (!c || nlaser < 0 || nlaser > PM2D_MAX_LASERS || (nlaser > 0 && !lasers)) return fail(PM2D_EINVAL, "bad laser table");
    for (int l = 0; l < nlaser; l++) {
        int rc = validate_laser_angle(lasers[l], c->g.ny * c->g.dy);
        if (rc) return rc;
    }
    for (int l = 0; l < nlaser; l++)
        if (lasers[l].comp < 0 || lasers[l].comp >= c->g.ncomp) return fail(PM2D_EINVAL, "laser component out of range");
    for (int l = 0; l < nlaser; l++) c->laser[l] = lasers[l];
    c->nlaser = nlaser;
    return PM2D_OK;
}

// ---- the time step: items (1)-(8) of P:L229-238 --------------------------------------------------
static int enqueue_step(pm2d_ctx *c)
{
    int rc;
    // (2) a^{n+1} from a^n, a^{n-1}, n_e^n ; E^n from n_i^n - n_e^n
    if (c->nsub == 1) {
        phase_begin(c, PM2D_PH_FIELD);
        if ((rc = launch_field_step(c, 0))) return rc;
        phase_end(c);
    }
    for (int stage = 0; stage < 2; stage++) {
        // E^n from n^n resp. E^ from n^ (Eqs. 9-11), and in the epilogue of the inverse transform the nodal
        // force of (3) / (7): Eq. 16 with a^n, n^n / Eq. 18 with a^{n+1}, n^
        phase_begin(c, PM2D_PH_POISSON);
        if ((rc = launch_poisson(c, false, stage == 0 ? c->a[1] : c->a[0], stage == 1))) return rc;
        phase_end(c);
        if (stage == 0 && c->nsub > 1) {
            // sub-cycling (Q21): the force of (3) has taken a^n; now S wave steps with n_e^n held (it is zeroed
            // only below), the ring turning after each but the last, so that a[0] = a^{n+1} for stage B
            phase_begin(c, PM2D_PH_FIELD);
            for (int sub = 0; sub < c->nsub; sub++) {
                if ((rc = launch_field_step(c, sub))) return rc;
                if (sub + 1 < c->nsub) {
                    float *t = c->a[2];
                    c->a[2] = c->a[1];
                    c->a[1] = c->a[0];
                    c->a[0] = t;
                }
            }
            phase_end(c);
        }
        // the set just read (n^n resp. n^) is the target of the stage after next: zero it on the side stream now;
        // the target of this stage was zeroed while the previous stage ran
        if ((rc = zero_set_async(c, stage))) return rc;
        PM2D_CUDA_CHECK(cudaStreamWaitEvent(c->stream, c->ev_zero[1 - stage], 0));
        // (3)-(5) gather, predictor, deposit / (7)-(8)+(1) gather, corrector, deposit -- one fused kernel
        phase_begin(c, stage == 0 ? PM2D_PH_STAGE_A : PM2D_PH_STAGE_B);
        for (int s = 0; s < c->nsp; s++)
            if (c->sp[s].cfg.mobile && (rc = launch_stage(c, s, stage))) return rc;
        phase_end(c);
    }
    float *t = c->a[2];
    c->a[2] = c->a[1];
    c->a[1] = c->a[0];
    c->a[0] = t;
    c->step++;
    c->uh_valid = true;
    if (c->prof_on) c->prof_steps++;
    if (c->g.rebin_every > 0 && c->step % c->g.rebin_every == 0) {
        c->uh_valid = false;             // the rebin uses u^ as scratch
        phase_begin(c, PM2D_PH_REBIN);
        for (int s = 0; s < c->nsp; s++)
            if (c->sp[s].cfg.mobile && !c->sp[s].random && (rc = launch_rebin(c, s, nullptr, nullptr, nullptr))) return rc;
        phase_end(c);
    }
    return PM2D_OK;
}

extern "C" int pm2d_step_async(pm2d_ctx *c, int nsteps)
{
    if (!c || nsteps < 0) return fail(PM2D_EINVAL, "bad argument");
    for (int n = 0; n < nsteps; n++) {
        int rc = enqueue_step(c);
        if (rc) return rc;
    }
    return PM2D_OK;
}

extern "C" int pm2d_step(pm2d_ctx *c, int nsteps)
{
    int rc = pm2d_step_async(c, nsteps);
    if (rc) return rc;
    return check_flags(c);
}

extern "C" int64_t pm2d_launch_count(pm2d_ctx *c) { return c ? c->launches : 0; }

extern "C" int64_t pm2d_stray_count(pm2d_ctx *c)
{
    if (!c) return fail(PM2D_EINVAL, "null ctx");
    unsigned long long h = 0;
    PM2D_CUDA_CHECK(cudaMemcpyAsync(&h, c->stray_total, sizeof(h), cudaMemcpyDeviceToHost, c->stream));
    PM2D_CUDA_CHECK(cudaMemsetAsync(c->stray_total, 0, sizeof(h), c->stream));
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    return (int64_t)h;
}
extern "C" int pm2d_lane_subs(pm2d_ctx *c, int s)
{
    if (!c || s < 0 || s >= c->nsp) return fail(PM2D_EINVAL, "bad species");
    return c->sp[s].lanes ? c->sp[s].lane_subs : 0;
}
extern "C" int64_t pm2d_particle_count(pm2d_ctx *c, int s) { return (c && s >= 0 && s < c->nsp) ? c->sp[s].np : -1; }

extern "C" int pm2d_profile_enable(pm2d_ctx *c, int on)
{
    if (!c) return fail(PM2D_EINVAL, "null ctx");
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    c->ev.clear();
    c->ev_phase.clear();
    for (int p = 0; p < PM2D_PH_COUNT; p++) { c->prof_ms[p] = 0; c->prof_launch[p] = 0; }
    c->prof_steps = 0;
    c->prof_on = on != 0;
    return PM2D_OK;
}

extern "C" int pm2d_profile_get(pm2d_ctx *c, double ms[PM2D_PH_COUNT], int64_t launches[PM2D_PH_COUNT], int64_t *steps)
{
    if (!c) return fail(PM2D_EINVAL, "null ctx");
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    for (size_t k = 0; k + 1 < c->ev.size(); k += 2) {
        float t = 0.f;
        PM2D_CUDA_CHECK(cudaEventElapsedTime(&t, c->ev[k], c->ev[k + 1]));
        c->prof_ms[c->ev_phase[k]] += t;
    }
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    c->ev.clear();
    c->ev_phase.clear();
    for (int p = 0; p < PM2D_PH_COUNT; p++) {
        if (ms) ms[p] = c->prof_ms[p];
        if (launches) launches[p] = c->prof_launch[p];
    }
    if (steps) *steps = c->prof_steps;
    return PM2D_OK;
}

// ---- accessors ---------------------------------------------------------------------------------
static int64_t copy_window(pm2d_ctx *c, const float *dev, int i0, int i1, int j0, int j1, float *host, size_t cap)
{
    const int nx = c->g.nx, ny = c->g.ny;
    if (i0 < 0 || i1 > nx + 1 || i0 >= i1 || j0 < 0 || j1 > ny || j0 >= j1 || !host) return fail(PM2D_EINVAL, "bad window");
    const size_t cnt = (size_t)(i1 - i0) * (j1 - j0);
    if (cnt > cap) return fail(PM2D_ENOMEM, "host buffer too small");
    PM2D_CUDA_CHECK(cudaMemcpy2DAsync(host, (size_t)(j1 - j0) * sizeof(float), dev + (size_t)i0 * ny + j0, (size_t)ny * sizeof(float),
                                      (size_t)(j1 - j0) * sizeof(float), (size_t)(i1 - i0), cudaMemcpyDeviceToHost, c->stream));
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    return (int64_t)cnt;
}

extern "C" int64_t pm2d_get_fields(pm2d_ctx *c, int field, int comp, int level, int i0, int i1, int j0, int j1, float *host,
                                   size_t cap)
{
    if (!c) return fail(PM2D_EINVAL, "null ctx");
    const unsigned blocks = (unsigned)((c->nn + 255) / 256);
    int rc;
    switch (field) {
    case PM2D_FIELD_A:
        if (comp < 0 || comp >= c->g.ncomp || level < 0 || level > 1) return fail(PM2D_EINVAL, "bad comp/level");
        return copy_window(c, c->a[1 + level] + (size_t)comp * c->nn, i0, i1, j0, j1, host, cap);
    case PM2D_FIELD_PHI:
        if ((rc = launch_poisson(c, true))) return rc;
        return copy_window(c, c->phi, i0, i1, j0, j1, host, cap);
    case PM2D_FIELD_ENODE:
        if (comp < 0 || comp > 1) return fail(PM2D_EINVAL, "bad comp");
        if ((rc = launch_poisson(c, false))) return rc;
        k_extract_comp<<<blocks, 256, 0, c->stream>>>(c->Enode, comp, c->phi, (size_t)c->nn);
        count_launch(c);
        return copy_window(c, c->phi, i0, i1, j0, j1, host, cap);
    case PM2D_FIELD_FORCE:
        if (comp < 0 || comp > 1 || level < 0 || level >= c->nsp || !c->sp[level].cfg.mobile) return fail(PM2D_EINVAL, "bad comp/species");
        // Eq. 16 for the current state (E of the current densities, a^n, n^n) by the PRODUCTION route: the Poisson solve
        // whose inverse transform evaluates the force of every mobile species in its epilogue, exactly the launches of a step
        if ((rc = launch_poisson(c, false, c->a[1], false))) return rc;
        k_extract_comp<<<blocks, 256, 0, c->stream>>>(c->sp[level].F, comp, c->phi, (size_t)c->nn);
        count_launch(c);
        return copy_window(c, c->phi, i0, i1, j0, j1, host, cap);
    case PM2D_FIELD_FORCE_REF:
        if (comp < 0 || comp > 1 || level < 0 || level >= c->nsp || !c->sp[level].cfg.mobile) return fail(PM2D_EINVAL, "bad comp/species");
        // the same force by the stand-alone kernel k_force on the nodal E grid: a cross-check of the fused epilogue
        if ((rc = launch_poisson(c, false))) return rc;
        if ((rc = launch_force(c, level, c->a[1]))) return rc;
        k_extract_comp<<<blocks, 256, 0, c->stream>>>(c->sp[level].F, comp, c->phi, (size_t)c->nn);
        count_launch(c);
        return copy_window(c, c->phi, i0, i1, j0, j1, host, cap);
    default:
        return fail(PM2D_EINVAL, "unknown field");
    }
}

extern "C" int64_t pm2d_get_moments(pm2d_ctx *c, int s, int moment, int i0, int i1, int j0, int j1, float *host, size_t cap)
{
    if (!c || s < 0 || s >= c->nsp) return fail(PM2D_EINVAL, "bad species");
    SpeciesDev &S = c->sp[s];
    int rc;
    if (moment == PM2D_MOMENT_N) {
        if ((rc = launch_fix_to_float(c, S.nfix, c->inv_nscale, c->phi))) return rc;
    } else if (moment == PM2D_MOMENT_PX || moment == PM2D_MOMENT_PY) {
        if (!S.cfg.mobile) return fail(PM2D_EINVAL, "immobile species has no momentum");
        if (!c->g.eager_moments) {   // build P on demand from the current particles (Eq. 14)
            if ((rc = zero_moments(c, s, false, true))) return rc;
            if ((rc = launch_deposit_only(c, s, false, true))) return rc;
        }
        if ((rc = launch_fix_to_float(c, moment == PM2D_MOMENT_PX ? S.pxfix : S.pyfix, c->inv_pscale, c->phi))) return rc;
    } else
        return fail(PM2D_EINVAL, "unknown moment");
    return copy_window(c, c->phi, i0, i1, j0, j1, host, cap);
}

extern "C" int pm2d_set_fields(pm2d_ctx *c, int field, int comp, int level, const float *host)
{
    if (!c || !host) return fail(PM2D_EINVAL, "null argument");
    if (field != PM2D_FIELD_A || comp < 0 || comp >= c->g.ncomp || level < 0 || level > 1) return fail(PM2D_EINVAL, "only a (level 0/1) can be set");
    PM2D_CUDA_CHECK(cudaMemcpyAsync(c->a[1 + level] + (size_t)comp * c->nn, host, (size_t)c->nn * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    return PM2D_OK;
}

extern "C" int pm2d_set_background(pm2d_ctx *c, int s, const float *host)
{
    if (!c || !host || s < 0 || s >= c->nsp || c->sp[s].cfg.mobile) return fail(PM2D_EINVAL, "not an immobile species");
    PM2D_CUDA_CHECK(cudaMemcpyAsync(c->phi, host, (size_t)c->nn * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    int rc = launch_float_to_fix(c, c->phi, c->nscale, c->sp[s].nfix);
    if (rc) return rc;
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    return PM2D_OK;
}

extern "C" int64_t pm2d_get_particles(pm2d_ctx *c, int s, int64_t first, int64_t count, int32_t *ix, int32_t *iy, float *fx, float *fy,
                                      float *ux, float *uy, float *w, int64_t *id)
{
    if (!c || s < 0 || s >= c->nsp || !c->sp[s].cfg.mobile) return fail(PM2D_EINVAL, "bad species");
    SpeciesDev &S = c->sp[s];
    if (first < 0 || count < 0 || first > S.np) return fail(PM2D_EINVAL, "bad range");
    count = std::min(count, S.np - first);
    if (count == 0) return 0;
    if (id && !S.id) return fail(PM2D_EINVAL, "ids need track_ids");
    // canonical cell + offset and velocity of every particle as separate arrays in the (idle) rebin and
    // predictor buffers: pv2 holds 4 arrays of cap words, uh holds 2
    c->uh_valid = false;                 // u^ is scratch of the unpacking below
    const size_t capw = (size_t)std::max<int64_t>(S.cap, 1);
    int32_t *dix = (int32_t *)S.pv2, *diy = dix + capw;
    float *dfx = (float *)(diy + capw), *dfy = dfx + capw;
    float *dux = (float *)S.uh, *duy = dux + capw;
    int rc = launch_unpack_particles(c, s, dix, diy, dfx, dfy, dux, duy);
    if (rc) return rc;
    auto d2h = [&](void *dst, const void *src, size_t esz) -> cudaError_t {
        if (!dst) return cudaSuccess;
        return cudaMemcpyAsync(dst, (const char *)src + (size_t)first * esz, (size_t)count * esz, cudaMemcpyDeviceToHost, c->stream);
    };
    PM2D_CUDA_CHECK(d2h(ix, dix, 4));
    PM2D_CUDA_CHECK(d2h(iy, diy, 4));
    PM2D_CUDA_CHECK(d2h(fx, dfx, 4));
    PM2D_CUDA_CHECK(d2h(fy, dfy, 4));
    PM2D_CUDA_CHECK(d2h(ux, dux, 4));
    PM2D_CUDA_CHECK(d2h(uy, duy, 4));
    PM2D_CUDA_CHECK(d2h(w, S.w, 4));
    PM2D_CUDA_CHECK(d2h(id, S.id, 8));
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    return count;
}

extern "C" int64_t pm2d_get_predictor(pm2d_ctx *c, int s, int64_t first, int64_t count, float *uhx, float *uhy)
{
    if (!c || s < 0 || s >= c->nsp || !c->sp[s].cfg.mobile || !uhx || !uhy) return fail(PM2D_EINVAL, "bad argument");
    SpeciesDev &S = c->sp[s];
    if (!c->uh_valid) return fail(PM2D_ESTATE, "the predictor velocities of the last step are gone (rebin, pm2d_get_particles or no step yet)");
    if (first < 0 || count < 0 || first > S.np) return fail(PM2D_EINVAL, "bad range");
    count = std::min(count, S.np - first);
    if (count == 0) return 0;
    std::vector<float2> h((size_t)count);
    PM2D_CUDA_CHECK(cudaMemcpyAsync(h.data(), S.uh + first, (size_t)count * sizeof(float2), cudaMemcpyDeviceToHost, c->stream));
    PM2D_CUDA_CHECK(cudaStreamSynchronize(c->stream));
    for (int64_t p = 0; p < count; p++) { uhx[p] = h[(size_t)p].x; uhy[p] = h[(size_t)p].y; }
    return count;
}

extern "C" int pm2d_set_particles(pm2d_ctx *c, int s, int64_t count, const int32_t *ix, const int32_t *iy, const float *fx,
                                  const float *fy, const float *ux, const float *uy, const float *w, int refix_background)
{
    if (!c || s < 0 || s >= c->nsp || !c->sp[s].cfg.mobile) return fail(PM2D_EINVAL, "bad species");
    SpeciesDev &S = c->sp[s];
    if (S.random) return fail(PM2D_ESTATE, "PM2D_ORDER_RANDOM takes its particles from the loader only");
    if (count < 0 || count > S.cap) return fail(PM2D_ENOMEM, "more particles than capacity");
    if (count > 0 && (!ix || !iy || !fx || !fy || !ux || !uy || !w)) return fail(PM2D_EINVAL, "null particle array");
    const int nx = c->g.nx, ny = c->g.ny, nty = c->nty, ntiles = c->ntiles;
    // host-side stable counting sort by (tile, cell) (test / restart path, not the hot path)
    std::vector<int64_t> off(ntiles + 1, 0);
    std::vector<int32_t> coff((size_t)ntiles * CPITCH, 0);
    std::vector<int64_t> key((size_t)count);
    for (int64_t p = 0; p < count; p++) {
        if (ix[p] < 0 || ix[p] >= nx || iy[p] < 0 || iy[p] >= ny || !(fx[p] >= 0.f && fx[p] < 1.f) || !(fy[p] >= 0.f && fy[p] < 1.f))
            return fail(PM2D_EINVAL, "particle outside the box or offset outside [0,1)");
        const int t = (ix[p] / TILE) * nty + iy[p] / TILE, cl = (ix[p] % TILE) * TILE + iy[p] % TILE;
        key[p] = (int64_t)t * CPITCH + cl;
        off[t + 1]++;
        coff[key[p] + 1]++;      // count of cell cl lands in slot cl+1 of the same tile (slot TCELLS = last cell)
    }
    for (int t = 0; t < ntiles; t++) off[t + 1] += off[t];
    std::vector<int64_t> cur((size_t)ntiles * CPITCH);
    for (int t = 0; t < ntiles; t++) {
        int32_t *co = coff.data() + (size_t)t * CPITCH;
        co[0] = 0;
        for (int cl = 0; cl < TCELLS; cl++) co[cl + 1] += co[cl];       // exclusive scan: co[cl] = first slot of cell cl
        for (int cl = 0; cl < TCELLS; cl++) cur[(size_t)t * CPITCH + cl] = off[t] + co[cl];
    }
    std::vector<PV> hpv((size_t)count);
    std::vector<float> hw((size_t)count);
    std::vector<int64_t> hid(S.id ? (size_t)count : 0);
    std::vector<int64_t> slot_of((size_t)count);          // cell-major slot of every particle (stable)
    for (int64_t p = 0; p < count; p++) slot_of[p] = cur[key[p]]++;
    if (S.layered) {
        // the layered order of k_cellsort inside every tile: layer r < LAYERS = particle r of every cell with more than r
        // particles, by (rank of the cell among the occupied cells of its column, column); then the cell-major tail
        std::vector<int64_t> remap((size_t)count);
        for (int t = 0; t < ntiles; t++) {
            const int32_t *co = coff.data() + (size_t)t * CPITCH;
            if (co[TCELLS] == 0) continue;
            int64_t run = off[t];
            for (int r = 0; r < PM2D_LAYERS; r++) {
                int rows[TILE][TILE], nocc[TILE];
                for (int j = 0; j < TILE; j++) {
                    nocc[j] = 0;
                    for (int i = 0; i < TILE; i++)
                        if (co[i * TILE + j + 1] - co[i * TILE + j] > r) rows[j][nocc[j]++] = i;
                }
                for (int k = 0; k < TILE; k++)
                    for (int j = 0; j < TILE; j++)
                        if (k < nocc[j]) remap[(size_t)(off[t] + co[rows[j][k] * TILE + j] + r)] = run++;
            }
            for (int cl = 0; cl < TCELLS; cl++)
                for (int q = PM2D_LAYERS; q < co[cl + 1] - co[cl]; q++) remap[(size_t)(off[t] + co[cl] + q)] = run++;
        }
        for (int64_t p = 0; p < count; p++) slot_of[p] = remap[(size_t)slot_of[p]];
    }
    for (int64_t p = 0; p < count; p++) {
        const int64_t q = slot_of[p];
        int li = ix[p] % TILE, lj = iy[p] % TILE;
        hpv[q].x = ((uint32_t)(li + POS_BIAS) << POS_FRAC_BITS) | (uint32_t)std::floor((double)fx[p] * 16777216.0);
        hpv[q].y = ((uint32_t)(lj + POS_BIAS) << POS_FRAC_BITS) | (uint32_t)std::floor((double)fy[p] * 16777216.0);
        hpv[q].ux = ux[p]; hpv[q].uy = uy[p]; hw[q] = w[p];
        if (S.id) hid[q] = p;
    }
    auto h2d = [&](void *dst, const void *src, size_t bytes) { return cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, c->stream); };
    if (count > 0) {
        PM2D_CUDA_CHECK(h2d(S.pv, hpv.data(), (size_t)count * sizeof(PV)));
        PM2D_CUDA_CHECK(h2d(S.w, hw.data(), (size_t)count * 4));
        if (S.id) PM2D_CUDA_CHECK(h2d(S.id, hid.data(), (size_t)count * 8));
    }
    PM2D_CUDA_CHECK(h2d(S.tile_off, off.data(), (size_t)(ntiles + 1) * 8));
    PM2D_CUDA_CHECK(h2d(S.cell_off, coff.data(), coff.size() * 4));
    S.np = count;
    c->uh_valid = false;
    int rc = launch_build_chunks(c, s);
    if (rc) return rc;
    if (S.lanes && (rc = launch_lanesort(c, s, true, nullptr, nullptr, nullptr))) return rc;
    if ((rc = redeposit(c, s))) return rc;
    if (refix_background && (rc = refix_backgrounds(c))) return rc;
    return check_flags(c);   // synchronises: the host vectors may now go
}

extern "C" int pm2d_rebin(pm2d_ctx *c, int s, int32_t *keys_out, int64_t *perm_out)
{
    if (!c || s < 0 || s >= c->nsp || !c->sp[s].cfg.mobile) return fail(PM2D_EINVAL, "bad species");
    SpeciesDev &S = c->sp[s];
    if (S.random) return fail(PM2D_ESTATE, "PM2D_ORDER_RANDOM has no rebin");
    int32_t *dk = nullptr;
    int64_t *dp = nullptr, *dt = nullptr;
    const size_t n = (size_t)std::max<int64_t>(S.np, 1);
    if (keys_out) PM2D_CUDA_CHECK(cudaMalloc(&dk, n * sizeof(int32_t)));
    if (perm_out) PM2D_CUDA_CHECK(cudaMalloc(&dp, n * sizeof(int64_t)));
    if (keys_out || perm_out) PM2D_CUDA_CHECK(cudaMalloc(&dt, n * sizeof(int64_t)));
    c->uh_valid = false;
    int rc = launch_rebin(c, s, dk, dp, dt);
    if (!rc && keys_out) rc = cudaMemcpyAsync(keys_out, dk, (size_t)S.np * 4, cudaMemcpyDeviceToHost, c->stream) == cudaSuccess ? 0 : PM2D_ECUDA;
    if (!rc && perm_out) rc = cudaMemcpyAsync(perm_out, dp, (size_t)S.np * 8, cudaMemcpyDeviceToHost, c->stream) == cudaSuccess ? 0 : PM2D_ECUDA;
    if (!rc) rc = check_flags(c);
    else cudaStreamSynchronize(c->stream);
    cudaFree(dk);
    cudaFree(dp);
    cudaFree(dt);
    return rc;
}

extern "C" int pm2d_diagnostics(pm2d_ctx *c, pm2d_diag *out)
{
    if (!c || !out) return fail(PM2D_EINVAL, "null argument");
    int rc = launch_poisson(c, true);   // phi of the current densities, so every term is at one time level
    if (rc) return rc;
    return launch_diagnostics(c, out);
}
