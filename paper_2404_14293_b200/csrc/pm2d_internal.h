// pm2d_internal.h -- context layout and launcher prototypes shared by the .cu files of libpm2d.so.
// Not part of the public ABI (include/pm2d.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/pm2d.h"

// ---- geometry of the particle tiles -----------------------------------------------------------
constexpr int TILE = PM2D_TILE;          // cells per tile side
constexpr int HALO = 2;                  // window nodes beyond the tile on each side
constexpr int WIN = TILE + 2 * HALO + 1; // window nodes per side (37)
constexpr int WPITCH = WIN;              // odd pitch: rows start on different banks
constexpr int CHUNK = 8192;              // max particles per CTA work item (loader, tile rebin, unpack)
constexpr int PTHREADS = 256;            // threads per CTA of the chunk kernels
constexpr int TCELLS = TILE * TILE;      // cells per tile
constexpr int CPITCH = TCELLS + 1;       // ints per tile in cell_off (last = particles in the tile)
constexpr int PM2D_ZEROS_BYTES = 64 * 1024;   // a block of zeros in the workspace (>= the deposit windows of k_stage_lanes)
constexpr int PM2D_LAYERS = 16;          // layered order: ranks >= PM2D_LAYERS form a cell-major tail
constexpr int TRI_M = 32;                // rows per x-partition of the tridiagonal solve
// fixed-point tile-relative position: (cell_rel + POS_BIAS) << 24 | frac24
constexpr int POS_BIAS = 64;
constexpr int POS_FRAC_BITS = 24;
constexpr uint32_t POS_FRAC_MASK = (1u << POS_FRAC_BITS) - 1u;

// one particle: fixed-point tile-relative position and velocity, 16 bytes (one 128-bit access)
struct __align__(16) PV {
    uint32_t x, y;
    float ux, uy;
};

struct SpeciesDev {
    // host copy of the parameters
    pm2d_species cfg;
    double vth2;
    int64_t np;          // particles held (constant: walls reflect, y wraps)
    int64_t cap;
    bool random;         // PM2D_ORDER_RANDOM: permuted storage + ptile, global gather / deposit, no rebin
    int32_t *ptile;      // [cap] tile of every particle (random order only)
    bool layered;        // storage order inside a tile: (rank in cell, cell) + thread-per-particle stage kernel;
                         // else (cell, rank) + strip kernel
    bool lanes;          // PM2D_ORDER_LANES: slot = 32 * (rank in x inside a y-slab) + y-slab; k_stage_lanes (pm2d_lanes.cu)
    int lane_copies;     // window copies of k_stage_lanes: 4 (species that drift a cell or more per rebin period) or 2
    int lane_subs;       // sub-tiles per tile in the lane order: 2 (16 cell rows each; hot species, 4 window copies) or 1
    int32_t *sub0;       // [ntiles] lane order: particles of sub-tile 0 of every tile (the tile's first sub0[t] slots)
    alignas(64) unsigned long long tmapF[16];   // CUtensorMap of F (lane order: the force windows are bulk-async box loads)
    int32_t *lane_exp;   // [ntiles] lane order: window units of the tile, sn | sp << 8 (pm2d_lanes.cu)
    // particles (device), stored tile by tile and, inside a tile, cell by cell (as of the last rebin)
    PV *pv;              // position + velocity
    float *w;            // density weight
    float2 *uh;          // predictor velocity u^ (Eq. 17); scratch outside a step
    PV *pv2;             // rebin double buffers
    float *w2;
    int64_t *id, *id2;   // optional
    int32_t *cell_off;   // [ntiles][CPITCH] first slot (relative to the tile) of each cell's run
    // binning
    int64_t *tile_off;   // [ntiles+1] first slot of each tile
    int64_t *tile_off2;
    int32_t *chunk_tile; // [max_chunks]
    int64_t *chunk_beg;  // [max_chunks+1]
    int32_t *chunk_cnt9; // [max_chunks][9] movers per direction (rebin)
    int64_t *chunk_rel9; // [max_chunks][9] offset inside the destination tile
    int32_t *tile_first_chunk; // [ntiles+1]
    int32_t *tile_cnt;         // [ntiles] scratch: particles per tile after a rebin
    int32_t *nchunks_dev;      // [1]
    int32_t max_chunks;
    int32_t nchunks;     // host copy (refreshed after a rebin)
    // grids (device)
    int32_t *nfix;       // density, fixed point, [(nx+1)*ny] (current)
    int32_t *pxfix, *pyfix;
    int32_t *nhat, *pxhat, *pyhat; // second set: deposits of stage A (x^, u^); zeroed on the side stream
    float2 *F;           // nodal force (Eq. 16)
};

struct pm2d_ctx {
    pm2d_grid g;
    int nsp, nlaser;
    SpeciesDev sp[PM2D_MAX_SPECIES];
    pm2d_laser laser[PM2D_MAX_LASERS];
    pm2d_profile profile;
    uint64_t seed;
    cudaStream_t stream;
    cudaStream_t zstream;            // side stream: zeroes the idle deposit set while a stage kernel runs
    cudaEvent_t ev_free[2], ev_zero[2];   // [0] main set (n^n, stage B target), [1] hat set (stage A target)
    int64_t step;        // particle steps taken
    bool uh_valid;       // the u^ arrays still hold the predictor velocities of the last step (pm2d_get_predictor)
    int nsub;            // wave-equation steps per particle step (Q21)
    double dtp;          // particle time step = nsub * g.dt
    int64_t nn;          // nodes
    int ntx, nty, ntiles;
    int LP;              // pitch (complex elements) of spectral rows: ny/2 + 2
    float nscale, inv_nscale; // density fixed point: n = fix * inv_nscale (power of two)
    float pscale, inv_pscale; // momentum fixed point
    // fields
    float *a[3];         // ring of time levels, each [ncomp][nn]; a[0] = n+1 target, a[1] = n, a[2] = n-1
    float2 *rho_hat;     // [(nx+1)][LP]
    // partitioned chasing method (pm2d_poisson.cu): tables [2][TRI_M][LP], sums [P][LP], g [P+1][LP]
    double *tri_cp, *tri_V, *tri_W, *tri_den;
    double2 *tri_sumV, *tri_sumW, *tri_g;
    int tri_P, tri_mlast;
    float2 *ehx, *ehy;   // [(nx+1)][LP] spectra of nodal E (or phi^ in ehx for diagnostics)
    float2 *Enode;       // [nn]
    float *phi;          // [nn] (diagnostics only)
    float2 *twiddle;     // [ny/2]
    double *red;         // [64] reduction scratch
    double *hist;        // [PM2D_MAX_BINS] velocity histogram scratch
    float *probe;        // [probe_steps][ncomp][2][ny] ring of boundary records (slot = (q-1) % probe_steps), or nullptr
    int32_t *flags;      // [4] device error flags
    double *shape_y, *taper_x;   // [ny], [nx] relative density tables of the number-weighted loader
    unsigned long long *stray_total; // [1] statistics
    int32_t *zeros;                  // [PM2D_ZEROS_BYTES / 4] never written: source of the bulk zero fill of the lanes windows
    int64_t *ovf_p;      // [ovf_cap] particles deferred by k_stage (footprint outside the tile window)
    int32_t *ovf_tile, *ovf_count;
    int ovf_cap;
    int cap_extra;       // tuning: see PartParams::cap_extra
    // profile
    bool prof_on;
    std::vector<cudaEvent_t> ev;   // 2 per phase per step while profiling is on; pm2d_profile_get folds them into prof_ms and frees them
    std::vector<int> ev_phase;
    double prof_ms[PM2D_PH_COUNT];
    int64_t prof_launch[PM2D_PH_COUNT];
    int64_t prof_steps;
    int cur_phase;
    int64_t launches;
};

void pm2d_set_error(const std::string &s);
#define PM2D_CUDA_CHECK(call)                                                                  \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess) {                                                               \
            pm2d_set_error(std::string(#call) + ": " + cudaGetErrorString(e_));                \
            return PM2D_ECUDA;                                                                 \
        }                                                                                      \
    } while (0)

static inline void count_launch(pm2d_ctx *c, int n = 1)
{
    c->launches += n;
    if (c->prof_on && c->cur_phase >= 0) c->prof_launch[c->cur_phase] += n;
}

// ---- launchers (each enqueues on c->stream and returns a PM2D_* code) --------------------------
// pm2d_particles.cu
int launch_load_particles(pm2d_ctx *c, int s);
int launch_shuffle_random(pm2d_ctx *c, int s);
int launch_stage(pm2d_ctx *c, int s, int stage);            // 0 = A (Eq. 17), 1 = B (Eq. 19)
int launch_deposit_only(pm2d_ctx *c, int s, bool density, bool momentum);
int launch_rebin(pm2d_ctx *c, int s, int32_t *keys_dev, int64_t *perm_dev, int64_t *perm_tmp_dev);
int launch_set_cell_offsets_uniform(pm2d_ctx *c, int s);
int launch_build_chunks(pm2d_ctx *c, int s);
int launch_unpack_particles(pm2d_ctx *c, int s, int32_t *ix, int32_t *iy, float *fx, float *fy, float *ux, float *uy);
// pm2d_lanes.cu
int launch_lanesort(pm2d_ctx *c, int s, bool from_primary, int32_t *keys_dev, int64_t *perm_dev, const int64_t *perm1_dev);
int launch_stage_lanes(pm2d_ctx *c, int s, int stage, int qmask);
double lane_ucap(const SpeciesDev &S);
float lane_pred(const pm2d_ctx *c, int axis);
int lanes_make_tensor_map(pm2d_ctx *c, int s);
// pm2d_fields.cu
int launch_field_step(pm2d_ctx *c, int sub);
int launch_force(pm2d_ctx *c, int s, const float *a_level);
int launch_fix_background(pm2d_ctx *c, int s);
int launch_fix_to_float(pm2d_ctx *c, const int32_t *src, float scale, float *dst);
int launch_float_to_fix(pm2d_ctx *c, const float *src, float scale, int32_t *dst);
// pm2d_poisson.cu
int launch_poisson_init(pm2d_ctx *c);
int launch_poisson(pm2d_ctx *c, bool want_phi, const float *force_a = nullptr, bool use_hat = false);
// pm2d_diag.cu
int launch_diagnostics(pm2d_ctx *c, pm2d_diag *out);
