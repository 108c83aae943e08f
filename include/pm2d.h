/*
 * pm2d.h -- C ABI of the B200-native PM2D particle-mesh library (libpm2d.so).
 *
 * One time step of PM2D (arXiv 2404.14293): deposit -> wave update + Poisson -> force grid ->
 * gather + predictor -> deposit -> Poisson -> force grid -> gather + corrector (program flow,
 * PAPER.md L229-238, Fig. 3).  Every step of that path runs in hand-written sm_100a kernels;
 * there is no CPU fallback.  "P:Lnnn" below cites /root/reference/PAPER.md line nnn; "Qn" cites
 * a reading listed in DESIGN.md section 3.
 *
 * Conventions
 *   - Units: lengths in lambda0, times in T0 = lambda0/c; velocities in c; densities in
 *     n_c; E in 2 pi c omega0 m_e / e; phi in the unit that makes Eq. 3 hold.
 *   - Nodes (i, j), i = 0..nx, j = 0..ny-1 (y periodic, ny a power of two >= 8); nodal arrays
 *     handed to / returned from the library are row-major float[(nx+1)][ny], index i*ny + j.
 *   - Canonical particle position: x = (ix + fx) dx, y = (iy + fy) dy with integer cell
 *     0 <= ix < nx, 0 <= iy < ny and fx, fy in [0,1) multiples of 2^-24 -- exact in double, so a
 *     checker sees exactly the device state.
 *   - Every call returns PM2D_OK (0) or a negative PM2D_E* code; pm2d_last_error() gives the
 *     text of the last failure on the calling thread's context.  No exceptions, no abort, no
 *     printing.  A ctx is not thread-safe.
 *   - Ownership: the caller owns `dev_workspace` (device memory, e.g. a torch uint8 tensor) and
 *     the CUDA stream for the life of the ctx.  The library carves every device array out of the
 *     workspace and never allocates device memory on the hot path.  `host` pointers are host
 *     memory owned by the caller (pinned memory makes the copies asynchronous-capable, pageable
 *     works).  The ctx itself is a small host object freed by pm2d_free.
 */
#ifndef PM2D_H
#define PM2D_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PM2D_OK 0
#define PM2D_EINVAL (-1)  /* bad argument: ny not a power of two, dt above the stability bound, ... */
#define PM2D_ENOMEM (-2)  /* workspace or host buffer too small */
#define PM2D_ECUDA (-3)   /* a CUDA call or kernel failed */
#define PM2D_ESTATE (-4)  /* call not valid in the current state (e.g. particle left the rebin range; a deposit left the
                             fixed-point range of the grids: density above 4 n_max of the profile, lane order only) */

#define PM2D_MAX_SPECIES 4
#define PM2D_MAX_LASERS 4
#define PM2D_MAX_MODES 16
#define PM2D_MAX_BINS 1024
#define PM2D_MAX_OMEGAS 64
#define PM2D_TILE 32 /* particles are binned by tiles of PM2D_TILE x PM2D_TILE cells */

/* particle shape: 1-D cumulative weight G(s); weights are G differences over the control volumes
 * [i-1/2, i+1/2] of the nodes.  SINE is the paper's cloud, Eq. 12-13. */
enum { PM2D_CIC = 0, PM2D_TSC = 1, PM2D_SINE = 2 };
/* particle loading: NONE = no particles generated (fixed background or
 * particles supplied by pm2d_set_particles); LATTICE_COLD = even lattice, u = 0;
 * RANDOM_MAXWELL = uniform-random offsets, Maxwellian u (BASELINE.json configs; Q7);
 * NUMBER_WEIGHTED = equal weights p[0]/(ppc_x ppc_y), the number of particles of a cell follows the profile
 * (floor(ppc * taper(i) * filament(j) + dither), BASELINE.json config 5); needs `capacity` >= the total. */
enum { PM2D_LOAD_NONE = 0, PM2D_LATTICE_COLD = 1, PM2D_RANDOM_MAXWELL = 2, PM2D_NUMBER_WEIGHTED = 3 };
enum { PM2D_PROFILE_UNIFORM = 0, PM2D_PROFILE_LINEAR = 1, PM2D_PROFILE_EXP_CAPPED = 2, PM2D_PROFILE_FILAMENT_Y = 3 };
/* fields for pm2d_get_fields / pm2d_set_fields */
enum {
    PM2D_FIELD_A = 0,      /* vector potential component `comp`, time level `level` (0 = n, 1 = n-1) */
    PM2D_FIELD_PHI = 1,    /* electrostatic potential on nodes (Eq. 3), recomputed from the current densities */
    PM2D_FIELD_ENODE = 2,  /* E averaged to nodes (Q3), comp 0 = x, 1 = y, from the current densities */
    PM2D_FIELD_FORCE = 3,  /* nodal force of species `level` (Eq. 16) for the current E, a^n, n^n; comp 0 = x, 1 = y.
                              Produced by the launches of a step: the Poisson solve with the force epilogue of its inverse
                              transform (what the stage kernels gather from) */
    PM2D_FIELD_FORCE_REF = 4 /* the same force by the stand-alone kernel on the nodal E grid (cross-check of the epilogue) */
};
/* Storage order of a species inside a tile (as of the last rebin).  CELL_MAJOR: (cell, rank in cell), walked by
 * strip threads with register accumulation (dense species).  LAYERED: layer r < 16 holds particle number r of every
 * cell with more than r particles, its cells ordered by (rank of the cell among those cells of its tile column iy,
 * iy); particles of rank >= 16 follow cell-major.  32 consecutive particles then lie in 32 different cells of 32
 * different columns (a full layer is simply row-major); walked one particle per thread.  AUTO: LAYERED up to 16
 * particles per cell on average (and never for PM2D_NUMBER_WEIGHTED), else CELL_MAJOR.
 * RANDOM (BASELINE.json config 5, "particles stored in random order"): the loader's particles are stored in a
 * pseudo-random permutation with an explicit tile index each (+4 B per particle); no tile is staged: every particle
 * gathers from the global force grid and deposits with integer atomics on the global grids (L2).  No rebin (the
 * positions stay relative to the tile a particle was loaded into: a run may drift at most 64 cells from it, else
 * PM2D_ESTATE), pm2d_rebin and pm2d_set_particles return PM2D_ESTATE.  It exists to measure what the sort buys.
 * LANES (what AUTO picks up to 16 particles per cell; never for PM2D_NUMBER_WEIGHTED): inside a sub-tile (a whole
 * tile, or for species that drift a cell or more per rebin period its two halves of 16 cell rows) the particles are
 * ranked by y and cut into 32 slabs of equal population; slot = 32 * (rank in x inside the slab) + slab, so lane i of a
 * warp always works on slab i and its shared-memory accesses fall on its own bank (pm2d_lanes.cu); see pm2d_rebin. */
enum { PM2D_ORDER_AUTO = 0, PM2D_ORDER_CELL_MAJOR = 1, PM2D_ORDER_LAYERED = 2, PM2D_ORDER_RANDOM = 3, PM2D_ORDER_LANES = 4 };
enum { PM2D_BC_Y_PERIODIC = 0, PM2D_BC_Y_ABSORB = 1 };
enum { PM2D_MOMENT_N = 0, PM2D_MOMENT_PX = 1, PM2D_MOMENT_PY = 2 }; /* n_s, (n u_x)_s, (n u_y)_s, Eq. 14 */

/* The edge taper ends at 1 % of the profile: macro-particles of neighbouring cells must not differ in weight by
 * orders of magnitude, or a light particle that wanders next to heavy ones sees grad(n)/n ~ (n_heavy/n_light)/dx in
 * the pressure term of Eq. 16 and runs away (Q20). */
#define PM2D_TAPER_FLOOR 0.01

typedef struct pm2d_ctx pm2d_ctx; /* opaque */

typedef struct {
    int32_t nx, ny;        /* cells; nx >= 8, ny a power of two in [8, 8192]                          */
    int32_t ncomp;         /* active components of a (Eq. 1): 1..3                                   */
    int32_t rebin_every;   /* tile rebin period in steps, 1..32; 0 = never (tests)                   */
    int32_t eager_moments; /* 1: deposit n, Px, Py at both RK stages as the flow chart says (P:L197,
                              L229, L234); 0: deposit n only and build Px, Py when pm2d_get_moments
                              asks (nothing in the step reads them)                                   */
    int32_t track_ids;     /* 1: carry a particle id through the rebin (tests); costs 8 B/particle   */
    int32_t particle_order; /* PM2D_ORDER_*: storage order inside a tile and the stage kernel that goes with it */
    int32_t subcycle;      /* S in 0..16 (0, 1 = none): the particle step is S wave-equation steps long, "the time step
                              for updating the particle motion is five times larger" (Q21).
                              One pm2d_step is then S steps of Eq. 6/8 with n_e held, and Eqs. 17/19 with S*dt;
                              S*dt/min(dx,dy) <= 4                                                    */
    int32_t bc_y;          /* PM2D_BC_Y_PERIODIC (BASELINE.json configs) | PM2D_BC_Y_ABSORB: "the second-order absorbing
                              boundary condition ... on all of four boundaries": Eq. 8 with x and
                              y exchanged on the walls j = 0 and j = ny-1 of `a`, first-order outgoing condition along
                              the diagonal at the four corners (Q23).  Particles, densities, Poisson and the
                              force grid stay periodic in y                                           */
    int32_t probe_steps;   /* 0: off.  R in 1..65536: the library keeps, on the device, the boundary records of the last R
                              particle steps (pm2d_get_probe, pm2d_probe_spectrum; Fig. 12): R * ncomp * 2 * ny
                              floats of workspace, written by the boundary kernels themselves (no extra launch)  */
    double dx, dy, dt;     /* lambda0, lambda0, T0; dt = step of the wave equation,
                              dt*sqrt(1/dx^2 + 1/dy^2 + pi^2 n_max) < 1                     */
} pm2d_grid;

typedef struct {
    double mass;           /* m_s / m_e (electron 1, deuterium 3672)                                  */
    double T_keV;          /* v_th = sqrt(T/511/mass)                                         */
    double pressure_coeff; /* C in  -C v_th^2 grad(n)/n ; Eq. 2 prints 2 (Q8)               */
    double DD;             /* side length of the cloud in cells: 1 for CIC, 2 for TSC, < 2 for SINE   */
    int32_t sign;          /* -1 electron, +1 ion (Z = 1), 0 neutral (tests: pressure force alone)    */
    int32_t shape;         /* PM2D_CIC | PM2D_TSC | PM2D_SINE                                         */
    int32_t mobile;        /* 0: fixed neutralising background (Q13)                                  */
    int32_t load;          /* PM2D_LOAD_*                                                             */
    int32_t ppc_x, ppc_y;  /* N, M of P:L154                                                          */
    int64_t capacity;      /* particle slots when load == NONE (pm2d_set_particles) or NUMBER_WEIGHTED; else 0 */
} pm2d_species;

typedef struct {
    int32_t kind;          /* PM2D_PROFILE_*                                                          */
    int32_t taper_cells;   /* edge taper at both x walls (Q9): within taper_cells of a wall the profile is
                              multiplied by PM2D_TAPER_FLOOR + (1 - PM2D_TAPER_FLOOR) sin^2(pi d / 2 taper_cells),
                              d = distance of the cell centre from the wall in cells; 0 = none           */
    double p[4];           /* UNIFORM: n0. LINEAR: n(0), n(Lx). EXP_CAPPED: n0, Lx/L, cap.
                              FILAMENT_Y: mean n0, amplitude A, sigma in cells: n(j) ~ 1 + A exp(-(y-Ly/2)^2/2 sigma^2) */
    int32_t taper_cells_y; /* the same taper at both y walls (0 = none): with taper_cells it makes the paper's slab "at the
                              center of the simulation box" with margins on all sides, the
                              margins at PM2D_TAPER_FLOOR of the profile instead of vacuum (Q20).  Weights only: not
                              with PM2D_NUMBER_WEIGHTED                                               */
    int32_t pad_;
    int32_t slab[4];       /* x_lo, x_hi, y_lo, y_hi in cells; all zero = the whole box.  Only cells with x_lo <= i < x_hi and
                              y_lo <= j < y_hi hold particles: "a plasma slab is set at the center of the simulation box, and
                              the vacuum space is usually set around the plasma slab ... allowing the plasma expanding"
                              (P:L81).  The loaded cells get the ids, offsets, momenta and weights they have without the slab
                              (the profile still spans the box; use taper_cells = 0 for a hard edge).  The margins are true
                              vacuum: no particles, Q10 keeps the pressure term out where n = 0.  Not with
                              PM2D_NUMBER_WEIGHTED.  EINVAL unless 0 <= lo < hi <= nx resp. ny                       */
} pm2d_profile;

typedef struct {
    double a0, omega;      /* amplitude; frequency in omega0 (Eq. 4)                        */
    double y0, w0;         /* beam centre and width in lambda0; w0 <= 0: plane wave                   */
    double t_rise;         /* sin^2 turn-on over t_rise (Q14); 0: none                                */
    double alpha;          /* angle of incidence in radians, |alpha| <= 1 (Eq. 5; Q22): the
                              beam axis is (cos alpha, -sin alpha) in box coordinates and crosses the boundary at y0.
                              A plane wave (w0 <= 0) at alpha != 0 must fit the periodic box:
                              omega*sin(alpha)*Ly an integer, else PM2D_EINVAL                       */
    int32_t comp;          /* component of a that carries the beam                                    */
    int32_t pad_;
} pm2d_laser;

typedef struct {
    int64_t step;
    double time;                        /* step * dt                                                  */
    double W_es, W_int, W_em;           /* energy terms of DESIGN.md Q11, per dx*dy                   */
    double W_kin[PM2D_MAX_SPECIES], W_th[PM2D_MAX_SPECIES];
    double charge[PM2D_MAX_SPECIES];    /* sum over nodes of n_s * control volume (cells)            */
    int64_t count[PM2D_MAX_SPECIES];    /* particles held                                             */
    double W_total;
} pm2d_diag;

/* phases timed by the built-in CUDA-event profile (pm2d_profile_*); the nodal force is evaluated in the epilogue
 * of the Poisson solve, so PM2D_PH_FORCE stays 0 during steps */
enum { PM2D_PH_FIELD = 0, PM2D_PH_POISSON = 1, PM2D_PH_FORCE = 2, PM2D_PH_STAGE_A = 3,
       PM2D_PH_STAGE_B = 4, PM2D_PH_REBIN = 5, PM2D_PH_COUNT = 6 };

/* Bytes of device workspace pm2d_init needs for this problem; 0 on invalid arguments. */
size_t pm2d_query_workspace(const pm2d_grid *grid, const pm2d_species *species, int nsp);

/* Build a context: validates arguments, carves the workspace, zeroes the fields, loads the
 * particles (profile x loader x seed, Philox-4x32-10), bins them by tile,
 * deposits item (1) of the flow and fixes immobile backgrounds (Q13).  `cuda_stream` is
 * a cudaStream_t (NULL = default stream).  Synchronises the stream before returning. */
int pm2d_init(const pm2d_grid *grid, const pm2d_species *species, int nsp, const pm2d_profile *profile,
              const pm2d_laser *lasers, int nlaser, uint64_t seed, void *dev_workspace, size_t bytes,
              void *cuda_stream, pm2d_ctx **out);

/* Advance `nsteps` time steps (items (1)-(8)).  Enqueues everything on the stream
 * with no host round trip inside, then synchronises the stream once. */
int pm2d_step(pm2d_ctx *ctx, int nsteps);
/* Same, without the final synchronisation (the caller synchronises its stream). */
int pm2d_step_async(pm2d_ctx *ctx, int nsteps);

/* Polarisation decomposition of one beam (Fig. 1(a)): "assuming the direction of vector potential a has an angle
 * of theta with respect to the z-axis, then the components of a in the S-polarization direction (z direction) is
 * a_sz = a cos(theta) ... a_px = a sin(theta) cos(beta) and a_py = a sin(theta) sin(beta)".  Components of `a` are
 * numbered 0 = z (S polarisation, the one BASELINE.json's configs use), 1 = x, 2 = y; every component obeys the same
 * wave equation (Eq. 1), so the beam becomes up to three laser-table entries that differ in `a0` and `comp` only.
 * proto: host, the beam (its a0 is the amplitude a, its comp is ignored); theta, beta in radians; out: host array of 3
 * entries.  Returns the number of entries written (components whose amplitude is not exactly zero, in the order z, x,
 * y), or PM2D_EINVAL on a null pointer.  The grid needs ncomp = 3 unless only the z entry comes back. */
int pm2d_polarised_beam(const pm2d_laser *proto, double theta, double beta, pm2d_laser out[3]);

/* Replace the laser table (e.g. a time-varying drive); nlaser <= PM2D_MAX_LASERS. */
int pm2d_set_lasers(pm2d_ctx *ctx, const pm2d_laser *lasers, int nlaser);

/* Copy the window rows i0..i1-1, columns j0..j1-1 of a nodal field / moment into host[(i1-i0)*(j1-j0)].
 * Returns the element count or a negative code; cap = capacity of `host` in elements. */
int64_t pm2d_get_fields(pm2d_ctx *ctx, int field, int comp, int level, int i0, int i1, int j0, int j1,
                        float *host, size_t cap);
int64_t pm2d_get_moments(pm2d_ctx *ctx, int species, int moment, int i0, int i1, int j0, int j1,
                         float *host, size_t cap);
/* Write one full nodal array of `a` (component comp, level 0 = n, 1 = n-1) from host[(nx+1)*ny]. */
int pm2d_set_fields(pm2d_ctx *ctx, int field, int comp, int level, const float *host);

/* Particles first..first+count-1 of a species in storage order (binned by tile, then by cell as of the last
 * rebin), canonical form.
 * Any output pointer may be NULL.  `id` needs track_ids.  Returns the number written. */
int64_t pm2d_get_particles(pm2d_ctx *ctx, int species, int64_t first, int64_t count, int32_t *ix, int32_t *iy,
                           float *fx, float *fy, float *ux, float *uy, float *w, int64_t *id);
/* Predictor velocities u^ (Eq. 17) that the last pm2d_step left for the slots first..first+count-1 of a
 * species, in the storage order pm2d_get_particles had BEFORE that step (a step without rebin keeps the order).  For
 * tests of the gather + predictor at full size.  uhx, uhy: host float[count].  PM2D_ESTATE when the arrays have been
 * reused since (a rebin at the end of the step, pm2d_get_particles, pm2d_set_particles) or no step was taken.
 * Returns the number written. */
int64_t pm2d_get_predictor(pm2d_ctx *ctx, int species, int64_t first, int64_t count, float *uhx, float *uhy);

/* Replace all particles of a mobile species (count <= capacity; any order; ids = 0..count-1 in
 * the order given), bin them, re-deposit every moment.  If `refix_background` != 0 the immobile
 * species of opposite sign are re-set to neutralise the new deposit (Q13). */
int pm2d_set_particles(pm2d_ctx *ctx, int species, int64_t count, const int32_t *ix, const int32_t *iy,
                       const float *fx, const float *fy, const float *ux, const float *uy, const float *w,
                       int refix_background);
/* Set the nodal density of an immobile species from host[(nx+1)*ny] (n_c). */
int pm2d_set_background(pm2d_ctx *ctx, int species, const float *host);

/* Run the rebin now.  keys_out[count] (optional, host) receives, in the OLD storage order, the
 * destination key of every particle, key = tile * PM2D_TILE^2 + (ix % PM2D_TILE) * PM2D_TILE + iy % PM2D_TILE
 * with tile = (ix / PM2D_TILE) * ceil(ny / PM2D_TILE) + iy / PM2D_TILE; perm_out[count] (optional, host)
 * receives for every NEW slot the OLD slot it came from.  CELL_MAJOR species: the result equals a stable counting
 * sort by key.  LAYERED species: with r = the rank of a particle among those of equal key in the old order, the
 * result is sorted by tile, then layer min(r, 16); inside a layer below 16 by (rank of the cell among the cells of
 * the same tile and the same iy that hold more than r particles, in ix order; iy), inside the tail by (cell, r).
 * LANES species are sorted by their SORT position: the position plus the free flight of half a rebin period, in
 * units of 2^-24 cell,
 *     xs = ix 2^24 + fx 2^24 + rint(float(ux) * float(rebin_every * S dt / (2 dx) * 2^24))      (float32 product, round to nearest)
 * clamped to [0, nx 2^24 - 1] (a sort position beyond a wall stays in the wall tile), ys likewise but wrapped into [0, ny 2^24).
 * The tile is that of (xs, ys); keys_out = tile * PM2D_TILE^2 + cell of (xs, ys) in the tile.  After the stable sort by tile,
 * inside every tile, with ix', fx', iy', fy' the tile-relative cell and offset of (xs, ys):
 * h = sub-tile (ix' >= 16 when pm2d_lane_subs is 2,
 * else 0); rho = rank in the stable sort by key_A = (h, iy', floor(32 fy')); slab = the rho-th of the N_h particles
 * of the sub-tile cut into 32 slabs whose sizes differ by at most one (the first N_h mod 32 slabs hold one more);
 * w = rank inside the slab in the stable sort by key_B = (h, slab, x bin), x bin = (2 (ix' % 16) + floor(2 fx')) resp.
 * ix'; slot = first slot of the sub-tile + 32 w + slab.  (A particle may therefore be listed in a tile next to the one
 * it sits in; pm2d_get_particles always returns its true cell.) */
int pm2d_rebin(pm2d_ctx *ctx, int species, int32_t *keys_out, int64_t *perm_out);

int pm2d_diagnostics(pm2d_ctx *ctx, pm2d_diag *out);

/* Fourier-mode amplitudes of a species' current nodal density (the k-spectra of Figs. 7 and 14,
 * P:L356, are |A|^2 of delta n_e):
 *     A(m_x, m_y) = sum_{i=0..nx} sum_{j<ny} v_i n_s(i,j) exp(-2 pi i (m_x i / nx + m_y j / ny)),
 * v_i = 1/2 on the wall columns i = 0, nx (half control volumes, Q9), 1 elsewhere; in units of n_c * cells.
 * mx, my: host int32[nmodes] (any sign), 1 <= nmodes <= PM2D_MAX_MODES; re, im: host double[nmodes].
 * float32/fixed-point input, float64 accumulation; synchronises the stream. */
/* Velocity distribution of a species inside a sub-box (Fig. 9): hist[b] = sum of the weights
 * w_p of the particles whose cell (ix, iy) lies in [i0, i1) x [j0, j1) and whose velocity component u (comp 0 = u_x,
 * 1 = u_y, in c) falls into bin b = floor((u - umin) * (nbins / (umax - umin))) evaluated in float32 (u, umin and the
 * scale rounded to float32 first); particles outside [umin, umax) are not counted.  hist: host double[nbins],
 * 1 <= nbins <= PM2D_MAX_BINS.  Synchronises the stream.  Sums in float64; the order of the additions is not fixed. */
int pm2d_velocity_histogram(pm2d_ctx *ctx, int species, int i0, int i1, int j0, int j1, int comp, double umin, double umax,
                            int nbins, double *hist);

/* Boundary records ("the time evolution of back-scattering laser light on the left boundary", P:L320;
 * Fig. 12(b), (d)).  With pm2d_grid.probe_steps = R > 0 every particle step q = 1, 2, ... (time q * S * dt)
 * leaves one record per component and wall: wall 0 = left, the scattered field a - a_inc on the nodes (0, j) (the
 * incident wave split off as in P:L122); wall 1 = right, a on the nodes (nx, j).  The last min(q, R) records are kept.
 * pm2d_get_probe copies them in time order into host[n * ny] (host float32, capacity `cap` elements), stores the step
 * index q of the first one in *first_step (host, may be NULL) and returns n (0 before the first step) or a negative
 * code (PM2D_ESTATE if probe_steps = 0).  Synchronises the stream. */
int64_t pm2d_get_probe(pm2d_ctx *ctx, int wall, int comp, float *host, size_t cap, int64_t *first_step);
/* Frequency spectrum of those records (Fig. 12(c), (e)), over the columns j0 <= j < j1:
 *     A_j(w) = dt_s sum_m h[m, j] exp(-2 pi i w m dt_s),   power[k] = sum_j |A_j(omega[k])|^2,
 * m = 0 .. n-1 over the kept records in time order, dt_s = S * dt, omega in units of omega0 (host double[nomega],
 * 1 <= nomega <= PM2D_MAX_OMEGAS); power: host double[nomega].  float32 records, float64 phases and sums.
 * Returns n, the number of records used, or a negative code.  Synchronises the stream. */
int64_t pm2d_probe_spectrum(pm2d_ctx *ctx, int wall, int comp, int j0, int j1, int nomega, const double *omega, double *power);

int pm2d_mode_amplitudes(pm2d_ctx *ctx, int species, int nmodes, const int32_t *mx, const int32_t *my, double *re, double *im);
/* The same sum for callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
 * no ctx, no workspace, no cudaMalloc / cudaFree / allocating library routine, no synchronisation.
 *   n_dev    DEVICE float[(nx + 1) * ny], a nodal density in the layout of pm2d_get_moments (read only)
 *   mx, my   HOST int32[nmodes], copied into the launch parameters before the call returns
 *   out_dev  DEVICE double[2 * nmodes]: Re A, Im A of mode k in out_dev[2 k], out_dev[2 k + 1], written on `stream`
 *   stream   cudaStream_t (NULL = the default stream); two kernels are enqueued on it
 * ny is any size >= 1 here (no FFT).  Scratch: per-row partial sums in ONE file-scope device array of the library,
 * PM2D_STATIC_MAX_ROWS * PM2D_MAX_MODES * 16 bytes = 4.0 MiB, held by every GPU that loads libpm2d.so until the process
 * exits.  nx + 1 > PM2D_STATIC_MAX_ROWS is refused with PM2D_EINVAL (use pm2d_mode_amplitudes).  The first call on a
 * device resolves the array's device address (cudaGetSymbolAddress, once per device, that device current): make that
 * call outside a graph capture.  Every call shares the array and leaves its partial sums in it; a call overwrites all
 * the entries it reads, so nothing has to be cleared, but two calls that OVERLAP on the GPU (different streams, or
 * graphs replayed concurrently) race on it: order them.  float32 input, float64 sums in a fixed order (the result is
 * reproducible bit for bit, unlike pm2d_mode_amplitudes' atomics). */
#define PM2D_STATIC_MAX_ROWS 16385
int pm2d_mode_amplitudes_static(const float *n_dev, int nx, int ny, int nmodes, const int32_t *mx, const int32_t *my,
                                double *out_dev, void *stream);
int64_t pm2d_particle_count(pm2d_ctx *ctx, int species);

/* CUDA-event profile of the step phases on the ctx's stream.  enable(1) starts recording one event
 * pair per phase per step (no synchronisation added); get() synchronises and returns the summed
 * milliseconds and kernel-launch counts per phase since enable(1), and the steps covered. */
int pm2d_profile_enable(pm2d_ctx *ctx, int on);
int pm2d_profile_get(pm2d_ctx *ctx, double ms[PM2D_PH_COUNT], int64_t launches[PM2D_PH_COUNT], int64_t *steps);
/* Kernels launched by this ctx since init. */
int64_t pm2d_launch_count(pm2d_ctx *ctx);
/* Statistics: particle-stage visits, since the last call, that were not served from a strip thread's
 * register patch (the particle had drifted more than half a cell from its cell of the last rebin) but
 * from the tile's shared windows or the global grids.  Synchronises the stream; resets the counter. */
int64_t pm2d_stray_count(pm2d_ctx *ctx);
/* Lane order of a species: sub-tiles per tile (2: two halves of 16 cell rows; 1: whole tiles), 0 if the species is
 * stored in another order, negative code on a bad argument. */
int pm2d_lane_subs(pm2d_ctx *ctx, int species);

void pm2d_free(pm2d_ctx *ctx);
const char *pm2d_last_error(void);
const char *pm2d_version(void);

/* sizeof of the structs above as this library was compiled: which = 0 pm2d_grid, 1 pm2d_species, 2 pm2d_profile,
 * 3 pm2d_laser, 4 pm2d_diag; -1 for any other value.  Host only, no ctx, no GPU: a binding checks its own layout
 * against it before it hands a struct over (tests/test_abi.py does, on a machine without a GPU). */
int pm2d_struct_size(int which);

#ifdef __cplusplus
}
#endif
#endif /* PM2D_H */
