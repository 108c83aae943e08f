/*
 * pm2d_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, double-precision, single-threaded CPU statement of the PM2D time step
 * (arXiv 2404.14293), written from the paper, one function per passage.  It shares no code,
 * header, table or constant with the CUDA path under paper_2404_14293_b200/csrc/.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 *
 * Citations: "P:Lnnn" = /root/reference/PAPER.md line nnn.  "Qn" = a reading of a silent,
 * ambiguous or garbled passage, listed in DESIGN.md section 3.
 *
 * Conventions
 *   nodes (i,j), i = 0..nx, j = 0..ny-1 (y periodic), stored row-major as  i*ny + j.
 *   cell-centred arrays (E) have i = 0..nx-1:  (i+1/2, j+1/2)  stored as  i*ny + j.
 *   particle positions X, Y are in CELL units (x = X*dx), velocities in c, weights in n_c.
 *   lengths in lambda0, times in T0, u in c, E in 2 pi c omega0 m_e / e.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P1..P14 of DESIGN.md section 3; the S8(f) widenings in
 * tests/test_oracle_next.py: P15 oblique incidence, P16 sub-cycling, P17 mode amplitudes, P18 velocity
 * histogram, P19 absorbing y walls and corners (Q23), P20 boundary records and their spectrum; round 2
 * (tests/test_oracle_physics.py, test_oracle_pins.py, test_oracle_loader.py): P21 mobile species of mass != 1 (ion
 * plasma oscillation, heavy neutral sound wave), P22 the ponderomotive coefficient of Eq. 16, P7b the transverse term
 * of Eq. 8 (oblique reflection is second order), P23 the ion-acoustic wave of two mobile species (two-fluid
 * dispersion), Q20 (a hard-edged slab expands with bounded velocities, a weight taper to zero runs away), the
 * loader (oracle/loader.py: Philox known-answer vectors, counts, weights, moments, the slab extent of P:L81) and
 * orc_polarised (Fig. 1(a)).
 * Eq. 21 (SBS growth rate) is not pinned: parity unpinned for that formula (DESIGN.md section 9 says why a
 * slab between walls cannot show it); P23 pins the sound wave it scatters from.
 * Parity unpinned (conventions only, identical by construction on both sides):
 * Q5 (Dirichlet phi at the x walls), Q13, Q14, Q24, the value 0 of Q10 and the taper recipe of Q9 (the wall weights of Q9
 * and the cell-centre sampling of Q17 are pinned: uniform lattice on wall nodes, loader weights; Q3, E to the nodes, by
 * the closed-form transfer factors of a Fourier mode).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_PI 3.14159265358979323846

enum { ORC_CIC = 0, ORC_TSC = 1, ORC_SINE = 2 };

typedef struct {
    int32_t nx, ny;      /* cells; nodes are (nx+1) x ny */
    int32_t ncomp;       /* active components of a (1..3) */
    int32_t subcycle;    /* S: the particle step is S wave-equation steps long (Q21); 0, 1 = none */
    int32_t bc_y;        /* boundary condition of a at the y walls: 0 periodic (BJ configs), 1 absorbing (Q23) */
    int32_t pad_;
    double dx, dy, dt;   /* dt: time step of the wave equation */
} orc_grid;

typedef struct {
    double mass;         /* m_s / m_e */
    double vth2;         /* v_th^2 = T_keV / 511 / mass */
    double C;            /* pressure coefficient, 2 in Eq. 2 */
    double DD;           /* side length of the particle in cells (Q1) */
    int32_t sign;        /* -1 electron, +1 ion, 0 neutral */
    int32_t shape;       /* ORC_CIC / ORC_TSC / ORC_SINE */
    int32_t mobile;
    int32_t pad_;
    int64_t np;
    double *X, *Y, *ux, *uy, *w;      /* np each */
    double *uhx, *uhy;                /* predictor velocity u^ (scratch, np each) */
    double *n, *Px, *Py;              /* nodal moments, (nx+1)*ny each */
    double *Fx, *Fy;                  /* nodal force, (nx+1)*ny each */
} orc_species;

typedef struct {
    double a0, omega, y0, w0, t_rise;
    double alpha;        /* angle of incidence in radians, Eq. 5 (Q22) */
    int32_t comp, pad_;
} orc_laser;

typedef struct {
    orc_grid g;
    int32_t nsp, nlaser;
    orc_species *sp;
    orc_laser *laser;
    double *a_new, *a_now, *a_old;    /* ncomp * (nx+1)*ny each */
    double *rho, *phi;                /* (nx+1)*ny */
    double *Ex, *Ey;                  /* nx*ny, cell centred */
    int64_t step;
} orc_state;

/* ------------------------------------------------------------------------------------------ */
/* O1. One-dimensional cumulative shape G(s), s in [0, DD] (cells), G(0)=0, G(DD)=1.
 * Sine cloud: Eq. 12-13.  Eq. 13 integrates the sine shape over [x1,x2] to
 * (1/2)[cos(pi x1 / 2D) - cos(pi x2 / 2D)] per axis, with 2D = DD the side length (Q1), so
 * G(s) = (1/2)[1 - cos(pi s / DD)].  CIC (uniform cloud, DD = 1 cell) and TSC (triangular cloud,
 * DD = 2 cells) are the textbook shapes of ref. [42], written the same way.           */
double orc_G(int shape, double DD, double s)
{
    if (s <= 0.0) return 0.0;
    if (s >= DD) return 1.0;
    if (shape == ORC_SINE) return 0.5 * (1.0 - cos(ORC_PI * s / DD));
    if (shape == ORC_CIC) return s / DD;               /* DD == 1 */
    /* TSC, DD == 2: density (per cell) rises linearly 0..1 on [0,1] and falls on [1,2] */
    if (s < 1.0) return 0.5 * s * s;
    return 1.0 - 0.5 * (2.0 - s) * (2.0 - s);
}

/* O1. Weights of one particle along one axis (the control volume of node i is
 * [i-1/2, i+1/2]; the weight is the integral of the normalised shape over the overlap, Eq. 13).
 * xp: particle centre in cells.  Returns the first node index; W[0..*count-1] are the weights of
 * nodes first, first+1, ...  At most 4 nodes can overlap for DD <= 2.                           */
int orc_weights_1d(int shape, double DD, double xp, double W[4], int *count)
{
    double xL = xp - 0.5 * DD;
    int first = (int)floor(xL + 0.5);          /* node whose control volume contains xL */
    int k;
    for (k = 0; k < 4; k++) {
        double node = (double)(first + k);
        double hi = node + 0.5 - xL, lo = node - 0.5 - xL;
        W[k] = orc_G(shape, DD, hi) - orc_G(shape, DD, lo);
    }
    *count = 4;
    return first;
}

/* Q9: fold a node index at the x walls (mirror), i -> -i, i -> 2nx - i. */
static int fold_x(int i, int nx)
{
    if (i < 0) i = -i;
    if (i > nx) i = 2 * nx - i;
    return i;
}
static int wrap_y(int j, int ny)
{
    j %= ny;
    if (j < 0) j += ny;
    return j;
}

/* O2. Deposit, Eq. 14, particles as the loop variable: density and
 * momentum ("densities and momentums").  Wall columns hold half a control volume, so
 * they are multiplied by 2 after the sum (Q9).                                                 */
void orc_deposit(const orc_grid *g, int shape, double DD, int64_t np, const double *X,
                 const double *Y, const double *ux, const double *uy, const double *w, double *n,
                 double *Px, double *Py)
{
    const int nx = g->nx, ny = g->ny;
    const int64_t nn = (int64_t)(nx + 1) * ny;
    int64_t p;
    int a, b, j;
    memset(n, 0, sizeof(double) * nn);
    memset(Px, 0, sizeof(double) * nn);
    memset(Py, 0, sizeof(double) * nn);
    for (p = 0; p < np; p++) {
        double Wx[4], Wy[4];
        int cx, cy;
        int i0 = orc_weights_1d(shape, DD, X[p], Wx, &cx);
        int j0 = orc_weights_1d(shape, DD, Y[p], Wy, &cy);
        for (a = 0; a < cx; a++) {
            if (Wx[a] == 0.0) continue;
            int i = fold_x(i0 + a, nx);
            for (b = 0; b < cy; b++) {
                if (Wy[b] == 0.0) continue;
                int64_t k = (int64_t)i * ny + wrap_y(j0 + b, ny);
                double ww = Wx[a] * Wy[b] * w[p];
                n[k] += ww;
                Px[k] += ww * ux[p];
                Py[k] += ww * uy[p];
            }
        }
    }
    for (j = 0; j < ny; j++) {
        n[j] *= 2.0; Px[j] *= 2.0; Py[j] *= 2.0;
        n[(int64_t)nx * ny + j] *= 2.0; Px[(int64_t)nx * ny + j] *= 2.0; Py[(int64_t)nx * ny + j] *= 2.0;
    }
}

/* O7. Gather, Eq. 15: force on a particle with the deposit weights and index fold. */
void orc_gather(const orc_grid *g, int shape, double DD, double Xp, double Yp, const double *Fx,
                const double *Fy, double *fx, double *fy)
{
    const int nx = g->nx, ny = g->ny;
    double Wx[4], Wy[4], sx = 0.0, sy = 0.0;
    int cx, cy, a, b;
    int i0 = orc_weights_1d(shape, DD, Xp, Wx, &cx);
    int j0 = orc_weights_1d(shape, DD, Yp, Wy, &cy);
    for (a = 0; a < cx; a++) {
        if (Wx[a] == 0.0) continue;
        int i = fold_x(i0 + a, nx);
        for (b = 0; b < cy; b++) {
            if (Wy[b] == 0.0) continue;
            int64_t k = (int64_t)i * ny + wrap_y(j0 + b, ny);
            sx += Wx[a] * Wy[b] * Fx[k];
            sy += Wx[a] * Wy[b] * Fy[k];
        }
    }
    *fx = sx;
    *fy = sy;
}

/* A3c (Fig. 1(a)).  "Assuming the direction of vector potential a has an angle of theta with respect to the
 * z-axis, then the components of a in the S-polarization direction (z direction) is a_sz = a cos(theta), and in the
 * P-polarization plane (x-y plane) is a_p = a sin(theta). if a_p has a angle of beta with respect to the x direction
 * ... a_px = a sin(theta) cos(beta) and a_py = a sin(theta) sin(beta)".  out[0] = a_sz, out[1] = a_px, out[2] = a_py;
 * the components of `a` are numbered 0 = z, 1 = x, 2 = y throughout.  Pin: the three axes of Fig. 1(a) and |a|. */
void orc_polarised(double a, double theta, double beta, double out[3])
{
    out[0] = a * cos(theta);
    out[1] = a * sin(theta) * cos(beta);
    out[2] = a * sin(theta) * sin(beta);
}

/* Incident wave, Eq. 4: a = a0 env(y) cos(omega t - k x), k = omega in vacuum, time in
 * T0 and x in lambda0 so the phase is 2 pi omega (t - x).  Turn-on (Q14): ramp(tau) =
 * sin^2(pi tau / (2 t_rise)) of the retarded time tau = t - x; t_rise = 0 is the paper's literal
 * substitution.  w0 <= 0: plane wave.
 * Oblique incidence, Eq. 5: (x, y) here are the box coordinates (the paper's x', y');
 * the beam coordinates that go into Eq. 4 are  xb = x cos(alpha) - y' sin(alpha),
 * yb = x sin(alpha) + y' cos(alpha), with y' measured from the beam centre y0 so that y0 stays
 * the centre of the beam on the boundary, and taken at the nearest periodic image (y is periodic
 * with period Ly) -- Q22.  The turn-on front is the plane t - xb = (Ly/2)|sin(alpha)|, the earliest
 * one that leaves the whole box field-free at t = 0 (the boundary reaches back to xb =
 * -(Ly/2)|sin(alpha)|); the carrier keeps the phase of Eq. 4.  alpha = 0 is the normal incidence of
 * P:L93, untouched.                                                                              */
double orc_a_inc(const orc_laser *L, double x, double y, double t, double Ly)
{
    double xb = x, yb = y - L->y0, tau, phase, env = 1.0, ramp = 1.0, lead = 0.0;
    if (L->alpha != 0.0) {
        double d = y - L->y0;
        d -= Ly * floor(d / Ly + 0.5);
        xb = x * cos(L->alpha) - d * sin(L->alpha);       /* Eq. 5 */
        yb = x * sin(L->alpha) + d * cos(L->alpha);
        lead = 0.5 * Ly * fabs(sin(L->alpha));
    }
    phase = t - xb;
    tau = phase - lead;
    if (tau <= 0.0) return 0.0;
    if (L->w0 > 0.0) {
        double r = yb / L->w0;
        env = exp(-r * r);
    }
    if (L->t_rise > 0.0 && tau < L->t_rise) {
        double s = sin(0.5 * ORC_PI * tau / L->t_rise);
        ramp = s * s;
    }
    return L->a0 * env * ramp * cos(2.0 * ORC_PI * L->omega * phase);
}

static double a_inc_sum(const orc_state *S, int comp, double x, double y, double t)
{
    double s = 0.0;
    int l;
    for (l = 0; l < S->nlaser; l++)
        if (S->laser[l].comp == comp) s += orc_a_inc(&S->laser[l], x, y, t, S->g.ny * S->g.dy);
    return s;
}

/* O3 + O4. Wave update for every active component: Eq. 6 on interior nodes, then
 * Eq. 8 solved for the boundary node (needs a^{n+1} at the neighbour), with
 * the incident wave split off at the left boundary.  t_now = n dt.                    */
void orc_field_step(orc_state *S, const double *ne, double t_now)
{
    const int nx = S->g.nx, ny = S->g.ny;
    const double dx = S->g.dx, dy = S->g.dy, dt = S->g.dt;
    const int64_t nn = (int64_t)(nx + 1) * ny;
    const double alpha = 1.0 / (2.0 * dt * dx), beta = 1.0 / (2.0 * dt * dt), gam = 1.0 / (4.0 * dy * dy);
    int c, i, j;
    for (c = 0; c < S->g.ncomp; c++) {
        double *ap = S->a_new + c * nn;
        const double *a = S->a_now + c * nn, *am = S->a_old + c * nn;
        for (i = 1; i < nx; i++)
            for (j = 0; j < ny; j++) {
                int jp = wrap_y(j + 1, ny), jm = wrap_y(j - 1, ny);
                int64_t k = (int64_t)i * ny + j;
                double lap = (a[k + ny] - 2.0 * a[k] + a[k - ny]) / (dx * dx) +
                             (a[(int64_t)i * ny + jp] - 2.0 * a[k] + a[(int64_t)i * ny + jm]) / (dy * dy);
                ap[k] = 2.0 * a[k] - am[k] + dt * dt * (lap - 4.0 * ORC_PI * ORC_PI * ne[k] * a[k]);
            }
        /* Eq. 8 rearranged for a_0^{n+1} (all terms of Eq. 8 kept, nothing else):
         *   alpha[(a1p - a1m) - (a0p - a0m)] - beta[(a0p - 2a0 + a0m) + (a1p - 2a1 + a1m)]
         *   + gam (D0 + D1) = 0 ,  D_i = a_{i,j+1} - 2 a_{i,j} + a_{i,j-1} at level n.          */
        for (j = 0; j < ny; j++) {
            int jp = wrap_y(j + 1, ny), jm = wrap_y(j - 1, ny);
            double y = j * dy, yp = jp * dy, ym = jm * dy;
            /* left: scattered part s = a - a_inc at i = 0, 1 */
            double s0 = a[j] - a_inc_sum(S, c, 0.0, y, t_now);
            double s0m = am[j] - a_inc_sum(S, c, 0.0, y, t_now - dt);
            double s1 = a[ny + j] - a_inc_sum(S, c, dx, y, t_now);
            double s1m = am[ny + j] - a_inc_sum(S, c, dx, y, t_now - dt);
            double s1p = ap[ny + j] - a_inc_sum(S, c, dx, y, t_now + dt);
            double D0 = (a[jp] - a_inc_sum(S, c, 0.0, yp, t_now)) - 2.0 * s0 +
                        (a[jm] - a_inc_sum(S, c, 0.0, ym, t_now));
            double D1 = (a[ny + jp] - a_inc_sum(S, c, dx, yp, t_now)) - 2.0 * s1 +
                        (a[ny + jm] - a_inc_sum(S, c, dx, ym, t_now));
            double s0p = (alpha * (s1p - s1m + s0m) - beta * (s1p + s1m + s0m - 2.0 * s0 - 2.0 * s1) +
                          gam * (D0 + D1)) / (alpha + beta);
            ap[j] = s0p + a_inc_sum(S, c, 0.0, y, t_now + dt);
            /* right: mirror image, no incident wave */
            {
                int64_t r0 = (int64_t)nx * ny, r1 = (int64_t)(nx - 1) * ny;
                double E0 = a[r0 + jp] - 2.0 * a[r0 + j] + a[r0 + jm];
                double E1 = a[r1 + jp] - 2.0 * a[r1 + j] + a[r1 + jm];
                ap[r0 + j] = (alpha * (ap[r1 + j] - am[r1 + j] + am[r0 + j]) -
                              beta * (ap[r1 + j] + am[r1 + j] + am[r0 + j] - 2.0 * a[r0 + j] - 2.0 * a[r1 + j]) +
                              gam * (E0 + E1)) / (alpha + beta);
            }
        }
        if (S->g.bc_y == 1) {
            /* "the second-order absorbing boundary condition ... on all of four boundaries": Eq. 8 with the
             * roles of x and y exchanged on the walls j = 0 and j = ny-1 (no incident wave there), for i = 1..nx-1;
             * it overwrites what the periodic stencil and the x-wall loop above left in those two columns.  The
             * corners are not treated by the paper: first-order outgoing condition along the diagonal (Q23).   */
            const double alpha_y = 1.0 / (2.0 * dt * dy), gam_x = 1.0 / (4.0 * dx * dx);
            const double hd = sqrt(dx * dx + dy * dy), kap = (dt - hd) / (dt + hd);
            int side;
            for (side = 0; side < 2; side++) {
                const int j0 = side ? ny - 1 : 0, j1 = side ? ny - 2 : 1;
                for (i = 1; i < nx; i++) {
                    int64_t k0 = (int64_t)i * ny + j0, k1 = (int64_t)i * ny + j1;
                    double D0 = a[k0 + ny] - 2.0 * a[k0] + a[k0 - ny];
                    double D1 = a[k1 + ny] - 2.0 * a[k1] + a[k1 - ny];
                    ap[k0] = (alpha_y * (ap[k1] - am[k1] + am[k0]) -
                              beta * (ap[k1] + am[k1] + am[k0] - 2.0 * a[k0] - 2.0 * a[k1]) + gam_x * (D0 + D1)) /
                             (alpha_y + beta);
                }
                /* corners: a_c^{n+1} = a_d^n + kappa (a_d^{n+1} - a_c^n), d the diagonal neighbour */
                ap[j0] = a[ny + j1] + kap * (ap[ny + j1] - a[j0]);
                ap[(int64_t)nx * ny + j0] = a[(int64_t)(nx - 1) * ny + j1] + kap * (ap[(int64_t)(nx - 1) * ny + j1] - a[(int64_t)nx * ny + j0]);
            }
        }
    }
}

/* Textbook iterative radix-2 FFT (Cooley-Tukey), in place, n a power of two.
 * sign = -1: forward  sum x_j e^{-2 pi i jl/n};  sign = +1: inverse without the 1/n.            */
void orc_fft(double *re, double *im, int n, int sign)
{
    int i, j = 0, len;
    for (i = 1; i < n; i++) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double t = re[i]; re[i] = re[j]; re[j] = t;
            t = im[i]; im[i] = im[j]; im[j] = t;
        }
    }
    for (len = 2; len <= n; len <<= 1) {
        double ang = sign * 2.0 * ORC_PI / len;
        for (i = 0; i < n; i += len) {
            int k;
            for (k = 0; k < len / 2; k++) {
                double wr = cos(ang * k), wi = sin(ang * k);
                int p = i + k, q = i + k + len / 2;
                double xr = re[q] * wr - im[q] * wi, xi = re[q] * wi + im[q] * wr;
                re[q] = re[p] - xr; im[q] = im[p] - xi;
                re[p] += xr; im[p] += xi;
            }
        }
    }
}

/* The definition the FFT must equal: O(n^2) DFT (used by the tests to pin orc_fft). */
void orc_dft(const double *re, const double *im, double *ore, double *oim, int n, int sign)
{
    int l, j;
    for (l = 0; l < n; l++) {
        double sr = 0.0, si = 0.0;
        for (j = 0; j < n; j++) {
            double ang = sign * 2.0 * ORC_PI * (double)((int64_t)j * l % n) / n;
            sr += re[j] * cos(ang) - im[j] * sin(ang);
            si += re[j] * sin(ang) + im[j] * cos(ang);
        }
        ore[l] = sr; oim[l] = si;
    }
}

/* O5. Poisson, Eqs. 9-11: Fourier series in y with the continuous wavenumber
 * k_y = 2 pi l / L_y (Eq. 10), central differences in x (Eq. 11), one tridiagonal system per l
 * solved by the chasing (Thomas) method; phi^ = 0 on both x walls for every l (Q5).
 * use_dft != 0 replaces the FFT by the O(n^2) definition (small grids, tests).                 */
void orc_poisson(const orc_grid *g, const double *rho, double *phi, int use_dft)
{
    const int nx = g->nx, ny = g->ny;
    const double dx = g->dx, Ly = g->ny * g->dy;
    const int64_t nn = (int64_t)(nx + 1) * ny;
    double *hr = (double *)calloc(nn, sizeof(double)), *hi = (double *)calloc(nn, sizeof(double));
    double *tr = (double *)malloc(sizeof(double) * ny), *ti = (double *)malloc(sizeof(double) * ny);
    double *cp = (double *)malloc(sizeof(double) * (nx + 1));
    double *dr = (double *)malloc(sizeof(double) * (nx + 1)), *di = (double *)malloc(sizeof(double) * (nx + 1));
    int i, j, l;
    for (i = 0; i <= nx; i++) {
        for (j = 0; j < ny; j++) { hr[(int64_t)i * ny + j] = rho[(int64_t)i * ny + j]; hi[(int64_t)i * ny + j] = 0.0; }
        if (use_dft) {
            orc_dft(hr + (int64_t)i * ny, hi + (int64_t)i * ny, tr, ti, ny, -1);
            memcpy(hr + (int64_t)i * ny, tr, sizeof(double) * ny);
            memcpy(hi + (int64_t)i * ny, ti, sizeof(double) * ny);
        } else
            orc_fft(hr + (int64_t)i * ny, hi + (int64_t)i * ny, ny, -1);
    }
    for (l = 0; l < ny; l++) {
        int ls = (l <= ny / 2) ? l : l - ny;                 /* l = -N/2 .. N/2 (Eq. 10) */
        double ky = 2.0 * ORC_PI * ls / Ly;
        double b = -2.0 - ky * ky * dx * dx;                 /* Eq. 11 times dx^2 */
        /* unknowns i = 1..nx-1, sub = super = 1, diag = b, rhs = dx^2 rho^_i */
        cp[1] = 1.0 / b;
        dr[1] = dx * dx * hr[(int64_t)1 * ny + l] / b;
        di[1] = dx * dx * hi[(int64_t)1 * ny + l] / b;
        for (i = 2; i < nx; i++) {
            double m = b - cp[i - 1];
            cp[i] = 1.0 / m;
            dr[i] = (dx * dx * hr[(int64_t)i * ny + l] - dr[i - 1]) / m;
            di[i] = (dx * dx * hi[(int64_t)i * ny + l] - di[i - 1]) / m;
        }
        hr[l] = hi[l] = 0.0;
        hr[(int64_t)nx * ny + l] = hi[(int64_t)nx * ny + l] = 0.0;
        if (nx >= 2) {
            hr[(int64_t)(nx - 1) * ny + l] = dr[nx - 1];
            hi[(int64_t)(nx - 1) * ny + l] = di[nx - 1];
            for (i = nx - 2; i >= 1; i--) {
                hr[(int64_t)i * ny + l] = dr[i] - cp[i] * hr[(int64_t)(i + 1) * ny + l];
                hi[(int64_t)i * ny + l] = di[i] - cp[i] * hi[(int64_t)(i + 1) * ny + l];
            }
        }
    }
    for (i = 0; i <= nx; i++) {
        if (use_dft) {
            orc_dft(hr + (int64_t)i * ny, hi + (int64_t)i * ny, tr, ti, ny, +1);
            for (j = 0; j < ny; j++) phi[(int64_t)i * ny + j] = tr[j] / ny;
        } else {
            orc_fft(hr + (int64_t)i * ny, hi + (int64_t)i * ny, ny, +1);
            for (j = 0; j < ny; j++) phi[(int64_t)i * ny + j] = hr[(int64_t)i * ny + j] / ny;
        }
    }
    free(hr); free(hi); free(tr); free(ti); free(cp); free(dr); free(di);
}

/* O5 (second half). Cell-centred E, with E = -grad phi (Q2). */
void orc_efield(const orc_grid *g, const double *phi, double *Ex, double *Ey)
{
    const int nx = g->nx, ny = g->ny;
    int i, j;
    for (i = 0; i < nx; i++)
        for (j = 0; j < ny; j++) {
            int jp = wrap_y(j + 1, ny);
            double p00 = phi[(int64_t)i * ny + j], p01 = phi[(int64_t)i * ny + jp];
            double p10 = phi[(int64_t)(i + 1) * ny + j], p11 = phi[(int64_t)(i + 1) * ny + jp];
            Ex[(int64_t)i * ny + j] = -0.5 * ((p11 - p01) / g->dx + (p10 - p00) / g->dx);
            Ey[(int64_t)i * ny + j] = -0.5 * ((p11 - p10) / g->dy + (p01 - p00) / g->dy);
        }
}

/* central difference of a nodal array, one-sided at the x walls (O6) */
static double ddx(const double *q, int i, int j, int nx, int ny, double dx)
{
    if (i == 0) return (q[(int64_t)ny + j] - q[j]) / dx;
    if (i == nx) return (q[(int64_t)nx * ny + j] - q[(int64_t)(nx - 1) * ny + j]) / dx;
    return (q[(int64_t)(i + 1) * ny + j] - q[(int64_t)(i - 1) * ny + j]) / (2.0 * dx);
}
static double ddy(const double *q, int i, int j, int ny, double dy)
{
    return (q[(int64_t)i * ny + wrap_y(j + 1, ny)] - q[(int64_t)i * ny + wrap_y(j - 1, ny)]) / (2.0 * dy);
}

/* O6. Fluid force on the nodes, Eq. 16 / 18, from Eq. 2:
 *   F_e = 4 pi^2 E - (1/2) grad(sum_c a_c^2) - C v_eth^2 grad(n_e) / n_e
 *   F_i = -(4 pi^2 / m_i) E - C v_ith^2 grad(n_i) / n_i
 * written for a species of charge sign q and mass m as  -q (4 pi^2 / m) E, the ponderomotive
 * term for electrons only (P:L62 has none for ions).  E at a node = mean of the adjacent cell
 * centres (Q3); gradients central, one-sided at the x walls; pressure term 0 where n = 0 (Q10). */
void orc_force(const orc_grid *g, const orc_species *s, const double *a, const double *Ex,
               const double *Ey, double *Fx, double *Fy)
{
    const int nx = g->nx, ny = g->ny;
    const int64_t nn = (int64_t)(nx + 1) * ny;
    const double fourpi2 = 4.0 * ORC_PI * ORC_PI;
    double *a2 = (double *)calloc(nn, sizeof(double));
    int i, j, c;
    int64_t k;
    for (c = 0; c < g->ncomp; c++)
        for (k = 0; k < nn; k++) a2[k] += a[c * nn + k] * a[c * nn + k];
    for (i = 0; i <= nx; i++)
        for (j = 0; j < ny; j++) {
            int jm = wrap_y(j - 1, ny), cnt = 0;
            double ex = 0.0, ey = 0.0, fx, fy;
            k = (int64_t)i * ny + j;
            if (i > 0) {
                ex += Ex[(int64_t)(i - 1) * ny + jm] + Ex[(int64_t)(i - 1) * ny + j];
                ey += Ey[(int64_t)(i - 1) * ny + jm] + Ey[(int64_t)(i - 1) * ny + j];
                cnt += 2;
            }
            if (i < nx) {
                ex += Ex[(int64_t)i * ny + jm] + Ex[(int64_t)i * ny + j];
                ey += Ey[(int64_t)i * ny + jm] + Ey[(int64_t)i * ny + j];
                cnt += 2;
            }
            ex /= cnt; ey /= cnt;
            fx = -(double)s->sign * fourpi2 / s->mass * ex;
            fy = -(double)s->sign * fourpi2 / s->mass * ey;
            if (s->sign < 0) {
                fx -= 0.5 * ddx(a2, i, j, nx, ny, g->dx);
                fy -= 0.5 * ddy(a2, i, j, ny, g->dy);
            }
            if (s->n[k] > 0.0) {
                fx -= s->C * s->vth2 * ddx(s->n, i, j, nx, ny, g->dx) / s->n[k];
                fy -= s->C * s->vth2 * ddy(s->n, i, j, ny, g->dy) / s->n[k];
            }
            Fx[k] = fx; Fy[k] = fy;
        }
    free(a2);
}

static void charge_density(const orc_state *S, double *rho)
{
    const int64_t nn = (int64_t)(S->g.nx + 1) * S->g.ny;
    int64_t k;
    int s;
    for (k = 0; k < nn; k++) rho[k] = 0.0;
    for (s = 0; s < S->nsp; s++)
        for (k = 0; k < nn; k++) rho[k] += (double)S->sp[s].sign * S->sp[s].n[k];   /* n_i - n_e */
}

static void deposit_species(const orc_state *S, orc_species *s, const double *ux, const double *uy,
                            const double *X, const double *Y)
{
    orc_deposit(&S->g, s->shape, s->DD, s->np, X, Y, ux, uy, s->w, s->n, s->Px, s->Py);
}

/* Item (1) of the flow for step 0: deposit every mobile species from (x^0, u^0). */
void orc_initial_deposit(orc_state *S)
{
    int s;
    for (s = 0; s < S->nsp; s++)
        if (S->sp[s].mobile) deposit_species(S, &S->sp[s], S->sp[s].ux, S->sp[s].uy, S->sp[s].X, S->sp[s].Y);
}


/* Eq. 17: predictor.  h = dt / (2 dx) converts (u^ + u) to cells. */
void orc_predictor(double dt, double h, double x, double u, double F, double *uh, double *xh)
{
    *uh = u + dt * F;
    *xh = x + h * (*uh + u);
}
/* Eq. 19: corrector. */
void orc_corrector(double dt, double h, double x, double u, double uh, double Fh, double *un, double *xn)
{
    *un = 0.5 * (uh + u) + 0.5 * dt * Fh;
    *xn = x + h * (*un + u);
}

/* rho^n, phi^n, E^n from the densities currently on the grids (used by the diagnostics so that
 * the energy terms refer to one time level). */
void orc_refresh_fields(orc_state *S)
{
    charge_density(S, S->rho);
    orc_poisson(&S->g, S->rho, S->phi, 0);
    orc_efield(&S->g, S->phi, S->Ex, S->Ey);
}

/* O8. One time step, items (1)-(8) of P:L229-238.  Item (1) of this step is item-(8)-deposit of
 * the previous one (or orc_initial_deposit): s->n holds n^n on entry and n^{n+1} on exit.      */
void orc_step(orc_state *S)
{
    const orc_grid *g = &S->g;
    const int nx = g->nx, ny = g->ny;
    const int64_t nn = (int64_t)(nx + 1) * ny;
    /* Q21: the particles advance with dt = S dt_wave; the wave equation takes S steps of
     * dt_wave per particle step with the electron density of item (1) held fixed                 */
    const int nsub = g->subcycle > 1 ? g->subcycle : 1;
    const double dt = nsub * g->dt;
    const double hx = dt / (2.0 * g->dx), hy = dt / (2.0 * g->dy);   /* cells per unit u */
    double *Xh = NULL, *Yh = NULL, *ne, *a_n;
    int s, sub;
    int64_t p, k;

    /* electron density for the wave source: sum over negative species */
    ne = (double *)calloc(nn, sizeof(double));
    for (s = 0; s < S->nsp; s++)
        if (S->sp[s].sign < 0)
            for (k = 0; k < nn; k++) ne[k] += S->sp[s].n[k];

    /* (2) a^{n+1} from a^n, a^{n-1}, n_e^n (Eq. 6, 8): S wave steps, a^n kept for item (3);
     * E^n from n_i^n - n_e^n (Eqs. 9-11) */
    a_n = (double *)malloc(sizeof(double) * g->ncomp * nn);
    memcpy(a_n, S->a_now, sizeof(double) * g->ncomp * nn);
    for (sub = 0; sub < nsub; sub++) {
        orc_field_step(S, ne, (double)(S->step * nsub + sub) * g->dt);
        if (sub + 1 < nsub) {
            double *t = S->a_old;
            S->a_old = S->a_now; S->a_now = S->a_new; S->a_new = t;
        }
    }
    charge_density(S, S->rho);
    orc_poisson(g, S->rho, S->phi, 0);
    orc_efield(g, S->phi, S->Ex, S->Ey);

    /* (3) F^n with a^n (Eq. 16), gathered at x^n (Eq. 15); (4) predictor, Eq. 17 */
    for (s = 0; s < S->nsp; s++) {
        orc_species *q = &S->sp[s];
        if (!q->mobile) continue;
        orc_force(g, q, a_n, S->Ex, S->Ey, q->Fx, q->Fy);
    }
    free(a_n);
    for (s = 0; s < S->nsp; s++) {
        orc_species *q = &S->sp[s];
        if (!q->mobile) continue;
        Xh = (double *)malloc(sizeof(double) * (q->np > 0 ? q->np : 1));
        Yh = (double *)malloc(sizeof(double) * (q->np > 0 ? q->np : 1));
        for (p = 0; p < q->np; p++) {
            double fx, fy;
            orc_gather(g, q->shape, q->DD, q->X[p], q->Y[p], q->Fx, q->Fy, &fx, &fy);
            orc_predictor(dt, hx, q->X[p], q->ux[p], fx, &q->uhx[p], &Xh[p]);
            orc_predictor(dt, hy, q->Y[p], q->uy[p], fy, &q->uhy[p], &Yh[p]);
        }
        /* (5) n^, P^ from (x^, u^) (Eq. 14) */
        deposit_species(S, q, q->uhx, q->uhy, Xh, Yh);
        /* keep x^ for stage 2: store in place of scratch by recomputing below */
        free(Xh); free(Yh);
    }
    /* (6) E^{n+1} */
    charge_density(S, S->rho);
    orc_poisson(g, S->rho, S->phi, 0);
    orc_efield(g, S->phi, S->Ex, S->Ey);
    /* (7) F^{n+1} with a^{n+1} and n^ (Eq. 18), gathered at x^ (Q4); (8) corrector, Eq. 19 */
    for (s = 0; s < S->nsp; s++) {
        orc_species *q = &S->sp[s];
        if (!q->mobile) continue;
        orc_force(g, q, S->a_new, S->Ex, S->Ey, q->Fx, q->Fy);
    }
    for (s = 0; s < S->nsp; s++) {
        orc_species *q = &S->sp[s];
        if (!q->mobile) continue;
        for (p = 0; p < q->np; p++) {
            double fx, fy, xh, yh, unx, uny, xn, yn;
            xh = q->X[p] + hx * (q->uhx[p] + q->ux[p]);     /* x^ of Eq. 17 again */
            yh = q->Y[p] + hy * (q->uhy[p] + q->uy[p]);
            orc_gather(g, q->shape, q->DD, xh, yh, q->Fx, q->Fy, &fx, &fy);
            orc_corrector(dt, hx, q->X[p], q->ux[p], q->uhx[p], fx, &unx, &xn);
            orc_corrector(dt, hy, q->Y[p], q->uy[p], q->uhy[p], fy, &uny, &yn);
            /* particle boundaries (Q9): reflect at the x walls, wrap in y */
            if (xn < 0.0) { xn = -xn; unx = -unx; }
            if (xn > (double)nx) { xn = 2.0 * nx - xn; unx = -unx; }
            yn -= floor(yn / ny) * ny;
            if (yn >= (double)ny) yn -= ny;
            q->X[p] = xn; q->Y[p] = yn; q->ux[p] = unx; q->uy[p] = uny;
        }
        /* item (1) of the next step */
        deposit_species(S, q, q->ux, q->uy, q->X, q->Y);
    }
    /* rotate time levels of a */
    {
        double *t = S->a_old;
        S->a_old = S->a_now; S->a_now = S->a_new; S->a_new = t;
    }
    S->step += 1;
    free(ne);
}

/* O9 / Q11. Energy terms of the invariant of Eqs. 1-3, per unit dx*dy, in m_e c^2 n_c lambda0^2
 * / (dx dy).  out[0] = W_es = 2 pi^2 sum_cells |E|^2; out[1] = W_int = (1/2) sum n_e |a|^2;
 * out[2] = W_em = (1/8 pi^2) sum (|d_t a|^2 + |grad a|^2)  (d_t a between levels now and old,
 * grad a at level now, forward differences);  out[3+2s] = W_kin[s] = sum_p (1/2) m w |u|^2;
 * out[4+2s] = W_th[s] = m C v_th^2 sum n ln n.  Node sums carry half weight on the wall columns. */
void orc_energies(const orc_state *S, double *out)
{
    const orc_grid *g = &S->g;
    const int nx = g->nx, ny = g->ny;
    const int64_t nn = (int64_t)(nx + 1) * ny;
    int i, j, s, c;
    int64_t k, p;
    double wes = 0.0, wint = 0.0, wem = 0.0;
    for (k = 0; k < (int64_t)nx * ny; k++) wes += S->Ex[k] * S->Ex[k] + S->Ey[k] * S->Ey[k];
    out[0] = 2.0 * ORC_PI * ORC_PI * wes;
    for (i = 0; i <= nx; i++)
        for (j = 0; j < ny; j++) {
            double vol = (i == 0 || i == nx) ? 0.5 : 1.0, ne = 0.0, a2 = 0.0;
            k = (int64_t)i * ny + j;
            for (s = 0; s < S->nsp; s++)
                if (S->sp[s].sign < 0) ne += S->sp[s].n[k];
            for (c = 0; c < g->ncomp; c++) {
                double a = S->a_now[c * nn + k], am = S->a_old[c * nn + k];
                double at = (a - am) / g->dt;
                double ay = (S->a_now[c * nn + (int64_t)i * ny + wrap_y(j + 1, ny)] - a) / g->dy;
                a2 += a * a;
                wem += vol * (at * at + ay * ay);
                if (i < nx) {
                    double ax = (S->a_now[c * nn + k + ny] - a) / g->dx;
                    wem += ax * ax;
                }
            }
            wint += 0.5 * vol * ne * a2;
        }
    out[1] = wint;
    out[2] = wem / (8.0 * ORC_PI * ORC_PI);
    for (s = 0; s < S->nsp; s++) {
        const orc_species *q = &S->sp[s];
        double wk = 0.0, wt = 0.0;
        if (q->mobile)
            for (p = 0; p < q->np; p++) wk += 0.5 * q->mass * q->w[p] * (q->ux[p] * q->ux[p] + q->uy[p] * q->uy[p]);
        for (i = 0; i <= nx; i++)
            for (j = 0; j < ny; j++) {
                double vol = (i == 0 || i == nx) ? 0.5 : 1.0;
                double n = q->n[(int64_t)i * ny + j];
                if (n > 0.0) wt += vol * n * log(n);
            }
        out[3 + 2 * s] = wk;
        out[4 + 2 * s] = q->mass * q->C * q->vth2 * wt;
    }
}
