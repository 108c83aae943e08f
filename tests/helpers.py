"""Shared test helpers: build an Oracle (CPU) from a pm2d_inputs config."""
import numpy as np

import oracle
import oracle.loader as L
import pm2d_inputs as I


def oracle_from_config(cfg, particles=None):
    return oracle.from_config(cfg, particles)


# ---- quasi-1D SRS slab (paper section 6.1: a0 = 0.06, 0.15 n_c, dx = 0.05, dt = 0.035, 1 particle per cell,
# DD = 1.6 dx), cold and with the pressure term off so that the vacuum edges stay put
def srs_slab(nx=1600, ny=8, dx=0.05, n0=0.15, seed=1, ripple=0.0, k_ripple=0.0):
    """Particles (canonical form) of a slab with 8 lambda0 vacuum margins and 5 lambda0 sin^2 ramps, one per
    cell at the cell centre plus 1e-3 cell of seeded position noise in x.  ripple > 0: plus a coherent displacement
    ripple * sin(2 pi k_ripple x) cells (k_ripple in 1/lambda0), a plasma-wave seed far above the rounding noise of
    a float32 run."""
    def prof(x_cells):
        x, Lx, r = x_cells * dx, nx * dx, 5.0
        up, dn = np.clip((x - 8.0) / r, 0, 1), np.clip((Lx - 8.0 - x) / r, 0, 1)
        return n0 * np.sin(0.5 * np.pi * up) ** 2 * np.sin(0.5 * np.pi * dn) ** 2
    ix, iy = [a.ravel() for a in np.meshgrid(np.arange(nx), np.arange(ny), indexing="ij")]
    w = prof(ix + 0.5)
    keep = w > 0
    ix, iy, w = ix[keep].astype(np.int32), iy[keep].astype(np.int32), w[keep].astype(np.float32)
    rng = np.random.default_rng(seed)
    disp = 1e-3 * rng.standard_normal(ix.size) + ripple * np.sin(2.0 * np.pi * k_ripple * (ix + 0.5) * dx)
    fx = (np.floor((0.5 + disp) * 2 ** 24) / 2 ** 24).astype(np.float32)
    z = np.zeros(ix.size, np.float32)
    return dict(ix=ix, iy=iy, fx=fx, fy=np.full(ix.size, 0.5, np.float32), ux=z, uy=z.copy(), w=w)


def srs_oracle(parts, nx, ny, dx=0.05, dt=0.035, a0=0.06, DD=1.6):
    X = parts["ix"] + parts["fx"].astype(np.float64)
    Y = parts["iy"] + parts["fy"].astype(np.float64)
    w = parts["w"].astype(np.float64)
    g = oracle.make_grid(nx, ny, dx, dx, dt)
    n_bg, _, _ = oracle.deposit(g, oracle.SINE, DD, X, Y, 0 * X, 0 * X, w)
    sp = [dict(sign=-1, mass=1.0, T_keV=0.0, C=0.0, shape=oracle.SINE, DD=DD, mobile=1, X=X, Y=Y, ux=0 * X, uy=0 * X, w=w),
          dict(sign=1, mass=1836.0, T_keV=0.0, mobile=0, shape=oracle.SINE, DD=DD, n_fixed=n_bg)]
    laser = dict(a0=a0, omega=1.0, y0=0.0, w0=0.0, t_rise=5.0, comp=0)
    return oracle.Oracle(nx, ny, dx, dx, dt, sp, [laser]), laser


def backscatter_growth_rate(t, scattered, dt=0.035, lo=2e-4, hi=2e-2):
    """Log-slope (per T0) of the rms envelope (2 T0 windows) of the scattered field at the left boundary
     while it rises from `lo` to `hi`."""
    win = int(round(2.0 / dt))
    env = np.array([np.sqrt(np.mean(scattered[i:i + win] ** 2)) for i in range(0, len(scattered) - win, win)])
    te = t[::win][:len(env)]
    i0, i1 = int(np.argmax(env > lo)), int(np.argmax(env > hi))
    assert i1 - i0 >= 10, "no clean exponential phase"
    return float(np.polyfit(te[i0:i1], np.log(env[i0:i1]), 1)[0])
