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


# ---- the lane storage order (include/pm2d.h, pm2d_rebin) as a numpy specification: the GPU test
# checks the device's permutation against it bit for bit, tests/test_lane_order_spec.py checks on the CPU what the order is for
def rank_in_group(group_sorted):
    """rank of every element inside its run of equal values (the array is sorted by group)"""
    n = group_sorted.size
    start = np.r_[0, np.flatnonzero(np.diff(group_sorted)) + 1]
    return np.arange(n) - np.repeat(start, np.diff(np.r_[start, n]))


def lane_order_perm(pp, T, nx, ny, subs, predx=0.0, predy=0.0):
    """The lane order as include/pm2d.h states it for pm2d_rebin, written out with numpy's stable sorts.
    -> (perm, key) with key = destination tile * T^2 + cell of the sort position."""
    n = pp["ix"].size
    nty = (ny + T - 1) // T

    def sort_pos(i, f, u, pred):            # global, 2^-24 cells: position + free flight of half a rebin period
        v = i.astype(np.int64) * 2 ** 24 + np.round(f.astype(np.float64) * 2 ** 24).astype(np.int64)
        return v + np.rint((u.astype(np.float32) * np.float32(pred)).astype(np.float64)).astype(np.int64)
    xg = np.clip(sort_pos(pp["ix"], pp["fx"], pp["ux"], predx), 0, nx * 2 ** 24 - 1)     # beyond a wall: stays in the wall tile
    yg = sort_pos(pp["iy"], pp["fy"], pp["uy"], predy) % (ny * 2 ** 24)                  # y is periodic
    tile = ((xg >> 24) // T) * nty + (yg >> 24) // T
    xs, ys = xg - ((xg >> 24) // T) * T * 2 ** 24, yg - ((yg >> 24) // T) * T * 2 ** 24
    cx, cy, fx24, fy24 = xs >> 24, ys >> 24, xs & (2 ** 24 - 1), ys & (2 ** 24 - 1)
    h = (cx >> 4) if subs == 2 else np.zeros_like(cx)
    key_a = (h << 10) | (cy << 5) | (fy24 >> 19)
    xb = (((cx & 15) << 1) | (fx24 >> 23)) if subs == 2 else cx
    o1 = np.argsort(tile, kind="stable")                                   # the tile pass
    t1, ka, xb1, h1 = tile[o1], key_a[o1], xb[o1], h[o1]
    tstart = np.searchsorted(t1, np.arange(t1.max() + 2))                  # first slot of every tile
    n0 = np.bincount(t1[h1 == 0], minlength=t1.max() + 1)                  # particles of sub-tile 0
    oa = np.lexsort((ka, t1))
    rho = np.empty(n, np.int64)
    rho[oa] = rank_in_group(t1[oa])
    hb = np.where(h1 == 1, n0[t1], 0)
    nh = np.where(h1 == 1, (tstart[t1 + 1] - tstart[t1]) - n0[t1], n0[t1])
    rho_h = rho - hb
    base, rem = nh // 32, nh % 32
    cut = rem * (base + 1)
    slab = np.where(rho_h < cut, rho_h // (base + 1), rem + (rho_h - cut) // np.maximum(base, 1))
    key_b = (h1 << 10) | (slab << 5) | xb1
    ob = np.lexsort((key_b, t1))
    rb = np.empty(n, np.int64)
    rb[ob] = rank_in_group(t1[ob])
    w = rb - hb - (slab * base + np.minimum(slab, rem))
    q = tstart[t1] + hb + 32 * w + slab
    perm = np.empty(n, np.int64)
    perm[q] = o1
    return perm, tile * (T * T) + cx * T + cy
