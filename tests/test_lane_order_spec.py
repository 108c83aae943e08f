"""What the lane storage order is for, checked on the CPU with its numpy specification (tests/helpers.py lane_order_perm: the
GPU test test_rebin_is_a_stable_counting_sort[lanes] holds the device's permutation to it bit for bit).  DESIGN.md sections 5,
6.1c: lane i of every warp works y-slab i of a sub-tile and owns bank i + b of shifted copies of the shared windows, so the
fused stage kernel has no bank conflicts as long as a particle's nearest node column stays within m = cy - i in -1..2 of
its lane; sorting by the position half a rebin period ahead keeps it there."""
import math

import numpy as np

import oracle.loader as L
import pm2d_inputs as I
from helpers import lane_order_perm

T = 32


def _particles(nx=64, ny=64, seed=2):
    cfg = I.config("c3", nx=nx, ny=ny)
    cfg["seed"] = seed
    cfg["profile"]["taper_cells"] = 0
    return cfg, L.generate_particles(cfg, 0)            # electrons: 4 per cell, 3 keV


def _lanes(cfg, p, every):
    """Slot of every particle in the lane order of a period of `every` steps -> (tile, sub-tile, lane, rank in slab)."""
    g = cfg["grid"]
    pred = [every * g["dt"] / (2.0 * g[d]) * 2.0 ** 24 for d in ("dx", "dy")]
    perm, key = lane_order_perm(p, T, g["nx"], g["ny"], 2, pred[0], pred[1])
    slot = np.empty(perm.size, np.int64)
    slot[perm] = np.arange(perm.size)                   # perm[q] = old index of the particle at slot q
    tile = key // (T * T)
    cx = (key % (T * T)) // T
    sub = cx >> 4
    # slots of a tile are contiguous, sub-tile 0 first: position inside the sub-tile
    order = np.lexsort((slot, sub, tile))
    grp = tile[order] * 2 + sub[order]
    start = np.r_[0, np.flatnonzero(np.diff(grp)) + 1]
    pos = np.empty(perm.size, np.int64)
    pos[order] = np.arange(perm.size) - np.repeat(start, np.diff(np.r_[start, perm.size]))
    return perm, tile, sub, pos & 31, pos >> 5


def test_lane_order_is_a_permutation_with_balanced_slabs():
    """Every particle gets exactly one slot; inside a sub-tile the 32 slabs (= lanes) hold populations that differ by at most
    one; a slab is a contiguous range in y, and inside it the particles are in x order (by half-cell bins)."""
    cfg, p = _particles()
    perm, tile, sub, lane, w = _lanes(cfg, p, 16)
    assert np.array_equal(np.sort(perm), np.arange(perm.size))
    g = cfg["grid"]
    y = p["iy"] + p["fy"].astype(np.float64) + p["uy"].astype(np.float64) * 16 * g["dt"] / (2 * g["dy"])
    x = p["ix"] + p["fx"].astype(np.float64) + p["ux"].astype(np.float64) * 16 * g["dt"] / (2 * g["dx"])
    x = np.clip(x, 0.0, g["nx"] - 1e-9)                                  # a sort position beyond a wall stays in the wall tile
    for t in np.unique(tile):
        for h in (0, 1):
            m = (tile == t) & (sub == h)
            cnt = np.bincount(lane[m], minlength=32)
            assert cnt.max() - cnt.min() <= 1
            yy, ll = y[m] % g["ny"], lane[m]
            hi = np.array([yy[ll == k].max() for k in range(32)])
            lo = np.array([yy[ll == k].min() for k in range(32)])
            assert (lo[1:] >= hi[:-1] - 1.0 / 32 - 1e-6).all()           # slabs are cut from the y order (1/32-cell bins)
            for k in (0, 13, 31):
                xs, ws = x[m][ll == k], w[m][ll == k]
                o = np.argsort(ws)
                assert (np.diff(np.floor(2 * xs[o])) >= 0).all()         # rank in the slab follows x (half-cell bins)


def _out_of_lane_fraction(cfg, p, every, steps):
    """Free flight for `steps` steps after a sort for a period of `every`: fraction of the (particle, step) visits whose
    nearest node column is outside the four window copies of the particle's lane (m = cy - lane not in -1..2), or whose
    nearest node row has left the window of its sub-tile (2 halo rows)."""
    g = cfg["grid"]
    _, tile, sub, lane, _ = _lanes(cfg, p, every)
    nty = g["ny"] // T
    x0 = p["ix"] + p["fx"].astype(np.float64)
    y0 = p["iy"] + p["fy"].astype(np.float64)
    vx, vy = p["ux"].astype(np.float64) * g["dt"] / g["dx"], p["uy"].astype(np.float64) * g["dt"] / g["dy"]
    gy0, gx0 = (tile % nty) * T, (tile // nty) * T
    bad = 0
    for k in range(1, steps + 1):
        cy = np.floor(y0 + k * vy + 0.5) - gy0
        cy = (cy - 16 + g["ny"] / 2) % g["ny"] - g["ny"] / 2 + 16             # nearest periodic image, seen from the tile's centre
        m = cy - lane
        r = np.floor(x0 + k * vx + 0.5) - gx0 - 16 * sub                       # nearest node row relative to the sub-tile
        bad += int(((m < -1) | (m > 2) | (r < -1) | (r > 17)).sum())
    return bad / (steps * x0.size)


def test_sorting_by_the_position_half_a_period_ahead_keeps_the_particles_in_their_lanes():
    """3 keV electrons (thermal drift 0.054 cell per step) over a rebin period of 16 steps leave the
    reach of their lane (four window copies, two halo rows) in 1e-4 of the visits when the order is built from the position
    half a period ahead, in 5e-3 when it is built from the position at the time of the sort -- the numbers behind
    `rebin_every = 16` and `NCOPY = 4`.  The device counts the same through pm2d_stray_count: bench.py's `stray_fraction` on
    full c3 is 1.0e-4, and 4.1e-3 was measured before the sort looked ahead."""
    cfg, p = _particles()
    ahead = _out_of_lane_fraction(cfg, p, 16, 16)
    cfg0, p0 = _particles()
    now = _out_of_lane_fraction(cfg0, p0, 0, 16)
    assert ahead < 3e-4 and now > 3e-3, (ahead, now)                 # measured 1.0e-4 and 5.2e-3
    vth = math.sqrt(3.0 / 511.0)
    assert 0.05 < vth * cfg["grid"]["dt"] / cfg["grid"]["dx"] < 0.06


def test_shifted_window_copies_remove_the_bank_conflicts_a_single_window_has():
    """a warp of the lane order holds one particle of every slab.  With ONE copy of the shared windows the bank
    of a deposit is its node column: lanes whose particles round to the same column modulo 32 collide (slab i straddles
    the node columns i and i + 1, so neighbours collide all the time) and a shared atomic costs as many wavefronts as the
    fullest bank -- the model gives 2.1-2.3 per atomic, what ncu measured on round 1's single-window kernel (2.0-2.4,
    profiles/r01i).  With the copies shifted by one column each, lane i takes copy m = cy - i and index i + b: its bank is
    i + b whatever cy is, one wavefront, for every visit that is in lane (all but 1e-4)."""
    cfg, p = _particles()
    g = cfg["grid"]
    perm, tile, sub, lane, w = _lanes(cfg, p, 16)
    nty = g["ny"] // T
    y0 = p["iy"] + p["fy"].astype(np.float64)
    vy = p["uy"].astype(np.float64) * g["dt"] / g["dy"]
    gy0 = (tile % nty) * T
    warp = (tile * 2 + sub) * 1024 + w                       # 32 consecutive slots of a sub-tile = one rank w of every slab
    o = np.lexsort((lane, warp))
    full = np.flatnonzero(np.bincount(np.unique(warp[o], return_inverse=True)[1]) == 32)
    _, inv = np.unique(warp[o], return_inverse=True)
    rows = o[np.isin(inv, full)].reshape(-1, 32)             # particle indices, one row per full warp, lanes in order
    assert rows.shape[0] > 400 and (lane[rows] == np.arange(32)).all()
    single, copies = [], []
    for k in (1, 8, 16):
        cy = np.floor(y0 + k * vy + 0.5) - gy0
        cy = ((cy - 16 + g["ny"] / 2) % g["ny"] - g["ny"] / 2 + 16).astype(np.int64)
        c = cy[rows]
        in_lane = ((c - lane[rows] >= -1) & (c - lane[rows] <= 2)).all(axis=1)
        c = c[in_lane]
        one = np.array([np.bincount(r % 32, minlength=32).max() for r in c])            # bank = node column
        m = c - np.arange(32)
        shifted = np.array([np.bincount((r - mm) % 32, minlength=32).max() for r, mm in zip(c, m)])   # index c - m = lane
        single.append(one.mean())
        copies.append(shifted.mean())
    assert all(v == 1.0 for v in copies)
    assert all(1.9 < v < 2.6 for v in single), single

