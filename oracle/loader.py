"""The particle loader of the oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT (survey item A7).

"the electron and ion macro-particles are initially distributed evenly within the grids ... the density weight of a
macro-particle n_sp^0 = n_s^0(i dx, j dy) / (N M)", here with BASELINE.json's "uniform-random positions
within each cell, Maxwellian momenta ... all drawn from seed" (Q7).  Recipe:
  cell (i, j), i < nx, j < ny, k-th particle of the cell, k < ppc_x*ppc_y:
     id      = k * (nx*ny) + i*ny + j
     r0..r3  = philox4x32_10(counter=(id_lo, id_hi, species, 0), key=(seed_lo, seed_hi))
     LATTICE_COLD  : fx = ((k // ppc_y) + 1/2)/ppc_x, fy = ((k % ppc_y) + 1/2)/ppc_y, u = 0
     RANDOM_MAXWELL: fx = (r0 >> 8) * 2^-24, fy = (r1 >> 8) * 2^-24,
                     U1 = (r2 + 1) * 2^-32, U2 = r3 * 2^-32   (double),
                     ux = vth*sqrt(-2 ln U1)*cos(2 pi U2), uy = vth*sqrt(-2 ln U1)*sin(2 pi U2)
                     evaluated in double, rounded once to float32
     w = profile(x at cell centre) * taper / (ppc_x*ppc_y), double rounded once to float32     (Q17)
     NUMBER_WEIGHTED (config c5): equal weights w = n0/ppc; the NUMBER of particles of a cell follows the
                     profile: count(i, j) = floor(ppc * shape(i, j) + U), shape = taper(i) * filament(j) with
                     mean 1 over j, U = philox(counter=(cell_lo, cell_hi, species, 1))[0] * 2^-32 (a
                     dithered rounding, so the expected count is exact); offsets and momenta as RANDOM_MAXWELL
     profile["slab"] = [x_lo, x_hi, y_lo, y_hi] (cells; absent or all zero: the whole box): only cells with
                     x_lo <= i < x_hi and y_lo <= j < y_hi hold particles -- "a plasma slab is set at the center of the
                     simulation box, and the vacuum space is usually set around the plasma slab"; ids, offsets,
                     momenta and weights of the loaded cells are what they are without the slab
The CUDA library runs the same recipe on the device (k_load); the two share no code.  Pins (tests/test_oracle_loader.py):
Philox-4x32-10 against the Random123 known-answer vectors (tests/golden/philox4x32_10_kat.txt), particles per cell exact,
w * N * M = profile at the cell centre, moments of the Maxwellian, expected counts of the number-weighted loading.
"""
from __future__ import annotations

import math

import numpy as np

from pm2d_inputs import (LATTICE_COLD, LOAD_NONE, NUMBER_WEIGHTED, PROFILE_EXP_CAPPED, PROFILE_FILAMENT_Y, PROFILE_LINEAR, PROFILE_UNIFORM,
                         RANDOM_MAXWELL, TAPER_FLOOR)

_M0, _M1 = np.uint64(0xD2511F53), np.uint64(0xCD9E8D57)
_W0, _W1 = 0x9E3779B9, 0xBB67AE85
_MASK = np.uint64(0xFFFFFFFF)


def philox4x32_10(c0, c1, c2, c3, k0, k1):
    """Philox-4x32-10 (Salmon et al., SC'11).  Arrays of uint32 counters, scalar uint32 keys."""
    c0, c1, c2, c3 = (np.asarray(c, dtype=np.uint64) & _MASK for c in (c0, c1, c2, c3))
    k0, k1 = int(k0) & 0xFFFFFFFF, int(k1) & 0xFFFFFFFF
    for _ in range(10):
        p0 = _M0 * c0
        p1 = _M1 * c2
        hi0, lo0 = p0 >> np.uint64(32), p0 & _MASK
        hi1, lo1 = p1 >> np.uint64(32), p1 & _MASK
        c0, c1, c2, c3 = (hi1 ^ c1 ^ np.uint64(k0)), lo1, (hi0 ^ c3 ^ np.uint64(k1)), lo0
        k0 = (k0 + _W0) & 0xFFFFFFFF
        k1 = (k1 + _W1) & 0xFFFFFFFF
    return tuple(c.astype(np.uint32) for c in (c0, c1, c2, c3))


# ---------------------------------------------------------------------------------------------
def profile_density(profile: dict, nx: int, i_cell):
    """Density (n_c) at the centre of cells with x-index i_cell (float64), taper included."""
    xc = (np.asarray(i_cell, dtype=np.float64) + 0.5) / nx           # in units of Lx
    kind = profile["kind"]
    p = profile["p"]
    if kind == PROFILE_UNIFORM:
        n = np.full_like(xc, p[0])
    elif kind == PROFILE_LINEAR:
        n = p[0] + (p[1] - p[0]) * xc
    elif kind == PROFILE_EXP_CAPPED:                                  # n0 exp(x/L) capped
        n = np.minimum(p[0] * np.exp(xc * p[1]), p[2])                # p[1] = Lx/L
    elif kind == PROFILE_FILAMENT_Y:                                  # uniform in x; the y-dependence is in filament_shape
        n = np.full_like(xc, p[0])
    else:
        raise ValueError(kind)
    return n * taper_factor(profile, nx, i_cell)


def taper_factor(profile: dict, nx: int, i_cell):
    """Edge taper (Q9) alone, float64: FLOOR + (1 - FLOOR) sin^2(pi d / 2 tc) within tc cells of an x wall."""
    i = np.asarray(i_cell, dtype=np.float64)
    tc = int(profile.get("taper_cells", 0))
    if tc <= 0:
        return np.ones_like(i)
    d = np.minimum(i + 0.5, nx - 0.5 - i)
    sn = np.sin(0.5 * math.pi * d / tc)
    return np.where(d < tc, TAPER_FLOOR + (1.0 - TAPER_FLOOR) * (sn * sn), 1.0)


def taper_factor_y(profile: dict, ny: int, j_cell):
    """The same taper at the y walls over profile["taper_cells_y"] cells (0 / absent: none)."""
    j = np.asarray(j_cell, dtype=np.float64)
    tc = int(profile.get("taper_cells_y", 0))
    if tc <= 0:
        return np.ones_like(j)
    d = np.minimum(j + 0.5, ny - 0.5 - j)
    sn = np.sin(0.5 * math.pi * d / tc)
    return np.where(d < tc, TAPER_FLOOR + (1.0 - TAPER_FLOOR) * (sn * sn), 1.0)


def filament_shape(profile: dict, ny: int):
    """Relative density of the cells of column index j (mean 1 over j): a Gaussian filament along x centred
    in y, 1 + A exp(-(y - Ly/2)^2 / 2 sigma^2), normalised; p = [n0, A, sigma in cells].  float64[ny]."""
    A, sig = float(profile["p"][1]), float(profile["p"][2])
    yc = np.arange(ny, dtype=np.float64) + 0.5
    r = (yc - 0.5 * ny) / sig
    g = 1.0 + A * np.exp(-0.5 * r * r)
    return g / (g.sum() / ny)


def profile_max(profile: dict) -> float:
    kind, p = profile["kind"], profile["p"]
    if kind == PROFILE_UNIFORM:
        return float(p[0])
    if kind == PROFILE_FILAMENT_Y:
        return float(p[0]) * (1.0 + float(p[1]))
    if kind == PROFILE_LINEAR:
        return float(max(p[0], p[1]))
    return float(min(p[0] * math.exp(max(p[1], 0.0)), p[2]))


def slab_extent(cfg: dict):
    """(x_lo, x_hi, y_lo, y_hi) of the cells that hold particles; the whole box without profile["slab"]."""
    g = cfg["grid"]
    sl = cfg["profile"].get("slab")
    if not sl or not any(sl):
        return 0, g["nx"], 0, g["ny"]
    x_lo, x_hi, y_lo, y_hi = (int(v) for v in sl)
    assert 0 <= x_lo < x_hi <= g["nx"] and 0 <= y_lo < y_hi <= g["ny"], sl
    return x_lo, x_hi, y_lo, y_hi


def generate_particles(cfg: dict, s: int, i_lo: int = 0, i_hi: int | None = None):
    """Particles of species ``s`` for cells with i_lo <= i < i_hi (all j), in id order
    (k-major, then cell).  Returns dict(id, ix, iy, fx, fy, ux, uy, w) -- int64/int32/float32."""
    g, sp = cfg["grid"], cfg["species"][s]
    nx, ny = g["nx"], g["ny"]
    i_hi = nx if i_hi is None else i_hi
    ppc = sp["ppc_x"] * sp["ppc_y"]
    x_lo, x_hi, y_lo, y_hi = slab_extent(cfg)
    ii, jj = np.meshgrid(np.arange(max(i_lo, x_lo), min(i_hi, x_hi), dtype=np.int64), np.arange(y_lo, y_hi, dtype=np.int64), indexing="ij")
    cell = (ii * ny + jj).ravel()
    if sp["load"] == NUMBER_WEIGHTED:
        assert (x_lo, x_hi, y_lo, y_hi) == (0, nx, 0, ny), "the number-weighted loading has no slab extent"
        cnt = cell_counts(cfg, s)[i_lo:i_hi].ravel()
        kmax = int(cnt.max()) if cnt.size else 0
        k = np.concatenate([np.full(int((cnt > kk).sum()), kk, dtype=np.int64) for kk in range(kmax)]) if kmax else np.zeros(0, np.int64)
        cell = np.concatenate([cell[cnt > kk] for kk in range(kmax)]) if kmax else np.zeros(0, np.int64)
    else:
        k = np.repeat(np.arange(ppc, dtype=np.int64), cell.size)
        cell = np.tile(cell, ppc)
    pid = k * (nx * ny) + cell
    ix = (cell // ny).astype(np.int32)
    iy = (cell % ny).astype(np.int32)
    seed = int(cfg["seed"])
    r0, r1, r2, r3 = philox4x32_10(pid & 0xFFFFFFFF, pid >> 32, np.full_like(pid, s), np.zeros_like(pid),
                                   seed & 0xFFFFFFFF, seed >> 32)
    if sp["load"] == LATTICE_COLD:
        fx = (((k // sp["ppc_y"]) + 0.5) / sp["ppc_x"]).astype(np.float32)
        fy = (((k % sp["ppc_y"]) + 0.5) / sp["ppc_y"]).astype(np.float32)
        ux = np.zeros(pid.size, np.float32)
        uy = np.zeros(pid.size, np.float32)
    elif sp["load"] in (RANDOM_MAXWELL, NUMBER_WEIGHTED):
        fx = ((r0 >> np.uint32(8)).astype(np.float64) * 2.0 ** -24).astype(np.float32)
        fy = ((r1 >> np.uint32(8)).astype(np.float64) * 2.0 ** -24).astype(np.float32)
        vth = math.sqrt(sp["T_keV"] / 511.0 / sp["mass"])
        U1 = (r2.astype(np.float64) + 1.0) * 2.0 ** -32
        U2 = r3.astype(np.float64) * 2.0 ** -32
        R = vth * np.sqrt(-2.0 * np.log(U1))
        ux = (R * np.cos(2.0 * math.pi * U2)).astype(np.float32)
        uy = (R * np.sin(2.0 * math.pi * U2)).astype(np.float32)
    else:
        raise ValueError(sp["load"])
    if sp["load"] == NUMBER_WEIGHTED:
        w = np.full(pid.size, np.float32(cfg["profile"]["p"][0] / ppc), np.float32)
    else:
        w = (profile_density(cfg["profile"], nx, ix) * taper_factor_y(cfg["profile"], ny, iy) / ppc).astype(np.float32)
    return dict(id=pid, ix=ix, iy=iy, fx=fx, fy=fy, ux=ux, uy=uy, w=w)


def cell_counts(cfg: dict, s: int):
    """NUMBER_WEIGHTED: particles per cell, int64[nx][ny] (see the module docstring)."""
    g, sp = cfg["grid"], cfg["species"][s]
    nx, ny = g["nx"], g["ny"]
    ppc = float(sp["ppc_x"] * sp["ppc_y"])
    shape_y = filament_shape(cfg["profile"], ny) if cfg["profile"]["kind"] == PROFILE_FILAMENT_Y else np.ones(ny)
    tap = taper_factor(cfg["profile"], nx, np.arange(nx))
    cell = np.arange(nx * ny, dtype=np.int64)
    seed = int(cfg["seed"])
    r0, _, _, _ = philox4x32_10(cell & 0xFFFFFFFF, cell >> 32, np.full_like(cell, s), np.ones_like(cell),
                                seed & 0xFFFFFFFF, seed >> 32)
    u = r0.astype(np.float64) * 2.0 ** -32
    lam = (ppc * tap)[:, None] * shape_y[None, :]
    return np.floor(lam + u.reshape(nx, ny)).astype(np.int64)


def n_particles(cfg: dict, s: int) -> int:
    sp = cfg["species"][s]
    if sp["load"] == LOAD_NONE:
        return 0
    if sp["load"] == NUMBER_WEIGHTED:
        return int(cell_counts(cfg, s).sum())
    x_lo, x_hi, y_lo, y_hi = slab_extent(cfg)
    return (x_hi - x_lo) * (y_hi - y_lo) * sp["ppc_x"] * sp["ppc_y"]
