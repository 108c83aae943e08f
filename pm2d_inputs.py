"""Seeded synthetic inputs for PM2D runs: configurations and the particle loader.

This module serves BOTH the CUDA library's tests/bench and the CPU oracle, and therefore holds
none of the method's arithmetic (no shape function, deposit, field update, push ...): only
  * the five workload configurations of BASELINE.json (shapes, profiles, species, laser, seed)
    plus reduced-size copies of them for parity tests, and
  * the counter-based particle loader: Philox-4x32-10 keyed by the seed, counter = particle id,
    species and stream.  The CUDA library implements the same generator on the device
    (csrc/pm2d_init.cu); tests check that the two agree.

Loader recipe:
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
"""
from __future__ import annotations

import copy
import math

import numpy as np

# enums shared with include/pm2d.h (values only; no code shared)
CIC, TSC, SINE = 0, 1, 2
LOAD_NONE, LATTICE_COLD, RANDOM_MAXWELL, NUMBER_WEIGHTED = 0, 1, 2, 3
PROFILE_UNIFORM, PROFILE_LINEAR, PROFILE_EXP_CAPPED, PROFILE_FILAMENT_Y = 0, 1, 2, 3

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


TAPER_FLOOR = 0.01   # the edge taper ends at 1 % of the profile, not at 0 (Q9 / Q20)


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


def generate_particles(cfg: dict, s: int, i_lo: int = 0, i_hi: int | None = None):
    """Particles of species ``s`` for cells with i_lo <= i < i_hi (all j), in id order
    (k-major, then cell).  Returns dict(id, ix, iy, fx, fy, ux, uy, w) -- int64/int32/float32."""
    g, sp = cfg["grid"], cfg["species"][s]
    nx, ny = g["nx"], g["ny"]
    i_hi = nx if i_hi is None else i_hi
    ppc = sp["ppc_x"] * sp["ppc_y"]
    ii, jj = np.meshgrid(np.arange(i_lo, i_hi, dtype=np.int64), np.arange(ny, dtype=np.int64), indexing="ij")
    cell = (ii * ny + jj).ravel()
    if sp["load"] == NUMBER_WEIGHTED:
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


# ---------------------------------------------------------------------------------------------
def _species(sign, mass, T, ppc_x, ppc_y, shape, DD, mobile=1, load=RANDOM_MAXWELL, C=2.0):
    return dict(sign=sign, mass=float(mass), T_keV=float(T), pressure_coeff=float(C), ppc_x=ppc_x, ppc_y=ppc_y,
                mobile=mobile, shape=shape, DD=float(DD), load=load)


def _laser(a0, w0=0.0, y0=0.0, t_rise=5.0, omega=1.0, comp=0):
    return dict(a0=float(a0), omega=float(omega), y0=float(y0), w0=float(w0), alpha=0.0, comp=comp, t_rise=float(t_rise))


_DX = 0.05  # lambda0/20 (BASELINE.json configs)


def _base(nx, ny, dt, steps, seed, rebin_every=16):
    return dict(grid=dict(nx=nx, ny=ny, dx=_DX, dy=_DX, dt=dt, ncomp=1, rebin_every=rebin_every),
                steps=steps, seed=seed)


def config(name: str, nx: int | None = None, ny: int | None = None) -> dict:
    """BASELINE.json configs 'c1'..'c5'.  nx/ny override the grid size to make
    a reduced copy (same dx, dt, particles per cell, profile shape over the box, species, laser)."""
    if name == "c1":      # tiny slab: 256x128, CFL 0.5, uniform 0.1 n_c, 4 e/cell 1 keV, CIC, a0=0.01
        c = _base(256, 128, 0.5 * _DX, 100, 0)
        c["profile"] = dict(kind=PROFILE_UNIFORM, p=[0.1, 0, 0, 0])
        c["species"] = [_species(-1, 1.0, 1.0, 2, 2, CIC, 1.0),
                        _species(+1, 1836.0, 0.0, 0, 0, CIC, 1.0, mobile=0, load=LOAD_NONE)]
        c["lasers"] = [_laser(0.01)]
    elif name == "c2":    # medium ramp: 2048x1024, 0.05->0.25, 8 e/cell 2 keV, TSC, a0=0.02
        c = _base(2048, 1024, 0.035, 1000, 1)
        c["profile"] = dict(kind=PROFILE_LINEAR, p=[0.05, 0.25, 0, 0])
        c["species"] = [_species(-1, 1.0, 2.0, 4, 2, TSC, 2.0),
                        _species(+1, 1836.0, 0.0, 0, 0, TSC, 2.0, mobile=0, load=LOAD_NONE)]
        c["lasers"] = [_laser(0.02)]
    elif name == "c3":    # SRS-scale slab: 8192x4096, 0.1 exp(x/L) capped 0.25, 4 e/cell 3 keV + D ions 1/cell 1 keV
        c = _base(8192, 4096, 0.035, 500, 2)
        c["profile"] = dict(kind=PROFILE_EXP_CAPPED, p=[0.1, math.log(2.5), 0.25, 0])
        c["species"] = [_species(-1, 1.0, 3.0, 2, 2, SINE, 1.9),
                        _species(+1, 3672.0, 1.0, 1, 1, SINE, 1.9)]
        c["lasers"] = [_laser(0.015)]
    elif name == "c4":    # large box: 16384x8192, 0.1->0.3, 2 e/cell 3 keV + ions 1/cell 1 keV, Gaussian beam
        c = _base(16384, 8192, 0.035, 200, 3)
        c["profile"] = dict(kind=PROFILE_LINEAR, p=[0.1, 0.3, 0, 0])
        c["species"] = [_species(-1, 1.0, 3.0, 2, 1, SINE, 1.9),
                        _species(+1, 3672.0, 1.0, 1, 1, SINE, 1.9)]
        c["lasers"] = [_laser(0.03, w0=0.3, y0=0.5)]     # w0, y0 in units of Ly, resolved below
    elif name == "c5":    # stress: 4096x4096, ~60 e/cell (1.0e9), 5 keV, Gaussian filament in y (peak 20x mean, sigma 64 cells)
        c = _base(4096, 4096, 0.035, 50, 4, rebin_every=4)     # cell-major + strip kernel: the register patches want fresh cells
        c["profile"] = dict(kind=PROFILE_FILAMENT_Y, p=[0.01, 87.7, 64.0, 0])
        c["species"] = [_species(-1, 1.0, 5.0, 10, 6, SINE, 1.9, load=NUMBER_WEIGHTED),
                        _species(+1, 1836.0, 0.0, 0, 0, SINE, 1.9, mobile=0, load=LOAD_NONE)]
        c["lasers"] = [_laser(0.01)]
    elif name == "cbet":  # S§8(f).1, the paper's CBET run: 8000x8000 there, 8192x8192 here (ny a power of two);
        # 0.4 n_c hydrogen slab (the standard edge taper stands in for the 20 lambda0 vacuum margins), 1 e + 1 ion per
        # cell, 1 keV / 200 eV, DD = 1.85 dx, two beams a0 = 0.008 at +-15 degrees, lambda0 and 0.9995 lambda0, centres
        # -+50 lambda0 from the axis, w0 = 30 lambda0, particle step = 5 wave steps, absorbing y walls for a
        c = _base(8192, 8192, 0.035, 200, 5, rebin_every=6)
        c["grid"]["subcycle"] = 5
        c["grid"]["bc_y"] = 1                                # "absorbing ... on all of four boundaries" (Q23)
        c["profile"] = dict(kind=PROFILE_UNIFORM, p=[0.4, 0, 0, 0])
        c["species"] = [_species(-1, 1.0, 1.0, 1, 1, SINE, 1.85),
                        _species(+1, 1836.0, 0.2, 1, 1, SINE, 1.85)]
        al = math.radians(15.0)
        c["lasers"] = [dict(_laser(0.008, w0=30.0 / 409.6, y0=0.5 - 50.0 / 409.6), alpha=al),
                       dict(_laser(0.008, w0=30.0 / 409.6, y0=0.5 + 50.0 / 409.6, omega=1.0 / 0.9995), alpha=-al)]
    else:
        raise ValueError(name)
    if nx is not None:
        c["grid"]["nx"] = nx
    if ny is not None:
        c["grid"]["ny"] = ny
    g = c["grid"]
    c["name"] = name if (nx is None and ny is None) else f"{name}@{g['nx']}x{g['ny']}"
    c["profile"]["taper_cells"] = g["nx"] // 16          # Q9
    if name == "cbet":                                    # the paper's slab has margins on all four sides
        c["profile"]["taper_cells_y"] = g["ny"] // 16
    if name == "c5":                                      # sigma = ny/64 cells, amplitude A such that peak = 20 x mean
        sig = g["ny"] / 64.0
        c["profile"]["p"][2] = sig
        c["profile"]["p"][1] = 19.0 / (1.0 - 20.0 * sig * math.sqrt(2.0 * math.pi) / g["ny"])
    for sp in c["species"]:
        if sp["load"] == NUMBER_WEIGHTED:                 # slots: an upper bound of the dithered counts
            sp["capacity"] = g["nx"] * g["ny"] * sp["ppc_x"] * sp["ppc_y"] + 4096
    if name in ("c4", "cbet"):
        Ly = g["ny"] * g["dy"]
        for las in c["lasers"]:
            las["w0"] *= Ly
            las["y0"] *= Ly
    return copy.deepcopy(c)


def n_particles(cfg: dict, s: int) -> int:
    sp = cfg["species"][s]
    if sp["load"] == LOAD_NONE:
        return 0
    if sp["load"] == NUMBER_WEIGHTED:
        return int(cell_counts(cfg, s).sum())
    return cfg["grid"]["nx"] * cfg["grid"]["ny"] * sp["ppc_x"] * sp["ppc_y"]
