"""Seeded synthetic inputs for PM2D runs: the workload configurations.

This module serves BOTH the CUDA library's tests/bench and the CPU oracle, and therefore holds none of the method's
arithmetic (no shape function, deposit, field update, push, and no particle loader): only the five workload
configurations of BASELINE.json (shapes, profiles, species, laser, seed), the paper's CBET set-up, and reduced-size
copies of them for parity tests.  The loader recipe they refer to (survey item A7: weights from the profile,
lattice offsets, Maxwellian velocities, the counter-based generator) is stated in DESIGN.md section 4 and implemented
twice, independently: on the device (k_load, pm2d_particles.cu) and in oracle/loader.py.
"""
from __future__ import annotations

import copy
import math

# enums shared with include/pm2d.h (values only; no code shared)
CIC, TSC, SINE = 0, 1, 2
LOAD_NONE, LATTICE_COLD, RANDOM_MAXWELL, NUMBER_WEIGHTED = 0, 1, 2, 3
PROFILE_UNIFORM, PROFILE_LINEAR, PROFILE_EXP_CAPPED, PROFILE_FILAMENT_Y = 0, 1, 2, 3

TAPER_FLOOR = 0.01   # the edge taper ends at 1 % of the profile, not at 0 (Q9 / Q20)


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
    elif name in ("cbet", "cbet_vac"):  # S§8(f).1, the paper's CBET run: 8000x8000 there, 8192x8192 here (ny a power of two);
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
    if name == "cbet_vac":                                # S§8(f).2: the same slab with TRUE vacuum margins (a
        # 360 x 360 lambda slab in the centre of a 400 x 400 lambda box = margins of a twentieth of the box on every
        # side), hard-edged: no particles outside, no taper by weight (Q20)
        c["profile"]["taper_cells"] = 0
        mx, my = max(g["nx"] // 20, 1), max(g["ny"] // 20, 1)
        c["profile"]["slab"] = [mx, g["nx"] - mx, my, g["ny"] - my]
    if name == "c5":                                      # sigma = ny/64 cells, amplitude A such that peak = 20 x mean
        sig = g["ny"] / 64.0
        c["profile"]["p"][2] = sig
        c["profile"]["p"][1] = 19.0 / (1.0 - 20.0 * sig * math.sqrt(2.0 * math.pi) / g["ny"])
    for sp in c["species"]:
        if sp["load"] == NUMBER_WEIGHTED:                 # slots: an upper bound of the dithered counts
            sp["capacity"] = g["nx"] * g["ny"] * sp["ppc_x"] * sp["ppc_y"] + 4096
    if name in ("c4", "cbet", "cbet_vac"):
        Ly = g["ny"] * g["dy"]
        for las in c["lasers"]:
            las["w0"] *= Ly
            las["y0"] *= Ly
    return copy.deepcopy(c)
