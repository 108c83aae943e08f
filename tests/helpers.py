"""Shared test helpers: build an Oracle (CPU) from a pm2d_inputs config."""
import numpy as np

import oracle
import pm2d_inputs as I


def oracle_species_from_arrays(sp_cfg, parts=None, n_fixed=None):
    d = dict(mass=sp_cfg["mass"], sign=sp_cfg["sign"], T_keV=sp_cfg["T_keV"], C=sp_cfg["pressure_coeff"],
             shape=sp_cfg["shape"], DD=sp_cfg["DD"], mobile=sp_cfg["mobile"])
    if parts is not None:
        d["X"] = parts["ix"].astype(np.float64) + parts["fx"].astype(np.float64)
        d["Y"] = parts["iy"].astype(np.float64) + parts["fy"].astype(np.float64)
        d["ux"] = parts["ux"].astype(np.float64)
        d["uy"] = parts["uy"].astype(np.float64)
        d["w"] = parts["w"].astype(np.float64)
    if n_fixed is not None:
        d["n_fixed"] = n_fixed
    return d


def oracle_from_config(cfg, particles=None):
    """particles: optional list (per species) of dicts as returned by generate_particles."""
    g = cfg["grid"]
    grid = oracle.make_grid(g["nx"], g["ny"], g["dx"], g["dy"], g["dt"], g["ncomp"])
    if particles is None:
        particles = [I.generate_particles(cfg, s) if sp["load"] != I.LOAD_NONE else None
                     for s, sp in enumerate(cfg["species"])]
    species = []
    # Q13: an immobile species without particles neutralises the summed deposit of the mobile
    # species of opposite sign at t = 0
    for s, sp in enumerate(cfg["species"]):
        if particles[s] is not None:
            species.append(oracle_species_from_arrays(sp, particles[s]))
        else:
            species.append(None)
    for s, sp in enumerate(cfg["species"]):
        if species[s] is None:
            nfix = np.zeros((g["nx"] + 1, g["ny"]))
            for t, sq in enumerate(cfg["species"]):
                if particles[t] is not None and sq["sign"] == -sp["sign"]:
                    d = species[t]
                    n, _, _ = oracle.deposit(grid, sq["shape"], sq["DD"], d["X"], d["Y"], d["ux"], d["uy"], d["w"])
                    nfix += n
            species[s] = oracle_species_from_arrays(sp, None, nfix)
    lasers = [dict(a0=l["a0"], omega=l["omega"], y0=l["y0"], w0=l["w0"], t_rise=l["t_rise"], comp=l["comp"])
              for l in cfg["lasers"]]
    return oracle.Oracle(g["nx"], g["ny"], g["dx"], g["dy"], g["dt"], species, lasers, g["ncomp"]), particles
