"""The number formats of the CUDA path, modelled on the CPU: int32 fixed-point deposits and the
float -> int conversion by a magic-number FMA.  Nothing here runs device code; the models are exact emulations of the
arithmetic the kernels are documented to do, checked against the float64 oracle and against the integers."""
import math

import numpy as np

import oracle
import oracle.loader as L
import pm2d_inputs as I


def test_the_magic_number_conversion_is_round_to_nearest_even_below_2_to_the_22():
    """DESIGN.md 6.1c / pm2d_lanes.cu: float -> int without the XU pipe.  fma(w, q, 1.5 * 2^23) in float32 has the integer
    rint(w q) in its mantissa -- bits(result) - bits(1.5 * 2^23) -- for every |w q| <= 2^22, ties to even, both signs; one
    step beyond 2^22 the sum leaves the binade of 1.5 * 2^23 and the trick breaks, which is why the kernel sends particles
    faster than `ucap` (4 thermal velocities) down the exact F2I path and chooses the per-tile momentum unit 2^sp so that
    a single contribution stays below 2^22.  The float32 FMA is emulated exactly in float64 (a 48-bit product plus a
    constant 50 bits above its last bit is exact there, then rounded once)."""
    MAGIC, BITS = np.float32(12582912.0), np.int32(0x4B400000)
    assert MAGIC.view(np.int32) == BITS

    def magic_int(w, q):
        s = np.float64(w) * np.float64(q) + np.float64(MAGIC)                  # exact
        return s.astype(np.float32).view(np.int32) - BITS

    rng = np.random.default_rng(11)
    w = rng.uniform(0.0, 2.0, 200000).astype(np.float32)                        # weights (scale 2 of the sine cloud)
    q = (rng.uniform(-1.0, 1.0, 200000) * 2.0 ** 21).astype(np.float32)         # |w q| < 2^22
    exact = np.float64(w) * np.float64(q)
    assert np.array_equal(magic_int(w, q), np.rint(exact).astype(np.int64).astype(np.int32))
    # ties go to even, on both sides of zero
    half = np.array([0.5, 1.5, 2.5, -0.5, -1.5, -2.5, 4194303.5, -4194303.5], np.float32)
    assert list(magic_int(np.float32(1.0), half)) == [0, 2, 2, 0, -2, -2, 4194304, -4194304]
    # the edge of the range: 2^22 itself still converts, 2^22 + 1 on the negative side does not
    assert magic_int(np.float32(1.0), np.float32(4194304.0)) == 4194304 and magic_int(np.float32(1.0), np.float32(-4194304.0)) == -4194304
    assert magic_int(np.float32(1.0), np.float32(-4194305.0)) != -4194305


def _fixed_point_deposit(cfg, s, unit):
    """Eq. 14 with every contribution rounded once to `unit` (what the kernels add into their int32 grids), from the
    oracle's own 1-D weights; interior particles only (the wall fold is not what is modelled here) -> (grid, used)."""
    g, q = cfg["grid"], cfg["species"][s]
    p = L.generate_particles(cfg, s)
    X = p["ix"] + p["fx"].astype(np.float64)
    Y = p["iy"] + p["fy"].astype(np.float64)
    use = (X > 2.0) & (X < g["nx"] - 2.0)
    out = np.zeros((g["nx"] + 1, g["ny"]), np.int64)
    for x, y, w in zip(X[use], Y[use], p["w"][use].astype(np.float64)):
        fx, Wx = oracle.weights_1d(q["shape"], q["DD"], x)
        fy, Wy = oracle.weights_1d(q["shape"], q["DD"], y)
        c = np.rint(w * np.outer(Wx, Wy) / unit).astype(np.int64)
        out[fx:fx + len(Wx), (fy + np.arange(len(Wy))) % g["ny"]] += c
    return out * unit, p, use


def test_int32_fixed_point_deposits_resolve_the_density_to_1e_7_of_the_grid_and_absolutely():
    """the deposit grids are int32 with the unit n_cap / 2^31, n_cap the power of two >= 8 n_max
    (0.25 n_c for c3 -> n_cap = 2, unit 9.3e-10 n_c); every contribution is rounded to it once.  Against the float64 deposit
    of the same particles the relative L2 error of the density is below 1e-7 (BASELINE.json asks for 1e-5), and the error
    of a node is absolute -- a few units whatever the node holds: a thousandth of a per cent in the slab, but 1e-4 and more
    of a node that carries 1e-5 of the slab's density, which is what the vacuum-margin parity test runs into."""
    cfg = I.config("c3", nx=48, ny=32)
    g, q = cfg["grid"], cfg["species"][0]
    unit = 2.0 / 2.0 ** 31
    got, p, use = _fixed_point_deposit(cfg, 0, unit)
    grid = oracle.make_grid(g["nx"], g["ny"], g["dx"], g["dy"], g["dt"])
    X = (p["ix"] + p["fx"].astype(np.float64))[use]
    Y = (p["iy"] + p["fy"].astype(np.float64))[use]
    ref, _, _ = oracle.deposit(grid, q["shape"], q["DD"], X, Y, 0 * X, 0 * X, p["w"][use].astype(np.float64))
    err = got - ref
    assert math.sqrt((err ** 2).sum() / (ref ** 2).sum()) < 1e-7                 # measured 9e-9
    assert np.abs(err).max() < 8 * unit                                          # measured 5.4 units: ~36 contributions per node, each off by at most half a unit
    assert np.abs(err).max() / ref.max() < 1e-7 and 3 * unit / (1e-5 * ref.max()) > 1e-4


def test_per_tile_momentum_units_of_the_lane_kernel_cost_a_third_of_the_tolerance():
    """k_stage_lanes converts a momentum contribution with the magic-number FMA, which holds 2^22; the shared
    windows therefore count momentum in units of 2^sp global units (global unit = n_cap / 2^35: |n u| <= n_cap / 16), sp =
    ilogb(w_max pscale u_cap) + 1 - 22 from the tile's largest weight and u_cap = 4 v_th.  For the electrons of c3 that is
    sp = 7: each contribution is rounded to 7.5e-9 n_c c.  Modelled against the float64 momentum deposit of the same
    particles: 3.5e-6 relative L2 -- inside BASELINE.json's 1e-5, and the largest single share of it (the density, in
    global units, is at 9e-9)."""
    cfg = I.config("c3", nx=48, ny=32)
    g, q = cfg["grid"], cfg["species"][0]
    p = L.generate_particles(cfg, 0)
    pscale = 2.0 ** 35 / 2.0                                               # n_cap = 2 n_c
    ucap = max(4.0 * math.sqrt(q["T_keV"] / 511.0 / q["mass"]), 0.004)
    sp = max(0, math.frexp(float(p["w"].max()) * pscale * ucap)[1] - 1 + 1 - 22)
    assert sp == 7
    unit = 2.0 ** sp / pscale
    X = p["ix"] + p["fx"].astype(np.float64)
    Y = p["iy"] + p["fy"].astype(np.float64)
    use = (X > 2.0) & (X < g["nx"] - 2.0) & (np.hypot(p["ux"], p["uy"]) <= ucap)      # the others take the exact path
    out = np.zeros((g["nx"] + 1, g["ny"]), np.int64)
    for x, y, w, u in zip(X[use], Y[use], p["w"][use].astype(np.float64), p["ux"][use].astype(np.float64)):
        fx, Wx = oracle.weights_1d(q["shape"], q["DD"], x)
        fy, Wy = oracle.weights_1d(q["shape"], q["DD"], y)
        out[fx:fx + len(Wx), (fy + np.arange(len(Wy))) % g["ny"]] += np.rint(w * u * np.outer(Wx, Wy) / unit).astype(np.int64)
    grid = oracle.make_grid(g["nx"], g["ny"], g["dx"], g["dy"], g["dt"])
    _, ref, _ = oracle.deposit(grid, q["shape"], q["DD"], X[use], Y[use], p["ux"][use].astype(np.float64), 0 * X[use], p["w"][use].astype(np.float64))
    rel = math.sqrt(((out * unit - ref) ** 2).sum() / (ref ** 2).sum())
    assert 5e-7 < rel < 5e-6, rel
