"""Pins of the oracle's particle loader (oracle/loader.py; survey item A7) and of the polarisation
decomposition (A3c).  CPU only.  Each test names the mistake it would catch."""
import math
import os

import numpy as np
import pytest

import oracle
import oracle.loader as L
import pm2d_inputs as I

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def test_philox_known_answer_vectors():
    """Philox-4x32-10 against the Random123 known-answer vectors (a wrong round constant, key schedule, word order or
    round count changes every word)."""
    rows = [ln.split() for ln in open(os.path.join(GOLDEN, "philox4x32_10_kat.txt")) if ln.strip() and not ln.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        c = [int(v, 16) for v in r[:4]]
        k = [int(v, 16) for v in r[4:6]]
        want = [int(v, 16) for v in r[6:10]]
        got = L.philox4x32_10(*[np.array([v], np.uint64) for v in c], k[0], k[1])
        assert [int(g[0]) for g in got] == want
    # vectorised over counters: every lane independent
    c0 = np.array([0, 0xffffffff, 0x243f6a88], np.uint64)
    got = L.philox4x32_10(c0, c0 * 0, c0 * 0, c0 * 0, 0, 0)
    assert int(got[0][0]) == 0x6627e8d5 and len({int(v) for v in got[0]}) == 3


@pytest.mark.parametrize("name", ["c1", "c2", "c3", "cbet"])
def test_particles_per_cell_ids_and_weights(name):
    """"N and M macro-particles per grid in x and y": exactly ppc_x * ppc_y particles in every cell, ids k *
    nx * ny + cell, offsets in [0, 1) on the 2^-24 lattice, and the weight n_s^0(cell centre) / (N M) (Q17) --
    a profile sampled at the node instead of the centre, a missing 1/(NM) or a taper in the wrong direction fail."""
    cfg = I.config(name, nx=48, ny=32)
    g = cfg["grid"]
    nx, ny = g["nx"], g["ny"]
    for s, sp in enumerate(cfg["species"]):
        if sp["load"] == I.LOAD_NONE:
            continue
        p = L.generate_particles(cfg, s)
        ppc = sp["ppc_x"] * sp["ppc_y"]
        assert p["ix"].size == nx * ny * ppc == L.n_particles(cfg, s)
        cell = p["ix"].astype(np.int64) * ny + p["iy"]
        assert np.array_equal(np.bincount(cell, minlength=nx * ny), np.full(nx * ny, ppc))
        k = p["id"] // (nx * ny)
        assert np.array_equal(p["id"] % (nx * ny), cell) and k.min() == 0 and k.max() == ppc - 1
        for f in (p["fx"], p["fy"]):
            assert f.min() >= 0.0 and f.max() < 1.0
            assert np.array_equal(f.astype(np.float64) * 2 ** 24, np.round(f.astype(np.float64) * 2 ** 24))
        # w N M = profile at the cell centre, written out here from the config (not through the loader's helpers)
        xc = (p["ix"] + 0.5) / nx
        pr = cfg["profile"]
        if pr["kind"] == I.PROFILE_UNIFORM:
            n0 = np.full(xc.shape, pr["p"][0])
        elif pr["kind"] == I.PROFILE_LINEAR:
            n0 = pr["p"][0] + (pr["p"][1] - pr["p"][0]) * xc
        else:
            n0 = np.minimum(pr["p"][0] * np.exp(xc * pr["p"][1]), pr["p"][2])
        def taper(idx, n, tc):
            d = np.minimum(idx + 0.5, n - 0.5 - idx)
            return np.where(d < tc, I.TAPER_FLOOR + (1 - I.TAPER_FLOOR) * np.sin(0.5 * math.pi * d / max(tc, 1)) ** 2, 1.0) if tc > 0 else 1.0
        want = n0 * taper(p["ix"].astype(np.float64), nx, pr["taper_cells"]) * taper(p["iy"].astype(np.float64), ny, pr.get("taper_cells_y", 0)) / ppc
        assert np.abs(p["w"] / want - 1).max() < 1e-7                      # one float32 rounding
    if name == "c1":
        p = L.generate_particles(cfg, 0)
        wx = p["w"][(p["iy"] == 0) & (p["id"] < nx * ny)]
        assert wx[0] == pytest.approx(0.1 / 4 * (I.TAPER_FLOOR + (1 - I.TAPER_FLOOR) * math.sin(0.5 * math.pi * 0.5 / 3) ** 2), rel=1e-6)
        assert wx[nx // 2] == pytest.approx(0.1 / 4, rel=1e-7)


def test_maxwellian_moments_and_uniform_offsets():
    """"Maxwellian momenta Te" (BASELINE.json configs; v_th = sqrt(T / 511 / m)): mean 0, variance v_th^2 per
    component, kurtosis 3, no x-y correlation, offsets uniform -- within 5 sigma of 4.9e5 draws.  A Box-Muller with the
    wrong radius (sqrt(-ln U) instead of sqrt(-2 ln U)), v_th without the mass, or cos in both components fail."""
    cfg = I.config("c3", nx=384, ny=256)
    for s, sp in enumerate(cfg["species"]):
        p = L.generate_particles(cfg, s)
        n = p["ux"].size
        vth = math.sqrt(sp["T_keV"] / 511.0 / sp["mass"])
        for u in (p["ux"].astype(np.float64), p["uy"].astype(np.float64)):
            assert abs(u.mean()) < 5 * vth / math.sqrt(n)
            assert abs((u ** 2).mean() / vth ** 2 - 1) < 5 * math.sqrt(2.0 / n)
            assert abs((u ** 4).mean() / vth ** 4 - 3) < 5 * math.sqrt(96.0 / n)
        assert abs((p["ux"].astype(np.float64) * p["uy"]).mean()) < 5 * vth ** 2 / math.sqrt(n)
        for f in (p["fx"].astype(np.float64), p["fy"].astype(np.float64)):
            assert abs(f.mean() - 0.5) < 5 * math.sqrt(1 / 12.0 / n)
            assert abs(f.var() - 1 / 12.0) < 5 * math.sqrt(1 / 180.0 / n)
        # the two species draw from different streams
    a, b = L.generate_particles(cfg, 0), L.generate_particles(cfg, 1)
    assert not np.array_equal(a["fx"][: b["fx"].size], b["fx"])


def test_lattice_cold_loading():
    """The paper's own loading: "distributed evenly within the grids ... the spatial intervals between two
    adjacent macro-particles in x and y directions are dx/N and dy/M", zero drift velocity."""
    cfg = I.config("c2", nx=16, ny=8)
    cfg["species"][0]["load"] = I.LATTICE_COLD
    p = L.generate_particles(cfg, 0)
    N, M = cfg["species"][0]["ppc_x"], cfg["species"][0]["ppc_y"]
    sel = (p["ix"] == 5) & (p["iy"] == 3)
    xs, ys = np.unique(p["fx"][sel]), np.unique(p["fy"][sel])
    assert xs.size == N and ys.size == M and sel.sum() == N * M
    assert np.allclose(np.diff(xs), 1.0 / N) and np.allclose(np.diff(ys), 1.0 / M)
    assert xs[0] == pytest.approx(0.5 / N) and ys[0] == pytest.approx(0.5 / M)          # centred: the lattice continues across cells
    assert not p["ux"].any() and not p["uy"].any()


def test_number_weighted_counts_follow_the_profile():
    """BASELINE.json config 5 ("density concentrated in a Gaussian filament (peak 20x mean, sigma = 64 cells)"): equal
    weights, the particle NUMBER follows the profile; the dithered rounding makes the expected count exact."""
    cfg = I.config("c5", nx=128, ny=256)
    sp = cfg["species"][0]
    ppc = sp["ppc_x"] * sp["ppc_y"]
    cnt = L.cell_counts(cfg, 0)
    shape = L.filament_shape(cfg["profile"], 256)
    assert shape.mean() == pytest.approx(1.0, rel=1e-12) and shape.max() / shape.mean() == pytest.approx(20.0, rel=1e-2)
    bulk = slice(cfg["profile"]["taper_cells"], 128 - cfg["profile"]["taper_cells"])
    per_col = cnt[bulk].mean(axis=0)                                   # over 112 rows: +- sqrt(1/12/112) from the dither
    assert np.abs(per_col - ppc * shape).max() < 5 * math.sqrt(1.0 / 12.0 / 112) + 1e-9
    assert abs(cnt[bulk].sum() / (112 * 256 * ppc) - 1.0) < 1e-3
    p = L.generate_particles(cfg, 0)
    assert p["ix"].size == cnt.sum() == L.n_particles(cfg, 0)
    assert np.array_equal(np.bincount(p["ix"].astype(np.int64) * 256 + p["iy"], minlength=128 * 256).reshape(128, 256), cnt)
    assert np.all(p["w"] == np.float32(cfg["profile"]["p"][0] / ppc))


def test_polarisation_decomposition_on_the_axes_of_fig_1a():
    """A3c (Fig. 1(a)): theta is measured from the z axis, beta from the x axis inside the x-y plane.  theta = 0:
    pure S polarisation, a_sz = a; theta = 90 deg, beta = 0: a_px = a; theta = 90 deg, beta = 90 deg: a_py = a; and
    |a| is kept.  Swapping sine and cosine of either angle, or the x and y components, fails one of the three."""
    a = 0.02
    z, x, y = oracle.polarised(a, 0.0, 0.7)
    assert z == a and x == 0.0 and y == 0.0
    z, x, y = oracle.polarised(a, math.pi / 2, 0.0)
    assert abs(z) < 1e-17 and x == pytest.approx(a, rel=1e-15) and y == 0.0
    z, x, y = oracle.polarised(a, math.pi / 2, math.pi / 2)
    assert abs(z) < 1e-17 and abs(x) < 1e-17 and y == pytest.approx(a, rel=1e-15)
    for th, be in ((0.3, 1.1), (1.2, -0.4), (2.0, 2.5)):
        c = oracle.polarised(a, th, be)
        assert math.sqrt(sum(v * v for v in c)) == pytest.approx(a, rel=1e-14)
        assert c[0] == pytest.approx(a * math.cos(th), rel=1e-14)         # a_sz = a cos(theta) as printed
        assert math.hypot(c[1], c[2]) == pytest.approx(a * abs(math.sin(th)), rel=1e-14)      # a_p = a sin(theta)
        assert math.atan2(c[2], c[1]) == pytest.approx(math.atan2(math.sin(be) * math.sin(th), math.cos(be) * math.sin(th)), abs=1e-14)


def test_slab_extent_loads_only_the_slab_cells():
    """profile["slab"] ("a plasma slab is set at the center of the simulation box, and the vacuum space is usually
    set around the plasma slab"): exactly the cells x_lo <= i < x_hi, y_lo <= j < y_hi hold particles, and each of them
    holds what it holds without the slab (same ids, offsets, momenta, weights) -- an off-by-one edge, a profile
    re-stretched over the slab or re-drawn random numbers fail."""
    cfg = I.config("cbet_vac", nx=80, ny=64)
    x_lo, x_hi, y_lo, y_hi = cfg["profile"]["slab"]
    assert (x_lo, x_hi, y_lo, y_hi) == (4, 76, 3, 61) and cfg["profile"]["taper_cells"] == 0
    assert L.slab_extent(cfg) == (4, 76, 3, 61)
    full = I.config("cbet_vac", nx=80, ny=64)
    del full["profile"]["slab"]
    assert L.slab_extent(full) == (0, 80, 0, 64)
    for s in (0, 1):
        p, q = L.generate_particles(cfg, s), L.generate_particles(full, s)
        assert len(p["id"]) == L.n_particles(cfg, s) == 72 * 58
        inside = (q["ix"] >= x_lo) & (q["ix"] < x_hi) & (q["iy"] >= y_lo) & (q["iy"] < y_hi)
        assert inside.sum() == len(p["id"])
        for key in ("id", "ix", "iy", "fx", "fy", "ux", "uy", "w"):
            assert np.array_equal(p[key], q[key][inside]), key
        assert p["ix"].min() == x_lo and p["ix"].max() == x_hi - 1 and p["iy"].min() == y_lo and p["iy"].max() == y_hi - 1
        assert np.all(p["w"] == np.float32(0.4))          # hard edge: no taper by weight
    # the x-range argument of generate_particles intersects the slab
    part = L.generate_particles(cfg, 0, 0, 10)
    assert set(np.unique(part["ix"])) == set(range(4, 10))
