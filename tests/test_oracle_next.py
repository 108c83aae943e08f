"""Pins of the S§8(f).1 widening of the oracle: oblique incidence (Eq. 5; Q22) and particle
sub-cycling (Q21).  Closed forms and invariants only; no GPU."""
import math

import numpy as np
import pytest

import oracle


def _vacuum_oracle(nx, ny, dx, dt, lasers, subcycle=1):
    sp = [dict(sign=-1, mass=1.0, T_keV=0.0, mobile=0, shape=oracle.CIC, DD=1.0, n_fixed=np.zeros((nx + 1, ny)))]
    return oracle.Oracle(nx, ny, dx, dx, dt, sp, lasers, subcycle=subcycle)


# ---- Eq. 5 -------------------------------------------------------------------------------------------
def test_P15_eq5_rotation_worked_values():
    """Eq. 5 substituted into Eq. 4 by hand: box point (x', y') -> beam point (x, y), y' from the beam centre."""
    al = math.radians(15.0)
    las = dict(a0=0.008, w0=30.0, y0=50.0, t_rise=0.0, omega=1.0 / 0.9995, alpha=al)     # beam 2 of P:L380
    Ly = 400.0
    lead = 0.5 * Ly * math.sin(al)            # turn-on front (Q22): 51.76 T0 here
    hit = 0
    for xq, yq, t in ((0.0, 50.0, 3.0), (0.0, 50.0, 53.0), (0.0, 62.0, 60.0), (0.05, 31.5, 80.0), (0.05, 50.0 - 7.25, 47.3),
                      (0.05, 50.0 - 7.25, 97.3)):
        d = yq - 50.0
        xb = xq * math.cos(al) - d * math.sin(al)
        yb = xq * math.sin(al) + d * math.cos(al)
        on = t - xb > lead
        hit += on
        ref = 0.008 * math.exp(-(yb / 30.0) ** 2) * math.cos(2 * math.pi / 0.9995 * (t - xb)) if on else 0.0
        assert oracle.a_inc(las, xq, yq, t, Ly) == pytest.approx(ref, abs=1e-15)
    assert hit == 4
    # nearest periodic image of the beam centre: y' and y' + Ly are the same boundary point
    assert oracle.a_inc(las, 0.0, 60.0 - Ly, 70.0, Ly) == pytest.approx(oracle.a_inc(las, 0.0, 60.0, 70.0, Ly), abs=1e-15)
    assert oracle.a_inc(las, 0.0, 60.0, 70.0, Ly) != 0.0
    # alpha = 0 is Eq. 4 at normal incidence, whatever Ly
    l0 = dict(las, alpha=0.0)
    assert oracle.a_inc(l0, 0.05, 62.0, 40.0, Ly) == oracle.a_inc(l0, 0.05, 62.0, 40.0, 1.0)


def test_P15_oblique_plane_wave_fills_vacuum_box():
    """A plane wave injected at an angle that fits the periodic box (omega sin(alpha) Ly = m) fills a vacuum box
    with a0 cos(2 pi (t - x' cos(alpha) + y' sin(alpha))): amplitude a0, transverse mode exactly -m (the sign of
    Eq. 5 as printed: the beam axis is (cos alpha, -sin alpha) in box coordinates), longitudinal wavenumber
    cos(alpha) up to the dispersion of the stencil, nothing coming back from either wall."""
    nx, ny, dx, dt, a0, m = 240, 256, 0.05, 0.035, 0.01, 3
    Ly = ny * dx
    al = math.asin(m / Ly)
    o = _vacuum_oracle(nx, ny, dx, dt, [dict(a0=a0, t_rise=3.0, alpha=al)])
    nsteps = int(26.0 / dt)
    o.step(nsteps)
    a = o.a_now[0]                                   # (nx+1, ny)
    A = np.fft.fft(a, axis=1) / ny                   # transverse modes, row by row
    rows = slice(10, nx - 10)
    power = (np.abs(A[rows]) ** 2).sum(axis=0)
    # a real field cos(.. + 2 pi m y / Ly) has modes +m and -m of equal size; the direction sits in the x phase
    assert set(np.argsort(power)[-2:]) == {m, ny - m}
    assert power[[m, ny - m]].sum() / power.sum() > 0.9995
    # a = Re[a0 exp(i(2 pi t - kx x' + 2 pi m y'/Ly))]: the coefficient of exp(+i 2 pi m y'/Ly) is (a0/2) exp(i(2 pi t - kx x'))
    c = A[:, m]
    assert np.abs(2 * np.abs(c[rows]) / a0 - 1.0).max() < 0.015
    ph = np.unwrap(np.angle(c[rows]))
    kx = -np.polyfit(np.arange(nx + 1)[rows] * dx, ph, 1)[0] / (2 * math.pi)
    # discrete dispersion of Eq. 6 in vacuum: sin^2(pi dt)/dt^2 = sin^2(kx' dx/2)/dx^2 + sin^2(ky' dx/2)/dx^2
    ky = m / Ly
    kx_d = math.asin(math.sqrt((math.sin(math.pi * dt) / dt) ** 2 - (math.sin(math.pi * ky * dx) / dx) ** 2) * dx) / (math.pi * dx)
    assert kx == pytest.approx(kx_d, rel=2e-3)
    assert kx == pytest.approx(math.cos(al), rel=1e-2)
    # with the opposite sign of alpha the wave goes the other way in y: conj pattern, i.e. the phase of mode +m
    # now decreases with -x'... checked through the mode that carries exp(-i kx x')
    o2 = _vacuum_oracle(nx, ny, dx, dt, [dict(a0=a0, t_rise=3.0, alpha=-al)])
    o2.step(nsteps)
    c2 = (np.fft.fft(o2.a_now[0], axis=1) / ny)[:, ny - m]
    ph2 = np.unwrap(np.angle(c2[rows]))
    assert -np.polyfit(np.arange(nx + 1)[rows] * dx, ph2, 1)[0] / (2 * math.pi) == pytest.approx(kx_d, rel=2e-3)


def test_P15_oblique_gaussian_beam_axis():
    """The centre of a Gaussian beam injected at alpha moves along (cos alpha, -sin alpha): at depth x' the
    centroid of the cycle-averaged a^2 sits at y0 - x' tan(alpha)."""
    nx, ny, dx, dt = 200, 256, 0.05, 0.035
    al, y0, w0 = math.radians(15.0), 7.0, 1.5
    o = _vacuum_oracle(nx, ny, dx, dt, [dict(a0=0.01, t_rise=2.0, alpha=al, y0=y0, w0=w0)])
    o.step(int(16.0 / dt))
    acc = np.zeros((nx + 1, ny))
    per = int(round(1.0 / dt))
    for _ in range(per):
        o.step()
        acc += o.a_now[0] ** 2
    y = np.arange(ny) * dx
    for i in (20, 100, 180):
        cen = (acc[i] * y).sum() / acc[i].sum()
        shift = i * dx * math.tan(al)
        # one cell + 4 % of the shift: Eq. 4 prescribes a flat phase front on a boundary that cuts the beam obliquely,
        # so a beam this narrow (w0 = 1.5 lambda0) steers slightly; a wrong sign or a sin/cos swap is off by > 100 %
        assert cen == pytest.approx(y0 - shift, abs=0.05 + 0.04 * shift)
    # width across the beam axis stays w0 (Rayleigh length pi w0^2 = 7 lambda0: mild spreading allowed)
    i = 20
    var = (acc[i] * (y - (acc[i] * y).sum() / acc[i].sum()) ** 2).sum() / acc[i].sum()
    # a^2 ~ exp(-2 yb^2 / w0^2), yb = (y' - centre) cos(alpha)  =>  var(y') = w0^2 / (4 cos^2 alpha)
    assert math.sqrt(var) == pytest.approx(w0 / (2 * math.cos(al)), rel=0.05)


# ---- sub-cycling ----------------------------------------------------------------------------------------
def test_P16_subcycled_wave_steps_equal_plain_steps_without_plasma():
    """Without plasma the particle step plays no part: N particle steps of S wave steps are S N plain steps,
    bit for bit (pins the time of every sub-step that goes into the boundary condition)."""
    nx, ny, dx, dt, S = 96, 16, 0.05, 0.035, 5
    las = [dict(a0=0.02, t_rise=1.0, w0=0.3, y0=0.4)]
    o1 = _vacuum_oracle(nx, ny, dx, dt, las)
    o5 = _vacuum_oracle(nx, ny, dx, dt, las, subcycle=S)
    o1.step(12 * S)
    o5.step(12)
    assert np.abs(o1.a_now[0]).max() > 0.01
    assert np.array_equal(o1.a_now[0], o5.a_now[0])
    assert np.array_equal(o1.a_old[0], o5.a_old[0])


def test_P16_subcycled_free_streaming_and_constant_force():
    """A neutral pressure-free particle moves by u S dt per step (exact); Heun's step is exact for a constant
    force, so a uniform E = -grad(phi) cannot be built here -- the free flight pins dt_p = S dt in Eq. 17/19."""
    nx, ny, dx, dt, S = 32, 8, 0.05, 0.035, 5
    X, Y = np.array([10.25]), np.array([3.5])
    sp = [dict(sign=0, mass=1.0, T_keV=0.0, C=0.0, shape=oracle.SINE, DD=1.9, mobile=1, X=X, Y=Y,
               ux=np.array([0.02]), uy=np.array([-0.03]), w=np.array([0.1]))]
    o = oracle.Oracle(nx, ny, dx, dx, dt, sp, subcycle=S)
    o.step(7)
    assert o.sp[0]["X"][0] == pytest.approx(10.25 + 0.02 * 7 * S * dt / dx, abs=1e-12)
    assert o.sp[0]["Y"][0] == pytest.approx(3.5 - 0.03 * 7 * S * dt / dx, abs=1e-12)


def test_P16_subcycled_plasma_oscillation_period():
    """Cold plasma oscillation with S = 5: the period, on the time axis t = step S dt, is 1/sqrt(n0) T0 up to the
    phase error of Heun's method at omega_pe dt_p (the same pin as P11 at five times the step)."""
    nx, ny, dx, dt, S, n0, px = 64, 2, 0.05, 0.035, 5, 0.1, 8
    g = oracle.make_grid(nx, ny, dx, dx, dt)
    xs = (np.arange(nx * px) + 0.5) / px
    X0, Y0 = [a.ravel() for a in np.meshgrid(xs, np.arange(ny) + 0.5, indexing="ij")]
    w = np.full(X0.size, n0 / px)
    n_bg, _, _ = oracle.deposit(g, oracle.TSC, 2.0, X0, Y0, 0 * X0, 0 * X0, w)
    K = 2 * math.pi * 2 / nx
    X = X0 + 0.02 * np.sin(K * X0)
    sp = [dict(sign=-1, mass=1.0, T_keV=0.0, C=0.0, shape=oracle.TSC, DD=2.0, mobile=1, X=X, Y=Y0, ux=0 * X, uy=0 * X, w=w),
          dict(sign=1, mass=1836.0, T_keV=0.0, mobile=0, shape=oracle.TSC, DD=2.0, n_fixed=n_bg)]
    o = oracle.Oracle(nx, ny, dx, dx, dt, sp, subcycle=S)
    i = np.arange(nx + 1)[:, None]
    amp, t = [], []
    for n in range(120):
        amp.append((o.moment(0, "n") * np.cos(K * i)).sum())
        t.append(n * S * dt)
        o.step()
    y = np.asarray(amp) - np.mean(amp)
    s = np.sign(y)
    idx = np.where(s[:-1] * s[1:] < 0)[0]
    t = np.asarray(t)
    tc = t[idx] - y[idx] * (t[idx + 1] - t[idx]) / (y[idx + 1] - y[idx])
    period = 2.0 * (tc[-1] - tc[0]) / (len(tc) - 1)
    th = 2 * math.pi * math.sqrt(n0) * S * dt                      # omega_pe dt_p
    # one step of Eqs. 17, 19 on x'' = -omega^2 x is the matrix [[1 - th^2/2 + th^4/8, th - th^3/4], [-th + th^3/4,
    # 1 - th^2/2]] in (x, u/omega): phase per step phi = arccos(trace / (2 sqrt(det))) = th (1 - th^2/12 + ...)
    tr, det = 2 - th * th + th ** 4 / 8, 1 - th ** 4 / 8
    phi = math.acos(tr / (2 * math.sqrt(det)))
    assert phi / th == pytest.approx(1 - th * th / 12, abs=2e-4)
    # the finite-grid factors of mode 2 on 64 cells (TSC smoothing, differenced E) lengthen the period by 0.6 %
    assert period == pytest.approx(1.0 / math.sqrt(n0) * th / phi, rel=0.01)
    # a push with dt instead of S dt would give a period S times longer on this time axis


def test_P15_oblique_turning_point_cos2_theta():
    """"the propagation of the incident laser beam is stopped when n_e = cos^2(theta) n_c".  A plane wave at
    theta = asin(1/3.2) = 18.2 degrees in a fixed linear ramp n_e = x'/L_n (L_n = 10 lambda0) is an Airy pattern
    Ai((x' - x_t)/l) with x_t = L_n cos^2(theta) = 9.02 lambda0 (10 lambda0 at normal incidence) and l =
    (L_n/k0^2)^(1/3) = 0.633 lambda0: last maximum of the cycle-averaged a^2 at x_t - 1.0188 l, evanescent beyond."""
    nx, ny, dx, dt, Ln = 240, 64, 0.05, 0.035, 10.0
    Ly = ny * dx
    ne = np.repeat((np.arange(nx + 1) * dx / Ln)[:, None], ny, axis=1)
    ell = (Ln / (2 * math.pi) ** 2) ** (1.0 / 3.0)
    xs = np.arange(nx + 1) * dx
    found = {}
    for name, al in (("normal", 0.0), ("oblique", math.asin(1.0 / Ly))):
        sp = [dict(sign=-1, mass=1.0, T_keV=0.0, mobile=0, shape=oracle.CIC, DD=1.0, n_fixed=ne)]
        o = oracle.Oracle(nx, ny, dx, dx, dt, sp, [dict(a0=0.01, t_rise=3.0, alpha=al)])
        o.step(int(34.0 / dt))                     # in, back, and a few periods to settle
        acc = np.zeros(nx + 1)
        per = int(round(2.0 / dt))
        for _ in range(per):
            o.step()
            acc += (o.a_now[0] ** 2).mean(axis=1)
        # last interior maximum of the standing pattern, refined by a parabola through its neighbours
        i = max(k for k in range(2, nx - 1) if acc[k] > acc[k - 1] and acc[k] >= acc[k + 1] and acc[k] > 0.2 * acc.max())
        off = 0.5 * (acc[i - 1] - acc[i + 1]) / (acc[i - 1] - 2 * acc[i] + acc[i + 1])
        found[name] = (i + off) * dx
        xt = Ln * math.cos(al) ** 2
        assert found[name] == pytest.approx(xt - 1.0188 * ell, abs=0.12)
        beyond = acc[xs > xt + 2.0 * ell]
        assert beyond.max() < 0.02 * acc.max()
    assert found["normal"] - found["oblique"] == pytest.approx(Ln * (1.0 / Ly) ** 2, abs=0.1)      # L_n sin^2(theta)


# ---- a8: Fourier-mode amplitudes ---------------------------------------------------------------------------
def test_P17_mode_amplitudes_closed_form_and_fft():
    """A single cosine product has the closed-form amplitude eps nx ny / 4 in its four modes and nx ny in (0, 0);
    for any field the wall-halved sum over i = 0..nx is the periodic DFT of the field with its two wall columns
    averaged into one (numpy's fft2 as the independent routine)."""
    nx, ny, m, l, eps = 24, 16, 3, 2, 0.25
    i, j = np.arange(nx + 1)[:, None], np.arange(ny)[None, :]
    n = 1.0 + eps * np.cos(2 * np.pi * m * i / nx) * np.cos(2 * np.pi * l * j / ny)
    A = oracle.mode_amplitudes(n, [0, m, -m, m, 1, m], [0, l, l, -l, l, 0])
    assert A[0] == pytest.approx(nx * ny, abs=1e-9)
    for k in (1, 2, 3):
        assert A[k] == pytest.approx(eps * nx * ny / 4, abs=1e-9)
    assert abs(A[4]) < 1e-9 and abs(A[5]) < 1e-9
    # a phase: n = sin(2 pi (m i/nx + l j/ny)) has A(m, l) = nx ny / (2i), A(-m, -l) = -nx ny / (2i)
    n2 = np.sin(2 * np.pi * (m * i / nx + l * j / ny))
    B = oracle.mode_amplitudes(n2, [m, -m], [l, -l])
    assert B[0] == pytest.approx(nx * ny / 2j, abs=1e-9) and B[1] == pytest.approx(-nx * ny / 2j, abs=1e-9)
    rng = np.random.default_rng(7)
    r = rng.random((nx + 1, ny))
    per = r[:nx].copy()
    per[0] = 0.5 * (r[0] + r[nx])
    F = np.fft.fft2(per)
    mxs, mys = [0, 1, 5, -2, 11], [0, 3, -1, 7, 8]
    C = oracle.mode_amplitudes(r, mxs, mys)
    for k in range(len(mxs)):
        assert C[k] == pytest.approx(F[mxs[k] % nx, mys[k] % ny], abs=1e-9)


def test_P18_velocity_histogram_of_a_maxwellian_and_a_box():
    """The histogram of 4e5 seeded normal velocities follows the Gaussian bin integrals within counting noise; the
    box selects by cell; the total weight inside [umin, umax) is conserved; numpy's histogram agrees where no value
    sits on a bin edge."""
    rng = np.random.default_rng(3)
    N, vth = 400000, 0.05
    X, Y = rng.random(N) * 40, rng.random(N) * 16
    u = (vth * rng.standard_normal(N)).astype(np.float32)
    w = np.full(N, 0.25)
    nb, lo, hi = 64, -0.2, 0.2
    h = oracle.velocity_histogram(X, Y, u, w, (0, 40, 0, 16), lo, hi, nb)
    assert h.sum() == pytest.approx(0.25 * ((u >= lo) & (u < hi)).sum(), rel=1e-12)
    edges = np.linspace(lo, hi, nb + 1)
    cdf = np.array([0.5 * (1 + math.erf(e / (vth * math.sqrt(2)))) for e in edges])
    expect = N * 0.25 * np.diff(cdf)
    big = expect > 200
    assert np.abs(h[big] / expect[big] - 1).max() < 5 * np.sqrt(1.0 / (4 * expect[big].min()))
    ref, _ = np.histogram(u.astype(np.float64), bins=nb, range=(lo, hi), weights=w)
    assert np.abs(h - ref).sum() <= 0.25 * 4                      # at most a few values on a rounded edge
    sub = oracle.velocity_histogram(X, Y, u, w, (10, 20, 4, 8), lo, hi, nb)
    sel = (np.floor(X) >= 10) & (np.floor(X) < 20) & (np.floor(Y) >= 4) & (np.floor(Y) < 8) & (u >= lo) & (u < hi)
    assert sub.sum() == pytest.approx(0.25 * sel.sum(), rel=1e-12)
    # a single particle: bin 3 of 8 on [0, 0.8) holds u = 0.35
    one = oracle.velocity_histogram([1.5], [2.5], [0.35], [2.0], (1, 2, 2, 3), 0.0, 0.8, 8)
    assert list(one) == [0, 0, 0, 2.0, 0, 0, 0, 0]
    assert oracle.velocity_histogram([1.5], [2.5], [0.35], [2.0], (2, 3, 2, 3), 0.0, 0.8, 8).sum() == 0.0


# ---- S§8(f).2: absorbing y walls for a ("on all of four boundaries"; Q23) ------------------------------
def _vac(nx, ny, dx, dt, bc_y, lasers=()):
    sp = [dict(sign=-1, mass=1.0, T_keV=0.0, mobile=0, shape=oracle.CIC, DD=1.0, n_fixed=np.zeros((nx + 1, ny)))]
    return oracle.Oracle(nx, ny, dx, dx, dt, sp, lasers, bc_y=bc_y)


def test_P19_four_absorbing_walls_let_a_ring_out():
    """A wave packet at rest in the middle of a square vacuum box splits into an outgoing ring.  With absorbing y
    walls it leaves through all four sides and the corners: under 0.5 % of the field energy is left once the ring
    has passed the corners; in the y-periodic box the part that crossed the y walls comes back in and stays."""
    nx, ny, dx, dt = 127, 128, 0.05, 0.035                 # 128 x 128 nodes (ny: a power of two for the Poisson FFT)
    x = np.arange(nx + 1)[:, None] * dx
    y = np.arange(ny)[None, :] * dx
    r2 = (x - 3.175) ** 2 + (y - 3.175) ** 2
    blob = np.exp(-r2 / 0.6 ** 2) * np.cos(2 * math.pi * np.sqrt(r2))
    left = {}
    for bc in (0, 1):
        o = _vac(nx, ny, dx, dt, bc)
        o.a_now[0][:] = blob
        o.a_old[0][:] = blob
        e0 = o.energies()["W_em"]
        o.step(int(7.5 / dt))                    # half diagonal 4.5 + packet
        left[bc] = o.energies()["W_em"] / e0
    assert left[1] < 5e-3
    assert left[0] > 0.2


def test_P19_y_wall_transmits_an_oblique_beam():
    """A Gaussian beam aimed at the lower y wall (alpha = +30 degrees: axis (cos, -sin)) crosses it: with the absorbing
    wall the upper half of the box stays dark (reflection coefficient of the second-order condition at 60 degrees
    from the wall normal: ((1 - cos 60)/(1 + cos 60))^2 = 1/9 in amplitude, 1.2 % in energy; measured against the
    periodic box, where the beam re-enters through the upper wall)."""
    nx, ny, dx, dt = 200, 128, 0.05, 0.035
    las = [dict(a0=0.01, t_rise=2.0, alpha=math.radians(30.0), y0=2.2, w0=0.9)]
    up = {}
    for bc in (0, 1):
        o = _vac(nx, ny, dx, dt, bc, las)
        o.step(int(20.0 / dt))
        acc = np.zeros((nx + 1, ny))
        for _ in range(int(round(1.0 / dt))):
            o.step()
            acc += o.a_now[0] ** 2
        # the beam meets the wall y = 0 near x' = 2.2 / tan(30) = 3.8; beyond x' = 5 everything above mid-height is
        # either reflected or re-entered light
        up[bc] = acc[100:, ny // 2:].sum() / acc.sum()
    assert up[0] > 0.2                      # periodic: the beam comes back in from above
    assert up[1] < 0.02                     # absorbing: only the reflected part


# ---- S§8(f).4: boundary records and their frequency spectrum (Fig. 12) --------------------------------
def test_P20_probe_spectrum_closed_form_fft_and_parseval():
    """The defining sum against what mathematics fixes: a sampled cosine whose period divides the record has
    A(w0) = T/2 exactly and nothing in the other bins; at the bin frequencies k/T the sum is numpy's FFT; Parseval."""
    M, dt_s, ny = 400, 0.035, 3
    T = M * dt_s                                            # 14: w0 = 1 -> 14 periods, w = 0.5 -> 7
    m = np.arange(M)[:, None]
    h = np.cos(2 * math.pi * 1.0 * m * dt_s) * np.array([1.0, 2.0, -0.5])[None, :]
    P = oracle.probe_spectrum(h, dt_s, [1.0, 0.5, 2.0 / T, 0.0])
    assert P[0] == pytest.approx((T / 2) ** 2 * (1 + 4 + 0.25), rel=1e-12)
    assert np.all(P[1:] < 1e-20 * P[0])
    rng = np.random.default_rng(5)
    r = rng.standard_normal((M, ny))
    ks = np.arange(M // 2 + 1)
    Pr = oracle.probe_spectrum(r, dt_s, ks / T)
    assert np.allclose(Pr, (np.abs(dt_s * np.fft.rfft(r, axis=0)) ** 2).sum(axis=1), rtol=1e-10)
    Pall = oracle.probe_spectrum(r, dt_s, np.arange(M) / T)
    assert Pall.sum() == pytest.approx(M * dt_s ** 2 * (r ** 2).sum(), rel=1e-10)
    # a phase-shifted sine has the same power: the time origin drops out
    h2 = np.sin(2 * math.pi * 1.0 * (m + 17.3) * dt_s) * np.ones((1, ny))
    assert oracle.probe_spectrum(h2, dt_s, [1.0])[0] == pytest.approx(ny * (T / 2) ** 2, rel=1e-12)


def test_P20_probe_of_a_plane_wave_crossing_a_vacuum_box():
    """Oracle.probe(): once a plane wave fills a vacuum box, the left record (a - a_inc at the level just reached)
    is empty — a wrong sign, a record one time level off (2 pi dt = 22 % of a0) or a missing beam would all show —
    and the right record is the transmitted wave: amplitude a0, spectrum peaked at omega0."""
    nx, ny, dx, dt, a0 = 200, 8, 0.05, 0.035, 0.01
    o = _vac(nx, ny, dx, dt, 0, [dict(a0=a0, t_rise=3.0)])
    o.step(int(20.0 / dt))
    M = 400                                                 # 14 periods
    left, right = np.zeros((M, ny)), np.zeros((M, ny))
    for k in range(M):
        o.step()
        left[k], right[k] = o.probe(0)
    assert np.abs(left).max() < 0.01 * a0
    assert np.abs(right).max() == pytest.approx(a0, rel=0.01)
    P = oracle.probe_spectrum(right, dt, [1.0, 0.5, 1.5])       # bins of the 14-period record
    assert P[0] == pytest.approx(ny * (a0 * M * dt / 2) ** 2, rel=0.02)
    assert P[1] < 1e-3 * P[0] and P[2] < 1e-3 * P[0]
