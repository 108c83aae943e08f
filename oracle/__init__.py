"""CPU oracle for the PM2D time step -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes wrapper around ``pm2d_oracle.c`` (plain C, double precision, written from the paper;
see that file's header for citations).  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.  It imports
nothing from ``paper_2404_14293_b200`` and the product imports nothing from here.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pm2d_oracle.c")
_LIB = os.path.join(_HERE, "libpm2d_oracle.so")

CIC, TSC, SINE = 0, 1, 2


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no fast-math, no OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("ncomp", C.c_int32), ("subcycle", C.c_int32),
                ("bc_y", C.c_int32), ("pad_", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dt", C.c_double)]


_dp = C.POINTER(C.c_double)


class _Species(C.Structure):
    _fields_ = [("mass", C.c_double), ("vth2", C.c_double), ("C", C.c_double), ("DD", C.c_double),
                ("sign", C.c_int32), ("shape", C.c_int32), ("mobile", C.c_int32), ("pad_", C.c_int32),
                ("np", C.c_int64),
                ("X", _dp), ("Y", _dp), ("ux", _dp), ("uy", _dp), ("w", _dp),
                ("uhx", _dp), ("uhy", _dp),
                ("n", _dp), ("Px", _dp), ("Py", _dp), ("Fx", _dp), ("Fy", _dp)]


class _Laser(C.Structure):
    _fields_ = [("a0", C.c_double), ("omega", C.c_double), ("y0", C.c_double), ("w0", C.c_double),
                ("t_rise", C.c_double), ("alpha", C.c_double), ("comp", C.c_int32), ("pad_", C.c_int32)]


class _State(C.Structure):
    _fields_ = [("g", _Grid), ("nsp", C.c_int32), ("nlaser", C.c_int32),
                ("sp", C.POINTER(_Species)), ("laser", C.POINTER(_Laser)),
                ("a_new", _dp), ("a_now", _dp), ("a_old", _dp),
                ("rho", _dp), ("phi", _dp), ("Ex", _dp), ("Ey", _dp), ("step", C.c_int64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_G.restype = C.c_double
        L.orc_G.argtypes = [C.c_int, C.c_double, C.c_double]
        L.orc_weights_1d.restype = C.c_int
        L.orc_weights_1d.argtypes = [C.c_int, C.c_double, C.c_double, _dp, C.POINTER(C.c_int)]
        L.orc_deposit.restype = None
        L.orc_deposit.argtypes = [C.POINTER(_Grid), C.c_int, C.c_double, C.c_int64] + [_dp] * 8
        L.orc_gather.restype = None
        L.orc_gather.argtypes = [C.POINTER(_Grid), C.c_int, C.c_double, C.c_double, C.c_double, _dp, _dp, _dp, _dp]
        L.orc_polarised.restype = None
        L.orc_polarised.argtypes = [C.c_double, C.c_double, C.c_double, _dp]
        L.orc_a_inc.restype = C.c_double
        L.orc_a_inc.argtypes = [C.POINTER(_Laser), C.c_double, C.c_double, C.c_double, C.c_double]
        L.orc_field_step.restype = None
        L.orc_field_step.argtypes = [C.POINTER(_State), _dp, C.c_double]
        L.orc_fft.restype = None
        L.orc_fft.argtypes = [_dp, _dp, C.c_int, C.c_int]
        L.orc_dft.restype = None
        L.orc_dft.argtypes = [_dp, _dp, _dp, _dp, C.c_int, C.c_int]
        L.orc_poisson.restype = None
        L.orc_poisson.argtypes = [C.POINTER(_Grid), _dp, _dp, C.c_int]
        L.orc_efield.restype = None
        L.orc_efield.argtypes = [C.POINTER(_Grid), _dp, _dp, _dp]
        L.orc_force.restype = None
        L.orc_force.argtypes = [C.POINTER(_Grid), C.POINTER(_Species), _dp, _dp, _dp, _dp, _dp]
        L.orc_initial_deposit.restype = None
        L.orc_initial_deposit.argtypes = [C.POINTER(_State)]
        L.orc_step.restype = None
        L.orc_step.argtypes = [C.POINTER(_State)]
        L.orc_predictor.restype = None
        L.orc_predictor.argtypes = [C.c_double] * 5 + [_dp, _dp]
        L.orc_corrector.restype = None
        L.orc_corrector.argtypes = [C.c_double] * 6 + [_dp, _dp]
        L.orc_refresh_fields.restype = None
        L.orc_refresh_fields.argtypes = [C.POINTER(_State)]
        L.orc_energies.restype = None
        L.orc_energies.argtypes = [C.POINTER(_State), _dp]
        _lib = L
    return _lib


def _p(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def _f64(a, n=None):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if n is not None:
        assert a.size == n, (a.size, n)
    return a


# ---------------------------------------------------------------------------------------------
# primitive calls (used by the pin tests)

def G(shape: int, DD: float, s: float) -> float:
    return lib().orc_G(shape, DD, s)


def weights_1d(shape: int, DD: float, xp: float):
    """-> (first node, np.ndarray of 4 weights)   [O1]"""
    W = np.zeros(4)
    cnt = C.c_int(0)
    first = lib().orc_weights_1d(shape, DD, xp, _p(W), C.byref(cnt))
    return first, W[: cnt.value]


def make_grid(nx, ny, dx, dy, dt, ncomp=1, subcycle=1, bc_y=0):
    return _Grid(nx, ny, ncomp, subcycle, bc_y, 0, dx, dy, dt)


def deposit(g: _Grid, shape, DD, X, Y, ux, uy, w):
    """-> n, Px, Py nodal arrays of shape (nx+1, ny)   [O2]"""
    X, Y, ux, uy, w = map(_f64, (X, Y, ux, uy, w))
    nn = (g.nx + 1) * g.ny
    n, Px, Py = np.zeros(nn), np.zeros(nn), np.zeros(nn)
    lib().orc_deposit(C.byref(g), shape, DD, X.size, _p(X), _p(Y), _p(ux), _p(uy), _p(w), _p(n), _p(Px), _p(Py))
    sh = (g.nx + 1, g.ny)
    return n.reshape(sh), Px.reshape(sh), Py.reshape(sh)


def gather(g: _Grid, shape, DD, Xp, Yp, Fx, Fy):
    Fx, Fy = _f64(Fx), _f64(Fy)
    fx, fy = C.c_double(0), C.c_double(0)
    lib().orc_gather(C.byref(g), shape, DD, Xp, Yp, _p(Fx), _p(Fy), C.byref(fx), C.byref(fy))
    return fx.value, fy.value


def fft(re, im, sign):
    re, im = _f64(re).copy(), _f64(im).copy()
    lib().orc_fft(_p(re), _p(im), re.size, sign)
    return re, im


def dft(re, im, sign):
    re, im = _f64(re), _f64(im)
    ore, oim = np.zeros_like(re), np.zeros_like(im)
    lib().orc_dft(_p(re), _p(im), _p(ore), _p(oim), re.size, sign)
    return ore, oim


def poisson(g: _Grid, rho, use_dft=False):
    rho = _f64(rho, (g.nx + 1) * g.ny)
    phi = np.zeros_like(rho)
    lib().orc_poisson(C.byref(g), _p(rho), _p(phi), int(use_dft))
    return phi.reshape(g.nx + 1, g.ny)


def efield(g: _Grid, phi):
    phi = _f64(phi, (g.nx + 1) * g.ny)
    Ex, Ey = np.zeros(g.nx * g.ny), np.zeros(g.nx * g.ny)
    lib().orc_efield(C.byref(g), _p(phi), _p(Ex), _p(Ey))
    return Ex.reshape(g.nx, g.ny), Ey.reshape(g.nx, g.ny)


def predictor(dt, h, x, u, F):
    uh, xh = C.c_double(0), C.c_double(0)
    lib().orc_predictor(dt, h, x, u, F, C.byref(uh), C.byref(xh))
    return uh.value, xh.value


def corrector(dt, h, x, u, uh, Fh):
    un, xn = C.c_double(0), C.c_double(0)
    lib().orc_corrector(dt, h, x, u, uh, Fh, C.byref(un), C.byref(xn))
    return un.value, xn.value


def polarised(a, theta, beta):
    """(a_sz, a_px, a_py) of P:L81 / Fig. 1(a): components 0 = z, 1 = x, 2 = y of the vector potential."""
    out = (C.c_double * 3)()
    lib().orc_polarised(float(a), float(theta), float(beta), out)
    return [out[0], out[1], out[2]]


def a_inc(laser: dict, x, y, t, Ly=1.0):
    L = _Laser(laser["a0"], laser.get("omega", 1.0), laser.get("y0", 0.0), laser.get("w0", 0.0),
               laser.get("t_rise", 0.0), laser.get("alpha", 0.0), laser.get("comp", 0), 0)
    return lib().orc_a_inc(C.byref(L), x, y, t, Ly)


def velocity_histogram(X, Y, u, w, box, umin, umax, nbins):
    """SURVEY 8f.4 (Fig. 9): weighted distribution of one velocity component over the particles whose cell
    (floor X, floor Y) lies in box = (i0, i1, j0, j1): hist[b] = sum of w_p over the particles with
    b = floor((u_p - umin) nbins / (umax - umin)), 0 <= b < nbins -- the definition, in float64."""
    X, Y, w = np.asarray(X, np.float64), np.asarray(Y, np.float64), np.asarray(w, np.float64)
    i0, i1, j0, j1 = box
    ix, iy = np.floor(X).astype(np.int64), np.floor(Y).astype(np.int64)
    inside = (ix >= i0) & (ix < i1) & (iy >= j0) & (iy < j1)
    t = np.floor((np.asarray(u, np.float64) - float(umin)) * (float(nbins) / (float(umax) - float(umin))))
    ok = inside & (t >= 0) & (t < nbins)
    h = np.zeros(nbins)
    np.add.at(h, t[ok].astype(np.int64), w[ok])
    return h


def probe_spectrum(h, dt_s, omegas):
    """SURVEY 8f.4 (Fig. 12(c), (e): "the frequent spectrum of the back-scattering laser light" recorded on the
    left boundary, of the transmitted light on the right one): power spectrum of a boundary history h[m, j] (record m
    taken at time (m0 + m) dt_s; the origin m0 drops out of the power), written out as the sum that defines it:
        A_j(w) = dt_s sum_m h[m, j] exp(-2 pi i w m dt_s),    P(w) = sum_j |A_j(w)|^2,    w in units of omega0."""
    h = np.asarray(h, np.float64)
    m = np.arange(h.shape[0])[:, None]
    out = np.zeros(len(omegas))
    for k, w in enumerate(omegas):
        A = dt_s * (h * np.exp(-2j * np.pi * float(w) * m * dt_s)).sum(axis=0)
        out[k] = (np.abs(A) ** 2).sum()
    return out


def mode_amplitudes(n, mx, my):
    """O9: Fourier-mode amplitudes of a nodal density n[(nx+1), ny], written out as the sum that
    defines them: A(mx, my) = sum_i sum_j v_i n[i, j] exp(-2 pi i (mx i/nx + my j/ny)), v_i = 1/2 on the wall columns
    (half control volumes, Q9).  The k-spectra of Figs. 7 and 14 are |A|^2 of delta n_e."""
    n = np.asarray(n, np.float64)
    nx, ny = n.shape[0] - 1, n.shape[1]
    v = np.ones(nx + 1)
    v[0] = v[nx] = 0.5
    i, j = np.arange(nx + 1)[:, None], np.arange(ny)[None, :]
    out = np.zeros(len(mx), complex)
    for k, (a, b) in enumerate(zip(mx, my)):
        out[k] = (v[:, None] * n * np.exp(-2j * np.pi * (a * i / nx + b * j / ny))).sum()
    return out


# ---------------------------------------------------------------------------------------------
class Oracle:
    """The whole step (O8) over numpy-owned arrays.

    species: list of dicts with keys mass, sign, T_keV, C (pressure_coeff), shape, DD, mobile and
    particle arrays X, Y (cell units), ux, uy, w; an immobile species may instead give ``n_fixed``
    (nodal density, shape (nx+1, ny)).  lasers: list of dicts (a0, omega, y0, w0, t_rise, alpha [rad], comp).
    subcycle: wave-equation steps of dt per particle step (Q21).  bc_y: 0 periodic, 1 absorbing y walls for a (Q23).
    """

    def __init__(self, nx, ny, dx, dy, dt, species, lasers=(), ncomp=1, subcycle=1, bc_y=0):
        self.g = make_grid(nx, ny, dx, dy, dt, ncomp, subcycle, bc_y)
        self.nn = nn = (nx + 1) * ny
        self.a = [np.zeros(ncomp * nn) for _ in range(3)]       # new, now, old
        self.rho, self.phi = np.zeros(nn), np.zeros(nn)
        self.Ex, self.Ey = np.zeros(nx * ny), np.zeros(nx * ny)
        self._sp = (_Species * len(species))()
        self.sp = []
        for k, s in enumerate(species):
            d = {}
            mobile = int(s.get("mobile", 1))
            npart = 0 if (not mobile and "X" not in s) else len(s["X"])
            for key in ("X", "Y", "ux", "uy", "w"):
                d[key] = _f64(s[key]).copy() if npart else np.zeros(1)
            d["uhx"], d["uhy"] = np.zeros(max(npart, 1)), np.zeros(max(npart, 1))
            for key in ("n", "Px", "Py", "Fx", "Fy"):
                d[key] = np.zeros(nn)
            mass = float(s.get("mass", 1.0))
            shape = int(s.get("shape", SINE))
            DD = float(s.get("DD", {CIC: 1.0, TSC: 2.0}.get(shape, 1.9)))
            if shape == CIC:
                assert DD == 1.0
            if shape == TSC:
                assert DD == 2.0
            self._sp[k] = _Species(mass, float(s.get("T_keV", 0.0)) / 511.0 / mass, float(s.get("C", 2.0)), DD,
                                   int(s["sign"]), shape, mobile, 0, npart,
                                   _p(d["X"]), _p(d["Y"]), _p(d["ux"]), _p(d["uy"]), _p(d["w"]),
                                   _p(d["uhx"]), _p(d["uhy"]),
                                   _p(d["n"]), _p(d["Px"]), _p(d["Py"]), _p(d["Fx"]), _p(d["Fy"]))
            d["np"] = npart
            d["mobile"] = mobile
            d["sign"] = int(s["sign"])
            self.sp.append(d)
        self._las = (_Laser * max(len(lasers), 1))()
        for k, l in enumerate(lasers):
            self._las[k] = _Laser(l["a0"], l.get("omega", 1.0), l.get("y0", 0.0), l.get("w0", 0.0),
                                  l.get("t_rise", 0.0), l.get("alpha", 0.0), l.get("comp", 0), 0)
        self.st = _State(self.g, len(species), len(lasers), self._sp, self._las,
                         _p(self.a[0]), _p(self.a[1]), _p(self.a[2]),
                         _p(self.rho), _p(self.phi), _p(self.Ex), _p(self.Ey), 0)
        # item (1) at step 0; immobile species: n_fixed if given, else deposited once from their
        # particles (Q13: callers pass the electron deposit as n_fixed for exact neutrality)
        lib().orc_initial_deposit(C.byref(self.st))
        for k, s in enumerate(species):
            if not self.sp[k]["mobile"]:
                if "n_fixed" in s:
                    self.sp[k]["n"][:] = _f64(s["n_fixed"], nn).ravel()
                elif self.sp[k]["np"]:
                    d = self.sp[k]
                    n, _, _ = deposit(self.g, self._sp[k].shape, self._sp[k].DD, d["X"], d["Y"], d["ux"], d["uy"], d["w"])
                    d["n"][:] = n.ravel()

    # views ----------------------------------------------------------------------------------
    def _abuf(self, which):
        ptr = {"new": self.st.a_new, "now": self.st.a_now, "old": self.st.a_old}[which]
        addr = C.addressof(ptr.contents)
        for b in self.a:
            if b.ctypes.data == addr:
                return b.reshape(self.g.ncomp, self.g.nx + 1, self.g.ny)
        raise RuntimeError("lost buffer")

    @property
    def a_now(self):
        return self._abuf("now")

    @property
    def a_old(self):
        return self._abuf("old")

    def probe(self, comp=0):
        """Boundary records of the current time level t = step * S * dt (Fig. 12(b), (d); "the time
        evolution of back-scattering laser light on the left boundary"): the scattered field a - a_inc on the left
        wall (the incident wave split off as in P:L122) and a on the right wall, each [ny]."""
        g = self.g
        t = self.st.step * max(g.subcycle, 1) * g.dt
        a = self.a_now[comp]
        inc = np.zeros(g.ny)
        for k in range(self.st.nlaser):
            L = self._las[k]
            if L.comp == comp:
                for j in range(g.ny):
                    inc[j] += lib().orc_a_inc(C.byref(L), 0.0, j * g.dy, t, g.ny * g.dy)
        return a[0] - inc, a[g.nx].copy()

    def moment(self, s, name):
        return self.sp[s][name].reshape(self.g.nx + 1, self.g.ny)

    @property
    def step_index(self):
        return self.st.step

    def step(self, nsteps=1):
        for _ in range(nsteps):
            lib().orc_step(C.byref(self.st))

    def refresh_fields(self):
        lib().orc_refresh_fields(C.byref(self.st))

    def force_now(self, s):
        """Eq. 16 for the current state: E of the current densities, a^n, n^n  -> (Fx, Fy)."""
        self.refresh_fields()
        Fx, Fy = np.zeros(self.nn), np.zeros(self.nn)
        lib().orc_force(C.byref(self.g), C.byref(self._sp[s]), self.st.a_now, _p(self.Ex), _p(self.Ey), _p(Fx), _p(Fy))
        sh = (self.g.nx + 1, self.g.ny)
        return Fx.reshape(sh), Fy.reshape(sh)

    def energies(self):
        self.refresh_fields()
        out = np.zeros(3 + 2 * len(self.sp))
        lib().orc_energies(C.byref(self.st), _p(out))
        d = {"W_es": out[0], "W_int": out[1], "W_em": out[2],
             "W_kin": out[3::2].copy(), "W_th": out[4::2].copy()}
        d["W_total"] = float(out.sum())
        return d


# ---- an Oracle from a pm2d_inputs config (tests, smoke, the CPU legs of bench.py) ----------------------------------
def species_from_arrays(sp_cfg, parts=None, n_fixed=None):
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


def from_config(cfg, particles=None):
    """particles: optional list (per species) of dicts as returned by oracle.loader.generate_particles."""
    from . import loader
    g = cfg["grid"]
    grid = make_grid(g["nx"], g["ny"], g["dx"], g["dy"], g["dt"], g["ncomp"])
    if particles is None:
        particles = [loader.generate_particles(cfg, s) if sp["load"] != 0 else None
                     for s, sp in enumerate(cfg["species"])]
    species = []
    # Q13: an immobile species without particles neutralises the summed deposit of the mobile
    # species of opposite sign at t = 0
    for s, sp in enumerate(cfg["species"]):
        if particles[s] is not None:
            species.append(species_from_arrays(sp, particles[s]))
        else:
            species.append(None)
    for s, sp in enumerate(cfg["species"]):
        if species[s] is None:
            nfix = np.zeros((g["nx"] + 1, g["ny"]))
            for t, sq in enumerate(cfg["species"]):
                if particles[t] is not None and sq["sign"] == -sp["sign"]:
                    d = species[t]
                    n, _, _ = deposit(grid, sq["shape"], sq["DD"], d["X"], d["Y"], d["ux"], d["uy"], d["w"])
                    nfix += n
            species[s] = species_from_arrays(sp, None, nfix)
    lasers = [dict(a0=l["a0"], omega=l["omega"], y0=l["y0"], w0=l["w0"], t_rise=l["t_rise"], comp=l["comp"],
                   alpha=l.get("alpha", 0.0)) for l in cfg["lasers"]]
    return Oracle(g["nx"], g["ny"], g["dx"], g["dy"], g["dt"], species, lasers, g["ncomp"],
                         subcycle=g.get("subcycle", 1), bc_y=g.get("bc_y", 0)), particles
