"""ctypes binding of libpm2d.so (include/pm2d.h): argument marshalling only.

PyTorch supplies the device workspace (a uint8 CUDA tensor) and the CUDA stream; every step of the
method runs inside the library's kernels.  There is no CPU path: importing works without a GPU
(symbols are checked), but creating a simulation raises if CUDA or the library is missing.
"""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpm2d.so")

MAX_SPECIES, MAX_LASERS, TILE = 4, 4, 32
CIC, TSC, SINE = 0, 1, 2
LOAD_NONE, LATTICE_COLD, RANDOM_MAXWELL, NUMBER_WEIGHTED = 0, 1, 2, 3
PROFILE_UNIFORM, PROFILE_LINEAR, PROFILE_EXP_CAPPED, PROFILE_FILAMENT_Y = 0, 1, 2, 3
FIELD_A, FIELD_PHI, FIELD_ENODE, FIELD_FORCE, FIELD_FORCE_REF = 0, 1, 2, 3, 4
MOMENT_N, MOMENT_PX, MOMENT_PY = 0, 1, 2
BC_Y_PERIODIC, BC_Y_ABSORB = 0, 1
ORDER_AUTO, ORDER_CELL_MAJOR, ORDER_LAYERED, ORDER_RANDOM, ORDER_LANES, LAYERS = 0, 1, 2, 3, 4, 16
PHASES = ("field", "poisson", "force", "stage_a", "stage_b", "rebin")


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("ncomp", C.c_int32), ("rebin_every", C.c_int32),
                ("eager_moments", C.c_int32), ("track_ids", C.c_int32), ("particle_order", C.c_int32), ("subcycle", C.c_int32),
                ("bc_y", C.c_int32), ("probe_steps", C.c_int32),
                ("dx", C.c_double), ("dy", C.c_double), ("dt", C.c_double)]


class Species(C.Structure):
    _fields_ = [("mass", C.c_double), ("T_keV", C.c_double), ("pressure_coeff", C.c_double), ("DD", C.c_double),
                ("sign", C.c_int32), ("shape", C.c_int32), ("mobile", C.c_int32), ("load", C.c_int32),
                ("ppc_x", C.c_int32), ("ppc_y", C.c_int32), ("capacity", C.c_int64)]


class Profile(C.Structure):
    _fields_ = [("kind", C.c_int32), ("taper_cells", C.c_int32), ("p", C.c_double * 4), ("taper_cells_y", C.c_int32), ("pad_", C.c_int32),
                ("slab", C.c_int32 * 4)]


class Laser(C.Structure):
    _fields_ = [("a0", C.c_double), ("omega", C.c_double), ("y0", C.c_double), ("w0", C.c_double),
                ("t_rise", C.c_double), ("alpha", C.c_double), ("comp", C.c_int32), ("pad_", C.c_int32)]


class Diag(C.Structure):
    _fields_ = [("step", C.c_int64), ("time", C.c_double), ("W_es", C.c_double), ("W_int", C.c_double), ("W_em", C.c_double),
                ("W_kin", C.c_double * MAX_SPECIES), ("W_th", C.c_double * MAX_SPECIES),
                ("charge", C.c_double * MAX_SPECIES), ("count", C.c_int64 * MAX_SPECIES), ("W_total", C.c_double)]


_vp = C.c_void_p
_fp = C.POINTER(C.c_float)
_ip = C.POINTER(C.c_int32)
_lp = C.POINTER(C.c_int64)

# every symbol include/pm2d.h declares: name -> (restype, argtypes)
SYMBOLS = {
    "pm2d_query_workspace": (C.c_size_t, [C.POINTER(Grid), C.POINTER(Species), C.c_int]),
    "pm2d_init": (C.c_int, [C.POINTER(Grid), C.POINTER(Species), C.c_int, C.POINTER(Profile), C.POINTER(Laser), C.c_int,
                            C.c_uint64, _vp, C.c_size_t, _vp, C.POINTER(_vp)]),
    "pm2d_step": (C.c_int, [_vp, C.c_int]),
    "pm2d_step_async": (C.c_int, [_vp, C.c_int]),
    "pm2d_set_lasers": (C.c_int, [_vp, C.POINTER(Laser), C.c_int]),
    "pm2d_polarised_beam": (C.c_int, [C.POINTER(Laser), C.c_double, C.c_double, C.POINTER(Laser)]),
    "pm2d_get_fields": (C.c_int64, [_vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, _fp, C.c_size_t]),
    "pm2d_get_moments": (C.c_int64, [_vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, _fp, C.c_size_t]),
    "pm2d_set_fields": (C.c_int, [_vp, C.c_int, C.c_int, C.c_int, _fp]),
    "pm2d_get_particles": (C.c_int64, [_vp, C.c_int, C.c_int64, C.c_int64, _ip, _ip, _fp, _fp, _fp, _fp, _fp, _lp]),
    "pm2d_get_predictor": (C.c_int64, [_vp, C.c_int, C.c_int64, C.c_int64, _fp, _fp]),
    "pm2d_set_particles": (C.c_int, [_vp, C.c_int, C.c_int64, _ip, _ip, _fp, _fp, _fp, _fp, _fp, C.c_int]),
    "pm2d_set_background": (C.c_int, [_vp, C.c_int, _fp]),
    "pm2d_rebin": (C.c_int, [_vp, C.c_int, _ip, _lp]),
    "pm2d_diagnostics": (C.c_int, [_vp, C.POINTER(Diag)]),
    "pm2d_velocity_histogram": (C.c_int, [_vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int,
                                         C.POINTER(C.c_double)]),
    "pm2d_get_probe": (C.c_int64, [_vp, C.c_int, C.c_int, _fp, C.c_size_t, _lp]),
    "pm2d_probe_spectrum": (C.c_int64, [_vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "pm2d_mode_amplitudes": (C.c_int, [_vp, C.c_int, C.c_int, _ip, _ip, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "pm2d_mode_amplitudes_static": (C.c_int, [_vp, C.c_int, C.c_int, C.c_int, _ip, _ip, _vp, _vp]),
    "pm2d_particle_count": (C.c_int64, [_vp, C.c_int]),
    "pm2d_profile_enable": (C.c_int, [_vp, C.c_int]),
    "pm2d_profile_get": (C.c_int, [_vp, C.POINTER(C.c_double), _lp, _lp]),
    "pm2d_launch_count": (C.c_int64, [_vp]),
    "pm2d_stray_count": (C.c_int64, [_vp]),
    "pm2d_lane_subs": (C.c_int, [_vp, C.c_int]),
    "pm2d_free": (None, [_vp]),
    "pm2d_last_error": (C.c_char_p, []),
    "pm2d_version": (C.c_char_p, []),
    "pm2d_struct_size": (C.c_int, [C.c_int]),
}

_lib = None


def load_library():
    """dlopen libpm2d.so (built in-tree by build.py) and type every exported symbol."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -m paper_2404_14293_b200.build` (there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            f = getattr(L, name)            # AttributeError if the library does not export it
            f.restype = res
            f.argtypes = args
        # the ctypes mirrors must have the layout the library was compiled with (a struct grown on one side only would be
        # read past its end on the other)
        for which, st in enumerate((Grid, Species, Profile, Laser, Diag)):
            if L.pm2d_struct_size(which) != C.sizeof(st):
                raise RuntimeError(f"{st.__name__}: the binding has {C.sizeof(st)} bytes, {LIB_PATH} has {L.pm2d_struct_size(which)}: rebuild the library")
        _lib = L
    return _lib


class PM2DError(RuntimeError):
    pass


def _check(rc):
    if rc < 0:
        raise PM2DError(f"pm2d error {rc}: {load_library().pm2d_last_error().decode()}")
    return rc


def _np(a, dtype):
    return np.ascontiguousarray(np.asarray(a, dtype=dtype))


def _ptr(a, ctype):
    return None if a is None else a.ctypes.data_as(C.POINTER(ctype))


def polarised_beam(a0, theta, beta, **laser):
    """Laser-table entries of one beam of arbitrary polarisation (Fig. 1(a)): pm2d_polarised_beam does the
    decomposition; this wrapper only marshals the beam in and the up to three entries out."""
    proto = Laser(float(a0), float(laser.get("omega", 1.0)), float(laser.get("y0", 0.0)), float(laser.get("w0", 0.0)),
                  float(laser.get("t_rise", 0.0)), float(laser.get("alpha", 0.0)), 0, 0)
    out = (Laser * 3)()
    n = _check(load_library().pm2d_polarised_beam(C.byref(proto), float(theta), float(beta), out))
    return [dict(laser, a0=out[k].a0, comp=out[k].comp) for k in range(n)]


STATIC_MAX_ROWS, MAX_MODES = 16385, 16


def mode_amplitudes_static(n_dev, nx, ny, mx, my, out_dev, stream=0):
    """pm2d_mode_amplitudes_static: n_dev a CUDA float32 tensor of (nx + 1) * ny nodes, out_dev a CUDA float64 tensor of
    2 * len(mx) values (Re, Im interleaved), stream a raw cudaStream_t (0 = default stream).  Allocates nothing and does
    not synchronise; two calls that overlap on the GPU race on the library's static scratch array."""
    import torch
    if not (n_dev.is_cuda and n_dev.dtype == torch.float32 and n_dev.is_contiguous() and n_dev.numel() == (nx + 1) * ny):
        raise ValueError("n_dev: contiguous CUDA float32 tensor of (nx + 1) * ny elements")
    mx, my = np.ascontiguousarray(mx, np.int32), np.ascontiguousarray(my, np.int32)
    if mx.size != my.size:
        raise ValueError("mx and my differ in length")
    if not (out_dev.is_cuda and out_dev.dtype == torch.float64 and out_dev.is_contiguous() and out_dev.numel() >= 2 * mx.size):
        raise ValueError("out_dev: contiguous CUDA float64 tensor of at least 2 * len(mx) elements")
    _check(load_library().pm2d_mode_amplitudes_static(n_dev.data_ptr(), int(nx), int(ny), int(mx.size), mx.ctypes.data_as(_ip),
                                                      my.ctypes.data_as(_ip), out_dev.data_ptr(), int(stream)))


def make_structs(cfg: dict, eager_moments=1, track_ids=0, rebin_every=None, particle_order=0):
    """Translate a pm2d_inputs-style config dict into the C structs."""
    g = cfg["grid"]
    grid = Grid(g["nx"], g["ny"], g.get("ncomp", 1), g.get("rebin_every", 8) if rebin_every is None else rebin_every,
                int(eager_moments), int(track_ids), int(particle_order), int(g.get("subcycle", 1)),
                int(g.get("bc_y", 0)), int(g.get("probe_steps", 0)), g["dx"], g["dy"], g["dt"])
    sp = (Species * len(cfg["species"]))()
    for k, s in enumerate(cfg["species"]):
        sp[k] = Species(s["mass"], s["T_keV"], s["pressure_coeff"], s["DD"], s["sign"], s["shape"], s["mobile"], s["load"],
                        s.get("ppc_x", 0), s.get("ppc_y", 0), int(s.get("capacity", 0)))
    p = cfg["profile"]
    prof = Profile(p["kind"], p.get("taper_cells", 0), (C.c_double * 4)(*[float(v) for v in p["p"]]), int(p.get("taper_cells_y", 0)), 0,
                   (C.c_int32 * 4)(*[int(v) for v in (p.get("slab") or (0, 0, 0, 0))]))
    las = (Laser * max(len(cfg["lasers"]), 1))()
    for k, l in enumerate(cfg["lasers"]):
        las[k] = Laser(l["a0"], l["omega"], l["y0"], l["w0"], l["t_rise"], l.get("alpha", 0.0), l["comp"], 0)
    return grid, sp, prof, las


class PM2D:
    """One simulation context.  Method names mirror the C ABI (pm2d_step -> .step, ...)."""

    def __init__(self, cfg: dict, device="cuda:0", eager_moments=1, track_ids=0, rebin_every=None, stream=None, particle_order=0):
        import torch

        self.lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("pm2d needs a CUDA device (sm_100a); there is no CPU fallback")
        self.cfg = cfg
        self.device = torch.device(device)
        self.grid, self.species, self.profile, self.lasers = make_structs(cfg, eager_moments, track_ids, rebin_every, particle_order)
        self.nsp, self.nlaser = len(cfg["species"]), len(cfg["lasers"])
        self.nx, self.ny = self.grid.nx, self.grid.ny
        nbytes = self.lib.pm2d_query_workspace(C.byref(self.grid), self.species, self.nsp)
        if nbytes == 0:
            raise PM2DError("pm2d_query_workspace: " + self.lib.pm2d_last_error().decode())
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)     # owns the device memory
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.ctx = _vp()
            _check(self.lib.pm2d_init(C.byref(self.grid), self.species, self.nsp, C.byref(self.profile), self.lasers, self.nlaser,
                                      C.c_uint64(int(cfg.get("seed", 0))), _vp(self.workspace.data_ptr()), nbytes,
                                      _vp(self.stream.cuda_stream), C.byref(self.ctx)))
        self.workspace_bytes = nbytes

    def close(self):
        if getattr(self, "ctx", None):
            self.lib.pm2d_free(self.ctx)
            self.ctx = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- stepping ------------------------------------------------------------------------------
    def step(self, nsteps=1):
        _check(self.lib.pm2d_step(self.ctx, int(nsteps)))

    def step_async(self, nsteps=1):
        _check(self.lib.pm2d_step_async(self.ctx, int(nsteps)))

    def set_lasers(self, lasers):
        las = (Laser * max(len(lasers), 1))()
        for k, l in enumerate(lasers):
            las[k] = Laser(l["a0"], l["omega"], l["y0"], l["w0"], l["t_rise"], l.get("alpha", 0.0), l["comp"], 0)
        _check(self.lib.pm2d_set_lasers(self.ctx, las, len(lasers)))

    # -- grids ---------------------------------------------------------------------------------
    def _window(self, win):
        i0, i1, j0, j1 = win if win is not None else (0, self.nx + 1, 0, self.ny)
        return i0, i1, j0, j1, np.empty((i1 - i0, j1 - j0), np.float32)

    def get_fields(self, field, comp=0, level=0, window=None, out=None):
        i0, i1, j0, j1, buf = self._window(window)
        if out is not None:
            buf = out
        _check(self.lib.pm2d_get_fields(self.ctx, field, comp, level, i0, i1, j0, j1, _ptr(buf, C.c_float), buf.size))
        return buf

    def get_moments(self, species, moment, window=None):
        i0, i1, j0, j1, buf = self._window(window)
        _check(self.lib.pm2d_get_moments(self.ctx, species, moment, i0, i1, j0, j1, _ptr(buf, C.c_float), buf.size))
        return buf

    def set_fields(self, field, comp, level, arr):
        a = _np(arr, np.float32)
        assert a.size == (self.nx + 1) * self.ny
        _check(self.lib.pm2d_set_fields(self.ctx, field, comp, level, _ptr(a, C.c_float)))

    def set_background(self, species, arr):
        a = _np(arr, np.float32)
        assert a.size == (self.nx + 1) * self.ny
        _check(self.lib.pm2d_set_background(self.ctx, species, _ptr(a, C.c_float)))

    # -- particles -----------------------------------------------------------------------------
    def particle_count(self, species):
        return int(_check(self.lib.pm2d_particle_count(self.ctx, species)))

    def get_particles(self, species, first=0, count=None, with_id=False):
        n = self.particle_count(species) - first if count is None else count
        out = dict(ix=np.empty(n, np.int32), iy=np.empty(n, np.int32), fx=np.empty(n, np.float32), fy=np.empty(n, np.float32),
                   ux=np.empty(n, np.float32), uy=np.empty(n, np.float32), w=np.empty(n, np.float32))
        ids = np.empty(n, np.int64) if with_id else None
        got = _check(self.lib.pm2d_get_particles(self.ctx, species, first, n, _ptr(out["ix"], C.c_int32), _ptr(out["iy"], C.c_int32),
                                                 _ptr(out["fx"], C.c_float), _ptr(out["fy"], C.c_float), _ptr(out["ux"], C.c_float),
                                                 _ptr(out["uy"], C.c_float), _ptr(out["w"], C.c_float), _ptr(ids, C.c_int64)))
        assert got == n
        if with_id:
            out["id"] = ids
        return out

    def get_predictor(self, species, first=0, count=None):
        n = self.particle_count(species) - first if count is None else count
        uhx, uhy = np.empty(n, np.float32), np.empty(n, np.float32)
        got = _check(self.lib.pm2d_get_predictor(self.ctx, species, first, n, _ptr(uhx, C.c_float), _ptr(uhy, C.c_float)))
        assert got == n
        return uhx, uhy

    def set_particles(self, species, parts, refix_background=True):
        ix, iy = _np(parts["ix"], np.int32), _np(parts["iy"], np.int32)
        f = {k: _np(parts[k], np.float32) for k in ("fx", "fy", "ux", "uy", "w")}
        _check(self.lib.pm2d_set_particles(self.ctx, species, ix.size, _ptr(ix, C.c_int32), _ptr(iy, C.c_int32),
                                           _ptr(f["fx"], C.c_float), _ptr(f["fy"], C.c_float), _ptr(f["ux"], C.c_float),
                                           _ptr(f["uy"], C.c_float), _ptr(f["w"], C.c_float), int(refix_background)))

    def rebin(self, species, want_keys=True, want_perm=True):
        n = self.particle_count(species)
        keys = np.empty(n, np.int32) if want_keys else None
        perm = np.empty(n, np.int64) if want_perm else None
        _check(self.lib.pm2d_rebin(self.ctx, species, _ptr(keys, C.c_int32), _ptr(perm, C.c_int64)))
        return keys, perm

    # -- diagnostics ---------------------------------------------------------------------------
    def diagnostics(self):
        d = Diag()
        _check(self.lib.pm2d_diagnostics(self.ctx, C.byref(d)))
        return dict(step=d.step, time=d.time, W_es=d.W_es, W_int=d.W_int, W_em=d.W_em, W_total=d.W_total,
                    W_kin=list(d.W_kin)[: self.nsp], W_th=list(d.W_th)[: self.nsp], charge=list(d.charge)[: self.nsp],
                    count=list(d.count)[: self.nsp])

    def velocity_histogram(self, species, box, comp, umin, umax, nbins):
        """weighted histogram of u_x (comp 0) or u_y (comp 1) of the particles in the cells box = (i0, i1, j0, j1)
        [pm2d_velocity_histogram]"""
        h = np.zeros(int(nbins))
        i0, i1, j0, j1 = box
        _check(self.lib.pm2d_velocity_histogram(self.ctx, int(species), int(i0), int(i1), int(j0), int(j1), int(comp), float(umin),
                                                float(umax), int(nbins), h.ctypes.data_as(C.POINTER(C.c_double))))
        return h

    def get_probe(self, wall, comp=0):
        """(records[n, ny], first_step): the kept boundary records of a wall (0 left: a - a_inc, 1 right: a) in time
        order; needs grid["probe_steps"] > 0  [pm2d_get_probe]"""
        n = int(self.grid.probe_steps)
        out = np.empty((max(n, 1), self.ny), np.float32)
        first = C.c_int64(0)
        got = _check(self.lib.pm2d_get_probe(self.ctx, int(wall), int(comp), _ptr(out, C.c_float), out.size, C.byref(first)))
        return out[:got], int(first.value)

    def probe_spectrum(self, wall, omegas, comp=0, j0=0, j1=None):
        """power[k] = sum_j |dt_s sum_m h[m, j] exp(-2 pi i omega_k m dt_s)|^2 over the kept records  [pm2d_probe_spectrum]"""
        om = _np(omegas, np.float64)
        out = np.zeros(om.size)
        _check(self.lib.pm2d_probe_spectrum(self.ctx, int(wall), int(comp), int(j0), int(self.ny if j1 is None else j1), int(om.size),
                                            om.ctypes.data_as(C.POINTER(C.c_double)), out.ctypes.data_as(C.POINTER(C.c_double))))
        return out

    def mode_amplitudes(self, species, mx, my):
        """complex A(m_x, m_y) of the species' nodal density for the mode pairs (mx[k], my[k])  [pm2d_mode_amplitudes]"""
        mx, my = np.ascontiguousarray(mx, np.int32), np.ascontiguousarray(my, np.int32)
        re, im = np.zeros(mx.size), np.zeros(mx.size)
        _dp = C.POINTER(C.c_double)
        _check(self.lib.pm2d_mode_amplitudes(self.ctx, int(species), int(mx.size), mx.ctypes.data_as(_ip), my.ctypes.data_as(_ip),
                                             re.ctypes.data_as(_dp), im.ctypes.data_as(_dp)))
        return re + 1j * im

    def profile_enable(self, on=True):
        _check(self.lib.pm2d_profile_enable(self.ctx, int(on)))

    def profile_get(self):
        ms = (C.c_double * len(PHASES))()
        la = (C.c_int64 * len(PHASES))()
        st = C.c_int64(0)
        _check(self.lib.pm2d_profile_get(self.ctx, ms, la, C.byref(st)))
        return dict(ms=dict(zip(PHASES, ms)), launches=dict(zip(PHASES, la)), steps=st.value)

    def launch_count(self):
        return int(self.lib.pm2d_launch_count(self.ctx))

    def stray_count(self):
        return int(_check(self.lib.pm2d_stray_count(self.ctx)))

    def version(self):
        return self.lib.pm2d_version().decode()

    def lane_subs(self, s):
        return int(_check(self.lib.pm2d_lane_subs(self.ctx, int(s))))
