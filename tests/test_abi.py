"""The C-ABI library loads and exports every symbol include/pm2d.h declares (no GPU needed)."""
import os
import re

import paper_2404_14293_b200 as P
from paper_2404_14293_b200 import build as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    txt = open(os.path.join(ROOT, "include", "pm2d.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(pm2d_[a-z_0-9]+)\s*\(", txt)))


def test_library_builds_and_exports_every_declared_symbol():
    B.build()
    lib = P.load_library()
    declared = _declared_symbols()
    assert len(declared) >= 18
    for name in declared:
        assert hasattr(lib, name), name
        assert name in P.SYMBOLS, f"binding does not type {name}"
    assert sorted(P.SYMBOLS) == declared
    assert b"sm_100a" in lib.pm2d_version()


def test_argument_validation_needs_no_gpu():
    import ctypes as C
    import pm2d_inputs as I
    from paper_2404_14293_b200.binding import make_structs

    lib = P.load_library()
    cfg = I.config("c1", nx=64, ny=32)
    grid, sp, prof, las = make_structs(cfg)
    assert lib.pm2d_query_workspace(C.byref(grid), sp, len(cfg["species"])) > 0
    grid.ny = 48                                   # not a power of two
    assert lib.pm2d_query_workspace(C.byref(grid), sp, len(cfg["species"])) == 0
    assert b"power of two" in lib.pm2d_last_error()
    grid.ny = 32
    grid.dt = 0.06                                 # dt/dx > 1
    assert lib.pm2d_query_workspace(C.byref(grid), sp, len(cfg["species"])) == 0


def test_slab_extent_is_validated_before_any_device_work():
    """pm2d_profile.slab: 0 <= lo < hi <= nx resp. ny or all zero, never with the number-weighted loading; the check
    sits in front of every CUDA call, so it answers on a machine without a GPU."""
    import ctypes as C
    import pm2d_inputs as I
    from paper_2404_14293_b200.binding import make_structs

    lib = P.load_library()
    out = C.c_void_p()

    def init(cfg):
        grid, sp, prof, las = make_structs(cfg)
        return lib.pm2d_init(C.byref(grid), sp, len(cfg["species"]), C.byref(prof), las, len(cfg["lasers"]), 0, None, 0, None, C.byref(out))

    for bad in ([0, 65, 0, 32], [10, 10, 0, 32], [-1, 20, 0, 32], [4, 60, 8, 33], [4, 60, 20, 8]):
        cfg = I.config("c1", nx=64, ny=32)
        cfg["profile"]["slab"] = bad
        assert init(cfg) == -1 and b"profile slab" in lib.pm2d_last_error(), bad          # PM2D_EINVAL
    cfg = I.config("c5", nx=64, ny=32)
    cfg["profile"]["slab"] = [4, 60, 4, 28]
    assert init(cfg) == -1 and b"NUMBER_WEIGHTED" in lib.pm2d_last_error()
    cfg = I.config("c1", nx=64, ny=32)
    cfg["profile"]["slab"] = [4, 60, 4, 28]              # a valid slab gets past the check (and then fails for want of a workspace / GPU)
    assert init(cfg) != 0 and b"profile slab" not in lib.pm2d_last_error()


def test_struct_layouts_of_the_binding_match_the_library():
    """pm2d_struct_size: the ctypes mirrors of pm2d_grid / species / profile / laser / diag have the sizes the library was
    compiled with (load_library refuses a mismatch); the fields the header lists last sit at the end of the mirrors."""
    import ctypes as C
    from paper_2404_14293_b200 import binding as B
    lib = P.load_library()
    for which, st in enumerate((B.Grid, B.Species, B.Profile, B.Laser, B.Diag)):
        assert lib.pm2d_struct_size(which) == C.sizeof(st) > 0, st.__name__
    assert lib.pm2d_struct_size(5) == -1 and lib.pm2d_struct_size(-1) == -1
    assert B.Profile.slab.offset + 16 == C.sizeof(B.Profile) and B.Profile.p.offset == 8
    hdr = open(os.path.join(ROOT, "include", "pm2d.h")).read()
    body = "    " + hdr[hdr.index("int32_t kind;          /* PM2D_PROFILE_*"):hdr.index("} pm2d_profile;")]
    order = [m for m in re.findall(r"^\s+(?:int32_t|double)\s+(\w+)", body, flags=re.M)]
    assert order == [n for n, _ in B.Profile._fields_], order


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2404_14293_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "pm2d_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(import|from)\s+paper_2404_14293_b200", txt, flags=re.M), f
            assert not re.search(r"#include\s+\"[^\"]*(csrc|pm2d\.h|pm2d_internal)", txt), f


def test_polarised_beam_decomposition():
    """a_sz = a cos(theta), a_px = a sin(theta) cos(beta), a_py = a sin(theta) sin(beta); host logic only."""
    import math
    import pytest
    b = P.polarised_beam(0.02, math.radians(90.0), math.radians(0.0), omega=1.0, y0=0.0, w0=0.0, alpha=0.0, t_rise=1.0)
    assert [(l["comp"], round(l["a0"], 15)) for l in b if abs(l["a0"]) > 1e-15] == [(1, 0.02)]      # pure P, along x
    b = P.polarised_beam(0.02, 0.0, 1.0, omega=1.0, y0=0.0, w0=0.0, alpha=0.0, t_rise=1.0)
    assert [(l["comp"], l["a0"]) for l in b] == [(0, 0.02)]                                         # pure S
    b = P.polarised_beam(0.02, math.radians(30.0), math.radians(90.0), omega=2.0, y0=1.0, w0=3.0, alpha=0.1, t_rise=1.0)
    amp = {l["comp"]: l["a0"] for l in b}
    assert amp[0] == 0.02 * math.cos(math.radians(30.0)) and abs(amp[2] - 0.01) < 1e-15 and abs(amp.get(1, 0.0)) < 1e-15
    assert sum(l["a0"] ** 2 for l in b) == pytest.approx(0.02 ** 2, rel=1e-14)
    assert all(l["omega"] == 2.0 and l["y0"] == 1.0 and l["w0"] == 3.0 and l["alpha"] == 0.1 for l in b)
