"""pm2d_mode_amplitudes_static (include/pm2d.h): the entry point that allocates nothing -- its scratch is a file-scope
device array of libpm2d.so -- against the existing pm2d_mode_amplitudes, on two calls in a row.  Collected last (zz): the
suite runs with pytest -x."""
import ctypes as C

import numpy as np
import pytest

import pm2d_inputs as I


def _pkg():
    import paper_2404_14293_b200 as pkg
    from paper_2404_14293_b200 import build
    build.build()
    return pkg


def test_sizes_beyond_the_static_scratch_are_refused():
    """nx + 1 > PM2D_STATIC_MAX_ROWS and nmodes > PM2D_MAX_MODES: PM2D_EINVAL with a message, before any CUDA call."""
    P = _pkg()
    lib = P.load_library()
    m = (C.c_int32 * 17)()
    dummy = C.c_void_p(256)                                    # never dereferenced: the sizes are checked first
    assert lib.pm2d_mode_amplitudes_static(dummy, P.STATIC_MAX_ROWS, 8, 1, m, m, dummy, None) == -1
    assert b"PM2D_STATIC_MAX_ROWS" in lib.pm2d_last_error()
    assert lib.pm2d_mode_amplitudes_static(dummy, 64, 8, 17, m, m, dummy, None) == -1
    assert lib.pm2d_mode_amplitudes_static(None, 64, 8, 1, m, m, dummy, None) == -1


@pytest.mark.gpu
def test_static_scratch_entry_point_equals_the_ctx_path_twice():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    P = _pkg()
    cfg = I.config("c3", nx=72, ny=64)                          # ragged nx, walls included, two mobile species
    sim = P.PM2D(cfg, eager_moments=1, rebin_every=2)
    nx, ny = cfg["grid"]["nx"], cfg["grid"]["ny"]
    mx = [0, 1, 0, 3, -2, 7, 36, 71, 5, 1, 2, 3, 4, 5, 6, 9]
    my = [0, 0, 1, 2, 5, -3, 32, 63, 31, 1, 1, 1, 1, 1, 1, 9]
    out = torch.full((2 * len(mx),), float("nan"), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    first = None
    for call in range(2):                                       # second call: other species, later step, scratch holds call 1's sums
        sim.step(3)
        s = call
        ref = sim.mode_amplitudes(s, mx, my)                    # existing path: ctx scratch, atomics
        n_dev = torch.from_numpy(np.ascontiguousarray(sim.get_moments(s, P.MOMENT_N), np.float32)).cuda()
        before = torch.cuda.memory_allocated()
        P.mode_amplitudes_static(n_dev, nx, ny, mx, my, out, stream)
        assert torch.cuda.memory_allocated() == before
        torch.cuda.synchronize()
        got = out.cpu().numpy()
        got = got[0::2] + 1j * got[1::2]
        scale = np.abs(ref[0])                                  # the (0, 0) amplitude: total charge; tolerance of test_mode_amplitudes_parity
        assert scale > 0 and np.isfinite(got).all()
        assert np.abs(got - ref).max() < 1e-5 * scale, (call, np.abs(got - ref).max() / scale)
        assert np.abs(ref[1:]).max() > 1e-4 * scale
        if first is not None:
            assert np.abs(got - first).max() > 1e-4 * scale     # the two calls did not compute the same thing
        first = got
        # the same input again: fixed summation order, bit-identical
        P.mode_amplitudes_static(n_dev, nx, ny, mx, my, out, stream)
        torch.cuda.synchronize()
        again = out.cpu().numpy()
        assert np.array_equal(again[0::2] + 1j * again[1::2], got)
    # fewer modes than the scratch holds, on a non-default stream
    side = torch.cuda.Stream()
    out2 = torch.zeros(4, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    P.mode_amplitudes_static(n_dev, nx, ny, mx[3:5], my[3:5], out2, side.cuda_stream)
    side.synchronize()
    o = out2.cpu().numpy()
    assert np.array_equal(o[0::2] + 1j * o[1::2], first[3:5])
    sim.close()
