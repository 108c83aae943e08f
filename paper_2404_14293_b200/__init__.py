"""paper_2404_14293_b200 -- B200-native (sm_100a) PM2D particle-mesh cycle (arXiv 2404.14293).

The product is the C-ABI library ``libpm2d.so`` (include/pm2d.h, sources under ``csrc/``); this
package holds its build script and a thin ctypes binding.  It never imports ``oracle``.
"""
from .binding import (CIC, TSC, SINE, LOAD_NONE, LATTICE_COLD, RANDOM_MAXWELL, PROFILE_UNIFORM, PROFILE_LINEAR,
                      PROFILE_EXP_CAPPED, FIELD_A, FIELD_PHI, FIELD_ENODE, FIELD_FORCE, FIELD_FORCE_REF, MOMENT_N, MOMENT_PX, MOMENT_PY,
                      PHASES, TILE, BC_Y_PERIODIC, BC_Y_ABSORB, ORDER_AUTO, ORDER_CELL_MAJOR, ORDER_LAYERED, ORDER_RANDOM, ORDER_LANES, LAYERS, PM2D, PM2DError, polarised_beam, load_library, SYMBOLS, LIB_PATH,
                      mode_amplitudes_static, STATIC_MAX_ROWS)

__all__ = ["PM2D", "PM2DError", "polarised_beam", "mode_amplitudes_static", "load_library", "SYMBOLS", "LIB_PATH"]
