"""paper_2010_11540_b200: B200-native hot path of the 2D PIC space-charge tracker of arXiv 2010.11540.

The product is libsc_track.so (hand-written CUDA for sm_100a, C ABI in include/sc_track.h); this
package is its thin ctypes binding.  Build the library with `python -m paper_2010_11540_b200.build`.
"""
from .binding import (ERRORS, EXPORTS, LIB_PATH, SC_DEPOSIT_F64, SC_DEPOSIT_FIXED, SC_DRIFT, SC_GRID_EX, SC_GRID_EY,
                      SC_GRID_LAMBDA, SC_GRID_PHI, SC_GRID_RHO_F64, SC_GRID_RHO_I64, SC_LINMAP, SC_MULT, SC_BOUNDARY_OPEN, SC_BOUNDARY_PIPE, SC_INTERP_BILINEAR, SC_INTERP_BICUBIC, SC_FLAG_NO_PDL, SC_FLAG_FUSED_POISSON, SC_FLAG_NO_FIELD_WINDOW, SC_REPLAY_TURN, SC_REPLAY_PUSH, SC_REPLAY_POISSON, SC_REPLAY_EMPTY, SC_N_MOMENTS,
                      SC_QUAD, SC_RF, SC_SCNODE, ScError, Tracker, load_library)

__all__ = ["Tracker", "ScError", "load_library", "LIB_PATH", "EXPORTS", "ERRORS", "SC_N_MOMENTS", "SC_FLAG_NO_PDL", "SC_FLAG_FUSED_POISSON", "SC_FLAG_NO_FIELD_WINDOW", "SC_REPLAY_TURN", "SC_REPLAY_PUSH", "SC_REPLAY_POISSON", "SC_REPLAY_EMPTY", "SC_BOUNDARY_OPEN", "SC_BOUNDARY_PIPE", "SC_INTERP_BILINEAR", "SC_INTERP_BICUBIC",
           "SC_DRIFT", "SC_LINMAP", "SC_MULT", "SC_RF", "SC_SCNODE", "SC_QUAD", "SC_DEPOSIT_F64", "SC_DEPOSIT_FIXED",
           "SC_GRID_RHO_F64", "SC_GRID_RHO_I64", "SC_GRID_PHI", "SC_GRID_EX", "SC_GRID_EY", "SC_GRID_LAMBDA"]
