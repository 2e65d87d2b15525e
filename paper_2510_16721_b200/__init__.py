"""B200-native hot path of the cell-filter nudged elastic band method (CFNEB, arXiv:2510.16721).

One CFNEB iteration over all images at once -- cell map, cell-list neighbours, batched force / energy /
virial, improved tangent, perpendicular projection + springs in the rotation-free generalized coordinates
(Eq. 17), climbing image, FIRE -- as hand-written fp64 CUDA for sm_100a behind the C ABI of
include/cfneb.h.  This package is the thin ctypes binding (argument marshalling only) plus the in-tree
build of libcfneb.so; see DESIGN.md.
"""
from .binding import (HISTORY_LEN, HistoryEntry, NOALLOC_MAX_IMAGES, band_dots_noalloc, CELL_B, CELL_D, CELL_FIXED, CFNEB, EXPORTS, KERNEL_CLASSES, LIB_PATH, POT_FS_MORSE,
                      POT_DNN, POT_LJ_SF, POT_NEP, POT_SW, CfnebError, FireState, Params, Status, default_params, fp64_peak_tflops, lib,
                      workspace_bytes)
from .workload import params_for

__all__ = ["CFNEB", "CfnebError", "Params", "Status", "FireState", "default_params", "workspace_bytes", "fp64_peak_tflops",
           "lib", "params_for", "band_dots_noalloc", "NOALLOC_MAX_IMAGES", "HistoryEntry", "HISTORY_LEN", "EXPORTS", "KERNEL_CLASSES", "LIB_PATH", "POT_LJ_SF", "POT_FS_MORSE", "POT_SW", "POT_DNN", "POT_NEP", "CELL_FIXED",
           "CELL_B", "CELL_D"]
