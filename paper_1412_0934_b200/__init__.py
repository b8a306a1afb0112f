"""B200-native per-patch Godunov hydro/MHD update of arXiv 1412.0934.

The product is ``libamrgodunov.so`` (C-ABI in ``include/amr_godunov.h``, hand-written sm_100a CUDA
kernels in ``csrc/``).  This package is the thin Python binding: same names, argument marshalling
only.  PyTorch supplies device memory and the stream; there is no CPU fallback -- importing works
anywhere, but every compute call needs the built library and a CUDA device.
"""
from .binding import (  # noqa: F401
    AMR_F32, AMR_F64, AMR_BC_PERIODIC, AMR_BC_OUTFLOW, AMR_LIM_NONE, AMR_LIM_MINMOD, AMR_LIM_MC,
    AMR_RS_HLL, AMR_RS_HLLC, AMR_RS_HLLD, CNT_NAMES, AmrError, PatchBatch, LevelLink, Hierarchy, PatchBuilder, lib, library_path,
    EXPORTS, measure_fma_peak, conserved_totals_noalloc,
)
