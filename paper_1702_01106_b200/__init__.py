"""paper_1702_01106_b200 -- thin Python binding of the grim B200 hot-path library (include/grim.h).

Argument marshalling only: every step of the path runs in the CUDA kernels of csrc/.  PyTorch is used for
device memory and streams.  There is no CPU fallback: loading fails loudly if libgrim_b200.so is missing, and
every compute call fails with GrimError if no sm_100 device is usable.
"""
from .binding import (  # noqa: F401
    BC_NONE, BC_OUTFLOW, BC_PERIODIC, BC_REFLECT_POLAR, EMHD, IDEAL, KERR_MKS, LLF, MINKOWSKI, MINMOD, MP5,
    ST_CONVERGED, ST_KMAX, ST_LS_EXHAUSTED, ST_NONFINITE, ST_SINGULAR, ST_TERMINAL, TAU_CONST, TAU_R32,
    Grid, GridDesc, GrimError, KERNEL_CLASSES, STATIC_MAX_ZONES, StepStats, exported_symbols,
    invert_primitives_static, lib, lib_path,
)

__all__ = [n for n in dir() if not n.startswith("_")]
