"""paper_1705_02028_b200 -- B200-native residual-distribution hydrodynamics sweep (arXiv:1705.02028).

Thin Python binding of the C-ABI in `include/mrd.h` (same names, argument marshalling only): every
step of the path runs in the CUDA kernels of `csrc/`.  PyTorch is used for device memory and
streams only.  There is no CPU fallback: without the built library or without a CUDA device the
calls raise.
"""
from .binding import (  # noqa: F401
    MRD_OK, MRD_EINVAL, MRD_ENOMEM, MRD_ECUDA, MRD_ENONPHYSICAL,
    SCHEME_N, SCHEME_LDA, SCHEME_B, SCHEME_BMAX, SCHEME_BMIN, SCHEME_BX, FP64, FP32,
    MrdError, Params, Layout, Partition, Mesh, lib, measure_peaks, exported_symbols, version,
)
