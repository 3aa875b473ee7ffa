"""paper_2202_02840_b200 -- B200-native CRKSPH short-range gas interaction pipeline (CRK-HACC, arxiv 2202.02840).

The product is the C-ABI CUDA library ``libcrk.so`` (include/crk.h); this package is its thin Python binding
(argument marshalling only -- every step of the path runs in the library's kernels).  PyTorch is used for device
memory and streams.  There is no CPU fallback: importing ``binding`` without a built library raises.
"""
from .binding import (  # noqa: F401
    Crk,
    CrkError,
    crk_create,
    crk_destroy,
    crk_build_cells,
    crk_volumes,
    crk_rk_coefficients,
    crk_hydro_derivs,
    crk_step_derivs,
    crk_step_derivs_host,
    crk_measure_fp32_peak,
    crk_sfc_order_noalloc,
    NOALLOC_MAX_N,
    library_path,
    EXPORTED_SYMBOLS,
)
