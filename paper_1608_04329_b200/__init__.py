"""B200-native Gibbs sweep for the Horseshoe Probit model (arXiv 1608.04329).

The product is the C-ABI library `libhsp.so` (include/hsp.h; CUDA kernels in csrc/).  This package
is the thin Python binding with the same names: it marshals arguments and nothing else.  There is
no CPU fallback: importing works anywhere, but every compute call needs the CUDA library and a GPU.
"""
from .binding import (HSP_F32, HSP_F64, HSP_STORE_Z, HSP_FREEZE_SCALES, HSP_FREEZE_Z, HSP_FREEZE_BETA,  # noqa: F401
                      HSP_NO_GRAPH, HSP_SERIAL, HSP_PAPER_DESIGN, HspError, HorseshoeProbit, lib, lib_path, declared_symbols,
                      dbg_philox, dbg_uniform, dbg_tnpos, dbg_norm_inv, dbg_cheng, set_option, reset_options, get_option, chol_schedule, xtz_noalloc,
                      noalloc_scratch_bytes)
