"""B200-native coarse-grid multi-RHS operator and block CG (arXiv:2409.03904 hot path).

The product is the C-ABI library (include/coarse_mrhs.h, csrc/); this package is its ctypes binding.
"""
from .binding import (C64, C128, BlockCGResult, CoarseError, CoarseOperator, block_gram_noalloc, block_project, block_promote,  # noqa: F401
                      fill_block, fill_synthetic, launch_count, lib, library_path, measure_peaks, small_cholesky, small_hpd_inverse)
