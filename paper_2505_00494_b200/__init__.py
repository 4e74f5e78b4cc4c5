"""paper_2505_00494_b200 -- B200-native (sm_100a) QR-CTMRG hot path.

The product is the C-ABI shared library `libqrctm.so` (include/qrctm.h, sources in
csrc/); `binding` is a thin ctypes layer with the same names.  Importing this
package does not load the library; the first call does, and fails loudly when
the library or a CUDA device is missing (there is no CPU fallback).
"""
from .binding import (QRCTM, QrctmError, chol_inv_f64, eigh_top_f64, gemm_f64, gemm_f64_noalloc, load_library, probe_fp64, qr_f64, shard_exchange, shard_range, tridiag_f64, version,  # noqa: F401
                      OPT_CHECK_EVERY, OPT_CORNER_MODE, OPT_GEMM_PATH, OPT_SYMMETRIZE, OPT_TIME_STAGES, OPT_QR_PATH, OPT_OVERLAP_CHECK, OPT_USE_GRAPH, OPT_ABSORB_MODE, OPT_K8_PATH, OPT_SMALL_PATH, STAGE_NAMES, STAGE_NAMES_RUN,
                      SYMBOLS, LIB_PATH)
