"""B200-native periodogram scan of FREDEC (Baluev 2013, arXiv:1309.0100).

The product is the C-ABI library libfredec_b200.so (include/fredec.h, sources under csrc/);
this package is its thin Python binding plus the seeded input generators (`inputs`).
"""
from ._binding import (  # noqa: F401
    FREDEC_D_MAX, FREDEC_ECUDA, FREDEC_EDATA, FREDEC_EINVAL, FREDEC_ELIMIT, FREDEC_ESINGULAR, FREDEC_OK,
    FREDEC_TOPK_MAX, FREDEC_TOPK_NOALLOC_K_MAX, fredec_topk_noalloc, fredec_topk_noalloc_scratch_bytes, FredecError, LIB_PATH,
    fredec_chi2_base, fredec_chi2_base_batched, fredec_bench_fp64, fredec_bench_fp64_name, fredec_last_launches,
    fredec_last_timing, fredec_scan, fredec_scan_batched, fredec_scan_topk, fredec_scan_topk_batched, fredec_set_stream, fredec_set_async, fredec_set_timing, fredec_last_status, fredec_shutdown,
    fredec_topk, fredec_topk_batched, fredec_version, lib,
    fredec_bandwidth, fredec_fap1, fredec_phase1, fredec_refine, fredec_refine_batched, fredec_subset_fits, fredec_trig_averages, fredec_zstat,
)
