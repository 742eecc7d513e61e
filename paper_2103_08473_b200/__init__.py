"""B200-native complex spinor-basis CCSD hot path (arXiv 2103.08473, Appendix 7.1).

Thin Python binding over the C ABI in include/ccsd.h; every step runs in the CUDA library.  PyTorch is used only
for device memory and streams.  There is no CPU fallback: without the built library or without a CUDA device the
compute entry points raise.
"""
from .binding import (CCSD, CCSDError, TENSOR_IDS, TERM_IDS, STEP_NAMES, contract, energy_static, gemm_plan, launch_count, lib_path,
                      load_library, measure_fp64_peak, real_flops_per_cmac, shard_ranges, sum_plane, transpose, zgemm_nt, zgemm_nt_strassen)

__all__ = ["CCSD", "CCSDError", "TENSOR_IDS", "TERM_IDS", "STEP_NAMES", "contract", "energy_static", "gemm_plan", "launch_count", "lib_path",
           "load_library", "measure_fp64_peak", "real_flops_per_cmac", "shard_ranges", "sum_plane", "transpose", "zgemm_nt", "zgemm_nt_strassen"]
