"""paper_2502_17963_b200 — B200-native (sm_100a) closed-shell CCSD(T) triples energy.

The product is the C-ABI library `lib/libbqc_t.so` (sources in `csrc/`, interface in
`include/bqc_t.h`); this package is its build script and a ctypes binding with the same
function names.  PyTorch only owns device memory and streams.
"""
from .binding import (BQC_T_FLAG_NO_T1, BQC_T_FLAG_PROFILE, BQC_T_FLAG_ABC_DRIVEN, BQC_T_FLAG_SHARD_BLOCKS, BqcError, LIB_PATH, bqc_dgemm_nt, bqc_error_detail,
                      bqc_error_string, bqc_fp64_peak_tflops, bqc_last_error, bqc_sum_fixed_noalloc, bqc_sum_fixed_noalloc_max, bqc_release_cached, bqc_sum_in_order, bqc_t_plan, bqc_t_debug_slabs, bqc_debug_tiling,
                      bqc_t_debug_wv, bqc_t_energy, bqc_t_energy_ex, bqc_t_energy_host, bqc_t_flops, bqc_t_last_profile,
                      bqc_t_num_triplets, bqc_t_opts, bqc_t_plan_occ_block, bqc_t_triplet_index,
                      bqc_t_triplet_owner, bqc_t_triplet_owner_ex, bqc_t_workspace_bytes, bqc_version, lib, make_opts,
                      bqc_mp2_energy, bqc_mp2_energy_ex, bqc_mp2_energy_host, bqc_mp2_flops, bqc_mp2_last_profile,
                      bqc_mp2_opts, bqc_mp2_plan_occ_block, bqc_mp2_workspace_bytes, make_mp2_opts)

from .distributed import bqc_t_energy_sharded, combine_partials

__all__ = [n for n in dir() if n.startswith("bqc_") or n in ("BqcError", "LIB_PATH", "lib", "make_opts", "make_mp2_opts",
                                                               "BQC_T_FLAG_NO_T1", "BQC_T_FLAG_PROFILE",
                                                               "BQC_T_FLAG_ABC_DRIVEN", "BQC_T_FLAG_SHARD_BLOCKS", "combine_partials")]
