"""paper_1306_5076_b200 -- B200-native bank-conflict-free sorting (arXiv 1306.5076).

A thin Python binding over the C-ABI CUDA library `libbcf.so` (include/bcf.h): argument
marshalling only, every step of the path runs in the sm_100a kernels under csrc/.
PyTorch is used for device memory and streams.  There is no CPU fallback: if the library is
missing or the device is not a B200, calls raise.

    import paper_1306_5076_b200 as bcf
    bcf.sort_tiles(keys)                      # in place, 32x32 tiles        (bcf_sort_tiles)
    out = bcf.merge_runs(keys, run_len)       # sorted runs -> one sequence  (bcf_merge_runs)
    bcf.sort(keys, vals)                      # in place BCFMergesort        (bcf_sort)
"""
from . import binding  # noqa: F401
from .binding import (  # noqa: F401
    BcfError,
    KERNEL_CLASSES,
    kernel_info,
    launch_counts,
    layout_access,
    layout_word,
    lib,
    colored_prefix_sums,
    SCAN_BANK_PER_THREAD,
    SCAN_THREAD_MAJOR,
    find_buckets,
    merge_partition,
    merge_partition4,
    merge_pass_count,
    merge_pieces,
    debug_merge_round_isolated,
    debug_sort_tiles_isolated,
    sort_buckets,
    options,
    Options,
    KERNEL_IDS,
    kernel_name,
    last_cuda_error,
    profile_dropped,
    MERGE_IMPL_AUTO,
    MERGE_IMPL_GENERIC,
    MERGE_IMPL_BARRIER4,
    MERGE_IMPL_PARTITION_LAUNCH,
    LAUNCH_AUTO,
    LAUNCH_PLAIN,
    LAUNCH_PDL,
    merge_round_static,
    merge_round_static_max_shares,
    merge_round_static_shares,
    merge_runs,
    merge_runs_pagewise,
    num_shares,
    profile_enable,
    profile_read,
    sort,
    sort_host,
    sort_tiles,
    sort_tiles_mergesort,
    BASE_SHEARSORT,
    BASE_TILE_MERGESORT,
    BASE_LONG_TILES,
    BASE_AUTO,
    sort_long_tiles,
    version,
    workspace_bytes,
)
