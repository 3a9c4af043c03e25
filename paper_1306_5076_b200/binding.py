"""ctypes binding of libbcf.so -- same names as the C ABI (include/bcf.h), marshalling only."""
import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libbcf.so")
_LIB = None

BCF_KEY_U32, BCF_KEY_U64 = 0, 1
BCF_VAL_NONE, BCF_VAL_U32 = 0, 1
OP_SORT_TILES, OP_MERGE_RUNS, OP_SORT, OP_SORT_HOST, OP_MERGE_PAGEWISE = range(5)
KERNEL_CLASSES = ("tile_sort", "partition", "merge", "merge_pagewise")
# bcf_kernel_id (include/bcf.h): every kernel the library can launch
KERNEL_IDS = ("tile_sort", "tile_mergesort", "long_tile_2", "long_tile_4", "long_tile_8", "partition", "merge",
              "partition_share_1", "partition_share_32", "merge_pipe", "partition4", "merge4_pipe", "merge_pagewise",
              "merge_pieces", "merge4_stream")
BASE_SHEARSORT, BASE_TILE_MERGESORT, BASE_LONG_TILES, BASE_AUTO = 0, 1, 2, 3
MERGE_IMPL_AUTO, MERGE_IMPL_GENERIC, MERGE_IMPL_BARRIER4, MERGE_IMPL_PARTITION_LAUNCH = 0, 1, 2, 3
LAUNCH_AUTO, LAUNCH_PLAIN, LAUNCH_PDL = 0, 1, 2


class Options(ctypes.Structure):
    """struct bcf_options (include/bcf.h): per-call algorithm selection; the library keeps no settings."""
    _fields_ = [("struct_size", ctypes.c_uint32), ("base_case", ctypes.c_int32), ("rounds_per_pass", ctypes.c_int32),
                ("merge_impl", ctypes.c_int32), ("partition_warp_search_max", ctypes.c_int32),
                ("launch_mode", ctypes.c_int32)]


def options(base_case=None, rounds_per_pass=None, merge_impl=None, partition_warp_search_max=None, launch_mode=None):
    """A bcf_options filled by bcf_options_init with the given fields overridden (None = the library default)."""
    o = Options()
    _check(lib().bcf_options_init(ctypes.byref(o)), "bcf_options_init")
    if base_case is not None:
        o.base_case = int(base_case)
    if rounds_per_pass is not None:
        o.rounds_per_pass = int(rounds_per_pass)
    if merge_impl is not None:
        o.merge_impl = int(merge_impl)
    if partition_warp_search_max is not None:
        o.partition_warp_search_max = int(partition_warp_search_max)
    if launch_mode is not None:
        o.launch_mode = int(launch_mode)
    return o


def _opt(opts):
    """None, an Options, or a dict of options() keywords -> pointer argument."""
    if opts is None:
        return None
    if isinstance(opts, dict):
        opts = options(**opts)
    return ctypes.byref(opts)
TILE = 1024
SHARE = 8192


class BcfError(RuntimeError):
    def __init__(self, status, name, where):
        super().__init__(f"{where}: {name} ({status})")
        self.status = status
        self.name = name


def lib():
    """Load libbcf.so (built in-tree by paper_1306_5076_b200.build).  Fails loudly if absent."""
    global _LIB
    if _LIB is not None:
        return _LIB
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} not found: build it with `python -m paper_1306_5076_b200.build` "
            "(there is no CPU fallback)")
    L = ctypes.CDLL(_LIB_PATH)
    vp, sz, ci, u64 = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int, ctypes.c_ulonglong
    L.bcf_status_string.restype = ctypes.c_char_p
    L.bcf_status_string.argtypes = [ci]
    L.bcf_version.restype = ctypes.c_char_p
    L.bcf_workspace_bytes.restype = sz
    L.bcf_workspace_bytes.argtypes = [ci, sz, sz, ci, ci]
    L.bcf_sort_tiles.argtypes = [vp, vp, sz, ci, ci, vp]
    L.bcf_sort_tiles_mergesort.argtypes = [vp, vp, sz, ci, ci, vp]
    L.bcf_options_init.argtypes = [ctypes.POINTER(Options)]
    L.bcf_last_cuda_error.restype = ci
    L.bcf_profile_dropped.restype = u64
    L.bcf_kernel_name.restype = ctypes.c_char_p
    L.bcf_kernel_name.argtypes = [ci]
    L.bcf_sort_long_tiles.argtypes = [vp, vp, sz, ci, ci, ci, vp]
    L.bcf_merge_partition.argtypes = [vp, vp, sz, sz, ci, ci, vp, sz, vp]
    L.bcf_merge_partition4.argtypes = [vp, vp, sz, sz, ci, ci, vp, sz, vp]
    L.bcf_merge_pass_count.argtypes = [sz, sz, ci, ci, vp]
    L.bcf_colored_prefix_sums_workspace_bytes.restype = sz
    L.bcf_colored_prefix_sums_workspace_bytes.argtypes = [sz]
    L.bcf_colored_prefix_sums.argtypes = [vp, vp, sz, ci, ci, vp, vp, sz, vp]
    L.bcf_find_buckets_workspace_bytes.restype = sz
    L.bcf_find_buckets_workspace_bytes.argtypes = [sz, sz, ci, ci, ci, ci]
    L.bcf_find_buckets.argtypes = [vp, sz, sz, ci, ci, ci, ci, vp, vp, vp, vp, sz, vp]
    L.bcf_merge_runs.argtypes = [vp, vp, vp, vp, sz, sz, ci, ci, vp, sz, vp]
    L.bcf_merge_runs_pagewise.argtypes = [vp, vp, vp, vp, sz, sz, ci, ci, vp, sz, vp]
    L.bcf_merge_runs_ex.argtypes = [vp, vp, vp, vp, sz, sz, ci, ci, vp, sz, vp, vp]
    L.bcf_merge_round_static_max_shares.restype = sz
    L.bcf_merge_round_static_max_shares.argtypes = []
    L.bcf_merge_round_static_shares.restype = sz
    L.bcf_merge_round_static_shares.argtypes = [sz, sz]
    L.bcf_merge_round_static.argtypes = [vp, vp, vp, vp, sz, sz, ci, ci, vp]
    L.bcf_sort.argtypes = [vp, vp, sz, ci, ci, vp, sz, vp]
    L.bcf_sort_ex.argtypes = [vp, vp, sz, ci, ci, vp, sz, vp, vp]
    L.bcf_sort_host.argtypes = [vp, vp, sz, ci, ci, vp, sz, vp]
    L.bcf_sort_host_ex.argtypes = [vp, vp, sz, ci, ci, vp, sz, vp, vp]
    L.bcf_sort_buckets_workspace_bytes.restype = sz
    L.bcf_sort_buckets_workspace_bytes.argtypes = [sz, ci, ci, ci, ci]
    L.bcf_sort_buckets.argtypes = [vp, sz, ci, ci, ci, ci, vp, vp, sz, vp, vp]
    L.bcf_merge_pieces_workspace_bytes.restype = sz
    L.bcf_merge_pieces_workspace_bytes.argtypes = [sz, sz, sz, ci]
    L.bcf_merge_pieces.argtypes = [vp, vp, sz, vp, sz, sz, ci, ci, vp, sz, vp]
    L.bcf_debug_merge_round_isolated.argtypes = [vp, vp, sz, sz, ci, vp, sz, vp]
    L.bcf_debug_sort_tiles_isolated.argtypes = [vp, sz, ci, vp]
    L.bcf_profile_enable.argtypes = [ci]
    L.bcf_profile_read.argtypes = [ctypes.POINTER(ctypes.c_float), ctypes.POINTER(u64)]
    L.bcf_launch_counts.argtypes = [ctypes.POINTER(u64)]
    L.bcf_launch_counts.restype = None
    L.bcf_kernel_info.argtypes = [ci, ci, ci] + [ctypes.POINTER(ci)] * 5
    L.bcf_layout_word.argtypes = [ci, ci]
    L.bcf_layout_access.argtypes = [ci, ci, ci, ctypes.POINTER(ci)]
    _LIB = L
    return L


def _check(status, where):
    if status != 0:
        raise BcfError(status, lib().bcf_status_string(status).decode(), where)


def version():
    return lib().bcf_version().decode()


def _torch():
    import torch
    return torch


def _types(keys, vals):
    torch = _torch()
    if keys.dtype == torch.uint32 or keys.dtype == torch.int32:
        kt = BCF_KEY_U32
    elif keys.dtype == torch.uint64 or keys.dtype == torch.int64:
        kt = BCF_KEY_U64
    else:
        raise TypeError(f"keys must be a 32- or 64-bit integer tensor (bit pattern = unsigned key), got {keys.dtype}")
    if vals is None:
        return kt, BCF_VAL_NONE
    if vals.dtype not in (torch.uint32, torch.int32):
        raise TypeError(f"vals must be a 32-bit integer tensor, got {vals.dtype}")
    if vals.numel() != keys.numel():
        raise ValueError("keys and vals must have the same number of elements")
    return kt, BCF_VAL_U32


def _dev(t, name):
    if t is None:
        return None
    if not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor (there is no CPU path)")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    return t.data_ptr()


def _stream(stream):
    torch = _torch()
    s = torch.cuda.current_stream() if stream is None else stream
    return s.cuda_stream


def workspace_bytes(op, n, run_len=0, key_dtype=None, has_vals=False, kt=None, vt=None):
    if kt is None:
        torch = _torch()
        kt = BCF_KEY_U64 if key_dtype in (torch.uint64, torch.int64, np.uint64) else BCF_KEY_U32
    if vt is None:
        vt = BCF_VAL_U32 if has_vals else BCF_VAL_NONE
    return int(lib().bcf_workspace_bytes(int(op), int(n), int(run_len), kt, vt))


def _workspace(op, n, run_len, kt, vt, device, workspace):
    torch = _torch()
    need = int(lib().bcf_workspace_bytes(int(op), int(n), int(run_len), kt, vt))
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=device)
    return workspace, workspace.numel() * workspace.element_size()


def num_shares(n, run_len):
    """Share slots of one merge round (include/bcf.h, bcf_merge_partition)."""
    pairs = -(-n // (2 * run_len))
    return pairs * (-(-2 * run_len // TILE))


def sort_tiles(keys, vals=None, stream=None):
    """bcf_sort_tiles: in place ShearSort of consecutive 32x32 tiles."""
    kt, vt = _types(keys, vals)
    n = keys.numel()
    if n % TILE:
        raise ValueError("sort_tiles needs a whole number of 1024-element tiles")
    _check(lib().bcf_sort_tiles(_dev(keys, "keys"), _dev(vals, "vals"), n // TILE, kt, vt, _stream(stream)),
           "bcf_sort_tiles")
    return keys if vals is None else (keys, vals)


def sort_tiles_mergesort(keys, vals=None, stream=None):
    """bcf_sort_tiles_mergesort: same result as sort_tiles, merger network instead of ShearSort phases."""
    kt, vt = _types(keys, vals)
    n = keys.numel()
    if n % TILE:
        raise ValueError("sort_tiles_mergesort needs a whole number of 1024-element tiles")
    _check(lib().bcf_sort_tiles_mergesort(_dev(keys, "keys"), _dev(vals, "vals"), n // TILE, kt, vt, _stream(stream)),
           "bcf_sort_tiles_mergesort")
    return keys if vals is None else (keys, vals)


def sort_long_tiles(keys, h, vals=None, stream=None):
    """bcf_sort_long_tiles: in place sort of consecutive long tiles of 1024 * h elements (h = 2, 4, 8)."""
    kt, vt = _types(keys, vals)
    n = keys.numel()
    if h not in (2, 4, 8) or n % (TILE * h):
        raise ValueError("sort_long_tiles needs h in (2, 4, 8) and a whole number of 1024*h-element long tiles")
    _check(lib().bcf_sort_long_tiles(_dev(keys, "keys"), _dev(vals, "vals"), n // (TILE * h), int(h), kt, vt,
                                     _stream(stream)), "bcf_sort_long_tiles")
    return keys if vals is None else (keys, vals)


def merge_partition(keys, run_len, vals=None, stream=None):
    """bcf_merge_partition: split points (uint32 tensor) of one merge round."""
    torch = _torch()
    kt, vt = _types(keys, vals)
    n = keys.numel()
    shares = num_shares(n, run_len) if n else 0
    splits = torch.empty(max(shares, 1), dtype=torch.int32, device=keys.device)
    _check(lib().bcf_merge_partition(_dev(keys, "keys"), _dev(vals, "vals"), n, int(run_len), kt, vt,
                                     splits.data_ptr(), shares, _stream(stream)), "bcf_merge_partition")
    return splits[:shares]


def merge_partition4(keys, run_len, vals=None, stream=None):
    """bcf_merge_partition4: (ceil(n / 8192) + 1, 4) int32 tensor, row s = the four-run split of boundary s."""
    torch = _torch()
    kt, vt = _types(keys, vals)
    n = keys.numel()
    bounds = -(-n // SHARE) + 1
    splits = torch.empty((bounds, 4), dtype=torch.int32, device=keys.device)
    _check(lib().bcf_merge_partition4(_dev(keys, "keys"), _dev(vals, "vals"), n, int(run_len), kt, vt,
                                      splits.data_ptr(), bounds, _stream(stream)), "bcf_merge_partition4")
    return splits


def merge_pass_count(n, run_len, key_dtype=None, has_vals=False, kt=None, vt=None, opts=None):
    """bcf_merge_pass_count: passes over global memory bcf_merge_runs takes from runs of run_len under opts."""
    if kt is None:
        kt = BCF_KEY_U64 if np.dtype(key_dtype).itemsize == 8 else BCF_KEY_U32
        vt = BCF_VAL_U32 if has_vals else BCF_VAL_NONE
    return int(lib().bcf_merge_pass_count(int(n), int(run_len), kt, vt, _opt(opts)))


def find_buckets(keys, run_len, t, P, pivot_buckets=False, stream=None):
    """bcf_find_buckets: returns (keys regrouped by bucket, pivots, piece_offsets[(nb*s + 1)])."""
    torch = _torch()
    kt, vt = _types(keys, None)
    n = keys.numel()
    s = -(-n // int(run_len))
    nb = 2 * P - 1 if pivot_buckets else P
    need = int(lib().bcf_find_buckets_workspace_bytes(n, int(run_len), int(t), int(P), int(bool(pivot_buckets)), kt))
    if need == 0:
        raise ValueError("find_buckets: invalid n / run_len / t / P")
    ws = torch.empty(need, dtype=torch.uint8, device=keys.device)
    out = torch.empty_like(keys)
    pivots = torch.empty(P - 1, dtype=keys.dtype, device=keys.device)
    offsets = torch.empty(nb * s + 1, dtype=torch.int32, device=keys.device)
    _check(lib().bcf_find_buckets(_dev(keys, "keys"), n, int(run_len), int(t), int(P), int(bool(pivot_buckets)), kt,
                                  out.data_ptr(), pivots.data_ptr(), offsets.data_ptr(), ws.data_ptr(), need,
                                  _stream(stream)), "bcf_find_buckets")
    return out, pivots, offsets


SCAN_BANK_PER_THREAD, SCAN_THREAD_MAJOR = 0, 1


def colored_prefix_sums(values, colors, num_colors, layout=SCAN_BANK_PER_THREAD, out=None, workspace=None, stream=None):
    """bcf_colored_prefix_sums: values int32/uint32 tensor, colors uint8 tensor (< num_colors) -> out."""
    torch = _torch()
    if values.dtype not in (torch.int32, torch.uint32) or colors.dtype != torch.uint8:
        raise TypeError("values must be a 32-bit integer tensor and colors a uint8 tensor")
    n = values.numel()
    if colors.numel() != n:
        raise ValueError("values and colors must have the same number of elements")
    if out is None:
        out = torch.empty_like(values)
    need = int(lib().bcf_colored_prefix_sums_workspace_bytes(n))
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=values.device)
    _check(lib().bcf_colored_prefix_sums(_dev(values, "values"), _dev(colors, "colors"), n, int(num_colors), int(layout),
                                         _dev(out, "out"), workspace.data_ptr(), workspace.numel(), _stream(stream)),
           "bcf_colored_prefix_sums")
    return out


def _merge(fn, name, op, keys, run_len, vals, out_keys, out_vals, workspace, stream, opts=False):
    torch = _torch()
    kt, vt = _types(keys, vals)
    n = keys.numel()
    if out_keys is None:
        out_keys = torch.empty_like(keys)
    if vals is not None and out_vals is None:
        out_vals = torch.empty_like(vals)
    ws, ws_bytes = _workspace(op, n, run_len, kt, vt, keys.device, workspace)
    args = (_dev(keys, "keys"), _dev(vals, "vals"), _dev(out_keys, "out_keys"), _dev(out_vals, "out_vals"),
            n, int(run_len), kt, vt, ws.data_ptr(), ws_bytes, _stream(stream))
    _check(fn(*args) if opts is False else fn(*args, _opt(opts)), name)
    return out_keys if vals is None else (out_keys, out_vals)


def merge_runs(keys, run_len, vals=None, out_keys=None, out_vals=None, workspace=None, stream=None, opts=None):
    """bcf_merge_runs(_ex): merge sorted runs of run_len into one sorted sequence (out of place)."""
    return _merge(lib().bcf_merge_runs_ex, "bcf_merge_runs_ex", OP_MERGE_RUNS, keys, run_len, vals, out_keys, out_vals,
                  workspace, stream, opts)


def merge_runs_pagewise(keys, run_len, vals=None, out_keys=None, out_vals=None, workspace=None, stream=None):
    """bcf_merge_runs_pagewise: the paper's streaming Alg. 6, one warp per pair of runs."""
    return _merge(lib().bcf_merge_runs_pagewise, "bcf_merge_runs_pagewise", OP_MERGE_PAGEWISE, keys, run_len, vals,
                  out_keys, out_vals, workspace, stream)


def merge_round_static_max_shares():
    """bcf_merge_round_static_max_shares: size of the library's built-in split-point array (entries)."""
    return int(lib().bcf_merge_round_static_max_shares())


def merge_round_static_shares(n, run_len):
    """bcf_merge_round_static_shares: split points one round of (n, run_len) needs; 0 for invalid sizes."""
    return int(lib().bcf_merge_round_static_shares(int(n), int(run_len)))


def merge_round_static(keys, run_len, out_keys, vals=None, out_vals=None, stream=None):
    """bcf_merge_round_static: one merge round (runs 2p, 2p+1 -> a run of 2 run_len) for callers that cannot
    allocate device memory where they merge.  The library brings its own split-point scratch (a fixed 256 KiB
    array per GPU), so this wrapper allocates nothing either: the caller passes every tensor, outputs included.
    Rounds needing more than merge_round_static_max_shares() split points raise BcfError(BCF_ERR_TOO_LARGE).
    Calls on one GPU share that scratch: keep them on one stream.  The first call per device does a one-off
    set-up; make it before any stream capture."""
    kt, vt = _types(keys, vals)
    _check(lib().bcf_merge_round_static(_dev(keys, "keys"), _dev(vals, "vals"), _dev(out_keys, "out_keys"),
                                        _dev(out_vals, "out_vals"), keys.numel(), int(run_len), kt, vt, _stream(stream)),
           "bcf_merge_round_static")
    return out_keys if vals is None else (out_keys, out_vals)


def sort(keys, vals=None, workspace=None, stream=None, opts=None):
    """bcf_sort(_ex): in place BCFMergesort of device tensors.  opts: None, options(...) or a dict of its keywords."""
    kt, vt = _types(keys, vals)
    n = keys.numel()
    ws, ws_bytes = _workspace(OP_SORT, n, 0, kt, vt, keys.device, workspace)
    _check(lib().bcf_sort_ex(_dev(keys, "keys"), _dev(vals, "vals"), n, kt, vt, ws.data_ptr(), ws_bytes,
                             _stream(stream), _opt(opts)), "bcf_sort_ex")
    return keys if vals is None else (keys, vals)


def sort_buckets(keys, P, t=None, pivot_buckets=False, workspace=None, stream=None, opts=None, return_bucket_starts=False):
    """bcf_sort_buckets: BCFMergesort with the paper's bucket distribution (BCFMergesortPB with pivot_buckets),
    keys only, in place.  With return_bucket_starts also the nb + 1 bucket starts (int32 tensor; only meaningful
    when the distribution ran, i.e. more than one run was left after the first merge phase)."""
    torch = _torch()
    kt, _ = _types(keys, None)
    n = keys.numel()
    t = P if t is None else t
    need = int(lib().bcf_sort_buckets_workspace_bytes(n, int(t), int(P), int(bool(pivot_buckets)), kt))
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=keys.device)
    nb = 2 * P - 1 if pivot_buckets else P
    starts = torch.full((nb + 1,), -1, dtype=torch.int32, device=keys.device) if return_bucket_starts else None
    _check(lib().bcf_sort_buckets(_dev(keys, "keys"), n, kt, int(t), int(P), int(bool(pivot_buckets)),
                                  None if starts is None else starts.data_ptr(), workspace.data_ptr(), workspace.numel(),
                                  _stream(stream), _opt(opts)), "bcf_sort_buckets")
    return (keys, starts) if return_bucket_starts else keys


def merge_pieces(keys, piece_offsets, groups, s, copy_odd_groups=False, out_keys=None, workspace=None, stream=None):
    """bcf_merge_pieces: the final merge phase alone on the layout bcf_find_buckets writes."""
    torch = _torch()
    kt, _ = _types(keys, None)
    n = keys.numel()
    if out_keys is None:
        out_keys = torch.empty_like(keys)
    need = int(lib().bcf_merge_pieces_workspace_bytes(n, int(groups), int(s), kt))
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=keys.device)
    _check(lib().bcf_merge_pieces(_dev(keys, "keys"), _dev(out_keys, "out_keys"), n, _dev(piece_offsets, "piece_offsets"),
                                  int(groups), int(s), int(bool(copy_odd_groups)), kt, workspace.data_ptr(),
                                  workspace.numel(), _stream(stream)), "bcf_merge_pieces")
    return out_keys


def sort_host(keys, vals=None, scratch=None, device="cuda", stream=None, opts=None):
    """bcf_sort_host: in place sort of HOST tensors (ideally pinned); H2D + sort + D2H + sync."""
    torch = _torch()
    kt, vt = _types(keys, vals)
    if keys.is_cuda or (vals is not None and vals.is_cuda):
        raise ValueError("sort_host takes host tensors")
    n = keys.numel()
    need = int(lib().bcf_workspace_bytes(OP_SORT_HOST, n, 0, kt, vt))
    if scratch is None:
        scratch = torch.empty(max(need, 16), dtype=torch.uint8, device=device)
    _check(lib().bcf_sort_host_ex(keys.data_ptr(), None if vals is None else vals.data_ptr(), n, kt, vt,
                                  scratch.data_ptr(), scratch.numel(), _stream(stream), _opt(opts)), "bcf_sort_host_ex")
    return keys if vals is None else (keys, vals)


def debug_merge_round_isolated(keys, run_len, exclusive=True, out_keys=None, stream=None):
    """bcf_debug_merge_round_isolated: one merge round of uint32 runs with the phase-separated kernel (experiment)."""
    torch = _torch()
    n = keys.numel()
    if out_keys is None:
        out_keys = torch.empty_like(keys)
    ws = torch.empty((n // SHARE + 1) * 4 + 16, dtype=torch.uint8, device=keys.device)
    _check(lib().bcf_debug_merge_round_isolated(_dev(keys, "keys"), _dev(out_keys, "out_keys"), n, int(run_len),
                                                int(bool(exclusive)), ws.data_ptr(), ws.numel(), _stream(stream)),
           "bcf_debug_merge_round_isolated")
    return out_keys


def debug_sort_tiles_isolated(keys, exclusive=True, stream=None):
    """bcf_debug_sort_tiles_isolated: tile mergesort of uint32 tiles with the phase-separated kernel (experiment)."""
    n = keys.numel()
    if n % TILE:
        raise ValueError("whole tiles only")
    _check(lib().bcf_debug_sort_tiles_isolated(_dev(keys, "keys"), n // TILE, int(bool(exclusive)), _stream(stream)),
           "bcf_debug_sort_tiles_isolated")
    return keys


def profile_enable(on=True):
    _check(lib().bcf_profile_enable(1 if on else 0), "bcf_profile_enable")


def profile_read():
    """{class: (milliseconds, launches)} of the launches timed since the last read."""
    ms = (ctypes.c_float * len(KERNEL_CLASSES))()
    cnt = (ctypes.c_ulonglong * len(KERNEL_CLASSES))()
    _check(lib().bcf_profile_read(ms, cnt), "bcf_profile_read")
    return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(KERNEL_CLASSES)}


def launch_counts():
    cnt = (ctypes.c_ulonglong * len(KERNEL_CLASSES))()
    lib().bcf_launch_counts(cnt)
    return {k: int(cnt[i]) for i, k in enumerate(KERNEL_CLASSES)}


def profile_dropped():
    """Launches the profiler could not time because its event pool was full (bcf_profile_dropped)."""
    return int(lib().bcf_profile_dropped())


def last_cuda_error():
    return int(lib().bcf_last_cuda_error())


def kernel_name(kernel_id):
    cid = kernel_id if isinstance(kernel_id, int) else KERNEL_IDS.index(kernel_id)
    name = lib().bcf_kernel_name(cid)
    return None if name is None else name.decode()


def kernel_info(kernel_id, kt=BCF_KEY_U32, vt=BCF_VAL_NONE):
    """bcf_kernel_info of a kernel named in KERNEL_IDS (or its integer id)."""
    vals = [ctypes.c_int() for _ in range(5)]
    cid = kernel_id if isinstance(kernel_id, int) else KERNEL_IDS.index(kernel_id)
    _check(lib().bcf_kernel_info(cid, kt, vt, *[ctypes.byref(v) for v in vals]),
           "bcf_kernel_info")
    names = ("regs_per_thread", "smem_bytes_per_cta", "threads_per_cta", "ctas_per_sm", "local_bytes_per_thread")
    return dict(zip(names, (v.value for v in vals)))


def layout_word(row, col):
    return int(lib().bcf_layout_word(int(row), int(col)))


def layout_access(pattern, step, lane):
    """(first_word, words) a lane touches in one step of an access pattern (host-only)."""
    first = ctypes.c_int()
    nwords = lib().bcf_layout_access(int(pattern), int(step), int(lane), ctypes.byref(first))
    return first.value, int(nwords)
