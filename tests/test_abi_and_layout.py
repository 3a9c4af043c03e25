"""CPU-only checks of the boundary: libbcf.so loads and exports every symbol include/bcf.h
declares, the host-only entry points behave as documented, and a host-side bank model proves that
every shared-memory access pattern the kernels use is conflict-free (section 2.1)."""
import ctypes
import os
import re

import numpy as np
import pytest

import paper_1306_5076_b200 as bcf
from paper_1306_5076_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def declared_functions():
    text = open(os.path.join(ROOT, "include", "bcf.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(bcf_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = declared_functions()
    assert {"bcf_sort_tiles", "bcf_merge_runs", "bcf_sort", "bcf_merge_partition", "bcf_sort_host",
            "bcf_merge_runs_pagewise", "bcf_workspace_bytes"} <= set(names)
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_1306_5076_b200", "libbcf.so"))
    for n in names:
        assert hasattr(lib, n), f"{n} declared in include/bcf.h but not exported"


def test_host_only_entry_points():
    assert bcf.version().startswith("bcf")
    L = bcf.lib()
    assert L.bcf_status_string(0) == b"BCF_OK"
    assert L.bcf_status_string(3) == b"BCF_ERR_WORKSPACE_TOO_SMALL"
    # workspace: tiles need none; the sort needs a ping-pong copy + split points
    assert bcf.workspace_bytes(binding.OP_SORT_TILES, 1 << 20) == 0
    assert bcf.workspace_bytes(binding.OP_SORT, 1024) == 0
    n = 1 << 20
    ws = bcf.workspace_bytes(binding.OP_SORT, n)
    assert 4 * n < ws < 4 * n + 64 * 1024
    ws_kv = bcf.workspace_bytes(binding.OP_SORT, n, kt=binding.BCF_KEY_U64, vt=binding.BCF_VAL_U32)
    assert 12 * n < ws_kv < 12 * n + 64 * 1024
    assert bcf.workspace_bytes(binding.OP_SORT_HOST, n) >= ws + 4 * n
    assert bcf.workspace_bytes(binding.OP_MERGE_RUNS, n, n) == 0            # a single run
    assert bcf.workspace_bytes(binding.OP_MERGE_RUNS, n, n // 2) < 64 * 1024  # one round: splits only
    assert bcf.workspace_bytes(binding.OP_MERGE_RUNS, n, 1) > 4 * n + 4 * (n // 2)
    assert bcf.workspace_bytes(99, n) == 0


def test_share_slot_count():
    assert bcf.num_shares(8192, 1024) == 8
    assert bcf.num_shares(5000, 1024) == 6      # 3 pairs x 2 slots
    assert bcf.num_shares(3000, 700) == 6       # 3 pairs x ceil(1400/1024)
    assert bcf.num_shares(1024, 1) == 512


def test_no_gpu_means_loud_failure():
    torch = pytest.importorskip("torch")
    if torch.cuda.is_available():
        pytest.skip("this box has a GPU")
    with pytest.raises(ValueError):
        bcf.sort(torch.zeros(2048, dtype=torch.int32))        # host tensor: refused, no CPU path
    buf = np.zeros(4096 + 64, dtype=np.uint8)
    ptr = (buf.ctypes.data + 15) & ~15
    st = bcf.lib().bcf_sort(ptr, None, 1024, 0, 0, None, 0, None)
    assert st in (4, 5)                                       # UNSUPPORTED_DEVICE or CUDA error, never OK


# ---------------------------------------------------------------- host-side bank model


def banks_conflict_free(first_words, width):
    """Hardware rule: a warp access of `width` words per lane is served 32/width lanes at a time
    (128-bit: quarter-warps, 64-bit: half-warps); within each group all touched banks must differ
    unless the word is the same."""
    group = 32 // width
    for g in range(0, 32, group):
        seen = {}
        for lane in range(g, g + group):
            for i in range(width):
                w = first_words[lane] + i
                b = w % 32
                if b in seen and seen[b] != w:
                    return False
                seen[b] = w
    return True


def test_layout_is_a_bijection_on_the_tile():
    words = sorted(bcf.layout_word(r, c) for r in range(32) for c in range(32))
    assert words == list(range(1024))
    # a row stays inside its own 128-byte line
    for r in range(32):
        assert {bcf.layout_word(r, c) // 32 for c in range(32)} == {r}


STEPS = {0: 8, 1: 8, 2: 32, 3: 32, 4: 32, 5: 8, 6: 16, 7: 32, 8: 160, 9: 8, 10: 32, 11: 64, 12: 64}


@pytest.mark.parametrize("pattern", sorted(STEPS))
def test_every_access_pattern_is_conflict_free(pattern):
    for step in range(STEPS[pattern]):
        acc = [bcf.layout_access(pattern, step, lane) for lane in range(32)]
        widths = {w for _, w in acc}
        assert len(widths) == 1
        width = widths.pop()
        first = [f for f, _ in acc]
        assert all(f % width == 0 for f in first)            # vector accesses are naturally aligned
        assert banks_conflict_free(first, width), (pattern, step)


def test_access_patterns_touch_the_right_logical_elements():
    lw = bcf.layout_word
    for step in range(8):
        for lane in range(32):
            assert bcf.layout_access(0, step, lane) == (lw(lane, 4 * step), 4)      # row chunk
            assert bcf.layout_access(1, step, lane) == (lw(lane, 4 * step), 4)
            pos = 128 * step + 4 * lane                                            # coalesced 16-byte store
            assert bcf.layout_access(5, step, lane) == (lw(pos // 32, pos % 32), 4)
    for step in range(32):
        for lane in range(32):
            col = 31 - lane if step % 2 else lane                                   # odd rows mirrored
            assert bcf.layout_access(2, step, lane) == (lw(step, col), 1)
            assert bcf.layout_access(3, step, lane) == (lw(step, col), 1)
            assert bcf.layout_access(4, step, lane) == (lw(step, lane), 1)
            assert bcf.layout_access(7, step, lane) == (lw(step, lane), 1)
    for step in range(16):
        for lane in range(32):
            pos = 64 * step + 2 * lane
            assert bcf.layout_access(6, step, lane) == (lw(pos // 32, pos % 32), 2)
    # within a chunk consecutive columns are consecutive words
    for r in range(32):
        for q in range(8):
            assert [lw(r, 4 * q + i) for i in range(4)] == list(range(lw(r, 4 * q), lw(r, 4 * q) + 4))


def test_long_tile_and_stage_buffer_patterns_touch_the_right_elements():
    """The patterns added in r3 (bcf_long_tile.cuh's flip row load and fused column read of the partner tile, the
    merge pipeline's stage-buffer slot loads): right logical elements, and each covers its line exactly once."""
    lw = bcf.layout_word
    for lane in range(32):
        got = []
        for step in range(8):
            first, width = bcf.layout_access(9, step, lane)
            assert (first, width) == (lw(31 - lane, 4 * (7 - step)), 4)
            got += [4 * (7 - step) + i for i in range(4)]
        assert sorted(got) == list(range(32))                    # the whole partner row, chunks in reverse order
    for step in range(32):
        assert sorted(bcf.layout_access(10, step, lane)[0] for lane in range(32)) == \
            sorted(lw(31 - step, c) for c in range(32))          # one row of the partner, every column once
    for off in range(32):
        assert [bcf.layout_access(11, off, lane)[0] for lane in range(32)] == list(range(off, off + 32))
        assert [bcf.layout_access(11, 32 + off, lane)[0] for lane in range(32)] == list(range(1023 - off, 991 - off, -1))
        assert bcf.layout_access(12, off, 5) == (2 * (off + 5), 2)


def test_linear_layout_would_conflict():
    """Sanity of the bank model itself: thread-per-row on an unskewed tile is a 32-way conflict."""
    first = [32 * r + 5 for r in range(32)]
    assert not banks_conflict_free(first, 1)


# ---------------------------------------------------------------- the paper's own schemes (A5-A7)


def test_fig2_bank_view_golden():
    """PAPER.md Fig. 2: word A_i of a contiguous array sits in bank i mod b, column i div b."""
    rows = [list(map(int, l.split())) for l in open(os.path.join(GOLDEN, "fig2_bank_layout.txt"))
            if not l.startswith("#")]
    b = len(rows)
    assert b == 8
    for bank, row in enumerate(rows):
        for col, idx in enumerate(row):
            assert idx % b == bank and idx // b == col


def test_paper_alg2_addressing_bank_sets():
    """Reading A6/A7: with m[row][col] at bank `row`, every index formula of Alg. 2
    is conflict-free at w = 32 except the un-skew step L361, which puts two threads on each bank."""
    w = 32

    def worst(bank_of):
        worst_case = 1
        for j in range(w):
            banks = [bank_of(t, j) for t in range(w)]
            worst_case = max(worst_case, max(banks.count(x) for x in set(banks)))
        return worst_case

    assert worst(lambda t, j: (t + j) % w) == 1                 # L347, L350, L353, L355, L357, L359
    assert worst(lambda t, j: (t + w - j) % w) == 1             # L351 (ELSE restored, index w-1-j)
    assert worst(lambda t, j: (2 * t + j) % w) == 2             # L361: the 2-way conflict
    # and the addressing is a bijection: diagonal d, position k  <->  (bank (d+k) mod w, column k)
    cells = {((d + k) % w, k) for d in range(w) for k in range(w)}
    assert len(cells) == w * w


def test_paper_transpose_round_count():
    """Reading A5: rounds i = 1 .. w/2-1 of PAPER.md:L95 swap only w^2/2 - w of the w(w-1)/2
    off-diagonal pairs; the w/2 pairs at distance w/2 need one more half-round."""
    w = 32
    pairs = set()
    for i in range(1, w // 2):
        for t in range(w):
            a, b = t, (i + t) % w
            pairs.add((min(a, b), max(a, b)))
    assert len(pairs) == w * w // 2 - w == 480
    missing = {(a, b) for a in range(w) for b in range(a + 1, w)} - pairs
    assert len(missing) == w // 2 and all(b - a == w // 2 for a, b in missing)


def test_tile_mergesort_column_sweep_reads_P_then_reversed_Q():
    """Pattern 8: at level T the thread of column c reads, as register k, position 32 k + c of the
    sequence P || reverse(Q) of its block of 2^T rows (P, Q = the block's sorted halves, row-major).
    Checked against that definition written out on a tile whose word at (r, c) holds 32 r + c."""
    where = {bcf.layout_word(r, c): (r, c) for r in range(32) for c in range(32)}
    for T in range(1, 6):
        size, half = 1 << T, 1 << (T - 1)
        for k in range(32):
            base = k - k % size
            P = [(base + i, c) for i in range(half) for c in range(32)]
            Q = [(base + half + i, c) for i in range(half) for c in range(32)]
            seq = P + Q[::-1]
            for lane in range(32):
                w, width = bcf.layout_access(8, 32 * (T - 1) + k, lane)
                assert width == 1 and where[w] == seq[32 * (k - base) + lane]


def test_argument_errors_are_reported_before_any_device_work():
    """Status codes for bad arguments come back on a box without a GPU too (include/bcf.h, ERRORS)."""
    L = bcf.lib()
    INVALID, MISALIGNED, TOO_SMALL = 1, 2, 3
    buf = np.zeros(1 << 16, dtype=np.uint8)
    p = (buf.ctypes.data + 255) & ~255
    assert L.bcf_options_init(None) == INVALID
    assert L.bcf_sort_long_tiles(p, None, 1, 3, 0, 0, None) == INVALID                 # h must be 2, 4 or 8
    assert L.bcf_sort_long_tiles(p + 4, None, 1, 2, 0, 0, None) == MISALIGNED
    assert L.bcf_sort_tiles_mergesort(None, None, 1, 0, 0, None) == INVALID
    assert L.bcf_sort_tiles_mergesort(p, None, 0, 0, 0, None) == 0                      # nothing to do
    # FIND-BUCKETS: P >= 2, s * t >= P, workspace
    assert L.bcf_find_buckets_workspace_bytes(4096, 1024, 4, 1, 0, 0) == 0
    assert L.bcf_find_buckets_workspace_bytes(4096, 1024, 1, 8, 0, 0) == 0              # 4 samples, 8 buckets
    need = L.bcf_find_buckets_workspace_bytes(4096, 1024, 4, 8, 1, 0)
    assert need > 0
    assert L.bcf_find_buckets(p, 4096, 1024, 4, 1, 0, 0, p + 16384, p + 40000, p + 44000, p + 48000, need, None) == INVALID
    assert L.bcf_find_buckets(p, 4096, 1024, 4, 8, 0, 0, p + 16384, p + 40000, p + 44000, p + 48000, 16, None) == TOO_SMALL
    assert L.bcf_find_buckets(p, 4096, 1024, 4, 8, 0, 0, p + 1024, p + 40000, p + 44000, p + 48000, need, None) == INVALID  # in/out overlap
    # coloured prefix sums: 1..16 colours, known layout, no aliasing
    assert L.bcf_colored_prefix_sums_workspace_bytes(0) == 0 and L.bcf_colored_prefix_sums_workspace_bytes(1000) > 0
    ws = L.bcf_colored_prefix_sums_workspace_bytes(1000)
    assert L.bcf_colored_prefix_sums(p, p + 8192, 1000, 17, 0, p + 16384, p + 32768, ws, None) == INVALID
    assert L.bcf_colored_prefix_sums(p, p + 8192, 1000, 0, 0, p + 16384, p + 32768, ws, None) == INVALID
    assert L.bcf_colored_prefix_sums(p, p + 8192, 1000, 4, 2, p + 16384, p + 32768, ws, None) == INVALID
    assert L.bcf_colored_prefix_sums(p, p + 8192, 1000, 4, 0, p, p + 32768, ws, None) == INVALID          # out aliases values
    assert L.bcf_colored_prefix_sums(p, p + 8192, 1000, 4, 0, p + 16384, p + 32768, 0, None) == TOO_SMALL
    # pass structure of the merging phase (host only)
    one, two = ctypes.byref(bcf.options(rounds_per_pass=1)), ctypes.byref(bcf.options(rounds_per_pass=2))
    assert L.bcf_merge_pass_count(1 << 28, 1024, 0, 0, one) == 18 and L.bcf_merge_pass_count(1 << 28, 8192, 0, 0, one) == 15
    assert L.bcf_merge_pass_count(1 << 28, 1024, 0, 0, two) == 9
    assert L.bcf_merge_pass_count(1 << 27, 1024, 0, 0, two) == 9     # 17 rounds: one two-way pass + 8 four-run passes
    assert L.bcf_merge_pass_count(1 << 26, 1024, 1, 1, two) == 16    # (u64,u32): the four-run stage buffers do not fit
    # the two option sets do not interact: no process-wide state is left behind by either call
    assert L.bcf_merge_pass_count(1 << 28, 1024, 0, 0, one) == 18 and L.bcf_merge_pass_count(1 << 28, 1024, 0, 0, two) == 9
    # bcf_options validation (host side, before any device work)
    bad = bcf.options()
    bad.base_case = 9
    assert L.bcf_sort_ex(p, None, 4096, 0, 0, p + 32768, 1 << 15, None, ctypes.byref(bad)) == INVALID
    bad = bcf.options()
    bad.merge_impl = 4                                            # one past BCF_MERGE_IMPL_PARTITION_LAUNCH
    assert L.bcf_sort_ex(p, None, 4096, 0, 0, p + 32768, 1 << 15, None, ctypes.byref(bad)) == INVALID
    bad = bcf.options()
    bad.struct_size = 8
    assert L.bcf_merge_pass_count(1 << 20, 1024, 0, 0, ctypes.byref(bad)) == 0
    # BCFMergesort with buckets: P >= 2, t >= 1, workspace
    assert L.bcf_sort_buckets_workspace_bytes(1 << 20, 8, 1, 0, 0) == 0 and L.bcf_sort_buckets_workspace_bytes(1 << 20, 0, 8, 0, 0) == 0
    need = L.bcf_sort_buckets_workspace_bytes(1 << 14, 4, 4, 1, 0)
    assert need >= 2 * 4 * (1 << 14)
    assert L.bcf_sort_buckets(p, 1 << 14, 0, 4, 1, 0, None, p, need, None, None) == INVALID
    assert L.bcf_sort_buckets(p, 1 << 14, 0, 4, 4, 0, None, p + (1 << 20), 64, None, None) == TOO_SMALL
    assert L.bcf_sort_buckets(p, 0, 0, 4, 4, 0, None, None, 0, None, None) == 0
    assert L.bcf_merge_pieces_workspace_bytes(1 << 14, 4, 1, 0) > 0 and L.bcf_merge_pieces_workspace_bytes(0, 4, 4, 0) == 0
    assert L.bcf_merge_pieces(p, p, 100, p, 4, 4, 0, 0, p, 1 << 14, None) == INVALID            # in/out aliasing


@pytest.mark.parametrize("kt,P,t,pb,n", [(1, 4096, 1, 1, 4095 * 1024 - 5), (0, 2048, 1, 0, 2047 * 1024 - 5),
                                         (0, 2048, 1, 1, 2048 * 1024 - 3), (1, 128, 128, 1, 1 << 22), (0, 4096, 3, 1, 3000 * 1024)])
def test_sort_buckets_workspace_covers_the_distribution_when_t_is_raised(kt, P, t, pb, n):
    """bcf_sort_buckets raises t to ceil(P / s) where the s runs of phase 2 give fewer than P samples; its
    workspace must be sized with that same t (r2 advisor: with t = 1 and a large P the FIND-BUCKETS region was
    sized as 0 bytes and the call wrote ~34 MB past the caller's workspace).  Host arithmetic only: the region
    after [keys copy][piece offsets][pivots] must hold bcf_find_buckets_workspace_bytes for both base run lengths."""
    L = binding.lib()
    total = L.bcf_sort_buckets_workspace_bytes(n, t, P, pb, kt)
    assert total > 0
    up = lambda x: (x + 255) // 256 * 256      # noqa: E731
    kb = 8 if kt else 4
    nb = 2 * P - 1 if pb else P
    rest_off = up(n * kb) + up((nb * P + 1) * 4) + up(P * kb)
    for base in (1024, 8192):
        run = base
        while -(-n // run) > P:
            run *= 2
        s = -(-n // run)
        tt = t if s * t >= P else -(-P // s)
        need = L.bcf_find_buckets_workspace_bytes(n, run, tt, P, pb, kt)
        assert need > 0
        assert total - rest_off >= need, (base, s, tt, total - rest_off, need)
