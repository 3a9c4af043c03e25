"""Pins for the CPU oracle (oracle/): what the paper and the mathematics fix, none of it the oracle
re-typed.  SURVEY.md section 8c lists them; each test names the reading (A1..A15) it pins.

 * 0-1 principle, exhaustively
 * exhaustive permutations / small alphabets against the closed form "sorted order"
 * the dirty-row halving invariant and the snake order of classic ShearSort
 * textbook library sorts (numpy) on every config shape
 * the trace of a stable two-finger merge, written out in Python, for the co-rank
 * the paper's pass count (Lemma 2)
"""
import itertools
import math
import os

import numpy as np
import pytest

import oracle
from paper_1306_5076_b200 import workloads

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def all_01_matrices(w):
    m = w * w
    idx = np.arange(1 << m, dtype=np.uint64)
    bits = ((idx[:, None] >> np.arange(m, dtype=np.uint64)[None, :]) & np.uint64(1)).astype(np.uint32)
    return bits  # shape (2^m, m), one row-major tile per row


def expected_01(tiles):
    """Closed form of a sorted 0/1 tile: (#zeros) zeros, then ones."""
    m = tiles.shape[1]
    ones = tiles.sum(axis=1)
    return (np.arange(m)[None, :] >= (m - ones)[:, None]).astype(np.uint32)


# ---------------------------------------------------------------- ShearSort (Alg. 1), A1-A4


@pytest.mark.parametrize("w", [1, 2, 3, 4])
def test_shearsort_sorts_every_01_matrix(w):
    tiles = all_01_matrices(w)
    out = oracle.shearsort_tiles(tiles.reshape(-1), w=w).reshape(tiles.shape)
    assert np.array_equal(out, expected_01(tiles))


def test_shearsort_one_phase_fewer_fails():
    """A2: ceil(log2 w) phases are necessary: with one fewer, w = 4 fails (mutation pin)."""
    tiles = all_01_matrices(4)
    out = oracle.shearsort_tiles(tiles.reshape(-1), w=4, phases=1).reshape(tiles.shape)
    bad = int((out != expected_01(tiles)).any(axis=1).sum())
    assert bad > 0
    assert bad == 17696  # an independent check found the same count


@pytest.mark.parametrize("w", [2, 3, 4])
def test_shearsort_classic_snake_order(w):
    """A4: with an alternating final row pass the tile is in snake order (Sen et al.)."""
    tiles = all_01_matrices(w)
    out = oracle.shearsort_tiles(tiles.reshape(-1), w=w, final_snake=True).reshape(-1, w, w)
    snake = out.copy()
    snake[:, 1::2, :] = snake[:, 1::2, ::-1]
    assert np.array_equal(snake.reshape(tiles.shape), expected_01(tiles))


@pytest.mark.parametrize("w", [8, 16, 32])
def test_shearsort_dirty_rows_halve(w):
    """0-1 argument behind L109: after k phases at most ceil(w / 2^k) rows are dirty."""
    rng = np.random.default_rng(1234 + w)
    num = 64
    dens = rng.random((num, 1, 1))
    tiles = (rng.random((num, w, w)) < dens).astype(np.uint32)
    # structured worst-ish cases: staircase and checkerboard
    tiles[0] = (np.add.outer(np.arange(w), np.arange(w)) % 2).astype(np.uint32)
    tiles[1] = (np.arange(w)[:, None] > np.arange(w)[None, :]).astype(np.uint32)
    for k in range(0, int(math.log2(w)) + 1):
        out = oracle.shearsort_tiles(tiles.reshape(-1), w=w, phases=k).reshape(num, w, w)
        rowsum = out.sum(axis=2)
        dirty = ((rowsum != 0) & (rowsum != w)).sum(axis=1)
        assert dirty.max() <= math.ceil(w / 2 ** k)
    final = oracle.shearsort_tiles(tiles.reshape(-1), w=w).reshape(num, -1)
    assert np.array_equal(final, expected_01(tiles.reshape(num, -1)))


@pytest.mark.parametrize("w", [2, 3, 5, 8, 32])
def test_shearsort_random_vs_library_sort(w):
    rng = np.random.default_rng(99 + w)
    x = rng.integers(0, 1 << 32, size=(37, w * w), dtype=np.uint64).astype(np.uint32)
    x[3] = 7  # all equal
    x[4] = np.arange(w * w, dtype=np.uint32)[::-1]
    x[5, : w * w // 2] = 0xFFFFFFFF  # the padding value is a legal key (A10)
    out = oracle.shearsort_tiles(x.reshape(-1), w=w).reshape(x.shape)
    assert np.array_equal(out, np.sort(x, axis=1))


def test_shearsort_key_value_lexicographic():
    """A11: order is (key, value) lexicographic; with value = index it equals a stable sort."""
    k, v = workloads.cfg2_tiles_u32_u32(num_tiles=5)
    ko, vo = oracle.shearsort_tiles(k, v)
    for t in range(5):
        s = slice(t * 1024, (t + 1) * 1024)
        order = np.argsort(k[s], kind="stable")
        assert np.array_equal(ko[s], k[s][order])
        assert np.array_equal(vo[s], v[s][order])
    # scrambled values: plain lexicographic order
    rng = np.random.default_rng(5)
    v2 = rng.permutation(v.size).astype(np.uint32)
    ko, vo = oracle.shearsort_tiles(k[:2048], v2[:2048])
    for t in range(2):
        s = slice(t * 1024, (t + 1) * 1024)
        order = np.lexsort((v2[s], k[s]))
        assert np.array_equal(ko[s], k[s][order]) and np.array_equal(vo[s], v2[s][order])


def test_shearsort_u64_keys():
    k, v = workloads.cfg5a_sort_u64_u32(n=3 * 1024)
    ko, vo = oracle.shearsort_tiles(k, v)
    for t in range(3):
        s = slice(t * 1024, (t + 1) * 1024)
        order = np.lexsort((v[s], k[s]))
        assert np.array_equal(ko[s], k[s][order]) and np.array_equal(vo[s], v[s][order])


# ---------------------------------------------------------------- merge (L125), co-rank (A12)


def python_merge_trace(a, b):
    """A stable two-finger merge written out in Python; returns (output, i after d outputs)."""
    i = j = 0
    out, trace = [], [0]
    while i < len(a) or j < len(b):
        if j >= len(b) or (i < len(a) and a[i] <= b[j]):
            out.append(a[i]); i += 1
        else:
            out.append(b[j]); j += 1
        trace.append(i)
    return out, trace


def test_merge_two_and_corank_match_stable_merge_trace():
    rng = np.random.default_rng(7)
    for case in range(300):
        na, nb = int(rng.integers(0, 40)), int(rng.integers(0, 40))
        hi = int(rng.choice([2, 5, 1000]))
        a = np.sort(rng.integers(0, hi, size=na)).astype(np.uint32)
        b = np.sort(rng.integers(0, hi, size=nb)).astype(np.uint32)
        out, trace = python_merge_trace(a.tolist(), b.tolist())
        assert oracle.merge_two(a, b).tolist() == out
        for d in range(na + nb + 1):
            i = oracle.corank(a, b, d)
            assert i == trace[d]
            j = d - i
            assert 0 <= i <= na and 0 <= j <= nb
            if i > 0 and j < nb:
                assert a[i - 1] <= b[j]
            if j > 0 and i < na:
                assert b[j - 1] < a[i]


def test_corank_ties_take_from_A_first():
    a = np.array([5, 5], dtype=np.uint32)
    b = np.array([5, 5], dtype=np.uint32)
    assert [oracle.corank(a, b, d) for d in range(5)] == [0, 1, 2, 2, 2]
    # with values the tie is broken by value
    assert oracle.corank(a, b, 2, va=np.array([1, 3], np.uint32), vb=np.array([0, 2], np.uint32)) == 1


def test_merge_two_key_value_u64():
    rng = np.random.default_rng(11)
    ka = rng.integers(0, 4, size=50, dtype=np.uint64) << np.uint64(40)
    kb = rng.integers(0, 4, size=70, dtype=np.uint64) << np.uint64(40)
    va = rng.integers(0, 1 << 32, size=50, dtype=np.uint64).astype(np.uint32)
    vb = rng.integers(0, 1 << 32, size=70, dtype=np.uint64).astype(np.uint32)
    oa = np.lexsort((va, ka)); ka, va = ka[oa], va[oa]
    ob = np.lexsort((vb, kb)); kb, vb = kb[ob], vb[ob]
    ko, vo = oracle.merge_two(ka, kb, va, vb)
    k = np.concatenate([ka, kb]); v = np.concatenate([va, vb])
    o = np.lexsort((v, k))
    assert np.array_equal(ko, k[o]) and np.array_equal(vo, v[o])


# ---------------------------------------------------------------- full sort / merge rounds (L103)


def test_sort_full_all_permutations_n_le_8():
    """Two (or fewer) 2x2 tiles + merge rounds on every permutation of n <= 8 keys."""
    for n in range(0, 9):
        want = np.arange(n, dtype=np.uint32)
        for p in itertools.permutations(range(n)):
            x = np.array(p, dtype=np.uint32)
            assert np.array_equal(oracle.sort_full(x, w=2), want)


def test_sort_full_all_ternary_words_of_length_8():
    for word in itertools.product(range(3), repeat=8):
        x = np.array(word, dtype=np.uint32)
        assert oracle.sort_full(x, w=2).tolist() == sorted(word)


def test_merge_runs_all_sorted_pairs_of_permutations_n8():
    """merge_runs on every permutation of 8 keys whose runs of length r were pre-sorted."""
    for r in (1, 2, 3, 4, 5):
        for p in itertools.islice(itertools.permutations(range(8)), 0, None, 7):
            x = workloads.sorted_runs(np.array(p, dtype=np.uint32), r)
            assert np.array_equal(oracle.merge_runs(x, r), np.arange(8, dtype=np.uint32))


@pytest.mark.parametrize("n", [0, 1, 2, 1023, 1024, 1025, 5000, 3 * 1024 + 17])
def test_sort_full_ragged_sizes_and_padding_value(n):
    """A10: partial tiles are padded with all-ones in scratch only; 0xFFFFFFFF is a legal key."""
    rng = np.random.default_rng(n)
    x = rng.integers(0, 1 << 32, size=n, dtype=np.uint64).astype(np.uint32)
    if n > 4:
        x[:: max(1, n // 5)] = 0xFFFFFFFF
    out, rounds = oracle.sort_full(x, return_rounds=True)
    assert np.array_equal(out, np.sort(x))
    tiles = max(1, math.ceil(n / 1024))
    assert rounds == math.ceil(math.log2(tiles))  # Lemma 2: 1 + ceil(log2(N/M)) scans


def test_sort_full_config_shapes_vs_library_sort():
    x = workloads.cfg3_sort_u32(n=1 << 14)
    assert np.array_equal(oracle.sort_full(x), np.sort(x))
    for dist in workloads.CFG4_VARIANTS:
        x = workloads.cfg4_sort_u32(dist, n=(1 << 13) + 77)
        out = oracle.sort_full(x)
        assert np.array_equal(out, np.sort(x)), dist
        assert np.all(out[:-1] <= out[1:])
    k, v = workloads.cfg5a_sort_u64_u32(n=(1 << 13) + 5)
    ko, vo = oracle.sort_full(k, v)
    o = np.lexsort((v, k))
    assert np.array_equal(ko, k[o]) and np.array_equal(vo, v[o])
    o2 = np.argsort(k, kind="stable")  # value = index  =>  stable sort by key
    assert np.array_equal(vo, v[o2])


@pytest.mark.parametrize("k", [2, 64, 1024])
def test_merge_runs_config_5b_shape(k):
    keys, run_len = workloads.cfg5b_merge_runs_u32(k, n=1 << 15)
    out, rounds = oracle.merge_runs(keys, run_len, return_rounds=True)
    assert rounds == int(math.log2(k))
    assert np.array_equal(out, np.sort(keys))


def test_merge_runs_ragged_runs():
    rng = np.random.default_rng(3)
    for n, r in [(10, 3), (1000, 7), (4097, 1024), (5000, 1), (777, 1000)]:
        x = rng.integers(0, 50, size=n).astype(np.uint32)
        xs = workloads.sorted_runs(x, r)
        assert np.array_equal(oracle.merge_runs(xs, r), np.sort(x))


# ---------------------------------------------------------------- SHEARSORT-MERGE (A8), Alg. 6 (A9)


def test_a8_contiguous_placement_counterexample():
    """One ShearSort round on contiguously placed half-pages does not merge (golden fixture)."""
    rows = {}
    with open(os.path.join(GOLDEN, "a8_counterexample.txt")) as f:
        for line in f:
            if line.startswith("#"):
                continue
            name, *vals = line.split()
            rows[name] = np.array(vals, dtype=np.uint32)
    page = np.concatenate([rows["A"], rows["B"]])
    out = oracle.shearsort_tiles(page, w=4, phases=1)
    assert np.array_equal(out, rows["AFTER"])
    assert not np.array_equal(out, np.sort(page))
    # the reading adopted (second page reversed, {column sort; row sort}) does merge it
    assert np.array_equal(oracle.shearsort_merge(page, na=8, w=4), np.sort(page))


@pytest.mark.parametrize("w", [2, 4, 8])
def test_shearsort_merge_every_sorted_01_pair_every_split(w):
    """0-1 principle for merging networks: all sorted-0/1 (A, B) with |A| + |B| = w^2."""
    m = w * w
    for na in range(m + 1):
        nb = m - na
        for za in range(na + 1):
            for zb in range(nb + 1):
                page = np.concatenate([np.arange(na) >= za, np.arange(nb) >= zb]).astype(np.uint32)
                out = oracle.shearsort_merge(page, na=na, w=w)
                assert out.sum() == page.sum() and np.all(out[:-1] <= out[1:]), (na, za, zb)


def test_shearsort_merge_random_w32():
    rng = np.random.default_rng(8)
    for _ in range(60):
        na = int(rng.integers(0, 1025))
        x = rng.integers(0, int(rng.choice([3, 1 << 32])), size=1024, dtype=np.uint64).astype(np.uint32)
        page = np.concatenate([np.sort(x[:na]), np.sort(x[na:])])
        assert np.array_equal(oracle.shearsort_merge(page, na=na), np.sort(x))


@pytest.mark.parametrize("w", [2, 4, 8, 32])
def test_binary_merge_pagewise_equals_sorted_union(w):
    rng = np.random.default_rng(40 + w)
    m = w * w
    sizes = [(0, 0), (0, 5), (5, 0), (1, 1), (m // 2, m // 2), (m, m), (3 * m, 3 * m),
             (m // 2 - 1, 2 * m + 3), (5 * m + 1, 7), (4 * m, m // 2)]
    sizes += [tuple(int(s) for s in rng.integers(0, 6 * m, size=2)) for _ in range(60)]
    for na, nb in sizes:
        hi = int(rng.choice([2, 7, 1 << 32]))
        a = np.sort(rng.integers(0, hi, size=na, dtype=np.uint64).astype(np.uint32))
        b = np.sort(rng.integers(0, hi, size=nb, dtype=np.uint64).astype(np.uint32))
        if na and rng.random() < 0.3:
            a[-1] = 0xFFFFFFFF  # a real key equal to the padding value
        out = oracle.binary_merge_pagewise(a, b, w=w)
        assert np.array_equal(out, np.sort(np.concatenate([a, b]))), (w, na, nb)


def test_binary_merge_pagewise_key_value():
    rng = np.random.default_rng(77)
    k = rng.integers(0, 9, size=3000, dtype=np.uint64)
    v = np.arange(3000, dtype=np.uint32)
    o = np.lexsort((v[:1300], k[:1300])); ka, va = k[:1300][o], v[:1300][o]
    o = np.lexsort((v[1300:], k[1300:])); kb, vb = k[1300:][o], v[1300:][o]
    ko, vo = oracle.binary_merge_pagewise(ka, kb, va, vb)
    o = np.lexsort((v, k))
    assert np.array_equal(ko, k[o]) and np.array_equal(vo, v[o])


def _kway_merge_trace(runs, d):
    """Brute force: repeatedly take the smallest head, lowest run index on ties; counts after d steps."""
    pos = [0] * len(runs)
    for _ in range(d):
        best = None
        for r, run in enumerate(runs):
            if pos[r] < len(run) and (best is None or run[pos[r]] < runs[best][pos[best]]):
                best = r
        pos[best] += 1
    return pos


def test_corank_multi_equals_kway_merge_trace_and_two_way_corank():
    rng = np.random.default_rng(77)
    for trial in range(300):
        k = int(rng.integers(1, 5))
        hi = int(rng.choice([2, 3, 50, 1 << 32]))
        runs = [np.sort(rng.integers(0, hi, size=int(rng.integers(0, 12)), dtype=np.uint64).astype(np.uint32))
                for _ in range(k)]
        total = sum(r.size for r in runs)
        for d in range(total + 1):
            got = oracle.corank_multi(runs, d)
            assert got == _kway_merge_trace([list(map(int, r)) for r in runs], d)
            if k == 2:
                assert got[0] == oracle.corank(runs[0], runs[1], d)
    # (key, value) order: equal keys are split by value before run index
    ka = [np.array([5, 5], np.uint32), np.array([5, 5], np.uint32)]
    va = [np.array([2, 9], np.uint32), np.array([1, 3], np.uint32)]
    assert [oracle.corank_multi(ka, d, va) for d in range(5)] == [[0, 0], [0, 1], [1, 1], [1, 2], [2, 2]]


def _bucket_ranges(Q, s, nb):
    return [(int(Q[b * s]), int(Q[(b + 1) * s])) for b in range(nb)]


@pytest.mark.parametrize("pb", [False, True])
def test_find_buckets_is_an_ordered_partition_and_meets_lemma_1(pb):
    """Pins for oracle.find_buckets (section 3.2, Alg. 7): O is a permutation of the input,
    every piece keeps its run's order, buckets are in ascending value order (so sorting each bucket gives
    the sorted input), bucket contents match their definition by the pivots, and -- all keys distinct --
    no bucket exceeds Lemma 1's bound s*ceil(N/(s t)) + ceil(s t / P)*ceil(N/(s t)) (L139-141)."""
    rng = np.random.default_rng(5 + pb)
    for trial in range(40):
        s = int(rng.integers(2, 9)); run_len = int(rng.integers(8, 200)); t = int(rng.integers(1, 9))
        P = int(rng.integers(2, min(s * t, 12) + 1))
        n = s * run_len - int(rng.integers(0, run_len // 2))
        distinct = trial % 2 == 0
        if distinct:
            keys = rng.permutation(1 << 16)[:n].astype(np.uint32)
        else:
            keys = rng.integers(0, 6, size=n).astype(np.uint32)
        keys = workloads.sorted_runs(keys, run_len)
        O, F, Q = oracle.find_buckets(keys, run_len, t, P, pivot_buckets=pb)
        s_runs = -(-n // run_len)
        nb = 2 * P - 1 if pb else P
        assert np.array_equal(np.sort(O), np.sort(keys)) and Q[-1] == n and np.all(np.diff(Q) >= 0)
        assert np.all(F[:-1] <= F[1:])
        rngs = _bucket_ranges(Q, s_runs, nb)
        for b, (lo, hi) in enumerate(rngs):
            x = O[lo:hi]
            if x.size == 0:
                continue
            if not pb:
                if b > 0: assert x.min() > F[b - 1]
                if b < P - 1: assert x.max() <= F[b]
            elif b % 2 == 1:                                  # pivot bucket j = (b - 1) / 2: all equal to it
                assert np.all(x == F[(b - 1) // 2])
            else:
                j = b // 2
                if j > 0: assert x.min() > F[j - 1]
                if j < P - 1: assert x.max() < F[j]
            for r in range(s_runs):                           # pieces stay sorted
                piece = O[Q[b * s_runs + r]:Q[b * s_runs + r + 1]]
                assert np.all(piece[:-1] <= piece[1:])
        sorted_by_bucket = np.concatenate([np.sort(O[lo:hi]) for lo, hi in rngs])
        assert np.array_equal(sorted_by_bucket, np.sort(keys))
        if distinct and not pb and n == s * run_len:
            per = -(-n // (s * t))
            bound = s * per + (-(-(s * t) // P)) * per
            assert max(hi - lo for lo, hi in rngs) <= bound


def test_find_buckets_pivot_buckets_finish_zero_one_data():
    """on 0-1 data BCFMergesortPB "has nothing more to do after rearranging the data"."""
    rng = np.random.default_rng(9)
    keys = workloads.sorted_runs(rng.integers(0, 2, size=16 * 256).astype(np.uint32), 256)
    O, F, Q = oracle.find_buckets(keys, 256, 8, 8, pivot_buckets=True)
    assert np.array_equal(O, np.sort(keys))
    s, nb = 16, 15
    sizes = [int(Q[(b + 1) * s] - Q[b * s]) for b in range(nb)]
    assert sum(sizes[1::2]) == keys.size and sum(sizes[0::2]) == 0     # every key sits in a pivot bucket


def test_colored_prefix_sums_pins():
    """oracle.colored_prefix_sums (App. A): one colour = the textbook inclusive scan (numpy cumsum);
    d colours = the scan of each colour's subsequence, put back in place; the last element of every colour
    carries that colour's total; wrap-around modulo 2^32."""
    rng = np.random.default_rng(21)
    v = rng.integers(0, 1 << 32, size=5000, dtype=np.uint64).astype(np.uint32)
    one = oracle.colored_prefix_sums(v, np.zeros(v.size, np.uint8), 1)
    assert np.array_equal(one, np.cumsum(v.astype(np.uint64)).astype(np.uint32))      # mod 2^32 by truncation
    for d in (2, 3, 16):
        c = rng.integers(0, d, size=v.size).astype(np.uint8)
        out = oracle.colored_prefix_sums(v, c, d)
        for k in range(d):
            m = c == k
            assert np.array_equal(out[m], np.cumsum(v[m].astype(np.uint64)).astype(np.uint32))
            if m.any():
                assert int(out[np.flatnonzero(m)[-1]]) == int(v[m].astype(np.uint64).sum() & 0xFFFFFFFF)
    assert oracle.colored_prefix_sums(np.array([1, 2, 3, 4], np.uint32), np.array([0, 1, 0, 1], np.uint8), 2).tolist() == [1, 2, 4, 6]
    assert oracle.colored_prefix_sums(np.array([0xFFFFFFFF, 2], np.uint32), np.array([0, 0], np.uint8), 1).tolist() == [0xFFFFFFFF, 1]


# ---------------------------------------------------------------- Alg. 7 golden (hand-worked) and mutation pins


def _load_alg7_golden():
    """tests/golden/alg7_worked_example.txt -> list of dicts (every number in it was worked by hand from
    PAPER.md L133-135, Alg. 7 L503-520 and L155; see the file header)."""
    cases, cur = [], None
    with open(os.path.join(os.path.dirname(__file__), "golden", "alg7_worked_example.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            key, *rest = line.split()
            if key == "CASE":
                cur = {"name": rest[0], "RANK_LE": []}
            elif key == "END":
                cases.append(cur)
                cur = None
            elif key == "RANK_LE":
                cur["RANK_LE"].append([int(x) for x in rest])
            elif key in ("RUN_LEN", "T", "P", "PIVOT_BUCKETS"):
                cur[key] = int(rest[0])
            else:
                cur[key] = [int(x) for x in rest]
    assert len(cases) == 4
    return cases


def _alg7_matches_golden(c, dtype=np.uint32):
    O, F, Q, steps = oracle.find_buckets(np.array(c["I"], dtype=dtype), c["RUN_LEN"], c["T"], c["P"],
                                         pivot_buckets=bool(c["PIVOT_BUCKETS"]), return_steps=True)
    return (steps["S_unsorted"].tolist() == c["S_UNSORTED"] and steps["S_sorted"].tolist() == c["S_SORTED"]
            and F.tolist() == c["F"] and steps["rank_le"].tolist() == c["RANK_LE"]
            and O.tolist() == c["O"] and Q.tolist() == c["Q"])


@pytest.mark.parametrize("dtype", [np.uint32, np.uint64])
def test_find_buckets_reproduces_the_hand_worked_alg7_examples(dtype):
    """oracle.find_buckets step by step against tests/golden/alg7_worked_example.txt: samples (L503),
    sorted samples (L505), pivots (L506, L135), ranks (L507-510), regrouped output and offsets (L512-520),
    with a ragged last run, a repeated pivot, and pivot buckets (L155)."""
    for c in _load_alg7_golden():
        assert _alg7_matches_golden(c, dtype), c["name"]


@pytest.mark.parametrize("mutant", ["pivot_j_instead_of_j_plus_1", "pivot_minus_1", "sample_last_of_each_stride"])
def test_alg7_golden_rejects_plausible_misreadings(monkeypatch, mutant):
    """Mutation pins: each plausible misreading of Alg. 7's two index formulas (pivot j at S[j s t / P], at
    S[(j+1) s t / P - 1], sample i at floor((i+1) len / t) - 1) must make the golden comparison fail -- the
    Lemma 1 bound and the partition properties alone do not see them."""
    if mutant == "pivot_j_instead_of_j_plus_1":
        monkeypatch.setattr(oracle, "alg7_pivot_index", lambda j, s, t, P: (j * s * t) // P)
    elif mutant == "pivot_minus_1":
        monkeypatch.setattr(oracle, "alg7_pivot_index", lambda j, s, t, P: ((j + 1) * s * t) // P - 1)
    else:
        monkeypatch.setattr(oracle, "alg7_sample_index", lambda i, length, t: ((i + 1) * length) // t - 1)
    results = [_alg7_matches_golden(c) for c in _load_alg7_golden()]
    assert not all(results), (mutant, results)
    assert not results[0], "the distinct-key example alone must catch the mutant"


# ---------------------------------------------------------------- BCFMergesort with buckets, end to end


def _ceil_log2(x):
    return max(0, int(math.ceil(math.log2(x)))) if x > 1 else 0


@pytest.mark.parametrize("pb", [False, True])
def test_sort_full_buckets_equals_library_sort_and_counts_its_phases(pb):
    """oracle.sort_full_buckets (PAPER.md 3.2, App. B): the result is the sorted input (numpy's sort, an
    independent routine) for distinct keys, heavy duplicates, 0-1 data, ragged n and every P; the number of
    rounds of both merge phases is the paper's: ceil(log2(tiles / P)) before the distribution ("suspend the
    merge at s = P", L131) and ceil(log2 s) = log P inside the buckets (L143)."""
    rng = np.random.default_rng(31 + pb)
    w, M = 4, 16                                        # small tiles keep the ShearSort cheap; w = 32 below
    for trial in range(60):
        P = int(rng.choice([2, 3, 4, 8]))
        tiles = int(rng.integers(1, 40))
        n = tiles * M - int(rng.integers(0, M))
        kind = trial % 3
        if kind == 0:
            keys = rng.permutation(1 << 14)[:n].astype(np.uint32)
        elif kind == 1:
            keys = rng.integers(0, 5, size=n).astype(np.uint32)
        else:
            keys = rng.integers(0, 2, size=n).astype(np.uint32)
        t = int(rng.choice([1, 2, P, 2 * P]))
        runs0 = -(-n // M)
        r1 = 0
        while -(-runs0 // (1 << r1)) > P:
            r1 += 1
        s = -(-n // (M << r1))
        if s > 1 and s * t < P:
            t = P
        out, info = oracle.sort_full_buckets(keys, P, t=t, pivot_buckets=pb, w=w, return_info=True)
        assert np.array_equal(out, np.sort(keys, kind="stable"))
        assert info["first_phase_rounds"] == r1 and info["s"] == s and info["run_len"] == M << r1
        if s > 1:
            # log P rounds wherever a bucket is non-empty; only all-pivot data (pivot buckets) has none to merge
            assert info["final_phase_rounds"] in ((0, _ceil_log2(s)) if pb else (_ceil_log2(s),))
            assert sum(info["bucket_sizes"]) == n and len(info["bucket_sizes"]) == (2 * P - 1 if pb else P)
    keys = np.random.default_rng(5).integers(0, 1 << 32, size=20 * 1024 + 77, dtype=np.uint64).astype(np.uint32)
    assert np.array_equal(oracle.sort_full_buckets(keys, 8, pivot_buckets=pb), np.sort(keys))
    assert np.array_equal(oracle.sort_full_buckets(keys, 8, pivot_buckets=pb), oracle.sort_full(keys))
    k64 = np.random.default_rng(6).integers(0, 1 << 63, size=9 * 1024 + 5, dtype=np.uint64)
    assert np.array_equal(oracle.sort_full_buckets(k64, 4, pivot_buckets=pb), np.sort(k64))


def test_sort_full_buckets_pivot_buckets_skip_the_final_phase_on_zero_one_data():
    """with pivot buckets every key of 0-1 data equals a pivot, so the final merge phase
    has nothing to merge (0 rounds), while the plain distribution still runs log P rounds in its buckets."""
    rng = np.random.default_rng(77)
    keys = rng.integers(0, 2, size=64 * 16).astype(np.uint32)
    out, info = oracle.sort_full_buckets(keys, 8, pivot_buckets=True, w=4, return_info=True)
    assert np.array_equal(out, np.sort(keys)) and info["final_phase_rounds"] == 0
    assert sum(info["bucket_sizes"][0::2]) == 0
    out, info = oracle.sort_full_buckets(keys, 8, pivot_buckets=False, w=4, return_info=True)
    assert np.array_equal(out, np.sort(keys)) and info["final_phase_rounds"] == 3


def test_merge_round_and_merge_pieces_pins():
    """oracle.merge_round = one round of oracle.merge_runs (pinned elsewhere against library sorts);
    oracle.merge_pieces of sorted pieces = the sorted concatenation, ceil(log2 s) rounds, empty pieces allowed."""
    rng = np.random.default_rng(8)
    for trial in range(50):
        n = int(rng.integers(1, 300)); L = int(rng.integers(1, 40))
        keys = workloads.sorted_runs(rng.integers(0, 9, size=n).astype(np.uint32), L)
        one = oracle.merge_round(keys, L)
        assert np.array_equal(one, workloads.sorted_runs(keys, 2 * L))
        s = int(rng.integers(1, 9))
        pieces = [np.sort(rng.integers(0, 7, size=int(rng.integers(0, 12))).astype(np.uint32)) for _ in range(s)]
        merged, rounds = oracle.merge_pieces(pieces)
        assert np.array_equal(merged, np.sort(np.concatenate(pieces))) and rounds == _ceil_log2(s)
