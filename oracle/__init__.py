"""CPU oracle for the hot path of arXiv 1306.5076 -- TEST INFRASTRUCTURE, not the product.

Thin ctypes wrapper over oracle/libbcf_oracle.so (plain C, see bcf_oracle_impl.h for the
arithmetic and its PAPER.md citations).  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package; the CUDA path
(paper_1306_5076_b200) never does, and this package never imports it.

All functions take numpy arrays (keys: uint32 or uint64; vals: uint32 or None), leave their
inputs untouched and return new arrays.
"""
import ctypes
import os

import numpy as np

from . import build as _build

_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        path = _build.build()
        lib = ctypes.CDLL(path)
        vp, sz, ci = ctypes.c_void_p, ctypes.c_size_t, ctypes.c_int
        for s in ("k32", "k64"):
            getattr(lib, f"bcf_oracle_shearsort_tiles_{s}").argtypes = [vp, vp, sz, sz, ci, ci]
            getattr(lib, f"bcf_oracle_merge_two_{s}").argtypes = [vp, vp, sz, vp, vp, sz, vp, vp]
            getattr(lib, f"bcf_oracle_merge_runs_{s}").argtypes = [vp, vp, sz, sz]
            getattr(lib, f"bcf_oracle_sort_full_{s}").argtypes = [vp, vp, sz, sz]
            getattr(lib, f"bcf_oracle_corank_{s}").argtypes = [vp, vp, sz, vp, vp, sz, sz]
            getattr(lib, f"bcf_oracle_corank_{s}").restype = sz
            getattr(lib, f"bcf_oracle_shearsort_merge_{s}").argtypes = [vp, vp, sz, sz]
            getattr(lib, f"bcf_oracle_binary_merge_pagewise_{s}").argtypes = [vp, vp, sz, vp, vp, sz, vp, vp, sz]
        _LIB = lib
    return _LIB


def _suffix(keys):
    if keys.dtype == np.uint32:
        return "k32"
    if keys.dtype == np.uint64:
        return "k64"
    raise TypeError(f"keys must be uint32 or uint64, got {keys.dtype}")


def _prep(keys, vals, copy=True):
    k = np.array(keys, copy=True) if copy else np.ascontiguousarray(keys)
    k = np.ascontiguousarray(k)
    _suffix(k)
    v = None
    if vals is not None:
        v = np.array(vals, dtype=np.uint32, copy=True) if copy else np.ascontiguousarray(vals, dtype=np.uint32)
        if v.shape != k.shape:
            raise ValueError("keys and vals must have the same shape")
    return k, v


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _ret(k, v):
    return k if v is None else (k, v)


def _check(rc, what):
    if rc < 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")
    return rc


def shearsort_tiles(keys, vals=None, w=32, final_snake=False, phases=-1):
    """ShearSort (Alg. 1) each consecutive row-major w*w tile of a flat array."""
    k, v = _prep(keys, vals)
    k = k.reshape(-1)
    if v is not None:
        v = v.reshape(-1)
    if w <= 0 or k.size % (w * w):
        raise ValueError("size must be a multiple of w*w")
    fn = getattr(_lib(), f"bcf_oracle_shearsort_tiles_{_suffix(k)}")
    _check(fn(_p(k), _p(v), k.size // (w * w), w, int(bool(final_snake)), int(phases)), "shearsort_tiles")
    return _ret(k, v)


def merge_two(ka, kb, va=None, vb=None):
    """Two-finger merge of two sorted sequences, ties from A."""
    a, av = _prep(ka, va, copy=False)
    b, bv = _prep(kb, vb, copy=False)
    if a.dtype != b.dtype or (av is None) != (bv is None):
        raise TypeError("A and B must have the same element type")
    ko = np.empty(a.size + b.size, dtype=a.dtype)
    vo = None if av is None else np.empty(a.size + b.size, dtype=np.uint32)
    fn = getattr(_lib(), f"bcf_oracle_merge_two_{_suffix(a)}")
    _check(fn(_p(a), _p(av), a.size, _p(b), _p(bv), b.size, _p(ko), _p(vo)), "merge_two")
    return _ret(ko, vo)


def merge_runs(keys, run_len, vals=None, return_rounds=False):
    """Pairwise merge rounds over sorted runs of run_len."""
    k, v = _prep(keys, vals)
    fn = getattr(_lib(), f"bcf_oracle_merge_runs_{_suffix(k)}")
    rounds = _check(fn(_p(k), _p(v), k.size, int(run_len)), "merge_runs")
    out = _ret(k, v)
    return (out, rounds) if return_rounds else out


def sort_full(keys, vals=None, w=32, return_rounds=False):
    """BCFMergesort: ShearSort base case on w*w tiles + merge rounds (section 3)."""
    k, v = _prep(keys, vals)
    fn = getattr(_lib(), f"bcf_oracle_sort_full_{_suffix(k)}")
    rounds = _check(fn(_p(k), _p(v), k.size, int(w)), "sort_full")
    out = _ret(k, v)
    return (out, rounds) if return_rounds else out


def corank(ka, kb, d, va=None, vb=None):
    """Number of elements the A-first two-finger merge takes from A for its first d outputs."""
    a, av = _prep(ka, va, copy=False)
    b, bv = _prep(kb, vb, copy=False)
    if a.dtype != b.dtype or (av is None) != (bv is None):
        raise TypeError("A and B must have the same element type")
    fn = getattr(_lib(), f"bcf_oracle_corank_{_suffix(a)}")
    r = fn(_p(a), _p(av), a.size, _p(b), _p(bv), b.size, int(d))
    if r == ctypes.c_size_t(-1).value:
        raise RuntimeError("oracle corank failed")
    return int(r)


def shearsort_merge(keys, na, vals=None, w=32):
    """SHEARSORT-MERGE on one page of w*w elements: [0,na) and [na,w*w) sorted (A8)."""
    k, v = _prep(keys, vals)
    if k.size != w * w:
        raise ValueError("page must hold w*w elements")
    fn = getattr(_lib(), f"bcf_oracle_shearsort_merge_{_suffix(k)}")
    _check(fn(_p(k), _p(v), int(w), int(na)), "shearsort_merge")
    return _ret(k, v)


def binary_merge_pagewise(ka, kb, va=None, vb=None, w=32):
    """BINARY-MERGE, the page-wise streaming merge of PAPER.md Alg. 6 with M = w*w."""
    a, av = _prep(ka, va, copy=False)
    b, bv = _prep(kb, vb, copy=False)
    if a.dtype != b.dtype or (av is None) != (bv is None):
        raise TypeError("A and B must have the same element type")
    ko = np.empty(a.size + b.size, dtype=a.dtype)
    vo = None if av is None else np.empty(a.size + b.size, dtype=np.uint32)
    fn = getattr(_lib(), f"bcf_oracle_binary_merge_pagewise_{_suffix(a)}")
    _check(fn(_p(a), _p(av), a.size, _p(b), _p(bv), b.size, _p(ko), _p(vo), int(w)), "binary_merge_pagewise")
    return _ret(ko, vo)


def corank_multi(runs_keys, d, runs_vals=None):
    """Split of the first d outputs of the stable k-way merge of sorted runs (ties: lower run first,
    then lower position) -- the definition the four-run partition of a pass must meet (the pass does
    two rounds of PAPER.md:L103 at once; north_star: "split-point search so each CTA gets an equal
    share of output").  Written out as the definition: concatenate the runs, sort STABLY by
    (key, value) -- a stable sort of the concatenation orders equal elements by run, then position --
    and count how many of the first d come from each run.  Returns a list of k counts summing to d."""
    ks = [np.ascontiguousarray(r) for r in runs_keys]
    lens = [r.size for r in ks]
    if not 0 <= d <= sum(lens):
        raise ValueError("d out of range")
    cat = np.concatenate(ks) if ks else np.empty(0, dtype=np.uint32)
    if runs_vals is None:
        order = np.argsort(cat, kind="stable")
    else:
        vcat = np.concatenate([np.ascontiguousarray(v, dtype=np.uint32) for v in runs_vals])
        order = np.lexsort((vcat, cat))      # lexsort is stable: last key is primary
    first = order[:d]
    bounds = np.cumsum([0] + lens)
    return [int(np.count_nonzero((first >= bounds[r]) & (first < bounds[r + 1]))) for r in range(len(ks))]


def alg7_sample_index(i, length, t):
    """Position of potential splitter i (0 <= i < t) in a sorted run of `length` elements.
    PAPER.md Alg. 7: "S[pid t + i] = I_pid[i n/t]" -> floor(i length / t): the first sample is the
    run's first element.  Pinned by tests/golden/alg7_worked_example.txt (S_UNSORTED)."""
    return (i * length) // t


def alg7_pivot_index(j, s, t, P):
    """Position in the sorted sample array S (s t entries) of final pivot j (0 <= j < P - 1).
    PAPER.md L135 "P-1 evenly spaced items from S", Alg. 7 "every t-th element of S" (s = P runs):
    S[t], S[2t], .. = S[floor((j+1) s t / P)].  Pinned by tests/golden/alg7_worked_example.txt (F)."""
    return ((j + 1) * s * t) // P


def find_buckets(keys, run_len, t, P, pivot_buckets=False, return_steps=False):
    """FIND-BUCKETS, section 3.2 "Distribution" (L131-137) / Algorithm 7 (L492-520), with the
    pivot buckets of L155 as an option; reading A18 of DESIGN.md for the garbled lines.  Step by step:
      1. S: t samples of each of the s sorted runs, sample i of run r = its element floor(i len_r / t)
         (Alg. 7: "S[pid t + i] = I_pid[i n/t]");
      2. MERGESORT(S) (L505) -- a library sort serves as the step;
      3. pivots F[j] = S[floor((j+1) s t / P)], j = 0..P-2 ("P-1 evenly spaced items from S", L135);
      4. rank of every pivot in every run = number of elements <= pivot (L507-510: first i with
         I[i] > F[c]); with pivot buckets also the number of elements < pivot;
      5. bucket sizes summed over the runs, exclusive prefix sums (L512-513);
      6. O = the runs' pieces regrouped by bucket, inside a bucket by run (L515-520).
    Keys only.  Returns (O, F, Q) with Q[b s + r] = start of piece (bucket b, run r) in O, Q[-1] = n;
    with return_steps also a dict of the intermediate arrays (S unsorted, S sorted, ranks) the golden pins."""
    k = np.ascontiguousarray(keys)
    _suffix(k)
    n = k.size
    s = -(-n // run_len)
    runs = [k[r * run_len:min(n, (r + 1) * run_len)] for r in range(s)]
    S_unsorted = np.array([run[alg7_sample_index(i, run.size, t)] for run in runs for i in range(t)], dtype=k.dtype)
    S = np.sort(S_unsorted, kind="stable")
    F = np.array([S[alg7_pivot_index(j, s, t, P)] for j in range(P - 1)], dtype=k.dtype)
    nb = 2 * P - 1 if pivot_buckets else P
    bounds = np.zeros((s, nb + 1), dtype=np.int64)
    for r, run in enumerate(runs):
        le = np.searchsorted(run, F, side="right")
        if not pivot_buckets:
            bounds[r, 1:P] = le
        else:
            lt = np.searchsorted(run, F, side="left")
            for j in range(P - 1):
                dup = j > 0 and F[j] == F[j - 1]        # the second copy of a repeated pivot owns nothing
                bounds[r, 2 * j + 1] = le[j] if dup else lt[j]
                bounds[r, 2 * j + 2] = le[j]
        bounds[r, nb] = run.size
    O = np.empty_like(k)
    Q = np.zeros(nb * s + 1, dtype=np.int64)
    oc = 0
    for b in range(nb):
        for r, run in enumerate(runs):
            piece = run[bounds[r, b]:bounds[r, b + 1]]
            Q[b * s + r] = oc
            O[oc:oc + piece.size] = piece
            oc += piece.size
    Q[nb * s] = oc
    if return_steps:
        rank_le = np.array([[int(np.searchsorted(run, f, side="right")) for run in runs] for f in F], dtype=np.int64)
        return O, F, Q, {"S_unsorted": S_unsorted, "S_sorted": S, "rank_le": rank_le.reshape(P - 1, s)}
    return O, F, Q


def base_case_runs(keys, w=32):
    """Base case phase alone (section 3, App. B): every tile of w*w keys ShearSorted, a last
    partial tile padded with the maximum key (L420) and cut back.  Returns the array of sorted runs of w*w."""
    k = np.ascontiguousarray(keys)
    M = w * w
    out = np.empty_like(k)
    full = (k.size // M) * M
    if full:
        out[:full] = shearsort_tiles(k[:full], w=w)
    if full < k.size:
        pad = np.full(M, np.iinfo(k.dtype).max, dtype=k.dtype)
        pad[:k.size - full] = k[full:]
        out[full:] = shearsort_tiles(pad, w=w)[:k.size - full]
    return out


def merge_round(keys, run_len):
    """ONE round of pairwise merging: runs 2p, 2p+1 of run_len -> one run of 2 run_len,
    two-finger merge (L125); an odd last run is copied through."""
    k = np.ascontiguousarray(keys)
    out = np.empty_like(k)
    for a0 in range(0, k.size, 2 * run_len):
        a1 = min(k.size, a0 + run_len)
        b1 = min(k.size, a1 + run_len)
        out[a0:b1] = merge_two(k[a0:a1], k[a1:b1]) if b1 > a1 else k[a0:a1]
    return out


def merge_pieces(pieces):
    """Final merge phase inside ONE bucket (section 3.2 "Final merge phase" L141-143, App. B):
    the bucket's sorted subsequences (one per run, any lengths, possibly empty) merged pairwise in
    ceil(log2 s) rounds of two-finger merges; a piece without a partner is carried to the next round.
    Returns (sorted bucket, rounds)."""
    cur = [np.ascontiguousarray(p) for p in pieces]
    rounds = 0
    while len(cur) > 1:
        cur = [merge_two(cur[i], cur[i + 1]) if i + 1 < len(cur) else cur[i] for i in range(0, len(cur), 2)]
        rounds += 1
    return (cur[0] if cur else np.empty(0, dtype=np.uint32)), rounds


def sort_full_buckets(keys, P, t=None, pivot_buckets=False, w=32, return_info=False):
    """BCFMergesort with the paper's bucket distribution, end to end (BCFMergesortPB when pivot_buckets):
    PAPER.md section 3.2 and App. B, the four phases in the paper's order:
      1. base case: tiles of M = w*w keys ShearSorted (L103, L236);
      2. first merge phase: rounds of pairwise merging while more than P runs remain -- "we suspend the
         merge at s = P" (L131; for run counts that are not P * 2^k: at the first s <= P);
      3. bucket distribution: FIND-BUCKETS on the s runs with t samples per run (default t = P, L139) and
         P buckets (2P-1 with pivot buckets, L155) -- find_buckets above;
      4. final merge phase: "CTA p_i then sorts the i-th bucket by merging the sorted subsequences of the
         bucket" (L141), ceil(log2 s) rounds inside every bucket (L143); a pivot bucket holds copies of one
         key and is already final (L155).
    A single run after phase 2 (s = 1) is the result.  Keys only.  With return_info also a dict: runs s at the
    distribution, run length, rounds of both merge phases, bucket sizes."""
    k = np.ascontiguousarray(keys)
    _suffix(k)
    n, M = k.size, w * w
    t = P if t is None else t
    cur = base_case_runs(k, w)
    run_len, rounds1 = M, 0
    while -(-n // run_len) > P:
        cur = merge_round(cur, run_len)
        run_len *= 2
        rounds1 += 1
    s = -(-n // run_len) if n else 0
    info = {"s": s, "run_len": run_len, "first_phase_rounds": rounds1, "final_phase_rounds": 0, "bucket_sizes": []}
    if s <= 1:
        return (cur, info) if return_info else cur
    O, F, Q = find_buckets(cur, run_len, t, P, pivot_buckets=pivot_buckets)
    nb = 2 * P - 1 if pivot_buckets else P
    out = np.empty_like(k)
    for b in range(nb):
        lo, hi = int(Q[b * s]), int(Q[(b + 1) * s])
        info["bucket_sizes"].append(hi - lo)
        if hi == lo:
            continue                                    # an empty bucket has nothing to merge
        if pivot_buckets and b % 2 == 1:
            out[lo:hi] = O[lo:hi]                       # copies of pivot (b-1)/2: already in final position
            continue
        merged, r = merge_pieces([O[int(Q[b * s + i]):int(Q[b * s + i + 1])] for i in range(s)])
        out[lo:hi] = merged
        info["final_phase_rounds"] = max(info["final_phase_rounds"], r)
    return (out, info) if return_info else out


def colored_prefix_sums(values, colors, num_colors):
    """Coloured prefix sums (Appendix A): "given an array of N elements and a set of d
    colors, with a color associated with each element, compute d independent prefix sums among the
    elements of the same color".  The definition written out, one element after the other:
    out[i] = sum of values[j], j <= i, colors[j] == colors[i] (inclusive), uint32 arithmetic."""
    v = np.ascontiguousarray(values, dtype=np.uint32)
    c = np.ascontiguousarray(colors, dtype=np.uint8)
    if v.shape != c.shape or (c.size and int(c.max()) >= num_colors):
        raise ValueError("bad colours")
    running = [0] * num_colors
    out = np.empty_like(v)
    vi, ci = v.tolist(), c.tolist()
    res = [0] * len(vi)
    for i in range(len(vi)):
        k = ci[i]
        running[k] = (running[k] + vi[i]) & 0xFFFFFFFF
        res[i] = running[k]
    out[:] = np.array(res, dtype=np.uint32) if res else out
    return out
