"""Seeded synthetic inputs for BASELINE.json's five configs.

This module holds NONE of the method's arithmetic: it only draws numbers.  It is the one
module that both the CPU oracle's tests and the CUDA path's tests/bench use, so that parity
never depends on two generators agreeing: every input is generated once on the host, as a
numpy array, and the same buffer is handed to both sides.

Generator: numpy's counter-based Philox bit generator, raw 64-bit outputs
(`np.random.Philox(key=seed).random_raw(n)`, a stream numpy guarantees bit-for-bit),
seed = 0x5EED0000 + 16 * config + variant.  The paper's own data sets (PAPER.md:L165:
uniform keys, a shuffled permutation, 0-1, k copies of n/k keys) are synthetic by
description; these configs stand in for them.

Every function takes the element count as a parameter (default: BASELINE.json's size) so
parity tests can use the same recipe at sizes the oracle finishes in seconds.
"""
import numpy as np

TILE = 1024  # w*w, w = 32


def seed_for(config: int, variant: int = 0) -> int:
    return 0x5EED0000 + 16 * int(config) + int(variant)


def raw_draws(seed: int, n: int) -> np.ndarray:
    """n raw 64-bit draws of the Philox stream keyed by `seed`."""
    return np.random.Philox(key=int(seed)).random_raw(int(n)).astype(np.uint64, copy=False)


def cfg1_tiles_u32(num_tiles: int = 1024, variant: int = 0):
    """Config 1: `num_tiles` independent 32x32 tiles of uint32 keys, i.i.d. uniform over [0, 2^32)."""
    d = raw_draws(seed_for(1, variant), num_tiles * TILE)
    return (d & np.uint64(0xFFFFFFFF)).astype(np.uint32)


def cfg2_tiles_u32_u32(num_tiles: int = 1 << 16, variant: int = 0):
    """Config 2: tiles of (uint32 key, uint32 value): key uniform over [0, 16), value = global index."""
    n = num_tiles * TILE
    d = raw_draws(seed_for(2, variant), n)
    keys = (d % np.uint64(16)).astype(np.uint32)
    vals = np.arange(n, dtype=np.uint32)
    return keys, vals


def cfg3_sort_u32(n: int = 1 << 24, variant: int = 0):
    """Config 3: n uint32 keys i.i.d. uniform over [0, 2^32)."""
    d = raw_draws(seed_for(3, variant), n)
    return (d & np.uint64(0xFFFFFFFF)).astype(np.uint32)


CFG4_VARIANTS = ("uniform", "sorted", "reverse", "dup256", "zipf")


def cfg4_sort_u32(dist: str = "uniform", n: int = 1 << 28):
    """Config 4: n uint32 keys under one of five distributions (cfg 4a-4e).

    uniform : i.i.d. over [0, 2^32)
    sorted  : key[i] = i
    reverse : key[i] = n - 1 - i
    dup256  : 256 distinct values: a table of 256 distinct draws, key = table[draw mod 256]
    zipf    : Zipf(s = 1.1) over [0, 2^20): key = rank - 1 by inverse-CDF lookup in a
              2^20-entry cumulative table of k^-1.1
    """
    variant = CFG4_VARIANTS.index(dist)
    seed = seed_for(4, variant)
    if dist == "sorted":
        return np.arange(n, dtype=np.uint32)
    if dist == "reverse":
        return (np.uint32(n - 1) - np.arange(n, dtype=np.uint32)).astype(np.uint32)
    d = raw_draws(seed, n)
    if dist == "uniform":
        return (d & np.uint64(0xFFFFFFFF)).astype(np.uint32)
    if dist == "dup256":
        t = raw_draws(seed ^ 0x7AB1E, 4096)
        t = (t & np.uint64(0xFFFFFFFF)).astype(np.uint32)
        _, first = np.unique(t, return_index=True)
        table = t[np.sort(first)][:256]
        assert table.size == 256
        return table[(d % np.uint64(256)).astype(np.int64)]
    if dist == "zipf":
        k = np.arange(1, (1 << 20) + 1, dtype=np.float64)
        cdf = np.cumsum(k ** -1.1)
        u = (d >> np.uint64(11)).astype(np.float64) * (2.0 ** -53) * cdf[-1]
        r = np.searchsorted(cdf, u, side="right")
        return np.minimum(r, (1 << 20) - 1).astype(np.uint32)
    raise ValueError(dist)


def cfg5a_sort_u64_u32(n: int = 1 << 26, variant: int = 0):
    """Config 5a: (uint64 key, uint32 value): per element the draw's top bit picks a uniform
    64-bit key or one of 1024 repeated 64-bit values; value = input index."""
    seed = seed_for(5, variant)
    d = raw_draws(seed, n)
    u = raw_draws(seed ^ 0x0F0F0F, n)
    table = raw_draws(seed ^ 0x7AB1E, 1024)
    rep = table[(d % np.uint64(1024)).astype(np.int64)]
    top = (d >> np.uint64(63)).astype(bool)
    keys = np.where(top, u, rep).astype(np.uint64)
    vals = np.arange(n, dtype=np.uint32)
    return keys, vals


def cfg5b_merge_runs_u32(k: int, n: int = 1 << 27, variant: int = 0):
    """Config 5b (merge-only): n uniform uint32 keys in k equal runs, each run pre-sorted on the
    host with numpy's library sort.  Returns (keys, run_len)."""
    assert n % k == 0
    d = raw_draws(seed_for(5, 8 + variant), n)
    keys = (d & np.uint64(0xFFFFFFFF)).astype(np.uint32)
    run_len = n // k
    keys = np.sort(keys.reshape(k, run_len), axis=1).reshape(-1)
    return keys, run_len


def sorted_runs(keys: np.ndarray, run_len: int, vals: np.ndarray = None):
    """Sort each run [i*run_len, min(n,(i+1)*run_len)) of an arbitrary input by (key, value) with
    numpy's library sort -- input preparation for merge tests with ragged runs."""
    keys = np.array(keys, copy=True)
    vals = None if vals is None else np.array(vals, copy=True)
    n = keys.size
    for lo in range(0, n, run_len):
        hi = min(n, lo + run_len)
        if vals is None:
            keys[lo:hi] = np.sort(keys[lo:hi])
        else:
            order = np.lexsort((vals[lo:hi], keys[lo:hi]))
            keys[lo:hi] = keys[lo:hi][order]
            vals[lo:hi] = vals[lo:hi][order]
    return keys if vals is None else (keys, vals)
