"""GPU checks at BASELINE.json's FULL sizes, in the launch configuration bench.py times (library
defaults: base case AUTO, one merge round per pass).  Where the oracle finishes in seconds the output is
compared element by element (config 3); elsewhere the output is pinned by properties that hold at any
size and determine it uniquely:
  keys only   non-decreasing, permutation-invariant checksums equal to the input's, and for sampled
              positions i the rank bounds  #(input < out[i]) <= i < #(input <= out[i])  -- the plain
              definition of "the i-th smallest", counted over the whole input;
  key-value   (values = input index) non-decreasing in (key, value), the values are a permutation of
              0..n-1 and out_key[i] == in_key[out_val[i]] for every i;
plus sampled tiles / one full variant against the oracle itself and against numpy's library sort."""
import numpy as np
import pytest

import oracle
from paper_1306_5076_b200 import workloads

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bcf():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1306_5076_b200 as m
    m.lib()
    assert m.get_base_case() == m.BASE_AUTO and m.get_rounds_per_pass() == 1   # what bench.py times
    return m


def dev(a):
    signed = {np.dtype(np.uint32): np.int32, np.dtype(np.uint64): np.int64}[a.dtype]
    return torch.from_numpy(np.ascontiguousarray(a).view(signed)).cuda()


def host(t, like):
    return t.cpu().numpy().view(like.dtype)


def checksums(a):
    a64 = a.astype(np.uint64, copy=False)
    return (int(a64.sum(dtype=np.uint64)), int((a64 * a64).sum(dtype=np.uint64)), int(np.bitwise_xor.reduce(a64)))


def check_keys_only(inp, out, samples=6, seed=0):
    assert out.shape == inp.shape
    assert bool(np.all(out[:-1] <= out[1:])), "not sorted"
    assert checksums(inp) == checksums(out), "not a permutation of the input"
    rng = np.random.default_rng(seed)
    n = inp.size
    for i in [0, n - 1] + [int(x) for x in rng.integers(0, n, size=samples)]:
        v = out[i]
        less = int(np.count_nonzero(inp < v))
        leq = less + int(np.count_nonzero(inp == v))
        assert less <= i < leq, (i, int(v), less, leq)


def check_key_value(in_keys, out_keys, out_vals):
    n = in_keys.size
    dk = out_keys[1:].astype(np.int64 if out_keys.dtype == np.uint32 else np.uint64)
    same = out_keys[1:] == out_keys[:-1]
    assert bool(np.all((out_keys[1:] > out_keys[:-1]) | (same & (out_vals[1:] > out_vals[:-1])))), "not sorted by (key, value)"
    del dk
    seen = np.zeros(n, dtype=np.bool_)
    seen[out_vals] = True
    assert bool(seen.all()), "values are not a permutation of the input indices"
    assert bool(np.array_equal(out_keys, in_keys[out_vals])), "a key travelled without its value"


def test_config3_full_size_exact(bcf):
    """2^24 uint32 keys: element by element against the oracle (ShearSort tiles + merge rounds)."""
    keys = workloads.cfg3_sort_u32()
    d = dev(keys)
    bcf.sort(d)
    assert np.array_equal(host(d, keys), oracle.sort_full(keys))


@pytest.mark.parametrize("dist", workloads.CFG4_VARIANTS)
def test_config4_full_size(bcf, dist):
    """2^28 uint32 keys, each of the five distributions."""
    keys = workloads.cfg4_sort_u32(dist)
    d = dev(keys)
    bcf.sort(d)
    out = host(d, keys)
    del d
    torch.cuda.empty_cache()
    check_keys_only(keys, out, seed=len(dist))
    if dist == "uniform":                       # one variant against the textbook library sort, in full
        assert np.array_equal(out, np.sort(keys, kind="stable"))
    if dist in ("sorted", "reverse"):
        assert np.array_equal(out, np.arange(keys.size, dtype=np.uint32))


def test_config4_full_size_paper_base_case_and_two_rounds_per_pass(bcf):
    """The paper's tile ShearSort as base case, and the four-run kernel, at 2^28: same output as the default."""
    keys = workloads.cfg4_sort_u32("dup256")
    d = dev(keys)
    bcf.sort(d)
    want = host(d, keys).copy()
    for base, rpp in ((bcf.BASE_SHEARSORT, 1), (bcf.BASE_TILE_MERGESORT, 2)):
        bcf.set_base_case(base)
        bcf.set_rounds_per_pass(rpp)
        try:
            d.copy_(dev(keys))
            bcf.sort(d)
            assert np.array_equal(host(d, keys), want), (base, rpp)
        finally:
            bcf.set_base_case(bcf.BASE_AUTO)
            bcf.set_rounds_per_pass(1)


def test_config5a_full_size(bcf):
    """2^26 (u64 key, u32 value = index) pairs: the properties determine the output uniquely."""
    keys, vals = workloads.cfg5a_sort_u64_u32()
    dk, dv = dev(keys), dev(vals)
    bcf.sort(dk, dv)
    check_key_value(keys, host(dk, keys), host(dv, vals))


@pytest.mark.parametrize("k", [2, 64, 1024])
def test_config5b_full_size(bcf, k):
    """merge-only: k sorted runs totalling 2^27 uint32 keys."""
    keys, run_len = workloads.cfg5b_merge_runs_u32(k)
    out = host(bcf.merge_runs(dev(keys), run_len), keys)
    torch.cuda.empty_cache()
    check_keys_only(keys, out, samples=4, seed=k)


def test_config2_full_size_sampled_tiles(bcf):
    """2^16 tiles of (u32 key in [0,16), u32 value = index): every tile by the key-value properties,
    every 257th tile against the oracle's ShearSort; both tile networks."""
    keys, vals = workloads.cfg2_tiles_u32_u32()
    for fn in (bcf.sort_tiles, bcf.sort_tiles_mergesort):
        dk, dv = dev(keys), dev(vals)
        fn(dk, dv)
        ok, ov = host(dk, keys), host(dv, vals)
        tk, tv = ok.reshape(-1, 1024), ov.reshape(-1, 1024)
        same = tk[:, 1:] == tk[:, :-1]
        assert bool(np.all((tk[:, 1:] > tk[:, :-1]) | (same & (tv[:, 1:] > tv[:, :-1]))))
        assert bool(np.array_equal(ok, keys[ov]))                         # every key with its value
        assert bool(np.all(tv // 1024 == np.arange(tk.shape[0])[:, None]))  # nothing left its tile
        for t in range(0, tk.shape[0], 257):
            sl = slice(1024 * t, 1024 * (t + 1))
            wk, wv = oracle.shearsort_tiles(keys[sl], vals[sl])
            assert np.array_equal(ok[sl], wk) and np.array_equal(ov[sl], wv)
