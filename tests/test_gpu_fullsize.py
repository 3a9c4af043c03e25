"""GPU checks at BASELINE.json's FULL sizes, in the launch configuration bench.py times (library
defaults, bcf_options = NULL).  Where the oracle finishes in seconds the output is compared element by
element with it (config 3); elsewhere:
  keys only   EVERY element against numpy's library sort of the same input (the result is the unique
              ascending arrangement of the input multiset, so any correct sort is the expected value) --
              all five distributions of config 4 and all three run counts of config 5b, the duplicate-heavy
              ones included (they are the ones that stress the tie rule of the co-rank searches);
  key-value   (values = input index) non-decreasing in (key, value), the values are a permutation of
              0..n-1 and out_key[i] == in_key[out_val[i]] for every i -- together these determine the
              output uniquely;
plus sampled tiles against the oracle's ShearSort."""
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
    return m


def dev(a):
    signed = {np.dtype(np.uint32): np.int32, np.dtype(np.uint64): np.int64}[a.dtype]
    return torch.from_numpy(np.ascontiguousarray(a).view(signed)).cuda()


def host(t, like):
    return t.cpu().numpy().view(like.dtype)


def check_keys_only(inp, out):
    """Element by element against numpy's sort of the input."""
    assert out.shape == inp.shape
    want = np.sort(inp, kind="stable")
    if not np.array_equal(out, want):
        bad = np.flatnonzero(out != want)
        raise AssertionError("first mismatch at %d of %d (%d wrong): got %d want %d"
                             % (bad[0], inp.size, bad.size, out[bad[0]], want[bad[0]]))


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
def test_config4_full_size_vs_numpy_sort_unique_result(bcf, dist):
    """2^28 uint32 keys, each of the five distributions."""
    keys = workloads.cfg4_sort_u32(dist)
    d = dev(keys)
    bcf.sort(d)
    out = host(d, keys)
    del d
    torch.cuda.empty_cache()
    check_keys_only(keys, out)
    if dist in ("sorted", "reverse"):
        assert np.array_equal(out, np.arange(keys.size, dtype=np.uint32))


def test_config4_full_size_paper_base_case_and_two_rounds_per_pass(bcf):
    """The paper's tile ShearSort as base case, and the four-run kernel, at 2^28: same output as the default."""
    keys = workloads.cfg4_sort_u32("dup256")
    d = dev(keys)
    bcf.sort(d)
    want = host(d, keys).copy()
    for base, rpp, mode in ((bcf.BASE_SHEARSORT, 1, bcf.LAUNCH_PLAIN), (bcf.BASE_TILE_MERGESORT, 2, bcf.LAUNCH_PDL),
                            (bcf.BASE_LONG_TILES, 2, bcf.LAUNCH_PLAIN), (bcf.BASE_LONG_TILES, 1, bcf.LAUNCH_PDL)):
        d.copy_(dev(keys))
        bcf.sort(d, opts={"base_case": base, "rounds_per_pass": rpp, "launch_mode": mode})
        assert np.array_equal(host(d, keys), want), (base, rpp, mode)


@pytest.mark.parametrize("data", ["zero_one", "dup256", "uniform"])
def test_sort_buckets_full_size_vs_numpy_sort_unique_result(bcf, data):
    """BCFMergesort with the paper's distribution (t = P = 128, the paper's p) and BCFMergesortPB at 2^27 keys
    (the size of bench.py's side line): every element against numpy's sort; 0-1 data is the paper's 15.5x case."""
    n = 1 << 27
    rng = np.random.Generator(np.random.Philox(key=workloads.seed_for(6, 1)))
    if data == "zero_one":
        keys = rng.integers(0, 2, size=n, dtype=np.uint32)
    elif data == "dup256":
        keys = workloads.cfg4_sort_u32("dup256", n=n)
    else:
        keys = workloads.cfg4_sort_u32("uniform", n=n)
    want = np.sort(keys)
    for pb in (False, True):
        d = dev(keys)
        bcf.sort_buckets(d, 128, pivot_buckets=pb)
        assert np.array_equal(host(d, keys), want), (data, pb)
        del d
        torch.cuda.empty_cache()


def test_config5a_full_size_by_the_properties_that_fix_the_unique_result(bcf):
    """2^26 (u64 key, u32 value = index) pairs: the properties determine the output uniquely."""
    keys, vals = workloads.cfg5a_sort_u64_u32()
    dk, dv = dev(keys), dev(vals)
    bcf.sort(dk, dv)
    check_key_value(keys, host(dk, keys), host(dv, vals))


@pytest.mark.parametrize("k", [2, 64, 1024])
def test_config5b_full_size_vs_numpy_sort_unique_result(bcf, k):
    """merge-only: k sorted runs totalling 2^27 uint32 keys."""
    keys, run_len = workloads.cfg5b_merge_runs_u32(k)
    out = host(bcf.merge_runs(dev(keys), run_len), keys)
    torch.cuda.empty_cache()
    check_keys_only(keys, out)


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


# ---------------------------------------------------------------- the size range include/bcf.h promises (n < 2^32)


def _flip(t):
    """int tensor holding unsigned bit patterns -> same tensor with unsigned order mapped onto signed order."""
    return t ^ torch.iinfo(t.dtype).min


def test_sort_more_than_2_pow_31_uint32_keys_by_rank_counting(bcf):
    """n = 2^31 + 4099 uint32 keys (8 GiB + 8 GiB workspace): past every 31-bit index.  numpy / the oracle cannot hold
    this in reasonable time, so the unique result is checked by what defines it: the output is ascending (unsigned), it
    has the input's histogram over the top 16 key bits and the input's wrapping sums of x and x^2, and at 48 sampled
    positions p (the ends, the 2^31 boundary, random ones) the element is the one of rank p: #(input < out[p]) <= p <
    #(input <= out[p]), counted over the whole input."""
    n = (1 << 31) + 4099
    g = torch.Generator(device="cuda")
    g.manual_seed(0x5EED31)
    src = torch.randint(-2**31, 2**31, (n,), dtype=torch.int32, device="cuda", generator=g)
    src[12345] = -1                                    # 0xFFFFFFFF, the padding value, as a real key
    d = src.clone()
    bcf.sort(d)
    torch.cuda.synchronize()
    fd = _flip(d)
    assert bool((fd[1:] >= fd[:-1]).all())
    del fd
    hist = lambda t: torch.bincount(((t >> 16) & 0xFFFF).to(torch.int64), minlength=1 << 16)   # noqa: E731
    assert torch.equal(hist(d), hist(src))
    for power in (1, 2):
        assert int((d.to(torch.int64) ** power).sum()) == int((src.to(torch.int64) ** power).sum())
    fs = _flip(src)
    rng = np.random.default_rng(31)
    for p in [0, 1, n - 1, n - 2, (1 << 31) - 1, 1 << 31, (1 << 31) + 1] + [int(x) for x in rng.integers(0, n, size=41)]:
        v = int(d[p]) ^ -2**31                          # flipped value, python int
        below, upto = int((fs < v).sum()), int((fs <= v).sum())
        assert below <= p < upto, (p, below, upto)


def test_sort_2_pow_30_key_value_pairs_by_properties(bcf):
    """n = 2^30 + 77 (u64 key, u32 value = input index) pairs, keys with many duplicates: ascending by (key, value),
    the values are a permutation of the indices, and every key travelled with its value -- together these fix the output."""
    n = (1 << 30) + 77
    g = torch.Generator(device="cuda")
    g.manual_seed(0x5EED30)
    keys = (torch.randint(0, 1 << 22, (n,), dtype=torch.int64, device="cuda", generator=g) << 41) | 5   # bit 63 set for half
    vals = torch.arange(n, dtype=torch.int32, device="cuda")
    dk, dv = keys.clone(), vals.clone()
    bcf.sort(dk, dv)
    torch.cuda.synchronize()
    fk = _flip(dk)
    later = fk[1:] > fk[:-1]
    tie = fk[1:] == fk[:-1]
    assert bool((later | tie).all())
    assert bool((~tie | (dv[1:] > dv[:-1])).all())      # equal keys: by value (indices < 2^31, signed compare is right)
    assert int(tie.sum()) > n // 2                       # the tie rule really was exercised
    del fk, later, tie
    seen = torch.zeros(n, dtype=torch.bool, device="cuda")
    seen[dv.to(torch.int64)] = True
    assert bool(seen.all())
    assert torch.equal(keys[dv.to(torch.int64)], dk)
