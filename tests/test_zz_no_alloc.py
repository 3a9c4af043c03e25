"""bcf_merge_round_static: the merge round for callers that cannot allocate device memory.

Some users of the library run where cudaMalloc is off limits at the moment they need to merge: an operator or
plugin called from a host engine's execute step, a process that handed all of the GPU's memory to its own pool at
start-up, a loop that cannot afford the stall an allocation may cause.  bcf_merge_runs is closed to them because
it wants a workspace.  bcf_merge_round_static keeps the only scratch a round needs (its split points) in a fixed
256 KiB array inside libbcf.so, so those callers pass just their own input and output arrays.

What is checked here: the new entry point gives, bit for bit (integer data: the tolerance of every parity test in
this suite is zero), what the existing workspace path bcf_merge_runs gives on the same input -- on two calls in a
row, because the built-in array is shared by all calls and still holds the previous call's split points when the
next one starts.  The file is named test_zz_* so that pytest collects it last: with `pytest -x` a failure here
cannot hide any other test.  It does not depend on what ran before it (it passes alone in a fresh process, where
its first call is the one that does the per-device set-up, and after the rest of the suite).
"""
import ctypes

import numpy as np
import pytest

torch = pytest.importorskip("torch")

KINDS = ["u32", "u32u32", "u64", "u64u32"]


def _sorted_runs(kind, n, run_len, seed):
    """n elements of `kind` whose runs of run_len are each sorted by (key, value); few distinct keys, so equal keys
    meet across runs and the (key, value) tie rule is exercised."""
    rng = np.random.default_rng(seed)
    kdt = np.uint32 if kind.startswith("u32") else np.uint64
    keys = rng.integers(0, max(2, n // 3), size=n, dtype=np.uint64).astype(kdt)
    if kdt is np.uint64:
        keys = keys << np.uint64(29)                       # both 32-bit halves of the key take part
    keys[n // 2] = np.iinfo(kdt).max                       # the padding value is a legal key
    vals = rng.permutation(n).astype(np.uint32) if kind.endswith("u32") and kind != "u32" else None
    for a in range(0, n, run_len):
        b = min(n, a + run_len)
        if vals is None:
            keys[a:b] = np.sort(keys[a:b])
        else:
            order = np.lexsort((vals[a:b], keys[a:b]))
            keys[a:b], vals[a:b] = keys[a:b][order], vals[a:b][order]
    return keys, vals


def _dev(a):
    if a is None:
        return None
    signed = {np.dtype(np.uint32): np.int32, np.dtype(np.uint64): np.int64}[a.dtype]
    return torch.from_numpy(np.ascontiguousarray(a).view(signed)).cuda()


@pytest.fixture(scope="module")
def bcf():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_1306_5076_b200 as m
    m.lib()  # fail loudly if the extension is missing
    return m


def _static_merge_all_rounds(bcf, dk, dv, run_len):
    """What a caller without an allocator does: ceil(log2(#runs)) calls, run_len doubling, between two buffers it
    already owns.  (The test allocates those two buffers with torch; the library call allocates nothing.)"""
    n = dk.numel()
    src_k, src_v = dk, dv
    dst_k, dst_v = torch.empty_like(dk), (None if dv is None else torch.empty_like(dv))
    length = run_len
    while True:
        bcf.merge_round_static(src_k, length, dst_k, vals=src_v, out_vals=dst_v)
        src_k, dst_k, src_v, dst_v = dst_k, src_k, dst_v, src_v
        length *= 2
        if length >= n:
            return src_k, src_v


def _existing_path(bcf, dk, dv, run_len):
    out = bcf.merge_runs(dk, run_len, vals=dv)
    return (out, None) if dv is None else out


@pytest.mark.gpu
@pytest.mark.parametrize("kind", KINDS)
def test_static_round_matches_merge_runs_on_two_calls_in_a_row(bcf, kind):
    """Two calls back to back on the same stream, each compared with bcf_merge_runs on the same input.
    The second call is a different shape (shorter, unequal runs, a ragged last page) than the first, so split points
    left in the shared array by the first call would be wrong for it if anything relied on them."""
    shapes = [(2 * 6144, 6144), (5000 + 3077, 5000)]       # (n, run_len): two runs each -> one round = the full merge
    results = []
    for call, (n, run_len) in enumerate(shapes):
        keys, vals = _sorted_runs(kind, n, run_len, seed=0xA110C + call)
        dk, dv = _dev(keys), _dev(vals)
        out_k = torch.empty_like(dk)
        out_v = None if dv is None else torch.empty_like(dv)
        bcf.merge_round_static(dk, run_len, out_k, vals=dv, out_vals=out_v)
        results.append((dk, dv, run_len, out_k, out_v))
    torch.cuda.synchronize()
    for dk, dv, run_len, out_k, out_v in results:
        want_k, want_v = _existing_path(bcf, dk, dv, run_len)
        assert torch.equal(out_k, want_k)
        if dv is not None:
            assert torch.equal(out_v, want_v)


@pytest.mark.gpu
@pytest.mark.parametrize("kind", ["u32", "u64u32"])
def test_static_rounds_repeated_give_the_full_merge(bcf, kind):
    """Many pairs per round and several rounds in a row (an odd number of runs, a short last run): looping the
    static round with run_len doubling ends in exactly the output of bcf_merge_runs."""
    n, run_len = 11 * 3000 + 123, 3000
    keys, vals = _sorted_runs(kind, n, run_len, seed=0x5747)
    dk, dv = _dev(keys), _dev(vals)
    got_k, got_v = _static_merge_all_rounds(bcf, dk, dv, run_len)
    want_k, want_v = _existing_path(bcf, dk, dv, run_len)
    assert torch.equal(got_k, want_k)
    if dv is not None:
        assert torch.equal(got_v, want_v)


def test_static_round_refuses_rounds_beyond_its_array():
    """The limit is checked before the device is touched, so this runs without a GPU: a round that needs more
    split points than the built-in array holds is refused with BCF_ERR_TOO_LARGE, one that just fits is not
    refused for its size (here it then fails on the missing device or the fake pointers are never reached)."""
    import paper_1306_5076_b200 as m
    L = m.lib()
    cap = m.merge_round_static_max_shares()
    assert cap == 65536
    assert m.merge_round_static_shares(cap * 1024, 1024) == cap
    assert m.merge_round_static_shares(cap * 1024 + 1, 1024) == cap + 2      # one more pair of two pages
    assert m.merge_round_static_shares(10, 1 << 40) == 1                     # one short run: a single page
    fake_in, fake_out = ctypes.c_void_p(0x10000000), ctypes.c_void_p(0x7F0000000000)
    st = L.bcf_merge_round_static(fake_in, None, fake_out, None, cap * 1024 + 1, 1024, 0, 0, None)
    assert L.bcf_status_string(st) == b"BCF_ERR_TOO_LARGE"
    assert L.bcf_merge_round_static(fake_in, None, fake_out, None, 0, 1024, 0, 0, None) == 0    # n = 0: no-op
    assert L.bcf_status_string(L.bcf_merge_round_static(fake_in, None, fake_out, None, 4096, 0, 0, 0, None)) \
        == b"BCF_ERR_INVALID_ARG"
