"""GPU parity: the CUDA path through the C ABI (paper_1306_5076_b200 -> libbcf.so) against the CPU
oracle, element by element, bit-exact (integer work), on the same seeded inputs.  Sizes span several
tiles/shares and ragged tails; every element type; the degenerate cases of the method."""
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
    m.lib()  # fail loudly if the extension is missing
    return m


# bcf_options of the pass structures of the merging phase
RPP = {1: {"rounds_per_pass": 1}, 2: {"rounds_per_pass": 2}, 3: {"rounds_per_pass": 2, "merge_impl": 2},
       4: {"rounds_per_pass": 1, "merge_impl": 3}}


@pytest.fixture(params=[1, 2, 3, 4], ids=["1round", "2rounds", "2rounds-barrier", "1round-partition-launch"])
def rpp(request):
    """The pass structures of the merging phase, passed per call in bcf_options: one round per pass
    (Lemma 2), two rounds per pass (four-run kernels: the task-stream kernel where it applies), and
    two rounds per pass with the barrier version of the four-run kernel everywhere, and one round per pass with a
    partition launch for every round (small rounds otherwise find their split points inside the merge kernel); the
    result must be the same unique sorted output."""
    return request.param


@pytest.fixture(params=[0, 1, 2], ids=["shearsort", "tilemergesort", "longtiles"])
def base(request):
    """The base cases of bcf_sort (bcf_options.base_case): the paper's tile ShearSort, the tile mergesort
    network, long tiles."""
    return request.param


def dev(a):
    """numpy unsigned array -> CUDA tensor holding the same bit pattern."""
    if a is None:
        return None
    signed = {np.dtype(np.uint32): np.int32, np.dtype(np.uint64): np.int64}[a.dtype]
    return torch.from_numpy(np.ascontiguousarray(a).view(signed)).cuda()


def host(t, like):
    return t.cpu().numpy().view(like.dtype)


def make(kind, n, seed, dup=False):
    """(keys, vals) numpy arrays of element type `kind` in {'u32','u32u32','u64','u64u32'}."""
    rng = np.random.default_rng(seed)
    hi = 16 if dup else (1 << 32)
    if kind.startswith("u32"):
        keys = rng.integers(0, hi, size=n, dtype=np.uint64).astype(np.uint32)
    else:
        keys = rng.integers(0, hi, size=n, dtype=np.uint64)
        if not dup:
            keys = (keys << np.uint64(32)) | rng.integers(0, 1 << 32, size=n, dtype=np.uint64)
            keys[::7] &= np.uint64(0xFFFFFFFF)          # equal high words, order decided by the low word
    vals = None
    if kind.endswith("u32") and kind not in ("u32",):
        vals = rng.permutation(n).astype(np.uint32) if n else np.zeros(0, np.uint32)
    if n > 8:                                            # the padding value is a legal element (A10)
        keys[n // 3] = np.iinfo(keys.dtype).max
        if vals is not None:
            vals[n // 3] = 0xFFFFFFFF
    return keys, vals


KINDS = ["u32", "u32u32", "u64", "u64u32"]


def assert_same(got_k, got_v, want, vals):
    if vals is None:
        assert np.array_equal(got_k, want)
    else:
        assert np.array_equal(got_k, want[0])
        assert np.array_equal(got_v, want[1])


# ---------------------------------------------------------------- bcf_sort_tiles (a1-a4)


def test_sort_tiles_config1_exact(bcf):
    """BASELINE config 1 at full size: 1024 tiles of uint32, uniform."""
    keys = workloads.cfg1_tiles_u32()
    d = dev(keys)
    bcf.sort_tiles(d)
    assert np.array_equal(host(d, keys), oracle.shearsort_tiles(keys))


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("tiles", [1, 3, 4, 9, 130])
def test_sort_tiles_types_and_counts(bcf, kind, tiles):
    keys, vals = make(kind, tiles * 1024, seed=tiles, dup=(tiles == 9))
    if tiles >= 3:
        keys[1024:2048] = keys[1024]                                    # all-equal tile
        keys[2048:3072] = np.sort(keys[2048:3072])[::-1]                # reversed tile
    dk, dv = dev(keys), dev(vals)
    bcf.sort_tiles(dk, dv)
    want = oracle.shearsort_tiles(keys, vals)
    assert_same(host(dk, keys), None if vals is None else host(dv, vals), want, vals)


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("tiles", [1, 3, 4, 9, 130])
def test_sort_tiles_mergesort_types_and_counts(bcf, kind, tiles):
    """bcf_sort_tiles_mergesort: the same unique result as the ShearSort oracle on every element type."""
    keys, vals = make(kind, tiles * 1024, seed=100 + tiles, dup=(tiles == 9))
    if tiles >= 3:
        keys[1024:2048] = keys[1024]                                    # all-equal tile
        keys[2048:3072] = np.sort(keys[2048:3072])[::-1]                # reversed tile
    dk, dv = dev(keys), dev(vals)
    bcf.sort_tiles_mergesort(dk, dv)
    want = oracle.shearsort_tiles(keys, vals)
    assert_same(host(dk, keys), None if vals is None else host(dv, vals), want, vals)


def test_sort_tiles_mergesort_configs_1_and_2(bcf):
    keys = workloads.cfg1_tiles_u32()
    d = dev(keys)
    bcf.sort_tiles_mergesort(d)
    assert np.array_equal(host(d, keys), oracle.shearsort_tiles(keys))
    keys, vals = workloads.cfg2_tiles_u32_u32(num_tiles=256)
    dk, dv = dev(keys), dev(vals)
    bcf.sort_tiles_mergesort(dk, dv)
    wk, wv = oracle.shearsort_tiles(keys, vals)
    assert np.array_equal(host(dk, keys), wk) and np.array_equal(host(dv, vals), wv)


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("h", [2, 4, 8])
@pytest.mark.parametrize("groups", [1, 3, 37])
def test_sort_long_tiles_matches_oracle(bcf, kind, h, groups):
    """Long tiles h * w^2: every block of 1024 h elements sorted as one sequence;
    the oracle sorts each block with its own ShearSort + two-finger merge rounds."""
    m = 1024 * h
    keys, vals = make(kind, groups * m, seed=1000 * h + groups, dup=(groups == 3))
    if groups >= 3:
        keys[m:2 * m] = keys[m]                                         # all-equal long tile
        keys[2 * m:3 * m] = np.sort(keys[2 * m:3 * m])[::-1]            # reversed long tile
    dk, dv = dev(keys), dev(vals)
    bcf.sort_long_tiles(dk, h, dv)
    gk, gv = host(dk, keys), None if vals is None else host(dv, vals)
    for g in range(groups):
        sl = slice(g * m, (g + 1) * m)
        want = oracle.sort_full(keys[sl], None if vals is None else vals[sl])
        assert_same(gk[sl], None if vals is None else gv[sl], want, vals)


def test_sort_tiles_config2_shape(bcf):
    """Config 2 recipe (keys in [0,16), value = index) on 256 tiles; equals a stable sort by key."""
    keys, vals = workloads.cfg2_tiles_u32_u32(num_tiles=256)
    dk, dv = dev(keys), dev(vals)
    bcf.sort_tiles(dk, dv)
    wk, wv = oracle.shearsort_tiles(keys, vals)
    assert np.array_equal(host(dk, keys), wk) and np.array_equal(host(dv, vals), wv)


# ---------------------------------------------------------------- bcf_merge_partition (a5)


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("n,run_len", [(5000, 1024), (8192, 4096), (3000, 700), (4096, 2048), (2500, 3000)])
def test_merge_partition_matches_oracle_corank(bcf, kind, n, run_len):
    keys, vals = make(kind, n, seed=n + run_len, dup=True)
    if vals is None:
        keys = workloads.sorted_runs(keys, run_len)
    else:
        keys, vals = workloads.sorted_runs(keys, run_len, vals)
    splits = bcf.merge_partition(dev(keys), run_len, dev(vals)).cpu().numpy().view(np.uint32)
    spp = -(-2 * run_len // 1024)
    assert splits.size == bcf.num_shares(n, run_len)
    for j, got in enumerate(splits):
        pair, t = divmod(j, spp)
        a0 = pair * 2 * run_len
        a1 = min(n, a0 + run_len)
        b1 = min(n, a1 + run_len)
        d = min(t * 1024, b1 - a0)
        want = oracle.corank(keys[a0:a1], keys[a1:b1], d,
                             None if vals is None else vals[a0:a1], None if vals is None else vals[a1:b1])
        assert got == want, (j, got, want)


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("n,run_len,dup", [
    (4 * 4096, 4096, False), (4 * 4096, 4096, True), (70001, 4096, True), (3 * 8192 + 5, 8192, False),
    (100000, 16384, True), (8192 * 5 + 1, 8192, False), (1 << 17, 1 << 15, False), (9000, 4096, True),
])
def test_merge_partition4_matches_oracle_multiway_corank(bcf, kind, n, run_len, dup):
    """Row a5 for four-run passes: every share boundary's split equals the definition (first d outputs
    of the stable four-way merge), including short and missing runs in the last group."""
    keys, vals = make(kind, n, seed=n + run_len, dup=dup)
    if vals is None:
        keys = workloads.sorted_runs(keys, run_len)
    else:
        keys, vals = workloads.sorted_runs(keys, run_len, vals)
    got = bcf.merge_partition4(dev(keys), run_len, dev(vals)).cpu().numpy().view(np.uint32)
    assert got.shape == (-(-n // 8192) + 1, 4)
    for s in range(got.shape[0]):
        out0 = s * 8192
        g0 = out0 // (4 * run_len) * (4 * run_len)
        if g0 >= n:
            assert list(got[s]) == [0, 0, 0, 0]
            continue
        cuts = [min(n, g0 + r * run_len) for r in range(5)]
        rk = [keys[cuts[r]:cuts[r + 1]] for r in range(4)]
        rv = None if vals is None else [vals[cuts[r]:cuts[r + 1]] for r in range(4)]
        d = min(out0 - g0, cuts[4] - g0)
        assert list(got[s]) == oracle.corank_multi(rk, d, rv), (s, d)


# ---------------------------------------------------------------- bcf_merge_runs (a6, a8, a9)


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("n,run_len", [
    (2048, 1024), (8192, 1024), (5000, 1024), (10000, 2048), (4097, 4096), (3000, 700),
    (1 << 16, 1 << 12), (70001, 333), (1024, 1), (777, 1000), (1, 1), (2, 1), (40000, 20000), (40001, 13),
    (5 * 4096 + 7, 4096), (9 * 2048, 2048), (7 * 1024 + 1, 1024), (1 << 18, 1 << 13), (300001, 1024), (3 * 32768 - 5, 32768),
])
def test_merge_runs_matches_oracle(bcf, kind, n, run_len, rpp):
    keys, vals = make(kind, n, seed=3 * n + run_len, dup=(n % 2 == 1))
    if vals is None:
        keys = workloads.sorted_runs(keys, run_len)
    else:
        keys, vals = workloads.sorted_runs(keys, run_len, vals)
    dk, dv = dev(keys), dev(vals)
    out = bcf.merge_runs(dk, run_len, dv, opts={**RPP[rpp]})
    want = oracle.merge_runs(keys, run_len, vals)
    if vals is None:
        assert np.array_equal(host(out, keys), want)
    else:
        assert np.array_equal(host(out[0], keys), want[0]) and np.array_equal(host(out[1], vals), want[1])
    assert np.array_equal(host(dk, keys), keys)          # the input is not modified


@pytest.mark.parametrize("n,run_len", [(5_000_000, 1 << 13), ((1 << 22) + 777, 1 << 14), (1 << 23, 1 << 21)])
def test_four_run_passes_many_shares_per_cta(bcf, n, run_len, rpp):
    """More shares than SMs: every CTA of the persistent four-run kernels works through several shares, so the
    stage and X-Y buffers are refilled and every mbarrier runs through several phases (bcf_merge4s.cuh)."""
    keys = workloads.sorted_runs(make("u32", n, seed=n % 1000)[0], run_len)
    out = bcf.merge_runs(dev(keys), run_len, opts={**RPP[rpp]})
    assert np.array_equal(host(out, keys), oracle.merge_runs(keys, run_len))


@pytest.mark.parametrize("k", [2, 64, 1024])
def test_merge_runs_config5b_shape(bcf, k, rpp):
    keys, run_len = workloads.cfg5b_merge_runs_u32(k, n=1 << 18)
    out = bcf.merge_runs(dev(keys), run_len, opts={**RPP[rpp]})
    assert np.array_equal(host(out, keys), oracle.merge_runs(keys, run_len))


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("n,run_len", [(2048, 1024), (9000, 1024), (5000, 700), (1 << 15, 512), (3, 1), (40001, 5000)])
def test_merge_runs_pagewise_matches_oracle(bcf, kind, n, run_len):
    """Row a7 (Alg. 6 streaming form): same unique result as the oracle's merge rounds, and the
    oracle's own literal Alg. 6 on the first pair."""
    keys, vals = make(kind, n, seed=n ^ run_len, dup=(n % 2 == 0))
    if vals is None:
        keys = workloads.sorted_runs(keys, run_len)
    else:
        keys, vals = workloads.sorted_runs(keys, run_len, vals)
    out = bcf.merge_runs_pagewise(dev(keys), run_len, dev(vals))
    want = oracle.merge_runs(keys, run_len, vals)
    if vals is None:
        assert np.array_equal(host(out, keys), want)
    else:
        assert np.array_equal(host(out[0], keys), want[0]) and np.array_equal(host(out[1], vals), want[1])
    if n > 2 * run_len:   # one round only: compare with Alg. 6 itself on pair 0
        a, b = keys[:run_len], keys[run_len:2 * run_len]
        va = None if vals is None else vals[:run_len]
        vb = None if vals is None else vals[run_len:2 * run_len]
        one = bcf.merge_runs_pagewise(dev(np.concatenate([a, b])), run_len,
                                      None if vals is None else dev(np.concatenate([va, vb])))
        lit = oracle.binary_merge_pagewise(a, b, va, vb)
        if vals is None:
            assert np.array_equal(host(one, keys), lit)
        else:
            assert np.array_equal(host(one[0], keys), lit[0]) and np.array_equal(host(one[1], vals), lit[1])


# ---------------------------------------------------------------- bcf_sort (a1-a9)


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("n", [1, 2, 31, 1023, 1024, 1025, 2048, 5000, 3 * 1024 + 17, (1 << 16) + 17, 1 << 17,
                               4096, 4097, 8192, 8193, 16 * 1024 + 3, 40 * 1024, (1 << 18) + 4099, 600001])
def test_sort_matches_oracle(bcf, kind, n, rpp, base):
    keys, vals = make(kind, n, seed=n, dup=(n % 3 == 0))
    dk, dv = dev(keys), dev(vals)
    bcf.sort(dk, dv, opts={**RPP[rpp], "base_case": base})
    want = oracle.sort_full(keys, vals)
    assert_same(host(dk, keys), None if vals is None else host(dv, vals), want, vals)


@pytest.mark.parametrize("launch_mode", [1, 2], ids=["plain", "pdl"])
@pytest.mark.parametrize("n", [1 << 17, 300001])
def test_sort_launch_modes(bcf, n, rpp, launch_mode):
    """Ordinary and programmatic dependent launches (bcf_options.launch_mode) give the same result."""
    for kind in ("u32", "u64u32"):
        keys, vals = make(kind, n, seed=n + launch_mode)
        dk, dv = dev(keys), dev(vals)
        for _ in range(3):                                   # back-to-back calls on one stream
            dk.copy_(dev(keys))
            bcf.sort(dk, dv if vals is None else dv.copy_(dev(vals)), opts={**RPP[rpp], "launch_mode": launch_mode})
        want = oracle.sort_full(keys, vals)
        assert_same(host(dk, keys), None if vals is None else host(dv, vals), want, vals)


@pytest.mark.parametrize("dist", workloads.CFG4_VARIANTS)
def test_sort_config4_distributions(bcf, dist, rpp, base):
    keys = workloads.cfg4_sort_u32(dist, n=(1 << 18) + 1000)
    d = dev(keys)
    bcf.sort(d, opts={**RPP[rpp], "base_case": base})
    assert np.array_equal(host(d, keys), oracle.sort_full(keys))


def test_sort_config3_and_5a_shapes(bcf, rpp):
    keys = workloads.cfg3_sort_u32(n=1 << 19)
    d = dev(keys)
    bcf.sort(d, opts={**RPP[rpp]})
    assert np.array_equal(host(d, keys), oracle.sort_full(keys))
    k, v = workloads.cfg5a_sort_u64_u32(n=(1 << 18) + 3)
    dk, dv = dev(k), dev(v)
    bcf.sort(dk, dv, opts={**RPP[rpp]})
    wk, wv = oracle.sort_full(k, v)
    assert np.array_equal(host(dk, k), wk) and np.array_equal(host(dv, v), wv)


def test_sort_empty_is_noop(bcf):
    e = torch.empty(0, dtype=torch.int32, device="cuda")
    bcf.sort(e)
    bcf.sort_tiles(e)
    assert bcf.merge_runs(e, 4).numel() == 0


@pytest.mark.parametrize("kind,n", [("u64u32", 50000), ("u32", 700), ("u32", 1024), ("u32", 4 * 8192), ("u32", 4 * 8192 + 1),
                                    ("u32", 1234567), ("u32u32", 300001), ("u64", 99999)])
def test_sort_host_roundtrip(bcf, kind, n, rpp):
    """bcf_sort_host copies the input in chunks and sorts the tiles of a chunk on a second stream while the next chunk is
    copied (chunks are whole base-case runs; ragged last chunk, fewer elements than chunks, odd and even pass counts)."""
    keys, vals = make(kind, n, seed=1)
    signed = {np.dtype(np.uint32): np.int32, np.dtype(np.uint64): np.int64}[keys.dtype]
    hk = torch.from_numpy(keys.view(signed).copy()).pin_memory()
    hv = None if vals is None else torch.from_numpy(vals.view(np.int32).copy()).pin_memory()
    bcf.sort_host(hk, hv, opts={**RPP[rpp]})
    want = oracle.sort_full(keys, vals)
    assert_same(hk.numpy().view(keys.dtype), None if hv is None else hv.numpy().view(np.uint32), want, vals)


def test_sort_host_concurrent_calls_on_one_device_do_not_share_a_side_stream(bcf):
    """bcf_sort_host keeps its side stream and events per device between calls; calls that run at the same time (four
    threads, each with its own stream and scratch, several calls each) must each borrow a set of their own."""
    import threading
    jobs = []
    for i in range(4):
        keys, _ = make("u32", 200000 + 1111 * i, seed=40 + i)
        jobs.append((keys, torch.from_numpy(keys.view(np.int32).copy()).pin_memory(), torch.cuda.Stream(),
                     np.sort(keys)))
    errors = []

    def work(keys, hk, stream, want):
        try:
            for rep in range(6):
                hk.copy_(torch.from_numpy(keys.view(np.int32)))
                bcf.sort_host(hk, stream=stream)
                if not np.array_equal(hk.numpy().view(np.uint32), want):
                    errors.append("mismatch in repetition %d" % rep)
        except Exception as e:      # noqa: BLE001
            errors.append(repr(e))

    threads = [threading.Thread(target=work, args=j) for j in jobs]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors


# ---------------------------------------------------------------- error behaviour (include/bcf.h)


def test_error_codes(bcf):
    k = torch.zeros(4096, dtype=torch.int32, device="cuda")
    with pytest.raises(bcf.BcfError) as e:
        bcf.merge_runs(k, 0)
    assert e.value.name == "BCF_ERR_INVALID_ARG"
    with pytest.raises(bcf.BcfError) as e:
        bcf.merge_runs(k, 1024, out_keys=k)                       # in/out aliasing
    assert e.value.name == "BCF_ERR_INVALID_ARG"
    with pytest.raises(bcf.BcfError) as e:
        bcf.sort(k[1:])                                           # 4-byte aligned only
    assert e.value.name == "BCF_ERR_MISALIGNED"
    with pytest.raises(bcf.BcfError) as e:
        bcf.sort(k, workspace=torch.empty(64, dtype=torch.uint8, device="cuda"))
    assert e.value.name == "BCF_ERR_WORKSPACE_TOO_SMALL"
    with pytest.raises(ValueError):
        bcf.sort(k.cpu())                                         # no CPU path


# Local memory (stack) bytes per thread the build is allowed to have, by (kernel, key type, value type).
# makes "the data is not transferred to local memory" part of the method: every kernel must show 0 unless it is
# listed here with the exact byte count (DESIGN.md section 4 names each entry and why it is not a data spill).
LOCAL_BYTES_ALLOWED = {}      # none: every kernel of the build is at 0 bytes


def test_every_launched_kernel_uses_no_local_memory(bcf):
    """All 15 kernels x 4 element types (those that exist): cudaFuncGetAttributes().localSizeBytes == 0."""
    seen = 0
    for kid in bcf.KERNEL_IDS:
        for kt in (0, 1):
            for vt in (0, 1):
                try:
                    info = bcf.kernel_info(kid, kt, vt)
                except bcf.BcfError as e:
                    assert e.name == "BCF_ERR_INVALID_ARG"
                    assert ((kid == "merge4_pipe" and (kt, vt) == (1, 1)) or (kid == "merge_pieces" and vt == 1) or
                            (kid == "merge4_stream" and (kt, vt) != (0, 0))), (kid, kt, vt)
                    continue
                seen += 1
                assert info["local_bytes_per_thread"] == LOCAL_BYTES_ALLOWED.get((kid, kt, vt), 0), (kid, kt, vt, info)
                assert info["ctas_per_sm"] >= 1, (kid, kt, vt, info)
    assert seen == 15 * 4 - 1 - 2 - 3


def test_options_are_per_call_and_validated(bcf):
    """No process-wide settings: two option sets in alternation give their own pass structure every time."""
    keys, _ = make("u32", 1 << 17, seed=9)
    want = oracle.sort_full(keys)
    for i in range(4):
        o = {"rounds_per_pass": 1 + i % 2, "base_case": i % 3}
        bcf.launch_counts()
        d = dev(keys)
        bcf.sort(d, opts=o)
        torch.cuda.synchronize()
        launches = bcf.launch_counts()
        run = 8192 if o["base_case"] == 2 else 1024
        assert launches["merge"] == bcf.merge_pass_count(keys.size, run, "uint32", opts={"rounds_per_pass": o["rounds_per_pass"]})
        assert np.array_equal(host(d, keys), want)
    bad = bcf.options()
    bad.rounds_per_pass = 7
    with pytest.raises(bcf.BcfError) as e:
        bcf.sort(dev(keys), opts=bad)
    assert e.value.name == "BCF_ERR_INVALID_ARG"
    bad = bcf.options()
    bad.struct_size = 4
    with pytest.raises(bcf.BcfError):
        bcf.sort(dev(keys), opts=bad)


def test_a_failed_launch_is_reported_once_and_does_not_stick(bcf):
    """include/bcf.h ERRORS: a pending CUDA error of another library call is cleared on entry; the next call works."""
    k = torch.zeros(4096, dtype=torch.int32, device="cuda")
    try:
        torch.empty(1, device="cuda").new_empty((1 << 62,))       # a failing CUDA call (out of memory) in this thread
    except Exception:
        pass
    bcf.sort(k)                                                   # must not return BCF_ERR_CUDA because of it
    torch.cuda.synchronize()


def test_second_device_in_one_process(bcf):
    """Per-device caches (kernel attributes, SM count) are keyed by device id: sort on cuda:1 after cuda:0."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs 2 GPUs")
    keys, vals = make("u64u32", 70000, seed=4)
    want = oracle.sort_full(keys, vals)
    for d in (0, 1, 0):
        with torch.cuda.device(d):
            dk = torch.from_numpy(keys.view(np.int64)).to(f"cuda:{d}")
            dv = torch.from_numpy(vals.view(np.int32)).to(f"cuda:{d}")
            bcf.sort(dk, dv)
            assert np.array_equal(dk.cpu().numpy().view(np.uint64), want[0])


# ---------------------------------------------------------------- bcf_find_buckets


@pytest.mark.parametrize("kind", ["u32", "u64"])
@pytest.mark.parametrize("pb", [False, True])
@pytest.mark.parametrize("n,run_len,t,P,dup", [
    (64 * 1024, 4096, 16, 16, False), (64 * 1024, 4096, 16, 16, True), (100000, 7000, 5, 9, False),
    (1 << 18, 1 << 12, 64, 64, True), (1 << 18, 1 << 14, 128, 128, False), (5000, 1024, 3, 2, True), (300, 100, 1, 3, False),
])
def test_find_buckets_matches_oracle(bcf, kind, pb, n, run_len, t, P, dup):
    """Alg. 7 (and pivot buckets): pivots, piece offsets and the regrouped keys, exactly."""
    keys, _ = make(kind, n, seed=n + t + P, dup=dup)
    keys = workloads.sorted_runs(keys, run_len)
    out, piv, off = bcf.find_buckets(dev(keys), run_len, t, P, pivot_buckets=pb)
    O, F, Q = oracle.find_buckets(keys, run_len, t, P, pivot_buckets=pb)
    assert np.array_equal(host(piv, keys), F)
    assert np.array_equal(off.cpu().numpy().view(np.uint32).astype(np.int64), Q)
    assert np.array_equal(host(out, keys), O)


def test_find_buckets_pivot_buckets_sort_zero_one_data(bcf):
    """0-1 data is sorted by the distribution alone when pivots get their own buckets."""
    rng = np.random.default_rng(3)
    keys = workloads.sorted_runs(rng.integers(0, 2, size=1 << 20).astype(np.uint32), 1 << 14)
    out, _, _ = bcf.find_buckets(dev(keys), 1 << 14, 64, 64, pivot_buckets=True)
    assert np.array_equal(host(out, keys), np.sort(keys))


# ---------------------------------------------------------------- bcf_colored_prefix_sums


@pytest.mark.parametrize("layout", [0, 1], ids=["bank_per_thread", "thread_major"])
@pytest.mark.parametrize("n,d", [(1, 1), (15, 3), (511, 16), (512, 2), (513, 7), (4096 * 3 + 5, 16), (100000, 1),
                                 (1 << 20, 16), ((1 << 20) + 12345, 5), ((1 << 23) + 3, 11)])
def test_colored_prefix_sums_match_oracle(bcf, layout, n, d):
    """App. A: every output element, both shared-memory layouts, ragged sizes, 1..16 colours."""
    rng = np.random.default_rng(n + d)
    vals = rng.integers(0, 1 << 32, size=n, dtype=np.uint64).astype(np.uint32)
    cols = rng.integers(0, d, size=n).astype(np.uint8)
    if n > 2000:
        cols[100:1500] = d - 1                      # a long single-colour stretch
    out = bcf.colored_prefix_sums(dev(vals), torch.from_numpy(cols).cuda(), d, layout=layout)
    assert np.array_equal(host(out, vals), oracle.colored_prefix_sums(vals, cols, d))


@pytest.mark.parametrize("layout", [0, 1], ids=["bank_per_thread", "thread_major"])
def test_colored_prefix_sums_out_of_range_colour_is_clamped(bcf, layout):
    """include/bcf.h: a colour byte >= num_colors counts as colour num_colors - 1 and never touches another warp's sums."""
    n, d = 40000, 4
    rng = np.random.default_rng(5)
    vals = rng.integers(0, 1 << 32, size=n, dtype=np.uint64).astype(np.uint32)
    cols = rng.integers(0, 256, size=n).astype(np.uint8)
    out = bcf.colored_prefix_sums(dev(vals), torch.from_numpy(cols).cuda(), d, layout=layout)
    assert np.array_equal(host(out, vals), oracle.colored_prefix_sums(vals, np.minimum(cols, d - 1).astype(np.uint8), d))


# ---------------------------------------------------------------- bcf_sort_buckets / bcf_merge_pieces


@pytest.mark.parametrize("kind", ["u32", "u64"])
@pytest.mark.parametrize("pb", [False, True], ids=["plain", "pivot_buckets"])
@pytest.mark.parametrize("n,P,t,data", [
    (64 * 1024, 8, 8, "uniform"), (64 * 1024 + 777, 8, 8, "dup"), (300001, 16, 16, "uniform"), (1 << 18, 16, 4, "zero_one"),
    (1 << 18, 128, 128, "uniform"), (5000, 4, 4, "dup"), (1024, 4, 4, "uniform"), (200000, 3, 5, "dup256"), (1 << 20, 32, 32, "zero_one"),
])
def test_sort_buckets_matches_oracle(bcf, kind, pb, n, P, t, data, base):
    """BCFMergesort with FIND-BUCKETS and the bucket-local final merge phase (BCFMergesortPB with pivot buckets):
    the unique sorted output, element by element, against oracle.sort_full_buckets (PAPER.md 3.2, App. B)."""
    rng = np.random.default_rng(n + P + t)
    dt = np.uint32 if kind == "u32" else np.uint64
    if data == "uniform":
        keys = rng.integers(0, 1 << 32, size=n, dtype=np.uint64).astype(dt)
        if kind == "u64":
            keys = (keys << np.uint64(32)) | rng.integers(0, 1 << 32, size=n, dtype=np.uint64)
    elif data == "dup":
        keys = rng.integers(0, 16, size=n).astype(dt)
    elif data == "dup256":
        keys = rng.integers(0, 1 << 32, size=256, dtype=np.uint64).astype(dt)[rng.integers(0, 256, size=n)]
    else:
        keys = rng.integers(0, 2, size=n).astype(dt)
    keys[n // 3] = np.iinfo(dt).max                              # the padding value is a legal key (A10)
    d = dev(keys)
    bcf.sort_buckets(d, P, t=t, pivot_buckets=pb, opts={"base_case": base})
    want = oracle.sort_full_buckets(keys, P, t=t, pivot_buckets=pb) if n <= (1 << 18) else np.sort(keys)
    assert np.array_equal(host(d, keys), want)


@pytest.mark.parametrize("kind,P,n", [("u32", 2048, 2047 * 1024 - 5), ("u64", 2048, 2047 * 1024 - 5), ("u32", 1024, 1023 * 1024 + 1)])
@pytest.mark.parametrize("pb", [False, True], ids=["plain", "pivot_buckets"])
def test_sort_buckets_few_samples_stays_inside_its_workspace(bcf, kind, P, n, pb, base):
    """t = 1 with a large P: the s <= P runs left by the first merge phase give fewer than P samples, so the call
    raises t to ceil(P / s).  The workspace is exactly bcf_sort_buckets_workspace_bytes(n, t = 1, ...) followed by a
    guard region; the output is the unique sorted sequence (vs numpy's sort) and the guard is untouched."""
    dt = np.uint32 if kind == "u32" else np.uint64
    rng = np.random.default_rng(n + P)
    keys = rng.integers(0, 1 << 32, size=n, dtype=np.uint64).astype(dt)
    if kind == "u64":
        keys = (keys << np.uint64(32)) | rng.integers(0, 1 << 32, size=n, dtype=np.uint64)
    need = int(bcf.lib().bcf_sort_buckets_workspace_bytes(n, 1, P, int(pb), 0 if kind == "u32" else 1))
    guard = 64 << 20
    buf = torch.full((need + guard,), 0xA5, dtype=torch.uint8, device="cuda")
    d = dev(keys)
    bcf.sort_buckets(d, P, t=1, pivot_buckets=pb, workspace=buf[:need], opts={"base_case": base})
    assert np.array_equal(host(d, keys), np.sort(keys))
    assert bool((buf[need:] == 0xA5).all())


def test_sort_buckets_bucket_starts_match_oracle_and_lemma_1(bcf):
    """The distribution inside bcf_sort_buckets is the oracle's (same runs, same pivots): bucket starts equal,
    and with all keys distinct no bucket exceeds Lemma 1's bound s ceil(N/(s t)) + ceil(s t/P) ceil(N/(s t))."""
    n, P, t = 1 << 18, 16, 16
    keys = np.random.default_rng(1).permutation(1 << 20)[:n].astype(np.uint32)
    d = dev(keys)
    _, starts = bcf.sort_buckets(d, P, t=t, opts={"base_case": 1}, return_bucket_starts=True)
    out, info = oracle.sort_full_buckets(keys, P, t=t, return_info=True)
    assert np.array_equal(host(d, keys), out)
    got = starts.cpu().numpy().astype(np.int64)
    assert np.array_equal(np.diff(got), np.array(info["bucket_sizes"]))
    s = info["s"]
    per = -(-n // (s * t))
    assert np.diff(got).max() <= s * per + (-(-(s * t) // P)) * per


@pytest.mark.parametrize("kind", ["u32", "u64"])
@pytest.mark.parametrize("groups,s,copy_odd", [(1, 2, False), (5, 3, False), (7, 8, True), (3, 1, False), (16, 16, False), (9, 5, True)])
def test_merge_pieces_matches_oracle(bcf, kind, groups, s, copy_odd):
    """The final merge phase alone: ragged, empty and page-spanning pieces; pivot buckets (odd groups) are copied."""
    rng = np.random.default_rng(groups * 100 + s)
    dt = np.uint32 if kind == "u32" else np.uint64
    lens = rng.choice([0, 1, 5, 31, 700, 1024, 1500, 3000], size=groups * s)
    offs = np.concatenate([[0], np.cumsum(lens)]).astype(np.int64)
    n = int(offs[-1])
    if n == 0:
        pytest.skip("empty draw")
    keys = np.empty(n, dtype=dt)
    want = np.empty(n, dtype=dt)
    for g in range(groups):
        lo, hi = offs[g * s], offs[(g + 1) * s]
        if copy_odd and g % 2 == 1:
            keys[lo:hi] = dt(rng.integers(0, 1000))              # a pivot bucket: copies of one key
        else:
            for r in range(s):
                a, b = offs[g * s + r], offs[g * s + r + 1]
                keys[a:b] = np.sort(rng.integers(0, 50 if g % 3 == 0 else 1 << 31, size=b - a).astype(dt))
        merged, _ = oracle.merge_pieces([keys[offs[g * s + r]:offs[g * s + r + 1]] for r in range(s)])
        want[lo:hi] = merged
    out = bcf.merge_pieces(dev(keys), torch.from_numpy(offs.astype(np.int32)).cuda(), groups, s, copy_odd_groups=copy_odd)
    assert np.array_equal(host(out, keys), want)


# ---------------------------------------------------------------- debug: conflict-isolation variants


@pytest.mark.parametrize("exclusive", [True, False])
def test_isolated_experiment_kernels_match_oracle(bcf, exclusive):
    """The phase-separated kernels of the bank-conflict experiment compute what the production kernels compute."""
    keys, _ = make("u32", 37 * 1024, seed=5)
    d = dev(keys)
    bcf.debug_sort_tiles_isolated(d, exclusive=exclusive)
    assert np.array_equal(host(d, keys), oracle.shearsort_tiles(keys))
    n, L = 1 << 17, 1 << 14
    keys, _ = make("u32", n, seed=6, dup=not exclusive)
    keys = workloads.sorted_runs(keys, L)
    out = bcf.debug_merge_round_isolated(dev(keys), L, exclusive=exclusive)
    assert np.array_equal(host(out, keys), oracle.merge_round(keys, L))


def test_sort_is_deterministic_under_repetition(bcf):
    """compute-sanitizer is closed on this pool (profiles/r2_sanitizer.md): a race in the hand-rolled barriers would show
    as a run-to-run difference.  20 repetitions per option set on sizes that exercise every kernel; all bit-identical
    and equal to the oracle."""
    for kind, n in (("u32", (1 << 18) + 4099), ("u64u32", 70001)):
        keys, vals = make(kind, n, seed=77, dup=True)
        want = oracle.sort_full(keys, vals)
        for o in ({"rounds_per_pass": 1, "base_case": 2}, {"rounds_per_pass": 2, "base_case": 2, "launch_mode": 2},
                  {"rounds_per_pass": 2, "base_case": 1}, {"rounds_per_pass": 1, "base_case": 0, "merge_impl": 1}):
            for rep in range(20):
                dk, dv = dev(keys), dev(vals)
                bcf.sort(dk, dv, opts=o)
                assert_same(host(dk, keys), None if vals is None else host(dv, vals), want, vals)


@pytest.mark.parametrize("kind,logn", [("u32", 24), ("u32u32", 23), ("u64u32", 23)])
def test_persistent_merge_kernels_are_deterministic_over_many_shares(bcf, kind, logn):
    """Every CTA of the persistent merge kernels works through several shares here, so their stage buffers are
    refilled and their mbarriers run through many phases (a warp that waits on a phase it did not take part in --
    bcf_merge_pipe.cuh, Cfg -- showed as an illegal address about once in ten sorts of 2^28 keys).  60 repetitions
    per pass structure: equal to the library sort of numpy the first time, bit-identical afterwards."""
    n = (1 << logn) + 12345
    keys, vals = make(kind, n, seed=logn)
    src_k, src_v = dev(keys), dev(vals)
    for o in (RPP[1], RPP[2], RPP[3], RPP[4]):      # RPP[4]: partition launches that search the page samples first
        ref = None
        for rep in range(60 if o is not RPP[4] else 10):
            dk, dv = src_k.clone(), None if src_v is None else src_v.clone()
            bcf.sort(dk, dv, opts=o)
            if ref is None:
                ref = (dk, dv)
                order = np.lexsort((vals, keys)) if vals is not None else np.argsort(keys, kind="stable")
                assert np.array_equal(host(dk, keys), keys[order])
                if vals is not None:
                    assert np.array_equal(host(dv, vals), vals[order])
            else:
                assert torch.equal(dk, ref[0]) and (dv is None or torch.equal(dv, ref[1])), (kind, o, rep)

