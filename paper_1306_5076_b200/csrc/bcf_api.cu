// bcf_api.cu -- the C ABI of include/bcf.h: argument validation, workspace carving, the merge-round
// driver and the measurement hooks.  Every step of the path runs in the
// kernels (one translation unit per kernel family, bcf_tu_*.cu); there is no CPU fallback.
#include "bcf_internal.cuh"

#include <cstdio>
#include <cstring>
#include <initializer_list>
#include <mutex>

using namespace bcf;

namespace bcf {

int &last_cuda_error_ref()
{
    thread_local int e = 0;
    return e;
}

}  // namespace bcf

namespace {

// Largest split-point array any round of merging runs of `run_len` needs.
size_t max_shares(size_t n, size_t run_len)
{
    size_t m = 0;
    for (size_t l = run_len; l < n; l *= 2) {
        const PassGeom g = pass_geom(n, l);
        if (g.num_shares > m) m = g.num_shares;
    }
    return m;
}

// ------------------------------------------------------------------ per-device state (keyed by device id)

struct DevCache {
    std::atomic<int> state{0};   // 0 unknown, 1 supported, 2 unsupported
    int num_sms = 0;
};
DevCache g_dev[MAX_DEVICES];

// The current device: clears a stale pending error, checks compute capability 10.x once per device.
bcf_status current_device(Dev *d)
{
    (void)cudaGetLastError();
    int dev = -1;
    BCF_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return BCF_ERR_UNSUPPORTED_DEVICE;
    DevCache &c = g_dev[dev];
    int st = c.state.load(std::memory_order_acquire);
    if (st == 0) {
        int major = 0, sms = 0;
        BCF_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
        BCF_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
        c.num_sms = sms;
        st = (major == 10) ? 1 : 2;
        c.state.store(st, std::memory_order_release);
    }
    if (st != 1) return BCF_ERR_UNSUPPORTED_DEVICE;
    d->id = dev;
    d->num_sms = c.num_sms;
    return BCF_OK;
}

// ------------------------------------------------------------------ per-call options (bcf_options)

#ifndef BCF_DEFAULT_ROUNDS_PER_PASS
#define BCF_DEFAULT_ROUNDS_PER_PASS 1
#endif
// BCF_LAUNCH_AUTO = programmatic dependent launches at every size.  Measured on B200: they hide
// the launch latency between the ~2 launches of every merge round, which is 27 % of a 2^20-key sort, 11 % of a
// 2^24-key sort and still 1 % at 2^28 keys (6.89 against 6.95 ms; r2).

bool resolve_options(const bcf_options *o, Opt *r)
{
    *r = Opt();
    r->rounds_per_pass = BCF_DEFAULT_ROUNDS_PER_PASS;
    if (!o) return true;
    if (o->struct_size < sizeof(bcf_options)) return false;
    if (o->base_case < BCF_BASE_SHEARSORT || o->base_case > BCF_BASE_AUTO) return false;
    if (o->rounds_per_pass < 0 || o->rounds_per_pass > 2) return false;
    if (o->merge_impl < BCF_MERGE_IMPL_AUTO || o->merge_impl > BCF_MERGE_IMPL_PARTITION_LAUNCH) return false;
    if (o->launch_mode < BCF_LAUNCH_AUTO || o->launch_mode > BCF_LAUNCH_PDL) return false;
    r->base_case = o->base_case;
    if (o->rounds_per_pass) r->rounds_per_pass = o->rounds_per_pass;
    r->generic_merge = o->merge_impl == BCF_MERGE_IMPL_GENERIC;
    r->merge4_barrier = o->merge_impl == BCF_MERGE_IMPL_BARRIER4;
    r->no_self_partition = o->merge_impl == BCF_MERGE_IMPL_PARTITION_LAUNCH;
    if (o->partition_warp_search_max >= 0) r->warp_search_max = static_cast<unsigned long long>(o->partition_warp_search_max);
    r->launch_mode = o->launch_mode;
    return true;
}

// launch mode of a call that works on n elements
inline void resolve_launch_mode(Opt *o, size_t n)
{
    (void)n;
    o->pdl = o->launch_mode != BCF_LAUNCH_PLAIN;
}

bool overlap(const void *a, size_t an, const void *b, size_t bn)
{
    if (!a || !b || !an || !bn) return false;
    const uintptr_t x = reinterpret_cast<uintptr_t>(a), y = reinterpret_cast<uintptr_t>(b);
    return x < y + bn && y < x + an;
}

// ------------------------------------------------------------------ profiling (bcf_profile_*)

// One event per launch, recorded just before it; a launch ends where the next one of the same API call
// begins, and the last one where the call's closing event (ProfileGroup) is recorded.  One event between
// two kernels instead of two halves what the instrumentation costs the timed region.
constexpr int PROFILE_POOL = 8192;
struct Profile {
    bool on = false;
    int used = 0;
    cudaEvent_t ev[PROFILE_POOL];
    int cls[PROFILE_POOL];             // kernel class of the launch that starts at ev[i]; -1: closing event
    int created = 0;
    int open_since = -1;               // first entry of the API call in progress
    unsigned long long dropped = 0;    // launches not timed because the pool was full
    // launch counts are kept whether or not timing is on, by every thread that launches: relaxed atomics.
    // Everything else in this struct is touched only while timing is on (one thread, include/bcf.h).
    std::atomic<unsigned long long> launches[BCF_KERNEL_CLASSES];
} g_prof;

inline int profile_mark(int cls, cudaStream_t s)
{
    if (!g_prof.on) return -1;
    if (g_prof.used >= PROFILE_POOL) { g_prof.dropped++; return -1; }
    const int idx = g_prof.used++;
    if (idx >= g_prof.created) {
        cudaEventCreate(&g_prof.ev[idx]);
        g_prof.created = idx + 1;
    }
    g_prof.cls[idx] = cls;
    cudaEventRecord(g_prof.ev[idx], s);
    return idx;
}

}  // namespace

void bcf::profile_launch(int cls, cudaStream_t stream)
{
    g_prof.launches[cls].fetch_add(1, std::memory_order_relaxed);
    profile_mark(cls, stream);
}

namespace {

// Closes the timed launches of one public API call (outermost scope only).
struct ProfileGroup {
    cudaStream_t s;
    bool outer;
    explicit ProfileGroup(cudaStream_t stream) : s(stream), outer(g_prof.on && g_prof.open_since < 0)
    {
        if (outer) g_prof.open_since = g_prof.used;
    }
    ~ProfileGroup()
    {
        if (!outer) return;              // timing off: concurrent callers share no state here
        if (g_prof.used > g_prof.open_since && g_prof.cls[g_prof.used - 1] >= 0) profile_mark(-1, s);
        g_prof.open_since = -1;
    }
};

// ------------------------------------------------------------------ launch helpers of the driver

// Power-of-two multiples of the tile size take the pipelined kernel (bcf_merge_pipe.cuh).
inline bool pipe_eligible(size_t run_len, const Opt &o)
{
    if (run_len % TILE) return false;
    const size_t r = run_len / TILE;
    if (r & (r - 1)) return false;
    return !o.generic_merge;
}

// Element types whose two stage buffers of a four-run share fit one SM (bcf_merge4.cuh).
template <class E>
inline bool merge4_eligible(size_t run_len, const Opt &o)
{
    return merge4_fits<E>() && pipe_eligible(run_len, o) && o.rounds_per_pass == 2;
}

// Dispatch a templated callable on the runtime element type.
#define BCF_DISPATCH(kt, vt, CALL)                                                   \
    do {                                                                             \
        if ((kt) == BCF_KEY_U32 && (vt) == BCF_VAL_NONE) { using E = Elem<1, false>; CALL; } \
        else if ((kt) == BCF_KEY_U32) { using E = Elem<1, true>; CALL; }             \
        else if ((vt) == BCF_VAL_NONE) { using E = Elem<2, false>; CALL; }           \
        else { using E = Elem<2, true>; CALL; }                                      \
    } while (0)

struct Workspace {
    void *keys;
    uint32_t *vals;
    uint32_t *splits;
    PageSamples samples;     // page heads / tails between merge rounds (bcf_internal.cuh)
    size_t bytes;
};

// Carve [keys copy][vals copy][splits] out of a workspace; any of the three can be empty.
Workspace carve(void *base, size_t n, bcf_key_t kt, bcf_val_t vt, bool with_data, size_t shares)
{
    Workspace w;
    size_t off = 0;
    char *b = static_cast<char *>(base);
    w.keys = b ? b + off : nullptr;
    if (with_data) off += align_up(n * key_bytes(kt), 256);
    w.vals = reinterpret_cast<uint32_t *>(b ? b + off : nullptr);
    if (with_data && vt == BCF_VAL_U32) off += align_up(n * 4, 256);
    w.splits = reinterpret_cast<uint32_t *>(b ? b + off : nullptr);
    off += align_up((shares + 1) * 4 + 64, 256);   // + room for the uint4 entries of a four-run pass
#ifndef BCF_NO_PAGE_SAMPLES                          // A/B only
    if (shares) {                                  // two samples per page of 1024 elements
        const size_t pages = n / TILE + 1;
        w.samples.keys = b ? b + off : nullptr;
        off += align_up(2 * pages * key_bytes(kt), 256);
        if (vt == BCF_VAL_U32) {
            w.samples.vals = reinterpret_cast<uint32_t *>(b ? b + off : nullptr);
            off += align_up(2 * pages * 4, 256);
        }
    }
#endif
    w.bytes = off;
    return w;
}

// The passes of the merging phase from sorted runs of run_len up to runs of at least
// `stop_len`: ways[i] = 2 is one merge round per read + write of the data (Lemma 2), ways[i] = 4 two rounds
// per read + write (bcf_merge4.cuh).  An odd number of remaining rounds is made even by a two-way pass first.
constexpr int MAX_PASSES = 40;
template <class E>
int plan_passes(size_t n, size_t run_len, size_t stop_len, const Opt &o, int *ways)
{
    int np = 0;
    const size_t target = stop_len < n ? stop_len : n;
    for (size_t l = run_len; l < target && np < MAX_PASSES; ++np) {
        const int remaining = ceil_log2((target + l - 1) / l);
        const bool four = remaining % 2 == 0 && merge4_eligible<E>(l, o);
        ways[np] = four ? 4 : 2;
        l *= four ? 4 : 2;
    }
    return np;
}

int count_passes(size_t n, size_t run_len, size_t stop_len, bcf_key_t kt, bcf_val_t vt, const Opt &o)
{
    int ways[MAX_PASSES];
    int np = 0;
    BCF_DISPATCH(kt, vt, np = plan_passes<E>(n, run_len, stop_len, o, ways));
    return np;
}

// Pass i writes to dst[i]; each pass is one read + one write of all n elements.
template <class E>
bcf_status merge_rounds(const Call &c, const void *k0, const uint32_t *v0, void *ka, uint32_t *va, void *kb, uint32_t *vb,
                        bool first_to_a, size_t n, size_t run_len, size_t stop_len, uint32_t *splits, const PageSamples &samples)
{
    bool samples_valid = false;          // `samples` describes ksrc (the previous pass was a pipelined two-run round)
    const void *ksrc = k0;
    const uint32_t *vsrc = v0;
    bool to_a = first_to_a;
    int ways[MAX_PASSES];
    const int np = plan_passes<E>(n, run_len, stop_len, c.opt, ways);
    size_t l = run_len;
    for (int i = 0; i < np; ++i) {
        void *kd = to_a ? ka : kb;
        uint32_t *vd = to_a ? va : vb;
        bcf_status st;
        if (ways[i] == 4) {
            st = launch_merge4<E>(c, ksrc, vsrc, kd, vd, splits, n, l);
            samples_valid = false;
        } else if (pipe_eligible(l, c.opt)) {
            st = launch_merge_pipe<E>(c, ksrc, vsrc, kd, vd, splits, n, l, samples_valid ? samples : PageSamples(), samples);
            samples_valid = samples.keys != nullptr && E::NP < 3;      // the three-plane kernel writes none (bcf_merge_pipe.cuh)
        } else {
            samples_valid = false;
            const PassGeom g = pass_geom(n, l);
            st = launch_partition<E>(c, ksrc, vsrc, splits, g);
            if (st != BCF_OK) return st;
            st = launch_merge<E>(c, ksrc, vsrc, kd, vd, splits, g);
        }
        if (st != BCF_OK) return st;
        ksrc = kd;
        vsrc = vd;
        to_a = !to_a;
        l *= ways[i];
    }
    return BCF_OK;
}

template <class E>
bcf_status pagewise_rounds(const Call &c, const void *k0, const uint32_t *v0, void *ka, uint32_t *va, void *kb, uint32_t *vb,
                           bool first_to_a, size_t n, size_t run_len)
{
    const void *ksrc = k0;
    const uint32_t *vsrc = v0;
    bool to_a = first_to_a;
    for (size_t l = run_len; l < n; l *= 2) {
        void *kd = to_a ? ka : kb;
        uint32_t *vd = to_a ? va : vb;
        bcf_status st = launch_pagewise<E>(c, ksrc, vsrc, kd, vd, n, l);
        if (st != BCF_OK) return st;
        ksrc = kd;
        vsrc = vd;
        to_a = !to_a;
    }
    return BCF_OK;
}

bcf_status merge_runs_common(bool pagewise, const void *d_keys_in, const void *d_vals_in, void *d_keys_out,
                             void *d_vals_out, size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt,
                             void *d_workspace, size_t workspace_bytes, cudaStream_t s, const bcf_options *options)
{
    Call c;
    c.s = s;
    if (!valid_types(kt, vt) || !resolve_options(options, &c.opt)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32) || run_len == 0) return BCF_ERR_INVALID_ARG;
    if (!d_keys_in || !d_keys_out) return BCF_ERR_INVALID_ARG;
    if ((vt == BCF_VAL_U32) != (d_vals_in != nullptr) || (vt == BCF_VAL_U32) != (d_vals_out != nullptr))
        return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys_in) || !aligned16(d_keys_out) || !aligned16(d_vals_in) || !aligned16(d_vals_out) ||
        !aligned16(d_workspace))
        return BCF_ERR_MISALIGNED;
    const size_t kb = n * key_bytes(kt), vb = (vt == BCF_VAL_U32) ? n * 4 : 0;
    if (overlap(d_keys_in, kb, d_keys_out, kb) || overlap(d_vals_in, vb, d_vals_out, vb) ||
        overlap(d_keys_in, kb, d_vals_out, vb) || overlap(d_vals_in, vb, d_keys_out, kb))
        return BCF_ERR_INVALID_ARG;
    const size_t need = bcf_workspace_bytes(pagewise ? BCF_OP_MERGE_PAGEWISE : BCF_OP_MERGE_RUNS, n, run_len, kt, vt);
    if (need && (!d_workspace || workspace_bytes < need)) return BCF_ERR_WORKSPACE_TOO_SMALL;
    if (overlap(d_workspace, need, d_keys_in, kb) || overlap(d_workspace, need, d_keys_out, kb) ||
        overlap(d_workspace, need, d_vals_in, vb) || overlap(d_workspace, need, d_vals_out, vb))
        return BCF_ERR_INVALID_ARG;
    bcf_status st = current_device(&c.dev);
    if (st != BCF_OK) return st;
    resolve_launch_mode(&c.opt, n);
    ProfileGroup profile_group(s);

    const size_t runs = (n + run_len - 1) / run_len;
    const int rounds = ceil_log2(runs);
    if (rounds == 0) {   // a single run: the result is the input
        BCF_CUDA(cudaMemcpyAsync(d_keys_out, d_keys_in, kb, cudaMemcpyDeviceToDevice, s));
        if (vb) BCF_CUDA(cudaMemcpyAsync(d_vals_out, d_vals_in, vb, cudaMemcpyDeviceToDevice, s));
        return BCF_OK;
    }
    // pass i (1-based) writes to `out` when (passes - i) is even, so the last pass lands in out.
    const int passes = pagewise ? rounds : count_passes(n, run_len, n, kt, vt, c.opt);
    const Workspace w = carve(d_workspace, n, kt, vt, rounds >= 2, pagewise ? 0 : max_shares(n, run_len));
    const bool first_to_out = ((passes - 1) % 2 == 0);
    if (pagewise) {
        BCF_DISPATCH(kt, vt, st = pagewise_rounds<E>(c, d_keys_in, static_cast<const uint32_t *>(d_vals_in), d_keys_out,
                                                     static_cast<uint32_t *>(d_vals_out), w.keys, w.vals, first_to_out,
                                                     n, run_len));
    } else {
        BCF_DISPATCH(kt, vt, st = merge_rounds<E>(c, d_keys_in, static_cast<const uint32_t *>(d_vals_in), d_keys_out,
                                                  static_cast<uint32_t *>(d_vals_out), w.keys, w.vals, first_to_out, n,
                                                  run_len, n, w.splits, w.samples));
    }
    return st;
}

// base case of bcf_sort under `o` for an element type: the network and the length of the runs it leaves
void resolve_base_case(const Opt &o, bcf_key_t kt, bcf_val_t vt, int *bc, size_t *base_run)
{
    // AUTO: what measures fastest on B200 -- long tiles for 4-byte keys alone, the tile mergesort otherwise
    *bc = o.base_case;
    if (*bc == BCF_BASE_AUTO) *bc = (kt == BCF_KEY_U32 && vt == BCF_VAL_NONE) ? BCF_BASE_LONG_TILES : BCF_BASE_TILE_MERGESORT;
    *base_run = (*bc == BCF_BASE_LONG_TILES) ? size_t(BCF_LONG_TILE_H) * TILE : size_t(TILE);
}

// Base case + merge passes until runs of at least stop_len (stop_len >= n: the whole sort), in place: the
// result is in d_keys / d_vals.  Validation is the caller's.  The two phases are separate functions so that
// bcf_sort_host can run the base case chunk by chunk under the host-to-device copy.
struct SortPlan {
    int bc;                  // base case network
    size_t base_run;         // length of the runs it leaves
    int passes;              // merge passes after it
    Workspace w;
    void *k0;                // where the base case writes: with an odd number of merge passes the workspace, so that the
    uint32_t *v0;            // last pass lands in the caller's buffer without an extra copy
    bool base_to_ws;
};

SortPlan sort_plan(const Call &c, void *d_keys, void *d_vals, size_t n, size_t stop_len, bcf_key_t kt, bcf_val_t vt, void *d_workspace)
{
    SortPlan p;
    resolve_base_case(c.opt, kt, vt, &p.bc, &p.base_run);
    p.passes = n > p.base_run ? count_passes(n, p.base_run, stop_len, kt, vt, c.opt) : 0;
    p.w = carve(d_workspace, n, kt, vt, n > TILE, n > TILE ? max_shares(n, TILE) : 0);
    p.base_to_ws = (p.passes % 2 == 1);
    p.k0 = p.base_to_ws ? p.w.keys : d_keys;
    p.v0 = p.base_to_ws ? p.w.vals : static_cast<uint32_t *>(d_vals);
    return p;
}

// base case of elements [first, first + count) (first a multiple of the base run length)
bcf_status sort_base_case(const Call &c, const SortPlan &p, void *d_keys, void *d_vals, size_t first, size_t count, bcf_key_t kt,
                          bcf_val_t vt)
{
    const size_t kb = key_bytes(kt);
    const void *kin = static_cast<const char *>(d_keys) + first * kb;
    const uint32_t *vin = d_vals ? static_cast<const uint32_t *>(d_vals) + first : nullptr;
    void *kout = static_cast<char *>(p.k0) + first * kb;
    uint32_t *vout = p.v0 ? p.v0 + first : nullptr;
    bcf_status st;
    if (p.bc == BCF_BASE_LONG_TILES)
        BCF_DISPATCH(kt, vt, st = launch_long_tile<E>(c, kin, vin, kout, vout, count, BCF_LONG_TILE_H));
    else
        BCF_DISPATCH(kt, vt, st = launch_tile_sort<E>(c, kin, vin, kout, vout, count, p.bc));
    return st;
}

bcf_status sort_merge_phase(const Call &c, const SortPlan &p, void *d_keys, void *d_vals, size_t n, size_t stop_len, bcf_key_t kt,
                            bcf_val_t vt)
{
    if (p.passes == 0) return BCF_OK;
    bcf_status st;
    // pass 1 writes to the buffer the base case did not write.
    BCF_DISPATCH(kt, vt, st = merge_rounds<E>(c, p.k0, p.v0, d_keys, static_cast<uint32_t *>(d_vals), p.w.keys, p.w.vals,
                                              /*first_to_a=*/p.base_to_ws, n, p.base_run, stop_len, p.w.splits, p.w.samples));
    return st;
}

bcf_status sort_phases(const Call &c, void *d_keys, void *d_vals, size_t n, size_t stop_len, bcf_key_t kt, bcf_val_t vt,
                       void *d_workspace)
{
    const SortPlan p = sort_plan(c, d_keys, d_vals, n, stop_len, kt, vt, d_workspace);
    const bcf_status st = sort_base_case(c, p, d_keys, d_vals, 0, n, kt, vt);
    if (st != BCF_OK) return st;
    return sort_merge_phase(c, p, d_keys, d_vals, n, stop_len, kt, vt);
}

// Side stream + events of a bcf_sort_host call.  They are kept per device between calls instead of being created and
// destroyed every time (a stream and six events cost tens of microseconds: nothing against the copies of a large sort,
// most of the call for a small one).  A call borrows one set and hands it back when it returns; two calls that run at
// the same time on one device each get a set of their own (created on demand).  Sets are never destroyed.
struct HostOverlap {
#ifndef BCF_HOST_CHUNKS
#define BCF_HOST_CHUNKS 4      // measured on 2^28 u32 keys: 1 chunk 47.8 ms, 4: 45.3, 8: 46.3, 16: 46.0
#endif
    static constexpr int CHUNKS = BCF_HOST_CHUNKS;
    cudaStream_t side = nullptr;
    cudaEvent_t ev[CHUNKS + 1] = {};
    cudaEvent_t done = nullptr;
    HostOverlap *next_free = nullptr;
    bcf_status init()
    {
        BCF_CUDA(cudaStreamCreateWithFlags(&side, cudaStreamNonBlocking));
        for (auto &e : ev) BCF_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        BCF_CUDA(cudaEventCreateWithFlags(&done, cudaEventDisableTiming));
        return BCF_OK;
    }
};
std::mutex g_overlap_mutex;
HostOverlap *g_overlap_free[MAX_DEVICES] = {};

struct OverlapLease {
    HostOverlap *o = nullptr;
    int dev = -1;
    bool finished = false;          // the call synchronised its stream after the side stream's last work
    bcf_status acquire(int device)
    {
        dev = device;
        {
            std::lock_guard<std::mutex> lock(g_overlap_mutex);
            o = g_overlap_free[dev];
            if (o) g_overlap_free[dev] = o->next_free;
        }
        if (o) return BCF_OK;
        o = new HostOverlap();
        const bcf_status st = o->init();
        if (st != BCF_OK) { o = nullptr; }      // a half-made set is abandoned (process-lifetime objects anyway)
        return st;
    }
    ~OverlapLease()
    {
        if (!o) return;
        if (!finished) cudaStreamSynchronize(o->side);     // error path: nothing of this call may still run on it
        std::lock_guard<std::mutex> lock(g_overlap_mutex);
        o->next_free = g_overlap_free[dev];
        g_overlap_free[dev] = o;
    }
};

bcf_status validate_sort(const void *d_keys, const void *d_vals, size_t n, bcf_key_t kt, bcf_val_t vt, const void *d_workspace,
                         size_t workspace_bytes)
{
    if (n >= (size_t(1) << 32)) return BCF_ERR_INVALID_ARG;
    if (!d_keys || (vt == BCF_VAL_U32) != (d_vals != nullptr)) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys) || !aligned16(d_vals) || !aligned16(d_workspace)) return BCF_ERR_MISALIGNED;
    const size_t need = bcf_workspace_bytes(BCF_OP_SORT, n, 0, kt, vt);
    if (need && (!d_workspace || workspace_bytes < need)) return BCF_ERR_WORKSPACE_TOO_SMALL;
    const size_t kb = n * key_bytes(kt), vb = (vt == BCF_VAL_U32) ? n * 4 : 0;
    if (overlap(d_workspace, need, d_keys, kb) || overlap(d_workspace, need, d_vals, vb)) return BCF_ERR_INVALID_ARG;
    return BCF_OK;
}

// ------------------------------------------------------------------ FIND-BUCKETS and the final merge phase

bool buckets_geom(size_t n, size_t run_len, int t, int P, int pivot_buckets, BucketsGeom *g)
{
    if (n == 0 || n >= (size_t(1) << 32) || run_len == 0 || t < 1 || P < 2) return false;
    const size_t s = (n + run_len - 1) / run_len;
    if (s > 65536 || (size_t)t > 65536 || (size_t)P > 65536 || s * (size_t)t < (size_t)P) return false;
    g->n = n; g->run_len = run_len;
    g->s = (unsigned)s; g->t = (unsigned)t; g->P = (unsigned)P;
    g->pb = pivot_buckets ? 1 : 0;
    g->nb = pivot_buckets ? 2u * P - 1u : (unsigned)P;
    return (size_t)g->nb * s < (size_t(1) << 26);
}

bcf_status find_buckets_impl(const Call &c, const void *d_keys_in, const BucketsGeom &g, bcf_key_t kt, void *d_keys_out,
                             void *d_pivots, uint32_t *d_piece_offsets, void *d_workspace)
{
    const size_t ns = (size_t)g.s * g.t;
    char *ws = static_cast<char *>(d_workspace);
    void *samples = ws;
    uint32_t *bounds = reinterpret_cast<uint32_t *>(ws + align_up(ns * key_bytes(kt), 256));
    char *sort_ws = reinterpret_cast<char *>(bounds) + align_up((size_t)g.s * (g.nb + 1) * 4, 256);
    bcf_status st = launch_buckets_sample(c, d_keys_in, samples, g, kt);                      // Alg. 7
    if (st != BCF_OK) return st;
    st = sort_phases(c, samples, nullptr, ns, ns, kt, BCF_VAL_NONE, sort_ws);                  // MERGESORT(S), L505
    if (st != BCF_OK) return st;
    return launch_buckets_distribute(c, d_keys_in, samples, d_pivots, bounds, d_piece_offsets, d_keys_out, g, kt);
}

// pairs of the first round of the final merge phase (the round with the most pairs)
inline size_t pieces_max_pairs(size_t groups, size_t s) { return groups * ((s + 1) / 2); }

// Every kernel the library can launch, by bcf_kernel_id (each translation unit knows its own).
template <class E>
bool kernel_desc(int id, bcf_key_t kt, KernelDesc *k)
{
    if (kernel_desc_tile<E>(id, k) || kernel_desc_long<E>(id, k) || kernel_desc_merge<E>(id, k) || kernel_desc_pipe<E>(id, k) ||
        kernel_desc_merge4<E>(id, k))
        return true;
    if constexpr (!E::HAS_VAL) return kernel_desc_pieces(id, kt, k);
    return false;
}

}  // namespace

// ====================================================================== exported C ABI

extern "C" {

const char *bcf_status_string(bcf_status s)
{
    switch (s) {
    case BCF_OK: return "BCF_OK";
    case BCF_ERR_INVALID_ARG: return "BCF_ERR_INVALID_ARG";
    case BCF_ERR_MISALIGNED: return "BCF_ERR_MISALIGNED";
    case BCF_ERR_WORKSPACE_TOO_SMALL: return "BCF_ERR_WORKSPACE_TOO_SMALL";
    case BCF_ERR_UNSUPPORTED_DEVICE: return "BCF_ERR_UNSUPPORTED_DEVICE";
    case BCF_ERR_CUDA: return "BCF_ERR_CUDA";
    case BCF_ERR_TOO_LARGE: return "BCF_ERR_TOO_LARGE";
    }
    return "BCF_ERR_UNKNOWN";
}

const char *bcf_version(void) { return "bcf 0.3 (sm_100a)"; }

bcf_status bcf_options_init(bcf_options *opt)
{
    if (!opt) return BCF_ERR_INVALID_ARG;
    opt->struct_size = sizeof(bcf_options);
    opt->base_case = BCF_BASE_AUTO;
    opt->rounds_per_pass = 0;
    opt->merge_impl = BCF_MERGE_IMPL_AUTO;
    opt->partition_warp_search_max = -1;
    opt->launch_mode = BCF_LAUNCH_AUTO;
    return BCF_OK;
}

int bcf_last_cuda_error(void) { return last_cuda_error_ref(); }

size_t bcf_workspace_bytes(int op, size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt)
{
    if (!valid_types(kt, vt) || n == 0) return 0;
    switch (op) {
    case BCF_OP_SORT_TILES:
        return 0;
    case BCF_OP_MERGE_RUNS: {
        if (run_len == 0) return 0;
        const int rounds = ceil_log2((n + run_len - 1) / run_len);
        if (rounds == 0) return 0;
        return carve(nullptr, n, kt, vt, rounds >= 2, max_shares(n, run_len)).bytes;   // whatever the options
    }
    case BCF_OP_MERGE_PAGEWISE: {
        if (run_len == 0) return 0;
        const int rounds = ceil_log2((n + run_len - 1) / run_len);
        if (rounds < 2) return 0;
        return carve(nullptr, n, kt, vt, true, 0).bytes;
    }
    case BCF_OP_SORT:
        if (n <= TILE) return 0;
        return carve(nullptr, n, kt, vt, true, max_shares(n, TILE)).bytes;
    case BCF_OP_SORT_HOST: {
        size_t data = align_up(n * key_bytes(kt), 256) + (vt == BCF_VAL_U32 ? align_up(n * 4, 256) : 0);
        return data + bcf_workspace_bytes(BCF_OP_SORT, n, 0, kt, vt);
    }
    }
    return 0;
}

static bcf_status sort_tiles_common(void *d_keys, void *d_vals, size_t num_tiles, bcf_key_t kt, bcf_val_t vt, bcf_stream_t stream,
                                    int algo)
{
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
    if (num_tiles == 0) return BCF_OK;
    if (num_tiles >= (size_t(1) << 22)) return BCF_ERR_INVALID_ARG;
    if (!d_keys || (vt == BCF_VAL_U32) != (d_vals != nullptr)) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys) || !aligned16(d_vals)) return BCF_ERR_MISALIGNED;
    Call c;
    c.s = stream;
    resolve_options(nullptr, &c.opt);
    bcf_status st = current_device(&c.dev);
    if (st != BCF_OK) return st;
    ProfileGroup profile_group(stream);
    BCF_DISPATCH(kt, vt, st = launch_tile_sort<E>(c, d_keys, static_cast<uint32_t *>(d_vals), d_keys,
                                                  static_cast<uint32_t *>(d_vals), num_tiles * TILE, algo));
    return st;
}

bcf_status bcf_sort_tiles(void *d_keys, void *d_vals, size_t num_tiles, bcf_key_t kt, bcf_val_t vt, bcf_stream_t stream)
{
    return sort_tiles_common(d_keys, d_vals, num_tiles, kt, vt, stream, BCF_BASE_SHEARSORT);
}

bcf_status bcf_sort_tiles_mergesort(void *d_keys, void *d_vals, size_t num_tiles, bcf_key_t kt, bcf_val_t vt,
                                    bcf_stream_t stream)
{
    return sort_tiles_common(d_keys, d_vals, num_tiles, kt, vt, stream, BCF_BASE_TILE_MERGESORT);
}

bcf_status bcf_sort_long_tiles(void *d_keys, void *d_vals, size_t num_long_tiles, int h, bcf_key_t kt, bcf_val_t vt,
                               bcf_stream_t stream)
{
    if (!valid_types(kt, vt) || (h != 2 && h != 4 && h != 8)) return BCF_ERR_INVALID_ARG;
    if (num_long_tiles == 0) return BCF_OK;
    if (num_long_tiles * h >= (size_t(1) << 22)) return BCF_ERR_INVALID_ARG;
    if (!d_keys || (vt == BCF_VAL_U32) != (d_vals != nullptr)) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys) || !aligned16(d_vals)) return BCF_ERR_MISALIGNED;
    Call c;
    c.s = stream;
    resolve_options(nullptr, &c.opt);
    bcf_status st = current_device(&c.dev);
    if (st != BCF_OK) return st;
    ProfileGroup profile_group(stream);
    BCF_DISPATCH(kt, vt, st = launch_long_tile<E>(c, d_keys, static_cast<uint32_t *>(d_vals), d_keys, static_cast<uint32_t *>(d_vals),
                                                  num_long_tiles * h * TILE, h));
    return st;
}

bcf_status bcf_merge_partition(const void *d_keys_in, const void *d_vals_in, size_t n, size_t run_len, bcf_key_t kt,
                               bcf_val_t vt, uint32_t *d_splits, size_t num_shares, bcf_stream_t stream)
{
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32) || run_len == 0) return BCF_ERR_INVALID_ARG;
    if (!d_keys_in || !d_splits || (vt == BCF_VAL_U32) != (d_vals_in != nullptr)) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys_in) || !aligned16(d_vals_in)) return BCF_ERR_MISALIGNED;
    const PassGeom g = pass_geom(n, run_len);
    if (num_shares != g.num_shares) return BCF_ERR_INVALID_ARG;
    Call c;
    c.s = stream;
    resolve_options(nullptr, &c.opt);
    bcf_status st = current_device(&c.dev);
    if (st != BCF_OK) return st;
    ProfileGroup profile_group(stream);
    BCF_DISPATCH(kt, vt, st = launch_partition<E>(c, d_keys_in, static_cast<const uint32_t *>(d_vals_in), d_splits, g));
    return st;
}

bcf_status bcf_merge_partition4(const void *d_keys_in, const void *d_vals_in, size_t n, size_t run_len, bcf_key_t kt,
                                bcf_val_t vt, uint32_t *d_splits, size_t num_bounds, bcf_stream_t stream)
{
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32) || run_len == 0) return BCF_ERR_INVALID_ARG;
    if (!d_keys_in || !d_splits || (vt == BCF_VAL_U32) != (d_vals_in != nullptr)) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys_in) || !aligned16(d_vals_in) || !aligned16(d_splits)) return BCF_ERR_MISALIGNED;
    if (num_bounds != (n + BCF_SHARE - 1) / BCF_SHARE + 1) return BCF_ERR_INVALID_ARG;
    Call c;
    c.s = stream;
    resolve_options(nullptr, &c.opt);
    bcf_status st = current_device(&c.dev);
    if (st != BCF_OK) return st;
    ProfileGroup profile_group(stream);
    BCF_DISPATCH(kt, vt, st = launch_partition4<E>(c, d_keys_in, static_cast<const uint32_t *>(d_vals_in), d_splits, n, run_len,
                                                   num_bounds));
    return st;
}

// ------------------------------------------------------------------ FIND-BUCKETS (Alg. 7)

size_t bcf_find_buckets_workspace_bytes(size_t n, size_t run_len, int t, int P, int pivot_buckets, bcf_key_t kt)
{
    BucketsGeom g;
    if (!valid_types(kt, BCF_VAL_NONE) || !buckets_geom(n, run_len, t, P, pivot_buckets, &g)) return 0;
    const size_t st = (size_t)g.s * g.t;
    return align_up(st * key_bytes(kt), 256) + align_up((size_t)g.s * (g.nb + 1) * 4, 256) +
           align_up(bcf_workspace_bytes(BCF_OP_SORT, st, 0, kt, BCF_VAL_NONE), 256) + 256;
}

bcf_status bcf_find_buckets(const void *d_keys_in, size_t n, size_t run_len, int t, int P, int pivot_buckets, bcf_key_t kt,
                            void *d_keys_out, void *d_pivots, uint32_t *d_piece_offsets, void *d_workspace,
                            size_t workspace_bytes, bcf_stream_t stream)
{
    if (!valid_types(kt, BCF_VAL_NONE)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    BucketsGeom g;
    if (!buckets_geom(n, run_len, t, P, pivot_buckets, &g)) return BCF_ERR_INVALID_ARG;
    if (!d_keys_in || !d_keys_out || !d_pivots || !d_piece_offsets || !d_workspace) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys_in) || !aligned16(d_keys_out) || !aligned16(d_workspace)) return BCF_ERR_MISALIGNED;
    const size_t kb = n * key_bytes(kt);
    if (overlap(d_keys_in, kb, d_keys_out, kb)) return BCF_ERR_INVALID_ARG;
    const size_t need = bcf_find_buckets_workspace_bytes(n, run_len, t, P, pivot_buckets, kt);
    if (workspace_bytes < need) return BCF_ERR_WORKSPACE_TOO_SMALL;
    if (overlap(d_workspace, need, d_keys_in, kb) || overlap(d_workspace, need, d_keys_out, kb)) return BCF_ERR_INVALID_ARG;
    Call c;
    c.s = stream;
    resolve_options(nullptr, &c.opt);
    bcf_status st = current_device(&c.dev);
    if (st != BCF_OK) return st;
    ProfileGroup profile_group(stream);
    return find_buckets_impl(c, d_keys_in, g, kt, d_keys_out, d_pivots, d_piece_offsets, d_workspace);
}

// ------------------------------------------------------------------ final merge phase, BCFMergesort(PB) end to end

size_t bcf_merge_pieces_workspace_bytes(size_t n, size_t groups, size_t s, bcf_key_t kt)
{
    if (!valid_types(kt, BCF_VAL_NONE) || n == 0 || groups == 0 || s == 0) return 0;
    const size_t tmp = ceil_log2(s) >= 2 ? align_up(n * key_bytes(kt), 256) : 0;
    return tmp + align_up((pieces_max_pairs(groups, s) + 1) * 4, 256);
}

bcf_status bcf_merge_pieces(const void *d_keys_in, void *d_keys_out, size_t n, const uint32_t *d_piece_offsets, size_t groups,
                            size_t s, int copy_odd_groups, bcf_key_t kt, void *d_workspace, size_t workspace_bytes,
                            bcf_stream_t stream)
{
    if (!valid_types(kt, BCF_VAL_NONE)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32) || groups == 0 || s == 0 || s > 65536 || groups * s >= (size_t(1) << 26)) return BCF_ERR_INVALID_ARG;
    if (!d_keys_in || !d_keys_out || !d_piece_offsets || !d_workspace) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys_in) || !aligned16(d_keys_out) || !aligned16(d_workspace)) return BCF_ERR_MISALIGNED;
    const size_t kb = n * key_bytes(kt);
    const size_t need = bcf_merge_pieces_workspace_bytes(n, groups, s, kt);
    if (workspace_bytes < need) return BCF_ERR_WORKSPACE_TOO_SMALL;
    if (overlap(d_keys_in, kb, d_keys_out, kb) || overlap(d_workspace, need, d_keys_in, kb) ||
        overlap(d_workspace, need, d_keys_out, kb))
        return BCF_ERR_INVALID_ARG;
    Call c;
    c.s = stream;
    resolve_options(nullptr, &c.opt);
    bcf_status st = current_device(&c.dev);
    if (st != BCF_OK) return st;
    ProfileGroup profile_group(stream);
    if (s == 1) {
        BCF_CUDA(cudaMemcpyAsync(d_keys_out, d_keys_in, kb, cudaMemcpyDeviceToDevice, stream));
        return BCF_OK;
    }
    char *ws = static_cast<char *>(d_workspace);
    void *tmp = ws;
    uint32_t *first = reinterpret_cast<uint32_t *>(ws + (ceil_log2(s) >= 2 ? align_up(kb, 256) : 0));
    return launch_merge_pieces_rounds(c, d_keys_in, d_keys_out, tmp, n, d_piece_offsets, groups, s, copy_odd_groups, first, kt);
}

// run length at which the first merge phase is suspended: the first base_run * 2^r that leaves at most P runs
static size_t buckets_stop_len(size_t n, size_t base_run, int P)
{
    size_t l = base_run;
    while ((n + l - 1) / l > static_cast<size_t>(P)) l *= 2;
    return l;
}

// Samples per run the distribution really takes on runs of stop_len: the caller's t, raised to ceil(P / s) where
// s t < P (Alg. 7 needs at least P samples to choose P - 1 pivots from).  The workspace is sized with the same value.
static int buckets_samples_per_run(size_t n, size_t stop_len, int t, int P)
{
    const size_t s = (n + stop_len - 1) / stop_len;
    if (s * static_cast<size_t>(t) >= static_cast<size_t>(P)) return t;
    return static_cast<int>((static_cast<size_t>(P) + s - 1) / s);
}

// [keys copy W1][piece offsets][pivots][max(sort workspace, FIND-BUCKETS workspace, final-phase workspace)]
struct BucketsWs {
    size_t w1, offsets, pivots, rest, total;
};
static BucketsWs buckets_ws(size_t n, int t, int P, int pb, bcf_key_t kt)
{
    BucketsWs w;
    const size_t kb = align_up(n * key_bytes(kt), 256);
    const size_t nb = pb ? 2 * size_t(P) - 1 : size_t(P);
    w.w1 = 0;
    w.offsets = kb;
    w.pivots = w.offsets + align_up((nb * size_t(P) + 1) * 4, 256);
    w.rest = w.pivots + align_up(size_t(P) * key_bytes(kt), 256);
    size_t rest = bcf_workspace_bytes(BCF_OP_SORT, n, 0, kt, BCF_VAL_NONE);
    // the distribution runs on s <= P runs of any of the run lengths a base case can leave
    size_t fb = 0;
    for (size_t base : {size_t(TILE), size_t(BCF_LONG_TILE_H) * TILE}) {
        const size_t l = buckets_stop_len(n, base, P);
        const size_t v = bcf_find_buckets_workspace_bytes(n, l, buckets_samples_per_run(n, l, t, P), P, pb, kt);
        if (v > fb) fb = v;
    }
    if (fb > rest) rest = fb;
    const size_t mp = bcf_merge_pieces_workspace_bytes(n, nb, size_t(P), kt);
    if (mp > rest) rest = mp;
    w.total = w.rest + align_up(rest, 256);
    return w;
}

size_t bcf_sort_buckets_workspace_bytes(size_t n, int t, int P, int pivot_buckets, bcf_key_t kt)
{
    if (!valid_types(kt, BCF_VAL_NONE) || n == 0 || n >= (size_t(1) << 32) || t < 1 || t > 65536 || P < 2 || P > 65536) return 0;
    return buckets_ws(n, t, P, pivot_buckets, kt).total;
}

bcf_status bcf_sort_buckets(void *d_keys, size_t n, bcf_key_t kt, int t, int P, int pivot_buckets, uint32_t *d_bucket_starts,
                            void *d_workspace, size_t workspace_bytes, bcf_stream_t stream, const bcf_options *options)
{
    Call c;
    c.s = stream;
    if (!valid_types(kt, BCF_VAL_NONE) || !resolve_options(options, &c.opt)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32) || t < 1 || t > 65536 || P < 2 || P > 65536) return BCF_ERR_INVALID_ARG;
    if (!d_keys || !d_workspace) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys) || !aligned16(d_workspace)) return BCF_ERR_MISALIGNED;
    const BucketsWs w = buckets_ws(n, t, P, pivot_buckets, kt);
    if (workspace_bytes < w.total) return BCF_ERR_WORKSPACE_TOO_SMALL;
    const size_t kb = n * key_bytes(kt);
    if (overlap(d_workspace, w.total, d_keys, kb)) return BCF_ERR_INVALID_ARG;
    bcf_status st = current_device(&c.dev);
    if (st != BCF_OK) return st;
    resolve_launch_mode(&c.opt, n);
    ProfileGroup profile_group(stream);

    char *ws = static_cast<char *>(d_workspace);
    void *w1 = ws + w.w1;
    uint32_t *offsets = reinterpret_cast<uint32_t *>(ws + w.offsets);
    void *pivots = ws + w.pivots;
    void *rest = ws + w.rest;

    // phases 1 + 2: base case, merge rounds while more than P runs remain (result in d_keys).  The sort
    // workspace of these phases is [W1 = the ping-pong copy][..]: carve() puts its keys copy first.
    int bc;
    size_t base_run;
    resolve_base_case(c.opt, kt, BCF_VAL_NONE, &bc, &base_run);
    const size_t stop_len = buckets_stop_len(n, base_run, P);
    // the sort's own workspace layout (keys copy + splits) needs bcf_workspace_bytes(SORT) contiguous bytes:
    // W1 followed by the offsets / pivots / rest regions covers it (they are written only after these phases)
    st = sort_phases(c, d_keys, nullptr, n, stop_len, kt, BCF_VAL_NONE, d_workspace);
    if (st != BCF_OK) return st;
    const size_t s = (n + stop_len - 1) / stop_len;
    if (s <= 1) return BCF_OK;

    // phase 3: FIND-BUCKETS  d_keys -> W1
    BucketsGeom g;
    const int tt = buckets_samples_per_run(n, stop_len, t, P);                                           // s t >= P
    if (!buckets_geom(n, stop_len, tt, P, pivot_buckets, &g)) return BCF_ERR_INVALID_ARG;
    if (bcf_find_buckets_workspace_bytes(n, stop_len, tt, P, pivot_buckets, kt) > w.total - w.rest)
        return BCF_ERR_WORKSPACE_TOO_SMALL;      // cannot happen while buckets_ws sizes `rest` with the same tt
    st = find_buckets_impl(c, d_keys, g, kt, w1, pivots, offsets, rest);
    if (st != BCF_OK) return st;
    if (d_bucket_starts)
        BCF_CUDA(cudaMemcpy2DAsync(d_bucket_starts, 4, offsets, s * 4, 4, g.nb + 1, cudaMemcpyDeviceToDevice, stream));

    // phase 4: the final merge phase inside the buckets  W1 -> d_keys
    char *r = static_cast<char *>(rest);
    const int rounds = ceil_log2(s);
    void *tmp = r;
    uint32_t *first = reinterpret_cast<uint32_t *>(r + (rounds >= 2 ? align_up(kb, 256) : 0));
    return launch_merge_pieces_rounds(c, w1, d_keys, tmp, n, offsets, g.nb, s, pivot_buckets ? 1 : 0, first, kt);
}

// ------------------------------------------------------------------ coloured prefix sums (App. A)

size_t bcf_colored_prefix_sums_workspace_bytes(size_t n)
{
    if (n == 0) return 0;
    return colored_scan_workspace_bytes(n);
}

bcf_status bcf_colored_prefix_sums(const uint32_t *d_values, const uint8_t *d_colors, size_t n, int num_colors, int layout,
                                   uint32_t *d_out, void *d_workspace, size_t workspace_bytes, bcf_stream_t stream)
{
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32) || num_colors < 1 || num_colors > colored_scan_max_colors()) return BCF_ERR_INVALID_ARG;
    if (layout != BCF_SCAN_BANK_PER_THREAD && layout != BCF_SCAN_THREAD_MAJOR) return BCF_ERR_INVALID_ARG;
    if (!d_values || !d_colors || !d_out || !d_workspace) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_values) || !aligned16(d_colors) || !aligned16(d_out) || !aligned16(d_workspace)) return BCF_ERR_MISALIGNED;
    if (overlap(d_out, n * 4, d_values, n * 4) || overlap(d_out, n * 4, d_colors, n)) return BCF_ERR_INVALID_ARG;
    if (workspace_bytes < bcf_colored_prefix_sums_workspace_bytes(n)) return BCF_ERR_WORKSPACE_TOO_SMALL;
    Call c;
    c.s = stream;
    resolve_options(nullptr, &c.opt);
    const bcf_status st = current_device(&c.dev);
    if (st != BCF_OK) return st;
    ProfileGroup profile_group(stream);
    return launch_colored_scan(c, d_values, d_colors, n, num_colors, layout == BCF_SCAN_BANK_PER_THREAD,
                               static_cast<uint32_t *>(d_workspace), d_out);
}

int bcf_merge_pass_count(size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt, const bcf_options *options)
{
    Opt o;
    if (!valid_types(kt, vt) || n == 0 || run_len == 0 || !resolve_options(options, &o)) return 0;
    return count_passes(n, run_len, n, kt, vt, o);
}

bcf_status bcf_merge_runs_ex(const void *d_keys_in, const void *d_vals_in, void *d_keys_out, void *d_vals_out, size_t n,
                             size_t run_len, bcf_key_t kt, bcf_val_t vt, void *d_workspace, size_t workspace_bytes,
                             bcf_stream_t stream, const bcf_options *opt)
{
    return merge_runs_common(false, d_keys_in, d_vals_in, d_keys_out, d_vals_out, n, run_len, kt, vt, d_workspace,
                             workspace_bytes, stream, opt);
}

bcf_status bcf_merge_runs(const void *d_keys_in, const void *d_vals_in, void *d_keys_out, void *d_vals_out, size_t n,
                          size_t run_len, bcf_key_t kt, bcf_val_t vt, void *d_workspace, size_t workspace_bytes,
                          bcf_stream_t stream)
{
    return merge_runs_common(false, d_keys_in, d_vals_in, d_keys_out, d_vals_out, n, run_len, kt, vt, d_workspace,
                             workspace_bytes, stream, nullptr);
}

bcf_status bcf_merge_runs_pagewise(const void *d_keys_in, const void *d_vals_in, void *d_keys_out, void *d_vals_out,
                                   size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt, void *d_workspace,
                                   size_t workspace_bytes, bcf_stream_t stream)
{
    return merge_runs_common(true, d_keys_in, d_vals_in, d_keys_out, d_vals_out, n, run_len, kt, vt, d_workspace,
                             workspace_bytes, stream, nullptr);
}

bcf_status bcf_sort_ex(void *d_keys, void *d_vals, size_t n, bcf_key_t kt, bcf_val_t vt, void *d_workspace,
                       size_t workspace_bytes, bcf_stream_t stream, const bcf_options *options)
{
    Call c;
    c.s = stream;
    if (!valid_types(kt, vt) || !resolve_options(options, &c.opt)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    bcf_status st = validate_sort(d_keys, d_vals, n, kt, vt, d_workspace, workspace_bytes);
    if (st != BCF_OK) return st;
    if ((st = current_device(&c.dev)) != BCF_OK) return st;
    resolve_launch_mode(&c.opt, n);
    ProfileGroup profile_group(stream);
    return sort_phases(c, d_keys, d_vals, n, n, kt, vt, d_workspace);
}

bcf_status bcf_sort(void *d_keys, void *d_vals, size_t n, bcf_key_t kt, bcf_val_t vt, void *d_workspace,
                    size_t workspace_bytes, bcf_stream_t stream)
{
    return bcf_sort_ex(d_keys, d_vals, n, kt, vt, d_workspace, workspace_bytes, stream, nullptr);
}

bcf_status bcf_sort_host_ex(void *h_keys, void *h_vals, size_t n, bcf_key_t kt, bcf_val_t vt, void *d_scratch,
                            size_t scratch_bytes, bcf_stream_t stream, const bcf_options *options)
{
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32)) return BCF_ERR_INVALID_ARG;
    if (!h_keys || (vt == BCF_VAL_U32) != (h_vals != nullptr)) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_scratch)) return BCF_ERR_MISALIGNED;
    const size_t need = bcf_workspace_bytes(BCF_OP_SORT_HOST, n, 0, kt, vt);
    if (!d_scratch || scratch_bytes < need) return BCF_ERR_WORKSPACE_TOO_SMALL;
    (void)cudaGetLastError();
    const size_t kb = n * key_bytes(kt), vb = (vt == BCF_VAL_U32) ? n * 4 : 0;
    char *base = static_cast<char *>(d_scratch);
    void *dk = base;
    void *dv = vb ? base + align_up(kb, 256) : nullptr;
    const size_t data = align_up(kb, 256) + (vb ? align_up(vb, 256) : 0);
    Call c;
    c.s = stream;
    if (!resolve_options(options, &c.opt)) return BCF_ERR_INVALID_ARG;
    bcf_status st = current_device(&c.dev);
    if (st != BCF_OK) return st;
    resolve_launch_mode(&c.opt, n);
    if (n <= TILE) {
        BCF_CUDA(cudaMemcpyAsync(dk, h_keys, kb, cudaMemcpyHostToDevice, stream));
        if (vb) BCF_CUDA(cudaMemcpyAsync(dv, h_vals, vb, cudaMemcpyHostToDevice, stream));
        st = bcf_sort_ex(dk, dv, n, kt, vt, base + data, scratch_bytes - data, stream, options);
        if (st != BCF_OK) return st;
    } else {
        // The base case works on independent tiles, so it runs chunk by chunk on a second stream while the next
        // chunk is still being copied: only the last chunk's base case is left on the critical path.  The merge
        // rounds need all the data and follow on the caller's stream.
        ProfileGroup profile_group(stream);
        const SortPlan p = sort_plan(c, dk, dv, n, n, kt, vt, base + data);
        OverlapLease lease;
        if ((st = lease.acquire(c.dev.id)) != BCF_OK) return st;
        HostOverlap &ov = *lease.o;
        Call side = c;
        side.s = ov.side;
        const size_t unit = p.base_run;
        const size_t chunk = (n / HostOverlap::CHUNKS + unit - 1) / unit * unit;
        int i = 0;
        for (size_t first = 0; first < n; first += chunk, ++i) {
            const size_t count = n - first < chunk ? n - first : chunk;
            BCF_CUDA(cudaMemcpyAsync(static_cast<char *>(dk) + first * key_bytes(kt), static_cast<const char *>(h_keys) + first * key_bytes(kt),
                                     count * key_bytes(kt), cudaMemcpyHostToDevice, stream));
            if (vb)
                BCF_CUDA(cudaMemcpyAsync(static_cast<uint32_t *>(dv) + first, static_cast<const uint32_t *>(h_vals) + first, count * 4,
                                         cudaMemcpyHostToDevice, stream));
            BCF_CUDA(cudaEventRecord(ov.ev[i], stream));
            BCF_CUDA(cudaStreamWaitEvent(ov.side, ov.ev[i], 0));
            if ((st = sort_base_case(side, p, dk, dv, first, count, kt, vt)) != BCF_OK) return st;
        }
        BCF_CUDA(cudaEventRecord(ov.done, ov.side));
        BCF_CUDA(cudaStreamWaitEvent(stream, ov.done, 0));
        if ((st = sort_merge_phase(c, p, dk, dv, n, n, kt, vt)) != BCF_OK) return st;
        BCF_CUDA(cudaMemcpyAsync(h_keys, dk, kb, cudaMemcpyDeviceToHost, stream));
        if (vb) BCF_CUDA(cudaMemcpyAsync(h_vals, dv, vb, cudaMemcpyDeviceToHost, stream));
        BCF_CUDA(cudaStreamSynchronize(stream));      // `stream` waited for the side stream: both are idle now
        lease.finished = true;
        return BCF_OK;
    }
    BCF_CUDA(cudaMemcpyAsync(h_keys, dk, kb, cudaMemcpyDeviceToHost, stream));
    if (vb) BCF_CUDA(cudaMemcpyAsync(h_vals, dv, vb, cudaMemcpyDeviceToHost, stream));
    BCF_CUDA(cudaStreamSynchronize(stream));
    return BCF_OK;
}

bcf_status bcf_sort_host(void *h_keys, void *h_vals, size_t n, bcf_key_t kt, bcf_val_t vt, void *d_scratch,
                         size_t scratch_bytes, bcf_stream_t stream)
{
    return bcf_sort_host_ex(h_keys, h_vals, n, kt, vt, d_scratch, scratch_bytes, stream, nullptr);
}

// ------------------------------------------------------------------ bank-conflict isolation experiment (debug)

bcf_status bcf_debug_merge_round_isolated(const void *d_keys_in, void *d_keys_out, size_t n, size_t run_len, int exclusive,
                                          void *d_workspace, size_t workspace_bytes, bcf_stream_t stream)
{
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32) || run_len < isolated_share() || (run_len & (run_len - 1)) || n % (2 * run_len)) return BCF_ERR_INVALID_ARG;
    if (!d_keys_in || !d_keys_out || !d_workspace) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys_in) || !aligned16(d_keys_out) || !aligned16(d_workspace)) return BCF_ERR_MISALIGNED;
    if (overlap(d_keys_in, n * 4, d_keys_out, n * 4)) return BCF_ERR_INVALID_ARG;
    if (workspace_bytes < (n / BCF_SHARE + 1) * 4) return BCF_ERR_WORKSPACE_TOO_SMALL;
    Call c;
    c.s = stream;
    resolve_options(nullptr, &c.opt);
    bcf_status st = current_device(&c.dev);
    if (st != BCF_OK) return st;
    ProfileGroup profile_group(stream);
    uint32_t *splits = static_cast<uint32_t *>(d_workspace);
    st = launch_partition_share<E_U32>(c, d_keys_in, nullptr, splits, n, run_len, isolated_share(), nullptr, nullptr);
    if (st != BCF_OK) return st;
    return launch_isolated_merge_round(c, static_cast<const uint32_t *>(d_keys_in), static_cast<uint32_t *>(d_keys_out), splits, n,
                                       run_len, exclusive);
}

bcf_status bcf_debug_sort_tiles_isolated(void *d_keys, size_t num_tiles, int exclusive, bcf_stream_t stream)
{
    if (num_tiles == 0) return BCF_OK;
    if (num_tiles >= (size_t(1) << 22) || !d_keys) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys)) return BCF_ERR_MISALIGNED;
    Call c;
    c.s = stream;
    resolve_options(nullptr, &c.opt);
    const bcf_status st = current_device(&c.dev);
    if (st != BCF_OK) return st;
    ProfileGroup profile_group(stream);
    return launch_isolated_tile_mergesort(c, static_cast<uint32_t *>(d_keys), num_tiles, exclusive);
}

// ------------------------------------------------------------------ measurement hooks

bcf_status bcf_profile_enable(int on)
{
    g_prof.on = on != 0;
    g_prof.used = 0;
    g_prof.open_since = -1;
    g_prof.dropped = 0;
    return BCF_OK;
}

bcf_status bcf_profile_read(float *ms, unsigned long long *launches)
{
    if (!ms || !launches) return BCF_ERR_INVALID_ARG;
    for (int c = 0; c < BCF_KERNEL_CLASSES; ++c) { ms[c] = 0.f; launches[c] = 0; }
    for (int i = 0; i + 1 < g_prof.used; ++i) {
        if (g_prof.cls[i] < 0) continue;
        if (cudaEventSynchronize(g_prof.ev[i + 1]) != cudaSuccess) return BCF_ERR_CUDA;
        float t = 0.f;
        if (cudaEventElapsedTime(&t, g_prof.ev[i], g_prof.ev[i + 1]) != cudaSuccess) return BCF_ERR_CUDA;
        ms[g_prof.cls[i]] += t;
        launches[g_prof.cls[i]]++;
    }
    g_prof.used = 0;
    return BCF_OK;
}

unsigned long long bcf_profile_dropped(void) { return g_prof.dropped; }

void bcf_launch_counts(unsigned long long *launches)
{
    for (int c = 0; c < BCF_KERNEL_CLASSES; ++c) {
        const unsigned long long v = g_prof.launches[c].exchange(0, std::memory_order_relaxed);
        if (launches) launches[c] = v;
    }
}

const char *bcf_kernel_name(int kernel_id)
{
    static const char *names[BCF_KID_COUNT] = {
        "tile_sort_kernel", "tile_mergesort_kernel", "long_tile_sort_kernel<h=2>", "long_tile_sort_kernel<h=4>",
        "long_tile_sort_kernel<h=8>", "partition_kernel", "merge_kernel", "partition_share_kernel<G=1>",
        "partition_share_kernel<G=32>", "merge_pipe_kernel", "partition4_kernel", "merge4_pipe_kernel",
        "pagewise_merge_kernel", "merge_pieces_kernel", "merge4_stream_kernel"};
    return (kernel_id >= 0 && kernel_id < BCF_KID_COUNT) ? names[kernel_id] : nullptr;
}

bcf_status bcf_kernel_info(int kernel_id, bcf_key_t kt, bcf_val_t vt, int *regs_per_thread, int *smem_bytes_per_cta,
                           int *threads_per_cta, int *ctas_per_sm, int *local_bytes_per_thread)
{
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
    KernelDesc k = {nullptr, 0, 0};
    bool ok = false;
    BCF_DISPATCH(kt, vt, ok = kernel_desc<E>(kernel_id, kt, &k));
    if (!ok || !k.fn) return BCF_ERR_INVALID_ARG;
    (void)cudaGetLastError();
    cudaFuncAttributes a;
    BCF_CUDA(cudaFuncGetAttributes(&a, k.fn));
    if (k.smem > 48 * 1024) BCF_CUDA(cudaFuncSetAttribute(k.fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)k.smem));
    int occ = 0;
    BCF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k.fn, k.threads, k.smem));
    if (regs_per_thread) *regs_per_thread = a.numRegs;
    if (smem_bytes_per_cta) *smem_bytes_per_cta = static_cast<int>(a.sharedSizeBytes + k.smem);
    if (threads_per_cta) *threads_per_cta = k.threads;
    if (ctas_per_sm) *ctas_per_sm = occ;
    if (local_bytes_per_thread) *local_bytes_per_thread = static_cast<int>(a.localSizeBytes);
    return BCF_OK;
}

// ------------------------------------------------------------------ layout introspection (host only)

int bcf_layout_word(int row, int col)
{
    if (row < 0 || row > 31 || col < 0 || col > 31) return -1;
    return elem_word(row, col);
}

int bcf_layout_access(int pattern, int step, int lane, int *first_word)
{
    if (!first_word || lane < 0 || lane > 31 || step < 0) return 0;
    switch (pattern) {
    case BCF_ACCESS_ROW_STORE:
    case BCF_ACCESS_ROW_LOAD:
        if (step > 7) return 0;
        *first_word = chunk_word(lane, step);
        return 4;
    case BCF_ACCESS_COL_LOAD:
    case BCF_ACCESS_COL_STORE:
        if (step > 31) return 0;
        *first_word = elem_word(step, mirrored_col(step, lane));
        return 1;
    case BCF_ACCESS_COL_STORE_PLAIN:
    case BCF_ACCESS_OUT_LOAD32:
        if (step > 31) return 0;
        *first_word = elem_word(step, lane);
        return 1;
    case BCF_ACCESS_OUT_LOAD128:
        if (step > 7) return 0;
        *first_word = chunk_word(4 * step + (lane >> 3), lane & 7);
        return 4;
    case BCF_ACCESS_COL_LOAD_LEVEL: {
        if (step > 159) return 0;
        const int T = step / 32 + 1, k = step % 32;
        *first_word = elem_word(merge_level_row(T, k), merge_level_mirror(T, k) ? 31 - lane : lane);
        return 1;
    }
    case BCF_ACCESS_OUT_LOAD64:
        if (step > 15) return 0;
        *first_word = elem_word(2 * step + (lane >> 4), 2 * (lane & 15));
        return 2;
    case BCF_ACCESS_LT_FLIP_ROW_LOAD:          // bcf_long_tile.cuh cross_stage_keep<FLIP = true>
        if (step > 7) return 0;
        *first_word = chunk_word(31 - lane, 7 - step);
        return 4;
    case BCF_ACCESS_LT_FUSED_COL_LOAD:         // bcf_long_tile.cuh cross_stage_cols_keep<FLIP = true>, partner read
        if (step > 31) return 0;
        *first_word = elem_word(31 - step, 31 - lane);
        return 1;
    case BCF_ACCESS_SLOT_LOAD32:               // bcf_merge_pipe.cuh load_slot32: ascending A piece / descending B piece
        if (step > 63) return 0;
        *first_word = step < 32 ? step + lane : 1023 - (step - 32) - lane;
        return 1;
    case BCF_ACCESS_SLOT_LOAD64:               // bcf_merge_pipe.cuh load_slot64 (ld.shared.v2.u32)
        if (step > 63) return 0;
        *first_word = 2 * (step < 32 ? step + lane : 1023 - (step - 32) - lane);
        return 2;
    }
    return 0;
}

}  // extern "C"
