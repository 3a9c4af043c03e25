// bcf_api.cu -- the C ABI of include/bcf.h: argument validation, workspace carving, the merge-round
// driver and the measurement hooks.  Every step of the path runs in the
// kernels of bcf_kernels.cuh; there is no CPU fallback.
#include "../../include/bcf.h"

#include <cstdio>
#include <cstring>

#include "bcf_kernels.cuh"
#include "bcf_pagewise.cuh"
#include "bcf_merge_pipe.cuh"
#include "bcf_merge4.cuh"
#include "bcf_long_tile.cuh"
#include "bcf_buckets.cuh"
#include "bcf_colored_scan.cuh"
#include <cstdlib>

using namespace bcf;

namespace {

// ------------------------------------------------------------------ small host helpers

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline int ceil_log2(size_t x) { int l = 0; while ((size_t(1) << l) < x) ++l; return l; }
inline size_t key_bytes(bcf_key_t kt) { return kt == BCF_KEY_U64 ? 8 : 4; }
inline bool valid_types(bcf_key_t kt, bcf_val_t vt)
{
    return (kt == BCF_KEY_U32 || kt == BCF_KEY_U64) && (vt == BCF_VAL_NONE || vt == BCF_VAL_U32);
}

PassGeom pass_geom(size_t n, size_t run_len)
{
    PassGeom g;
    g.n = n;
    g.run_len = run_len;
    const unsigned long long two_l = 2ull * run_len;
    g.shares_per_pair = static_cast<unsigned int>((two_l + TILE - 1) / TILE);
    const unsigned long long pairs = (n + two_l - 1) / two_l;
    g.num_shares = pairs * g.shares_per_pair;
    return g;
}

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

bcf_status check_device()
{
    static int cached_dev = -1;
    static bcf_status cached = BCF_ERR_UNSUPPORTED_DEVICE;
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return BCF_ERR_CUDA;
    if (dev == cached_dev) return cached;
    int major = 0;
    if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess) return BCF_ERR_CUDA;
    cached_dev = dev;
    cached = (major == 10) ? BCF_OK : BCF_ERR_UNSUPPORTED_DEVICE;
    return cached;
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
    unsigned long long launches[BCF_KERNEL_CLASSES] = {0, 0, 0, 0};
} g_prof;

inline int profile_mark(int cls, cudaStream_t s)
{
    if (!g_prof.on || g_prof.used >= PROFILE_POOL) return -1;
    const int idx = g_prof.used++;
    if (idx >= g_prof.created) {
        cudaEventCreate(&g_prof.ev[idx]);
        g_prof.created = idx + 1;
    }
    g_prof.cls[idx] = cls;
    cudaEventRecord(g_prof.ev[idx], s);
    return idx;
}

struct LaunchTimer {
    LaunchTimer(int cls, cudaStream_t stream)
    {
        g_prof.launches[cls]++;
        profile_mark(cls, stream);
    }
};

// Closes the timed launches of one public API call (outermost scope only).
struct ProfileGroup {
    cudaStream_t s;
    bool outer;
    explicit ProfileGroup(cudaStream_t stream) : s(stream), outer(g_prof.open_since < 0)
    {
        if (outer) g_prof.open_since = g_prof.used;
    }
    ~ProfileGroup()
    {
        if (!outer) return;
        if (g_prof.used > g_prof.open_since && g_prof.cls[g_prof.used - 1] >= 0) profile_mark(-1, s);
        g_prof.open_since = -1;
    }
};

// ------------------------------------------------------------------ launchers

template <class E>
constexpr size_t warp_smem_bytes() { return size_t(E::NP) * TILE * 4; }

// Base case of bcf_sort: BCF_BASE_SHEARSORT (the paper's tile sort), BCF_BASE_TILE_MERGESORT (same tile,
// same movement, mergers instead of full line sorts; bcf_kernels.cuh), BCF_BASE_LONG_TILES (8 tiles per CTA,
// bcf_long_tile.cuh) or BCF_BASE_AUTO.  bcf_set_base_case().
#ifndef BCF_DEFAULT_BASE_CASE
#define BCF_DEFAULT_BASE_CASE BCF_BASE_AUTO
#endif
int g_base_case = -1;
inline int base_case()
{
    if (g_base_case < 0) {
        const char *e = std::getenv("BCF_BASE_CASE");
        const int v = e ? std::atoi(e) : BCF_DEFAULT_BASE_CASE;
        g_base_case = (v >= BCF_BASE_SHEARSORT && v <= BCF_BASE_AUTO) ? v : BCF_DEFAULT_BASE_CASE;
    }
    return g_base_case;
}

template <class E>
bcf_status launch_tile_sort(const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, size_t n,
                            cudaStream_t s, int algo = BCF_BASE_SHEARSORT)
{
    const size_t tiles = (n + TILE - 1) / TILE;
    if (tiles == 0) return BCF_OK;
    const size_t smem = WARPS_PER_CTA * warp_smem_bytes<E>();
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(tile_sort_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess ||
            cudaFuncSetAttribute(tile_mergesort_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return BCF_ERR_CUDA;
        attr_set = true;
    }
    const size_t blocks = (tiles + WARPS_PER_CTA - 1) / WARPS_PER_CTA;
    {
        LaunchTimer t(BCF_KERNEL_TILE_SORT, s);
        if (algo == BCF_BASE_TILE_MERGESORT)
            tile_mergesort_kernel<E><<<static_cast<unsigned>(blocks), WARPS_PER_CTA * 32, smem, s>>>(kin, vin, kout, vout, n);
        else
            tile_sort_kernel<E><<<static_cast<unsigned>(blocks), WARPS_PER_CTA * 32, smem, s>>>(kin, vin, kout, vout, n);
    }
    return cudaPeekAtLastError() == cudaSuccess ? BCF_OK : BCF_ERR_CUDA;
}

// Long tiles (bcf_long_tile.cuh): groups of h = 2, 4 or 8 tiles sorted by one CTA of h warps.
#ifndef BCF_LONG_TILE_H
#define BCF_LONG_TILE_H 8
#endif
template <class E, int H>
bcf_status launch_long_tile_h(const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, size_t n, cudaStream_t s)
{
    using C = LongTileCfg<E, H>;
    static int num_sms = 0, ctas = 0;
    if (!num_sms) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
            return BCF_ERR_CUDA;
        if (cudaFuncSetAttribute(long_tile_sort_kernel<E, H>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::smem) != cudaSuccess ||
            cudaOccupancyMaxActiveBlocksPerMultiprocessor(&ctas, long_tile_sort_kernel<E, H>, H * 32, C::smem) != cudaSuccess ||
            ctas < 1) {
            num_sms = 0;
            return BCF_ERR_CUDA;
        }
    }
    const size_t groups = ((n + TILE - 1) / TILE + H - 1) / H;
    if (groups == 0) return BCF_OK;
    const size_t cap = static_cast<size_t>(ctas) * num_sms * 8;     // a few waves; the kernel strides over groups
    {
        LaunchTimer t(BCF_KERNEL_TILE_SORT, s);
        long_tile_sort_kernel<E, H><<<static_cast<unsigned>(groups < cap ? groups : cap), H * 32, C::smem, s>>>(kin, vin, kout, vout, n);
    }
    return cudaPeekAtLastError() == cudaSuccess ? BCF_OK : BCF_ERR_CUDA;
}

template <class E>
bcf_status launch_long_tile(const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, size_t n, int h, cudaStream_t s)
{
    switch (h) {
    case 2: return launch_long_tile_h<E, 2>(kin, vin, kout, vout, n, s);
    case 4: return launch_long_tile_h<E, 4>(kin, vin, kout, vout, n, s);
    case 8: return launch_long_tile_h<E, 8>(kin, vin, kout, vout, n, s);
    }
    return BCF_ERR_INVALID_ARG;
}

template <class E>
bcf_status launch_partition(const void *kin, const uint32_t *vin, uint32_t *splits, const PassGeom &g, cudaStream_t s)
{
    if (g.num_shares == 0) return BCF_OK;
    const unsigned blocks = static_cast<unsigned>((g.num_shares + 127) / 128);
    {
        LaunchTimer t(BCF_KERNEL_PARTITION, s);
        partition_kernel<E><<<blocks, 128, 0, s>>>(kin, vin, splits, g);
    }
    return cudaPeekAtLastError() == cudaSuccess ? BCF_OK : BCF_ERR_CUDA;
}

template <class E>
bcf_status launch_merge(const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, const uint32_t *splits,
                        const PassGeom &g, cudaStream_t s)
{
    if (g.num_shares == 0) return BCF_OK;
    const size_t smem = WARPS_PER_CTA * warp_smem_bytes<E>();
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(merge_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return BCF_ERR_CUDA;
        attr_set = true;
    }
    const unsigned blocks = static_cast<unsigned>((g.num_shares + WARPS_PER_CTA - 1) / WARPS_PER_CTA);
    {
        LaunchTimer t(BCF_KERNEL_MERGE, s);
        merge_kernel<E><<<blocks, WARPS_PER_CTA * 32, smem, s>>>(kin, vin, kout, vout, splits, g);
    }
    return cudaPeekAtLastError() == cudaSuccess ? BCF_OK : BCF_ERR_CUDA;
}

// Power-of-two multiples of the tile size take the pipelined kernel (bcf_merge_pipe.cuh).
inline bool pipe_eligible(size_t run_len)
{
    if (run_len % TILE) return false;
    const size_t r = run_len / TILE;
    if (r & (r - 1)) return false;
    static int forced_v1 = -1;
    if (forced_v1 < 0) {
        const char *e = std::getenv("BCF_MERGE_IMPL");
        forced_v1 = (e && std::strcmp(e, "v1") == 0) ? 1 : 0;
    }
    return !forced_v1;
}

// Largest boundary count that takes the 32-lanes-per-boundary search (BCF_PART_WARP_MAX overrides).
inline unsigned long long pipe_warp_search_max()
{
    static long long v = -1;
    if (v < 0) {
        const char *e = std::getenv("BCF_PART_WARP_MAX");
        v = e ? std::atoll(e) : 4096;
    }
    return static_cast<unsigned long long>(v);
}

template <class E>
bcf_status launch_merge_pipe(const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, uint32_t *splits, size_t n,
                             size_t run_len, cudaStream_t s)
{
    using C = pipe::Cfg<E>;
    const unsigned long long shares = (n + pipe::SH - 1) / pipe::SH;
    if (shares == 0) return BCF_OK;
    static int num_sms = 0;
    if (!num_sms) {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
            return BCF_ERR_CUDA;
        if (cudaFuncSetAttribute(pipe::merge_pipe_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                 (int)C::total) != cudaSuccess) {
            num_sms = 0;
            return BCF_ERR_CUDA;
        }
    }
    if (2 * run_len > (size_t)pipe::SH) {
        LaunchTimer t(BCF_KERNEL_PARTITION, s);
        // few boundaries: latency-bound, 32 lanes per boundary; many: bandwidth-bound, one thread each
        if (shares + 1 <= pipe_warp_search_max()) {
            const unsigned blocks = static_cast<unsigned>(((shares + 1) * 32 + pipe::PART_THREADS - 1) / pipe::PART_THREADS);
            pipe::partition_share_kernel<E, 32><<<blocks, pipe::PART_THREADS, 0, s>>>(kin, vin, splits, n, run_len, shares);
        } else {
            const unsigned blocks = static_cast<unsigned>((shares + 1 + pipe::PART_THREADS - 1) / pipe::PART_THREADS);
            pipe::partition_share_kernel<E, 1><<<blocks, pipe::PART_THREADS, 0, s>>>(kin, vin, splits, n, run_len, shares);
        }
    }
    {
        LaunchTimer t(BCF_KERNEL_MERGE, s);
        const unsigned long long cap = static_cast<unsigned long long>(C::ctas_per_sm) * num_sms;
        const unsigned blocks = static_cast<unsigned>(shares < cap ? shares : cap);
        pipe::merge_pipe_kernel<E><<<blocks, pipe::THREADS, C::total, s>>>(kin, vin, kout, vout, splits, n, run_len, shares);
    }
    return cudaPeekAtLastError() == cudaSuccess ? BCF_OK : BCF_ERR_CUDA;
}

// Rounds per pass: 2 = the four-run kernel of bcf_merge4.cuh where it applies, 1 = one round per pass
// everywhere.  Set by bcf_set_rounds_per_pass(); the initial value comes from BCF_MERGE_WAYS (2 or 4 runs
// per pass) if set.
#ifndef BCF_DEFAULT_ROUNDS_PER_PASS
#define BCF_DEFAULT_ROUNDS_PER_PASS 1
#endif
int g_rounds_per_pass = -1;
inline int rounds_per_pass()
{
    if (g_rounds_per_pass < 0) {
        const char *e = std::getenv("BCF_MERGE_WAYS");
        g_rounds_per_pass = e ? (std::atoi(e) == 4 ? 2 : 1) : BCF_DEFAULT_ROUNDS_PER_PASS;
    }
    return g_rounds_per_pass;
}

// Element types whose two stage buffers of a four-run share fit one SM (bcf_merge4.cuh).
template <class E>
inline bool merge4_eligible(size_t run_len)
{
    return pipe4::Cfg4<E>::fits && pipe_eligible(run_len) && rounds_per_pass() == 2;
}

template <class E>
bcf_status launch_partition4(const void *kin, const uint32_t *vin, uint32_t *splits, size_t n, size_t run_len,
                             size_t num_bounds, cudaStream_t s)
{
    if (num_bounds == 0) return BCF_OK;
    const unsigned blocks = static_cast<unsigned>((num_bounds + pipe4::PART4_THREADS - 1) / pipe4::PART4_THREADS);
    {
        LaunchTimer t(BCF_KERNEL_PARTITION, s);
        pipe4::partition4_kernel<E><<<blocks, pipe4::PART4_THREADS, 0, s>>>(kin, vin, reinterpret_cast<uint4 *>(splits), n, run_len,
                                                                           num_bounds, pipe4::SH);
    }
    return cudaPeekAtLastError() == cudaSuccess ? BCF_OK : BCF_ERR_CUDA;
}

// One pass = two merge rounds: groups of four runs of run_len become one run of 4 run_len.
template <class E>
bcf_status launch_merge4(const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, uint32_t *splits, size_t n,
                         size_t run_len, cudaStream_t s)
{
    using C = pipe4::Cfg4<E>;
    if constexpr (!C::fits) {
        return BCF_ERR_INVALID_ARG;
    } else {
        const unsigned long long shares = (n + pipe4::SH - 1) / pipe4::SH;
        if (shares == 0) return BCF_OK;
        static int num_sms = 0;
        if (!num_sms) {
            int dev = 0;
            if (cudaGetDevice(&dev) != cudaSuccess ||
                cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
                return BCF_ERR_CUDA;
            if (cudaFuncSetAttribute(pipe4::merge4_pipe_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)C::total) != cudaSuccess) {
                num_sms = 0;
                return BCF_ERR_CUDA;
            }
        }
        if (4 * run_len > (size_t)pipe4::SH) {
            const bcf_status st = launch_partition4<E>(kin, vin, splits, n, run_len, shares + 1, s);
            if (st != BCF_OK) return st;
        }
        {
            LaunchTimer t(BCF_KERNEL_MERGE, s);
            const unsigned long long cap = static_cast<unsigned long long>(C::ctas_per_sm) * num_sms;
            const unsigned blocks = static_cast<unsigned>(shares < cap ? shares : cap);
            pipe4::merge4_pipe_kernel<E><<<blocks, pipe4::THREADS, C::total, s>>>(
                kin, vin, kout, vout, reinterpret_cast<const uint4 *>(splits), n, run_len, shares);
        }
        return cudaPeekAtLastError() == cudaSuccess ? BCF_OK : BCF_ERR_CUDA;
    }
}

template <class E>
bcf_status launch_pagewise(const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, size_t n, size_t run_len,
                           cudaStream_t s)
{
    const size_t pairs = (n + 2 * run_len - 1) / (2 * run_len);
    if (pairs == 0) return BCF_OK;
    const size_t smem = WARPS_PER_CTA * warp_smem_bytes<E>();
    static bool attr_set = false;
    if (!attr_set) {
        if (cudaFuncSetAttribute(pagewise_merge_kernel<E>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
            return BCF_ERR_CUDA;
        attr_set = true;
    }
    const unsigned blocks = static_cast<unsigned>((pairs + WARPS_PER_CTA - 1) / WARPS_PER_CTA);
    {
        LaunchTimer t(BCF_KERNEL_MERGE_PAGEWISE, s);
        pagewise_merge_kernel<E><<<blocks, WARPS_PER_CTA * 32, smem, s>>>(kin, vin, kout, vout, n, run_len);
    }
    return cudaPeekAtLastError() == cudaSuccess ? BCF_OK : BCF_ERR_CUDA;
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
    w.bytes = off;
    return w;
}

// The passes of the merging phase from sorted runs of run_len: ways[i] = 2 is one merge
// round per read + write of the data (Lemma 2), ways[i] = 4 two rounds per read + write
// (bcf_merge4.cuh).  An odd number of remaining rounds is made even by a two-way pass first.
constexpr int MAX_PASSES = 40;
template <class E>
int plan_passes(size_t n, size_t run_len, int *ways)
{
    int np = 0;
    for (size_t l = run_len; l < n && np < MAX_PASSES; ++np) {
        const int remaining = ceil_log2((n + l - 1) / l);
        const bool four = remaining % 2 == 0 && merge4_eligible<E>(l);
        ways[np] = four ? 4 : 2;
        l *= four ? 4 : 2;
    }
    return np;
}

int count_passes(size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt)
{
    int ways[MAX_PASSES];
    int np = 0;
    BCF_DISPATCH(kt, vt, np = plan_passes<E>(n, run_len, ways));
    return np;
}

// Pass i writes to dst[i]; each pass is one read + one write of all n elements.
template <class E>
bcf_status merge_rounds(const void *k0, const uint32_t *v0, void *ka, uint32_t *va, void *kb, uint32_t *vb,
                        bool first_to_a, size_t n, size_t run_len, uint32_t *splits, cudaStream_t s)
{
    const void *ksrc = k0;
    const uint32_t *vsrc = v0;
    bool to_a = first_to_a;
    int ways[MAX_PASSES];
    const int np = plan_passes<E>(n, run_len, ways);
    size_t l = run_len;
    for (int i = 0; i < np; ++i) {
        void *kd = to_a ? ka : kb;
        uint32_t *vd = to_a ? va : vb;
        bcf_status st;
        if (ways[i] == 4) {
            st = launch_merge4<E>(ksrc, vsrc, kd, vd, splits, n, l, s);
        } else if (pipe_eligible(l)) {
            st = launch_merge_pipe<E>(ksrc, vsrc, kd, vd, splits, n, l, s);
        } else {
            const PassGeom g = pass_geom(n, l);
            st = launch_partition<E>(ksrc, vsrc, splits, g, s);
            if (st != BCF_OK) return st;
            st = launch_merge<E>(ksrc, vsrc, kd, vd, splits, g, s);
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
bcf_status pagewise_rounds(const void *k0, const uint32_t *v0, void *ka, uint32_t *va, void *kb, uint32_t *vb,
                           bool first_to_a, size_t n, size_t run_len, cudaStream_t s)
{
    const void *ksrc = k0;
    const uint32_t *vsrc = v0;
    bool to_a = first_to_a;
    for (size_t l = run_len; l < n; l *= 2) {
        void *kd = to_a ? ka : kb;
        uint32_t *vd = to_a ? va : vb;
        bcf_status st = launch_pagewise<E>(ksrc, vsrc, kd, vd, n, l, s);
        if (st != BCF_OK) return st;
        ksrc = kd;
        vsrc = vd;
        to_a = !to_a;
    }
    return BCF_OK;
}

bcf_status merge_runs_common(bool pagewise, const void *d_keys_in, const void *d_vals_in, void *d_keys_out,
                             void *d_vals_out, size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt,
                             void *d_workspace, size_t workspace_bytes, cudaStream_t s)
{
    ProfileGroup profile_group(s);
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
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
    bcf_status st = check_device();
    if (st != BCF_OK) return st;

    const size_t runs = (n + run_len - 1) / run_len;
    const int rounds = ceil_log2(runs);
    if (rounds == 0) {   // a single run: the result is the input
        if (cudaMemcpyAsync(d_keys_out, d_keys_in, kb, cudaMemcpyDeviceToDevice, s) != cudaSuccess) return BCF_ERR_CUDA;
        if (vb && cudaMemcpyAsync(d_vals_out, d_vals_in, vb, cudaMemcpyDeviceToDevice, s) != cudaSuccess) return BCF_ERR_CUDA;
        return BCF_OK;
    }
    // pass i (1-based) writes to `out` when (passes - i) is even, so the last pass lands in out.
    const int passes = pagewise ? rounds : count_passes(n, run_len, kt, vt);
    const Workspace w = carve(d_workspace, n, kt, vt, passes >= 2, pagewise ? 0 : max_shares(n, run_len));
    const bool first_to_out = ((passes - 1) % 2 == 0);
    if (pagewise) {
        BCF_DISPATCH(kt, vt, st = pagewise_rounds<E>(d_keys_in, static_cast<const uint32_t *>(d_vals_in), d_keys_out,
                                                     static_cast<uint32_t *>(d_vals_out), w.keys, w.vals, first_to_out,
                                                     n, run_len, s));
    } else {
        BCF_DISPATCH(kt, vt, st = merge_rounds<E>(d_keys_in, static_cast<const uint32_t *>(d_vals_in), d_keys_out,
                                                  static_cast<uint32_t *>(d_vals_out), w.keys, w.vals, first_to_out, n,
                                                  run_len, w.splits, s));
    }
    return st;
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
    }
    return "BCF_ERR_UNKNOWN";
}

const char *bcf_version(void) { return "bcf 0.1 (sm_100a)"; }

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
        return carve(nullptr, n, kt, vt, count_passes(n, run_len, kt, vt) >= 2, max_shares(n, run_len)).bytes;
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
    ProfileGroup profile_group(stream);
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
    if (num_tiles == 0) return BCF_OK;
    if (num_tiles >= (size_t(1) << 22)) return BCF_ERR_INVALID_ARG;
    if (!d_keys || (vt == BCF_VAL_U32) != (d_vals != nullptr)) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys) || !aligned16(d_vals)) return BCF_ERR_MISALIGNED;
    bcf_status st = check_device();
    if (st != BCF_OK) return st;
    BCF_DISPATCH(kt, vt, st = launch_tile_sort<E>(d_keys, static_cast<uint32_t *>(d_vals), d_keys,
                                                  static_cast<uint32_t *>(d_vals), num_tiles * TILE, stream, algo));
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
    ProfileGroup profile_group(stream);
    if (!valid_types(kt, vt) || (h != 2 && h != 4 && h != 8)) return BCF_ERR_INVALID_ARG;
    if (num_long_tiles == 0) return BCF_OK;
    if (num_long_tiles * h >= (size_t(1) << 22)) return BCF_ERR_INVALID_ARG;
    if (!d_keys || (vt == BCF_VAL_U32) != (d_vals != nullptr)) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys) || !aligned16(d_vals)) return BCF_ERR_MISALIGNED;
    bcf_status st = check_device();
    if (st != BCF_OK) return st;
    BCF_DISPATCH(kt, vt, st = launch_long_tile<E>(d_keys, static_cast<uint32_t *>(d_vals), d_keys, static_cast<uint32_t *>(d_vals),
                                                  num_long_tiles * h * TILE, h, stream));
    return st;
}

bcf_status bcf_set_base_case(int base)
{
    if (base < BCF_BASE_SHEARSORT || base > BCF_BASE_AUTO) return BCF_ERR_INVALID_ARG;
    g_base_case = base;
    return BCF_OK;
}

int bcf_get_base_case(void) { return base_case(); }

bcf_status bcf_merge_partition(const void *d_keys_in, const void *d_vals_in, size_t n, size_t run_len, bcf_key_t kt,
                               bcf_val_t vt, uint32_t *d_splits, size_t num_shares, bcf_stream_t stream)
{
    ProfileGroup profile_group(stream);
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32) || run_len == 0) return BCF_ERR_INVALID_ARG;
    if (!d_keys_in || !d_splits || (vt == BCF_VAL_U32) != (d_vals_in != nullptr)) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys_in) || !aligned16(d_vals_in)) return BCF_ERR_MISALIGNED;
    const PassGeom g = pass_geom(n, run_len);
    if (num_shares != g.num_shares) return BCF_ERR_INVALID_ARG;
    bcf_status st = check_device();
    if (st != BCF_OK) return st;
    BCF_DISPATCH(kt, vt, st = launch_partition<E>(d_keys_in, static_cast<const uint32_t *>(d_vals_in), d_splits, g, stream));
    return st;
}

bcf_status bcf_merge_partition4(const void *d_keys_in, const void *d_vals_in, size_t n, size_t run_len, bcf_key_t kt,
                                bcf_val_t vt, uint32_t *d_splits, size_t num_bounds, bcf_stream_t stream)
{
    ProfileGroup profile_group(stream);
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32) || run_len == 0) return BCF_ERR_INVALID_ARG;
    if (!d_keys_in || !d_splits || (vt == BCF_VAL_U32) != (d_vals_in != nullptr)) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys_in) || !aligned16(d_vals_in) || !aligned16(d_splits)) return BCF_ERR_MISALIGNED;
    if (num_bounds != (n + BCF_SHARE - 1) / BCF_SHARE + 1) return BCF_ERR_INVALID_ARG;
    bcf_status st = check_device();
    if (st != BCF_OK) return st;
    BCF_DISPATCH(kt, vt, st = launch_partition4<E>(d_keys_in, static_cast<const uint32_t *>(d_vals_in), d_splits, n, run_len,
                                                   num_bounds, stream));
    return st;
}

// ------------------------------------------------------------------ FIND-BUCKETS (Alg. 7)

static bool buckets_geom(size_t n, size_t run_len, int t, int P, int pivot_buckets, buckets::Geom *g)
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

size_t bcf_find_buckets_workspace_bytes(size_t n, size_t run_len, int t, int P, int pivot_buckets, bcf_key_t kt)
{
    buckets::Geom g;
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
    buckets::Geom g;
    if (!buckets_geom(n, run_len, t, P, pivot_buckets, &g)) return BCF_ERR_INVALID_ARG;
    if (!d_keys_in || !d_keys_out || !d_pivots || !d_piece_offsets || !d_workspace) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys_in) || !aligned16(d_keys_out) || !aligned16(d_workspace)) return BCF_ERR_MISALIGNED;
    const size_t kb = n * key_bytes(kt);
    if (overlap(d_keys_in, kb, d_keys_out, kb)) return BCF_ERR_INVALID_ARG;
    const size_t need = bcf_find_buckets_workspace_bytes(n, run_len, t, P, pivot_buckets, kt);
    if (workspace_bytes < need) return BCF_ERR_WORKSPACE_TOO_SMALL;
    if (overlap(d_workspace, need, d_keys_in, kb) || overlap(d_workspace, need, d_keys_out, kb)) return BCF_ERR_INVALID_ARG;
    bcf_status st = check_device();
    if (st != BCF_OK) return st;
    ProfileGroup profile_group(stream);

    const size_t ns = (size_t)g.s * g.t;
    char *ws = static_cast<char *>(d_workspace);
    void *samples = ws;
    uint32_t *bounds = reinterpret_cast<uint32_t *>(ws + align_up(ns * key_bytes(kt), 256));
    char *sort_ws = reinterpret_cast<char *>(bounds) + align_up((size_t)g.s * (g.nb + 1) * 4, 256);
    const size_t sort_ws_bytes = workspace_bytes - static_cast<size_t>(sort_ws - ws);
    const bool k64 = (kt == BCF_KEY_U64);
    {
        const unsigned blocks = static_cast<unsigned>((ns + 255) / 256);
        LaunchTimer tm(BCF_KERNEL_PARTITION, stream);
        if (k64) buckets::sample_kernel<2><<<blocks, 256, 0, stream>>>(d_keys_in, samples, g);
        else buckets::sample_kernel<1><<<blocks, 256, 0, stream>>>(d_keys_in, samples, g);
    }
    if (cudaPeekAtLastError() != cudaSuccess) return BCF_ERR_CUDA;
    st = bcf_sort(samples, nullptr, ns, kt, BCF_VAL_NONE, sort_ws, sort_ws_bytes, stream);   // MERGESORT(S)
    if (st != BCF_OK) return st;
    {
        const size_t work = (size_t)g.s * (g.P - 1);
        const unsigned blocks = static_cast<unsigned>((work + 127) / 128);
        LaunchTimer tm(BCF_KERNEL_PARTITION, stream);
        if (k64) buckets::rank_kernel<2><<<blocks, 128, 0, stream>>>(d_keys_in, samples, d_pivots, bounds, g);
        else buckets::rank_kernel<1><<<blocks, 128, 0, stream>>>(d_keys_in, samples, d_pivots, bounds, g);
    }
    {
        LaunchTimer tm(BCF_KERNEL_PARTITION, stream);
        buckets::offsets_kernel<<<1, buckets::SCAN_THREADS, 0, stream>>>(bounds, d_piece_offsets, g);
    }
    {
        const size_t chunks = ((run_len + buckets::SCATTER_CHUNK - 1) / buckets::SCATTER_CHUNK) * g.s;
        const unsigned blocks = static_cast<unsigned>(chunks < 148 * 64 ? chunks : 148 * 64);
        LaunchTimer tm(BCF_KERNEL_MERGE, stream);
        if (k64) buckets::scatter_kernel<2><<<blocks, 256, 0, stream>>>(d_keys_in, d_keys_out, bounds, d_piece_offsets, g);
        else buckets::scatter_kernel<1><<<blocks, 256, 0, stream>>>(d_keys_in, d_keys_out, bounds, d_piece_offsets, g);
    }
    return cudaPeekAtLastError() == cudaSuccess ? BCF_OK : BCF_ERR_CUDA;
}

// ------------------------------------------------------------------ coloured prefix sums (App. A)

static unsigned colored_scan_grid(size_t n)
{
    const size_t pages = (n + cscan::PAGE - 1) / cscan::PAGE;
    const size_t ctas = (pages + cscan::WARPS - 1) / cscan::WARPS;
    return static_cast<unsigned>(ctas < 2048 ? ctas : 2048);
}

size_t bcf_colored_prefix_sums_workspace_bytes(size_t n)
{
    if (n == 0) return 0;
    return align_up(size_t(colored_scan_grid(n)) * cscan::WARPS * cscan::MAX_COLORS * 4, 256);
}

bcf_status bcf_colored_prefix_sums(const uint32_t *d_values, const uint8_t *d_colors, size_t n, int num_colors, int layout,
                                   uint32_t *d_out, void *d_workspace, size_t workspace_bytes, bcf_stream_t stream)
{
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32) || num_colors < 1 || num_colors > cscan::MAX_COLORS) return BCF_ERR_INVALID_ARG;
    if (layout != BCF_SCAN_BANK_PER_THREAD && layout != BCF_SCAN_THREAD_MAJOR) return BCF_ERR_INVALID_ARG;
    if (!d_values || !d_colors || !d_out || !d_workspace) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_values) || !aligned16(d_colors) || !aligned16(d_out) || !aligned16(d_workspace)) return BCF_ERR_MISALIGNED;
    if (overlap(d_out, n * 4, d_values, n * 4) || overlap(d_out, n * 4, d_colors, n)) return BCF_ERR_INVALID_ARG;
    if (workspace_bytes < bcf_colored_prefix_sums_workspace_bytes(n)) return BCF_ERR_WORKSPACE_TOO_SMALL;
    bcf_status st = check_device();
    if (st != BCF_OK) return st;
    ProfileGroup profile_group(stream);
    const unsigned grid = colored_scan_grid(n);
    const unsigned long long warps = static_cast<unsigned long long>(grid) * cscan::WARPS;
    uint32_t *partial = static_cast<uint32_t *>(d_workspace);
    const bool cf = (layout == BCF_SCAN_BANK_PER_THREAD);
    {
        LaunchTimer t(BCF_KERNEL_PARTITION, stream);
        if (cf) cscan::reduce_kernel<true><<<grid, cscan::WARPS * 32, 0, stream>>>(d_values, d_colors, n, num_colors, partial);
        else cscan::reduce_kernel<false><<<grid, cscan::WARPS * 32, 0, stream>>>(d_values, d_colors, n, num_colors, partial);
    }
    {
        LaunchTimer t(BCF_KERNEL_PARTITION, stream);
        cscan::offsets_kernel<<<1, cscan::MAX_COLORS * 32, 0, stream>>>(partial, warps, num_colors);
    }
    {
        LaunchTimer t(BCF_KERNEL_MERGE, stream);
        if (cf) cscan::scan_kernel<true><<<grid, cscan::WARPS * 32, 0, stream>>>(d_values, d_colors, n, num_colors, partial, d_out);
        else cscan::scan_kernel<false><<<grid, cscan::WARPS * 32, 0, stream>>>(d_values, d_colors, n, num_colors, partial, d_out);
    }
    return cudaPeekAtLastError() == cudaSuccess ? BCF_OK : BCF_ERR_CUDA;
}

bcf_status bcf_set_rounds_per_pass(int rounds)
{
    if (rounds != 1 && rounds != 2) return BCF_ERR_INVALID_ARG;
    g_rounds_per_pass = rounds;
    return BCF_OK;
}

int bcf_get_rounds_per_pass(void) { return rounds_per_pass(); }

int bcf_merge_pass_count(size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt)
{
    if (!valid_types(kt, vt) || n == 0 || run_len == 0) return 0;
    return count_passes(n, run_len, kt, vt);
}

bcf_status bcf_merge_runs(const void *d_keys_in, const void *d_vals_in, void *d_keys_out, void *d_vals_out, size_t n,
                          size_t run_len, bcf_key_t kt, bcf_val_t vt, void *d_workspace, size_t workspace_bytes,
                          bcf_stream_t stream)
{
    return merge_runs_common(false, d_keys_in, d_vals_in, d_keys_out, d_vals_out, n, run_len, kt, vt, d_workspace,
                             workspace_bytes, stream);
}

bcf_status bcf_merge_runs_pagewise(const void *d_keys_in, const void *d_vals_in, void *d_keys_out, void *d_vals_out,
                                   size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt, void *d_workspace,
                                   size_t workspace_bytes, bcf_stream_t stream)
{
    return merge_runs_common(true, d_keys_in, d_vals_in, d_keys_out, d_vals_out, n, run_len, kt, vt, d_workspace,
                             workspace_bytes, stream);
}

bcf_status bcf_sort(void *d_keys, void *d_vals, size_t n, bcf_key_t kt, bcf_val_t vt, void *d_workspace,
                    size_t workspace_bytes, bcf_stream_t stream)
{
    ProfileGroup profile_group(stream);
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32)) return BCF_ERR_INVALID_ARG;
    if (!d_keys || (vt == BCF_VAL_U32) != (d_vals != nullptr)) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys) || !aligned16(d_vals) || !aligned16(d_workspace)) return BCF_ERR_MISALIGNED;
    const size_t need = bcf_workspace_bytes(BCF_OP_SORT, n, 0, kt, vt);
    if (need && (!d_workspace || workspace_bytes < need)) return BCF_ERR_WORKSPACE_TOO_SMALL;
    const size_t kb = n * key_bytes(kt), vb = (vt == BCF_VAL_U32) ? n * 4 : 0;
    if (overlap(d_workspace, need, d_keys, kb) || overlap(d_workspace, need, d_vals, vb)) return BCF_ERR_INVALID_ARG;
    bcf_status st = check_device();
    if (st != BCF_OK) return st;

    // base case: runs of base_run sorted elements (one tile, or a long tile of h tiles)
    // AUTO: what measures fastest on B200 -- long tiles for 4-byte keys alone, the tile mergesort otherwise
    int bc = base_case();
    if (bc == BCF_BASE_AUTO) bc = (kt == BCF_KEY_U32 && vt == BCF_VAL_NONE) ? BCF_BASE_LONG_TILES : BCF_BASE_TILE_MERGESORT;
    const size_t base_run = (bc == BCF_BASE_LONG_TILES) ? size_t(BCF_LONG_TILE_H) * TILE : size_t(TILE);
    const int passes = n > base_run ? count_passes(n, base_run, kt, vt) : 0;
    const Workspace w = carve(d_workspace, n, kt, vt, passes > 0, passes > 0 ? max_shares(n, TILE) : 0);
    uint32_t *vals = static_cast<uint32_t *>(d_vals);
    // With an odd number of merge passes the base case writes into the workspace, so that the
    // last pass lands in the caller's buffer without an extra copy.
    const bool base_to_ws = (passes % 2 == 1);
    void *k0 = base_to_ws ? w.keys : d_keys;
    uint32_t *v0 = base_to_ws ? w.vals : vals;
    if (bc == BCF_BASE_LONG_TILES)
        BCF_DISPATCH(kt, vt, st = launch_long_tile<E>(d_keys, vals, k0, v0, n, BCF_LONG_TILE_H, stream));
    else
        BCF_DISPATCH(kt, vt, st = launch_tile_sort<E>(d_keys, vals, k0, v0, n, stream, bc));
    if (st != BCF_OK || passes == 0) return st;
    // pass 1 writes to the buffer the base case did not write.
    BCF_DISPATCH(kt, vt, st = merge_rounds<E>(k0, v0, d_keys, vals, w.keys, w.vals, /*first_to_a=*/base_to_ws, n, base_run,
                                              w.splits, stream));
    return st;
}

bcf_status bcf_sort_host(void *h_keys, void *h_vals, size_t n, bcf_key_t kt, bcf_val_t vt, void *d_scratch,
                         size_t scratch_bytes, bcf_stream_t stream)
{
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32)) return BCF_ERR_INVALID_ARG;
    if (!h_keys || (vt == BCF_VAL_U32) != (h_vals != nullptr)) return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_scratch)) return BCF_ERR_MISALIGNED;
    const size_t need = bcf_workspace_bytes(BCF_OP_SORT_HOST, n, 0, kt, vt);
    if (!d_scratch || scratch_bytes < need) return BCF_ERR_WORKSPACE_TOO_SMALL;
    const size_t kb = n * key_bytes(kt), vb = (vt == BCF_VAL_U32) ? n * 4 : 0;
    char *base = static_cast<char *>(d_scratch);
    void *dk = base;
    void *dv = vb ? base + align_up(kb, 256) : nullptr;
    const size_t data = align_up(kb, 256) + (vb ? align_up(vb, 256) : 0);
    if (cudaMemcpyAsync(dk, h_keys, kb, cudaMemcpyHostToDevice, stream) != cudaSuccess) return BCF_ERR_CUDA;
    if (vb && cudaMemcpyAsync(dv, h_vals, vb, cudaMemcpyHostToDevice, stream) != cudaSuccess) return BCF_ERR_CUDA;
    const bcf_status st = bcf_sort(dk, dv, n, kt, vt, base + data, scratch_bytes - data, stream);
    if (st != BCF_OK) return st;
    if (cudaMemcpyAsync(h_keys, dk, kb, cudaMemcpyDeviceToHost, stream) != cudaSuccess) return BCF_ERR_CUDA;
    if (vb && cudaMemcpyAsync(h_vals, dv, vb, cudaMemcpyDeviceToHost, stream) != cudaSuccess) return BCF_ERR_CUDA;
    if (cudaStreamSynchronize(stream) != cudaSuccess) return BCF_ERR_CUDA;
    return BCF_OK;
}

// ------------------------------------------------------------------ measurement hooks

bcf_status bcf_profile_enable(int on)
{
    g_prof.on = on != 0;
    g_prof.used = 0;
    g_prof.open_since = -1;
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

void bcf_launch_counts(unsigned long long *launches)
{
    for (int c = 0; c < BCF_KERNEL_CLASSES; ++c) {
        if (launches) launches[c] = g_prof.launches[c];
        g_prof.launches[c] = 0;
    }
}

bcf_status bcf_kernel_info(int kernel_class, bcf_key_t kt, bcf_val_t vt, int *regs_per_thread, int *smem_bytes_per_cta,
                           int *threads_per_cta, int *ctas_per_sm, int *local_bytes_per_thread)
{
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
    const void *fn = nullptr;
    size_t smem = 0;
    int threads = WARPS_PER_CTA * 32;
    BCF_DISPATCH(kt, vt, {
        switch (kernel_class) {
        case BCF_KERNEL_TILE_SORT: fn = (const void *)tile_sort_kernel<E>; smem = WARPS_PER_CTA * warp_smem_bytes<E>(); break;
        case BCF_KERNEL_TILE_MERGESORT: fn = (const void *)tile_mergesort_kernel<E>; smem = WARPS_PER_CTA * warp_smem_bytes<E>(); break;
        case BCF_KERNEL_PARTITION: fn = (const void *)partition_kernel<E>; smem = 0; threads = 128; break;
        case BCF_KERNEL_MERGE: fn = (const void *)merge_kernel<E>; smem = WARPS_PER_CTA * warp_smem_bytes<E>(); break;
        case BCF_KERNEL_MERGE_PAGEWISE: fn = (const void *)pagewise_merge_kernel<E>; smem = WARPS_PER_CTA * warp_smem_bytes<E>(); break;
        default: break;
        }
    });
    if (!fn) return BCF_ERR_INVALID_ARG;
    cudaFuncAttributes a;
    if (cudaFuncGetAttributes(&a, fn) != cudaSuccess) return BCF_ERR_CUDA;
    if (smem > 48 * 1024 && cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess)
        return BCF_ERR_CUDA;
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, fn, threads, smem) != cudaSuccess) return BCF_ERR_CUDA;
    if (regs_per_thread) *regs_per_thread = a.numRegs;
    if (smem_bytes_per_cta) *smem_bytes_per_cta = static_cast<int>(a.sharedSizeBytes + smem);
    if (threads_per_cta) *threads_per_cta = threads;
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
    }
    return 0;
}

}  // extern "C"
