// bcf_internal.cuh -- host-side declarations shared by the translation units of libbcf.so (the library is
// built as several .cu files compiled in parallel; paper_1306_5076_b200/build.py): status / error helpers,
// per-device caches, the per-call options, the launch helper, the measurement hooks and the launchers each
// kernel file exports.  Nothing here is part of the C ABI (include/bcf.h).
#pragma once
#include "../../include/bcf.h"

#include <atomic>
#include <cstdint>
#include <cuda_runtime.h>

#include "bcf_layout.cuh"

namespace bcf {

// ------------------------------------------------------------------ small host helpers

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline bool aligned16(const void *p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline int ceil_log2(size_t x) { int l = 0; while ((size_t(1) << l) < x) ++l; return l; }
inline size_t key_bytes(bcf_key_t kt) { return kt == BCF_KEY_U64 ? 8 : 4; }
inline bool valid_types(bcf_key_t kt, bcf_val_t vt)
{
    return (kt == BCF_KEY_U32 || kt == BCF_KEY_U64) && (vt == BCF_VAL_NONE || vt == BCF_VAL_U32);
}

inline PassGeom pass_geom(size_t n, size_t run_len)
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

// ------------------------------------------------------------------ errors (include/bcf.h "ERRORS")

int &last_cuda_error_ref();            // thread-local, bcf_api.cu

inline bcf_status cuda_fail(cudaError_t e)
{
    last_cuda_error_ref() = static_cast<int>(e);
    (void)cudaGetLastError();          // consume it: one failure is reported once
    return BCF_ERR_CUDA;
}
// status of the launch just made on this thread
inline bcf_status launch_status()
{
    const cudaError_t e = cudaGetLastError();
    return e == cudaSuccess ? BCF_OK : cuda_fail(e);
}
#define BCF_CUDA(call)                                      \
    do {                                                    \
        const cudaError_t e_ = (call);                      \
        if (e_ != cudaSuccess) return ::bcf::cuda_fail(e_); \
    } while (0)

// ------------------------------------------------------------------ per-device state (keyed by device id)

constexpr int MAX_DEVICES = 64;
struct Dev {
    int id = -1;
    int num_sms = 0;
};

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) applies to one device: done once per (kernel, device).
template <auto Kernel>
bcf_status ensure_dyn_smem(const Dev &d, size_t bytes)
{
    static std::atomic<unsigned long long> done{0};
    const unsigned long long bit = 1ull << d.id;
    if (done.load(std::memory_order_acquire) & bit) return BCF_OK;
    BCF_CUDA(cudaFuncSetAttribute(Kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, static_cast<int>(bytes)));
    done.fetch_or(bit, std::memory_order_release);
    return BCF_OK;
}

// resident CTAs per SM of a kernel at (threads, smem), cached per (kernel, device)
template <auto Kernel>
bcf_status resident_ctas(const Dev &d, int threads, size_t smem, int *ctas)
{
    static std::atomic<int> cache[MAX_DEVICES];
    int c = cache[d.id].load(std::memory_order_acquire);
    if (c == 0) {
        BCF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&c, Kernel, threads, smem));
        if (c < 1) return cuda_fail(cudaErrorLaunchOutOfResources);
        cache[d.id].store(c, std::memory_order_release);
    }
    *ctas = c;
    return BCF_OK;
}

// ------------------------------------------------------------------ per-call options (bcf_options, resolved)

struct Opt {
    int base_case = BCF_BASE_AUTO;
    int rounds_per_pass = 1;             // resolved: 1 or 2
    bool generic_merge = false;
    bool no_self_partition = false;      // always a partition launch, even where the merge kernel could find its own split points
    bool merge4_barrier = false;         // four-run passes with the barrier kernel even where the task-stream kernel applies
    unsigned long long warp_search_max = 4096;
    int launch_mode = BCF_LAUNCH_AUTO;
    bool pdl = false;                    // resolved per call from launch_mode and the problem size (bcf_api.cu)
};

// Everything a launcher needs to know about the call it serves.
struct Call {
    Dev dev;
    Opt opt;
    cudaStream_t s;
};

// ------------------------------------------------------------------ measurement hooks (bcf_profile_*)

// counts the launch in its class and, when timing is on, records the event that starts it (bcf_api.cu)
void profile_launch(int kernel_class, cudaStream_t s);
struct LaunchTimer {
    LaunchTimer(int cls, cudaStream_t stream) { profile_launch(cls, stream); }
};

// ------------------------------------------------------------------ one launch

// With programmatic dependent launch (bcf_options.launch_mode) the kernel may be scheduled while its
// predecessor in the stream drains; every kernel of this library waits (griddepcontrol.wait, bcf_core.cuh
// pdl_wait) before it touches global memory, so the data dependence is the stream's as before.
template <class... KArgs, class... Args>
bcf_status launch(const Call &c, void (*kernel)(KArgs...), unsigned grid, unsigned block, size_t smem, Args... args)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = c.s;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = c.opt.pdl ? 1 : 0;
    const cudaError_t e = cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
    return e == cudaSuccess ? launch_status() : cuda_fail(e);
}

// ------------------------------------------------------------------ launchers (one .cu per kernel family)

// bcf_kernel_info: function, dynamic shared memory and threads per CTA of kernel `id` for element type E
struct KernelDesc {
    const void *fn;
    size_t smem;
    int threads;
};

#ifndef BCF_LONG_TILE_H
#define BCF_LONG_TILE_H 8      // long tiles of the default base case: 8 tiles per CTA
#endif

// bcf_tu_tile.cu
template <class E>
bcf_status launch_tile_sort(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, size_t n, int algo);
template <class E>
bool kernel_desc_tile(int id, KernelDesc *k);
// bcf_tu_long.cu
template <class E>
bcf_status launch_long_tile(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, size_t n, int h);
template <class E>
bool kernel_desc_long(int id, KernelDesc *k);
// bcf_tu_merge.cu
template <class E>
bcf_status launch_partition(const Call &c, const void *kin, const uint32_t *vin, uint32_t *splits, const PassGeom &g);
template <class E>
bcf_status launch_merge(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, const uint32_t *splits,
                        const PassGeom &g);
template <class E>
bcf_status launch_pagewise(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, size_t n, size_t run_len);
template <class E>
bool kernel_desc_merge(int id, KernelDesc *k);
// bcf_tu_pipe.cu
// First and last element of every full page (1024 elements) of an array of sorted runs, written by the merge round
// that produced the array and read by the partition of the next round: keys[2 p], keys[2 p + 1] (and vals) = head
// and tail of page p.  keys == nullptr: none (not asked for / not valid).
struct PageSamples {
    void *keys = nullptr;
    uint32_t *vals = nullptr;
};
// share = 0: the share size of the production merge kernel for E
template <class E>
bcf_status launch_partition_share(const Call &c, const void *kin, const uint32_t *vin, uint32_t *splits, size_t n, size_t run_len,
                                  size_t share, const void *samp_k, const uint32_t *samp_v);
// `in`: samples of kin (or none), `out`: where to write the samples of kout (or none)
template <class E>
bcf_status launch_merge_pipe(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, uint32_t *splits,
                             size_t n, size_t run_len, const PageSamples &in, const PageSamples &out);
template <class E>
bool kernel_desc_pipe(int id, KernelDesc *k);
// bcf_tu_merge4.cu
template <class E>
bool merge4_fits();
template <class E>
bcf_status launch_partition4(const Call &c, const void *kin, const uint32_t *vin, uint32_t *splits, size_t n, size_t run_len,
                             size_t num_bounds);
template <class E>
bcf_status launch_merge4(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, uint32_t *splits, size_t n,
                         size_t run_len);
template <class E>
bool kernel_desc_merge4(int id, KernelDesc *k);

// bcf_tu_buckets.cu: FIND-BUCKETS, the final merge phase, coloured prefix sums (keys only / fixed types)
// the steps of Alg. 7 around the sort of the samples (which bcf_api.cu's driver does in between)
bcf_status launch_buckets_sample(const Call &c, const void *kin, void *samples, const BucketsGeom &g, bcf_key_t kt);
bcf_status launch_buckets_distribute(const Call &c, const void *kin, const void *sorted_samples, void *pivots, uint32_t *bounds,
                                     uint32_t *piece_offsets, void *kout, const BucketsGeom &g, bcf_key_t kt);
bcf_status launch_merge_pieces_rounds(const Call &c, const void *kin, void *kout, void *ktmp, size_t n, const uint32_t *Q,
                                      size_t groups, size_t s, int copy_odd, uint32_t *first, bcf_key_t kt);
bool kernel_desc_pieces(int id, bcf_key_t kt, KernelDesc *k);
unsigned colored_scan_grid(size_t n);
size_t colored_scan_workspace_bytes(size_t n);
int colored_scan_max_colors();
bcf_status launch_colored_scan(const Call &c, const uint32_t *values, const uint8_t *colors, size_t n, int num_colors, bool cf,
                               uint32_t *partial, uint32_t *out);

// bcf_tu_isolate.cu: the bank-conflict isolation experiment (debug entry points of include/bcf.h)
size_t isolated_share();        // share size of the experiment's merge round
bcf_status launch_isolated_merge_round(const Call &c, const uint32_t *kin, uint32_t *kout, const uint32_t *splits, size_t n,
                                       size_t run_len, int exclusive);
bcf_status launch_isolated_tile_mergesort(const Call &c, uint32_t *keys, size_t num_tiles, int exclusive);

// the four element types every templated launcher is instantiated for
using E_U32 = Elem<1, false>;
using E_U32_U32 = Elem<1, true>;
using E_U64 = Elem<2, false>;
using E_U64_U32 = Elem<2, true>;

}  // namespace bcf
