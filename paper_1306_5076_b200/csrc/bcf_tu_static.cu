// bcf_tu_static.cu -- bcf_merge_round_static (include/bcf.h): one merge round (rows a5 + a6) whose split-point
// scratch lives inside the library instead of in a workspace the caller has to find memory for.
//
// Who this is for.  Every other entry point that merges needs a workspace from the caller, and getting one usually
// means cudaMalloc (or a framework allocator that ends in it).  Some callers cannot do that at the point where they
// want to merge: a plugin or operator that a host engine calls inside its execute step and that is forbidden to
// allocate there; a process whose memory budget was handed out in full at start-up, so a late cudaMalloc fails; a
// latency-bound loop that cannot afford the device-wide synchronisation an allocation or a free may bring.  Such a
// caller still owns its input and output arrays; only the split points (one uint32 per 1024 outputs) had nowhere to go.
//
// The scratch is the file-scope array g_static_splits below: BCF_STATIC_MAX_SHARES uint32 = 256 KiB that every GPU
// which loads libbcf.so holds until the process exits, used or not.  That fixed size is the limit of this entry
// point (a round of at most BCF_STATIC_MAX_SHARES output pages, i.e. up to 2^26 elements when 2 * run_len is a
// multiple of 1024); larger rounds are refused with BCF_ERR_TOO_LARGE and belong to bcf_merge_runs.
//
// The kernels are the library's own partition_kernel / merge_kernel (bcf_kernels.cuh), unchanged: they receive the
// scratch as an ordinary pointer argument and never name the array, so it does not matter that these templates are
// also instantiated in bcf_tu_merge.cu.
#include "bcf_internal.cuh"
#include "bcf_kernels.cuh"

#include <mutex>

using namespace bcf;

namespace {

// The scratch itself.  In HOST code this name is only a stand-in for the symbol (its host-side "address" is not
// device memory); the device address is looked up once per device in static_setup() and handed to the kernels.
static __device__ __align__(256) uint32_t g_static_splits[BCF_STATIC_MAX_SHARES];

struct StaticDev {
    std::atomic<int> state{0};      // 0 not set up, 1 ready, 2 unsupported device
    uint32_t *splits = nullptr;     // device address of g_static_splits on this device
    int num_sms = 0;
};
StaticDev g_static_dev[MAX_DEVICES];
std::mutex g_static_mutex;          // serialises the one-off set-up; never taken once a device is ready

template <class E>
constexpr size_t merge_smem() { return WARPS_PER_CTA * size_t(E::NP) * TILE * 4; }

// First call on the current device: compute-capability check, the device address of the scratch, and the
// dynamic shared memory opt-in of the four merge kernels.  Nothing here allocates through the CUDA API (the
// driver loads this file's module on first use, as for any kernel).
bcf_status static_setup(Dev *d)
{
    (void)cudaGetLastError();
    int dev = -1;
    BCF_CUDA(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAX_DEVICES) return BCF_ERR_UNSUPPORTED_DEVICE;
    StaticDev &sd = g_static_dev[dev];
    int st = sd.state.load(std::memory_order_acquire);
    if (st == 0) {
        std::lock_guard<std::mutex> lock(g_static_mutex);
        st = sd.state.load(std::memory_order_acquire);
        if (st == 0) {
            int major = 0, sms = 0;
            BCF_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
            BCF_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
            if (major != 10) {
                sd.state.store(2, std::memory_order_release);
                return BCF_ERR_UNSUPPORTED_DEVICE;
            }
            void *p = nullptr;
            BCF_CUDA(cudaGetSymbolAddress(&p, g_static_splits));      // this device's copy of the array
            if (!p) return cuda_fail(cudaErrorInvalidSymbol);
            Dev tmp;
            tmp.id = dev;
            tmp.num_sms = sms;
            bcf_status s;
            if ((s = ensure_dyn_smem<merge_kernel<E_U32>>(tmp, merge_smem<E_U32>())) != BCF_OK) return s;
            if ((s = ensure_dyn_smem<merge_kernel<E_U32_U32>>(tmp, merge_smem<E_U32_U32>())) != BCF_OK) return s;
            if ((s = ensure_dyn_smem<merge_kernel<E_U64>>(tmp, merge_smem<E_U64>())) != BCF_OK) return s;
            if ((s = ensure_dyn_smem<merge_kernel<E_U64_U32>>(tmp, merge_smem<E_U64_U32>())) != BCF_OK) return s;
            sd.splits = static_cast<uint32_t *>(p);
            sd.num_sms = sms;
            sd.state.store(1, std::memory_order_release);
            st = 1;
        }
    }
    if (st != 1) return BCF_ERR_UNSUPPORTED_DEVICE;
    d->id = dev;
    d->num_sms = sd.num_sms;
    return BCF_OK;
}

bool ranges_overlap(const void *a, size_t an, const void *b, size_t bn)
{
    if (!a || !b || !an || !bn) return false;
    const uintptr_t x = reinterpret_cast<uintptr_t>(a), y = reinterpret_cast<uintptr_t>(b);
    return x < y + bn && y < x + an;
}

// partition -> g_static_splits -> merge, both launched on the caller's stream (plain stream order)
template <class E>
bcf_status static_round(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, uint32_t *splits,
                        const PassGeom &g)
{
    const unsigned pblocks = static_cast<unsigned>((g.num_shares + 127) / 128);
    const bcf_status st = launch(c, partition_kernel<E>, pblocks, 128, 0, kin, vin, splits, g);
    if (st != BCF_OK) return st;
    const unsigned mblocks = static_cast<unsigned>((g.num_shares + WARPS_PER_CTA - 1) / WARPS_PER_CTA);
    return launch(c, merge_kernel<E>, mblocks, WARPS_PER_CTA * 32, merge_smem<E>(), kin, vin, kout, vout,
                  static_cast<const uint32_t *>(splits), g);
}

}  // namespace

extern "C" {

size_t bcf_merge_round_static_max_shares(void) { return BCF_STATIC_MAX_SHARES; }

size_t bcf_merge_round_static_shares(size_t n, size_t run_len)
{
    if (n == 0 || run_len == 0 || n >= (size_t(1) << 32)) return 0;
    return static_cast<size_t>(pass_geom(n, run_len > n ? n : run_len).num_shares);
}

bcf_status bcf_merge_round_static(const void *d_keys_in, const void *d_vals_in, void *d_keys_out, void *d_vals_out, size_t n,
                                  size_t run_len, bcf_key_t kt, bcf_val_t vt, bcf_stream_t stream)
{
    if (!valid_types(kt, vt)) return BCF_ERR_INVALID_ARG;
    if (n == 0) return BCF_OK;
    if (n >= (size_t(1) << 32) || run_len == 0) return BCF_ERR_INVALID_ARG;
    if (!d_keys_in || !d_keys_out) return BCF_ERR_INVALID_ARG;
    if ((vt == BCF_VAL_U32) != (d_vals_in != nullptr) || (vt == BCF_VAL_U32) != (d_vals_out != nullptr))
        return BCF_ERR_INVALID_ARG;
    if (!aligned16(d_keys_in) || !aligned16(d_keys_out) || !aligned16(d_vals_in) || !aligned16(d_vals_out))
        return BCF_ERR_MISALIGNED;
    const size_t kb = n * key_bytes(kt), vb = (vt == BCF_VAL_U32) ? n * 4 : 0;
    if (ranges_overlap(d_keys_in, kb, d_keys_out, kb) || ranges_overlap(d_vals_in, vb, d_vals_out, vb) ||
        ranges_overlap(d_keys_in, kb, d_vals_out, vb) || ranges_overlap(d_vals_in, vb, d_keys_out, kb))
        return BCF_ERR_INVALID_ARG;
    // the limit: the round's split points must fit the built-in array (checked before anything touches the device)
    // (a run_len beyond n means a single run, which the round copies; clamped so 2 * run_len cannot overflow)
    const PassGeom g = pass_geom(n, run_len > n ? n : run_len);
    if (g.num_shares > BCF_STATIC_MAX_SHARES) return BCF_ERR_TOO_LARGE;

    Call c;
    c.s = stream;
    c.opt.pdl = false;               // ordinary stream-ordered launches
    const bcf_status st = static_setup(&c.dev);
    if (st != BCF_OK) return st;
    uint32_t *splits = g_static_dev[c.dev.id].splits;
    const uint32_t *vin = static_cast<const uint32_t *>(d_vals_in);
    uint32_t *vout = static_cast<uint32_t *>(d_vals_out);
    if (kt == BCF_KEY_U32 && vt == BCF_VAL_NONE) return static_round<E_U32>(c, d_keys_in, vin, d_keys_out, vout, splits, g);
    if (kt == BCF_KEY_U32) return static_round<E_U32_U32>(c, d_keys_in, vin, d_keys_out, vout, splits, g);
    if (vt == BCF_VAL_NONE) return static_round<E_U64>(c, d_keys_in, vin, d_keys_out, vout, splits, g);
    return static_round<E_U64_U32>(c, d_keys_in, vin, d_keys_out, vout, splits, g);
}

}  // extern "C"
