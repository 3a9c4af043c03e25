// bcf_tu_pipe.cu -- translation unit of the production merge round (bcf_merge_pipe.cuh): the TMA-fed
// persistent merge kernel and its share-boundary partition kernel (rows a5-a9).
#include "bcf_internal.cuh"
#include "bcf_merge_pipe.cuh"

namespace bcf {

// split points of the share boundaries of one round (only rounds with 2 L > SH need them)
template <class E>
bcf_status launch_partition_share(const Call &c, const void *kin, const uint32_t *vin, uint32_t *splits, size_t n, size_t run_len,
                                  size_t share, const void *samp_k, const uint32_t *samp_v)
{
    if (share == 0) share = pipe::Cfg<E>::SH;
    const unsigned long long shares = (n + share - 1) / share;
    const unsigned long long ull_share = share;
    const unsigned long long ull_n = n, ull_l = run_len;
    LaunchTimer t(BCF_KERNEL_PARTITION, c.s);
    // few boundaries: latency-bound, 32 lanes per boundary; many: bandwidth-bound, one thread each
    if (shares + 1 <= c.opt.warp_search_max) {
        const unsigned blocks = static_cast<unsigned>(((shares + 1) * 32 + pipe::PART_THREADS - 1) / pipe::PART_THREADS);
        return launch(c, pipe::partition_share_kernel<E, 32>, blocks, pipe::PART_THREADS, 0, kin, vin, splits, ull_n, ull_l, shares, ull_share, samp_k, samp_v);
    }
    const unsigned blocks = static_cast<unsigned>((shares + 1 + pipe::PART_THREADS - 1) / pipe::PART_THREADS);
    return launch(c, pipe::partition_share_kernel<E, 1>, blocks, pipe::PART_THREADS, 0, kin, vin, splits, ull_n, ull_l, shares, ull_share, samp_k, samp_v);
}

template <class E>
bcf_status launch_merge_pipe(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, uint32_t *splits,
                             size_t n, size_t run_len, const PageSamples &in, const PageSamples &out)
{
    using C = pipe::Cfg<E>;
    const unsigned long long shares = (n + pipe::Cfg<E>::SH - 1) / pipe::Cfg<E>::SH;
    if (shares == 0) return BCF_OK;
    bcf_status st = ensure_dyn_smem<pipe::merge_pipe_kernel<E>>(c.dev, C::total);
    if (st != BCF_OK) return st;
    const unsigned long long cap = static_cast<unsigned long long>(C::ctas_per_sm) * c.dev.num_sms;
    const unsigned blocks = static_cast<unsigned>(shares < cap ? shares : cap);
    // shares that cut through the runs need split points: from a partition launch, or -- small launches -- worked
    // out by the merge kernel's own CTAs (merge_pipe_kernel, self_part)
    int self_part = 0;
    if (2 * run_len > (size_t)C::SH) {
        if ((shares + blocks - 1) / blocks <= (unsigned long long)C::SELF_MAX && !c.opt.no_self_partition) {
            self_part = 1;
        } else {
            st = launch_partition_share<E>(c, kin, vin, splits, n, run_len, 0, in.keys, in.vals);
            if (st != BCF_OK) return st;
        }
    }
    LaunchTimer t(BCF_KERNEL_MERGE, c.s);
    return launch(c, pipe::merge_pipe_kernel<E>, blocks, C::THREADS, C::total, kin, vin, kout, vout,
                  static_cast<const uint32_t *>(splits), static_cast<unsigned long long>(n),
                  static_cast<unsigned long long>(run_len), shares, self_part, out.keys, out.vals);
}

template <class E>
bool kernel_desc_pipe(int id, KernelDesc *k)
{
    switch (id) {
    case BCF_KID_PARTITION_SHARE_1: *k = {(const void *)pipe::partition_share_kernel<E, 1>, 0, pipe::PART_THREADS}; return true;
    case BCF_KID_PARTITION_SHARE_32: *k = {(const void *)pipe::partition_share_kernel<E, 32>, 0, pipe::PART_THREADS}; return true;
    case BCF_KID_MERGE_PIPE: *k = {(const void *)pipe::merge_pipe_kernel<E>, pipe::Cfg<E>::total, pipe::Cfg<E>::THREADS}; return true;
    }
    return false;
}

template bcf_status launch_partition_share<E_U32>(const Call &, const void *, const uint32_t *, uint32_t *, size_t, size_t, size_t, const void *,
                                                   const uint32_t *);
template bcf_status launch_merge_pipe<E_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, uint32_t *, size_t, size_t,
                                              const PageSamples &, const PageSamples &);
template bool kernel_desc_pipe<E_U32>(int, KernelDesc *);
template bcf_status launch_partition_share<E_U32_U32>(const Call &, const void *, const uint32_t *, uint32_t *, size_t, size_t, size_t, const void *,
                                                   const uint32_t *);
template bcf_status launch_merge_pipe<E_U32_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, uint32_t *, size_t, size_t,
                                              const PageSamples &, const PageSamples &);
template bool kernel_desc_pipe<E_U32_U32>(int, KernelDesc *);
template bcf_status launch_partition_share<E_U64>(const Call &, const void *, const uint32_t *, uint32_t *, size_t, size_t, size_t, const void *,
                                                   const uint32_t *);
template bcf_status launch_merge_pipe<E_U64>(const Call &, const void *, const uint32_t *, void *, uint32_t *, uint32_t *, size_t, size_t,
                                              const PageSamples &, const PageSamples &);
template bool kernel_desc_pipe<E_U64>(int, KernelDesc *);
template bcf_status launch_partition_share<E_U64_U32>(const Call &, const void *, const uint32_t *, uint32_t *, size_t, size_t, size_t, const void *,
                                                   const uint32_t *);
template bcf_status launch_merge_pipe<E_U64_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, uint32_t *, size_t, size_t,
                                              const PageSamples &, const PageSamples &);
template bool kernel_desc_pipe<E_U64_U32>(int, KernelDesc *);

}  // namespace bcf
