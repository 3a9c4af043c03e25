// bcf_tu_merge4.cu -- translation unit of the four-run pass (bcf_merge4.cuh): multi-sequence
// selection + two merge rounds per read + write of the data.
#include "bcf_internal.cuh"
#include "bcf_merge4.cuh"
#include "bcf_merge4s.cuh"

namespace bcf {

template <class E>
bool merge4_fits() { return pipe4::Cfg4<E>::fits; }

template <class E>
bcf_status launch_partition4(const Call &c, const void *kin, const uint32_t *vin, uint32_t *splits, size_t n, size_t run_len,
                             size_t num_bounds)
{
    if (num_bounds == 0) return BCF_OK;
    const unsigned blocks = static_cast<unsigned>((num_bounds + pipe4::PART4_THREADS - 1) / pipe4::PART4_THREADS);
    LaunchTimer t(BCF_KERNEL_PARTITION, c.s);
    return launch(c, pipe4::partition4_kernel<E>, blocks, pipe4::PART4_THREADS, 0, kin, vin, reinterpret_cast<uint4 *>(splits),
                  static_cast<unsigned long long>(n), static_cast<unsigned long long>(run_len),
                  static_cast<unsigned long long>(num_bounds), static_cast<unsigned long long>(pipe4::SH));
}

// One pass = two merge rounds: groups of four runs of run_len become one run of 4 run_len.
template <class E>
bcf_status launch_merge4(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, uint32_t *splits, size_t n,
                         size_t run_len)
{
    using C = pipe4::Cfg4<E>;
    if constexpr (!C::fits) {
        return BCF_ERR_INVALID_ARG;
    } else {
        const unsigned long long shares = (n + pipe4::SH - 1) / pipe4::SH;
        if (shares == 0) return BCF_OK;
        bcf_status st = ensure_dyn_smem<pipe4::merge4_pipe_kernel<E>>(c.dev, C::total);
        if (st != BCF_OK) return st;
        if (4 * run_len > (size_t)pipe4::SH) {
            st = launch_partition4<E>(c, kin, vin, splits, n, run_len, shares + 1);
            if (st != BCF_OK) return st;
            // shares that cut through the runs: the task-stream kernel (no CTA barrier between the two levels)
            if constexpr (pipe4s::Cfg4s<E>::fits) {
                if (!c.opt.merge4_barrier) {
                    using S = pipe4s::Cfg4s<E>;
                    st = ensure_dyn_smem<pipe4s::merge4_stream_kernel<E>>(c.dev, S::total);
                    if (st != BCF_OK) return st;
                    LaunchTimer t(BCF_KERNEL_MERGE, c.s);
                    const unsigned long long sms = c.dev.num_sms;
                    return launch(c, pipe4s::merge4_stream_kernel<E>, static_cast<unsigned>(shares < sms ? shares : sms), pipe4s::THREADS,
                                  S::total, kin, vin, kout, vout, reinterpret_cast<const uint4 *>(splits),
                                  static_cast<unsigned long long>(n), static_cast<unsigned long long>(run_len), shares);
                }
            }
        }
        LaunchTimer t(BCF_KERNEL_MERGE, c.s);
        const unsigned long long cap = static_cast<unsigned long long>(C::ctas_per_sm) * c.dev.num_sms;
        const unsigned blocks = static_cast<unsigned>(shares < cap ? shares : cap);
        return launch(c, pipe4::merge4_pipe_kernel<E>, blocks, pipe4::THREADS, C::total, kin, vin, kout, vout,
                      reinterpret_cast<const uint4 *>(splits), static_cast<unsigned long long>(n),
                      static_cast<unsigned long long>(run_len), shares);
    }
}

template <class E>
bool kernel_desc_merge4(int id, KernelDesc *k)
{
    switch (id) {
    case BCF_KID_PARTITION4: *k = {(const void *)pipe4::partition4_kernel<E>, 0, pipe4::PART4_THREADS}; return true;
    case BCF_KID_MERGE4_PIPE:
        if constexpr (pipe4::Cfg4<E>::fits) {
            *k = {(const void *)pipe4::merge4_pipe_kernel<E>, pipe4::Cfg4<E>::total, pipe4::THREADS};
            return true;
        } else {
            return false;
        }
    case BCF_KID_MERGE4_STREAM:
        if constexpr (pipe4s::Cfg4s<E>::fits) {
            *k = {(const void *)pipe4s::merge4_stream_kernel<E>, pipe4s::Cfg4s<E>::total, pipe4s::THREADS};
            return true;
        } else {
            return false;
        }
    }
    return false;
}

template bool merge4_fits<E_U32>();
template bcf_status launch_partition4<E_U32>(const Call &, const void *, const uint32_t *, uint32_t *, size_t, size_t, size_t);
template bcf_status launch_merge4<E_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, uint32_t *, size_t, size_t);
template bool kernel_desc_merge4<E_U32>(int, KernelDesc *);
template bool merge4_fits<E_U32_U32>();
template bcf_status launch_partition4<E_U32_U32>(const Call &, const void *, const uint32_t *, uint32_t *, size_t, size_t, size_t);
template bcf_status launch_merge4<E_U32_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, uint32_t *, size_t, size_t);
template bool kernel_desc_merge4<E_U32_U32>(int, KernelDesc *);
template bool merge4_fits<E_U64>();
template bcf_status launch_partition4<E_U64>(const Call &, const void *, const uint32_t *, uint32_t *, size_t, size_t, size_t);
template bcf_status launch_merge4<E_U64>(const Call &, const void *, const uint32_t *, void *, uint32_t *, uint32_t *, size_t, size_t);
template bool kernel_desc_merge4<E_U64>(int, KernelDesc *);
template bool merge4_fits<E_U64_U32>();
template bcf_status launch_partition4<E_U64_U32>(const Call &, const void *, const uint32_t *, uint32_t *, size_t, size_t, size_t);
template bcf_status launch_merge4<E_U64_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, uint32_t *, size_t, size_t);
template bool kernel_desc_merge4<E_U64_U32>(int, KernelDesc *);

}  // namespace bcf
