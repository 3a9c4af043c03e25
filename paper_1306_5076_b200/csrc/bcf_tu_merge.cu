// bcf_tu_merge.cu -- translation unit of the one-warp-per-page merge round for any run length
// (partition_kernel + merge_kernel, rows a5-a6, bcf_kernels.cuh) and of the paper's page-wise streaming
// merge (pagewise_merge_kernel, row a7, bcf_pagewise.cuh).
#include "bcf_internal.cuh"
#include "bcf_kernels.cuh"
#include "bcf_pagewise.cuh"

namespace bcf {

template <class E>
bcf_status launch_partition(const Call &c, const void *kin, const uint32_t *vin, uint32_t *splits, const PassGeom &g)
{
    if (g.num_shares == 0) return BCF_OK;
    const unsigned blocks = static_cast<unsigned>((g.num_shares + 127) / 128);
    LaunchTimer t(BCF_KERNEL_PARTITION, c.s);
    return launch(c, partition_kernel<E>, blocks, 128, 0, kin, vin, splits, g);
}

template <class E>
bcf_status launch_merge(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, const uint32_t *splits,
                        const PassGeom &g)
{
    if (g.num_shares == 0) return BCF_OK;
    const size_t smem = WARPS_PER_CTA * size_t(E::NP) * TILE * 4;
    const bcf_status st = ensure_dyn_smem<merge_kernel<E>>(c.dev, smem);
    if (st != BCF_OK) return st;
    const unsigned blocks = static_cast<unsigned>((g.num_shares + WARPS_PER_CTA - 1) / WARPS_PER_CTA);
    LaunchTimer t(BCF_KERNEL_MERGE, c.s);
    return launch(c, merge_kernel<E>, blocks, WARPS_PER_CTA * 32, smem, kin, vin, kout, vout, splits, g);
}

template <class E>
bcf_status launch_pagewise(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, size_t n, size_t run_len)
{
    const size_t pairs = (n + 2 * run_len - 1) / (2 * run_len);
    if (pairs == 0) return BCF_OK;
    const size_t smem = WARPS_PER_CTA * size_t(E::NP) * TILE * 4;
    const bcf_status st = ensure_dyn_smem<pagewise_merge_kernel<E>>(c.dev, smem);
    if (st != BCF_OK) return st;
    const unsigned blocks = static_cast<unsigned>((pairs + WARPS_PER_CTA - 1) / WARPS_PER_CTA);
    LaunchTimer t(BCF_KERNEL_MERGE_PAGEWISE, c.s);
    return launch(c, pagewise_merge_kernel<E>, blocks, WARPS_PER_CTA * 32, smem, kin, vin, kout, vout, n, run_len);
}

template <class E>
bool kernel_desc_merge(int id, KernelDesc *k)
{
    const size_t smem = WARPS_PER_CTA * size_t(E::NP) * TILE * 4;
    switch (id) {
    case BCF_KID_PARTITION: *k = {(const void *)partition_kernel<E>, 0, 128}; return true;
    case BCF_KID_MERGE: *k = {(const void *)merge_kernel<E>, smem, WARPS_PER_CTA * 32}; return true;
    case BCF_KID_MERGE_PAGEWISE: *k = {(const void *)pagewise_merge_kernel<E>, smem, WARPS_PER_CTA * 32}; return true;
    }
    return false;
}

template bcf_status launch_partition<E_U32>(const Call &, const void *, const uint32_t *, uint32_t *, const PassGeom &);
template bcf_status launch_merge<E_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, const uint32_t *, const PassGeom &);
template bcf_status launch_pagewise<E_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, size_t, size_t);
template bool kernel_desc_merge<E_U32>(int, KernelDesc *);
template bcf_status launch_partition<E_U32_U32>(const Call &, const void *, const uint32_t *, uint32_t *, const PassGeom &);
template bcf_status launch_merge<E_U32_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, const uint32_t *, const PassGeom &);
template bcf_status launch_pagewise<E_U32_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, size_t, size_t);
template bool kernel_desc_merge<E_U32_U32>(int, KernelDesc *);
template bcf_status launch_partition<E_U64>(const Call &, const void *, const uint32_t *, uint32_t *, const PassGeom &);
template bcf_status launch_merge<E_U64>(const Call &, const void *, const uint32_t *, void *, uint32_t *, const uint32_t *, const PassGeom &);
template bcf_status launch_pagewise<E_U64>(const Call &, const void *, const uint32_t *, void *, uint32_t *, size_t, size_t);
template bool kernel_desc_merge<E_U64>(int, KernelDesc *);
template bcf_status launch_partition<E_U64_U32>(const Call &, const void *, const uint32_t *, uint32_t *, const PassGeom &);
template bcf_status launch_merge<E_U64_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, const uint32_t *, const PassGeom &);
template bcf_status launch_pagewise<E_U64_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, size_t, size_t);
template bool kernel_desc_merge<E_U64_U32>(int, KernelDesc *);

}  // namespace bcf
