// bcf_tu_tile.cu -- translation unit of the one-warp-per-tile base cases: the paper's tile ShearSort
// (tile_sort_kernel, rows a1-a4) and the tile mergesort (tile_mergesort_kernel); bcf_kernels.cuh.
#include "bcf_internal.cuh"
#include "bcf_kernels.cuh"

namespace bcf {

template <class E>
bcf_status launch_tile_sort(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, size_t n, int algo)
{
    const size_t tiles = (n + TILE - 1) / TILE;
    if (tiles == 0) return BCF_OK;
    const size_t smem = WARPS_PER_CTA * size_t(E::NP) * TILE * 4;
    const unsigned blocks = static_cast<unsigned>((tiles + WARPS_PER_CTA - 1) / WARPS_PER_CTA);
    bcf_status st;
    if (algo == BCF_BASE_TILE_MERGESORT) {
        if ((st = ensure_dyn_smem<tile_mergesort_kernel<E>>(c.dev, smem)) != BCF_OK) return st;
        LaunchTimer t(BCF_KERNEL_TILE_SORT, c.s);
        return launch(c, tile_mergesort_kernel<E>, blocks, WARPS_PER_CTA * 32, smem, kin, vin, kout, vout, n);
    }
    if ((st = ensure_dyn_smem<tile_sort_kernel<E>>(c.dev, smem)) != BCF_OK) return st;
    LaunchTimer t(BCF_KERNEL_TILE_SORT, c.s);
    return launch(c, tile_sort_kernel<E>, blocks, WARPS_PER_CTA * 32, smem, kin, vin, kout, vout, n);
}

template <class E>
bool kernel_desc_tile(int id, KernelDesc *k)
{
    const size_t smem = WARPS_PER_CTA * size_t(E::NP) * TILE * 4;
    switch (id) {
    case BCF_KID_TILE_SORT: *k = {(const void *)tile_sort_kernel<E>, smem, WARPS_PER_CTA * 32}; return true;
    case BCF_KID_TILE_MERGESORT: *k = {(const void *)tile_mergesort_kernel<E>, smem, WARPS_PER_CTA * 32}; return true;
    }
    return false;
}

template bcf_status launch_tile_sort<E_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, size_t, int);
template bool kernel_desc_tile<E_U32>(int, KernelDesc *);
template bcf_status launch_tile_sort<E_U32_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, size_t, int);
template bool kernel_desc_tile<E_U32_U32>(int, KernelDesc *);
template bcf_status launch_tile_sort<E_U64>(const Call &, const void *, const uint32_t *, void *, uint32_t *, size_t, int);
template bool kernel_desc_tile<E_U64>(int, KernelDesc *);
template bcf_status launch_tile_sort<E_U64_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, size_t, int);
template bool kernel_desc_tile<E_U64_U32>(int, KernelDesc *);

}  // namespace bcf
