// bcf_tu_long.cu -- translation unit of the long-tile base case (bcf_long_tile.cuh).
#include "bcf_internal.cuh"
#include "bcf_long_tile.cuh"

namespace bcf {

template <class E, int H>
static bcf_status launch_long_tile_h(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, size_t n)
{
    using C = LongTileCfg<E, H>;
    const size_t groups = ((n + TILE - 1) / TILE + H - 1) / H;
    if (groups == 0) return BCF_OK;
    bcf_status st;
    int ctas = 0;
    if ((st = ensure_dyn_smem<long_tile_sort_kernel<E, H>>(c.dev, C::smem)) != BCF_OK) return st;
    if ((st = resident_ctas<long_tile_sort_kernel<E, H>>(c.dev, H * 32, C::smem, &ctas)) != BCF_OK) return st;
    const size_t cap = static_cast<size_t>(ctas) * c.dev.num_sms * 8;     // a few waves; the kernel strides over groups
    LaunchTimer t(BCF_KERNEL_TILE_SORT, c.s);
    return launch(c, long_tile_sort_kernel<E, H>, static_cast<unsigned>(groups < cap ? groups : cap), H * 32, C::smem, kin, vin,
                  kout, vout, n);
}

template <class E>
bcf_status launch_long_tile(const Call &c, const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, size_t n, int h)
{
    switch (h) {
    case 2: return launch_long_tile_h<E, 2>(c, kin, vin, kout, vout, n);
    case 4: return launch_long_tile_h<E, 4>(c, kin, vin, kout, vout, n);
    case 8: return launch_long_tile_h<E, 8>(c, kin, vin, kout, vout, n);
    }
    return BCF_ERR_INVALID_ARG;
}

template <class E>
bool kernel_desc_long(int id, KernelDesc *k)
{
    switch (id) {
    case BCF_KID_LONG_TILE_2: *k = {(const void *)long_tile_sort_kernel<E, 2>, LongTileCfg<E, 2>::smem, 64}; return true;
    case BCF_KID_LONG_TILE_4: *k = {(const void *)long_tile_sort_kernel<E, 4>, LongTileCfg<E, 4>::smem, 128}; return true;
    case BCF_KID_LONG_TILE_8: *k = {(const void *)long_tile_sort_kernel<E, 8>, LongTileCfg<E, 8>::smem, 256}; return true;
    }
    return false;
}

template bcf_status launch_long_tile<E_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, size_t, int);
template bool kernel_desc_long<E_U32>(int, KernelDesc *);
template bcf_status launch_long_tile<E_U32_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, size_t, int);
template bool kernel_desc_long<E_U32_U32>(int, KernelDesc *);
template bcf_status launch_long_tile<E_U64>(const Call &, const void *, const uint32_t *, void *, uint32_t *, size_t, int);
template bool kernel_desc_long<E_U64>(int, KernelDesc *);
template bcf_status launch_long_tile<E_U64_U32>(const Call &, const void *, const uint32_t *, void *, uint32_t *, size_t, int);
template bool kernel_desc_long<E_U64_U32>(int, KernelDesc *);

}  // namespace bcf
