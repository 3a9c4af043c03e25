// bcf_tu_buckets.cu -- translation unit of the paper's bucket distribution FIND-BUCKETS (bcf_buckets.cuh), the
// final merge phase inside the buckets (bcf_pieces.cuh) and the coloured prefix sums (bcf_colored_scan.cuh).
#include "bcf_internal.cuh"
#include "bcf_buckets.cuh"
#include "bcf_pieces.cuh"
#include "bcf_colored_scan.cuh"

namespace bcf {

bcf_status launch_buckets_sample(const Call &c, const void *kin, void *samples, const BucketsGeom &g, bcf_key_t kt)
{
    const size_t ns = (size_t)g.s * g.t;
    const unsigned blocks = static_cast<unsigned>((ns + 255) / 256);
    LaunchTimer tm(BCF_KERNEL_PARTITION, c.s);
    return kt == BCF_KEY_U64 ? launch(c, buckets::sample_kernel<2>, blocks, 256, 0, kin, samples, g)
                             : launch(c, buckets::sample_kernel<1>, blocks, 256, 0, kin, samples, g);
}

// ranks of the pivots (Alg. 7), offsets (L512-513), pieces moved bucket by bucket (L515-520)
bcf_status launch_buckets_distribute(const Call &c, const void *kin, const void *sorted_samples, void *pivots, uint32_t *bounds,
                                     uint32_t *piece_offsets, void *kout, const BucketsGeom &g, bcf_key_t kt)
{
    const bool k64 = (kt == BCF_KEY_U64);
    bcf_status st;
    {
        const size_t work = (size_t)g.s * (g.P - 1);
        const unsigned blocks = static_cast<unsigned>((work + 127) / 128);
        LaunchTimer tm(BCF_KERNEL_PARTITION, c.s);
        st = k64 ? launch(c, buckets::rank_kernel<2>, blocks, 128, 0, kin, sorted_samples, pivots, bounds, g)
                 : launch(c, buckets::rank_kernel<1>, blocks, 128, 0, kin, sorted_samples, pivots, bounds, g);
        if (st != BCF_OK) return st;
    }
    {
        LaunchTimer tm(BCF_KERNEL_PARTITION, c.s);
        st = launch(c, buckets::offsets_kernel, 1, buckets::SCAN_THREADS, 0, static_cast<const uint32_t *>(bounds), piece_offsets, g);
        if (st != BCF_OK) return st;
    }
    const size_t chunks = ((g.run_len + buckets::SCATTER_CHUNK - 1) / buckets::SCATTER_CHUNK) * g.s;
    const size_t cap = static_cast<size_t>(c.dev.num_sms) * 64;
    const unsigned blocks = static_cast<unsigned>(chunks < cap ? chunks : cap);
    LaunchTimer tm(BCF_KERNEL_MERGE, c.s);
    return k64 ? launch(c, buckets::scatter_kernel<2>, blocks, 256, 0, kin, kout, static_cast<const uint32_t *>(bounds),
                        static_cast<const uint32_t *>(piece_offsets), g)
               : launch(c, buckets::scatter_kernel<1>, blocks, 256, 0, kin, kout, static_cast<const uint32_t *>(bounds),
                        static_cast<const uint32_t *>(piece_offsets), g);
}

template <class E>
static bcf_status merge_pieces_rounds(const Call &c, const void *kin, void *kout, void *ktmp, size_t n, const uint32_t *Q, size_t groups,
                                      size_t s, int copy_odd, uint32_t *first)
{
    const size_t smem = WARPS_PER_CTA * size_t(E::NP) * TILE * 4;
    bcf_status st = ensure_dyn_smem<pieces::merge_pieces_kernel<E>>(c.dev, smem);
    if (st != BCF_OK) return st;
    const int rounds = ceil_log2(s);
    const void *src = kin;
    unsigned block = 1;
    for (int i = 1; i <= rounds; ++i, block *= 2) {
        void *dst = ((rounds - i) % 2 == 0) ? kout : ktmp;
        pieces::Geom g;
        g.groups = groups;
        g.s = static_cast<unsigned>(s);
        g.block = block;
        g.ppg = static_cast<unsigned>((s + 2 * size_t(block) - 1) / (2 * size_t(block)));
        g.copy_odd = copy_odd;
        {
            LaunchTimer t(BCF_KERNEL_PARTITION, c.s);
            st = launch(c, pieces::pages_scan_kernel, 1, pieces::SCAN_THREADS, 0, Q, first, g);
            if (st != BCF_OK) return st;
        }
        const size_t max_pages = n / TILE + groups * g.ppg + 1;
        const size_t cap = static_cast<size_t>(c.dev.num_sms) * 16;
        const size_t want = (max_pages + WARPS_PER_CTA - 1) / WARPS_PER_CTA;
        LaunchTimer t(BCF_KERNEL_MERGE, c.s);
        st = launch(c, pieces::merge_pieces_kernel<E>, static_cast<unsigned>(want < cap ? want : cap), WARPS_PER_CTA * 32, smem, src,
                    dst, Q, static_cast<const uint32_t *>(first), g);
        if (st != BCF_OK) return st;
        src = dst;
    }
    return BCF_OK;
}

bcf_status launch_merge_pieces_rounds(const Call &c, const void *kin, void *kout, void *ktmp, size_t n, const uint32_t *Q,
                                      size_t groups, size_t s, int copy_odd, uint32_t *first, bcf_key_t kt)
{
    if (kt == BCF_KEY_U64) return merge_pieces_rounds<E_U64>(c, kin, kout, ktmp, n, Q, groups, s, copy_odd, first);
    return merge_pieces_rounds<E_U32>(c, kin, kout, ktmp, n, Q, groups, s, copy_odd, first);
}

bool kernel_desc_pieces(int id, bcf_key_t kt, KernelDesc *k)
{
    if (id != BCF_KID_MERGE_PIECES) return false;
    if (kt == BCF_KEY_U64) *k = {(const void *)pieces::merge_pieces_kernel<E_U64>, WARPS_PER_CTA * size_t(2) * TILE * 4, WARPS_PER_CTA * 32};
    else *k = {(const void *)pieces::merge_pieces_kernel<E_U32>, WARPS_PER_CTA * size_t(1) * TILE * 4, WARPS_PER_CTA * 32};
    return true;
}

// ------------------------------------------------------------------ coloured prefix sums (App. A)

unsigned colored_scan_grid(size_t n)
{
    const size_t pages = (n + cscan::PAGE - 1) / cscan::PAGE;
    const size_t ctas = (pages + cscan::WARPS - 1) / cscan::WARPS;
    return static_cast<unsigned>(ctas < 2048 ? ctas : 2048);
}

size_t colored_scan_workspace_bytes(size_t n)
{
    return align_up(size_t(colored_scan_grid(n)) * cscan::WARPS * cscan::MAX_COLORS * 4, 256);
}

int colored_scan_max_colors() { return cscan::MAX_COLORS; }

bcf_status launch_colored_scan(const Call &c, const uint32_t *values, const uint8_t *colors, size_t n, int num_colors, bool cf,
                               uint32_t *partial, uint32_t *out)
{
    const unsigned grid = colored_scan_grid(n);
    const unsigned long long warps = static_cast<unsigned long long>(grid) * cscan::WARPS;
    bcf_status st;
    {
        LaunchTimer t(BCF_KERNEL_PARTITION, c.s);
        st = cf ? launch(c, cscan::reduce_kernel<true>, grid, cscan::WARPS * 32, 0, values, colors, n, num_colors, partial)
                : launch(c, cscan::reduce_kernel<false>, grid, cscan::WARPS * 32, 0, values, colors, n, num_colors, partial);
        if (st != BCF_OK) return st;
    }
    {
        LaunchTimer t(BCF_KERNEL_PARTITION, c.s);
        st = launch(c, cscan::offsets_kernel, 1, cscan::MAX_COLORS * 32, 0, partial, warps, num_colors);
        if (st != BCF_OK) return st;
    }
    LaunchTimer t(BCF_KERNEL_MERGE, c.s);
    return cf ? launch(c, cscan::scan_kernel<true>, grid, cscan::WARPS * 32, 0, values, colors, n, num_colors,
                       static_cast<const uint32_t *>(partial), out)
              : launch(c, cscan::scan_kernel<false>, grid, cscan::WARPS * 32, 0, values, colors, n, num_colors,
                       static_cast<const uint32_t *>(partial), out);
}

}  // namespace bcf
