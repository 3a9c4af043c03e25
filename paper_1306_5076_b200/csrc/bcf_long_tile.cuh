// bcf_long_tile.cuh -- long tiles: M = h * w^2 elements sorted by the h warps of one CTA in shared
// memory (section 3.1, Appendix E: "for any integer h
// that divides w, we can sort M = w^2 h elements using h warps of a CTA").
//
// The paper views the data as a w x (w h) matrix and sorts its long rows with a nested "Segmented
// ShearSort" after re-packing them by transposes (Alg. 3-5).  What still holds on sm_100a is the
// idea -- h warps, each owning one w x w tile in registers / conflict-free shared memory, combine
// their tiles without ever leaving the chip -- but not the nested ShearSort, which would cost
// ~6 x 6 full line sorts.  Here every warp sorts its own tile (tile mergesort, bcf_kernels.cuh) and
// the h sorted tiles are then merged pairwise, log2 h rounds, with the page merge of PAPER.md:L129
// in its data-oblivious form (reading A8: second piece reversed => bitonic => mergers only):
//
//   round B = 2, 4, .., h (blocks of B tiles, each block = two sorted halves of B/2 tiles):
//     * flip stage: tile i of the block meets tile B-1-i, position p meets position 1023-p; the lower
//       tile keeps the smaller element of every pair, the upper tile the larger;
//     * half-cleaner stages for tile strides B/4 .. 1: tile i meets tile i ^ stride, position p meets
//       position p;
//     * now every tile holds a bitonic sequence and the tiles are in order: column pass and row pass
//       of SHEARSORT-MERGE inside each tile (2 x 80 comparators per thread).
//   A cross-tile stage costs one min OR max per element: the warp writes its rows to an exchange set
//   (8 STS.128), one CTA barrier, reads the partner's rows (8 LDS.128, row 31-r and registers reversed
//   for the flip) -- all conflict-free by the same layout argument as row_store / row_load.
#pragma once
#include "bcf_kernels.cuh"

#ifndef BCF_LT_MINB8
#define BCF_LT_MINB8 2
#endif
// share of the max outputs formed on the FMA pipe (bcf_core.cuh ce<>): with 8 warps in lock step per
// CTA this kernel is bound by the ALU pipe, so the offload pays here (A/B in DESIGN.md 5.7)
#ifndef BCF_LT_FMA_MOD
#define BCF_LT_FMA_MOD 2
#endif

namespace bcf {

// this thread's element k of row `lane` against the partner tile's element at the same (or flipped)
// position: keep the smaller (LOW) or the larger one.
template <class E, bool FLIP, bool LOW>
__device__ __forceinline__ void cross_stage_keep(const uint32_t *partner, const int lane, uint32_t (&v)[E::NP][32])
{
    constexpr int NP = E::NP;
    const int row = FLIP ? 31 - lane : lane;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        uint32_t w[NP][4];
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const uint4 t = *reinterpret_cast<const uint4 *>(partner + p * TILE + chunk_word(row, FLIP ? 7 - q : q));
            if (FLIP) { w[p][0] = t.w; w[p][1] = t.z; w[p][2] = t.y; w[p][3] = t.x; }
            else { w[p][0] = t.x; w[p][1] = t.y; w[p][2] = t.z; w[p][3] = t.w; }
        }
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int k = 4 * q + e;
            if constexpr (NP == 1) {
                v[0][k] = LOW ? min(v[0][k], w[0][e]) : max(v[0][k], w[0][e]);
            } else {
                // mine > other, lexicographic over the planes
                bool gt = false, eq = true;
#pragma unroll
                for (int p = 0; p < NP; ++p) {
                    gt = gt || (eq && v[p][k] > w[p][e]);
                    eq = eq && v[p][k] == w[p][e];
                }
                const bool take = LOW ? gt : !(gt || eq);   // replace mine by the other element
#pragma unroll
                for (int p = 0; p < NP; ++p) v[p][k] = take ? w[p][e] : v[p][k];
            }
        }
    }
}

// Two sets of planes used alternately: the barrier of stage s + 1 also tells that every read of
// stage s is over, so the set written in stage s can be overwritten in stage s + 2 -- one CTA
// barrier per stage.
template <class E, bool FLIP>
__device__ __forceinline__ void cross_stage(uint32_t *set, const int warp, const int partner, const bool low, const int lane,
                                            uint32_t (&v)[E::NP][32])
{
    uint32_t *mine = set + warp * (E::NP * TILE);
#pragma unroll
    for (int p = 0; p < E::NP; ++p) row_store(mine + p * TILE, v[p], lane);
    __syncthreads();
    const uint32_t *other = set + partner * (E::NP * TILE);
    if (low) cross_stage_keep<E, FLIP, true>(other, lane, v);
    else cross_stage_keep<E, FLIP, false>(other, lane, v);
}

// column pass + row pass on a tile that holds a bitonic sequence in row registers
template <class E>
__device__ __forceinline__ void tile_bitonic_merge(uint32_t *planes, const int lane, uint32_t (&v)[E::NP][32])
{
#pragma unroll
    for (int p = 0; p < E::NP; ++p) row_store(planes + p * TILE, v[p], lane);
    __syncwarp();
#pragma unroll
    for (int p = 0; p < E::NP; ++p) col_load<false>(planes + p * TILE, v[p], lane);
    line_bitonic_merge<E::NP, BCF_LT_FMA_MOD>(v);
#pragma unroll
    for (int p = 0; p < E::NP; ++p) col_store<false>(planes + p * TILE, v[p], lane);
    __syncwarp();
#pragma unroll
    for (int p = 0; p < E::NP; ++p) row_load(planes + p * TILE, v[p], lane);
    line_bitonic_merge<E::NP, BCF_LT_FMA_MOD>(v);
}

// The LAST cross-tile stage of a round with the exchange doubling as the row -> column transpose of the tile merge
// that follows: the warp writes its rows to the exchange set as before, and after the barrier thread c reads BOTH
// tiles in the column layout -- its own position 32 k + c and the partner's (for the flip: position 1023 - p, i.e.
// row 31 - k, column 31 - c; for a fixed k one row in a permuted order, 32 distinct banks) -- and keeps the smaller
// or the larger element.  The result is the column registers the column pass needs, so the row_store + col_load of
// tile_bitonic_merge (one of this kernel's shared-memory sweeps per element and round) is not needed.
#ifndef BCF_LT_FUSED_TRANSPOSE
#define BCF_LT_FUSED_TRANSPOSE 1
#endif
template <class E, bool FLIP, bool LOW>
__device__ __forceinline__ void cross_stage_cols_keep(const uint32_t *own, const uint32_t *partner, const int lane,
                                                      uint32_t (&v)[E::NP][32])
{
    constexpr int NP = E::NP;
#pragma unroll
    for (int k = 0; k < 32; ++k) {
        uint32_t a[NP], b[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            a[p] = own[p * TILE + elem_word(k, lane)];
            b[p] = partner[p * TILE + (FLIP ? elem_word(31 - k, 31 - lane) : elem_word(k, lane))];
        }
        if constexpr (NP == 1) {
            v[0][k] = LOW ? min(a[0], b[0]) : max(a[0], b[0]);
        } else {
            bool gt = false, eq = true;      // mine > other, lexicographic over the planes
#pragma unroll
            for (int p = 0; p < NP; ++p) {
                gt = gt || (eq && a[p] > b[p]);
                eq = eq && a[p] == b[p];
            }
            const bool take = LOW ? gt : !(gt || eq);
#pragma unroll
            for (int p = 0; p < NP; ++p) v[p][k] = take ? b[p] : a[p];
        }
    }
}

template <class E, bool FLIP>
__device__ __forceinline__ void cross_stage_to_cols(uint32_t *set, const int warp, const int partner, const bool low, const int lane,
                                                    uint32_t (&v)[E::NP][32])
{
    uint32_t *mine = set + warp * (E::NP * TILE);
#pragma unroll
    for (int p = 0; p < E::NP; ++p) row_store(mine + p * TILE, v[p], lane);
    __syncthreads();
    const uint32_t *other = set + partner * (E::NP * TILE);
    if (low) cross_stage_cols_keep<E, FLIP, true>(mine, other, lane, v);
    else cross_stage_cols_keep<E, FLIP, false>(mine, other, lane, v);
}

// column pass + row pass on a tile that holds a bitonic sequence in COLUMN registers
template <class E>
__device__ __forceinline__ void tile_bitonic_merge_cols(uint32_t *planes, const int lane, uint32_t (&v)[E::NP][32])
{
    line_bitonic_merge<E::NP, BCF_LT_FMA_MOD>(v);
#pragma unroll
    for (int p = 0; p < E::NP; ++p) col_store<false>(planes + p * TILE, v[p], lane);
    __syncwarp();
#pragma unroll
    for (int p = 0; p < E::NP; ++p) row_load(planes + p * TILE, v[p], lane);
    line_bitonic_merge<E::NP, BCF_LT_FMA_MOD>(v);
}

template <class E, int H>
struct LongTileCfg {
    static constexpr size_t set_words = size_t(H) * E::NP * TILE;
    static constexpr size_t smem = 2 * set_words * 4;      // two exchange sets
    // resident CTAs the register cap is chosen for
    static constexpr int min_ctas = (E::NP == 1) ? (H >= 8 ? BCF_LT_MINB8 : 4) : (E::NP == 2 ? (H >= 8 ? 1 : 2) : 1);
};

template <class E, int H>
__global__ void __launch_bounds__(H * 32, LongTileCfg<E, H>::min_ctas)
long_tile_sort_kernel(const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, const size_t n)
{
    pdl_entry();
    extern __shared__ __align__(16) uint32_t smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    constexpr size_t SET = LongTileCfg<E, H>::set_words;
    // A warp's working planes (transposes inside its tile) are its own slot of the set the NEXT stage
    // writes: its last readers passed a barrier since.
    uint32_t *const slot = smem + warp * (E::NP * TILE);
    // 32-bit group / tile counters (n < 2^32): fewer live registers in the loop than size_t arithmetic
    const unsigned num_tiles = static_cast<unsigned>((n + TILE - 1) / TILE);
    const unsigned num_groups = (num_tiles + H - 1) / H;
    const unsigned full_tiles = static_cast<unsigned>(n / TILE);

    for (unsigned g = blockIdx.x; g < num_groups; g += gridDim.x) {
        const unsigned tile = g * H + warp;
        const size_t base = static_cast<size_t>(tile) * TILE;
        const int cnt = tile < full_tiles ? TILE : (tile < num_tiles ? static_cast<int>(n - base) : 0);
        uint32_t v[E::NP][32];
        if (cnt == TILE) load_tile_vec<E>(kin, vin, base, lane, v);
        else load_tile_guarded<E>(kin, vin, base, cnt, lane, v);    // missing elements: the maximum element
        line_sort<E::NP, BCF_LT_FMA_MOD>(v);
        tile_merge_level<E, 1, BCF_LT_FMA_MOD>(slot, lane, v);
        tile_merge_level<E, 2, BCF_LT_FMA_MOD>(slot, lane, v);
        tile_merge_level<E, 3, BCF_LT_FMA_MOD>(slot, lane, v);
        tile_merge_level<E, 4, BCF_LT_FMA_MOD>(slot, lane, v);
        tile_merge_level<E, 5, BCF_LT_FMA_MOD>(slot, lane, v);
        int stage = 0;
#pragma unroll
        for (int B = 2; B <= H; B *= 2) {
            const int i = warp & (B - 1);
#if BCF_LT_FUSED_TRANSPOSE
            if (B == 2) {
                cross_stage_to_cols<E, true>(smem + (stage++ & 1) * SET, warp, (warp - i) + (B - 1 - i), i < B / 2, lane, v);
            } else {
                cross_stage<E, true>(smem + (stage++ & 1) * SET, warp, (warp - i) + (B - 1 - i), i < B / 2, lane, v);
#pragma unroll
                for (int s = B / 4; s >= 2; s /= 2)
                    cross_stage<E, false>(smem + (stage++ & 1) * SET, warp, warp ^ s, (warp & s) == 0, lane, v);
                cross_stage_to_cols<E, false>(smem + (stage++ & 1) * SET, warp, warp ^ 1, (warp & 1) == 0, lane, v);
            }
            tile_bitonic_merge_cols<E>(slot + (stage & 1) * SET, lane, v);
#else
            cross_stage<E, true>(smem + (stage++ & 1) * SET, warp, (warp - i) + (B - 1 - i), i < B / 2, lane, v);
#pragma unroll
            for (int s = B / 4; s >= 1; s /= 2)
                cross_stage<E, false>(smem + (stage++ & 1) * SET, warp, warp ^ s, (warp & s) == 0, lane, v);
            tile_bitonic_merge<E>(slot + (stage & 1) * SET, lane, v);
#endif
        }
        // (storing the rows straight from the registers -- eight 16-byte stores per thread, 128 bytes apart across
        // the lanes -- would save this round trip through shared memory; measured slower, 1.71 -> 1.84 ms: the
        // half-filled store sectors cost more than the two shared-memory sweeps)
        if (cnt > 0) store_rows<E>(slot + (stage & 1) * SET, kout, vout, base, cnt, cnt == TILE, lane, v);
        __syncthreads();     // the exchange sets are reused by the CTA's next group
    }
}

}  // namespace bcf
