// bcf_pagewise.cuh -- hot-path row a7: BINARY-MERGE, the page-wise streaming merge of
// PAPER.md Algorithm 6 (L457-490, L127, L416-420), one warp per pair of runs.
//
// The warp keeps a page S of M = 1024 elements on chip.  S[0..M/2) is the page just loaded from
// the stream `e` whose previous page ended smaller; S[M/2..M) is the upper half kept from the
// previous merge.  SHEARSORT-MERGE(S) (bcf_kernels.cuh, reading A8) merges them, the lower half is
// written out, the upper half stays.  Sequential per pair: this kernel only fills
// the machine while there are many pairs; bcf_merge_runs (partition + share merge) is the
// production path.  Line numbers in comments are PAPER.md's.
#pragma once
#include "bcf_kernels.cuh"

namespace bcf {

template <int NP>
__device__ __forceinline__ bool planes_lt(const uint32_t (&x)[NP], const uint32_t (&y)[NP])
{
    bool lt = false, eq = true;
#pragma unroll
    for (int p = 0; p < NP; ++p) {
        lt = lt || (eq && x[p] < y[p]);
        eq = eq && (x[p] == y[p]);
    }
    return lt;
}

// Element g of a stream as planes (uniform address: every lane reads the same element).
template <class E>
__device__ __forceinline__ void load_scalar(const void *keys, const uint32_t *vals, const size_t g, uint32_t (&x)[E::NP])
{
    if constexpr (E::KEY_WORDS == 1) {
        x[0] = static_cast<const uint32_t *>(keys)[g];
    } else {
        const uint2 t = reinterpret_cast<const uint2 *>(keys)[g];
        x[0] = t.y;
        x[1] = t.x;
    }
    if constexpr (E::HAS_VAL) x[E::KEY_WORDS] = vals[g];
}

// Write rows [row0, row0 + 16) of the sorted page (held in the skewed planes) to out[oc ..),
// never past `total` (padding is not written, L141, L420).
template <class E>
__device__ __forceinline__ void emit_half(const uint32_t *planes, const int row0, void *kout, uint32_t *vout,
                                          const size_t obase, const size_t oc, const size_t total, const int lane)
{
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const size_t o = oc + 32 * k + lane;
        if (o < total) {
            const int w = elem_word(row0 + k, lane);
            if constexpr (E::KEY_WORDS == 1) static_cast<uint32_t *>(kout)[obase + o] = planes[w];
            else reinterpret_cast<uint2 *>(kout)[obase + o] = make_uint2(planes[TILE + w], planes[w]);
            if constexpr (E::HAS_VAL) vout[obase + o] = planes[E::KEY_WORDS * TILE + w];
        }
    }
}

template <class E>
__global__ void __launch_bounds__(WARPS_PER_CTA * 32)
pagewise_merge_kernel(const void *__restrict__ kin, const uint32_t *__restrict__ vin,
                      void *__restrict__ kout, uint32_t *__restrict__ vout, const size_t n, const size_t run_len)
{
    pdl_entry();
    constexpr int NP = E::NP;
    constexpr int H = TILE / 2;
    extern __shared__ __align__(16) uint32_t smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    uint32_t *planes = smem + warp * (NP * TILE);
    const size_t pair = static_cast<size_t>(blockIdx.x) * WARPS_PER_CTA + warp;
    const size_t a0 = pair * 2 * run_len;
    if (a0 >= n) return;
    // two scalars and a select per stream quantity: an array indexed by the runtime stream number `e`
    // would live in local memory
    const size_t len0 = min(run_len, n - a0);
    const size_t start0 = a0;
    const size_t start1 = a0 + len0;
    const size_t len1 = min(run_len, n - start1);
    size_t ic0 = 0, ic1 = 0;
    const size_t total = len0 + len1;
    size_t oc = 0;
    int e;

    uint32_t v[NP][32];
    uint32_t last_new[NP], top[NP];

    // L464: load a page of M/2 keys from each input stream into S (second page reversed, A8).
#pragma unroll
    for (int k = 0; k < 16; ++k) {
        const size_t q = 32 * k + lane;
        if (q < len0) load_elem<E>(kin, vin, start0 + q, v, k);
        else set_sentinel<E>(v, k);
    }
#pragma unroll
    for (int k = 16; k < 32; ++k) {
        const size_t q = TILE - 1 - (32 * k + lane);
        if (q < len1) load_elem<E>(kin, vin, start1 + q, v, k);
        else set_sentinel<E>(v, k);
    }
    ic0 = min(static_cast<size_t>(H), len0);
    ic1 = min(static_cast<size_t>(H), len1);
    // L466-468: the stream whose page will be exhausted first (e = 0 restored, reading A9).
    {
        uint32_t s0[NP], s1[NP];
#pragma unroll
        for (int p = 0; p < NP; ++p) s0[p] = s1[p] = SENTINEL;
        if (len0 >= static_cast<size_t>(H)) load_scalar<E>(kin, vin, start0 + H - 1, s0);
        if (len1 >= static_cast<size_t>(H)) load_scalar<E>(kin, vin, start1 + H - 1, s1);
        e = planes_lt<NP>(s1, s0) ? 1 : 0;           // S[M/2-1] <= S[M-1]  ->  e = 0
    }

    bool more = true;
    while (true) {
        // SHEARSORT-MERGE(S), L470 / L484
        line_bitonic_merge<NP>(v);
        __syncwarp();                                // upper-half reads of this round are done
#pragma unroll
        for (int p = 0; p < NP; ++p) col_store<false>(planes + p * TILE, v[p], lane);
        __syncwarp();
#pragma unroll
        for (int p = 0; p < NP; ++p) row_load(planes + p * TILE, v[p], lane);
        line_bitonic_merge<NP>(v);
#pragma unroll
        for (int p = 0; p < NP; ++p) row_store(planes + p * TILE, v[p], lane);
#pragma unroll
        for (int p = 0; p < NP; ++p) top[p] = __shfl_sync(0xFFFFFFFFu, v[p][31], 31);   // S[M-1]
        __syncwarp();
        // L472 / L486-487: write the lower half to the output stream.
        emit_half<E>(planes, 0, kout, vout, a0, oc, total, lane);
        oc += H;

        // L475: WHILE (ic[0] < n) OR (ic[1] < n)
        more = (ic0 < len0) || (ic1 < len1);
        if (!more) break;
        if ((e ? ic1 : ic0) >= (e ? len1 : len0)) e = 1 - e;              // L478
        const size_t len_e = e ? len1 : len0, ic_e = e ? ic1 : ic0, start_e = e ? start1 : start0;
        const size_t ls = min(static_cast<size_t>(H), len_e - ic_e);   // L420
        // L479: S[0..M/2) = next page of stream e (padded with infinity)
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const size_t q = 32 * k + lane;
            if (q < ls) load_elem<E>(kin, vin, start_e + ic_e + q, v, k);
            else set_sentinel<E>(v, k);
        }
#pragma unroll
        for (int p = 0; p < NP; ++p) last_new[p] = SENTINEL;
        if (ls == static_cast<size_t>(H)) load_scalar<E>(kin, vin, start_e + ic_e + H - 1, last_new);
        if (e) ic1 += ls; else ic0 += ls;            // L480
        if (planes_lt<NP>(top, last_new)) e = 1 - e; // L482: IF S[M/2-1] > S[M-1]
        // the kept upper half, reversed behind the new page: position 32k + lane, k >= 16, holds
        // sorted element (47 - k, 31 - lane); one shared-memory line per k -> conflict-free.
#pragma unroll
        for (int p = 0; p < NP; ++p) {
#pragma unroll
            for (int k = 16; k < 32; ++k) v[p][k] = planes[p * TILE + elem_word(47 - k, 31 - lane)];
        }
    }
    // L489: write the final remaining page.
    emit_half<E>(planes, 16, kout, vout, a0, oc, total, lane);
}

}  // namespace bcf
