// bcf_kernels.cuh -- the sm_100a kernels of the hot path.
//
//   tile_sort_kernel   a1-a4, a9 : ShearSort of 32 x 32 tiles, one warp per tile
//   partition_kernel   a5        : split-point (co-rank) search, one thread per output share
//   merge_kernel       a6, a8, a9: one warp per share of 1024 outputs, SHEARSORT-MERGE in registers
//
// One warp works alone on one tile/share: its 32 threads are the paper's "w threads" and own the
// 32 lines of the tile ("each thread processes a separate row of the matrix").
// Warps never talk to each other, so the only barrier in these kernels is __syncwarp(), which
// replaces the implicit lock-step the paper relies on and is required on every
// architecture since sm_70.
#pragma once
#include "bcf_core.cuh"

namespace bcf {

constexpr int WARPS_PER_CTA = 4;
constexpr uint32_t SENTINEL = 0xFFFFFFFFu;   // "infinity" in every plane (reading A10)

// ------------------------------------------------------------------ global memory access

// Every element is read once and written once per kernel: allocating those lines in L1 buys
// nothing, and the L1 data array is the SAME SRAM as shared memory, so L1 fills and write-through
// data compete with the warps' shared-memory wavefronts for its 32 banks.  Loads therefore carry
// L1::no_allocate and stores are streaming (.cs).  BCF_GMEM_HINT=0 restores the default policies
// (kept for the A/B measurement recorded in profiles/).
#ifndef BCF_GMEM_HINT
#define BCF_GMEM_HINT 1
#endif

__device__ __forceinline__ uint4 ldg128(const uint4 *p)
{
#if BCF_GMEM_HINT
    uint4 t;
    asm volatile("ld.global.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(t.x), "=r"(t.y), "=r"(t.z), "=r"(t.w) : "l"(p));
    return t;
#else
    return *p;
#endif
}
__device__ __forceinline__ uint2 ldg64(const uint2 *p)
{
#if BCF_GMEM_HINT
    uint2 t;
    asm volatile("ld.global.L1::no_allocate.v2.u32 {%0, %1}, [%2];" : "=r"(t.x), "=r"(t.y) : "l"(p));
    return t;
#else
    return *p;
#endif
}
__device__ __forceinline__ uint32_t ldg32(const uint32_t *p)
{
#if BCF_GMEM_HINT
    uint32_t t;
    asm volatile("ld.global.L1::no_allocate.u32 %0, [%1];" : "=r"(t) : "l"(p));
    return t;
#else
    return *p;
#endif
}
__device__ __forceinline__ void stg128(uint4 *p, const uint4 t)
{
#if BCF_GMEM_HINT
    __stcs(p, t);
#else
    *p = t;
#endif
}
__device__ __forceinline__ void stg64(uint2 *p, const uint2 t)
{
#if BCF_GMEM_HINT
    __stcs(p, t);
#else
    *p = t;
#endif
}
__device__ __forceinline__ void stg32(uint32_t *p, const uint32_t t)
{
#if BCF_GMEM_HINT
    __stcs(p, t);
#else
    *p = t;
#endif
}

// Element `g` of the SoA arrays into planes of register slot k.
template <class E>
__device__ __forceinline__ void load_elem(const void *keys, const uint32_t *vals, const size_t g,
                                          uint32_t (&v)[E::NP][32], const int k)
{
    if constexpr (E::KEY_WORDS == 1) {
        v[0][k] = ldg32(static_cast<const uint32_t *>(keys) + g);
    } else {
        const uint2 t = ldg64(reinterpret_cast<const uint2 *>(keys) + g);
        v[0][k] = t.y;   // high word first: planes are compared in order
        v[1][k] = t.x;
    }
    if constexpr (E::HAS_VAL) v[E::KEY_WORDS][k] = ldg32(vals + g);
}

template <class E>
__device__ __forceinline__ void set_sentinel(uint32_t (&v)[E::NP][32], const int k)
{
#pragma unroll
    for (int p = 0; p < E::NP; ++p) v[p][k] = SENTINEL;
}

// A1: whole tile, 128-bit coalesced loads.  Which 32 elements a thread receives is irrelevant:
// the first step of ShearSort is a full sort of each row and the sorted tile is unique, so every
// assignment of the tile's elements to rows gives the same result.
template <class E>
__device__ __forceinline__ void load_tile_vec(const void *keys, const uint32_t *vals, const size_t base,
                                              const int lane, uint32_t (&v)[E::NP][32])
{
    if constexpr (E::KEY_WORDS == 1) {
        const uint4 *pk = reinterpret_cast<const uint4 *>(static_cast<const uint32_t *>(keys) + base);
#pragma unroll
        for (int m = 0; m < 8; ++m) {
            const uint4 t = ldg128(pk + 32 * m + lane);
            v[0][4 * m] = t.x; v[0][4 * m + 1] = t.y; v[0][4 * m + 2] = t.z; v[0][4 * m + 3] = t.w;
        }
        if constexpr (E::HAS_VAL) {
            const uint4 *pv = reinterpret_cast<const uint4 *>(vals + base);
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const uint4 t = ldg128(pv + 32 * m + lane);
                v[1][4 * m] = t.x; v[1][4 * m + 1] = t.y; v[1][4 * m + 2] = t.z; v[1][4 * m + 3] = t.w;
            }
        }
    } else {
        const uint4 *pk = reinterpret_cast<const uint4 *>(static_cast<const uint64_t *>(keys) + base);
#pragma unroll
        for (int m = 0; m < 16; ++m) {
            const uint4 t = ldg128(pk + 32 * m + lane);   // keys 64m + 2 lane, +1
            v[0][2 * m] = t.y; v[1][2 * m] = t.x; v[0][2 * m + 1] = t.w; v[1][2 * m + 1] = t.z;
        }
        if constexpr (E::HAS_VAL) {
            const uint2 *pv = reinterpret_cast<const uint2 *>(vals + base);
#pragma unroll
            for (int m = 0; m < 16; ++m) {
                const uint2 t = ldg64(pv + 32 * m + lane);
                v[2][2 * m] = t.x; v[2][2 * m + 1] = t.y;
            }
        }
    }
}

// Partial tile (a9): element 32k + lane, padded with the sentinel past `cnt`.
template <class E>
__device__ __forceinline__ void load_tile_guarded(const void *keys, const uint32_t *vals, const size_t base,
                                                  const int cnt, const int lane, uint32_t (&v)[E::NP][32])
{
#pragma unroll
    for (int k = 0; k < 32; ++k) {
        if (32 * k + lane < cnt) load_elem<E>(keys, vals, base + 32 * k + lane, v, k);
        else set_sentinel<E>(v, k);
    }
}

// A4: thread r holds sorted logical row r.  Stage through the skewed planes (row_store), then
// every lane reads back the chunk it stores to global so that the global stores are coalesced
// 128-bit (or 64-bit) vector stores; the reads are conflict-free (bcf_layout.cuh).  This is the
// un-skew step of PAPER.md Alg. 2 L361-362 folded into the read pattern of the final store
// (reading A6: the step as printed has a 2-way conflict).
// `vec_ok`: the share is full and its global start is 16-byte aligned.
template <class E>
__device__ __forceinline__ void store_rows(uint32_t *planes, void *keys, uint32_t *vals, const size_t base,
                                           const int cnt, const bool vec_ok, const int lane,
                                           const uint32_t (&v)[E::NP][32])
{
#pragma unroll
    for (int p = 0; p < E::NP; ++p) row_store(planes + p * TILE, v[p], lane);
    __syncwarp();
    if (vec_ok) {
        if constexpr (E::KEY_WORDS == 1) {
            uint4 *pk = reinterpret_cast<uint4 *>(static_cast<uint32_t *>(keys) + base);
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int w = chunk_word(4 * m + (lane >> 3), lane & 7);
                stg128(pk + 32 * m + lane, *reinterpret_cast<const uint4 *>(planes + w));
            }
            if constexpr (E::HAS_VAL) {
                uint4 *pv = reinterpret_cast<uint4 *>(vals + base);
#pragma unroll
                for (int m = 0; m < 8; ++m) {
                    const int w = chunk_word(4 * m + (lane >> 3), lane & 7);
                    stg128(pv + 32 * m + lane, *reinterpret_cast<const uint4 *>(planes + TILE + w));
                }
            }
        } else {
            uint4 *pk = reinterpret_cast<uint4 *>(static_cast<uint64_t *>(keys) + base);
#pragma unroll
            for (int m = 0; m < 16; ++m) {
                const int w = elem_word(2 * m + (lane >> 4), 2 * (lane & 15));
                const uint2 hi = *reinterpret_cast<const uint2 *>(planes + w);
                const uint2 lo = *reinterpret_cast<const uint2 *>(planes + TILE + w);
                stg128(pk + 32 * m + lane, make_uint4(lo.x, hi.x, lo.y, hi.y));
            }
            if constexpr (E::HAS_VAL) {
                uint2 *pv = reinterpret_cast<uint2 *>(vals + base);
#pragma unroll
                for (int m = 0; m < 16; ++m) {
                    const int w = elem_word(2 * m + (lane >> 4), 2 * (lane & 15));
                    stg64(pv + 32 * m + lane, *reinterpret_cast<const uint2 *>(planes + 2 * TILE + w));
                }
            }
        }
    } else {
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            if (32 * k + lane < cnt) {
                const int w = elem_word(k, lane);
                const size_t g = base + 32 * k + lane;
                if constexpr (E::KEY_WORDS == 1) {
                    stg32(static_cast<uint32_t *>(keys) + g, planes[w]);
                } else {
                    stg64(reinterpret_cast<uint2 *>(keys) + g, make_uint2(planes[TILE + w], planes[w]));
                }
                if constexpr (E::HAS_VAL) stg32(vals + g, planes[E::KEY_WORDS * TILE + w]);
            }
        }
    }
    __syncwarp();   // the planes are reused by the warp's next tile
}

// ------------------------------------------------------------------ a1-a4: tile ShearSort
//
// PAPER.md Alg. 1 (L308-335) with the transposes removed as in section 3.3 / Alg. 2:
//   FOR i IN 1..log2(w):  row sort (alternating)   -> thread r sorts logical row r in registers
//                         column sort (ascending)  -> thread c sorts logical column c
//   clean-up row sort (ascending), store.
// Row data moves registers -> planes with 8 STS.128, planes -> column registers with 32 LDS.32
// (odd rows mirrored = descending rows), back with 32 STS.32 and 8 LDS.128; every one of these
// warp accesses hits 32 distinct banks.
template <class E>
__global__ void __launch_bounds__(WARPS_PER_CTA * 32)
tile_sort_kernel(const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, const size_t n)
{
    pdl_entry();
    extern __shared__ __align__(16) uint32_t smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    uint32_t *planes = smem + warp * (E::NP * TILE);
    const size_t num_tiles = (n + TILE - 1) / TILE;
    const size_t stride = static_cast<size_t>(gridDim.x) * WARPS_PER_CTA;

    for (size_t tile = static_cast<size_t>(blockIdx.x) * WARPS_PER_CTA + warp; tile < num_tiles; tile += stride) {
        const size_t base = tile * TILE;
        const int cnt = (n - base) < static_cast<size_t>(TILE) ? static_cast<int>(n - base) : TILE;
        uint32_t v[E::NP][32];
        if (cnt == TILE) load_tile_vec<E>(kin, vin, base, lane, v);
        else load_tile_guarded<E>(kin, vin, base, cnt, lane, v);

#pragma unroll 1
        for (int phase = 0; phase < 5; ++phase) {          // ceil(log2 32) phases (reading A2)
            line_sort<E::NP>(v);                            // rows (ascending in registers)
#pragma unroll
            for (int p = 0; p < E::NP; ++p) row_store(planes + p * TILE, v[p], lane);
            __syncwarp();
#pragma unroll
            for (int p = 0; p < E::NP; ++p) col_load<true>(planes + p * TILE, v[p], lane);
            line_sort<E::NP>(v);                            // columns, ascending
#pragma unroll
            for (int p = 0; p < E::NP; ++p) col_store<true>(planes + p * TILE, v[p], lane);
            __syncwarp();
#pragma unroll
            for (int p = 0; p < E::NP; ++p) row_load(planes + p * TILE, v[p], lane);
        }
        line_sort<E::NP>(v);                                // clean-up pass: all rows ascending
        store_rows<E>(planes, kout, vout, base, cnt, cnt == TILE, lane, v);
    }
}

// ------------------------------------------------------------------ tile mergesort (alternative base case)
//
// The same tile, the same conflict-free row <-> column movement, but the paper's own page merge
// (SHEARSORT-MERGE, in the form of reading A8) applied inside the tile instead
// of full ShearSort phases: rows are sorted once (Batcher, 191 comparators), then for T = 1..5 every
// block of 2^T rows is formed from its two sorted halves by ONE round {column pass, row pass} --
// the second half is read reversed, so every column of the block and then every row is bitonic and
// the line "sorts" are mergers (16 T + 80 comparators per thread).  831 comparators per thread
// instead of 2101, the same 10 sweeps through shared memory; the sorted tile is unique, so the
// result is bit-identical to ShearSort's.  bcf_sort_tiles stays ShearSort (row a2); this kernel is
// bcf_sort_tiles_mergesort and, by default, the base case of bcf_sort.
#ifndef BCF_TMS_FMA_MOD
#define BCF_TMS_FMA_MOD 0     // min/max only: this kernel is not bound by the ALU pipe (A/B in DESIGN.md 5.6)
#endif
// (Level T = 1 with warp shuffles instead of shared memory -- the two rows of a block live in neighbouring threads, both
// send register 31 - j and keep min / max with one predicated VIMNMX -- was built and measured in r2: 32 SHFL.BFLY in
// place of four sweeps through shared memory gain 0.5 % on the long-tile kernel; a shuffle occupies the same data
// path about as long as the wavefronts it replaces.  Not kept.)
template <class E, int T, int FM = BCF_TMS_FMA_MOD>
__device__ __forceinline__ void tile_merge_level(uint32_t *planes, const int lane, uint32_t (&v)[E::NP][32])
{
#pragma unroll
    for (int p = 0; p < E::NP; ++p) row_store(planes + p * TILE, v[p], lane);
    __syncwarp();
#pragma unroll
    for (int p = 0; p < E::NP; ++p) col_load_level<T>(planes + p * TILE, v[p], lane);
    block_bitonic_merge<E::NP, T, FM>(v);                // column pass: strides 2^(T-1) .. 1 rows
    __syncwarp();                                        // mirrored reads: another thread's words are overwritten next
#pragma unroll
    for (int p = 0; p < E::NP; ++p) col_store<false>(planes + p * TILE, v[p], lane);
    __syncwarp();
#pragma unroll
    for (int p = 0; p < E::NP; ++p) row_load(planes + p * TILE, v[p], lane);
    line_bitonic_merge<E::NP, FM>(v);                    // row pass: strides 16 .. 1
}

// resident CTAs per SM asked of the compiler (register cap), per number of planes
#ifndef BCF_TMS_MINB1
#define BCF_TMS_MINB1 4
#endif
#ifndef BCF_TMS_MINB2
#define BCF_TMS_MINB2 4
#endif
#ifndef BCF_TMS_MINB3
#define BCF_TMS_MINB3 3
#endif
template <class E>
__global__ void __launch_bounds__(WARPS_PER_CTA * 32, E::NP == 1 ? BCF_TMS_MINB1 : E::NP == 2 ? BCF_TMS_MINB2 : BCF_TMS_MINB3)
tile_mergesort_kernel(const void *kin, const uint32_t *vin, void *kout, uint32_t *vout, const size_t n)
{
    pdl_entry();
    extern __shared__ __align__(16) uint32_t smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    uint32_t *planes = smem + warp * (E::NP * TILE);
    const size_t num_tiles = (n + TILE - 1) / TILE;
    const size_t stride = static_cast<size_t>(gridDim.x) * WARPS_PER_CTA;

    for (size_t tile = static_cast<size_t>(blockIdx.x) * WARPS_PER_CTA + warp; tile < num_tiles; tile += stride) {
        const size_t base = tile * TILE;
        const int cnt = (n - base) < static_cast<size_t>(TILE) ? static_cast<int>(n - base) : TILE;
        uint32_t v[E::NP][32];
        if (cnt == TILE) load_tile_vec<E>(kin, vin, base, lane, v);
        else load_tile_guarded<E>(kin, vin, base, cnt, lane, v);
        line_sort<E::NP, BCF_TMS_FMA_MOD>(v);               // every row ascending
        tile_merge_level<E, 1>(planes, lane, v);
        tile_merge_level<E, 2>(planes, lane, v);
        tile_merge_level<E, 3>(planes, lane, v);
        tile_merge_level<E, 4>(planes, lane, v);
        tile_merge_level<E, 5>(planes, lane, v);
        store_rows<E>(planes, kout, vout, base, cnt, cnt == TILE, lane, v);
    }
}

// ------------------------------------------------------------------ a5: merge partitioning

// struct PassGeom: bcf_layout.cuh

template <class E>
__device__ __forceinline__ bool elem_le_global(const void *keys, const uint32_t *vals, const size_t ia, const size_t ib)
{
    if constexpr (E::KEY_WORDS == 1) {
        const uint32_t ka = __ldg(static_cast<const uint32_t *>(keys) + ia);
        const uint32_t kb = __ldg(static_cast<const uint32_t *>(keys) + ib);
        if constexpr (E::HAS_VAL) {
            if (ka != kb) return ka < kb;
            return __ldg(vals + ia) <= __ldg(vals + ib);
        } else {
            return ka <= kb;
        }
    } else {
        const unsigned long long ka = __ldg(static_cast<const unsigned long long *>(keys) + ia);
        const unsigned long long kb = __ldg(static_cast<const unsigned long long *>(keys) + ib);
        if constexpr (E::HAS_VAL) {
            if (ka != kb) return ka < kb;
            return __ldg(vals + ia) <= __ldg(vals + ib);
        } else {
            return ka <= kb;
        }
    }
}

// One thread per share slot: binary search on the share's first output diagonal for the unique
// split (i, d - i) with A[i-1] <= B[d-i] and B[d-i-1] < A[i] (A-first ties, include/bcf.h).
template <class E>
__global__ void __launch_bounds__(128)
partition_kernel(const void *__restrict__ kin, const uint32_t *__restrict__ vin,
                 uint32_t *__restrict__ splits, const PassGeom g)
{
    pdl_entry();
    const unsigned long long slot = static_cast<unsigned long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (slot >= g.num_shares) return;
    const unsigned long long pair = slot / g.shares_per_pair;
    const unsigned long long t = slot % g.shares_per_pair;
    const unsigned long long a0 = pair * 2ull * g.run_len;
    if (a0 >= g.n) { splits[slot] = 0; return; }
    const unsigned long long alen = min(g.run_len, g.n - a0);
    const unsigned long long b0 = a0 + alen;
    const unsigned long long blen = min(g.run_len, g.n - b0);
    const unsigned long long d = min(t * TILE, alen + blen);
    unsigned long long lo = d > blen ? d - blen : 0ull;
    unsigned long long hi = min(d, alen);
    while (lo < hi) {
        const unsigned long long mid = (lo + hi) >> 1;
        if (elem_le_global<E>(kin, vin, a0 + mid, b0 + (d - 1 - mid))) lo = mid + 1;
        else hi = mid;
    }
    splits[slot] = static_cast<uint32_t>(lo);
}

// ------------------------------------------------------------------ a6: conflict-free in-smem merge
//
// SHEARSORT-MERGE of one share: the warp's piece of A ascending followed by
// its piece of B REVERSED forms a bitonic sequence S of 1024 elements (padding, if any, sits in
// the middle as the maximum), seen as a row-major 32 x 32 page.  One ShearSort round, columns
// first: each column of S is bitonic, so the column "sort" is a 5-stage merger in the registers of
// thread c; afterwards every row is bitonic and all elements of row r are <= those of row r+1, so
// the row "sort" is a second 5-stage merger in the registers of thread r (reading A8).
//  * position 32k + lane is what a coalesced global load hands to lane `lane` in its k-th load:
//    the column layout comes straight from global memory, no shared-memory traffic;
//  * columns -> rows through the skewed planes: 32 STS.32 + 8 LDS.128 per plane, conflict-free;
//  * rows -> global through store_rows: 8 STS.128 + 8 LDS.128 + 8 STG.128 per plane.
template <class E>
__global__ void __launch_bounds__(WARPS_PER_CTA * 32)
merge_kernel(const void *__restrict__ kin, const uint32_t *__restrict__ vin,
             void *__restrict__ kout, uint32_t *__restrict__ vout,
             const uint32_t *__restrict__ splits, const PassGeom g)
{
    pdl_entry();
    extern __shared__ __align__(16) uint32_t smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    uint32_t *planes = smem + warp * (E::NP * TILE);
    const unsigned long long stride = static_cast<unsigned long long>(gridDim.x) * WARPS_PER_CTA;

    for (unsigned long long slot = static_cast<unsigned long long>(blockIdx.x) * WARPS_PER_CTA + warp;
         slot < g.num_shares; slot += stride) {
        const unsigned long long pair = slot / g.shares_per_pair;
        const unsigned int t = static_cast<unsigned int>(slot % g.shares_per_pair);
        const unsigned long long a0 = pair * 2ull * g.run_len;
        if (a0 >= g.n) continue;
        const unsigned long long alen = min(g.run_len, g.n - a0);
        const unsigned long long b0 = a0 + alen;
        const unsigned long long blen = min(g.run_len, g.n - b0);
        const unsigned long long plen = alen + blen;
        const unsigned long long d0 = static_cast<unsigned long long>(t) * TILE;
        if (d0 >= plen) continue;
        const unsigned long long d1 = min(d0 + TILE, plen);
        const unsigned long long i0 = splits[slot];
        const unsigned long long i1 = (t + 1 < g.shares_per_pair) ? splits[slot + 1] : alen;
        const int a = static_cast<int>(i1 - i0);                 // elements taken from A
        const int b = static_cast<int>((d1 - i1) - (d0 - i0));   // elements taken from B
        const size_t ga = a0 + i0;                               // first element of the A piece
        const size_t gb = b0 + (d0 - i0);                        // first element of the B piece

        uint32_t v[E::NP][32];
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            const int p = 32 * k + lane;
            if (p < a) load_elem<E>(kin, vin, ga + p, v, k);
            else if (p >= TILE - b) load_elem<E>(kin, vin, gb + (TILE - 1 - p), v, k);
            else set_sentinel<E>(v, k);
        }
        line_bitonic_merge<E::NP>(v);                            // column pass (strides 512..32)
#pragma unroll
        for (int p = 0; p < E::NP; ++p) col_store<false>(planes + p * TILE, v[p], lane);
        __syncwarp();
#pragma unroll
        for (int p = 0; p < E::NP; ++p) row_load(planes + p * TILE, v[p], lane);
        line_bitonic_merge<E::NP>(v);                            // row pass (strides 16..1)

        const size_t out = a0 + d0;
        const int cnt = static_cast<int>(d1 - d0);
        const bool vec_ok = (cnt == TILE) && ((out * E::KEY_BYTES) % 16 == 0) &&
                            (!E::HAS_VAL || (out * 4) % 16 == 0);
        store_rows<E>(planes, kout, vout, out, cnt, vec_ok, lane, v);
    }
}

}  // namespace bcf
