// bcf_core.cuh -- register-resident lines, compare-exchange networks and the conflict-free
// shared-memory sweeps shared by the tile-sort and merge kernels.
//
// An element is NP 32-bit "planes" compared lexicographically in plane order:
//      (u32 key)            NP = 1 : {key}
//      (u32 key, u32 val)   NP = 2 : {key, val}
//      (u64 key)            NP = 2 : {key_hi, key_lo}
//      (u64 key, u32 val)   NP = 3 : {key_hi, key_lo, val}
// A thread owns one LINE (a logical row or column of the 32 x 32 tile): 32 elements held in
// registers v[p][0..31].  Every register index below is a compile-time constant after
// unrolling ("the indices for accessing registers ... do not depend on the thread
// index and the data is not transferred to local memory").  In shared memory each plane is its
// own 4 KiB array of 4-byte words, so the paper's w = 32 four-byte-bank argument applies to
// every plane verbatim.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "bcf_layout.cuh"

namespace bcf {

template <int KW, bool HV>
struct Elem {
    static constexpr int KEY_WORDS = KW;           // 1: u32 key, 2: u64 key
    static constexpr bool HAS_VAL = HV;
    static constexpr int NP = KW + (HV ? 1 : 0);   // planes
    static constexpr int KEY_BYTES = 4 * KW;
};

// ------------------------------------------------------------------ compare-exchange

// After the call element i <= element j in the lexicographic plane order.
template <int NP>
__device__ __forceinline__ void ce(uint32_t (&v)[NP][32], const int i, const int j)
{
    if constexpr (NP == 1) {
        const uint32_t a = v[0][i], b = v[0][j];
        v[0][i] = min(a, b);
        v[0][j] = max(a, b);
    } else {
        const uint64_t x = (static_cast<uint64_t>(v[0][i]) << 32) | v[1][i];
        const uint64_t y = (static_cast<uint64_t>(v[0][j]) << 32) | v[1][j];
        bool sw = x > y;
        if constexpr (NP == 3) sw = sw || (x == y && v[2][i] > v[2][j]);
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const uint32_t a = v[p][i], b = v[p][j];
            v[p][i] = sw ? b : a;
            v[p][j] = sw ? a : b;
        }
    }
}

// ------------------------------------------------------------------ Batcher's odd-even mergesort
// PAPER.md:L111, L317 "BATCHERS-ODD-EVEN-MERGESORT(R)" on the 32 registers of one line
// (191 compare-exchanges, depth 15).  Template recursion = full unrolling.

template <int NP, int LO, int N, int R>
struct OddEvenMerge {
    static __device__ __forceinline__ void run(uint32_t (&v)[NP][32])
    {
        constexpr int M = R * 2;
        if constexpr (M < N) {
            OddEvenMerge<NP, LO, N, M>::run(v);
            OddEvenMerge<NP, LO + R, N, M>::run(v);
#pragma unroll
            for (int i = LO + R; i + R < LO + N; i += M) ce<NP>(v, i, i + R);
        } else {
            ce<NP>(v, LO, LO + R);
        }
    }
};

template <int NP, int LO, int N>
struct OddEvenMergeSort {
    static __device__ __forceinline__ void run(uint32_t (&v)[NP][32])
    {
        if constexpr (N > 1) {
            OddEvenMergeSort<NP, LO, N / 2>::run(v);
            OddEvenMergeSort<NP, LO + N / 2, N / 2>::run(v);
            OddEvenMerge<NP, LO, N, 1>::run(v);
        }
    }
};

// Sort the 32 elements of a line ascending.
template <int NP>
__device__ __forceinline__ void line_sort(uint32_t (&v)[NP][32])
{
    OddEvenMergeSort<NP, 0, 32>::run(v);
}

// The last five stages (strides 16, 8, 4, 2, 1) of a bitonic merger applied to a line that is a
// bitonic sequence: 80 compare-exchanges, depth 5.  Used by SHEARSORT-MERGE (reading A8): with
// the second piece stored reversed every column and then every row of the page is bitonic, so
// the line "sort" of PAPER.md:L129 needs only a merger.
template <int NP>
__device__ __forceinline__ void line_bitonic_merge(uint32_t (&v)[NP][32])
{
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
#pragma unroll
        for (int k = 0; k < 32; ++k)
            if ((k & s) == 0) ce<NP>(v, k, k + s);
    }
}

// ------------------------------------------------------------------ shared-memory sweeps
// `pl` points at one plane (1024 words) of the calling warp's tile.  All addresses are computed
// from the lane; all register indices are constants.

// thread `r` = logical row r: eight 16-byte chunks (STS.128 / LDS.128), conflict-free per
// quarter-warp (bcf_layout.cuh).
__device__ __forceinline__ void row_store(uint32_t *pl, const uint32_t (&v)[32], const int r)
{
#pragma unroll
    for (int q = 0; q < 8; ++q)
        *reinterpret_cast<uint4 *>(pl + chunk_word(r, q)) =
            make_uint4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]);
}

__device__ __forceinline__ void row_load(const uint32_t *pl, uint32_t (&v)[32], const int r)
{
#pragma unroll
    for (int q = 0; q < 8; ++q) {
        const uint4 t = *reinterpret_cast<const uint4 *>(pl + chunk_word(r, q));
        v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
    }
}

// thread `c` = logical column c: 32 single words, row k of the access touches the 32 words of
// line k in a permuted order.  MIRROR: rows of odd index are read/written at column 31 - c,
// which realises the alternating row direction of ShearSort without
// reversing registers; the thread writes back exactly the words it read.
template <bool MIRROR>
__device__ __forceinline__ void col_load(const uint32_t *pl, uint32_t (&v)[32], const int c)
{
#pragma unroll
    for (int k = 0; k < 32; ++k) v[k] = pl[elem_word(k, MIRROR ? mirrored_col(k, c) : c)];
}

template <bool MIRROR>
__device__ __forceinline__ void col_store(uint32_t *pl, const uint32_t (&v)[32], const int c)
{
#pragma unroll
    for (int k = 0; k < 32; ++k) pl[elem_word(k, MIRROR ? mirrored_col(k, c) : c)] = v[k];
}

}  // namespace bcf
