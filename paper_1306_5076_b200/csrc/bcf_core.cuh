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

// struct Elem<KEY_WORDS, HAS_VAL>: bcf_layout.cuh

// ------------------------------------------------------------------ programmatic dependent launch
// Every kernel of the library starts with pdl_entry(): it waits until the grids it depends on have completed and
// their writes are visible (griddepcontrol.wait) -- before its first access to global memory.  With the launch
// attribute (bcf_options.launch_mode = BCF_LAUNCH_PDL) the kernel's CTAs are scheduled as soon as the CTAs of
// its predecessor have exited, so the launch latency overlaps the predecessor's drain; without it the
// instruction does nothing.  No kernel triggers its dependents early (griddepcontrol.launch_dependents):
// measured on B200, dependents that sit on the SMs while a merge pass runs slow it down.
#ifndef BCF_PDL_EARLY_TRIGGER
#define BCF_PDL_EARLY_TRIGGER 0
#endif
__device__ __forceinline__ void pdl_entry()
{
#if BCF_PDL_EARLY_TRIGGER
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// ------------------------------------------------------------------ compare-exchange
//
// Pipe balance (measured on B200): integer min/max, compare, select and add/sub with
// carry all issue on the ALU pipe (16 lanes / clk / SM sub-partition), integer multiply-add on the
// FMA pipe.  A compare-exchange written with ALU instructions only leaves the FMA pipe idle, so part
// of the "larger" outputs are formed as  hi = a + b - lo  (mod 2^32, exact) with two IMADs whose
// multiplier comes from constant memory -- opaque to ptxas, which would otherwise turn them back
// into ALU adds.
static __constant__ uint32_t c_one = 1u;            // one copy per translation unit
static __constant__ uint32_t c_minus_one = 0xFFFFFFFFu;

// a + b - lo on the FMA pipe (lo is one of a, b; the result is the other one).
__device__ __forceinline__ uint32_t other_of(const uint32_t a, const uint32_t b, const uint32_t lo)
{
    uint32_t s, hi;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(s) : "r"(a), "r"(c_one), "r"(b));
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(hi) : "r"(lo), "r"(c_minus_one), "r"(s));
    return hi;
}

// x > y for elements of NP planes compared lexicographically: one subtract-with-borrow chain from
// the least significant plane up (NP ALU instructions).
template <int NP>
__device__ __forceinline__ bool elem_gt(const uint32_t (&v)[NP][32], const int i, const int j)
{
    uint32_t bo;
    if constexpr (NP == 2) {
        asm("{\n .reg .u32 t;\n sub.cc.u32 t, %2, %1;\n subc.cc.u32 t, %4, %3;\n subc.u32 %0, 0, 0;\n}"
            : "=r"(bo) : "r"(v[1][i]), "r"(v[1][j]), "r"(v[0][i]), "r"(v[0][j]));
    } else {
        asm("{\n .reg .u32 t;\n sub.cc.u32 t, %2, %1;\n subc.cc.u32 t, %4, %3;\n subc.cc.u32 t, %6, %5;\n"
            " subc.u32 %0, 0, 0;\n}"
            : "=r"(bo) : "r"(v[2][i]), "r"(v[2][j]), "r"(v[1][i]), "r"(v[1][j]), "r"(v[0][i]), "r"(v[0][j]));
    }
    return bo != 0;
}

// Tuning knobs (A/B measured on B200 in the real kernels, where register pressure limits what the
// micro-benchmark promises; the defaults are the fastest):
//   BCF_CE1_FMA_MOD     keys-only: comparator (i, j) forms its max on the FMA pipe when i % MOD != 0 (0: never)
//   BCF_CE2_FMA_PLANES  two-plane elements: the last this-many planes form their "larger" output on the FMA pipe
//   BCF_CE3_FMA_PLANES  same for three-plane elements
#ifndef BCF_CE1_FMA_MOD
#define BCF_CE1_FMA_MOD 3
#endif
#ifndef BCF_CE2_FMA_PLANES
#define BCF_CE2_FMA_PLANES 1
#endif
#ifndef BCF_CE3_FMA_PLANES
#define BCF_CE3_FMA_PLANES 0
#endif

// After the call element i <= element j in the lexicographic plane order.
// FMOD: keys-only comparator (i, j) forms its max on the FMA pipe when i % FMOD != 0 (0: never).  The
// default suits the ALU-bound ShearSort and the merge kernels; the tile mergesort, which is bound by
// issue slots and shared-memory latency instead, passes 0 (fewer instructions).
template <int NP, int FMOD = BCF_CE1_FMA_MOD>
__device__ __forceinline__ void ce(uint32_t (&v)[NP][32], const int i, const int j)
{
    if constexpr (NP == 1) {
        const uint32_t a = v[0][i], b = v[0][j];
        const uint32_t lo = min(a, b);
        v[0][i] = lo;
        // FMOD > 0: comparators with i % FMOD != 0; FMOD < 0: comparators with i % -FMOD == 0 (a smaller share)
        const bool fma = FMOD > 0 ? (i % (FMOD > 0 ? FMOD : 1)) != 0 : (FMOD < 0 && (i % (FMOD < 0 ? -FMOD : 1)) == 0);
        v[0][j] = fma ? other_of(a, b, lo) : max(a, b);
    } else {
        const bool sw = elem_gt<NP>(v, i, j);
#pragma unroll
        for (int p = 0; p < NP; ++p) {
            const uint32_t a = v[p][i], b = v[p][j];
            const uint32_t lo = sw ? b : a;
            v[p][i] = lo;
            constexpr int FMA_PLANES = (NP == 2) ? BCF_CE2_FMA_PLANES : BCF_CE3_FMA_PLANES;
            v[p][j] = (p >= NP - FMA_PLANES) ? other_of(a, b, lo) : (sw ? a : b);
        }
    }
}

// ------------------------------------------------------------------ Batcher's odd-even mergesort
// PAPER.md:L111, L317 "BATCHERS-ODD-EVEN-MERGESORT(R)" on the 32 registers of one line
// (191 compare-exchanges, depth 15).  Template recursion = full unrolling.

template <int NP, int LO, int N, int R, int FMOD>
struct OddEvenMerge {
    static __device__ __forceinline__ void run(uint32_t (&v)[NP][32])
    {
        constexpr int M = R * 2;
        if constexpr (M < N) {
            OddEvenMerge<NP, LO, N, M, FMOD>::run(v);
            OddEvenMerge<NP, LO + R, N, M, FMOD>::run(v);
#pragma unroll
            for (int i = LO + R; i + R < LO + N; i += M) ce<NP, FMOD>(v, i, i + R);
        } else {
            ce<NP, FMOD>(v, LO, LO + R);
        }
    }
};

template <int NP, int LO, int N, int FMOD>
struct OddEvenMergeSort {
    static __device__ __forceinline__ void run(uint32_t (&v)[NP][32])
    {
        if constexpr (N > 1) {
            OddEvenMergeSort<NP, LO, N / 2, FMOD>::run(v);
            OddEvenMergeSort<NP, LO + N / 2, N / 2, FMOD>::run(v);
            OddEvenMerge<NP, LO, N, 1, FMOD>::run(v);
        }
    }
};

// Sort the 32 elements of a line ascending.
template <int NP, int FMOD = BCF_CE1_FMA_MOD>
__device__ __forceinline__ void line_sort(uint32_t (&v)[NP][32])
{
    OddEvenMergeSort<NP, 0, 32, FMOD>::run(v);
}

// The last five stages (strides 16, 8, 4, 2, 1) of a bitonic merger applied to a line that is a
// bitonic sequence: 80 compare-exchanges, depth 5.  Used by SHEARSORT-MERGE (reading A8): with
// the second piece stored reversed every column and then every row of the page is bitonic, so
// the line "sort" of PAPER.md:L129 needs only a merger.
template <int NP, int FMOD = BCF_CE1_FMA_MOD>
__device__ __forceinline__ void line_bitonic_merge(uint32_t (&v)[NP][32])
{
#pragma unroll
    for (int s = 16; s >= 1; s >>= 1) {
#pragma unroll
        for (int k = 0; k < 32; ++k)
            if ((k & s) == 0) ce<NP, FMOD>(v, k, k + s);
    }
}

// Stages of stride 2^(T-1) .. 1 of a bitonic merger inside every block of 2^T consecutive registers
// (T = 5 is line_bitonic_merge).  Used on column registers by the tile mergesort: a block of 2^T
// rows of the page is a bitonic sequence of 32 * 2^T elements, and its stages of stride >= 32
// elements are exactly these register stages of the thread that owns the column.
template <int NP, int T, int FMOD = BCF_CE1_FMA_MOD>
__device__ __forceinline__ void block_bitonic_merge(uint32_t (&v)[NP][32])
{
#pragma unroll
    for (int s = (1 << (T - 1)); s >= 1; s >>= 1) {
#pragma unroll
        for (int k = 0; k < 32; ++k)
            if ((k & s) == 0) ce<NP, FMOD>(v, k, k + s);
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

// Column sweep of the tile mergesort at level T: blocks of 2^T rows, each made of two sorted blocks
// P (first half) and Q (second half) of 2^(T-1) rows.  The thread of column c reads, as register k,
// position 32 k + c of the bitonic sequence P || reverse(Q): rows of P as they are, the rows of Q
// in reverse order and mirrored (column 31 - c).  For a fixed k the 32 threads read the 32 words of
// ONE row in a permuted order -> 32 distinct banks, like col_load.
// merge_level_row / merge_level_mirror: bcf_layout.cuh

template <int T>
__device__ __forceinline__ void col_load_level(const uint32_t *pl, uint32_t (&v)[32], const int c)
{
#pragma unroll
    for (int k = 0; k < 32; ++k) v[k] = pl[elem_word(merge_level_row(T, k), merge_level_mirror(T, k) ? 31 - c : c)];
}

}  // namespace bcf
