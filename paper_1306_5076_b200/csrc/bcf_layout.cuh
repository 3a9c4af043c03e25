// bcf_layout.cuh -- the conflict-free shared-memory layout of one 32 x 32 plane of 4-byte words.
//
// PAPER.md section 2.1 (L89-93): shared memory is a matrix with one row per bank; an access of a
// warp is conflict-free when its 32 threads touch 32 distinct banks.  Section 3.3 (L153) and
// Alg. 2 (L337-363) avoid the explicit transposes of Alg. 1 by addressing logical rows and
// columns through a skew (wrapped diagonals / rotated columns).  Reading A7: any
// bijective skew with that property is equivalent.  We use an XOR skew at 16-byte-chunk
// granularity instead of the paper's rotation at word granularity:
//
//      logical element (row r, column c)  ->  word  32 r + 4 ((c >> 2) ^ (r & 7)) + (c & 3)
//
// i.e. row r stays in its own 128-byte line, and its eight 16-byte chunks are permuted by r & 7.
//  * thread-per-column, one word per thread (thread c touches (k, c) for a fixed k): the 32
//    threads touch the 32 words of line k in a permuted order -> 32 distinct banks.
//  * thread-per-row, one 16-byte chunk per thread (thread r touches chunk q of row r): a 128-bit
//    access is served per quarter-warp; threads 8a..8a+7 touch chunks q ^ (0..7) of 8 different
//    lines -> 8 distinct chunks -> 32 distinct banks.  This is what the paper's word rotation
//    cannot do, and it cuts the row-side instruction count by 4 (LDS.128 / STS.128).
//  * the same holds for the un-skewing reads that feed coalesced vector stores to global.
// Register indices never depend on the thread: only addresses do.
//
// These functions are `constexpr __host__ __device__`, used by the kernels and exported through
// bcf_layout_word / bcf_layout_access (include/bcf.h) for the host-side bank model in tests/.
#pragma once

#if defined(__CUDACC__)
#define BCF_HD __host__ __device__ __forceinline__
#else
#define BCF_HD inline
#endif

namespace bcf {

constexpr int W = 32;        // threads per warp = banks
constexpr int TILE = 1024;   // w*w

// word offset of chunk q (4 words) of logical row r
BCF_HD constexpr int chunk_word(int r, int q) { return 32 * r + 4 * (q ^ (r & 7)); }

// word offset of logical element (r, c)
BCF_HD constexpr int elem_word(int r, int c) { return chunk_word(r, c >> 2) + (c & 3); }

// column a thread-per-column access of thread c uses in row k when rows of odd index are
// mirrored (descending rows of ShearSort, read back-to-front instead of
// being written back-to-front).
BCF_HD constexpr int mirrored_col(int k, int c) { return (k & 1) ? (31 - c) : c; }

// Column sweep of the tile mergesort at level T (bcf_core.cuh col_load_level): register k of the thread of
// column c holds position 32 k + c of P || reverse(Q) of its block of 2^T rows -- which row, and mirrored or not.
BCF_HD constexpr int merge_level_row(int T, int k)
{
    const int size = 1 << T, half = size >> 1, i = k & (size - 1);
    return i < half ? k : (k - i) + half + (size - 1 - i);
}
BCF_HD constexpr bool merge_level_mirror(int T, int k) { return (k & ((1 << T) - 1)) >= (1 << (T - 1)); }

// ------------------------------------------------------------------ plain types shared by host and device code

// An element is NP 32-bit "planes" compared lexicographically in plane order (bcf_core.cuh).
template <int KW, bool HV>
struct Elem {
    static constexpr int KEY_WORDS = KW;           // 1: u32 key, 2: u64 key
    static constexpr bool HAS_VAL = HV;
    static constexpr int NP = KW + (HV ? 1 : 0);   // planes
    static constexpr int KEY_BYTES = 4 * KW;
};

// geometry of one merge round of the one-warp-per-page kernels (bcf_kernels.cuh)
struct PassGeom {
    unsigned long long n;         // elements
    unsigned long long run_len;   // L
    unsigned int shares_per_pair; // ceil(2L / 1024)
    unsigned long long num_shares;
};

// geometry of FIND-BUCKETS (bcf_buckets.cuh)
struct BucketsGeom {
    unsigned long long n, run_len;
    unsigned int s;        // runs
    unsigned int t;        // samples per run
    unsigned int P;        // buckets without pivot buckets
    unsigned int nb;       // buckets: P or 2P - 1
    int pb;
};

}  // namespace bcf
