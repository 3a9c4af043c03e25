// bcf_pieces.cuh -- the FINAL MERGE PHASE of BCFMergesort inside the buckets (
// PAPER.md section 3.2 "Final merge phase" L141-143, Appendix B): after FIND-BUCKETS every bucket
// holds s sorted subsequences ("pieces", one per run) of arbitrary lengths, possibly empty; "CTA p_i then
// sorts the i-th bucket by merging the sorted subsequences of the bucket ... padding is introduced
// implicitly in shared memory, but not written to the output array.  This phase requires log(P) additional
// merge rounds".
//
// A round merges, inside every group (bucket) of s pieces, blocks of B = 2^k adjacent pieces pairwise;
// the blocks are described by the piece offsets FIND-BUCKETS wrote (Q[g s + r]), so no per-round
// descriptor array exists.  The paper gives a bucket to one CTA; with duplicates a bucket can hold most of
// the input (L155), so here the unit of work is one PAGE of BCF_TILE outputs of one pair instead, whatever
// the piece lengths:
//   pages_scan_kernel   pages[q] = ceil((|A_q| + |B_q|) / 1024) for every pair q of the round, exclusive
//                       prefix sums -> first[q]; first[npairs] = number of pages of the round
//   merge_pieces_kernel warps stride over the pages of the round: pair by binary search in first[], the
//                       page's two split points by a 32-ary co-rank search (one probe per lane, A-first
//                       ties as in bcf_merge_partition), then SHEARSORT-MERGE of the page exactly as
//                       merge_kernel does (bitonic column layout straight from global memory, column
//                       merger, skewed transpose, row merger, coalesced stores); a partial page is padded
//                       with the maximum key in registers only.
// Pivot buckets (L155: "already in the correct position") are groups that are copied: their pieces are
// treated as ONE block whose partner is empty.  Keys only, like FIND-BUCKETS.
#pragma once
#include "bcf_kernels.cuh"

namespace bcf {
namespace pieces {

struct Geom {
    unsigned long long groups;   // buckets
    unsigned int s;              // pieces per group
    unsigned int block;          // B = 2^k pieces per sorted block at the start of this round
    unsigned int ppg;            // pairs per group = ceil(s / 2B)
    int copy_odd;                // groups of odd index are one block (pivot buckets)
};

// [a0, a1) and [a1, b1): the two sorted blocks of pair q.
__device__ __forceinline__ void pair_range(const uint32_t *__restrict__ Q, const Geom &g, const unsigned long long q,
                                           unsigned long long &a0, unsigned long long &a1, unsigned long long &b1)
{
    const unsigned long long grp = q / g.ppg;
    const unsigned int j = static_cast<unsigned int>(q % g.ppg);
    const uint32_t *row = Q + grp * g.s;
    if (g.copy_odd && (grp & 1)) {
        a0 = row[0];
        a1 = b1 = (j == 0) ? row[g.s] : row[0];       // pair 0 carries the whole group, the others nothing
        if (j) a0 = a1;
        return;
    }
    const unsigned long long p0 = min(static_cast<unsigned long long>(g.s), 2ull * j * g.block);
    const unsigned long long p1 = min(static_cast<unsigned long long>(g.s), p0 + g.block);
    const unsigned long long p2 = min(static_cast<unsigned long long>(g.s), p1 + g.block);
    a0 = row[p0]; a1 = row[p1]; b1 = row[p2];
}

constexpr int SCAN_THREADS = 1024;
__global__ void __launch_bounds__(SCAN_THREADS)
pages_scan_kernel(const uint32_t *__restrict__ Q, uint32_t *__restrict__ first, const Geom g)
{
    pdl_entry();
    __shared__ unsigned long long sums[SCAN_THREADS];
    const unsigned long long total = g.groups * g.ppg;
    const unsigned long long chunk = (total + SCAN_THREADS - 1) / SCAN_THREADS;
    const unsigned long long lo = min(total, threadIdx.x * chunk), hi = min(total, lo + chunk);
    unsigned long long acc = 0;
    for (unsigned long long q = lo; q < hi; ++q) {
        unsigned long long a0, a1, b1;
        pair_range(Q, g, q, a0, a1, b1);
        acc += (b1 - a0 + TILE - 1) / TILE;
    }
    sums[threadIdx.x] = acc;
    __syncthreads();
    for (int d = 1; d < SCAN_THREADS; d <<= 1) {            // inclusive Hillis-Steele scan
        const unsigned long long v = threadIdx.x >= d ? sums[threadIdx.x - d] : 0ull;
        __syncthreads();
        sums[threadIdx.x] += v;
        __syncthreads();
    }
    unsigned long long off = threadIdx.x ? sums[threadIdx.x - 1] : 0ull;
    for (unsigned long long q = lo; q < hi; ++q) {
        unsigned long long a0, a1, b1;
        pair_range(Q, g, q, a0, a1, b1);
        first[q] = static_cast<uint32_t>(off);
        off += (b1 - a0 + TILE - 1) / TILE;
    }
    if (threadIdx.x == SCAN_THREADS - 1) first[total] = static_cast<uint32_t>(sums[SCAN_THREADS - 1]);
}

// Co-rank of diagonal d of (A = la keys at A, B = lb keys at B): smallest i with NOT(A[i] <= B[d-1-i]).
// 32-ary: lane j probes lo + j * step, one ballot narrows the range 32-fold.
template <class E>
__device__ __forceinline__ unsigned long long corank_warp(const void *__restrict__ kin, const unsigned long long A,
                                                          const unsigned long long la, const unsigned long long B,
                                                          const unsigned long long lb, const unsigned long long d, const int lane)
{
    unsigned long long lo = d > lb ? d - lb : 0ull, hi = min(d, la);
    while (lo < hi) {
        const unsigned long long step = (hi - lo + 31) / 32;
        const unsigned long long mid = lo + lane * step;
        bool le = false;
        if (mid < hi) le = elem_le_global<E>(kin, nullptr, A + mid, B + (d - 1 - mid));
        const unsigned long long c = __popc(__ballot_sync(0xFFFFFFFFu, le));
        const unsigned long long nlo = c ? lo + (c - 1) * step + 1 : lo;
        hi = min(hi, lo + c * step);
        lo = nlo;
    }
    return lo;
}

template <class E>
__global__ void __launch_bounds__(WARPS_PER_CTA * 32)
merge_pieces_kernel(const void *__restrict__ kin, void *__restrict__ kout, const uint32_t *__restrict__ Q,
                    const uint32_t *__restrict__ first, const Geom g)
{
    pdl_entry();
    static_assert(!E::HAS_VAL, "keys only");
    extern __shared__ __align__(16) uint32_t smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    uint32_t *planes = smem + warp * (E::NP * TILE);
    const unsigned long long npairs = g.groups * g.ppg;
    const unsigned long long total = first[npairs];
    const unsigned long long stride = static_cast<unsigned long long>(gridDim.x) * WARPS_PER_CTA;

    for (unsigned long long w = static_cast<unsigned long long>(blockIdx.x) * WARPS_PER_CTA + warp; w < total; w += stride) {
        unsigned long long lo = 0, hi = npairs;              // last pair q with first[q] <= w (pairs without pages are skipped)
        while (lo + 1 < hi) {
            const unsigned long long mid = (lo + hi) >> 1;
            if (first[mid] <= w) lo = mid; else hi = mid;
        }
        unsigned long long a0, a1, b1;
        pair_range(Q, g, lo, a0, a1, b1);
        const unsigned long long la = a1 - a0, lb = b1 - a1;
        const unsigned long long d0 = (w - first[lo]) * TILE;
        const unsigned long long d1 = min(d0 + TILE, la + lb);
        const unsigned long long i0 = corank_warp<E>(kin, a0, la, a1, lb, d0, lane);
        const unsigned long long i1 = corank_warp<E>(kin, a0, la, a1, lb, d1, lane);
        const int a = static_cast<int>(i1 - i0);
        const int b = static_cast<int>((d1 - i1) - (d0 - i0));
        const size_t ga = a0 + i0, gb = a1 + (d0 - i0);

        uint32_t v[E::NP][32];
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            const int p = 32 * k + lane;
            if (p < a) load_elem<E>(kin, nullptr, ga + p, v, k);
            else if (p >= TILE - b) load_elem<E>(kin, nullptr, gb + (TILE - 1 - p), v, k);
            else set_sentinel<E>(v, k);
        }
        line_bitonic_merge<E::NP>(v);                            // column pass
#pragma unroll
        for (int p = 0; p < E::NP; ++p) col_store<false>(planes + p * TILE, v[p], lane);
        __syncwarp();
#pragma unroll
        for (int p = 0; p < E::NP; ++p) row_load(planes + p * TILE, v[p], lane);
        line_bitonic_merge<E::NP>(v);                            // row pass

        const size_t out = a0 + d0;
        const int cnt = static_cast<int>(d1 - d0);
        const bool vec_ok = (cnt == TILE) && ((out * E::KEY_BYTES) % 16 == 0);
        store_rows<E>(planes, kout, nullptr, out, cnt, vec_ok, lane, v);
    }
}

}  // namespace pieces
}  // namespace bcf
