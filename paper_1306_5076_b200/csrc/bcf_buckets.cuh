// bcf_buckets.cuh -- FIND-BUCKETS, the paper's deterministic bucket distribution (
// PAPER.md section 3.2 "Distribution" L131-137, Lemma 1, Algorithm 7) and the pivot
// buckets of section 3.3 "Duplicate keys" (L155, BCFMergesortPB).
//
// The hot path does not need it (exact co-ranking gives every CTA an equal share of the output
// whatever the key distribution); it is built as the paper's alternative partitioner:
//   s sorted runs -> t evenly spaced samples of each -> sort the s t samples -> P - 1 evenly spaced
//   pivots -> rank of every pivot in every run -> bucket sizes, exclusive prefix sums -> the runs'
//   pieces regrouped by bucket (then by run), buckets in ascending value order.
// Reading of the garbled Alg. 7 (A18): sample i of run r is element floor(i len_r / t);
// pivot j is sample floor((j + 1) s t / P) of the sorted samples, j = 0 .. P-2 ("P-1 evenly spaced
// items from S", L135); the rank of a pivot in a run is the number of elements <= pivot ("IF I[i] >
// F[c]", L507); bucket j holds F[j-1] < x <= F[j].  With pivot buckets, elements equal to pivot j
// get a bucket of their own between bucket j (now F[j-1] < x < F[j]) and bucket j+1: 2P-1 buckets.
// Keys only (the paper has no values, reading A13).
#pragma once
#include "bcf_kernels.cuh"

namespace bcf {
namespace buckets {

template <int KW>
struct KeyT { using type = uint32_t; };
template <>
struct KeyT<2> { using type = unsigned long long; };

using Geom = BucketsGeom;      // bcf_layout.cuh

__device__ __forceinline__ unsigned long long run_length(const Geom &g, const unsigned int r)
{
    const unsigned long long start = static_cast<unsigned long long>(r) * g.run_len;
    return min(g.run_len, g.n - start);
}

// S[r t + i] = I_r[floor(i len_r / t)]
template <int KW>
__global__ void sample_kernel(const void *__restrict__ kin, void *__restrict__ samples, const Geom g)
{
    pdl_entry();
    using K = typename KeyT<KW>::type;
    const unsigned long long id = static_cast<unsigned long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (id >= static_cast<unsigned long long>(g.s) * g.t) return;
    const unsigned int r = static_cast<unsigned int>(id / g.t), i = static_cast<unsigned int>(id % g.t);
    const unsigned long long len = run_length(g, r);
    const unsigned long long pos = static_cast<unsigned long long>(i) * len / g.t;
    static_cast<K *>(samples)[id] = static_cast<const K *>(kin)[static_cast<unsigned long long>(r) * g.run_len + pos];
}

// bounds[r][0 .. nb]: piece b of run r is elements [bounds[r][b], bounds[r][b+1]) of the run.
// One thread per (run, pivot): binary searches for #(< pivot) and #(<= pivot).
template <int KW>
__global__ void rank_kernel(const void *__restrict__ kin, const void *__restrict__ sorted_samples, void *__restrict__ pivots,
                            uint32_t *__restrict__ bounds, const Geom g)
{
    pdl_entry();
    using K = typename KeyT<KW>::type;
    const unsigned long long id = static_cast<unsigned long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    const unsigned int np = g.P - 1;
    if (id >= static_cast<unsigned long long>(g.s) * np) return;
    const unsigned int r = static_cast<unsigned int>(id / np), j = static_cast<unsigned int>(id % np);
    const unsigned long long st = static_cast<unsigned long long>(g.s) * g.t;
    const K *S = static_cast<const K *>(sorted_samples);
    const K f = S[(static_cast<unsigned long long>(j) + 1) * st / g.P];
    const K *run = static_cast<const K *>(kin) + static_cast<unsigned long long>(r) * g.run_len;
    const unsigned long long len = run_length(g, r);
    unsigned long long lo = 0, hi = len;                    // #(<= f)
    while (lo < hi) {
        const unsigned long long mid = (lo + hi) >> 1;
        if (run[mid] <= f) lo = mid + 1; else hi = mid;
    }
    const unsigned long long le = lo;
    uint32_t *row = bounds + static_cast<unsigned long long>(r) * (g.nb + 1);
    if (!g.pb) {
        row[j + 1] = static_cast<uint32_t>(le);
    } else {
        lo = 0; hi = le;                                    // #(< f)
        while (lo < hi) {
            const unsigned long long mid = (lo + hi) >> 1;
            if (run[mid] < f) lo = mid + 1; else hi = mid;
        }
        // a pivot repeated in F: its second copy owns nothing
        const bool dup = j > 0 && S[static_cast<unsigned long long>(j) * st / g.P] == f;
        row[2 * j + 1] = static_cast<uint32_t>(dup ? le : lo);
        row[2 * j + 2] = static_cast<uint32_t>(le);
    }
    if (j == 0) { row[0] = 0; row[g.nb] = static_cast<uint32_t>(len); }
    if (r == 0) static_cast<K *>(pivots)[j] = f;
}

// Q[b s + r] = start in O of piece (bucket b, run r); Q[nb s] = n.  One CTA: every thread sums a
// contiguous chunk of piece sizes, a shared-memory scan of the chunk sums, then the chunk is written.
constexpr int SCAN_THREADS = 1024;
__global__ void __launch_bounds__(SCAN_THREADS)
offsets_kernel(const uint32_t *__restrict__ bounds, uint32_t *__restrict__ Q, const Geom g)
{
    pdl_entry();
    __shared__ unsigned long long sums[SCAN_THREADS];
    const unsigned long long total = static_cast<unsigned long long>(g.nb) * g.s;
    const unsigned long long chunk = (total + SCAN_THREADS - 1) / SCAN_THREADS;
    const unsigned long long lo = min(total, threadIdx.x * chunk), hi = min(total, lo + chunk);
    unsigned long long acc = 0;
    for (unsigned long long e = lo; e < hi; ++e) {
        const unsigned int b = static_cast<unsigned int>(e / g.s), r = static_cast<unsigned int>(e % g.s);
        const uint32_t *row = bounds + static_cast<unsigned long long>(r) * (g.nb + 1);
        acc += row[b + 1] - row[b];
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
    for (unsigned long long e = lo; e < hi; ++e) {
        const unsigned int b = static_cast<unsigned int>(e / g.s), r = static_cast<unsigned int>(e % g.s);
        const uint32_t *row = bounds + static_cast<unsigned long long>(r) * (g.nb + 1);
        Q[e] = static_cast<uint32_t>(off);
        off += row[b + 1] - row[b];
    }
    if (threadIdx.x == SCAN_THREADS - 1) Q[total] = static_cast<uint32_t>(sums[SCAN_THREADS - 1]);
}

// O[Q[b s + r] ..] = piece (b, r).  One CTA per chunk of SCATTER_CHUNK consecutive elements of a run --
// equal work for every CTA whatever the bucket sizes (0-1 data puts half of the input into one bucket):
// the chunk's first bucket by binary search in the run's row of bounds, then bucket after bucket the
// part of the chunk that falls into it is copied, coalesced, to its place in O.
constexpr unsigned SCATTER_CHUNK = 8192;
template <int KW>
__global__ void __launch_bounds__(256)
scatter_kernel(const void *__restrict__ kin, void *__restrict__ kout, const uint32_t *__restrict__ bounds,
               const uint32_t *__restrict__ Q, const Geom g)
{
    pdl_entry();
    using K = typename KeyT<KW>::type;
    const unsigned long long chunks_per_run = (g.run_len + SCATTER_CHUNK - 1) / SCATTER_CHUNK;
    const unsigned long long total = chunks_per_run * g.s;
    for (unsigned long long e = blockIdx.x; e < total; e += gridDim.x) {
        const unsigned int r = static_cast<unsigned int>(e / chunks_per_run);
        const unsigned long long len = run_length(g, r);
        const unsigned long long c0 = (e % chunks_per_run) * SCATTER_CHUNK;
        if (c0 >= len) continue;
        const unsigned long long c1 = min(len, c0 + SCATTER_CHUNK);
        const uint32_t *row = bounds + static_cast<unsigned long long>(r) * (g.nb + 1);
        unsigned int lo = 0, hi = g.nb;                      // last b with row[b] <= c0
        while (lo + 1 < hi) {
            const unsigned int mid = (lo + hi) >> 1;
            if (row[mid] <= c0) lo = mid; else hi = mid;
        }
        const K *src = static_cast<const K *>(kin) + static_cast<unsigned long long>(r) * g.run_len;
        for (unsigned int b = lo; b < g.nb && row[b] < c1; ++b) {
            const unsigned long long from = max(c0, static_cast<unsigned long long>(row[b]));
            const unsigned long long to = min(c1, static_cast<unsigned long long>(row[b + 1]));
            if (from >= to) continue;
            K *dst = static_cast<K *>(kout) + Q[static_cast<unsigned long long>(b) * g.s + r] - row[b];
            // four independent loads in flight per thread
            unsigned long long i = from + threadIdx.x;
            for (; i + 3 * 256 < to; i += 4 * 256) {
                const K a = src[i], b2 = src[i + 256], c = src[i + 512], d = src[i + 768];
                dst[i] = a; dst[i + 256] = b2; dst[i + 512] = c; dst[i + 768] = d;
            }
            for (; i < to; i += 256) dst[i] = src[i];
        }
    }
}

}  // namespace buckets
}  // namespace bcf
