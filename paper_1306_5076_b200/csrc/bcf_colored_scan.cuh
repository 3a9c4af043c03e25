// bcf_colored_scan.cuh -- conflict-free coloured prefix sums (Appendix A
// L218-230): given n values and a colour in [0, d) for each, d independent inclusive prefix sums among
// the elements of the same colour (uint32 arithmetic, sums wrap modulo 2^32).
//
// The paper's three-phase scheme (L222-224): contiguous tiles; phase 1 reduces every tile to d sums,
// phase 2 turns the d x P tile sums into exclusive offsets, phase 3 scans every tile page by page,
// each thread owning a contiguous chunk of the page, its per-colour running sums kept in shared
// memory "one memory bank per thread" (L228).  Here a tile belongs to one WARP, a page is
// 32 lanes x 16 elements, and
//   * the per-thread per-colour sums live at word  32 c + lane  (bank = lane): the data-dependent
//     index c never changes the bank, so every access of the warp hits 32 distinct banks whatever
//     the colours are -- that is the paper's point, and LAYOUT_THREAD_MAJOR (word  d lane + c, the
//     layout the paper starts from, L226) is kept selectable to reproduce its Figure 1: there the
//     bank is (d lane + c) mod 32 and conflicts grow with d;
//   * the scan ACROSS the threads of one colour, for which the paper transposes the w x d matrix
//     (L228), is a warp-shuffle scan: lane t reads its own word of colour c, five shuffle steps,
//     no second layout needed.
#pragma once
#include "bcf_kernels.cuh"

namespace bcf {
namespace cscan {

#ifndef BCF_CSCAN_CH
#define BCF_CSCAN_CH 16
#endif
// A lane reads its chunk with 16-byte loads 64 bytes apart: the two halves of a 32-byte sector arrive in
// two different instructions, so these loads DO allocate in L1 (unlike the streaming loads of the sort).
#ifndef BCF_CSCAN_LD
#define BCF_CSCAN_LD(p) __ldg(p)
#endif
constexpr int CH = BCF_CSCAN_CH;       // elements per lane per page (a multiple of 16: 16-byte loads of colours)
constexpr int PAGE = 32 * CH;          // elements per warp per page
constexpr int WARPS = 8;               // warps per CTA
constexpr int MAX_COLORS = 16;

template <bool CF>
__device__ __forceinline__ int slot(const int c, const int lane, const int d)
{
    return CF ? 32 * c + lane : d * lane + c;
}

__device__ __forceinline__ uint32_t warp_inclusive_scan(uint32_t x, const int lane)
{
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) {
        const uint32_t y = __shfl_up_sync(0xFFFFFFFFu, x, s);
        if (lane >= s) x += y;
    }
    return x;
}

// pages [first, last) of warp `w` when the pages are dealt out in consecutive, equally long ranges
__device__ __forceinline__ void warp_pages(const unsigned long long n, const unsigned long long w,
                                           const unsigned long long num_warps, unsigned long long &first,
                                           unsigned long long &last)
{
    const unsigned long long pages = (n + PAGE - 1) / PAGE;
    const unsigned long long per = (pages + num_warps - 1) / num_warps;
    first = min(pages, w * per);
    last = min(pages, first + per);
}

// this lane's chunk of a page: CH values and CH colours (missing elements: value 0, colour 0)
__device__ __forceinline__ void load_chunk(const uint32_t *__restrict__ vals, const unsigned char *__restrict__ cols,
                                           const unsigned long long base, const unsigned long long n, const int d,
                                           uint32_t (&v)[CH], uint32_t (&c)[CH])
{
    if (base + CH <= n) {
        const uint4 *pv = reinterpret_cast<const uint4 *>(vals + base);
#pragma unroll
        for (int q = 0; q < CH / 4; ++q) {
            const uint4 t = BCF_CSCAN_LD(pv + q);
            v[4 * q] = t.x; v[4 * q + 1] = t.y; v[4 * q + 2] = t.z; v[4 * q + 3] = t.w;
        }
#pragma unroll
        for (int q = 0; q < CH / 16; ++q) {
            const uint4 t = BCF_CSCAN_LD(reinterpret_cast<const uint4 *>(cols + base) + q);
            const uint32_t w[4] = {t.x, t.y, t.z, t.w};
#pragma unroll
            for (int k = 0; k < 16; ++k) c[16 * q + k] = (w[k / 4] >> (8 * (k % 4))) & 0xFFu;
        }
    } else {
#pragma unroll
        for (int k = 0; k < CH; ++k) {
            const bool in = base + k < n;
            v[k] = in ? vals[base + k] : 0u;
            c[k] = in ? cols[base + k] : 0u;
        }
    }
    // a colour byte >= d comes straight from the caller's data and would index another warp's sums: counted as d - 1
#pragma unroll
    for (int k = 0; k < CH; ++k) c[k] = min(c[k], static_cast<uint32_t>(d - 1));
}

// Phase 1: partial[w][c] = sum of the values of colour c in warp w's tile.
template <bool CF>
__global__ void __launch_bounds__(WARPS * 32)
reduce_kernel(const uint32_t *__restrict__ vals, const unsigned char *__restrict__ cols, const unsigned long long n,
              const int d, uint32_t *__restrict__ partial)
{
    pdl_entry();
    __shared__ uint32_t sm[WARPS * MAX_COLORS * 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *s = sm + warp * (MAX_COLORS * 32);
    const unsigned long long w = static_cast<unsigned long long>(blockIdx.x) * WARPS + warp;
    unsigned long long first, last;
    warp_pages(n, w, static_cast<unsigned long long>(gridDim.x) * WARPS, first, last);
    for (int c = 0; c < d; ++c) s[slot<CF>(c, lane, d)] = 0;
    for (unsigned long long p = first; p < last; ++p) {
        uint32_t v[CH], c[CH];
        load_chunk(vals, cols, p * PAGE + lane * CH, n, d, v, c);
#pragma unroll
        for (int k = 0; k < CH; ++k) s[slot<CF>(c[k], lane, d)] += v[k];
    }
    for (int c = 0; c < d; ++c) {
        uint32_t x = s[slot<CF>(c, lane, d)];
#pragma unroll
        for (int sft = 16; sft >= 1; sft >>= 1) x += __shfl_xor_sync(0xFFFFFFFFu, x, sft);
        if (lane == 0) partial[w * MAX_COLORS + c] = x;
    }
}

// Phase 2: partial[w][c] becomes the exclusive prefix sum over the warps w, per colour.  One CTA, warp c
// scans colour c in strips of 32 tiles.
__global__ void __launch_bounds__(MAX_COLORS * 32)
offsets_kernel(uint32_t *__restrict__ partial, const unsigned long long num_warps, const int d)
{
    pdl_entry();
    const int lane = threadIdx.x & 31, c = threadIdx.x >> 5;
    if (c >= d) return;
    uint32_t carry = 0;
    for (unsigned long long w0 = 0; w0 < num_warps; w0 += 32) {
        const unsigned long long w = w0 + lane;
        const uint32_t x = w < num_warps ? partial[w * MAX_COLORS + c] : 0u;
        const uint32_t incl = warp_inclusive_scan(x, lane);
        if (w < num_warps) partial[w * MAX_COLORS + c] = carry + incl - x;
        carry += __shfl_sync(0xFFFFFFFFu, incl, 31);
    }
}

// Phase 3: the coloured prefix sums of every tile, seeded with the tile offsets.
template <bool CF>
__global__ void __launch_bounds__(WARPS * 32)
scan_kernel(const uint32_t *__restrict__ vals, const unsigned char *__restrict__ cols, const unsigned long long n, const int d,
            const uint32_t *__restrict__ offsets, uint32_t *__restrict__ out)
{
    pdl_entry();
    __shared__ uint32_t sm[WARPS * MAX_COLORS * 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint32_t *s = sm + warp * (MAX_COLORS * 32);
    const unsigned long long w = static_cast<unsigned long long>(blockIdx.x) * WARPS + warp;
    unsigned long long first, last;
    warp_pages(n, w, static_cast<unsigned long long>(gridDim.x) * WARPS, first, last);
    uint32_t carry = (lane < d && first < last) ? offsets[w * MAX_COLORS + lane] : 0u;   // lane c: colour c so far
    for (unsigned long long p = first; p < last; ++p) {
        const unsigned long long base = p * PAGE + lane * CH;
        uint32_t v[CH], c[CH];
        load_chunk(vals, cols, base, n, d, v, c);
        for (int k = 0; k < d; ++k) s[slot<CF>(k, lane, d)] = 0;
        // running sums inside the chunk: one read-modify-write of this lane's own word per element
#pragma unroll
        for (int k = 0; k < CH; ++k) {
            const int i = slot<CF>(c[k], lane, d);
            v[k] += s[i];
            s[i] = v[k];
        }
        // intra-page offsets: per colour, exclusive scan of the lanes' totals + what came before the page
        for (int k = 0; k < d; ++k) {
            const int i = slot<CF>(k, lane, d);
            const uint32_t x = s[i];
            const uint32_t incl = warp_inclusive_scan(x, lane);
            const uint32_t before = __shfl_sync(0xFFFFFFFFu, carry, k);
            s[i] = before + incl - x;
            const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
            if (lane == k) carry += total;
        }
#pragma unroll
        for (int k = 0; k < CH; ++k) v[k] += s[slot<CF>(c[k], lane, d)];
        if (base + CH <= n) {
            uint4 *po = reinterpret_cast<uint4 *>(out + base);
#pragma unroll
            for (int q = 0; q < CH / 4; ++q) stg128(po + q, make_uint4(v[4 * q], v[4 * q + 1], v[4 * q + 2], v[4 * q + 3]));
        } else {
#pragma unroll
            for (int k = 0; k < CH; ++k)
                if (base + k < n) out[base + k] = v[k];
        }
    }
}

}  // namespace cscan
}  // namespace bcf
