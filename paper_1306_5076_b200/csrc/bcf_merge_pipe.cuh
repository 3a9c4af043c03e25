// bcf_merge_pipe.cuh -- the production merge round for power-of-two run lengths (rows a5-a9), every
// element type: a persistent, warp-specialised kernel fed by TMA bulk copies.
//
// PAPER.md section 2 (L83-85): "we treat Theta(M) elements as a single contiguous block and transfer
// these blocks between the global and shared memories"; section 3.2 (L127-129): merge pages in
// shared memory with the conflict-free tile machinery.  The paper streams one page pair per warp
// sequentially (Alg. 6) and therefore needs its bucket distribution (L131-143) for parallelism;
// here every CTA takes an equal SHARE of the output of a round instead (north_star: "split-point
// search so each CTA gets an equal share of output"):
//
//   share      = SH = PAGES * 1024 consecutive outputs of the round (PAGES = 16 / 4 / 8 for 4- / 8- / 12-byte
//                elements), one page (sub-tile) of 1024 outputs per consumer warp at a time
//   producer   = one extra warp.  For share s it works out which input the share needs
//                  - run length 2L <= SH: the share's own input range (whole pairs),
//                  - otherwise: A[I0, I1) and B[D0 - I0, D1 - I1) from the global split points
//                    (partition_share_kernel), as 16-byte aligned supersets,
//                and issues cp.async.bulk (TMA, UBLKCP) copies global -> shared that complete on an
//                mbarrier.  NSTAGE stage buffers: the copies of share i+1 are in flight while the
//                consumers work on share i; no load ever occupies a register or an LSU slot.
//   consumers  = NWC warps (16 / 12 / 8 for 4- / 8- / 12-byte elements, Cfg below), each owning one page position
//                of the shares it works on.  Each finds the two split points of its own sub-tile INSIDE shared memory
//                with a conflict-free 32-ary search (corank_smem), reads its 1024 elements from the
//                stage buffer straight into the column layout (word address consecutive across
//                lanes: conflict-free for any offset), releases the stage, and runs SHEARSORT-MERGE
//                (column merger, skewed transpose, row merger, coalesced 128-bit stores).
//
// Multi-plane elements ((u32,u32), u64, (u64,u32)): the stage buffer holds the SoA pieces as they
// are in global memory (a key region of 4- or 8-byte keys, a value region), the search compares
// (key, value) lexicographically, and the transposes go through ONE 4 KiB scratch plane per warp,
// plane after plane, so that two stage buffers of 8192 twelve-byte elements still fit one SM.
#pragma once
#include <utility>

#include "bcf_kernels.cuh"

namespace bcf {
namespace pipe {

constexpr int NSTAGE = 2;                // stage buffers of the four-run kernel (bcf_merge4.cuh); this kernel: Cfg<E>::STAGES
constexpr int REGION_SLACK = 128;        // bytes: room for the 16-byte aligned supersets of two pieces

struct ShareMeta {
    int cnt;         // outputs of this share (<= SH)
    int a_len;       // elements taken from run A / run B ("large" rounds)
    int b_len;
    int ka_off;      // element offset of the first A / B key inside the key region
    int kb_off;
    int va_off;      // same for the value region (its alignment slack differs from the keys')
    int vb_off;
    int pad;
};

// Shape of the kernel per element type.  A share is PAGES pages of 1024 outputs in one of STAGES stage buffers; the
// NWC consumer warps form GROUPS = NWC / PAGES groups of PAGES warps, warp w owning page w mod PAGES of the shares
// of its group:
//   GROUPS = 1      every warp takes its page of EVERY share of the CTA (4-byte elements: 16 warps, 16 pages);
//   GROUPS = STAGES group j takes the shares that land in stage buffer j (every STAGES-th share of the CTA), so
//                   more warps than pages of a share can be busy (8-byte elements: 3 stage buffers of 4 pages, 12
//                   warps at 128 registers: 0.216 -> 0.185 ms per round at 2^26 (u32,u32) pairs against 8 warps on
//                   2 buffers of 8 pages).  Twelve-byte elements need 168 registers, which allows 8 consumer warps
//                   either way; one group on shares of 8 pages is the faster shape for them.
// No other assignment is allowed, for the sake of the barriers: an mbarrier wait names the phase it waits for by
// ONE parity bit, which is sound only if the waiting warp took part in the previous phase of that barrier (otherwise
// the barrier may be one phase behind -- the wait passes on stale data -- or two phases ahead -- the wait never
// returns).  In both shapes a warp waits on a stage buffer exactly in the phases in which it reads a page from it.
// (A first version dealt pages round robin to 19 / 15 / 11 warps; it was 0.2-6 % faster and crashed about once in
// ten runs of a 2^28-key sort on exactly this.)
#ifndef BCF_PIPE_PAGES4
#define BCF_PIPE_PAGES4 16   // pages per share, 4-byte elements
#endif
#ifndef BCF_PIPE_PAGES8
#define BCF_PIPE_PAGES8 4    // pages per share, 8-byte elements
#endif
#ifndef BCF_PIPE_STAGES8
#define BCF_PIPE_STAGES8 3
#endif
#ifndef BCF_PIPE_PAGES12
#define BCF_PIPE_PAGES12 8   // pages per share, 12-byte elements
#endif
#ifndef BCF_PIPE_STAGES12
#define BCF_PIPE_STAGES12 2
#endif
#ifndef BCF_PIPE_GROUPS12
#define BCF_PIPE_GROUPS12 1  // 8 warps at 168 registers; two groups on shares of 4 pages measured slower (0.322 against 0.314 ms)
#endif
template <class E>
struct Cfg {
    static constexpr int KB = E::KEY_BYTES;
    static constexpr int EB = KB + (E::HAS_VAL ? 4 : 0);
    static constexpr int PAGES = EB == 4 ? BCF_PIPE_PAGES4 : (EB == 8 ? BCF_PIPE_PAGES8 : BCF_PIPE_PAGES12);   // pages per share
    static constexpr int SH = PAGES * TILE;                    // outputs per share
    static constexpr int STAGES = EB == 4 ? 2 : (EB == 8 ? BCF_PIPE_STAGES8 : BCF_PIPE_STAGES12);
    static constexpr int GROUPS = EB == 4 ? 1 : (EB == 8 ? STAGES : BCF_PIPE_GROUPS12);
    static_assert(GROUPS == 1 || GROUPS == STAGES, "see above: a warp must take part in every phase it waits on");
    static constexpr int NWC = GROUPS * PAGES;
    static constexpr int THREADS = (NWC + 1) * 32;
    static constexpr size_t key_region = size_t(SH) * KB + REGION_SLACK;
    static constexpr size_t val_region = E::HAS_VAL ? size_t(SH) * 4 + REGION_SLACK : 0;
    static constexpr size_t stage_bytes = key_region + val_region;
    static constexpr size_t scratch_off = STAGES * stage_bytes;
    static constexpr size_t meta_off = scratch_off + size_t(NWC) * TILE * 4;
    static constexpr size_t bar_off = meta_off + STAGES * sizeof(ShareMeta);
    // split points a CTA works out for itself (small launches, SELF_MAX shares per CTA at most: merge_pipe_kernel)
    static constexpr int SELF_MAX = 8;
    static constexpr size_t self_off = bar_off + 2 * STAGES * 8;
    static constexpr size_t total = self_off + 2 * SELF_MAX * 4;
    static_assert(total + 1024 <= 227 * 1024, "stage buffers + scratch planes exceed the SM's shared memory");
    // 227 KiB of shared memory per SM, 1 KiB per CTA reserved by the system
    static constexpr int ctas_per_sm = (2 * (total + 1024) <= 227 * 1024) ? 2 : 1;
    // registers per thread that keep ctas_per_sm CTAs resident: the register file is 16 K registers per SM
    // sub-partition and the warps of the resident CTAs are dealt round the four of them, so the bound is set by the
    // sub-partition that gets ceil(warps / 4).  Stated to ptxas as the cap itself (__maxnreg__), because with
    // __launch_bounds__ alone it settles on fewer registers than the SM offers and spills element data for the
    // 64-bit key types.
    static constexpr int max_regs = (16384 / (((NWC + 1) * ctas_per_sm + 3) / 4 * 32)) / 8 * 8;
};

// ------------------------------------------------------------------ PTX wrappers (mbarrier, TMA)

__device__ __forceinline__ uint32_t smem_u32(const void *p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// 1-D bulk copy global -> shared (TMA engine; SASS UBLKCP).  dst, src 16-byte aligned, bytes % 16 == 0.
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ------------------------------------------------------------------ in-shared-memory split search
//
// Co-rank of diagonal d of (A = la elements at ka_off / va_off, B = lb elements at kb_off / vb_off):
// smallest i with NOT(A[i] <= B[d-1-i]) in the (key, value) order (A-first ties).  32-ary search:
// lane j probes i = lo + j * step with `step` ODD, so the 32 probe addresses of a 4-byte array fall
// into 32 distinct banks, and the 16 probes of each half-warp of an 8-byte array into 16 distinct
// bank pairs -- the search itself obeys the paper's rule.  3 rounds for 8192.
template <class E>
__device__ __forceinline__ bool elem_le_smem(const unsigned char *kreg, const unsigned char *vreg, const int ia, const int ib,
                                             const int va, const int vb)
{
    if constexpr (E::KEY_WORDS == 1) {
        const uint32_t x = reinterpret_cast<const uint32_t *>(kreg)[ia], y = reinterpret_cast<const uint32_t *>(kreg)[ib];
        if constexpr (E::HAS_VAL) {
            const uint32_t p = reinterpret_cast<const uint32_t *>(vreg)[va], q = reinterpret_cast<const uint32_t *>(vreg)[vb];
            return x < y || (x == y && p <= q);
        } else {
            return x <= y;
        }
    } else {
        const unsigned long long x = reinterpret_cast<const unsigned long long *>(kreg)[ia];
        const unsigned long long y = reinterpret_cast<const unsigned long long *>(kreg)[ib];
        if constexpr (E::HAS_VAL) {
            const uint32_t p = reinterpret_cast<const uint32_t *>(vreg)[va], q = reinterpret_cast<const uint32_t *>(vreg)[vb];
            return x < y || (x == y && p <= q);
        } else {
            return x <= y;
        }
    }
}

template <class E>
__device__ __forceinline__ int corank_smem(const unsigned char *kreg, const unsigned char *vreg, const ShareMeta &m,
                                           const int d, const int lane, const int lo_min = 0, const int hi_max = 1 << 30)
{
    // [lo_min, hi_max]: a range the caller already knows (the co-rank of an earlier diagonal bounds this one)
    int lo = max(max(0, d - m.b_len), lo_min), hi = min(min(d, m.a_len), hi_max);
    while (lo < hi) {
        const int step = (((hi - lo) + 31) >> 5) | 1;
        const int mid = lo + lane * step;
        bool le = false;
        if (mid < hi)
            le = elem_le_smem<E>(kreg, vreg, m.ka_off + mid, m.kb_off + d - 1 - mid, m.va_off + mid, m.vb_off + d - 1 - mid);
        const int c = __popc(__ballot_sync(0xFFFFFFFFu, le));
        const int nlo = c ? lo + (c - 1) * step + 1 : lo;
        hi = min(hi, lo + c * step);
        lo = nlo;
    }
    return lo;
}

// ------------------------------------------------------------------ a5 for shares: global split points
//
// G lanes per share boundary s in [0, num_shares]: co-rank of output diagonal SH * s inside its
// pair (clamped to the pair's length) by a G-ary search -- lane j of the group probes
// i = lo + j * step and one ballot narrows the range G-fold.  G = 32 needs 6 dependent rounds of
// global loads for a pair of 2^27-element runs instead of 27 and wins while the launch is
// latency-bound (few boundaries); with many boundaries the 64 probes per round make it
// bandwidth-bound and the plain binary search (G = 1) is faster (measured).
// Only launched for rounds with 2 L > SH.
constexpr int PART_THREADS = 128;

// Co-rank of share boundary s (output diagonal `share` * s of the round, inside its pair) by a 32-ary search of the
// calling warp: lane j probes i = lo + j * step, one ballot narrows the range 32-fold.  Same result in every lane.
template <class E>
__device__ __forceinline__ unsigned long long corank_global_warp(const void *__restrict__ kin, const uint32_t *__restrict__ vin,
                                                                 const unsigned long long n, const unsigned long long L,
                                                                 const unsigned long long out0, const int lane)
{
    const unsigned long long a0 = out0 / (2 * L) * (2 * L);
    if (a0 >= n) return 0ull;
    const unsigned long long alen = min(L, n - a0);
    const unsigned long long b0 = a0 + alen;
    const unsigned long long blen = min(L, n - b0);
    const unsigned long long d = min(out0 - a0, alen + blen);
    unsigned long long lo = d > blen ? d - blen : 0ull;
    unsigned long long hi = min(d, alen);
    while (lo < hi) {
        const unsigned long long step = (hi - lo + 31) / 32;
        const unsigned long long mid = lo + lane * step;
        bool le = false;
        if (mid < hi) le = elem_le_global<E>(kin, vin, a0 + mid, b0 + (d - 1 - mid));
        const unsigned long long c = __popc(__ballot_sync(0xFFFFFFFFu, le));
        const unsigned long long nlo = c ? lo + (c - 1) * step + 1 : lo;
        hi = min(hi, lo + c * step);
        lo = nlo;
    }
    return lo;
}

template <class E, int G>
__global__ void __launch_bounds__(PART_THREADS)
partition_share_kernel(const void *__restrict__ kin, const uint32_t *__restrict__ vin, uint32_t *__restrict__ splits,
                       const unsigned long long n, const unsigned long long L, const unsigned long long num_shares,
                       const unsigned long long share, const void *__restrict__ samp_k, const uint32_t *__restrict__ samp_v)
{
    pdl_entry();
    const int j = threadIdx.x % G;                       // lane inside the group
    const unsigned gmask = (G == 32) ? 0xFFFFFFFFu : (((1u << G) - 1u) << ((threadIdx.x & 31) / G * G));
    const unsigned long long s = (static_cast<unsigned long long>(blockIdx.x) * PART_THREADS + threadIdx.x) / G;
    if (s > num_shares) return;
    const unsigned long long out0 = s * share;
    const unsigned long long a0 = out0 / (2 * L) * (2 * L);
    if (a0 >= n) { if (j == 0) splits[s] = 0; return; }
    const unsigned long long alen = min(L, n - a0);
    const unsigned long long b0 = a0 + alen;
    const unsigned long long blen = min(L, n - b0);
    const unsigned long long d = min(out0 - a0, alen + blen);
    unsigned long long lo = d > blen ? d - blen : 0ull;
    unsigned long long hi = min(d, alen);
    if constexpr (G == 1) {
        // One thread per boundary, binary search.  ncu (profiles/r2_partition_full.md): 19 us for 16385 boundaries
        // of a pair of 2^27-key runs, 49 MB read from DRAM, every unit idle -- the ~54 probes of a boundary are
        // scattered over a 1 GiB array, each a DRAM (and TLB) miss, and several probes per round make it SLOWER
        // (4 / 8 / 16 independent, clamped probes per round: 0.027 / 0.037 / 0.054 ms per launch): the launch is
        // bound by the number of scattered probes.  So the probes are made local instead.  The merge kernel that
        // wrote this round's input also wrote the first and the last element of each of its output pages (1024
        // elements) to a small array (`samp`, 2 MB for 2^28 keys).  Because a share boundary is a multiple of the
        // page size, the predicate at i = 1024 k needs exactly a page head of A and a page tail of B: the first 17
        // of the 27 steps run on the samples, the last 10 inside one page of A and one of B.
        if (samp_k != nullptr && alen == L && lo < hi) {
            const unsigned long long pa = a0 / TILE;                   // page of A[0]
            const unsigned long long pb = (b0 + d) / TILE;             // B[d - 1 - 1024 k] = tail of page pb - k - 1
            const unsigned long long k0 = (lo + TILE - 1) / TILE;
            unsigned long long klo = k0, khi = (hi + TILE - 1) / TILE;  // smallest k in [klo, khi] with NOT P(1024 k)
            while (klo < khi) {
                const unsigned long long km = (klo + khi) >> 1;
                if (elem_le_global<E>(samp_k, samp_v, 2 * (pa + km), 2 * (pb - km - 1) + 1)) klo = km + 1;
                else khi = km;
            }
            if (klo > k0) lo = max(lo, (klo - 1) * TILE + 1);
            hi = min(hi, klo * TILE);
        }
        while (lo < hi) {
            const unsigned long long mid = (lo + hi) >> 1;
            if (elem_le_global<E>(kin, vin, a0 + mid, b0 + (d - 1 - mid))) lo = mid + 1;
            else hi = mid;
        }
    } else {
        while (lo < hi) {
            const unsigned long long step = (hi - lo + G - 1) / G;
            const unsigned long long mid = lo + j * step;
            bool le = false;
            if (mid < hi) le = elem_le_global<E>(kin, vin, a0 + mid, b0 + (d - 1 - mid));
            const unsigned long long c = __popc(__ballot_sync(gmask, le) & gmask);
            const unsigned long long nlo = c ? lo + (c - 1) * step + 1 : lo;
            hi = min(hi, lo + c * step);
            lo = nlo;
        }
    }
    if (j == 0) splits[s] = static_cast<uint32_t>(lo);
}

// ------------------------------------------------------------------ stage buffer -> column registers
//
// Register slot K of the column layout (position p = 32 K + lane of the bitonic sequence
// A' || max-padding || reverse(B')): two predicated shared loads with immediate offsets per array.
// Within each load the active lanes read consecutive elements: conflict-free for any offset.
template <int K>
__device__ __forceinline__ uint32_t load_slot32(const int xa, const int xb, const uint32_t addrA, const uint32_t addrB)
{
    uint32_t r = SENTINEL;
    asm volatile(
        "{\n"
        ".reg .pred pa, pb;\n"
        "setp.gt.s32 pa, %1, %3;\n"
        "setp.ge.s32 pb, %2, %4;\n"
        "@pa ld.shared.u32 %0, [%5+%7];\n"
        "@pb ld.shared.u32 %0, [%6+%8];\n"
        "}\n"
        : "+r"(r)
        : "r"(xa), "r"(xb), "n"(32 * K), "n"(-32 * K), "r"(addrA), "r"(addrB), "n"(128 * K), "n"(-128 * K));
    return r;
}

template <int K>
__device__ __forceinline__ void load_slot64(uint32_t &hi, uint32_t &lo, const int xa, const int xb, const uint32_t addrA,
                                            const uint32_t addrB)
{
    hi = SENTINEL;
    lo = SENTINEL;
    asm volatile(
        "{\n"
        ".reg .pred pa, pb;\n"
        "setp.gt.s32 pa, %2, %4;\n"
        "setp.ge.s32 pb, %3, %5;\n"
        "@pa ld.shared.v2.u32 {%0, %1}, [%6+%8];\n"
        "@pb ld.shared.v2.u32 {%0, %1}, [%7+%9];\n"
        "}\n"
        : "+r"(lo), "+r"(hi)
        : "r"(xa), "r"(xb), "n"(32 * K), "n"(-32 * K), "r"(addrA), "r"(addrB), "n"(256 * K), "n"(-256 * K));
}

template <class E, int... Ks>
__device__ __forceinline__ void load_columns(uint32_t (&v)[E::NP][32], const int xa, const int xb, const uint32_t kA,
                                             const uint32_t kB, const uint32_t vA, const uint32_t vB,
                                             std::integer_sequence<int, Ks...>)
{
    if constexpr (E::KEY_WORDS == 1) ((v[0][Ks] = load_slot32<Ks>(xa, xb, kA, kB)), ...);
    else (load_slot64<Ks>(v[0][Ks], v[1][Ks], xa, xb, kA, kB), ...);
    if constexpr (E::HAS_VAL) ((v[E::KEY_WORDS][Ks] = load_slot32<Ks>(xa, xb, vA, vB)), ...);
}

// ------------------------------------------------------------------ rows -> global through one scratch plane
//
// store_rows (bcf_kernels.cuh) with a single 4 KiB scratch plane per warp: the planes of the
// element go through it one after the other.  Same access patterns, same conflict-freedom.
template <class E>
__device__ __forceinline__ void store_rows_seq(uint32_t *scratch, void *keys, uint32_t *vals, const size_t base,
                                               const int cnt, const bool full, const int lane, uint32_t (&v)[E::NP][32],
                                               void *samp_k = nullptr, uint32_t *samp_v = nullptr)
{
    // samp_k / samp_v (optional): first and last element of a FULL page go to entries 2 p, 2 p + 1 (p = base / 1024)
    // of the sample arrays -- read by lane 0 from the scratch plane while the plane holds them (words of logical
    // (row 0, column 0) and (row 31, column 31)), so that no register of the page stays live for it.
    // Not for three-plane elements: their kernel sits at its register cap and any addition costs it 3-9 % per round
    // (measured), more than the partition launch gains; their partition searches the arrays themselves.
    const size_t se = 2 * (base / TILE);
    const bool sample = E::NP < 3 && samp_k != nullptr && lane == 0;
    if (full) {
        if constexpr (E::KEY_WORDS == 1) {
            row_store(scratch, v[0], lane);
            __syncwarp();
            if (sample)
                *reinterpret_cast<uint2 *>(static_cast<uint32_t *>(samp_k) + se) = make_uint2(scratch[elem_word(0, 0)], scratch[elem_word(31, 31)]);
            uint4 *pk = reinterpret_cast<uint4 *>(static_cast<uint32_t *>(keys) + base);
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int w = chunk_word(4 * m + (lane >> 3), lane & 7);
                stg128(pk + 32 * m + lane, *reinterpret_cast<const uint4 *>(scratch + w));
            }
        } else {
            row_store(scratch, v[0], lane);
            __syncwarp();
            uint32_t sh0 = 0, sh1 = 0;
            if (sample) { sh0 = scratch[elem_word(0, 0)]; sh1 = scratch[elem_word(31, 31)]; }
#pragma unroll
            for (int m = 0; m < 16; ++m) {     // this lane's high words of keys 64 m + 2 lane, + 1
                const int w = elem_word(2 * m + (lane >> 4), 2 * (lane & 15));
                const uint2 h = *reinterpret_cast<const uint2 *>(scratch + w);
                v[0][2 * m] = h.x; v[0][2 * m + 1] = h.y;
            }
            __syncwarp();
            row_store(scratch, v[1], lane);
            __syncwarp();
            if (sample)
                *reinterpret_cast<uint4 *>(static_cast<uint64_t *>(samp_k) + se) =
                    make_uint4(scratch[elem_word(0, 0)], sh0, scratch[elem_word(31, 31)], sh1);
            uint4 *pk = reinterpret_cast<uint4 *>(static_cast<uint64_t *>(keys) + base);
#pragma unroll
            for (int m = 0; m < 16; ++m) {
                const int w = elem_word(2 * m + (lane >> 4), 2 * (lane & 15));
                const uint2 l = *reinterpret_cast<const uint2 *>(scratch + w);
                stg128(pk + 32 * m + lane, make_uint4(l.x, v[0][2 * m], l.y, v[0][2 * m + 1]));
            }
        }
        if constexpr (E::HAS_VAL) {
            __syncwarp();
            row_store(scratch, v[E::KEY_WORDS], lane);
            __syncwarp();
            if (sample) *reinterpret_cast<uint2 *>(samp_v + se) = make_uint2(scratch[elem_word(0, 0)], scratch[elem_word(31, 31)]);
            uint4 *pv = reinterpret_cast<uint4 *>(vals + base);
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int w = chunk_word(4 * m + (lane >> 3), lane & 7);
                stg128(pv + 32 * m + lane, *reinterpret_cast<const uint4 *>(scratch + w));
            }
        }
    } else {
        // ragged end of the array: back to the column layout (position 32 k + lane), guarded stores
#pragma unroll
        for (int p = 0; p < E::NP; ++p) {
            row_store(scratch, v[p], lane);
            __syncwarp();
            col_load<false>(scratch, v[p], lane);
            __syncwarp();
        }
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            if (32 * k + lane < cnt) {
                const size_t g = base + 32 * k + lane;
                if constexpr (E::KEY_WORDS == 1) stg32(static_cast<uint32_t *>(keys) + g, v[0][k]);
                else stg64(reinterpret_cast<uint2 *>(keys) + g, make_uint2(v[1][k], v[0][k]));
                if constexpr (E::HAS_VAL) stg32(vals + g, v[E::KEY_WORDS][k]);
            }
        }
    }
    __syncwarp();   // the scratch plane is reused by the warp's next sub-tile
}

// ------------------------------------------------------------------ the merge round

// 16-byte aligned superset [s, e) of elements [g, g + len) of an array of EB-byte elements.
template <int EB>
__device__ __forceinline__ void aligned_superset(const unsigned long long g, const int len, unsigned long long &s,
                                                 unsigned long long &e)
{
    constexpr unsigned long long M = 16 / EB - 1;
    s = g & ~M;
    e = (g + len + M) & ~M;
}

template <class E>
__global__ void __maxnreg__(Cfg<E>::max_regs)
merge_pipe_kernel(const void *__restrict__ kin_, const uint32_t *__restrict__ vin, void *__restrict__ kout,
                  uint32_t *__restrict__ vout, const uint32_t *__restrict__ splits, const unsigned long long n,
                  const unsigned long long L, const unsigned long long num_shares, const int self_part,
                  void *__restrict__ samp_k, uint32_t *__restrict__ samp_v)
{
    pdl_entry();
    using C = Cfg<E>;
    constexpr int KB = C::KB;
    constexpr int SH = C::SH, NSTAGE = C::STAGES, NW = C::NWC;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint32_t *scratch_all = reinterpret_cast<uint32_t *>(smem_raw + C::scratch_off);
    ShareMeta *meta = reinterpret_cast<ShareMeta *>(smem_raw + C::meta_off);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + C::bar_off);
    uint64_t *empty = full + NSTAGE;
    const unsigned char *kin = static_cast<const unsigned char *>(kin_);

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const bool small_round = (2 * L <= static_cast<unsigned long long>(SH));

    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], C::PAGES);      // one arrival per page of the share
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // self_part: the launch is small (every CTA has at most SELF_MAX shares) and no partition launch preceded it.
    // The warps of the CTA work out the split points of the CTA's own share boundaries first -- boundary q = 2 i + e
    // is the start (e = 0) or the end (e = 1) of the CTA's i-th share -- one 32-ary search per warp at a time.  This
    // removes one launch per round where launches are what a round costs (2^24 keys and below).
    uint32_t *self_splits = reinterpret_cast<uint32_t *>(smem_raw + C::self_off);
    if (self_part) {
        const unsigned int mine =
            blockIdx.x < num_shares ? static_cast<unsigned int>((num_shares - blockIdx.x + gridDim.x - 1) / gridDim.x) : 0u;
        for (unsigned int q = warp; q < 2 * mine; q += NW + 1) {
            const unsigned long long sb = blockIdx.x + static_cast<unsigned long long>(q >> 1) * gridDim.x + (q & 1u);
            const unsigned long long c = corank_global_warp<E>(kin_, vin, n, L, sb * SH, lane);
            if (lane == 0) self_splits[q] = static_cast<uint32_t>(c);
        }
    }
    __syncthreads();

    if (warp == NW) {
        // ============================== producer warp
        unsigned int it = 0;
        for (unsigned long long s = blockIdx.x; s < num_shares; s += gridDim.x, ++it) {
            const int st = it % NSTAGE;
            const uint32_t ph = (it / NSTAGE) & 1u;
            unsigned char *kreg = smem_raw + st * C::stage_bytes;
            unsigned char *vreg = kreg + C::key_region;
            // (waiting for the stage only after the split points are loaded -- later than here -- was measured: it
            // changes nothing for the wide element types and costs the u32 kernel 10 %, 0.328 -> 0.363 ms per round)
            mbar_wait(&empty[st], ph ^ 1u);
            const unsigned long long out0 = s * SH;
            const int cnt = static_cast<int>(min(static_cast<unsigned long long>(SH), n - out0));
            ShareMeta m;
            m.cnt = cnt;
            m.pad = 0;
            if (small_round) {
                m.a_len = 0; m.b_len = 0; m.ka_off = 0; m.kb_off = 0; m.va_off = 0; m.vb_off = 0;
                if ((cnt & 3) == 0) {
                    if (lane == 0) {
                        meta[st] = m;
                        mbar_arrive_expect_tx(&full[st], static_cast<uint32_t>(cnt) * (KB + (E::HAS_VAL ? 4u : 0u)));
                        bulk_g2s(kreg, kin + out0 * KB, static_cast<uint32_t>(cnt) * KB, &full[st]);
                        if constexpr (E::HAS_VAL) bulk_g2s(vreg, vin + out0, static_cast<uint32_t>(cnt) * 4u, &full[st]);
                    }
                } else {   // ragged end of the array: plain cooperative copy
                    for (int i = lane; i < cnt * (KB / 4); i += 32)
                        reinterpret_cast<uint32_t *>(kreg)[i] = reinterpret_cast<const uint32_t *>(kin + out0 * KB)[i];
                    if constexpr (E::HAS_VAL)
                        for (int i = lane; i < cnt; i += 32) reinterpret_cast<uint32_t *>(vreg)[i] = vin[out0 + i];
                    __syncwarp();
                    if (lane == 0) { meta[st] = m; mbar_arrive(&full[st]); }
                }
            } else {
                const unsigned long long a0 = out0 / (2 * L) * (2 * L);
                const unsigned long long alen = min(L, n - a0);
                const unsigned long long b0 = a0 + alen;
                const unsigned long long blen = min(L, n - b0);
                const unsigned long long D0 = out0 - a0, D1 = D0 + cnt;
                const unsigned long long I0 = self_part ? self_splits[2 * it] : splits[s];
                const unsigned long long I1 = (D1 >= alen + blen) ? alen : (self_part ? self_splits[2 * it + 1] : splits[s + 1]);
                const unsigned long long ga = a0 + I0, gb = b0 + (D0 - I0);
                const int la = static_cast<int>(I1 - I0), lb = cnt - la;
                unsigned long long ksa, kea, ksb, keb, vsa = 0, vea = 0, vsb = 0, veb = 0;
                aligned_superset<KB>(ga, la, ksa, kea);
                aligned_superset<KB>(gb, lb, ksb, keb);
                const int kA = la ? static_cast<int>(kea - ksa) : 0;
                const int kB = lb ? static_cast<int>(keb - ksb) : 0;
                m.a_len = la;
                m.b_len = lb;
                m.ka_off = static_cast<int>(ga - ksa);
                m.kb_off = kA + static_cast<int>(gb - ksb);
                int vA = 0, vB = 0;
                m.va_off = 0;
                m.vb_off = 0;
                bool bulk_ok = (!la || kea <= n) && (!lb || keb <= n);
                if constexpr (E::HAS_VAL) {
                    aligned_superset<4>(ga, la, vsa, vea);
                    aligned_superset<4>(gb, lb, vsb, veb);
                    vA = la ? static_cast<int>(vea - vsa) : 0;
                    vB = lb ? static_cast<int>(veb - vsb) : 0;
                    m.va_off = static_cast<int>(ga - vsa);
                    m.vb_off = vA + static_cast<int>(gb - vsb);
                    bulk_ok = bulk_ok && (!la || vea <= n) && (!lb || veb <= n);
                }
                if (bulk_ok) {
                    if (lane == 0) {
                        meta[st] = m;
                        mbar_arrive_expect_tx(&full[st], static_cast<uint32_t>(kA + kB) * KB + static_cast<uint32_t>(vA + vB) * 4u);
                        if (la) bulk_g2s(kreg, kin + ksa * KB, static_cast<uint32_t>(kA) * KB, &full[st]);
                        if (lb) bulk_g2s(kreg + size_t(kA) * KB, kin + ksb * KB, static_cast<uint32_t>(kB) * KB, &full[st]);
                        if constexpr (E::HAS_VAL) {
                            if (la) bulk_g2s(vreg, vin + vsa, static_cast<uint32_t>(vA) * 4u, &full[st]);
                            if (lb) bulk_g2s(vreg + size_t(vA) * 4, vin + vsb, static_cast<uint32_t>(vB) * 4u, &full[st]);
                        }
                    }
                } else {
                    uint32_t *kw = reinterpret_cast<uint32_t *>(kreg);
                    const uint32_t *gk = reinterpret_cast<const uint32_t *>(kin);
                    for (int i = lane; i < la * (KB / 4); i += 32) kw[m.ka_off * (KB / 4) + i] = gk[ga * (KB / 4) + i];
                    for (int i = lane; i < lb * (KB / 4); i += 32) kw[m.kb_off * (KB / 4) + i] = gk[gb * (KB / 4) + i];
                    if constexpr (E::HAS_VAL) {
                        uint32_t *vw = reinterpret_cast<uint32_t *>(vreg);
                        for (int i = lane; i < la; i += 32) vw[m.va_off + i] = vin[ga + i];
                        for (int i = lane; i < lb; i += 32) vw[m.vb_off + i] = vin[gb + i];
                    }
                    __syncwarp();
                    if (lane == 0) { meta[st] = m; mbar_arrive(&full[st]); }
                }
            }
        }
        return;
    }

    // ============================== consumer warps
    // warp w: page w mod PAGES of the shares of group w / PAGES (Cfg above)
    uint32_t *scratch = scratch_all + warp * TILE;
    const int tile_off = (warp % C::PAGES) * TILE;
    for (unsigned int it = warp / C::PAGES;; it += C::GROUPS) {
        const unsigned long long s = blockIdx.x + static_cast<unsigned long long>(it) * gridDim.x;
        if (s >= num_shares) break;
        const int st = it % NSTAGE;
        const uint32_t ph = (it / NSTAGE) & 1u;
        const unsigned char *kreg = smem_raw + st * C::stage_bytes;
        const unsigned char *vreg = kreg + C::key_region;
        mbar_wait(&full[st], ph);
        ShareMeta m = meta[st];
        if (tile_off >= m.cnt) {            // ragged last share: nothing on this page
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[st]);
            continue;
        }
        int d0;
        if (small_round) {
            const int l = static_cast<int>(L);
            const int pb = tile_off / (2 * l) * (2 * l);
            m.a_len = min(l, m.cnt - pb);
            m.b_len = min(l, m.cnt - pb - m.a_len);
            m.ka_off = pb; m.kb_off = pb + m.a_len;
            m.va_off = pb; m.vb_off = pb + m.a_len;
            d0 = tile_off - pb;
        } else {
            d0 = tile_off;
        }
        const int d1 = min(d0 + TILE, m.a_len + m.b_len);
        const int i0 = corank_smem<E>(kreg, vreg, m, d0, lane);
        const int i1 = corank_smem<E>(kreg, vreg, m, d1, lane, i0, i0 + (d1 - d0));
        const int a = i1 - i0;                   // elements of A in this sub-tile
        const int b = (d1 - d0) - a;             // elements of B
        // column layout straight from the stage buffer: position p = 32 k + lane is A'[p] for p < a,
        // B'[1023 - p] for p >= 1024 - b, the maximum element in between (partial sub-tiles only).
        const uint32_t kA = smem_u32(kreg) + static_cast<uint32_t>(m.ka_off + i0 + lane) * KB;
        const uint32_t kB = smem_u32(kreg) + static_cast<uint32_t>(m.kb_off + (d0 - i0) + (TILE - 1) - lane) * KB;
        const uint32_t vA = smem_u32(vreg) + static_cast<uint32_t>(m.va_off + i0 + lane) * 4u;
        const uint32_t vB = smem_u32(vreg) + static_cast<uint32_t>(m.vb_off + (d0 - i0) + (TILE - 1) - lane) * 4u;
        const int xa = a - lane;                 // p < a        <=>  32 k < xa
        const int xb = lane - (TILE - b);        // p >= 1024-b  <=>  32 k + xb >= 0
        uint32_t v[E::NP][32];
        load_columns<E>(v, xa, xb, kA, kB, vA, vB, std::make_integer_sequence<int, 32>{});
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[st]);  // stage buffer may be refilled

        line_bitonic_merge<E::NP>(v);            // column pass
#pragma unroll
        for (int p = 0; p < E::NP; ++p) {
            if (p) __syncwarp();
            col_store<false>(scratch, v[p], lane);
            __syncwarp();
            row_load(scratch, v[p], lane);
        }
        line_bitonic_merge<E::NP>(v);            // row pass
        const int cnt = d1 - d0;
        // (full pages also leave their first and last element in `samp` for the partition of the next round)
        if constexpr (E::NP < 3) store_rows_seq<E>(scratch, kout, vout, s * SH + tile_off, cnt, cnt == TILE, lane, v, samp_k, samp_v);
        else store_rows_seq<E>(scratch, kout, vout, s * SH + tile_off, cnt, cnt == TILE, lane, v);
    }
}

}  // namespace pipe
}  // namespace bcf
