// bcf_merge_pipe.cuh -- the production merge round for power-of-two run lengths (rows a5-a9):
// a persistent, warp-specialised kernel fed by TMA bulk copies.
//
// PAPER.md section 2 (L83-85): "we treat Theta(M) elements as a single contiguous block and transfer
// these blocks between the global and shared memories"; section 3.2 (L127-129): merge pages in
// shared memory with the conflict-free tile machinery.  The paper streams one page pair per warp
// sequentially (Alg. 6) and therefore needs its bucket distribution (L131-143) for parallelism;
// here every CTA takes an equal SHARE of the output of a round instead (north_star: "split-point
// search so each CTA gets an equal share of output"):
//
//   share      = SH = 8 * 1024 consecutive outputs of the round = 8 sub-tiles, one per consumer warp
//   producer   = one extra warp.  For share s it works out which input the share needs
//                  - run length 2L <= SH: the share's own input range (whole pairs),
//                  - otherwise: A[I0, I1) and B[D0 - I0, D1 - I1) from the global split points
//                    (partition_share_kernel), as 16-byte aligned supersets,
//                and issues cp.async.bulk (TMA, UBLKCP) copies global -> shared that complete on an
//                mbarrier.  NSTAGE stage buffers: the copies of share i+1 are in flight while the
//                consumers work on share i; no load ever occupies a register or an LSU slot.
//   consumers  = 8 warps.  Each finds the two split points of its own sub-tile INSIDE shared memory
//                with a conflict-free 32-ary search (corank_smem), reads its 1024 elements from the
//                stage buffer straight into the column layout (word address consecutive across
//                lanes: conflict-free for any offset), releases the stage, and runs SHEARSORT-MERGE
//                (column merger, skewed transpose, row merger, coalesced 128-bit stores).
#pragma once
#include <utility>

#include "bcf_kernels.cuh"

namespace bcf {
namespace pipe {

constexpr int NW = 8;                    // consumer warps per CTA
constexpr int SH = NW * TILE;            // outputs per share
constexpr int NSTAGE = 2;
constexpr int STAGE_WORDS = SH + 32;     // room for the two aligned supersets
constexpr int THREADS = (NW + 1) * 32;

struct ShareMeta {
    int cnt;         // outputs of this share (<= SH)
    int a_off;       // word offset of the A piece in the stage buffer ("large" rounds)
    int a_len;
    int b_off;
    int b_len;
    int pad[3];
};

struct SmemLayout {
    static constexpr size_t stage_bytes = size_t(STAGE_WORDS) * 4;
    static constexpr size_t planes_off = NSTAGE * stage_bytes;
    static constexpr size_t meta_off = planes_off + size_t(NW) * TILE * 4;
    static constexpr size_t bar_off = meta_off + NSTAGE * sizeof(ShareMeta);
    static constexpr size_t total = bar_off + 2 * NSTAGE * 8;
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
// Co-rank of diagonal d of (A = buf[sA .. sA+la), B = buf[sB .. sB+lb)): smallest i with
// NOT(A[i] <= B[d-1-i]) (A-first ties).  32-ary search: lane j probes i = lo + j * step with `step`
// ODD, so the 32 probe addresses sA + i (and sB + d - 1 - i) fall into 32 distinct banks -- the
// search itself obeys the paper's rule.  3 rounds for a range of 8192.
__device__ __forceinline__ int corank_smem(const uint32_t *buf, const int sA, const int la, const int sB, const int lb,
                                           const int d, const int lane)
{
    int lo = max(0, d - lb), hi = min(d, la);
    while (lo < hi) {
        const int step = (((hi - lo) + 31) >> 5) | 1;
        const int mid = lo + lane * step;
        bool le = false;
        if (mid < hi) le = buf[sA + mid] <= buf[sB + d - 1 - mid];
        const int c = __popc(__ballot_sync(0xFFFFFFFFu, le));
        const int nlo = c ? lo + (c - 1) * step + 1 : lo;
        hi = min(hi, lo + c * step);
        lo = nlo;
    }
    return lo;
}

// ------------------------------------------------------------------ a5 for shares: global split points
//
// One thread per share boundary s in [0, num_shares]: co-rank of output diagonal SH * s inside its
// pair (clamped to the pair's length).  Only launched for rounds with 2 L > SH.
__global__ void __launch_bounds__(128)
partition_share_kernel(const uint32_t *__restrict__ kin, uint32_t *__restrict__ splits, const unsigned long long n,
                       const unsigned long long L, const unsigned long long num_shares)
{
    const unsigned long long s = static_cast<unsigned long long>(blockIdx.x) * blockDim.x + threadIdx.x;
    if (s > num_shares) return;
    const unsigned long long out0 = s * SH;
    const unsigned long long a0 = out0 / (2 * L) * (2 * L);
    if (a0 >= n) { splits[s] = 0; return; }
    const unsigned long long alen = min(L, n - a0);
    const unsigned long long b0 = a0 + alen;
    const unsigned long long blen = min(L, n - b0);
    const unsigned long long d = min(out0 - a0, alen + blen);
    unsigned long long lo = d > blen ? d - blen : 0ull;
    unsigned long long hi = min(d, alen);
    while (lo < hi) {
        const unsigned long long mid = (lo + hi) >> 1;
        if (__ldg(kin + a0 + mid) <= __ldg(kin + b0 + (d - 1 - mid))) lo = mid + 1;
        else hi = mid;
    }
    splits[s] = static_cast<uint32_t>(lo);
}

// Register slot K of the column layout: two predicated shared loads with immediate offsets.
template <int K>
__device__ __forceinline__ uint32_t load_column_slot(const int xa, const int xb, const uint32_t addrA, const uint32_t addrB)
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

template <int... Ks>
__device__ __forceinline__ void load_columns(uint32_t (&v)[32], const int xa, const int xb, const uint32_t addrA,
                                             const uint32_t addrB, std::integer_sequence<int, Ks...>)
{
    ((v[Ks] = load_column_slot<Ks>(xa, xb, addrA, addrB)), ...);
}

// ------------------------------------------------------------------ the merge round

__global__ void __launch_bounds__(THREADS, 2)
merge_pipe_kernel(const uint32_t *__restrict__ kin, uint32_t *__restrict__ kout, const uint32_t *__restrict__ splits,
                  const unsigned long long n, const unsigned long long L, const unsigned long long num_shares)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint32_t *stage_buf = reinterpret_cast<uint32_t *>(smem_raw);
    uint32_t *planes_all = reinterpret_cast<uint32_t *>(smem_raw + SmemLayout::planes_off);
    ShareMeta *meta = reinterpret_cast<ShareMeta *>(smem_raw + SmemLayout::meta_off);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + SmemLayout::bar_off);
    uint64_t *empty = full + NSTAGE;

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const bool small_round = (2 * L <= static_cast<unsigned long long>(SH));

    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NW) {
        // ============================== producer warp
        unsigned int it = 0;
        for (unsigned long long s = blockIdx.x; s < num_shares; s += gridDim.x, ++it) {
            const int st = it % NSTAGE;
            const uint32_t ph = (it / NSTAGE) & 1u;
            uint32_t *buf = stage_buf + st * STAGE_WORDS;
            mbar_wait(&empty[st], ph ^ 1u);
            const unsigned long long out0 = s * SH;
            const int cnt = static_cast<int>(min(static_cast<unsigned long long>(SH), n - out0));
            ShareMeta m;
            m.cnt = cnt;
            if (small_round) {
                m.a_off = 0; m.a_len = 0; m.b_off = 0; m.b_len = 0;
                if ((cnt & 3) == 0) {
                    if (lane == 0) {
                        meta[st] = m;
                        mbar_arrive_expect_tx(&full[st], static_cast<uint32_t>(cnt) * 4u);
                        bulk_g2s(buf, kin + out0, static_cast<uint32_t>(cnt) * 4u, &full[st]);
                    }
                } else {   // ragged end of the array: plain cooperative copy
                    for (int i = lane; i < cnt; i += 32) buf[i] = kin[out0 + i];
                    __syncwarp();
                    if (lane == 0) { meta[st] = m; mbar_arrive(&full[st]); }
                }
            } else {
                const unsigned long long a0 = out0 / (2 * L) * (2 * L);
                const unsigned long long alen = min(L, n - a0);
                const unsigned long long b0 = a0 + alen;
                const unsigned long long blen = min(L, n - b0);
                const unsigned long long D0 = out0 - a0, D1 = D0 + cnt;
                const unsigned long long I0 = splits[s];
                const unsigned long long I1 = (D1 >= alen + blen) ? alen : splits[s + 1];
                const unsigned long long ga = a0 + I0, gb = b0 + (D0 - I0);
                const int la = static_cast<int>(I1 - I0), lb = cnt - la;
                const unsigned long long sa = ga & ~3ull, ea = (ga + la + 3) & ~3ull;
                const unsigned long long sb = gb & ~3ull, eb = (gb + lb + 3) & ~3ull;
                const int wordsA = la ? static_cast<int>(ea - sa) : 0;
                const int wordsB = lb ? static_cast<int>(eb - sb) : 0;
                m.a_off = static_cast<int>(ga - sa);
                m.a_len = la;
                m.b_off = wordsA + static_cast<int>(gb - sb);
                m.b_len = lb;
                const bool bulk_ok = (!la || ea <= n) && (!lb || eb <= n);
                if (bulk_ok) {
                    if (lane == 0) {
                        meta[st] = m;
                        mbar_arrive_expect_tx(&full[st], static_cast<uint32_t>(wordsA + wordsB) * 4u);
                        if (la) bulk_g2s(buf, kin + sa, static_cast<uint32_t>(wordsA) * 4u, &full[st]);
                        if (lb) bulk_g2s(buf + wordsA, kin + sb, static_cast<uint32_t>(wordsB) * 4u, &full[st]);
                    }
                } else {
                    for (int i = lane; i < la; i += 32) buf[m.a_off + i] = kin[ga + i];
                    for (int i = lane; i < lb; i += 32) buf[m.b_off + i] = kin[gb + i];
                    __syncwarp();
                    if (lane == 0) { meta[st] = m; mbar_arrive(&full[st]); }
                }
            }
        }
        return;
    }

    // ============================== consumer warps
    uint32_t *planes = planes_all + warp * TILE;
    const int tile_off = warp * TILE;
    unsigned int it = 0;
    for (unsigned long long s = blockIdx.x; s < num_shares; s += gridDim.x, ++it) {
        const int st = it % NSTAGE;
        const uint32_t ph = (it / NSTAGE) & 1u;
        const uint32_t *buf = stage_buf + st * STAGE_WORDS;
        mbar_wait(&full[st], ph);
        const ShareMeta m = meta[st];
        if (tile_off >= m.cnt) {            // ragged last share: nothing for this warp
            __syncwarp();
            if (lane == 0) mbar_arrive(&empty[st]);
            continue;
        }
        int sA, la, sB, lb, d0;
        if (small_round) {
            const int l = static_cast<int>(L);
            const int pb = tile_off / (2 * l) * (2 * l);
            la = min(l, m.cnt - pb);
            lb = min(l, m.cnt - pb - la);
            sA = pb; sB = pb + la; d0 = tile_off - pb;
        } else {
            sA = m.a_off; la = m.a_len; sB = m.b_off; lb = m.b_len; d0 = tile_off;
        }
        const int d1 = min(d0 + TILE, la + lb);
        const int i0 = corank_smem(buf, sA, la, sB, lb, d0, lane);
        const int i1 = corank_smem(buf, sA, la, sB, lb, d1, lane);
        const int a = i1 - i0;                   // elements of A in this sub-tile
        const int b = (d1 - d0) - a;             // elements of B
        // column layout straight from the stage buffer: position p = 32 k + lane is A'[p] for p < a,
        // B'[1023 - p] for p >= 1024 - b, the maximum element in between (partial sub-tiles only).
        // Two predicated loads per k: within each the active lanes read consecutive words.
        const uint32_t addrA = smem_u32(buf + sA + i0 + lane);
        const uint32_t addrB = smem_u32(buf + sB + (d0 - i0) + (TILE - 1) - lane);
        const int xa = a - lane;                 // p < a        <=>  32 k < xa
        const int xb = lane - (TILE - b);        // p >= 1024-b  <=>  32 k >= -xb  <=>  32 k + xb >= 0
        uint32_t v[1][32];
        load_columns(v[0], xa, xb, addrA, addrB, std::make_integer_sequence<int, 32>{});
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[st]);  // stage buffer may be refilled

        line_bitonic_merge<1>(v);                // column pass
        col_store<false>(planes, v[0], lane);
        __syncwarp();
        row_load(planes, v[0], lane);
        line_bitonic_merge<1>(v);                // row pass
        const int cnt = d1 - d0;
        store_rows<Elem<1, false>>(planes, kout, nullptr, s * SH + tile_off, cnt, cnt == TILE, lane, v);
    }
}

}  // namespace pipe
}  // namespace bcf
