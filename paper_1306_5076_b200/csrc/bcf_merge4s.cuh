// bcf_merge4s.cuh -- the four-run pass (bcf_merge4.cuh) as a STREAM of page tasks: no CTA-wide barrier.
//
// Same work as pipe4::merge4_pipe_kernel for rounds with 4 L > SH -- X = merge(A, B), Y = merge(C, D) of a share
// into shared memory (level 1), Z = merge(X, Y) to global memory (level 2), every page the paper's conflict-free
// SHEARSORT-MERGE (reading A8) -- but the two levels of a share are not separated by
// barriers that stop all warps of the CTA (ncu on the barrier version: `barrier` was the largest stall, 1.2 per
// issued instruction, profiles/r1b_merge4_full.md).  Instead:
//
//   * X and Y go to their own buffer (two of them, alternating) instead of back into the stage buffer, so a stage
//     is released as soon as its level-1 pages are in registers;
//   * the page merges of the CTA form one sequence of TASKS
//         L1(0) | L1(1) L2(0) | L1(2) L2(1) | ...        L1(i) = 9 page slots of level 1 of the CTA's share i,
//                                                         L2(i) = 8 pages of level 2
//     and consumer warp w takes tasks w, w + NWC, w + 2 NWC, ... in this order, with NWC = 17 = the tasks of a
//     block: warps 0-8 are the level-1 page slots and warps 9-16 the level-2 pages of every share.  L2(i) comes a
//     whole block after L1(i), so by the time a warp reaches a level-2 page its inputs are normally complete.
//     (NWC must divide into the block like this: an mbarrier wait names its phase by ONE parity bit, which is
//     only sound if the waiting warp has itself seen the previous phase of that barrier complete.  With 19 warps
//     rotating through the slots a warp could reach the second use of a buffer without having taken part in the
//     first, and pass the wait on the first fill -- observed as an illegal address on garbage meta data.)
//   * four mbarrier pairs carry the dependences: full / empty per stage buffer (TMA landed / level-1 pages
//     loaded), xfull / xempty per X-Y buffer (all level-1 pages stored / all level-2 pages loaded).  Every task
//     waits only for tasks that precede it in the sequence and every warp works through its tasks in sequence
//     order, so the waits cannot form a cycle.
//
// One CTA per SM (4 share-sized buffers + one scratch plane per warp fill the shared memory), NWC consumer warps
// + the TMA producer warp.  Keys only (u32): for the wider element types four buffers do not fit and the barrier
// version stays in use, as it does for the rounds with 4 L <= SH.
#pragma once
#include "bcf_merge4.cuh"

namespace bcf {
namespace pipe4s {

using pipe::ShareMeta;
using pipe4::SH;
using pipe4::NT;

#ifndef BCF_M4S_NWC
#define BCF_M4S_NWC 17            // consumer warps = tasks per block (see above); 18 warps per SM, 96 registers
#endif
#ifndef BCF_M4S_FMOD
#define BCF_M4S_FMOD 2            // every second comparator forms its max on the FMA pipe (measured: 0 -> 0.702, 2 -> 0.675,
                                  // 3 -> 0.697 ms per launch at 2^28 keys: the ALU pipe and the issue slots are both near their limit)
#endif
constexpr int NWC = BCF_M4S_NWC;
constexpr int THREADS = (NWC + 1) * 32;
constexpr int L1_SLOTS = NT + 1;                 // level-1 page slots per share
constexpr int TASKS = L1_SLOTS + NT;             // tasks per block of the sequence
static_assert(TASKS % NWC == 0, "every warp must meet every phase of the barriers it waits on (see the header comment)");
constexpr int NBUF = 2;

struct StageMeta {
    ShareMeta pair[2];   // level-1 pairs (a, b) and (c, d) inside the stage buffer
    int cnt;             // outputs of the share
    int pad[3];
};
struct XYMeta {
    int len_x, len_y;    // |X|, |Y|
    int w_y;             // element offset of Y inside the X-Y buffer (multiple of 4)
    int cnt;
};

template <class E>
struct Cfg4s {
    using B = pipe4::Cfg4<E>;
    static constexpr size_t stage_bytes = B::stage_bytes;
    static constexpr size_t xy_off = NBUF * stage_bytes;
    static constexpr size_t scratch_off = xy_off + NBUF * stage_bytes;
    static constexpr size_t meta_off = scratch_off + size_t(NWC) * TILE * 4;
    static constexpr size_t xmeta_off = meta_off + NBUF * sizeof(StageMeta);
    static constexpr size_t bar_off = xmeta_off + NBUF * sizeof(XYMeta);
    static constexpr size_t total = bar_off + 4 * NBUF * 8;
    static constexpr bool fits = (total + 1024 <= 227 * 1024);
    static constexpr int max_regs = (16384 / (((NWC + 1) + 3) / 4 * 32)) / 8 * 8;
};

template <class E>
__global__ void __maxnreg__(Cfg4s<E>::max_regs)
merge4_stream_kernel(const void *__restrict__ kin_, const uint32_t *__restrict__ vin, void *__restrict__ kout,
                     uint32_t *__restrict__ vout, const uint4 *__restrict__ splits, const unsigned long long n,
                     const unsigned long long L, const unsigned long long num_shares)
{
    pdl_entry();
    using C = Cfg4s<E>;
    using B = typename C::B;
    constexpr int KB = B::KB;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint32_t *scratch_all = reinterpret_cast<uint32_t *>(smem_raw + C::scratch_off);
    StageMeta *meta = reinterpret_cast<StageMeta *>(smem_raw + C::meta_off);
    XYMeta *xmeta = reinterpret_cast<XYMeta *>(smem_raw + C::xmeta_off);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + C::bar_off);
    uint64_t *empty = full + NBUF;
    uint64_t *xfull = empty + NBUF;
    uint64_t *xempty = xfull + NBUF;
    const unsigned char *kin = static_cast<const unsigned char *>(kin_);

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    // shares of this CTA: blockIdx.x, blockIdx.x + gridDim.x, ...
    const unsigned int my_shares =
        blockIdx.x < num_shares ? static_cast<unsigned int>((num_shares - blockIdx.x + gridDim.x - 1) / gridDim.x) : 0u;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NBUF; ++s) {
            pipe::mbar_init(&full[s], 1);
            pipe::mbar_init(&empty[s], L1_SLOTS);
            pipe::mbar_init(&xfull[s], L1_SLOTS);
            pipe::mbar_init(&xempty[s], NT);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NWC) {
        // ============================== producer warp: the four pieces of a share by TMA (as in bcf_merge4.cuh)
        for (unsigned int it = 0; it < my_shares; ++it) {
            const unsigned long long s = blockIdx.x + static_cast<unsigned long long>(it) * gridDim.x;
            const int st = it % NBUF;
            const uint32_t ph = (it / NBUF) & 1u;
            unsigned char *kreg = smem_raw + st * C::stage_bytes;
            unsigned char *vreg = kreg + B::key_region;
            pipe::mbar_wait(&empty[st], ph ^ 1u);
            const unsigned long long out0 = s * SH;
            const int cnt = static_cast<int>(min(static_cast<unsigned long long>(SH), n - out0));
            const unsigned long long g0 = out0 / (4 * L) * (4 * L);
            const unsigned long long D0 = out0 - g0, D1 = D0 + cnt;
            const uint4 s0 = splits[s];
            uint4 s1 = splits[s + 1];
            unsigned long long rs[4], rl[4], total = 0;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                rs[r] = g0 + r * L;
                rl[r] = rs[r] < n ? min(L, n - rs[r]) : 0ull;
                total += rl[r];
            }
            if (D1 >= total) s1 = make_uint4((uint32_t)rl[0], (uint32_t)rl[1], (uint32_t)rl[2], (uint32_t)rl[3]);
            const uint32_t p0[4] = {s0.x, s0.y, s0.z, s0.w};
            const uint32_t p1[4] = {s1.x, s1.y, s1.z, s1.w};
            unsigned long long g[4], ks[4], vs[4];
            int len[4], koff[4], voff[4], kcnt[4], vcnt[4];
            int kacc = 0, vacc = 0;
            bool bulk_ok = true;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                g[r] = rs[r] + p0[r];
                len[r] = static_cast<int>(p1[r] - p0[r]);
                unsigned long long ke, ve;
                pipe::aligned_superset<KB>(g[r], len[r], ks[r], ke);
                kcnt[r] = len[r] ? static_cast<int>(ke - ks[r]) : 0;
                koff[r] = kacc + static_cast<int>(g[r] - ks[r]);
                kacc += kcnt[r];
                bulk_ok = bulk_ok && (!len[r] || ke <= n);
                vs[r] = 0; vcnt[r] = 0; voff[r] = 0;
                if constexpr (E::HAS_VAL) {
                    pipe::aligned_superset<4>(g[r], len[r], vs[r], ve);
                    vcnt[r] = len[r] ? static_cast<int>(ve - vs[r]) : 0;
                    voff[r] = vacc + static_cast<int>(g[r] - vs[r]);
                    vacc += vcnt[r];
                    bulk_ok = bulk_ok && (!len[r] || ve <= n);
                }
            }
            if (lane == 0) {
                StageMeta &M = meta[st];
                M.cnt = cnt;
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    ShareMeta m;
                    m.cnt = 0; m.pad = 0;
                    m.a_len = len[2 * q]; m.b_len = len[2 * q + 1];
                    m.ka_off = koff[2 * q]; m.kb_off = koff[2 * q + 1];
                    m.va_off = voff[2 * q]; m.vb_off = voff[2 * q + 1];
                    M.pair[q] = m;
                }
            }
            if (bulk_ok) {
                if (lane == 0) {
                    pipe::mbar_arrive_expect_tx(&full[st], static_cast<uint32_t>(kacc) * KB + static_cast<uint32_t>(vacc) * 4u);
                    int ka = 0, va = 0;
#pragma unroll
                    for (int r = 0; r < 4; ++r) {
                        if (len[r]) {
                            pipe::bulk_g2s(kreg + size_t(ka) * KB, kin + ks[r] * KB, static_cast<uint32_t>(kcnt[r]) * KB, &full[st]);
                            if constexpr (E::HAS_VAL)
                                pipe::bulk_g2s(vreg + size_t(va) * 4, vin + vs[r], static_cast<uint32_t>(vcnt[r]) * 4u, &full[st]);
                        }
                        ka += kcnt[r];
                        va += vcnt[r];
                    }
                }
            } else {   // a piece's aligned superset would reach past the end of the array: plain cooperative copy
                uint32_t *kw = reinterpret_cast<uint32_t *>(kreg);
                const uint32_t *gk = reinterpret_cast<const uint32_t *>(kin);
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    for (int i = lane; i < len[r] * (KB / 4); i += 32) kw[koff[r] * (KB / 4) + i] = gk[g[r] * (KB / 4) + i];
                    if constexpr (E::HAS_VAL) {
                        uint32_t *vw = reinterpret_cast<uint32_t *>(vreg);
                        for (int i = lane; i < len[r]; i += 32) vw[voff[r] + i] = vin[g[r] + i];
                    }
                }
                __syncwarp();
                if (lane == 0) pipe::mbar_arrive(&full[st]);
            }
        }
        return;
    }

    // ============================== consumer warps: tasks warp, warp + NWC, ... of the sequence
    uint32_t *scratch = scratch_all + warp * TILE;
    for (unsigned int t = warp;; t += NWC) {
        const unsigned int blk = t / TASKS;
        const int r = static_cast<int>(t % TASKS);
        if (blk > my_shares) break;
        uint32_t v[E::NP][32];
        if (r < L1_SLOTS) {
            // ---------------- level 1, share `blk` of the CTA, page slot r: a page of X = merge(A, B) or of Y = merge(C, D)
            if (blk >= my_shares) continue;
            const unsigned int it = blk;
            const int st = it % NBUF;
            const uint32_t ph = (it / NBUF) & 1u;
            const unsigned char *kreg = smem_raw + st * C::stage_bytes;
            const unsigned char *vreg = kreg + B::key_region;
            unsigned char *xk = smem_raw + C::xy_off + st * C::stage_bytes;       // X-Y buffer of this share
            unsigned char *xv = xk + B::key_region;
            pipe::mbar_wait(&full[st], ph);
            const StageMeta &M = meta[st];
            const int len_x = M.pair[0].a_len + M.pair[0].b_len;
            const int len_y = M.pair[1].a_len + M.pair[1].b_len;
            const int share_cnt = M.cnt;
            const int pages_x = (len_x + TILE - 1) / TILE;
            const int pages_y = (len_y + TILE - 1) / TILE;
            const int w_y = (len_x + 3) & ~3;
            const int q = r < pages_x ? 0 : 1;
            const int j = r - (q ? pages_x : 0);
            const bool work = j < (q ? pages_y : pages_x);
            int cnt1 = 0;
            if (work) {
                const ShareMeta m = M.pair[q];
                cnt1 = pipe4::load_page<E>(kreg, vreg, m, j, lane, v);
            }
            __syncwarp();
            if (lane == 0) pipe::mbar_arrive(&empty[st]);          // the stage may be refilled
            if (work) {
                line_bitonic_merge<E::NP, BCF_M4S_FMOD>(v);
#pragma unroll
                for (int p = 0; p < E::NP; ++p) {
                    if (p) __syncwarp();
                    col_store<false>(scratch, v[p], lane);
                    __syncwarp();
                    row_load(scratch, v[p], lane);
                }
                line_bitonic_merge<E::NP, BCF_M4S_FMOD>(v);
            }
            pipe::mbar_wait(&xempty[st], ph ^ 1u);                 // level 2 of the share two back has read this buffer
            if (r == 0 && lane == 0) {
                XYMeta xm;
                xm.len_x = len_x; xm.len_y = len_y; xm.w_y = w_y; xm.cnt = share_cnt;
                xmeta[st] = xm;
            }
            if (work)
                pipe4::store_rows_to<E, true>(scratch, xk, reinterpret_cast<uint32_t *>(xv), static_cast<size_t>((q ? w_y : 0) + j * TILE),
                                              cnt1, cnt1 == TILE, lane, v);
            __syncwarp();
            if (lane == 0) pipe::mbar_arrive(&xfull[st]);
        } else {
            // ---------------- level 2, share `blk - 1` of the CTA, page r - L1_SLOTS of Z = merge(X, Y)
            if (blk == 0) continue;
            const unsigned int it = blk - 1;
            const int st = it % NBUF;
            const uint32_t ph = (it / NBUF) & 1u;
            const unsigned char *xk = smem_raw + C::xy_off + st * C::stage_bytes;
            const unsigned char *xv = xk + B::key_region;
            const int j = r - L1_SLOTS;
            pipe::mbar_wait(&xfull[st], ph);
            const XYMeta xm = xmeta[st];
            int cnt2 = 0;
            if (j * TILE < xm.cnt) {
                ShareMeta m;
                m.cnt = 0; m.pad = 0;
                m.a_len = xm.len_x; m.b_len = xm.len_y;
                m.ka_off = 0; m.kb_off = xm.w_y;
                m.va_off = 0; m.vb_off = xm.w_y;
                cnt2 = pipe4::load_page<E>(xk, xv, m, j, lane, v);
            }
            __syncwarp();
            if (lane == 0) pipe::mbar_arrive(&xempty[st]);         // the X-Y buffer may be overwritten
            if (cnt2) {
                line_bitonic_merge<E::NP, BCF_M4S_FMOD>(v);
#pragma unroll
                for (int p = 0; p < E::NP; ++p) {
                    if (p) __syncwarp();
                    col_store<false>(scratch, v[p], lane);
                    __syncwarp();
                    row_load(scratch, v[p], lane);
                }
                line_bitonic_merge<E::NP, BCF_M4S_FMOD>(v);
                const unsigned long long s = blockIdx.x + static_cast<unsigned long long>(it) * gridDim.x;
                pipe4::store_rows_to<E, false>(scratch, kout, vout, s * SH + static_cast<unsigned long long>(j) * TILE, cnt2,
                                               cnt2 == TILE, lane, v);
            }
        }
    }
}

}  // namespace pipe4s
}  // namespace bcf
