// bcf_tu_isolate.cu -- the bank-conflict ISOLATION EXPERIMENT (debug entry points, never on the product path).
//
// north_star asks for l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_{ld,st} = 0 on the sort and merge kernels.
// Every LDS/STS of those kernels touches 32 distinct banks (host bank model, per-instruction "excessive wavefronts"
// = 0 in ncu's source view), yet the kernel-level hardware counter is not 0 on grids with more than one wave.
// DESIGN.md section 7 attributes the difference to arbitration: global-memory traffic of the same SM (LDG returns,
// STG data, TMA writes) moves through the same SRAM banks as the shared-memory wavefronts.  The two kernels below
// test that claim.  They execute the SAME shared-memory instruction streams as the production kernels (the same
// device functions: corank_smem, load_columns, line_bitonic_merge, col_store, row_load, row_store, the un-skewing
// LDS.128 of the store path; tile_merge_level) but in three phases separated by CTA barriers:
//     phase 1  global -> chip      (TMA bulk copies / LDG.128), nothing else
//     phase 2  every LDS / STS of the work item, results parked in registers
//     phase 3  registers -> global (STG.128), nothing else
// With `exclusive` = 1 the launch asks for enough dynamic shared memory that ONE CTA is resident per SM, so no other
// CTA's phase 1 / 3 can overlap this CTA's phase 2: if the counter is caused by arbitration it must read 0.  With
// `exclusive` = 0 the same code runs with several CTAs per SM (their phases interleave): the counter must come back.
// (The merge round has the production shape since r3 -- 16-page shares, 16 warps, ~196 KB of shared memory -- so one
// CTA per SM is all that fits and `exclusive` makes no difference for it; the production kernel it is compared with
// is also one CTA per SM, whose TMA writes and global stores overlap its own LDS / STS.)
// profiles/r3_conflict_isolation.md holds the measured table (r2_conflict_isolation.md: the older 8-page shape).
#include "bcf_internal.cuh"
#include "bcf_merge_pipe.cuh"

namespace bcf {
namespace isolate {

using E = Elem<1, false>;
// the shape of the experiment follows the production merge kernel for uint32 keys (pipe::Cfg<E>): the same share size
// (16 pages), one page per consumer warp (16 warps), two stage buffers -- so ONE CTA fills an SM here exactly as in
// merge_pipe_kernel<u32>, and whatever the production counter shows comes from that CTA's own concurrent traffic
// (TMA writes into the stage buffers, STG data), not from a neighbour CTA.
constexpr int NW = pipe::Cfg<E>::PAGES;
constexpr int SH = pipe::Cfg<E>::SH;
constexpr int NSTAGE = pipe::Cfg<E>::STAGES;
constexpr int THREADS = NW * 32;
static_assert(NW == pipe::Cfg<E>::NWC, "one consumer warp per page, as in the production kernel");
struct C {
    static constexpr size_t stage_bytes = size_t(SH) * 4 + pipe::REGION_SLACK;
    static constexpr size_t scratch_off = NSTAGE * stage_bytes;
    static constexpr size_t meta_off = scratch_off + size_t(NW) * TILE * 4;
    static constexpr size_t bar_off = meta_off + NSTAGE * sizeof(pipe::ShareMeta);
    static constexpr size_t total = bar_off + NSTAGE * 8;
};
static_assert(C::total + 1024 <= 227 * 1024, "the experiment's CTA must fit one SM");
constexpr size_t EXCLUSIVE_SMEM = 120 * 1024;      // more than half of the 227 KB an SM offers: one CTA per SM

// One merge round on u32 keys, runs of L = 1024 * 2^k >= SH, n a multiple of 2 L: each CTA merges NSTAGE shares.
__global__ void __launch_bounds__(THREADS, 1)
merge_round_isolated_kernel(const uint32_t *__restrict__ kin, uint32_t *__restrict__ kout, const uint32_t *__restrict__ splits,
                            const unsigned long long n, const unsigned long long L, const unsigned long long num_shares)
{
    pdl_entry();
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint32_t *scratch_all = reinterpret_cast<uint32_t *>(smem_raw + C::scratch_off);
    pipe::ShareMeta *meta = reinterpret_cast<pipe::ShareMeta *>(smem_raw + C::meta_off);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + C::bar_off);
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const unsigned long long s0 = static_cast<unsigned long long>(blockIdx.x) * NSTAGE;

    if (threadIdx.x == 0) {
        for (int st = 0; st < NSTAGE; ++st) pipe::mbar_init(&full[st], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    // ---------------- phase 1: the TMA engine writes the stage buffers; no thread touches shared data meanwhile
    // (the share descriptors of BOTH stages are written before the first bulk copy is issued)
    if (threadIdx.x == 0) {
        const uint32_t *src[NSTAGE][2];
        int cnt[NSTAGE][2];
        for (int st = 0; st < NSTAGE && s0 + st < num_shares; ++st) {
            const unsigned long long s = s0 + st;
            const unsigned long long out0 = s * SH;
            const unsigned long long a0 = out0 / (2 * L) * (2 * L);
            const unsigned long long b0 = a0 + L;
            const unsigned long long D0 = out0 - a0, D1 = D0 + SH;
            const unsigned long long I0 = splits[s];
            const unsigned long long I1 = (D1 >= 2 * L) ? L : splits[s + 1];
            const unsigned long long ga = a0 + I0, gb = b0 + (D0 - I0);
            const int la = static_cast<int>(I1 - I0), lb = SH - la;
            unsigned long long ksa, kea, ksb, keb;
            pipe::aligned_superset<4>(ga, la, ksa, kea);
            pipe::aligned_superset<4>(gb, lb, ksb, keb);
            const int kA = la ? static_cast<int>(kea - ksa) : 0;
            const int kB = lb ? static_cast<int>(keb - ksb) : 0;
            pipe::ShareMeta m;
            m.cnt = SH; m.pad = 0;
            m.a_len = la; m.b_len = lb;
            m.ka_off = static_cast<int>(ga - ksa);
            m.kb_off = kA + static_cast<int>(gb - ksb);
            m.va_off = 0; m.vb_off = 0;
            meta[st] = m;
            src[st][0] = kin + ksa; cnt[st][0] = kA;
            src[st][1] = kin + ksb; cnt[st][1] = kB;
        }
        for (int st = 0; st < NSTAGE && s0 + st < num_shares; ++st) {
            unsigned char *kreg = smem_raw + st * C::stage_bytes;
            pipe::mbar_arrive_expect_tx(&full[st], static_cast<uint32_t>(cnt[st][0] + cnt[st][1]) * 4u);
            if (cnt[st][0]) pipe::bulk_g2s(kreg, src[st][0], static_cast<uint32_t>(cnt[st][0]) * 4u, &full[st]);
            if (cnt[st][1]) pipe::bulk_g2s(kreg + size_t(cnt[st][0]) * 4, src[st][1], static_cast<uint32_t>(cnt[st][1]) * 4u, &full[st]);
        }
    }
    for (int st = 0; st < NSTAGE && s0 + st < num_shares; ++st) pipe::mbar_wait(&full[st], 0);
    __syncthreads();

    // ---------------- phase 2: all shared-memory work of both shares, outputs parked in registers
    uint32_t *scratch = scratch_all + warp * TILE;
    uint4 out[NSTAGE][8];
#pragma unroll
    for (int st = 0; st < NSTAGE; ++st) {
        if (s0 + st < num_shares) {
            const unsigned char *kreg = smem_raw + st * C::stage_bytes;
            const pipe::ShareMeta m = meta[st];
            const int d0 = warp * TILE, d1 = d0 + TILE;
            const int i0 = pipe::corank_smem<E>(kreg, kreg, m, d0, lane);
            const int i1 = pipe::corank_smem<E>(kreg, kreg, m, d1, lane, i0, i0 + TILE);
            const int a = i1 - i0, b = TILE - a;
            const uint32_t kA = pipe::smem_u32(kreg) + static_cast<uint32_t>(m.ka_off + i0 + lane) * 4u;
            const uint32_t kB = pipe::smem_u32(kreg) + static_cast<uint32_t>(m.kb_off + (d0 - i0) + (TILE - 1) - lane) * 4u;
            uint32_t v[1][32];
            pipe::load_columns<E>(v, a - lane, lane - (TILE - b), kA, kB, kA, kB, std::make_integer_sequence<int, 32>{});
            line_bitonic_merge<1>(v);
            col_store<false>(scratch, v[0], lane);
            __syncwarp();
            row_load(scratch, v[0], lane);
            line_bitonic_merge<1>(v);
            __syncwarp();
            row_store(scratch, v[0], lane);
            __syncwarp();
#pragma unroll
            for (int q = 0; q < 8; ++q)
                out[st][q] = *reinterpret_cast<const uint4 *>(scratch + chunk_word(4 * q + (lane >> 3), lane & 7));
            __syncwarp();
        }
    }
    __syncthreads();

    // ---------------- phase 3: global stores only
#pragma unroll
    for (int st = 0; st < NSTAGE; ++st) {
        if (s0 + st < num_shares) {
            uint4 *pk = reinterpret_cast<uint4 *>(kout + (s0 + st) * SH + warp * TILE);
#pragma unroll
            for (int q = 0; q < 8; ++q) stg128(pk + 32 * q + lane, out[st][q]);
        }
    }
}

// Tile mergesort of whole u32 tiles, one tile per warp, one CTA of WARPS_PER_CTA warps per WARPS_PER_CTA tiles.
__global__ void __launch_bounds__(WARPS_PER_CTA * 32, 1)
tile_mergesort_isolated_kernel(uint32_t *__restrict__ keys, const size_t num_tiles)
{
    pdl_entry();
    extern __shared__ __align__(16) uint32_t smem[];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    uint32_t *planes = smem + warp * TILE;
    const size_t tile = static_cast<size_t>(blockIdx.x) * WARPS_PER_CTA + warp;
    const bool active = tile < num_tiles;
    uint32_t v[1][32];
    // phase 1: global loads only
    if (active) load_tile_vec<E>(keys, nullptr, tile * TILE, lane, v);
    __syncthreads();
    // phase 2: the whole network, every LDS / STS of the tile
    uint4 out[8];
    if (active) {
        line_sort<1, BCF_TMS_FMA_MOD>(v);
        tile_merge_level<E, 1>(planes, lane, v);
        tile_merge_level<E, 2>(planes, lane, v);
        tile_merge_level<E, 3>(planes, lane, v);
        tile_merge_level<E, 4>(planes, lane, v);
        tile_merge_level<E, 5>(planes, lane, v);
        row_store(planes, v[0], lane);
        __syncwarp();
#pragma unroll
        for (int q = 0; q < 8; ++q) out[q] = *reinterpret_cast<const uint4 *>(planes + chunk_word(4 * q + (lane >> 3), lane & 7));
    }
    __syncthreads();
    // phase 3: global stores only
    if (active) {
        uint4 *pk = reinterpret_cast<uint4 *>(keys + tile * TILE);
#pragma unroll
        for (int q = 0; q < 8; ++q) stg128(pk + 32 * q + lane, out[q]);
    }
}

}  // namespace isolate

size_t isolated_share() { return isolate::SH; }

bcf_status launch_isolated_merge_round(const Call &c, const uint32_t *kin, uint32_t *kout, const uint32_t *splits, size_t n,
                                       size_t run_len, int exclusive)
{
    const unsigned long long shares = n / isolate::SH;
    const size_t smem = exclusive ? (isolate::EXCLUSIVE_SMEM > isolate::C::total ? isolate::EXCLUSIVE_SMEM : isolate::C::total)
                                  : isolate::C::total;
    // the attribute is set to the larger size once; the launch asks for what this call wants
    const bcf_status st = ensure_dyn_smem<isolate::merge_round_isolated_kernel>(
        c.dev, isolate::EXCLUSIVE_SMEM > isolate::C::total ? isolate::EXCLUSIVE_SMEM : isolate::C::total);
    if (st != BCF_OK) return st;
    LaunchTimer t(BCF_KERNEL_MERGE, c.s);
    return launch(c, isolate::merge_round_isolated_kernel, static_cast<unsigned>((shares + isolate::NSTAGE - 1) / isolate::NSTAGE),
                  isolate::THREADS, smem, kin, kout, splits, static_cast<unsigned long long>(n),
                  static_cast<unsigned long long>(run_len), shares);
}

bcf_status launch_isolated_tile_mergesort(const Call &c, uint32_t *keys, size_t num_tiles, int exclusive)
{
    const size_t own = WARPS_PER_CTA * size_t(TILE) * 4;
    const size_t smem = exclusive ? isolate::EXCLUSIVE_SMEM : own;
    const bcf_status st = ensure_dyn_smem<isolate::tile_mergesort_isolated_kernel>(c.dev, isolate::EXCLUSIVE_SMEM);
    if (st != BCF_OK) return st;
    LaunchTimer t(BCF_KERNEL_TILE_SORT, c.s);
    return launch(c, isolate::tile_mergesort_isolated_kernel, static_cast<unsigned>((num_tiles + WARPS_PER_CTA - 1) / WARPS_PER_CTA),
                  WARPS_PER_CTA * 32, smem, keys, num_tiles);
}

}  // namespace bcf
