// bcf_merge4.cuh -- four runs per pass: TWO merge rounds of BCFMergesort per read + write of the data
// ("multi-way merging per pass ... with the same in-smem machinery").
//
// PAPER.md section 3 (L103) merges pairs of runs in ceil(log2(N/M)) rounds and Lemma 2 (L145)
// charges one scan of global memory per round.  Every round is HBM-bound on B200 while the
// conflict-free SHEARSORT-MERGE of a page (L129, L418) leaves the ALUs mostly idle, so this kernel
// keeps a share on chip for two consecutive rounds: the four runs (A, B, C, D) of a group are merged
// as X = merge(A, B), Y = merge(C, D) -- level 1, written back into shared memory -- and
// Z = merge(X, Y) -- level 2, written to global memory.  Both levels are the paper's page merge
// unchanged (one bitonic page of w*w elements per warp, column pass, skewed transpose, row pass);
// the comparisons done and the result are those of two rounds of section 3, only the intermediate
// runs never travel to HBM.
//
//   share     = SH = 8 * 1024 consecutive outputs of the pass.
//   partition = partition4_kernel: for every share boundary the number of elements each of the four
//               runs contributes to the outputs before it (multi-sequence selection, below).
//   producer  = one warp: TMA bulk copies of the (up to) four pieces of a share into a stage buffer.
//   consumers = 9 warps.  Level 1 has up to 9 page merges (the pieces of X and of Y rarely end on a
//               page boundary), level 2 exactly ceil(cnt / 1024) <= 8.  Level 1 reads the stage
//               buffer into registers, a named barrier separates the last read from the first
//               write, and the merged pages go back INTO the same stage buffer (X at offset 0, Y
//               behind it), so no third buffer is needed and two CTAs fit one SM.
#pragma once
#include "bcf_merge_pipe.cuh"

namespace bcf {
namespace pipe4 {

using pipe::NSTAGE;
using pipe::ShareMeta;

constexpr int NT = 8;                    // pages per share = level-2 consumer warps
constexpr int SH = NT * TILE;            // outputs per share
constexpr int NWC = NT + 1;              // consumer warps (level 1 can have NT + 1 pages)
constexpr int THREADS = (NWC + 1) * 32;
constexpr int REGION_SLACK = 128;        // bytes: aligned supersets of four pieces + alignment of Y

struct Meta4 {
    ShareMeta pair[4];   // level-1 pairs: pieces (a, b) inside the stage buffer
    int w[4];            // element offset at which pair q's merged output is written (multiple of 4)
    int cnt;             // outputs of this share
    int npairs;          // level-1 pairs in use; level-2 pair p merges the outputs of pairs 2p, 2p+1
    int pad0, pad1;
};

template <class E>
struct Cfg4 {
    static constexpr int KB = E::KEY_BYTES;
    static constexpr size_t key_region = size_t(SH) * KB + REGION_SLACK;
    static constexpr size_t val_region = E::HAS_VAL ? size_t(SH) * 4 + REGION_SLACK : 0;
    static constexpr size_t stage_bytes = key_region + val_region;
    static constexpr size_t scratch_off = NSTAGE * stage_bytes;
    static constexpr size_t meta_off = scratch_off + size_t(NWC) * TILE * 4;
    static constexpr size_t bar_off = meta_off + NSTAGE * sizeof(Meta4);
    static constexpr size_t total = bar_off + 2 * NSTAGE * 8;
    static constexpr bool fits = (total + 1024 <= 227 * 1024);
    static constexpr int ctas_per_sm = (2 * (total + 1024) <= 227 * 1024) ? 2 : 1;
};

// ------------------------------------------------------------------ a5 for four runs: multi-sequence selection
//
// For share boundary s (output position out0 = SH * s of the pass) inside its group of four runs
// R_0..R_3 (run r = elements [g0 + r L, g0 + (r+1) L) clipped to n): the split (p_0, .., p_3),
// sum p_r = d = out0 - g0, such that every element left of the split precedes every element right
// of it in the order (element, run index, position) -- the first d outputs of the stable 4-way
// merge.  That order is strict, so the split is unique; elements that compare equal are bitwise
// identical, so the outputs do not depend on the tie rule (reading A11/A12).
//
// Search: the classical halving scheme for multi-sequence selection.  At step size h (a power of
// two, from H >= L down to 1) only the last element of every block of h elements of a run is
// looked at; c_r counts blocks of run r left of the split and the target is floor(d / h) blocks.
// Going from h to h / 2 doubles c_r, and the split is repaired by single-block moves: while the
// largest left boundary element exceeds the smallest right boundary element, the two runs
// exchange a block (each exchange moves both runs towards the unique solution, so the loop
// terminates; measured <= 4 moves per level).  At h = 1 the block split IS the element split.
// Runs shorter than H are padded with elements larger than every real one.  One thread per
// boundary; log2(H) + 1 levels of 4 independent loads plus ~1.2 dependent moves.
struct SelElem {
    unsigned long long key;
    uint32_t val;
    uint32_t kind;   // 0: -inf (no left neighbour), 1: real, 2: padding, 3: +inf (no right neighbour)
};

__device__ __forceinline__ bool sel_less(const SelElem &x, const int rx, const SelElem &y, const int ry)
{
    if (x.kind != y.kind) return x.kind < y.kind;
    if (x.key != y.key) return x.key < y.key;
    if (x.val != y.val) return x.val < y.val;
    return rx < ry;
}

template <class E>
__device__ __forceinline__ SelElem sel_load(const void *kin, const uint32_t *vin, const unsigned long long start,
                                            const unsigned long long len, const unsigned long long pos)
{
    SelElem e;
    e.key = 0;
    e.val = 0;
    if (pos >= len) { e.kind = 2; return e; }
    e.kind = 1;
    if constexpr (E::KEY_WORDS == 1) e.key = __ldg(static_cast<const uint32_t *>(kin) + start + pos);
    else e.key = __ldg(static_cast<const unsigned long long *>(kin) + start + pos);
    if constexpr (E::HAS_VAL) e.val = __ldg(vin + start + pos);
    return e;
}

constexpr int PART4_THREADS = 128;
template <class E>
__global__ void __launch_bounds__(PART4_THREADS, 1)
partition4_kernel(const void *__restrict__ kin, const uint32_t *__restrict__ vin, uint4 *__restrict__ splits,
                  const unsigned long long n, const unsigned long long L, const unsigned long long num_bounds,
                  const unsigned long long share)
{
    pdl_entry();
    const unsigned long long s = static_cast<unsigned long long>(blockIdx.x) * PART4_THREADS + threadIdx.x;
    if (s >= num_bounds) return;
    const unsigned long long out0 = s * share;
    const unsigned long long g0 = out0 / (4 * L) * (4 * L);
    if (g0 >= n) { splits[s] = make_uint4(0, 0, 0, 0); return; }
    unsigned long long start[4], len[4];
    unsigned long long total = 0;
#pragma unroll
    for (int r = 0; r < 4; ++r) {
        start[r] = g0 + r * L;
        len[r] = start[r] < n ? min(L, n - start[r]) : 0ull;
        total += len[r];
    }
    const unsigned long long d = min(out0 - g0, total);
    unsigned long long H = 1;
    while (H < L) H <<= 1;

    unsigned long long c[4] = {0, 0, 0, 0};
    SelElem lf[4], rt[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) { lf[r].key = 0; lf[r].val = 0; lf[r].kind = 0; }

    for (unsigned long long h = H;; h >>= 1) {
        const unsigned long long nb = H / h;       // blocks per (padded) run
        const unsigned long long D = d / h;
        // right boundary samples of every run (the left ones carry over: position c h - 1 is unchanged)
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            if (c[r] < nb) rt[r] = sel_load<E>(kin, vin, start[r], len[r], (c[r] + 1) * h - 1);
            else { rt[r].key = 0; rt[r].val = 0; rt[r].kind = 3; }
        }
        while (true) {
            const unsigned long long sum = c[0] + c[1] + c[2] + c[3];
            int a = 0, b = 0;                        // a: run with the largest left, b: smallest right
            SelElem la = lf[0], rb = rt[0];
#pragma unroll
            for (int q = 1; q < 4; ++q) {
                if (sel_less(la, a, lf[q], q)) { la = lf[q]; a = q; }
                if (sel_less(rt[q], q, rb, b)) { rb = rt[q]; b = q; }
            }
            bool retreat = false, advance = false;
            if (sum < D) advance = true;
            else if (sum > D) retreat = true;
            else if (a != b && sel_less(rb, b, la, a)) { advance = true; retreat = true; }
            if (!advance && !retreat) break;
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                if (retreat && q == a) {             // the block left of the split of run a moves right
                    c[q] -= 1;
                    rt[q] = lf[q];
                    if (c[q] > 0) lf[q] = sel_load<E>(kin, vin, start[q], len[q], c[q] * h - 1);
                    else { lf[q].key = 0; lf[q].val = 0; lf[q].kind = 0; }
                }
                if (advance && q == b) {             // the block right of the split of run b moves left
                    c[q] += 1;
                    lf[q] = rt[q];
                    if (c[q] < nb) rt[q] = sel_load<E>(kin, vin, start[q], len[q], (c[q] + 1) * h - 1);
                    else { rt[q].key = 0; rt[q].val = 0; rt[q].kind = 3; }
                }
            }
        }
        if (h == 1) break;
#pragma unroll
        for (int r = 0; r < 4; ++r) c[r] <<= 1;
    }
    splits[s] = make_uint4(static_cast<uint32_t>(c[0]), static_cast<uint32_t>(c[1]), static_cast<uint32_t>(c[2]),
                           static_cast<uint32_t>(c[3]));
}

// ------------------------------------------------------------------ rows -> linear shared memory / global
//
// pipe::store_rows_seq with the destination either global memory (streaming vector stores) or a
// linear region of shared memory (level-1 output): lane l stores 16 bytes at element offset
// base + 4 (32 m + l) -- a quarter-warp covers 32 consecutive words, conflict-free for a 16-byte
// aligned base.
template <bool SMEM>
__device__ __forceinline__ void st128(uint4 *p, const uint4 t)
{
    if constexpr (SMEM) *p = t;
    else stg128(p, t);
}
template <bool SMEM>
__device__ __forceinline__ void st64(uint2 *p, const uint2 t)
{
    if constexpr (SMEM) *p = t;
    else stg64(p, t);
}
template <bool SMEM>
__device__ __forceinline__ void st32(uint32_t *p, const uint32_t t)
{
    if constexpr (SMEM) *p = t;
    else stg32(p, t);
}

template <class E, bool SMEM>
__device__ __forceinline__ void store_rows_to(uint32_t *scratch, void *keys, uint32_t *vals, const size_t base,
                                              const int cnt, const bool full, const int lane, uint32_t (&v)[E::NP][32])
{
    if (full) {
        if constexpr (E::KEY_WORDS == 1) {
            row_store(scratch, v[0], lane);
            __syncwarp();
            uint4 *pk = reinterpret_cast<uint4 *>(static_cast<uint32_t *>(keys) + base);
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int w = chunk_word(4 * m + (lane >> 3), lane & 7);
                st128<SMEM>(pk + 32 * m + lane, *reinterpret_cast<const uint4 *>(scratch + w));
            }
        } else {
            row_store(scratch, v[0], lane);
            __syncwarp();
#pragma unroll
            for (int m = 0; m < 16; ++m) {     // this lane's high words of keys 64 m + 2 lane, + 1
                const int w = elem_word(2 * m + (lane >> 4), 2 * (lane & 15));
                const uint2 h = *reinterpret_cast<const uint2 *>(scratch + w);
                v[0][2 * m] = h.x; v[0][2 * m + 1] = h.y;
            }
            __syncwarp();
            row_store(scratch, v[1], lane);
            __syncwarp();
            uint4 *pk = reinterpret_cast<uint4 *>(static_cast<uint64_t *>(keys) + base);
#pragma unroll
            for (int m = 0; m < 16; ++m) {
                const int w = elem_word(2 * m + (lane >> 4), 2 * (lane & 15));
                const uint2 l = *reinterpret_cast<const uint2 *>(scratch + w);
                st128<SMEM>(pk + 32 * m + lane, make_uint4(l.x, v[0][2 * m], l.y, v[0][2 * m + 1]));
            }
        }
        if constexpr (E::HAS_VAL) {
            __syncwarp();
            row_store(scratch, v[E::KEY_WORDS], lane);
            __syncwarp();
            uint4 *pv = reinterpret_cast<uint4 *>(vals + base);
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const int w = chunk_word(4 * m + (lane >> 3), lane & 7);
                st128<SMEM>(pv + 32 * m + lane, *reinterpret_cast<const uint4 *>(scratch + w));
            }
        }
    } else {
        // partial page: back to the column layout (position 32 k + lane), guarded stores
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
                if constexpr (E::KEY_WORDS == 1) st32<SMEM>(static_cast<uint32_t *>(keys) + g, v[0][k]);
                else st64<SMEM>(reinterpret_cast<uint2 *>(keys) + g, make_uint2(v[1][k], v[0][k]));
                if constexpr (E::HAS_VAL) st32<SMEM>(vals + g, v[E::KEY_WORDS][k]);
            }
        }
    }
    __syncwarp();   // the scratch plane is reused by the warp's next page
}

// ------------------------------------------------------------------ one page merge out of a stage buffer
//
// Page j (outputs [1024 j, 1024 j + 1024) of the merge of the pair `m`) into row registers:
// in-smem co-rank of both page boundaries, bitonic column layout straight from the stage buffer.
// Returns the number of outputs of the page; the caller runs the two mergers after it released or
// synchronised on the stage buffer.
template <class E>
__device__ __forceinline__ int load_page(const unsigned char *kreg, const unsigned char *vreg, const ShareMeta &m, const int j,
                                         const int lane, uint32_t (&v)[E::NP][32])
{
    constexpr int KB = E::KEY_BYTES;
    const int d0 = j * TILE;
    const int d1 = min(d0 + TILE, m.a_len + m.b_len);
    const int i0 = pipe::corank_smem<E>(kreg, vreg, m, d0, lane);
    const int i1 = pipe::corank_smem<E>(kreg, vreg, m, d1, lane, i0, i0 + (d1 - d0));
    const int a = i1 - i0;
    const int b = (d1 - d0) - a;
    const uint32_t kA = pipe::smem_u32(kreg) + static_cast<uint32_t>(m.ka_off + i0 + lane) * KB;
    const uint32_t kB = pipe::smem_u32(kreg) + static_cast<uint32_t>(m.kb_off + (d0 - i0) + (TILE - 1) - lane) * KB;
    const uint32_t vA = pipe::smem_u32(vreg) + static_cast<uint32_t>(m.va_off + i0 + lane) * 4u;
    const uint32_t vB = pipe::smem_u32(vreg) + static_cast<uint32_t>(m.vb_off + (d0 - i0) + (TILE - 1) - lane) * 4u;
    pipe::load_columns<E>(v, a - lane, lane - (TILE - b), kA, kB, vA, vB, std::make_integer_sequence<int, 32>{});
    return d1 - d0;
}

// column merger, skewed transpose through the warp's scratch plane, row merger (SHEARSORT-MERGE)
template <class E>
__device__ __forceinline__ void merge_page(uint32_t *scratch, const int lane, uint32_t (&v)[E::NP][32])
{
    line_bitonic_merge<E::NP>(v);
#pragma unroll
    for (int p = 0; p < E::NP; ++p) {
        if (p) __syncwarp();
        col_store<false>(scratch, v[p], lane);
        __syncwarp();
        row_load(scratch, v[p], lane);
    }
    line_bitonic_merge<E::NP>(v);
}

__device__ __forceinline__ void consumer_barrier()
{
    asm volatile("bar.sync 1, %0;" ::"n"(NWC * 32) : "memory");
}

// ------------------------------------------------------------------ the two-round pass

template <class E>
__global__ void __launch_bounds__(THREADS, Cfg4<E>::ctas_per_sm)
merge4_pipe_kernel(const void *__restrict__ kin_, const uint32_t *__restrict__ vin, void *__restrict__ kout,
                   uint32_t *__restrict__ vout, const uint4 *__restrict__ splits, const unsigned long long n,
                   const unsigned long long L, const unsigned long long num_shares)
{
    pdl_entry();
    using C = Cfg4<E>;
    constexpr int KB = C::KB;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint32_t *scratch_all = reinterpret_cast<uint32_t *>(smem_raw + C::scratch_off);
    Meta4 *meta = reinterpret_cast<Meta4 *>(smem_raw + C::meta_off);
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw + C::bar_off);
    uint64_t *empty = full + NSTAGE;
    const unsigned char *kin = static_cast<const unsigned char *>(kin_);

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const bool small_round = (4 * L <= static_cast<unsigned long long>(SH));

    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) {
            pipe::mbar_init(&full[s], 1);
            pipe::mbar_init(&empty[s], NWC);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NWC) {
        // ============================== producer warp
        unsigned int it = 0;
        for (unsigned long long s = blockIdx.x; s < num_shares; s += gridDim.x, ++it) {
            const int st = it % NSTAGE;
            const uint32_t ph = (it / NSTAGE) & 1u;
            unsigned char *kreg = smem_raw + st * C::stage_bytes;
            unsigned char *vreg = kreg + C::key_region;
            pipe::mbar_wait(&empty[st], ph ^ 1u);
            const unsigned long long out0 = s * SH;
            const int cnt = static_cast<int>(min(static_cast<unsigned long long>(SH), n - out0));
            if (small_round) {
                // the share holds whole groups: pair q = runs 2q, 2q+1 of the share, in place
                const int l = static_cast<int>(L);
                if (lane == 0) {
                    Meta4 &M = meta[st];
                    M.cnt = cnt;
                    M.npairs = (cnt + 2 * l - 1) / (2 * l);
                    for (int q = 0; q < 4; ++q) {
                        const int pb = q * 2 * l;
                        ShareMeta m;
                        m.cnt = 0; m.pad = 0;
                        m.a_len = max(0, min(l, cnt - pb));
                        m.b_len = max(0, min(l, cnt - pb - l));
                        m.ka_off = pb; m.kb_off = pb + l; m.va_off = pb; m.vb_off = pb + l;
                        M.pair[q] = m;
                        M.w[q] = pb;
                    }
                }
                if ((cnt & 3) == 0) {
                    if (lane == 0) {
                        pipe::mbar_arrive_expect_tx(&full[st], static_cast<uint32_t>(cnt) * (KB + (E::HAS_VAL ? 4u : 0u)));
                        pipe::bulk_g2s(kreg, kin + out0 * KB, static_cast<uint32_t>(cnt) * KB, &full[st]);
                        if constexpr (E::HAS_VAL) pipe::bulk_g2s(vreg, vin + out0, static_cast<uint32_t>(cnt) * 4u, &full[st]);
                    }
                } else {   // ragged end of the array: plain cooperative copy
                    for (int i = lane; i < cnt * (KB / 4); i += 32)
                        reinterpret_cast<uint32_t *>(kreg)[i] = reinterpret_cast<const uint32_t *>(kin + out0 * KB)[i];
                    if constexpr (E::HAS_VAL)
                        for (int i = lane; i < cnt; i += 32) reinterpret_cast<uint32_t *>(vreg)[i] = vin[out0 + i];
                    __syncwarp();
                    if (lane == 0) pipe::mbar_arrive(&full[st]);
                }
            } else {
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
                    Meta4 &M = meta[st];
                    M.cnt = cnt;
                    M.npairs = 2;
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        ShareMeta m;
                        m.cnt = 0; m.pad = 0;
                        m.a_len = len[2 * q]; m.b_len = len[2 * q + 1];
                        m.ka_off = koff[2 * q]; m.kb_off = koff[2 * q + 1];
                        m.va_off = voff[2 * q]; m.vb_off = voff[2 * q + 1];
                        M.pair[q] = m;
                    }
                    M.w[0] = 0;
                    M.w[1] = (len[0] + len[1] + 3) & ~3;
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
                } else {
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
        }
        return;
    }

    // ============================== consumer warps
    uint32_t *scratch = scratch_all + warp * TILE;
    unsigned int it = 0;
    for (unsigned long long s = blockIdx.x; s < num_shares; s += gridDim.x, ++it) {
        const int st = it % NSTAGE;
        const uint32_t ph = (it / NSTAGE) & 1u;
        unsigned char *kreg = smem_raw + st * C::stage_bytes;
        unsigned char *vreg = kreg + C::key_region;
        pipe::mbar_wait(&full[st], ph);
        const Meta4 &M = meta[st];
        const int npairs = M.npairs;
        int len1[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) len1[q] = (q < npairs) ? M.pair[q].a_len + M.pair[q].b_len : 0;

        uint32_t v[E::NP][32];

        // ---------------- level 1: X = merge(A, B), Y = merge(C, D), page `warp` of the pages of all pairs
        int q1 = -1, j1 = warp;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int pages = (len1[q] + TILE - 1) / TILE;
            if (q1 < 0) {
                if (j1 < pages) q1 = q;
                else j1 -= pages;
            }
        }
        int cnt1 = 0, w1 = 0;
        if (q1 >= 0) {
            const ShareMeta m = M.pair[q1];
            cnt1 = load_page<E>(kreg, vreg, m, j1, lane, v);
            w1 = M.w[q1] + j1 * TILE;
        }
        const int w0 = M.w[0], wq1 = M.w[1], wq2 = M.w[2], wq3 = M.w[3];
        if (q1 >= 0) merge_page<E>(scratch, lane, v);
        consumer_barrier();          // every level-1 read of the stage buffer is done
        if (q1 >= 0) {
            store_rows_to<E, true>(scratch, kreg, reinterpret_cast<uint32_t *>(vreg), static_cast<size_t>(w1), cnt1,
                                   cnt1 == TILE, lane, v);
        }
        // the next writer of this stage buffer is the TMA engine (async proxy)
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        consumer_barrier();          // X and Y are complete

        // ---------------- level 2: Z = merge(X, Y), page `warp` of the share
        int p2 = -1, j2 = warp, out_rel = 0;
#pragma unroll
        for (int p = 0; p < 2; ++p) {
            const int l2 = len1[2 * p] + len1[2 * p + 1];
            const int pages = (l2 + TILE - 1) / TILE;
            if (p2 < 0) {
                if (j2 < pages) p2 = p;
                else { j2 -= pages; out_rel += l2; }
            }
        }
        int cnt2 = 0;
        if (p2 >= 0) {
            ShareMeta m;
            m.cnt = 0; m.pad = 0;
            m.a_len = p2 ? len1[2] : len1[0];
            m.b_len = p2 ? len1[3] : len1[1];
            m.ka_off = p2 ? wq2 : w0;
            m.kb_off = p2 ? wq3 : wq1;
            m.va_off = m.ka_off;
            m.vb_off = m.kb_off;
            cnt2 = load_page<E>(kreg, vreg, m, j2, lane, v);
        }
        __syncwarp();
        if (lane == 0) pipe::mbar_arrive(&empty[st]);   // stage buffer may be refilled
        if (p2 >= 0) {
            merge_page<E>(scratch, lane, v);
            store_rows_to<E, false>(scratch, kout, vout, s * SH + out_rel + j2 * TILE, cnt2, cnt2 == TILE, lane, v);
        }
    }
}

}  // namespace pipe4
}  // namespace bcf
