/*
 * bcf.h -- C ABI of the B200-native bank-conflict-free sorting library (libbcf.so).
 *
 * The library implements the data-parallel hot path of
 *   Sitchinava & Weichert, "Bank Conflict Free Comparison-based Sorting On GPUs",
 *   arXiv 1306.5076 (cited below as PAPER.md:L<line>, section / algorithm),
 * as hand-written sm_100a CUDA kernels:  the ShearSort of w x w = 32 x 32 tiles in shared
 * memory (section 3.1, Alg. 1/2) and BCFMergesort's merging of sorted runs larger
 * than shared memory (section 3, 3.2, Alg. 6).
 *
 * Conventions for every entry point
 *  - Elements are keys alone, or (key, value) pairs in two separate arrays (SoA).
 *    Supported element types: (U32, NONE), (U32, U32), (U64, NONE), (U64, U32).
 *  - ORDER: ascending by (key, value) compared lexicographically as unsigned integers; for
 *    keys-only, by key.  That order is total on element bit patterns, so exactly one output is
 *    correct for every input (reading A11).
 *  - POINTERS named d_* are DEVICE pointers, h_* are HOST pointers.  All device arrays must be
 *    16-byte aligned (BCF_ERR_MISALIGNED otherwise).  d_vals must be NULL iff the value type is
 *    BCF_VAL_NONE.
 *  - OWNERSHIP: the caller owns every byte, including the workspace; the library never
 *    allocates or frees device memory.  (One call, bcf_merge_round_static, takes no workspace: its
 *    scratch is a fixed 256 KiB array inside the library's device image; see there.)
 *  - ASYNCHRONY: device entry points only enqueue work on `stream` and return; they never
 *    synchronise.  (bcf_sort_host is the exception, see there.)
 *  - ERRORS: status codes only; no exceptions, no exit().  n == 0 is BCF_OK and a no-op.
 *    Every entry point that touches the device first clears a pending (non-sticky) CUDA error of the
 *    calling thread, checks every launch it makes, stops at the first failure and returns
 *    BCF_ERR_CUDA once; the CUDA error code of that failure is kept per thread (bcf_last_cuda_error)
 *    and is not left pending.  After a failure the contents of the output and workspace are unspecified.
 *  - STATE: the library keeps no settings.  Everything that selects an algorithm is passed per call in a
 *    bcf_options (below); two threads, or two calls, with different options do not interact.  The only
 *    process-wide state is the measurement hooks at the end of this file (timing: not thread-safe, off by
 *    default, and untouched by calls made while it is off; launch counts: atomic counters, safe from any
 *    number of threads), per-device caches of kernel attributes (thread-safe, keyed by device id), and a per-device
 *    pool of the side stream + events bcf_sort_host uses (thread-safe; a call borrows one set, concurrent calls get
 *    their own; kept until the process exits).
 *  - DEVICE: compute capability 10.x (B200, sm_100a) is required; anything else returns
 *    BCF_ERR_UNSUPPORTED_DEVICE.  There is no fallback path of any kind.
 *  - LIMIT: n < 2^32 elements.  Largest inputs tested on a B200 (tests/test_gpu_fullsize.py): 2^31 + 4099 uint32
 *    keys and 2^30 + 77 (uint64, uint32) pairs through bcf_sort.
 */
#ifndef BCF_H_
#define BCF_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BCF_W 32            /* warp size = number of 4-byte shared memory banks */
#define BCF_TILE 1024       /* M = w*w elements per tile / page           */
#define BCF_SHARE 8192      /* outputs per share of the four-run pass (bcf_merge_partition4): 8 pages.
                               The two-run merge kernel picks its own share
                               size per element type (16 / 4 / 8 pages for 4- / 8- / 12-byte elements).       */

/* A CUDA stream handle; identical to cudaStream_t / CUstream. */
typedef struct CUstream_st *bcf_stream_t;

typedef enum {
    BCF_OK = 0,
    BCF_ERR_INVALID_ARG = 1,         /* NULL pointer, bad enum, run_len == 0, in/out aliasing, n >= 2^32 */
    BCF_ERR_MISALIGNED = 2,          /* a device pointer is not 16-byte aligned                         */
    BCF_ERR_WORKSPACE_TOO_SMALL = 3, /* workspace_bytes < bcf_workspace_bytes(...)                      */
    BCF_ERR_UNSUPPORTED_DEVICE = 4,  /* current device is not compute capability 10.x                   */
    BCF_ERR_CUDA = 5,                /* a CUDA runtime call or kernel launch failed                     */
    BCF_ERR_TOO_LARGE = 6            /* bcf_merge_round_static only: the round needs more split points
                                        than the library's built-in scratch array holds                 */
} bcf_status;

typedef enum { BCF_KEY_U32 = 0, BCF_KEY_U64 = 1 } bcf_key_t;
typedef enum { BCF_VAL_NONE = 0, BCF_VAL_U32 = 1 } bcf_val_t;

typedef enum {
    BCF_OP_SORT_TILES = 0,
    BCF_OP_MERGE_RUNS = 1,
    BCF_OP_SORT = 2,
    BCF_OP_SORT_HOST = 3,
    BCF_OP_MERGE_PAGEWISE = 4
} bcf_op_t;

/* Human-readable name of a status code (static storage). */
const char *bcf_status_string(bcf_status s);

/* Library version, e.g. "bcf 0.1 (sm_100a)". */
const char *bcf_version(void);

/*
 * Bytes of device workspace the given operation needs for n elements.
 *   SORT_TILES      0
 *   MERGE_RUNS      one ping-pong copy of keys (+values) and the split-point array of the
 *                   first pass (run_len is the caller's run length)
 *   SORT            same with run_len = BCF_TILE (run_len argument ignored)
 *   SORT_HOST       the data itself (keys + values) plus the SORT workspace
 *   MERGE_PAGEWISE  same as MERGE_RUNS without the split-point array
 * Returns 0 for an invalid op / type.
 */
size_t bcf_workspace_bytes(int op, size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt);

/*
 * bcf_sort_tiles -- batched base case: ShearSort of independent 32 x 32 tiles.
 * PAPER.md section 3.1 (L105-111), Algorithm 1 (L308-335) with the implicit transposition of
 * section 3.3 / Algorithm 2 (L153, L337-363):  ceil(log2 w) = 5 phases of {row sort in
 * alternating direction, column sort ascending} and one clean-up row sort, every line sorted by
 * one thread with Batcher's odd-even mergesort in registers, every shared-memory access of a
 * warp touching 32 distinct banks.
 *
 *   d_keys, d_vals : in place; tile t is elements [1024 t, 1024 t + 1024), row-major 32 x 32.
 *   num_tiles      : number of whole tiles.
 * On return (after the stream drains) every tile is in ascending row-major order.
 */
bcf_status bcf_sort_tiles(void *d_keys, void *d_vals, size_t num_tiles,
                          bcf_key_t kt, bcf_val_t vt, bcf_stream_t stream);

/*
 * bcf_sort_tiles_mergesort -- same contract and same (unique) result as bcf_sort_tiles with a
 * cheaper network inside the same conflict-free framework: every row sorted once (Batcher), then
 * for T = 1..5 every block of 2^T rows is formed from its two sorted halves by ONE round
 * {column pass, row pass} of the paper's page merge (SHEARSORT-MERGE, with the
 * second half read reversed, reading A8), so all later line operations are bitonic mergers:
 * 831 comparators per thread instead of ShearSort's 2101, the same 10 sweeps through shared memory.
 */
bcf_status bcf_sort_tiles_mergesort(void *d_keys, void *d_vals, size_t num_tiles,
                                    bcf_key_t kt, bcf_val_t vt, bcf_stream_t stream);

/*
 * bcf_sort_long_tiles -- long tiles M = h * w^2 (section 3.1, Appendix E): every
 * group of h consecutive tiles (h = 2, 4 or 8; h divides w) is sorted as ONE sequence of 1024 h
 * elements by the h warps of one CTA without leaving the chip: each warp sorts its tile, then
 * log2 h rounds merge the sorted tiles pairwise with the data-oblivious form of the paper's page
 * merge (flip stage + half-cleaners between tiles through conflict-free shared memory, then the
 * column pass and row pass inside each tile).  The paper's own nested Segmented ShearSort
 * (Alg. 3-5) is not used.  In place; long tile t = elements [1024 h t, 1024 h (t+1)).
 */
bcf_status bcf_sort_long_tiles(void *d_keys, void *d_vals, size_t num_long_tiles, int h,
                               bcf_key_t kt, bcf_val_t vt, bcf_stream_t stream);

/*
 * bcf_options -- per-call algorithm selection.  Pass NULL for the defaults.  No environment variable and no
 * process-wide setter exists; the result of every entry point is the same for every option value (the
 * sorted output is unique), only the kernels and the number of passes over global memory differ.
 *   struct_size     sizeof(bcf_options) of the caller (bcf_options_init fills it); lets the struct grow.
 *   base_case       base case of bcf_sort: BCF_BASE_SHEARSORT = the paper's tile ShearSort (bcf_sort_tiles),
 *                   BCF_BASE_TILE_MERGESORT = bcf_sort_tiles_mergesort, BCF_BASE_LONG_TILES =
 *                   bcf_sort_long_tiles with h = 8 (runs of 8192, three merge rounds fewer), BCF_BASE_AUTO =
 *                   the fastest measured on B200 per element type.
 *   rounds_per_pass merge rounds per read + write of the data: 1 (Lemma 2), 2 (four-run kernel
 *                   where it applies) or 0 = the library's choice.
 *   merge_impl      BCF_MERGE_IMPL_AUTO, or BCF_MERGE_IMPL_GENERIC = one warp per page with loads from global
 *                   memory (merge_kernel) even where the TMA-fed pipeline applies; BCF_MERGE_IMPL_BARRIER4 =
 *                   four-run passes (rounds_per_pass = 2) always with the kernel that separates its two levels
 *                   by CTA barriers (bcf_merge4.cuh) instead of the task-stream kernel (bcf_merge4s.cuh);
 *                   BCF_MERGE_IMPL_PARTITION_LAUNCH = every round's split points from a partition launch, even
 *                   where the merge kernel's CTAs would find their own (rounds with at most 8 shares per CTA).
 *   partition_warp_search_max
 *                   largest number of share boundaries of a round searched with 32 lanes per boundary
 *                   (latency-bound case); above it one thread per boundary.  < 0 = default (4096).
 *   launch_mode     BCF_LAUNCH_PLAIN = ordinary stream-ordered launches; BCF_LAUNCH_PDL = programmatic
 *                   dependent launches (a kernel's CTAs are scheduled while its predecessor drains and wait
 *                   on griddepcontrol before touching its output); BCF_LAUNCH_AUTO = the library's choice
 *                   (dependent launches: measured faster at every size, 27 % at 2^20 keys, 1 % at 2^28).
 */
typedef enum { BCF_BASE_SHEARSORT = 0, BCF_BASE_TILE_MERGESORT = 1, BCF_BASE_LONG_TILES = 2, BCF_BASE_AUTO = 3 } bcf_base_case;
typedef enum { BCF_MERGE_IMPL_AUTO = 0, BCF_MERGE_IMPL_GENERIC = 1, BCF_MERGE_IMPL_BARRIER4 = 2, BCF_MERGE_IMPL_PARTITION_LAUNCH = 3 } bcf_merge_impl;
typedef enum { BCF_LAUNCH_AUTO = 0, BCF_LAUNCH_PLAIN = 1, BCF_LAUNCH_PDL = 2 } bcf_launch_mode;
typedef struct bcf_options {
    uint32_t struct_size;
    int32_t base_case;
    int32_t rounds_per_pass;
    int32_t merge_impl;
    int32_t partition_warp_search_max;
    int32_t launch_mode;
} bcf_options;
/* Fill *opt with the defaults (AUTO everywhere).  Returns BCF_ERR_INVALID_ARG for NULL. */
bcf_status bcf_options_init(bcf_options *opt);
/* CUDA error code (cudaError_t as int) of the calling thread's most recent BCF_ERR_CUDA; 0 if none. */
int bcf_last_cuda_error(void);

/*
 * bcf_merge_partition -- split-point search of ONE merge pass (hot-path row a5).
 * Not in the paper: it replaces the sampled bucket distribution of PAPER.md section 3.2
 * (L131-143, Alg. 7), which the paper needs because its page-wise merge is sequential per pair
 * (L121); north_star asks for "merge partitioning (split-point search so each CTA gets an equal
 * share of output)".  Runs are [i*run_len, min(n,(i+1)*run_len)); runs 2p and 2p+1 form pair p
 * (A, B).  Each pair's output is cut into shares of BCF_TILE elements; the pass has
 *      num_shares = ceil(n / (2 run_len)) * ceil(2 run_len / BCF_TILE)
 * share slots, slot j belonging to pair j / ceil(2 run_len / BCF_TILE).
 *   d_splits[j] (uint32, num_shares entries, device) receives the co-rank of the share's first
 *   output diagonal d: the number of elements of A among the first d outputs of the stable
 *   (A-first on ties) merge of A and B, i.e. the smallest i in [max(0,d-|B|), min(d,|A|)] with
 *   NOT (A[i] <= B[d-i-1]).  Slots past the end of a short last pair receive |A|.
 */
bcf_status bcf_merge_partition(const void *d_keys_in, const void *d_vals_in, size_t n, size_t run_len,
                               bcf_key_t kt, bcf_val_t vt, uint32_t *d_splits, size_t num_shares,
                               bcf_stream_t stream);

/*
 * bcf_merge_partition4 -- split-point search of one FOUR-RUN pass (two merge rounds of PAPER.md
 * section 3, done on chip per read + write of the data).
 * Runs 4g .. 4g+3 (run r = elements [r*run_len, min(n, (r+1)*run_len))) form group g; the pass
 * output is cut into shares of BCF_SHARE elements.  For every share boundary
 * s = 0 .. ceil(n / BCF_SHARE) at output position s * BCF_SHARE, inside the group that position
 * falls into (4 run_len must be a multiple of BCF_SHARE):
 *   d_splits[4 s + r] (uint32, device, 16-byte aligned) = number of elements of run r of the group
 *   among the first d = s * BCF_SHARE - group_start outputs of the stable four-way merge (ties:
 *   lower run first, then lower position), found by multi-sequence selection.
 * A boundary at or past n receives the split of d clipped to the group's length (0 0 0 0 for a
 * group that starts at or past n).  num_bounds must be ceil(n / BCF_SHARE) + 1.
 */
bcf_status bcf_merge_partition4(const void *d_keys_in, const void *d_vals_in, size_t n, size_t run_len,
                                bcf_key_t kt, bcf_val_t vt, uint32_t *d_splits, size_t num_bounds,
                                bcf_stream_t stream);

/*
 * bcf_find_buckets -- FIND-BUCKETS, the paper's deterministic bucket distribution (section 3.2
 * "Distribution" L131-137, Lemma 1, Algorithm 7), with the pivot buckets of
 * section 3.3 (L155, BCFMergesortPB) as an option.  Not on the hot path (bcf_merge_runs partitions
 * by exact co-ranking); provided as the paper's own partitioner.  Keys only.
 *   d_keys_in  : n keys, s = ceil(n / run_len) sorted runs of run_len (the last may be shorter).
 *   t          : samples per run; sample i of run r is its element floor(i * len_r / t).
 *   P          : buckets.  The s*t samples are sorted; pivot j = sorted sample floor((j+1) s t / P),
 *                j = 0..P-2.  Bucket j holds the keys with pivot[j-1] < key <= pivot[j].
 *   pivot_buckets != 0 : keys equal to pivot j get a bucket of their own right after bucket j
 *                (which then holds pivot[j-1] < key < pivot[j]): nb = 2P-1 buckets instead of nb = P;
 *                the second copy of a repeated pivot owns nothing.
 *   d_keys_out : n keys: the runs' pieces regrouped by bucket, inside a bucket by run, every piece
 *                in its original (sorted) order.  Buckets are in ascending key order.
 *   d_pivots   : P-1 keys.
 *   d_piece_offsets : nb*s + 1 uint32: entry b*s + r = position in d_keys_out of the piece of run r
 *                in bucket b; the last entry is n.  (Bucket b starts at entry b*s.)
 *   d_workspace: >= bcf_find_buckets_workspace_bytes(...) bytes.
 * Lemma 1: with all keys distinct every bucket has at most s*ceil(len/t) + ceil(s t / P)*ceil(len/t)
 * keys, len = run_len.  Requires t >= 1, P >= 2, s*t >= P, s, t, P <= 65536.
 */
size_t bcf_find_buckets_workspace_bytes(size_t n, size_t run_len, int t, int P, int pivot_buckets, bcf_key_t kt);
bcf_status bcf_find_buckets(const void *d_keys_in, size_t n, size_t run_len, int t, int P, int pivot_buckets,
                            bcf_key_t kt, void *d_keys_out, void *d_pivots, uint32_t *d_piece_offsets,
                            void *d_workspace, size_t workspace_bytes, bcf_stream_t stream);

/*
 * bcf_colored_prefix_sums -- conflict-free coloured prefix sums (Appendix A; SURVEY.md
 * 8f item 4): d_out[i] = sum of d_values[j] over j <= i with d_colors[j] == d_colors[i], in uint32
 * arithmetic (sums wrap modulo 2^32).  Three phases as in the paper (tile sums, exclusive scan of the
 * tile sums per colour, page-wise scan of every tile); a thread's per-colour running sums are kept in
 * shared memory.
 *   d_values  : n uint32.   d_colors : n bytes, each < num_colors.   num_colors : 1..16.
 *   layout    : BCF_SCAN_BANK_PER_THREAD -- word 32 c + lane, "one memory bank per thread" (L228): every
 *               warp access hits 32 distinct banks whatever the colours;
 *               BCF_SCAN_THREAD_MAJOR -- word d lane + c, the layout the paper starts from, kept to
 *               reproduce its Figure 1 (bank conflicts and run time grow with d).  Same result.
 *   d_out     : n uint32, may not overlap the inputs.
 *   d_workspace : >= bcf_colored_prefix_sums_workspace_bytes(n) bytes.
 * A colour >= num_colors is counted as colour num_colors - 1 (it never indexes outside the caller's d sums).
 */
typedef enum { BCF_SCAN_BANK_PER_THREAD = 0, BCF_SCAN_THREAD_MAJOR = 1 } bcf_scan_layout;
size_t bcf_colored_prefix_sums_workspace_bytes(size_t n);
bcf_status bcf_colored_prefix_sums(const uint32_t *d_values, const uint8_t *d_colors, size_t n, int num_colors,
                                   int layout, uint32_t *d_out, void *d_workspace, size_t workspace_bytes,
                                   bcf_stream_t stream);

/*
 * Number of passes over global memory (one read + one write of all n elements each) that
 * bcf_merge_runs(_ex) takes from runs of run_len under `opt` (NULL = defaults): a pass does two merge rounds
 * where the four-run kernel applies (rounds_per_pass = 2, run_len = 1024 * 2^k and the element type's stage
 * buffers fit one SM) and one round otherwise.  Host only.
 */
int bcf_merge_pass_count(size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt, const bcf_options *opt);

/*
 * bcf_merge_runs -- BCFMergesort's merging phase on already sorted runs.
 * PAPER.md section 3 (L103): ceil(log2(#runs)) rounds, each merging pairs of runs; the paper
 * charges one read + one write of all n elements per round (Lemma 2), this library
 * does two rounds per read + write where bcf_merge_pass_count says so.  Every pass is one
 * partition launch (above) and one merge launch in which a warp takes one page at a time: it loads its piece of A
 * and its piece of B (together BCF_TILE elements, coalesced), merges them in shared
 * memory/registers with ONE ShearSort round -- SHEARSORT-MERGE, with the
 * second piece stored reversed so that one {column pass, row pass} is sufficient (reading A8) --
 * and stores BCF_TILE outputs coalesced.  Partial shares are padded with the maximum element in
 * registers only.
 *
 *   d_keys_in/d_vals_in  : n elements, runs of run_len each already sorted (unchecked). Not modified.
 *   d_keys_out/d_vals_out: receive the single sorted sequence, whatever the number of rounds.
 *                          Must not overlap the inputs or the workspace.
 *   d_workspace          : >= bcf_workspace_bytes(BCF_OP_MERGE_RUNS, n, run_len, kt, vt) bytes.
 */
bcf_status bcf_merge_runs(const void *d_keys_in, const void *d_vals_in, void *d_keys_out, void *d_vals_out,
                          size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt,
                          void *d_workspace, size_t workspace_bytes, bcf_stream_t stream);
/* Same with per-call options (NULL = defaults = bcf_merge_runs). */
bcf_status bcf_merge_runs_ex(const void *d_keys_in, const void *d_vals_in, void *d_keys_out, void *d_vals_out,
                             size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt,
                             void *d_workspace, size_t workspace_bytes, bcf_stream_t stream, const bcf_options *opt);

/*
 * bcf_merge_round_static -- ONE merge round (section 3: adjacent runs merged in pairs) that needs
 * no workspace and allocates nothing.
 *
 * Why it exists.  bcf_merge_runs wants a workspace, and a caller normally gets one from cudaMalloc.  Not every
 * caller can: code that a host engine runs inside its execute step (an inference plugin, a framework operator)
 * is often not allowed to allocate there; a process that gave all device memory to its own pool at start-up has
 * none left to ask the driver for; a latency-bound loop cannot take the device-wide stall an allocation or free
 * may cause.  Those callers already own their input and output arrays.  What they lack is a place for the round's
 * split points, so this entry point keeps that scratch inside the library.
 *
 * The scratch and its limit.  The split points live in a fixed array of BCF_STATIC_MAX_SHARES uint32 (256 KiB)
 * that is part of libbcf.so's device image: every GPU on which the library is used holds those 256 KiB from first
 * use until the process exits, whether or not this function is ever called.  A round is accepted when
 *      bcf_merge_round_static_shares(n, run_len) = ceil(n / (2 run_len)) * ceil(2 run_len / BCF_TILE)
 * is at most BCF_STATIC_MAX_SHARES (n <= 2^26 elements when 2 run_len is a multiple of BCF_TILE); anything larger
 * returns BCF_ERR_TOO_LARGE before any work is enqueued -- use bcf_merge_runs with a workspace for those.
 *
 * What it computes.  Runs are [i run_len, min(n, (i+1) run_len)), each already sorted (unchecked); runs 2p and 2p+1
 * are merged into output positions [2p run_len, min(n, (2p+2) run_len)); an unpaired last run is copied.  The output
 * therefore consists of sorted runs of 2 run_len: for n <= 2 run_len it is the result of bcf_merge_runs, and a
 * caller with more runs repeats the call with run_len doubled, swapping its own two buffers (ceil(log2(#runs)) calls).
 * Same kernels as bcf_merge_runs with BCF_MERGE_IMPL_GENERIC (exact co-rank partition, then one warp per page
 * doing SHEARSORT-MERGE), same ordering contract, all four element types.
 *   d_keys_in / d_vals_in   : n elements, not modified.      d_keys_out / d_vals_out : n elements, no overlap with the inputs.
 *
 * Things to know.
 *  - No cudaMalloc, cudaFree or other allocating call is made, on the first call or later.  Two kernels are
 *    enqueued on `stream`; the call does not synchronise.
 *  - The FIRST call on each device does a one-off set-up with that device current: it checks the compute
 *    capability, asks the runtime for the device address of the built-in array (cudaGetSymbolAddress) and opts the
 *    merge kernels into their shared memory size.  Make that first call during start-up, before any stream capture
 *    is begun; later calls only launch.  The set-up is thread-safe.
 *  - All calls on a device share the one array, and it keeps whatever the previous call wrote.  Nothing in it has to
 *    start at zero (every entry a round reads is written by that round's partition kernel first), so there is
 *    nothing to clear.  But two calls whose kernels can run at the same time on one GPU -- different streams, or
 *    different host threads on different streams -- overwrite each other's split points and produce garbage:
 *    keep the calls of one device in one stream, or order them with events.
 *  - The measurement hooks at the end of this file do not count or time these launches.
 */
#define BCF_STATIC_MAX_SHARES 65536
size_t bcf_merge_round_static_max_shares(void);                 /* BCF_STATIC_MAX_SHARES, for callers that dlopen    */
size_t bcf_merge_round_static_shares(size_t n, size_t run_len); /* split points one round needs; 0 for invalid sizes */
bcf_status bcf_merge_round_static(const void *d_keys_in, const void *d_vals_in, void *d_keys_out, void *d_vals_out,
                                  size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt, bcf_stream_t stream);

/*
 * bcf_sort -- BCFMergesort (section 3, Appendix B): base case on
 * ceil(n / BCF_TILE) tiles (a last partial tile is padded with the maximum element on chip
 * only), then ceil(log2(ceil(n / BCF_TILE))) merge rounds in bcf_merge_pass_count(n, BCF_TILE, ..)
 * passes ping-ponging between the data and the workspace.  In place: the sorted result is in d_keys / d_vals for any n.
 *   d_workspace : >= bcf_workspace_bytes(BCF_OP_SORT, n, 0, kt, vt) bytes.
 */
bcf_status bcf_sort(void *d_keys, void *d_vals, size_t n, bcf_key_t kt, bcf_val_t vt,
                    void *d_workspace, size_t workspace_bytes, bcf_stream_t stream);
/* Same with per-call options (NULL = defaults = bcf_sort). */
bcf_status bcf_sort_ex(void *d_keys, void *d_vals, size_t n, bcf_key_t kt, bcf_val_t vt,
                       void *d_workspace, size_t workspace_bytes, bcf_stream_t stream, const bcf_options *opt);

/*
 * bcf_sort_buckets -- BCFMergesort with the paper's bucket distribution, end to end; with pivot_buckets != 0
 * this is BCFMergesortPB (section 3.2, section 3.3, Appendix B).  Keys only.
 * The four phases of the paper in its order:
 *   1. base case (as bcf_sort);
 *   2. first merge phase: merge rounds (as bcf_merge_runs) while more than P runs remain -- "we suspend the
 *      merge at s = P" (L131);
 *   3. bucket distribution: bcf_find_buckets on the s <= P runs with t samples per run and P buckets
 *      (2P-1 with pivot buckets);
 *   4. final merge phase (L141-143): inside every bucket its s sorted pieces (any lengths, possibly empty)
 *      are merged pairwise in ceil(log2 s) rounds; every round is one launch in which a warp takes one page
 *      of BCF_TILE outputs of one pair of pieces, finds its split points by co-ranking and merges with
 *      SHEARSORT-MERGE; partial pages are padded with the maximum key on chip only (L141).  A pivot bucket
 *      holds copies of one key and is only copied ("already in the correct position", L155).
 * If one run remains after phase 2 the result is complete and phases 3-4 are skipped.
 *   d_keys      : n keys, sorted in place.
 *   P, t        : buckets and samples per run; 2 <= P <= 65536, 1 <= t <= 65536 (the paper: t = P = 128).
 *                 Where the s runs left by phase 2 give fewer than P samples (s t < P), t is raised to
 *                 ceil(P / s) for this call; the workspace size below already accounts for that.
 *   d_workspace : >= bcf_sort_buckets_workspace_bytes(n, t, P, pivot_buckets, kt) bytes.
 *   d_bucket_starts : NULL, or nb + 1 uint32 (device): start of every bucket in the sorted output, last = n
 *                 (nb = P or 2P-1); written only when phases 3-4 ran (n > P runs of one tile, more than one run).
 */
size_t bcf_sort_buckets_workspace_bytes(size_t n, int t, int P, int pivot_buckets, bcf_key_t kt);
bcf_status bcf_sort_buckets(void *d_keys, size_t n, bcf_key_t kt, int t, int P, int pivot_buckets,
                            uint32_t *d_bucket_starts, void *d_workspace, size_t workspace_bytes,
                            bcf_stream_t stream, const bcf_options *opt);

/*
 * bcf_merge_pieces -- phase 4 alone: `groups` groups of `s` adjacent sorted pieces each
 * (piece (g, r) = elements [d_piece_offsets[g s + r], d_piece_offsets[g s + r + 1]) of d_keys_in, the layout
 * bcf_find_buckets writes) are merged group by group into d_keys_out at the same positions.
 * copy_odd_groups != 0: groups of odd index are copied instead of merged (pivot buckets).
 *   d_workspace : >= bcf_merge_pieces_workspace_bytes(n, groups, s, kt) bytes; d_keys_in is not modified.
 */
size_t bcf_merge_pieces_workspace_bytes(size_t n, size_t groups, size_t s, bcf_key_t kt);
bcf_status bcf_merge_pieces(const void *d_keys_in, void *d_keys_out, size_t n, const uint32_t *d_piece_offsets,
                            size_t groups, size_t s, int copy_odd_groups, bcf_key_t kt, void *d_workspace,
                            size_t workspace_bytes, bcf_stream_t stream);

/*
 * bcf_sort_host -- bcf_sort on HOST buffers (the end-to-end path bench.py's `e2e` times).
 * Copies h_keys / h_vals (n elements, host memory, ideally pinned) to the device scratch,
 * sorts there, copies the result back into h_keys / h_vals and SYNCHRONISES `stream` before
 * returning, so the host buffers hold the sorted data on return.
 *   d_scratch : >= bcf_workspace_bytes(BCF_OP_SORT_HOST, n, 0, kt, vt) bytes of device memory.
 */
bcf_status bcf_sort_host(void *h_keys, void *h_vals, size_t n, bcf_key_t kt, bcf_val_t vt,
                         void *d_scratch, size_t scratch_bytes, bcf_stream_t stream);
bcf_status bcf_sort_host_ex(void *h_keys, void *h_vals, size_t n, bcf_key_t kt, bcf_val_t vt,
                            void *d_scratch, size_t scratch_bytes, bcf_stream_t stream, const bcf_options *opt);

/*
 * bcf_merge_runs_pagewise -- the paper's own streaming form of the merge (hot-path row a7):
 * BINARY-MERGE, Algorithm 6 (L457-490), L127, L416-420.  One warp per pair of runs
 * keeps a page of M = BCF_TILE elements on chip, refills M/2 from the stream whose last loaded
 * page ends smaller, merges with SHEARSORT-MERGE and emits the M/2 smallest; partial pages are
 * padded with the maximum element on chip only.  Sequential per pair, so it only
 * fills the GPU while there are many pairs; same arguments and result as bcf_merge_runs.
 *   d_workspace : >= bcf_workspace_bytes(BCF_OP_MERGE_PAGEWISE, n, run_len, kt, vt) bytes.
 */
bcf_status bcf_merge_runs_pagewise(const void *d_keys_in, const void *d_vals_in, void *d_keys_out,
                                   void *d_vals_out, size_t n, size_t run_len, bcf_key_t kt, bcf_val_t vt,
                                   void *d_workspace, size_t workspace_bytes, bcf_stream_t stream);

/* ------------------------------------------------------------------ debug: conflict isolation --- */

/*
 * The bank-conflict isolation experiment (csrc/bcf_tu_isolate.cu; profiles/r3_conflict_isolation.md).  DEBUG entry
 * points: nothing in the library calls them.  They run the same shared-memory instruction streams as
 * merge_pipe_kernel and tile_mergesort_kernel (uint32 keys) in three phases separated by CTA barriers --
 * global -> chip, every LDS / STS of the work item, registers -> global -- so that ncu's
 * l1tex__data_bank_conflicts_pipe_lsu_mem_shared_op_{ld,st} can be read with (exclusive = 0, several CTAs per SM)
 * and without (exclusive = 1, one CTA per SM) other global-memory traffic on the SM during the LDS / STS phase.
 *   bcf_debug_merge_round_isolated : ONE merge round of runs of run_len = 16384 * 2^k (at least one share
 *       of the production uint32 merge kernel, whose shape -- 16-page shares, 16 warps, one CTA per SM -- it copies); n a
 *       multiple of 2 run_len; out of place; d_workspace >= (n / BCF_SHARE + 1) * 4 bytes (split points, production kernel).
 *   bcf_debug_sort_tiles_isolated  : bcf_sort_tiles_mergesort of whole tiles, in place.
 * Results are those of bcf_merge_runs / bcf_sort_tiles (parity-tested).
 */
bcf_status bcf_debug_merge_round_isolated(const void *d_keys_in, void *d_keys_out, size_t n, size_t run_len, int exclusive,
                                          void *d_workspace, size_t workspace_bytes, bcf_stream_t stream);
bcf_status bcf_debug_sort_tiles_isolated(void *d_keys, size_t num_tiles, int exclusive, bcf_stream_t stream);

/* ------------------------------------------------------------------ measurement hooks ------ */

typedef enum {
    BCF_KERNEL_TILE_SORT = 0,
    BCF_KERNEL_PARTITION = 1,
    BCF_KERNEL_MERGE = 2,
    BCF_KERNEL_MERGE_PAGEWISE = 3,
    BCF_KERNEL_CLASSES = 4           /* classes with timing / launch counters                           */
} bcf_kernel_class;

/*
 * Per-kernel timing with CUDA events recorded on the launching stream (bench.py's `roofline`).
 * bcf_profile_enable(1) makes the library record one event of its own before every later launch
 * and one at the end of the API call; a launch is timed from its event to the next one, so its
 * figure includes the gap to the following launch (a fixed pool; when it is exhausted further
 * launches are not timed);
 * bcf_profile_read synchronises those events, adds up elapsed milliseconds and launch counts
 * per kernel class into ms[BCF_KERNEL_CLASSES] / launches[BCF_KERNEL_CLASSES] (host arrays), and
 * resets the pool.  bcf_profile_enable(0) switches timing off.  Launch COUNTS per class are kept
 * whether or not timing is on; bcf_launch_counts copies and clears them.
 */
bcf_status bcf_profile_enable(int on);
bcf_status bcf_profile_read(float *ms, unsigned long long *launches);
void bcf_launch_counts(unsigned long long *launches);

/* Launches bcf_profile_enable(1) could not time because its fixed pool of events was full (then
 * bcf_profile_read's sums are incomplete and say so here); reset by bcf_profile_enable. */
unsigned long long bcf_profile_dropped(void);

/*
 * Static resource usage of every kernel the library can launch, for an element type (needs a device):
 * registers per thread, static+dynamic shared memory per CTA as launched, threads per CTA,
 * resident CTAs per SM at that configuration, local-memory bytes per thread.  PAPER.md:L151 makes "the
 * data is not transferred to local memory" part of the method: tests assert 0 bytes for every kernel.
 * BCF_ERR_INVALID_ARG for a kernel that does not exist for the element type (merge4_pipe for (u64,u32),
 * merge_pieces for key-value types).
 */
typedef enum {
    BCF_KID_TILE_SORT = 0,
    BCF_KID_TILE_MERGESORT = 1,
    BCF_KID_LONG_TILE_2 = 2,
    BCF_KID_LONG_TILE_4 = 3,
    BCF_KID_LONG_TILE_8 = 4,
    BCF_KID_PARTITION = 5,
    BCF_KID_MERGE = 6,
    BCF_KID_PARTITION_SHARE_1 = 7,
    BCF_KID_PARTITION_SHARE_32 = 8,
    BCF_KID_MERGE_PIPE = 9,
    BCF_KID_PARTITION4 = 10,
    BCF_KID_MERGE4_PIPE = 11,
    BCF_KID_MERGE_PAGEWISE = 12,
    BCF_KID_MERGE_PIECES = 13,
    BCF_KID_MERGE4_STREAM = 14,
    BCF_KID_COUNT = 15
} bcf_kernel_id;
const char *bcf_kernel_name(int kernel_id);
bcf_status bcf_kernel_info(int kernel_id, bcf_key_t kt, bcf_val_t vt, int *regs_per_thread,
                           int *smem_bytes_per_cta, int *threads_per_cta, int *ctas_per_sm,
                           int *local_bytes_per_thread);

/* ------------------------------------------------------------------ layout introspection --- */

typedef enum {
    BCF_ACCESS_ROW_STORE = 0,   /* thread r writes 16-byte chunk `step` (0..7) of logical row r      */
    BCF_ACCESS_ROW_LOAD = 1,    /* thread r reads  16-byte chunk `step` (0..7) of logical row r      */
    BCF_ACCESS_COL_LOAD = 2,    /* thread c reads  word `step` (0..31) of logical column c, rows of
                                   odd index mirrored (the alternating row direction)              */
    BCF_ACCESS_COL_STORE = 3,   /* thread c writes word `step` of logical column c (same mirroring) */
    BCF_ACCESS_COL_STORE_PLAIN = 4, /* thread c writes word `step` of column c, no mirroring (merge) */
    BCF_ACCESS_OUT_LOAD128 = 5, /* lane reads the 16-byte chunk it stores to global in vector store
                                   `step` (0..7): row 4*step + lane/8, chunk lane%8               */
    BCF_ACCESS_OUT_LOAD64 = 6,  /* lane reads 8 bytes: row 2*step + lane/16, words 2*(lane%16)..+1  */
    BCF_ACCESS_OUT_LOAD32 = 7,  /* lane reads 1 word: row step, column lane                        */
    BCF_ACCESS_COL_LOAD_LEVEL = 8, /* tile mergesort, step = 32 * (T - 1) + k for level T = 1..5, register k:
                                   thread c reads position 32 k + c of P || reverse(Q) of its block of 2^T rows */
    BCF_ACCESS_LT_FLIP_ROW_LOAD = 9, /* long tiles, flip stage between two tiles: thread r reads 16-byte chunk 7 - step
                                   (step 0..7) of the PARTNER tile's row 31 - r                       */
    BCF_ACCESS_LT_FUSED_COL_LOAD = 10, /* long tiles, last cross-tile stage fused with the transpose: thread c reads the
                                   partner's element (row 31 - step, column 31 - c), step 0..31     */
    BCF_ACCESS_SLOT_LOAD32 = 11, /* merge pipeline, stage buffer (plain linear words, no skew): lane reads word
                                   off + 32 k + lane of the A piece (step = off, 0..31) or word
                                   1023 - off - lane of the reversed B piece (step = 32 + off): 32 consecutive
                                   words from ANY offset; k only adds multiples of 32                   */
    BCF_ACCESS_SLOT_LOAD64 = 12, /* same for 8-byte keys: lane reads words 2 (off + lane), +1 (step = off) or
                                   2 (1023 - off - lane), +1 (step = 32 + off)                       */
    BCF_ACCESS_PATTERNS = 13
} bcf_access_pattern;

/*
 * The shared-memory word (0..1023, bank = word % 32) that holds logical element (row, col) of a
 * 32 x 32 plane, and the words a lane touches in each access pattern the kernels use.  Pure host
 * functions (no device needed) compiled from the SAME constexpr index functions the kernels
 * use, so a host-side bank model can prove every warp access conflict-free
 * (section 2.1; section 3.3).
 *   bcf_layout_access returns the number of consecutive words (1, 2 or 4) and stores the first.
 */
int bcf_layout_word(int row, int col);
int bcf_layout_access(int pattern, int step, int lane, int *first_word);

#ifdef __cplusplus
}
#endif
#endif /* BCF_H_ */
