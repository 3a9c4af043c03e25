/*
 * bcf_oracle_impl.h -- TEST INFRASTRUCTURE ONLY (CPU oracle, not the product).
 *
 * Plain, slow, single-threaded restatement of the hot path of
 * "Bank Conflict Free Comparison-based Sorting On GPUs" (Sitchinava & Weichert,
 * arXiv 1306.5076; /root/reference/PAPER.md, cited below as PAPER.md:L<line>).
 *
 * This file is included once per key type by bcf_oracle.c with
 *     ORC_K     the key type (uint32_t or uint64_t)
 *     ORC_(x)   a name-mangling macro
 * An element is the pair (key, value) compared lexicographically, unsigned
 * (reading A11; BASELINE.json north_star "ties ... broken by (key, value)
 * lexicographic order").  Keys-only inputs carry value 0 everywhere.
 *
 * Nothing here is shared with the CUDA path: no header, table, constant or helper.
 * Line sorts are insertion sorts on purpose (the kernels use Batcher networks).
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may call into this code.
 */

typedef struct { ORC_K k; uint32_t v; } ORC_(elem);

/* a <= b in the (key, value) lexicographic order. */
static int ORC_(le)(ORC_(elem) a, ORC_(elem) b)
{
    if (a.k != b.k) return a.k < b.k;
    return a.v <= b.v;
}

/* a < b, strictly. */
static int ORC_(lt)(ORC_(elem) a, ORC_(elem) b)
{
    if (a.k != b.k) return a.k < b.k;
    return a.v < b.v;
}

/*
 * Sort one line (a row or a column) of `len` elements that lie `stride` apart,
 * ascending, or descending when `descending` != 0.  Straight insertion sort:
 * t^(n) in PAPER.md:L111 is "the time it takes to sort a row or a column of n
 * elements using a single thread"; the paper's choice of Batcher's network for it
 * is an implementation detail of the result (a full sort of the line), reading A14.
 */
static void ORC_(line_sort)(ORC_(elem) *base, size_t stride, size_t len, int descending)
{
    for (size_t i = 1; i < len; ++i) {
        ORC_(elem) x = base[i * stride];
        size_t j = i;
        while (j > 0) {
            ORC_(elem) y = base[(j - 1) * stride];
            int out_of_order = descending ? ORC_(lt)(y, x) : ORC_(lt)(x, y);
            if (!out_of_order) break;
            base[j * stride] = y;
            --j;
        }
        base[j * stride] = x;
    }
}

static int ORC_(ceil_log2)(size_t w)
{
    int l = 0;
    while (((size_t)1 << l) < w) ++l;
    return l;
}

/*
 * SHEARSORT of one w x w tile, Algorithm 1 (L308-335), section 3.1 (L109-111).
 * T is row-major: T[r*w + c] (reading A1: rows = contiguous w-element chunks alternate
 * direction, columns = stride-w lines ascend).
 *
 *   FOR i IN 1 .. log2(w):                               (L314)
 *       sort the rows in alternating order               (L315-320; ELSE restored, A3)
 *       sort the columns (ascending)                     (L323-326)
 *   clean up and remove snake-like order: sort rows      (L329-332)
 *
 * The transposes of Alg. 1 (L322, L328, L334) are pure data movement between the
 * row view and the column view of shared memory and do not change which elements
 * form a row or a column; on a CPU they are the stride argument of line_sort.
 *
 * phases < 0  -> ceil(log2 w) full phases (reading A2).  A caller may pass fewer
 *               to exercise the "one phase fewer must fail" mutation pin.
 * final_snake -> last row pass alternates (classic ShearSort of Sen et al., snake
 *               order) instead of all-ascending (the paper's L329, reading A4).
 */
static void ORC_(shearsort_tile)(ORC_(elem) *T, size_t w, int final_snake, int phases)
{
    if (phases < 0) phases = ORC_(ceil_log2)(w);
    for (int i = 1; i <= phases; ++i) {
        for (size_t r = 0; r < w; ++r)                   /* rows, alternating */
            ORC_(line_sort)(T + r * w, 1, w, (int)(r & 1));
        for (size_t c = 0; c < w; ++c)                   /* columns, ascending */
            ORC_(line_sort)(T + c, w, w, 0);
    }
    for (size_t r = 0; r < w; ++r)                       /* clean-up row pass */
        ORC_(line_sort)(T + r * w, 1, w, final_snake ? (int)(r & 1) : 0);
}

/*
 * Binary merging: "starts off by loading the smallest element from
 * each sequence.  Then it repeatedly outputs the smaller of the two items and loads
 * the next element from the sequence whose element was written out."  Ties take
 * from A (reading A12; elements that tie are bitwise identical, so this fixes the
 * co-rank, not the output).
 */
static void ORC_(merge_two)(const ORC_(elem) *A, size_t na, const ORC_(elem) *B, size_t nb,
                            ORC_(elem) *out)
{
    size_t i = 0, j = 0, o = 0;
    while (i < na && j < nb) {
        if (ORC_(le)(A[i], B[j])) out[o++] = A[i++];
        else                      out[o++] = B[j++];
    }
    while (i < na) out[o++] = A[i++];
    while (j < nb) out[o++] = B[j++];
}

/*
 * The merging phase: "proceeds in ceil(log(N/M)) rounds, in each round
 * merging pairs of sorted sequences from the previous round to create increasingly
 * larger sequences, until only a single sorted sequence remains."  Runs are
 * [i*run_len, min(n,(i+1)*run_len)); an odd last run is copied through.
 * Result ends in buf; tmp is scratch of n elements.  Returns the number of rounds.
 */
static int ORC_(merge_runs)(ORC_(elem) *buf, ORC_(elem) *tmp, size_t n, size_t run_len)
{
    int rounds = 0;
    ORC_(elem) *src = buf, *dst = tmp;
    while (run_len < n) {
        for (size_t lo = 0; lo < n; lo += 2 * run_len) {
            size_t mid = lo + run_len < n ? lo + run_len : n;
            size_t hi  = lo + 2 * run_len < n ? lo + 2 * run_len : n;
            ORC_(merge_two)(src + lo, mid - lo, src + mid, hi - mid, dst + lo);
        }
        ORC_(elem) *t = src; src = dst; dst = t;
        run_len *= 2;
        ++rounds;
    }
    if (src != buf) memcpy(buf, src, n * sizeof(ORC_(elem)));
    return rounds;
}

/*
 * BCFMergesort, section 3 (L103) and Appendix B (L236-238): base case phase
 * sorts ceil(N/M) sequences of M = w*w elements with ShearSort, then the merging
 * phase.  A last partial tile is padded with "infinity" (all-ones key and value,
 * reading A10) in a scratch tile only: "padding is introduced
 * implicitly in shared memory, but not written to the output array".
 */
static int ORC_(sort_full)(ORC_(elem) *buf, ORC_(elem) *tmp, size_t n, size_t w)
{
    size_t M = w * w;
    size_t full = n / M, rem = n % M;
    for (size_t t = 0; t < full; ++t)
        ORC_(shearsort_tile)(buf + t * M, w, 0, -1);
    if (rem) {
        ORC_(elem) *pad = (ORC_(elem) *)malloc(M * sizeof(ORC_(elem)));
        if (!pad) return -1;
        memcpy(pad, buf + full * M, rem * sizeof(ORC_(elem)));
        for (size_t i = rem; i < M; ++i) { pad[i].k = (ORC_K)~(ORC_K)0; pad[i].v = 0xFFFFFFFFu; }
        ORC_(shearsort_tile)(pad, w, 0, -1);
        memcpy(buf + full * M, pad, rem * sizeof(ORC_(elem)));
        free(pad);
    }
    return ORC_(merge_runs)(buf, tmp, n, M);
}

/*
 * Split point ("co-rank") of output diagonal d of the merge of A and B: the number of
 * elements the two-finger merge above has taken from A when it has written d outputs.
 * Not in the paper (north_star's replacement for Alg. 7, reading A12).  Written as the
 * definition: smallest i in [max(0,d-nb), min(d,na)] such that NOT(A[i] <= B[d-i-1]),
 * found by a linear scan so that it shares nothing with the kernel's binary search.
 */
static size_t ORC_(corank)(const ORC_(elem) *A, size_t na, const ORC_(elem) *B, size_t nb, size_t d)
{
    size_t lo = d > nb ? d - nb : 0;
    size_t hi = d < na ? d : na;
    size_t i = lo;
    while (i < hi && ORC_(le)(A[i], B[d - i - 1])) ++i;
    return i;
}

/*
 * SHEARSORT-MERGE(S): "modify the SHEARSORT subroutine to only
 * perform one round of ShearSort instead of log2(w)".  Reading A8: with the two sorted
 * half-pages placed contiguously one round is NOT enough (pinned by a counter-example in
 * tests); with the second page stored reversed behind the first, one {column sort; row
 * sort} round merges every split.  S holds M = w*w elements, S[0..na) ascending,
 * S[na..M) ascending on entry; this routine reverses the second part, then does the round.
 */
static void ORC_(shearsort_merge)(ORC_(elem) *S, size_t w, size_t na)
{
    size_t M = w * w;
    for (size_t i = na, j = M; i + 1 < j; ++i) {         /* store B reversed after A */
        --j;
        ORC_(elem) t = S[i]; S[i] = S[j]; S[j] = t;
    }
    for (size_t c = 0; c < w; ++c) ORC_(line_sort)(S + c, w, w, 0);      /* columns */
    for (size_t r = 0; r < w; ++r) ORC_(line_sort)(S + r * w, 1, w, 0);  /* rows    */
}

/*
 * BINARY-MERGE, page-wise binary merge, Algorithm 6 (L457-490), L127, L416-420.
 * Streams I[0], I[1] of n[0], n[1] elements; shared array S[M], M = w*w; page = M/2.
 * Followed line by line; the repairs are reading A9 (e = 0 restored at L466-468) and
 * L420 (arbitrary stream sizes: ls = min(M/2, n[e] - ic[e]), partial pages padded with
 * infinity, padding subtracted from the output).
 * Because SHEARSORT-MERGE needs its two inputs sorted, and after a merge the upper half
 * S[M/2..M) is sorted and the freshly loaded page S[0..M/2) is sorted, each call merges
 * (page, upper half).
 */
static int ORC_(binary_merge_pagewise)(const ORC_(elem) *I0, size_t n0, const ORC_(elem) *I1, size_t n1,
                                       ORC_(elem) *O, size_t w)
{
    size_t M = w * w, H = M / 2;
    if (M < 2) return -2;
    const ORC_(elem) *I[2] = { I0, I1 };
    size_t n[2] = { n0, n1 }, ic[2] = { 0, 0 }, oc = 0, total = n0 + n1;
    ORC_(elem) INF; INF.k = (ORC_K)~(ORC_K)0; INF.v = 0xFFFFFFFFu;
    ORC_(elem) *S = (ORC_(elem) *)malloc(M * sizeof(ORC_(elem)));
    if (!S) return -1;
    int e = 0;

    /* L464: load a page of M/2 keys from each input stream into S (padded, L420) */
    for (int s = 0; s < 2; ++s) {
        size_t ls = n[s] < H ? n[s] : H;
        for (size_t i = 0; i < H; ++i) S[s * H + i] = i < ls ? I[s][i] : INF;
        ic[s] = ls;
    }
    /* L466-468: the input stream whose page will be exhausted first */
    e = ORC_(le)(S[H - 1], S[M - 1]) ? 0 : 1;
    /* L470: merge the first pages */
    ORC_(shearsort_merge)(S, w, H);
    /* L472: write the first page to the output stream (never write padding) */
    for (size_t i = 0; i < H && oc < total; ++i) O[oc++] = S[i];

    /* L475: WHILE (ic[0] < n) OR (ic[1] < n) */
    while (ic[0] < n[0] || ic[1] < n[1]) {
        if (ic[e] >= n[e]) e = 1 - e;                                  /* L478 */
        size_t ls = n[e] - ic[e] < H ? n[e] - ic[e] : H;               /* L420 */
        for (size_t i = 0; i < H; ++i) S[i] = i < ls ? I[e][ic[e] + i] : INF;   /* L479 */
        ic[e] += ls;                                                   /* L480 */
        /* L482: which is the next page to be exhausted.  S[H-1] is the last key loaded
         * from stream e, S[M-1] the largest key still held from before. */
        if (ORC_(lt)(S[M - 1], S[H - 1])) e = 1 - e;
        ORC_(shearsort_merge)(S, w, H);                                /* L484 */
        for (size_t i = 0; i < H && oc < total; ++i) O[oc++] = S[i];   /* L486-487 */
    }
    /* L489: write the final remaining page */
    for (size_t i = H; i < M && oc < total; ++i) O[oc++] = S[i];
    free(S);
    return oc == total ? 0 : -3;
}
