/*
 * bcf_oracle.c -- TEST INFRASTRUCTURE ONLY (CPU oracle, not the product).
 *
 * Exported C entry points of the CPU oracle for the hot path of arXiv 1306.5076
 * (PAPER.md).  The arithmetic lives in bcf_oracle_impl.h, instantiated here for
 * 32-bit and 64-bit keys; this file only converts between the caller's
 * structure-of-arrays buffers (keys[], optional vals[]) and the oracle's
 * array of (key, value) elements.  vals == NULL means "keys only" (value 0).
 *
 * Shares no code with paper_1306_5076_b200/csrc (the CUDA path) and is never
 * linked into it.  Build: python oracle/build.py  (gcc -O2 -shared).
 *
 * Return codes: 0 ok (or the number of merge rounds where stated), <0 error
 * (-1 out of memory, -2 bad argument, -3 internal inconsistency).
 */
#include <stdint.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>

#define ORC_K uint32_t
#define ORC_(x) orc32_##x
#include "bcf_oracle_impl.h"
#undef ORC_K
#undef ORC_

#define ORC_K uint64_t
#define ORC_(x) orc64_##x
#include "bcf_oracle_impl.h"
#undef ORC_K
#undef ORC_

#define DEFINE_SHIMS(P, S, KT)                                                                      \
static P##elem *P##pack(const KT *k, const uint32_t *v, size_t n)                                \
{                                                                                                \
    P##elem *e = (P##elem *)malloc((n ? n : 1) * sizeof(P##elem));                               \
    if (!e) return NULL;                                                                         \
    for (size_t i = 0; i < n; ++i) { e[i].k = k[i]; e[i].v = v ? v[i] : 0u; }                    \
    return e;                                                                                    \
}                                                                                                \
static void P##unpack(const P##elem *e, KT *k, uint32_t *v, size_t n)                            \
{                                                                                                \
    for (size_t i = 0; i < n; ++i) { k[i] = e[i].k; if (v) v[i] = e[i].v; }                      \
}                                                                                                \
/* ShearSort each of num_tiles consecutive w*w tiles (Alg. 1). */                                \
int bcf_oracle_shearsort_tiles_##S(KT *keys, uint32_t *vals, size_t num_tiles, size_t w,         \
                                   int final_snake, int phases)                                  \
{                                                                                                \
    if (w == 0) return -2;                                                                       \
    size_t n = num_tiles * w * w;                                                                \
    P##elem *e = P##pack(keys, vals, n);                                                         \
    if (!e) return -1;                                                                           \
    for (size_t t = 0; t < num_tiles; ++t) P##shearsort_tile(e + t * w * w, w, final_snake, phases); \
    P##unpack(e, keys, vals, n);                                                                 \
    free(e);                                                                                     \
    return 0;                                                                                    \
}                                                                                                \
/* Two-finger merge of sorted A and B into out (L125). */                                        \
int bcf_oracle_merge_two_##S(const KT *ka, const uint32_t *va, size_t na,                        \
                             const KT *kb, const uint32_t *vb, size_t nb,                        \
                             KT *kout, uint32_t *vout)                                           \
{                                                                                                \
    P##elem *a = P##pack(ka, va, na), *b = P##pack(kb, vb, nb);                                  \
    P##elem *o = (P##elem *)malloc((na + nb ? na + nb : 1) * sizeof(P##elem));                   \
    if (!a || !b || !o) { free(a); free(b); free(o); return -1; }                                \
    P##merge_two(a, na, b, nb, o);                                                               \
    P##unpack(o, kout, vout, na + nb);                                                           \
    free(a); free(b); free(o);                                                                   \
    return 0;                                                                                    \
}                                                                                                \
/* Merge rounds over sorted runs of run_len, in place (L103).  Returns rounds. */                \
int bcf_oracle_merge_runs_##S(KT *keys, uint32_t *vals, size_t n, size_t run_len)                \
{                                                                                                \
    if (run_len == 0) return -2;                                                                 \
    P##elem *e = P##pack(keys, vals, n);                                                         \
    P##elem *t = (P##elem *)malloc((n ? n : 1) * sizeof(P##elem));                               \
    if (!e || !t) { free(e); free(t); return -1; }                                               \
    int r = P##merge_runs(e, t, n, run_len);                                                     \
    P##unpack(e, keys, vals, n);                                                                 \
    free(e); free(t);                                                                            \
    return r;                                                                                    \
}                                                                                                \
/* BCFMergesort: ShearSort base case on w*w tiles, then merge rounds.  Returns rounds. */        \
int bcf_oracle_sort_full_##S(KT *keys, uint32_t *vals, size_t n, size_t w)                       \
{                                                                                                \
    if (w == 0) return -2;                                                                       \
    P##elem *e = P##pack(keys, vals, n);                                                         \
    P##elem *t = (P##elem *)malloc((n ? n : 1) * sizeof(P##elem));                               \
    if (!e || !t) { free(e); free(t); return -1; }                                               \
    int r = P##sort_full(e, t, n, w);                                                            \
    P##unpack(e, keys, vals, n);                                                                 \
    free(e); free(t);                                                                            \
    return r;                                                                                    \
}                                                                                                \
/* Co-rank of diagonal d (A-first ties).  Returns (size_t)-1 on error. */                        \
size_t bcf_oracle_corank_##S(const KT *ka, const uint32_t *va, size_t na,                        \
                             const KT *kb, const uint32_t *vb, size_t nb, size_t d)              \
{                                                                                                \
    if (d > na + nb) return (size_t)-1;                                                          \
    P##elem *a = P##pack(ka, va, na), *b = P##pack(kb, vb, nb);                                  \
    if (!a || !b) { free(a); free(b); return (size_t)-1; }                                       \
    size_t i = P##corank(a, na, b, nb, d);                                                       \
    free(a); free(b);                                                                            \
    return i;                                                                                    \
}                                                                                                \
/* SHEARSORT-MERGE on one page S of w*w elements: S[0..na) and S[na..w*w) sorted. */             \
int bcf_oracle_shearsort_merge_##S(KT *keys, uint32_t *vals, size_t w, size_t na)                \
{                                                                                                \
    if (w == 0 || na > w * w) return -2;                                                         \
    P##elem *e = P##pack(keys, vals, w * w);                                                     \
    if (!e) return -1;                                                                           \
    P##shearsort_merge(e, w, na);                                                                \
    P##unpack(e, keys, vals, w * w);                                                             \
    free(e);                                                                                     \
    return 0;                                                                                    \
}                                                                                                \
/* Page-wise binary merge, Alg. 6, with M = w*w. */                                              \
int bcf_oracle_binary_merge_pagewise_##S(const KT *ka, const uint32_t *va, size_t na,            \
                                         const KT *kb, const uint32_t *vb, size_t nb,            \
                                         KT *kout, uint32_t *vout, size_t w)                     \
{                                                                                                \
    if (w < 2 || (w * w) % 2) return -2;                                                         \
    P##elem *a = P##pack(ka, va, na), *b = P##pack(kb, vb, nb);                                  \
    P##elem *o = (P##elem *)malloc((na + nb ? na + nb : 1) * sizeof(P##elem));                   \
    if (!a || !b || !o) { free(a); free(b); free(o); return -1; }                                \
    int r = P##binary_merge_pagewise(a, na, b, nb, o, w);                                        \
    if (r == 0) P##unpack(o, kout, vout, na + nb);                                               \
    free(a); free(b); free(o);                                                                   \
    return r;                                                                                    \
}

DEFINE_SHIMS(orc32_, k32, uint32_t)
DEFINE_SHIMS(orc64_, k64, uint64_t)
