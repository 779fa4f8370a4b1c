/* oracle/qed_combi.h — TEST INFRASTRUCTURE (CPU oracle). Not part of the product path.
 *
 * Combinatorics of QED vertex graphs without lepton loops, as read from the paper
 * ("UV divergent subdiagrams", "forestlike formula"; PAPER.md:104 classes (k,m,n);
 * PAPER.md:153 fn5 mirror images) and fixed in DESIGN.md "Readings" R1-R4:
 *
 *  - a graph of loop order L is an open electron path with positions 0..2L; position e carries the
 *    external photon; the other 2L positions are joined pairwise by L photon chords (a_i<b_i).
 *  - electron line t joins positions t,t+1 (line index t); photon i (chords sorted by a) has line
 *    index 2L+i; M=3L internal lines.
 *  - valid graph (1PI vertex graph): every electron line t is spanned by a chord (a<=t<b).
 *  - UV-divergent subgraph: contiguous position segment [lo,hi] != [0,2L], vertex-induced, with
 *    ext = #positions whose photon leaves the segment (e counts) equal to 0 (type S, electron
 *    self-energy) or 1 (type V, vertex-like), and 1PI inside.
 *  - forest: set of pairwise nested-or-disjoint subgraphs.
 *
 * Plain C, no cleverness: everything is enumerated by brute force.
 */
#ifndef QED_COMBI_H
#define QED_COMBI_H
#include <stdint.h>
#include <string.h>
#include <stdlib.h>

#define MAXL 5
#define MAXPOS 11
#define MAXM 15
#define MAXSUB 24
#define MAXFOREST 256
#define MAXTERM 256

typedef struct {
  int L, M, npos, e;
  int a[MAXL], b[MAXL]; /* chords sorted by a */
  int chord_at[MAXPOS]; /* chord index at a position, -1 at e */
  int other[MAXPOS];    /* partner position, -1 at e */
} Graph;

typedef struct { int lo, hi, type; /* 0=S, 1=V */ } Sub;

/* returns 0 if ok, <0 if the input is not a valid graph */
static int graph_init(Graph *g, int L, int e, const int *ca, const int *cb) {
  if (L < 1 || L > MAXL) return -1;
  memset(g, 0, sizeof *g);
  g->L = L; g->M = 3 * L; g->npos = 2 * L + 1; g->e = e;
  if (e < 0 || e > 2 * L) return -2;
  int a[MAXL], b[MAXL];
  for (int i = 0; i < L; i++) {
    a[i] = ca[i]; b[i] = cb[i];
    if (a[i] > b[i]) { int t = a[i]; a[i] = b[i]; b[i] = t; }
    if (a[i] < 0 || b[i] > 2 * L || a[i] == b[i]) return -3;
  }
  /* sort by a (insertion sort) */
  for (int i = 1; i < L; i++)
    for (int j = i; j > 0 && a[j - 1] > a[j]; j--) {
      int t = a[j]; a[j] = a[j - 1]; a[j - 1] = t;
      t = b[j]; b[j] = b[j - 1]; b[j - 1] = t;
    }
  for (int p = 0; p < g->npos; p++) { g->chord_at[p] = -1; g->other[p] = -1; }
  for (int i = 0; i < L; i++) {
    g->a[i] = a[i]; g->b[i] = b[i];
    if (a[i] == e || b[i] == e) return -4;
    if (g->chord_at[a[i]] != -1 || g->chord_at[b[i]] != -1) return -5; /* not a matching */
    g->chord_at[a[i]] = i; g->chord_at[b[i]] = i;
    g->other[a[i]] = b[i]; g->other[b[i]] = a[i];
  }
  /* 1PI: every electron line covered */
  for (int t = 0; t < 2 * L; t++) {
    int cov = 0;
    for (int i = 0; i < L; i++) if (a[i] <= t && t < b[i]) cov = 1;
    if (!cov) return -6;
  }
  return 0;
}

/* ---- canonical enumeration: ascending e, then lexicographic sorted chord list ---- */
typedef struct { int *list_e, *list_a, *list_b; int L, e, count, want_idx, found; int target_a[MAXL], target_b[MAXL], target_e, match_idx; int out_a[MAXL], out_b[MAXL], out_e; } EnumCtx;

static void enum_rec(EnumCtx *c, int *used, int k, int *a, int *b) {
  int L = c->L, npos = 2 * L + 1;
  if (k == L) {
    Graph g;
    if (graph_init(&g, L, c->e, a, b) != 0) return;
    if (c->list_e) { c->list_e[c->count] = c->e; memcpy(c->list_a + c->count * MAXL, a, sizeof(int) * L); memcpy(c->list_b + c->count * MAXL, b, sizeof(int) * L); }
    if (c->want_idx == c->count) { c->found = 1; c->out_e = c->e; memcpy(c->out_a, a, sizeof(int) * L); memcpy(c->out_b, b, sizeof(int) * L); }
    if (c->target_e == c->e && memcmp(c->target_a, a, sizeof(int) * L) == 0 && memcmp(c->target_b, b, sizeof(int) * L) == 0) c->match_idx = c->count;
    c->count++;
    return;
  }
  int p = 0;
  while (p < npos && (used[p] || p == c->e)) p++;
  if (p >= npos) return;
  used[p] = 1; a[k] = p;
  for (int q = p + 1; q < npos; q++) {
    if (used[q] || q == c->e) continue;
    used[q] = 1; b[k] = q;
    enum_rec(c, used, k + 1, a, b);
    used[q] = 0;
  }
  used[p] = 0;
}

/* run the enumeration; want_idx<0: just count / match target */
static void enum_run(EnumCtx *c, int L) {
  c->L = L; c->count = 0; c->found = 0; c->match_idx = -1;
  for (int e = 0; e <= 2 * L; e++) {
    int used[MAXPOS] = {0}, a[MAXL], b[MAXL];
    c->e = e;
    enum_rec(c, used, 0, a, b);
  }
}

static int graph_count(int L) { EnumCtx c; memset(&c, 0, sizeof c); c.want_idx = -1; c.target_e = -1; enum_run(&c, L); return c.count; }

static int graph_by_index(int L, int idx, Graph *g) {
  EnumCtx c; memset(&c, 0, sizeof c); c.want_idx = idx; c.target_e = -1; enum_run(&c, L);
  if (!c.found) return -1;
  return graph_init(g, L, c.out_e, c.out_a, c.out_b);
}

static int graph_canonical_id(const Graph *g) {
  EnumCtx c; memset(&c, 0, sizeof c); c.want_idx = -1; c.target_e = g->e;
  memcpy(c.target_a, g->a, sizeof(int) * g->L); memcpy(c.target_b, g->b, sizeof(int) * g->L);
  enum_run(&c, g->L);
  return c.match_idx;
}

/* class (k,m,n) */
static void graph_class(const Graph *g, int *k, int *m, int *n) {
  int kk = 0, l = 0, r = 0;
  for (int i = 0; i < g->L; i++) {
    if (g->a[i] < g->e && g->e < g->b[i]) kk++;
    else if (g->b[i] < g->e) l++;
    else r++;
  }
  *k = kk; *m = l > r ? l : r; *n = l > r ? r : l;
}

/* mirror image x -> 2L-x */
static int graph_mirror(const Graph *g, Graph *out) {
  int a[MAXL], b[MAXL];
  for (int i = 0; i < g->L; i++) { a[i] = 2 * g->L - g->b[i]; b[i] = 2 * g->L - g->a[i]; }
  return graph_init(out, g->L, 2 * g->L - g->e, a, b);
}

/* ---- UV-divergent subgraphs ---- */
static int seg_is_1pi(const Graph *g, int lo, int hi) {
  for (int t = lo; t < hi; t++) {
    int cov = 0;
    for (int i = 0; i < g->L; i++)
      if (g->a[i] >= lo && g->b[i] <= hi && g->a[i] <= t && t < g->b[i]) cov = 1;
    if (!cov) return 0;
  }
  return 1;
}
static int seg_ext(const Graph *g, int lo, int hi) {
  int ext = 0;
  for (int x = lo; x <= hi; x++) {
    if (x == g->e) ext++;
    else if (g->other[x] < lo || g->other[x] > hi) ext++;
  }
  return ext;
}
static int enum_subgraphs(const Graph *g, Sub *subs) {
  int n = 0;
  for (int lo = 0; lo <= 2 * g->L; lo++)
    for (int hi = lo + 1; hi <= 2 * g->L; hi++) {
      if (lo == 0 && hi == 2 * g->L) continue;
      int ext = seg_ext(g, lo, hi);
      if (ext > 1) continue;
      if (!seg_is_1pi(g, lo, hi)) continue;
      subs[n].lo = lo; subs[n].hi = hi; subs[n].type = ext; n++;
    }
  return n; /* ascending (lo,hi) by construction */
}
static int subs_compatible(const Sub *x, const Sub *y) {
  if (x->lo <= y->lo && y->hi <= x->hi) return 1;
  if (y->lo <= x->lo && x->hi <= y->hi) return 1;
  if (x->hi < y->lo || y->hi < x->lo) return 1;
  return 0;
}
/* all forests of proper subgraphs (the empty one included), ascending bitmask */
static int enum_forests(const Sub *subs, int nsub, uint32_t *forests) {
  int n = 0;
  for (uint32_t m = 0; m < (1u << nsub); m++) {
    int ok = 1;
    for (int i = 0; i < nsub && ok; i++) if (m >> i & 1)
      for (int j = i + 1; j < nsub && ok; j++) if (m >> j & 1)
        if (!subs_compatible(&subs[i], &subs[j])) ok = 0;
    if (ok) forests[n++] = m;
  }
  return n;
}

/* terms of the forest-like formula: (forest, G') with G' in I[G]∩F; gprime=-1 means G'=G */
typedef struct { uint32_t forest; int gprime; int sign; } Term;
static int enum_terms(const Graph *g, const Sub *subs, int nsub, const uint32_t *forests, int nforest, Term *terms) {
  int n = 0;
  for (int f = 0; f < nforest; f++) {
    int size = 1 + __builtin_popcount(forests[f]); /* |F| including G */
    int sign = (size - 1) % 2 ? -1 : 1;
    terms[n].forest = forests[f]; terms[n].gprime = -1; terms[n].sign = sign; n++;
    for (int i = 0; i < nsub; i++)
      if ((forests[f] >> i & 1) && subs[i].type == 1 && subs[i].lo <= g->e && g->e <= subs[i].hi) {
        terms[n].forest = forests[f]; terms[n].gprime = i; terms[n].sign = sign; n++;
      }
  }
  return n;
}
#endif
