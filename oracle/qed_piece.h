/* oracle/qed_piece.h — TEST INFRASTRUCTURE (CPU oracle).
 *
 * A "piece" is a forest element H (or G) with its maximal children shrunk (R5):
 * a V-child becomes a point vertex carrying the child's scalar, an S-child becomes an insertion
 * slot on the electron line. This header builds the path-ordered element list, the momentum
 * slots and the routing vectors eps of a piece.
 */
#ifndef QED_PIECE_H
#define QED_PIECE_H
#include "qed_combi.h"

#define MAXCHILD 5
#define MAXSLOT 16
#define MAXELEM 40

enum { EL_VCHORD = 0, EL_VFREE = 1, EL_SLOT = 2 };
enum { SLOT_LINE = 0, SLOT_INS = 1 };

typedef struct {
  int lo, hi, type;               /* type 0=S, 1=V */
  int nchild, child_lo[MAXCHILD], child_hi[MAXCHILD], child_type[MAXCHILD];
  int nch, chord[MAXL];           /* own chords (global chord indices) */
  int nline, line[2 * MAXL];      /* own electron lines (global t) */
  int nslot;
  struct { int kind, line, child; unsigned eps; int sgn; } slot[MAXSLOT];
  int nelem;
  struct { int kind, chord /*local*/, slot, child; } elem[MAXELEM];
  int has_e;                      /* external vertex inside H (maybe inside a child) */
} Geom;

static int pos_child(const Geom *h, int pos) {
  for (int c = 0; c < h->nchild; c++) if (h->child_lo[c] <= pos && pos <= h->child_hi[c]) return c;
  return -1;
}

/* children must be given sorted by lo, pairwise disjoint, strictly inside [lo,hi] */
static void geom_build(const Graph *g, int lo, int hi, int type, int nchild, const Sub *children, Geom *h) {
  memset(h, 0, sizeof *h);
  h->lo = lo; h->hi = hi; h->type = type; h->nchild = nchild;
  for (int c = 0; c < nchild; c++) { h->child_lo[c] = children[c].lo; h->child_hi[c] = children[c].hi; h->child_type[c] = children[c].type; }
  h->has_e = (lo <= g->e && g->e <= hi);
  /* own chords: both ends inside H, not both inside the same child */
  int local_of[MAXL];
  for (int i = 0; i < g->L; i++) {
    local_of[i] = -1;
    if (g->a[i] < lo || g->b[i] > hi) continue;
    int ca = pos_child(h, g->a[i]), cb = pos_child(h, g->b[i]);
    if (ca >= 0 && ca == cb) continue;
    local_of[i] = h->nch; h->chord[h->nch++] = i;
  }
  /* free position of a V-type piece: e if inside, else the position whose chord leaves H */
  int freepos = -1;
  if (type == 1) {
    if (h->has_e) freepos = g->e;
    else for (int x = lo; x <= hi; x++) if (g->other[x] < lo || g->other[x] > hi) freepos = x;
  }
  /* walk the path */
  int pos = lo;
  while (pos <= hi) {
    int c = pos_child(h, pos);
    if (c >= 0 && h->child_type[c] == 0) {          /* S-child: insertion slot */
      int s = h->nslot++;
      h->slot[s].kind = SLOT_INS; h->slot[s].child = c; h->slot[s].line = h->child_lo[c] - 1;
      h->elem[h->nelem].kind = EL_SLOT; h->elem[h->nelem].slot = s; h->elem[h->nelem].child = c; h->nelem++;
      pos = h->child_hi[c] + 1;
    } else if (c >= 0) {                             /* V-child: a point vertex */
      int is_free = (freepos >= h->child_lo[c] && freepos <= h->child_hi[c]);
      if (is_free) { h->elem[h->nelem].kind = EL_VFREE; h->elem[h->nelem].chord = -1; }
      else {
        int leave = -1;
        for (int x = h->child_lo[c]; x <= h->child_hi[c]; x++)
          if (x != g->e && (g->other[x] < h->child_lo[c] || g->other[x] > h->child_hi[c])) leave = x;
        h->elem[h->nelem].kind = EL_VCHORD; h->elem[h->nelem].chord = local_of[g->chord_at[leave]];
      }
      h->elem[h->nelem].child = c; h->elem[h->nelem].slot = -1; h->nelem++;
      pos = h->child_hi[c] + 1;
    } else {                                         /* own vertex */
      if (pos == freepos) { h->elem[h->nelem].kind = EL_VFREE; h->elem[h->nelem].chord = -1; }
      else { h->elem[h->nelem].kind = EL_VCHORD; h->elem[h->nelem].chord = local_of[g->chord_at[pos]]; }
      h->elem[h->nelem].child = -1; h->elem[h->nelem].slot = -1; h->nelem++;
      pos++;
    }
    if (pos <= hi) {                                 /* own electron line pos-1 */
      int t = pos - 1, s = h->nslot++;
      h->line[h->nline++] = t;
      h->slot[s].kind = SLOT_LINE; h->slot[s].line = t; h->slot[s].child = -1;
      h->elem[h->nelem].kind = EL_SLOT; h->elem[h->nelem].slot = s; h->elem[h->nelem].child = -1; h->nelem++;
    }
  }
  /* routing: chord i spans slot iff a_i <= t < b_i (t = the slot's line; for an insertion the line before it) */
  for (int s = 0; s < h->nslot; s++) {
    int t = h->slot[s].line; unsigned eps = 0;
    for (int j = 0; j < h->nch; j++) { int i = h->chord[j]; if (g->a[i] <= t && t < g->b[i]) eps |= 1u << j; }
    h->slot[s].eps = eps;
    h->slot[s].sgn = (t < g->e) ? -1 : +1;
  }
}

/* maximal elements of forest F (bitmask over subs) strictly inside segment [lo,hi] (self excluded), sorted by lo */
static int forest_children(const Sub *subs, int nsub, uint32_t F, int lo, int hi, Sub *out, int *out_idx) {
  int n = 0;
  for (int i = 0; i < nsub; i++) {
    if (!(F >> i & 1)) continue;
    if (!(lo <= subs[i].lo && subs[i].hi <= hi) || (subs[i].lo == lo && subs[i].hi == hi)) continue;
    int maximal = 1;
    for (int j = 0; j < nsub; j++) {
      if (j == i || !(F >> j & 1)) continue;
      if (!(lo <= subs[j].lo && subs[j].hi <= hi) || (subs[j].lo == lo && subs[j].hi == hi)) continue;
      if (subs[j].lo <= subs[i].lo && subs[i].hi <= subs[j].hi) maximal = 0;
    }
    if (maximal) { out[n] = subs[i]; if (out_idx) out_idx[n] = i; n++; }
  }
  return n; /* subs are sorted by (lo,hi), so children come out sorted by lo */
}
#endif
