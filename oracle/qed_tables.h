/* oracle/qed_tables.h — TEST INFRASTRUCTURE (CPU oracle).
 *
 * Numerator of one piece under one operator, written out with explicit 4x4 complex Dirac
 * matrices (Dirac representation, metric (+,-,-,-), rest frame p=(m,0,0,0), m=1).
 * DESIGN.md O3-O5. The paper only names the operators; the definitions below
 * are the DESIGN.md reading of its ref. [14].
 *
 * String of a piece (reverse path order, i.e. M <- E * M while walking the path):
 *   photon vertex of own chord i : gamma^{alpha_i}, the two ends contracted with g (Feynman gauge)
 *   free vertex                  : gamma^mu (mu kept open)
 *   electron line t              : (A_t pslash + m + kappaslash_t [+ A'_t qslash])
 *                                  with A_t pslash + m = (1+A_t) P+ + (1-A_t) P-  = (2-x_t) P+ + x_t P-
 *   S-child insertion            : a + b (A_t pslash + kappaslash_t [+ A'_t qslash])
 * kappa's are Wick-paired: a pair (t,u) -> (-1/2) beta_tu gamma^rho ... gamma_rho.
 * Every way of choosing {P+, P-, kappa, q} per slot and pairing the kappas is one monomial; its
 * coefficient is the operator's linear functional applied to the constant matrix string, obtained
 * here by a depth-first walk over the choices that carries the partial product as a tensor over
 * the currently open Lorentz indices.
 */
#ifndef QED_TABLES_H
#define QED_TABLES_H
#include "qed_piece.h"
#include <complex.h>
#include <stdio.h>

typedef double complex cplx;
enum { OP_A = 0, OP_U = 1, OP_L = 2, OP_LMU = 3 };
/* factor kinds of a monomial */
enum { F_DPLUS = 0, F_DMINUS = 1, F_BETA = 2, F_AQ = 3, F_AT = 4 };
#define MAXFAC 24

typedef struct {
  double coef[2];           /* output 0 (and 1 for U on an S-type piece: a, b) */
  int grade;                /* own contractions c */
  int pattern;              /* bit c set: S-child c enters with its b part (else a part) */
  int nfac; struct { unsigned char kind, i, j; } fac[MAXFAC];
} Monomial;

typedef struct { int nout; int n, cap; Monomial *mono; } PieceTable;

/* ---------- Dirac matrices: sparse rows, (gamma M)[r][c] = val[r] * M[perm[r]][c] ---------- */
static const int GPERM[4][4] = {{0, 1, 2, 3}, {3, 2, 1, 0}, {3, 2, 1, 0}, {2, 3, 0, 1}};
static const cplx GVAL[4][4] = {{1, 1, -1, -1}, {1, 1, -1, -1}, {-I, I, I, -I}, {1, -1, -1, 1}};
static const double GMET[4] = {1, -1, -1, -1};

static void dense_gamma(int mu, cplx G[4][4]) {
  memset(G, 0, sizeof(cplx) * 16);
  for (int r = 0; r < 4; r++) G[r][GPERM[mu][r]] = GVAL[mu][r];
}
static void matmul(const cplx A[4][4], const cplx B[4][4], cplx C[4][4]) {
  cplx T[4][4];
  for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) { cplx s = 0; for (int k = 0; k < 4; k++) s += A[i][k] * B[k][j]; T[i][j] = s; }
  memcpy(C, T, sizeof T);
}
static cplx trace4(const cplx A[4][4]) { return A[0][0] + A[1][1] + A[2][2] + A[3][3]; }

/* ---------- tensor over open Lorentz indices; every axis has size 4, axis k has stride 4^k ---------- */
enum { AX_CHORD = 0, AX_KAPPA = 1, AX_MU = 2, AX_NU = 3 };
typedef struct { int nax; int tag[14], id[14]; cplx (*m)[4][4]; } Tens;

/* tensors live on a per-thread LIFO arena (the depth-first walk frees in reverse order of allocation) */
static __thread char *tens_arena = NULL;
static __thread size_t tens_top = 0, tens_cap = 0;
static Tens tens_alloc(int nax) {
  Tens t; t.nax = nax;
  size_t bytes = sizeof(cplx) * 16 * ((size_t)1 << (2 * nax));
  if (!tens_arena) { tens_cap = (size_t)6 << 30; tens_arena = (char *)malloc(tens_cap); /* virtual; touched lazily */ }
  if (tens_top + bytes > tens_cap) { fprintf(stderr, "oracle: tensor arena exhausted\n"); abort(); }
  t.m = (cplx(*)[4][4])(tens_arena + tens_top); tens_top += bytes;
  return t;
}
static void tens_free(Tens *t) { tens_top -= sizeof(cplx) * 16 * ((size_t)1 << (2 * t->nax)); t->m = NULL; }
static Tens tens_open(const Tens *src, int tag, int id) {     /* T'[.., rho] = gamma^rho T[..] */
  Tens t = tens_alloc(src->nax + 1);
  memcpy(t.tag, src->tag, sizeof(int) * src->nax); memcpy(t.id, src->id, sizeof(int) * src->nax);
  t.tag[src->nax] = tag; t.id[src->nax] = id;
  size_t n = (size_t)1 << (2 * src->nax);
  for (int rho = 0; rho < 4; rho++) for (size_t k = 0; k < n; k++)
    for (int r = 0; r < 4; r++) for (int c = 0; c < 4; c++) t.m[rho * n + k][r][c] = GVAL[rho][r] * src->m[k][GPERM[rho][r]][c];
  return t;
}
static Tens tens_close(const Tens *src, int ax) {            /* T'[rest] = sum_rho g_rr gamma^rho T[rest, rho@ax] */
  Tens t = tens_alloc(src->nax - 1);
  for (int k = 0, j = 0; k < src->nax; k++) if (k != ax) { t.tag[j] = src->tag[k]; t.id[j] = src->id[k]; j++; }
  size_t lowsz = (size_t)1 << (2 * ax), n = (size_t)1 << (2 * t.nax);
  for (size_t k = 0; k < n; k++) {
    size_t low = k & (lowsz - 1), high = k >> (2 * ax);
    for (int r = 0; r < 4; r++) for (int c = 0; c < 4; c++) {
      cplx s = 0;
      for (int rho = 0; rho < 4; rho++) {
        size_t src_idx = low + (size_t)rho * lowsz + high * lowsz * 4;
        s += GMET[rho] * GVAL[rho][r] * src->m[src_idx][GPERM[rho][r]][c];
      }
      t.m[k][r][c] = s;
    }
  }
  return t;
}
static Tens tens_diag(const Tens *src, const double d[4]) {  /* T' = diag(d) T */
  Tens t = tens_alloc(src->nax);
  memcpy(t.tag, src->tag, sizeof(int) * src->nax); memcpy(t.id, src->id, sizeof(int) * src->nax);
  size_t n = (size_t)1 << (2 * src->nax);
  for (size_t k = 0; k < n; k++) for (int r = 0; r < 4; r++) for (int c = 0; c < 4; c++) t.m[k][r][c] = d[r] * src->m[k][r][c];
  return t;
}
static int tens_find(const Tens *t, int tag, int id) { for (int k = 0; k < t->nax; k++) if (t->tag[k] == tag && (id < 0 || t->id[k] == id)) return k; return -1; }

/* ---------- operator functionals (O4) ---------- */
/* X[mu]: string with free index mu at q=0.   L[X] = Tr[(pslash+m) p_mu X^mu]/(4m^2) = Tr[(g0+1) X^0]/4 */
static cplx func_L(cplx X[4][4][4]) {
  cplx G0[4][4], P[4][4], T[4][4]; dense_gamma(0, G0);
  memcpy(P, G0, sizeof P); for (int i = 0; i < 4; i++) P[i][i] += 1.0;
  matmul(P, X[0], T); return trace4(T) / 4.0;
}
/* U_V[X] = ( Tr[gamma_mu X^mu] - Tr[pslash p_mu X^mu]/m^2 ) / 12.  func_UV12 returns 12 U_V[X]: the
 * traces are integers, so 12 U_V is exactly representable while U_V (a multiple of 1/12) is not; tables
 * of the operators U and (L-U) on vertex-like pieces therefore store 12*coefficient and the evaluation
 * divides by 12 once in its working precision (O5, "exact coefficients") */
static cplx func_UV12(cplx X[4][4][4]) {
  cplx s = 0, G[4][4], T[4][4];
  for (int mu = 0; mu < 4; mu++) { dense_gamma(mu, G); matmul(G, X[mu], T); s += GMET[mu] * trace4(T); }
  dense_gamma(0, G); matmul(G, X[0], T); s -= trace4(T);
  return s;
}
static cplx func_UV(cplx X[4][4][4]) { return func_UV12(X) / 12.0; }
/* R[T] = sum_{jkl} eps_jkl Tr[ Sigma^l P+ T^{jk} ] with
 * T^{jk} = (ps+m) Y^{jk} (ps+m) + 1/2 g^k X^j (ps+m) - 1/2 (ps+m) X^j g^k   (j,k spatial) */
static void sigma_Pplus(int l, cplx S[4][4]) { /* Sigma^l P+ , Sigma^l = diag(sigma^l, sigma^l) */
  memset(S, 0, sizeof(cplx) * 16);
  if (l == 1) { S[0][1] = 1; S[1][0] = 1; }
  if (l == 2) { S[0][1] = -I; S[1][0] = I; }
  if (l == 3) { S[0][0] = 1; S[1][1] = -1; }
}
static int eps3(int j, int k, int l) { return (j - k) * (k - l) * (l - j) / 2; } /* Levi-Civita on 1..3 */
static cplx func_R_X(cplx X[4][4][4]) {
  cplx s = 0, G0[4][4], PM[4][4], Gk[4][4], S[4][4], T1[4][4], T2[4][4];
  dense_gamma(0, G0); memcpy(PM, G0, sizeof PM); for (int i = 0; i < 4; i++) PM[i][i] += 1.0;
  for (int j = 1; j <= 3; j++) for (int k = 1; k <= 3; k++) for (int l = 1; l <= 3; l++) {
    int e = eps3(j, k, l); if (!e) continue;
    dense_gamma(k, Gk); sigma_Pplus(l, S);
    matmul(Gk, X[j], T1); matmul(T1, PM, T1);         /* g^k X^j (ps+m) */
    matmul(PM, X[j], T2); matmul(T2, Gk, T2);         /* (ps+m) X^j g^k */
    for (int r = 0; r < 4; r++) for (int c = 0; c < 4; c++) T1[r][c] = 0.5 * T1[r][c] - 0.5 * T2[r][c];
    matmul(S, T1, T1); s += (double)e * trace4(T1);
  }
  return s;
}
static cplx func_R_Y(cplx Y[4][4][4][4]) { /* Y[j][k] */
  cplx s = 0, G0[4][4], PM[4][4], S[4][4], T1[4][4];
  dense_gamma(0, G0); memcpy(PM, G0, sizeof PM); for (int i = 0; i < 4; i++) PM[i][i] += 1.0;
  for (int j = 1; j <= 3; j++) for (int k = 1; k <= 3; k++) for (int l = 1; l <= 3; l++) {
    int e = eps3(j, k, l); if (!e) continue;
    sigma_Pplus(l, S);
    matmul(PM, Y[j][k], T1); matmul(T1, PM, T1); matmul(S, T1, T1);
    s += (double)e * trace4(T1);
  }
  return s;
}
static cplx R_gamma(void) { /* normalisation: X^j = gamma^j, Y = 0 */
  cplx X[4][4][4]; for (int mu = 0; mu < 4; mu++) dense_gamma(mu, X[mu]);
  return func_R_X(X);
}

/* ---------- depth-first expansion ---------- */
typedef struct {
  const Geom *h; int op; PieceTable *tab; cplx Rg;
  int nfac; struct { unsigned char kind, i, j; } fac[MAXFAC];
  int grade, pattern, used_q, max_grade;
  int nopenk;
  int spawn_at;                 /* element index at which the walk is cut into independent sub-walks (-1: never) */
  struct Frontier *front;
} Dfs;
typedef struct Frontier { int n, cap; struct FrontierItem { Dfs d; Tens T; } *item; } Frontier;

static void table_push(PieceTable *t, const Monomial *m) {
  if (t->n == t->cap) { t->cap = t->cap ? 2 * t->cap : 256; t->mono = (Monomial *)realloc(t->mono, sizeof(Monomial) * t->cap); }
  t->mono[t->n++] = *m;
}
static void dfs_leaf(Dfs *d, const Tens *T) {
  const Geom *h = d->h;
  cplx out[2] = {0, 0};
  if (h->type == 0) {                    /* S-type: U_S = (Tr S/4, Tr[g0 S]/4) */
    cplx G0[4][4], Tm[4][4]; dense_gamma(0, G0);
    out[0] = trace4(T->m[0]) / 4.0; matmul(G0, T->m[0], Tm); out[1] = trace4(Tm) / 4.0;
  } else if (!d->used_q) {
    cplx X[4][4][4]; memcpy(X, T->m, sizeof X);   /* single axis MU */
    if (d->op == OP_L) out[0] = func_L(X);
    else if (d->op == OP_U) out[0] = func_UV12(X);                         /* 12 * coefficient, see func_UV12 */
    else if (d->op == OP_LMU) out[0] = 12.0 * func_L(X) - func_UV12(X);     /* 12 * coefficient */
    else out[0] = func_R_X(X) / d->Rg - func_L(X);
  } else {
    int amu = tens_find(T, AX_MU, -1), anu = tens_find(T, AX_NU, -1);
    cplx Y[4][4][4][4];
    for (int j = 0; j < 4; j++) for (int k = 0; k < 4; k++) {
      size_t idx = (size_t)j << (2 * amu) | (size_t)k << (2 * anu);
      memcpy(Y[j][k], T->m[idx], sizeof(cplx) * 16);
    }
    out[0] = func_R_Y(Y) / d->Rg;
  }
  double pref = 1.0;
  for (int i = 0; i < h->nch; i++) pref *= -0.25;
  for (int i = 0; i < d->grade; i++) pref *= -0.5;
  if (cabs(out[0]) < 1e-12 && cabs(out[1]) < 1e-12) return;
  if (fabs(cimag(out[0])) > 1e-9 || fabs(cimag(out[1])) > 1e-9) { fprintf(stderr, "oracle: complex coefficient %g%+gi\n", creal(out[0]), cimag(out[0])); abort(); }
  Monomial m; memset(&m, 0, sizeof m);
  m.coef[0] = pref * creal(out[0]); m.coef[1] = pref * creal(out[1]);
  m.grade = d->grade; m.pattern = d->pattern; m.nfac = d->nfac;
  memcpy(m.fac, d->fac, sizeof m.fac);
  table_push(d->tab, &m);
}

static void dfs_step(Dfs *d, int ei, const Tens *T);

static void dfs_choice_fixed(Dfs *d, int ei, const Tens *T, const double diag[4], int fkind, int slot) {
  Tens t2 = tens_diag(T, diag);
  int nf0 = d->nfac;
  if (fkind >= 0) { d->fac[d->nfac].kind = (unsigned char)fkind; d->fac[d->nfac].i = (unsigned char)slot; d->fac[d->nfac].j = 0; d->nfac++; }
  dfs_step(d, ei + 1, &t2);
  d->nfac = nf0; tens_free(&t2);
}

static void dfs_step(Dfs *d, int ei, const Tens *T) {
  const Geom *h = d->h;
  if (ei == h->nelem) { if (d->nopenk == 0) dfs_leaf(d, T); return; }
  if (ei == d->spawn_at && d->front) {     /* save the state; the sub-walk is run later, possibly on another thread */
    Frontier *f = d->front;
    if (f->n == f->cap) { f->cap = f->cap ? 2 * f->cap : 64; f->item = (struct FrontierItem *)realloc(f->item, sizeof(struct FrontierItem) * f->cap); }
    struct FrontierItem *it = &f->item[f->n++];
    it->d = *d; it->d.front = NULL; it->T = *T;
    size_t bytes = sizeof(cplx) * 16 * ((size_t)1 << (2 * T->nax));
    it->T.m = (cplx(*)[4][4])malloc(bytes); memcpy(it->T.m, T->m, bytes);
    return;
  }
  /* not enough slots left to close the open kappas? */
  int slots_left = 0;
  for (int k = ei; k < h->nelem; k++) if (h->elem[k].kind == EL_SLOT) slots_left++;
  if (d->nopenk > slots_left) return;
  int kind = h->elem[ei].kind;
  if (kind == EL_VCHORD) {
    int ch = h->elem[ei].chord, ax = tens_find(T, AX_CHORD, ch);
    Tens t2 = (ax < 0) ? tens_open(T, AX_CHORD, ch) : tens_close(T, ax);
    dfs_step(d, ei + 1, &t2); tens_free(&t2);
    return;
  }
  if (kind == EL_VFREE) {
    Tens t2 = tens_open(T, AX_MU, 0);
    dfs_step(d, ei + 1, &t2); tens_free(&t2);
    return;
  }
  /* momentum slot */
  int s = h->elem[ei].slot, ins = (h->slot[s].kind == SLOT_INS), child = h->slot[s].child;
  static const double PPLUS[4] = {1, 1, 0, 0}, PMINUS[4] = {0, 0, 1, 1}, ONE[4] = {1, 1, 1, 1}, G0D[4] = {1, 1, -1, -1};
  int pat0 = d->pattern;
  if (!ins) {
    dfs_choice_fixed(d, ei, T, PPLUS, F_DPLUS, s);
    dfs_choice_fixed(d, ei, T, PMINUS, F_DMINUS, s);
  } else {
    dfs_choice_fixed(d, ei, T, ONE, -1, s);            /* a-part: identity, pattern bit stays 0 */
    d->pattern = pat0 | (1 << child);
    dfs_choice_fixed(d, ei, T, G0D, F_AT, s);          /* b * A_t pslash */
  }
  if (ins) d->pattern = pat0 | (1 << child);
  /* kappa: open a new index ... */
  if (d->grade + d->nopenk + 1 <= d->max_grade) {
    Tens t2 = tens_open(T, AX_KAPPA, s);
    d->nopenk++;
    dfs_step(d, ei + 1, &t2);
    d->nopenk--; tens_free(&t2);
  }
  /* ... or close one of the open kappa indices (Wick pair (u,s), weight beta_us) */
  for (int ax = 0; ax < T->nax; ax++) if (T->tag[ax] == AX_KAPPA) {
    int u = T->id[ax];
    Tens t2 = tens_close(T, ax);
    d->fac[d->nfac].kind = F_BETA; d->fac[d->nfac].i = (unsigned char)u; d->fac[d->nfac].j = (unsigned char)s; d->nfac++;
    d->grade++; d->nopenk--;
    dfs_step(d, ei + 1, &t2);
    d->grade--; d->nopenk++; d->nfac--; tens_free(&t2);
  }
  /* q-part (only under operator A, at most once): gamma^nu with nu open, weight A'_s */
  if (d->op == OP_A && !d->used_q) {
    Tens t2 = tens_open(T, AX_NU, 0);
    d->fac[d->nfac].kind = F_AQ; d->fac[d->nfac].i = (unsigned char)s; d->fac[d->nfac].j = 0; d->nfac++;
    d->used_q = 1;
    dfs_step(d, ei + 1, &t2);
    d->used_q = 0; d->nfac--; tens_free(&t2);
  }
  d->pattern = pat0;
}

/* max_grade<0: no pruning */
static void build_piece_table(const Geom *h, int op, int max_grade, PieceTable *tab) {
  memset(tab, 0, sizeof *tab);
  tab->nout = (h->type == 0) ? 2 : 1;
  Dfs d; memset(&d, 0, sizeof d);
  d.h = h; d.op = op; d.tab = tab; d.Rg = R_gamma();
  d.max_grade = max_grade < 0 ? 99 : max_grade;
  Frontier fr; memset(&fr, 0, sizeof fr);
  d.spawn_at = h->nelem > 8 ? 6 : -1; d.front = d.spawn_at >= 0 ? &fr : NULL;
  Tens T = tens_alloc(0);
  memset(T.m[0], 0, sizeof(cplx) * 16); for (int i = 0; i < 4; i++) T.m[0][i][i] = 1.0;
  dfs_step(&d, 0, &T);
  tens_free(&T);
  if (fr.n) {   /* run the sub-walks in parallel, then concatenate their monomials in walk order */
    PieceTable *part = (PieceTable *)calloc(fr.n, sizeof(PieceTable));
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < fr.n; k++) {
      Dfs sub = fr.item[k].d; sub.tab = &part[k]; sub.front = NULL;
      dfs_step(&sub, sub.spawn_at, &fr.item[k].T);
    }
    for (int k = 0; k < fr.n; k++) {
      for (int i = 0; i < part[k].n; i++) table_push(tab, &part[k].mono[i]);
      free(part[k].mono); free(fr.item[k].T.m);
    }
    free(part); free(fr.item);
  }
}
#endif
