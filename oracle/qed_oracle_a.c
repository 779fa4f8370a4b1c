/* oracle/qed_oracle_a.c — TEST INFRASTRUCTURE: "Oracle-A", the subtracted integrand straight from its definition.
 *
 * Not part of the product path; only tests/ may load it (liboracle_a.so, oracle/build.py). It shares NO code with the
 * CUDA path and none with the table-driven oracle (qed_oracle.c and its headers, "Oracle-B" below): its own graph
 * type, its own enumeration of UV-divergent subgraphs and forests, its own operator assignment, piece geometry,
 * loop-matrix inverse (cofactors), Dirac matrices and traces. Per point, per term, per piece, with
 *   - numeric 4x4 complex matrices  (A_t pslash + m) for every electron line — NOT expanded into P+/P-,
 *   - every Wick pairing of the kappa's enumerated explicitly, each pair closed as (-1/2) beta_tu gamma^rho ... gamma_rho,
 *   - the operators A, U, L of the forest-like formula applied as explicit traces,
 *   - no coefficient tables, no prepare step, no memoisation between terms.
 * It is slow (seconds per point at 4 loops) and exists to pin Oracle-B where the paper gives no number:
 * tests/test_oracle_a.py requires the two to agree to 1e-12 on every 2- and 3-loop graph and on a few 4-loop graphs.
 *
 * What is evaluated (the paper names the operators and the "forestlike formula" and defers their
 * definition to its ref. [14]; the reading is DESIGN.md O1-O6, restated here so that this file can be checked alone):
 *
 *  Graph: open electron path, positions 0..2L, external photon at position e, L photon chords (a_i < b_i) joining the
 *  other positions in pairs. Electron line t joins positions t, t+1 and carries parameter z[t]; photon i (chords sorted
 *  by a) carries z[2L+i]. All electron masses 1, photons massless, Feynman gauge.
 *
 *  UV-divergent subgraph: a position segment [lo,hi] != [0,2L] such that at most one of its positions has its photon
 *  leaving the segment (the external vertex counts as leaving): none -> electron self-energy (S), one -> vertex-like (V);
 *  and every electron line inside is spanned by a chord inside (1PI). Forest: pairwise nested-or-disjoint set.
 *
 *  O1  f_G = sum_{F forest of proper subgraphs} sum_{G' in I[G] ∩ (F ∪ {G})} (-1)^{|F|} prod_{H in F ∪ {G}} M_H ,
 *      I[G] = {G} ∪ {V-type subgraphs containing e};   M_H = A      if H = G'
 *                                                             U      if H not in I[G], or H strictly inside G'
 *                                                             L      if H in I[G], G' strictly inside H, H != G
 *                                                             L - U  if H = G and G' != G
 *      on Gamma^mu(p,0) = a g^mu + b p^mu + c pslash p^mu + d [pslash, g^mu]:  U -> a,  L -> a + m b + m^2 c;
 *      A -> F2(0) (coefficient of i sigma^{mu nu} q_nu / 2m) of Gamma^mu(p,q); on Sigma = a + b pslash: U -> (a, b).
 *  O2  piece = forest element with its maximal children shrunk (V-child: point vertex times the child's scalar; S-child:
 *      insertion a + b (..) on the line). Loop matrix  A = sum_{own lines t} z_t eps_t eps_t^T + diag(z_photon),
 *      eps_ti = 1 iff own chord i spans line t;  U = det A;  beta_tu = eps_t^T A^-1 eps_u;
 *      x_t = sum_{own lines u} z_u beta_tu;  A_t = 1 - x_t;  A'_t = (s_t - sum_u z_u beta_tu s_u)/2, s = -1 before e, +1 after;
 *      V = sum_{own lines u} z_u x_u.
 *  O3  numerator string in reverse path order (each new factor multiplies from the left): own chord vertex gamma^alpha
 *      (two ends contracted with g), free vertex gamma^mu, line (A_t pslash + m + kappaslash_t [+ A'_t qslash]),
 *      insertion a + b (A_t pslash + kappaslash_t [+ A'_t qslash]); rest frame p = (1,0,0,0); kappa's Wick-paired.
 *  O4  L[X] = Tr[(g0+1) X^0]/4;  U_V[X] = (sum_mu g_mumu Tr[g^mu X^mu] - Tr[g0 X^0])/12;  U_S = (Tr S/4, Tr[g0 S]/4);
 *      A[X,Y] = R[T]/R[T_gamma] - L[X], T^{jk} = (g0+1) Y^{jk} (g0+1) + g^k X^j (g0+1)/2 - (g0+1) X^j g^k/2,
 *      R[T] = sum_{jkl} eps_jkl Tr[Sigma^l P+ T^{jk}].
 *  O5  piece value N_c = (-1/4)^{own chords} sum over configurations with c own pairs, graded product with the children.
 *  O6  f_term = sign sum_{c<L} (L-c-1)! N_c / ((prod_H U_H)^2 (sum_H V_H)^{L-c}).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cx;
#define AL 5          /* max loops */
#define ANG 6         /* grades kept */
#define AMAXSEG 32
#define AMAXEL 48
#define AMAXSLOT 16

typedef struct { int L, e, a[AL], b[AL], other[2 * AL + 1]; } AGraph;
typedef struct { int lo, hi, type; } ASeg;                    /* type 0 = S, 1 = V */
typedef struct { double v[2][ANG]; double U, V; } AVal;       /* graded scalar(s) of a forest element, product of U's, sum of V's inside */

/* ---- Dirac matrices, Dirac representation: g0 = diag(1,1,-1,-1), g^i = [[0, s_i], [-s_i, 0]] ---- */
static void a_gamma(int mu, cx G[4][4]) {
  static const cx s[4][2][2] = {{{1, 0}, {0, 1}}, {{0, 1}, {1, 0}}, {{0, -I}, {I, 0}}, {{1, 0}, {0, -1}}};
  memset(G, 0, sizeof(cx) * 16);
  if (mu == 0) { G[0][0] = G[1][1] = 1; G[2][2] = G[3][3] = -1; return; }
  for (int r = 0; r < 2; r++) for (int c = 0; c < 2; c++) { G[r][2 + c] = s[mu][r][c]; G[2 + r][c] = -s[mu][r][c]; }
}
static const double A_MET[4] = {1, -1, -1, -1};
static void a_mul(const cx A[4][4], const cx B[4][4], cx C[4][4]) {
  cx T[4][4];
  for (int i = 0; i < 4; i++) for (int j = 0; j < 4; j++) { cx s = 0; for (int k = 0; k < 4; k++) s += A[i][k] * B[k][j]; T[i][j] = s; }
  memcpy(C, T, sizeof T);
}
static cx a_tr(const cx A[4][4]) { return A[0][0] + A[1][1] + A[2][2] + A[3][3]; }

/* ---- graph, subgraphs ---- */
static int a_graph(AGraph *g, int L, int e, const int *ca, const int *cb) {
  if (L < 1 || L > AL || e < 0 || e > 2 * L) return -1;
  g->L = L; g->e = e;
  for (int x = 0; x <= 2 * L; x++) g->other[x] = -1;
  int a[AL], b[AL];
  for (int i = 0; i < L; i++) { a[i] = ca[i] < cb[i] ? ca[i] : cb[i]; b[i] = ca[i] < cb[i] ? cb[i] : ca[i]; }
  for (int i = 0; i < L; i++) for (int j = i + 1; j < L; j++) if (a[j] < a[i]) { int t = a[i]; a[i] = a[j]; a[j] = t; t = b[i]; b[i] = b[j]; b[j] = t; }
  for (int i = 0; i < L; i++) {
    if (a[i] < 0 || b[i] > 2 * L || a[i] == b[i] || a[i] == e || b[i] == e || g->other[a[i]] >= 0 || g->other[b[i]] >= 0) return -1;
    g->a[i] = a[i]; g->b[i] = b[i]; g->other[a[i]] = b[i]; g->other[b[i]] = a[i];
  }
  return 0;
}
static int a_divergent(const AGraph *g, int lo, int hi, int *type) {
  if (lo == 0 && hi == 2 * g->L) return 0;
  int leaving = 0;
  for (int x = lo; x <= hi; x++) if (x == g->e || g->other[x] < lo || g->other[x] > hi) leaving++;
  if (leaving > 1) return 0;
  for (int t = lo; t < hi; t++) {           /* 1PI: every line inside is spanned by a chord inside */
    int spanned = 0;
    for (int i = 0; i < g->L; i++) if (lo <= g->a[i] && g->b[i] <= hi && g->a[i] <= t && t < g->b[i]) spanned = 1;
    if (!spanned) return 0;
  }
  *type = leaving;
  return 1;
}
static int a_subgraphs(const AGraph *g, ASeg *s) {
  int n = 0;
  for (int lo = 0; lo <= 2 * g->L; lo++) for (int hi = lo + 1; hi <= 2 * g->L; hi++) { int ty; if (a_divergent(g, lo, hi, &ty)) { s[n].lo = lo; s[n].hi = hi; s[n].type = ty; n++; } }
  return n;
}
static int a_inside(const ASeg *x, const ASeg *y) { return y->lo <= x->lo && x->hi <= y->hi; }     /* x within y (or equal) */
static int a_is_forest(const ASeg *s, int n, unsigned F) {
  for (int i = 0; i < n; i++) if (F >> i & 1) for (int j = i + 1; j < n; j++) if (F >> j & 1)
    if (!(a_inside(&s[i], &s[j]) || a_inside(&s[j], &s[i]) || s[i].hi < s[j].lo || s[j].hi < s[i].lo)) return 0;
  return 1;
}

/* ---- tensor over open Lorentz indices: T[idx] is a 4x4 matrix, idx = sum_k i_k 4^k ---- */
enum { AX_CHORD, AX_KAPPA, AX_MU, AX_NU };
typedef struct { int nax, kind[12], id[12]; cx (*m)[4][4]; } ATen;
static ATen at_new(int nax) { ATen t; t.nax = nax; t.m = (cx(*)[4][4])malloc(sizeof(cx) * 16 * ((size_t)1 << (2 * nax))); return t; }
static size_t at_size(const ATen *t) { return (size_t)1 << (2 * t->nax); }
/* T'[idx, rho] = w * gamma^rho T[idx] : a new open index (appended as the most significant axis) */
static ATen at_open(const ATen *s, int kind, int id, double w) {
  ATen t = at_new(s->nax + 1);
  memcpy(t.kind, s->kind, sizeof(int) * s->nax); memcpy(t.id, s->id, sizeof(int) * s->nax);
  t.kind[s->nax] = kind; t.id[s->nax] = id;
  size_t n = at_size(s);
  for (int rho = 0; rho < 4; rho++) { cx G[4][4]; a_gamma(rho, G); for (size_t k = 0; k < n; k++) { a_mul(G, s->m[k], t.m[(size_t)rho * n + k]); for (int r = 0; r < 4; r++) for (int c = 0; c < 4; c++) t.m[(size_t)rho * n + k][r][c] *= w; } }
  return t;
}
/* T'[rest] = w * sum_rho g_{rho rho} gamma^rho T[rest, rho at axis ax] : closes an index */
static ATen at_close(const ATen *s, int ax, double w) {
  ATen t = at_new(s->nax - 1);
  for (int k = 0, j = 0; k < s->nax; k++) if (k != ax) { t.kind[j] = s->kind[k]; t.id[j] = s->id[k]; j++; }
  size_t low = (size_t)1 << (2 * ax), n = at_size(&t);
  cx G[4][4][4]; for (int rho = 0; rho < 4; rho++) a_gamma(rho, G[rho]);
  for (size_t k = 0; k < n; k++) {
    size_t lo = k & (low - 1), hi = k >> (2 * ax);
    memset(t.m[k], 0, sizeof(cx) * 16);
    for (int rho = 0; rho < 4; rho++) {
      cx P[4][4]; a_mul(G[rho], s->m[lo + (size_t)rho * low + hi * low * 4], P);
      for (int r = 0; r < 4; r++) for (int c = 0; c < 4; c++) t.m[k][r][c] += w * A_MET[rho] * P[r][c];
    }
  }
  return t;
}
/* T' = E T for a fixed matrix E */
static ATen at_left(const ATen *s, const cx E[4][4]) {
  ATen t = at_new(s->nax);
  memcpy(t.kind, s->kind, sizeof(int) * s->nax); memcpy(t.id, s->id, sizeof(int) * s->nax);
  size_t n = at_size(s);
  for (size_t k = 0; k < n; k++) a_mul(E, s->m[k], t.m[k]);
  return t;
}
static int at_find(const ATen *t, int kind, int id) { for (int k = 0; k < t->nax; k++) if (t->kind[k] == kind && (id < 0 || t->id[k] == id)) return k; return -1; }

/* ---- operator functionals (O4) as explicit traces ---- */
static cx a_func_L(cx X[4][4][4]) { cx P[4][4], T[4][4]; a_gamma(0, P); for (int i = 0; i < 4; i++) P[i][i] += 1; a_mul(P, X[0], T); return a_tr(T) / 4; }
static cx a_func_UV(cx X[4][4][4]) {
  cx s = 0, G[4][4], T[4][4];
  for (int mu = 0; mu < 4; mu++) { a_gamma(mu, G); a_mul(G, X[mu], T); s += A_MET[mu] * a_tr(T); }
  a_gamma(0, G); a_mul(G, X[0], T); s -= a_tr(T);
  return s / 12;
}
static int a_eps(int j, int k, int l) { return (j - k) * (k - l) * (l - j) / 2; }
/* R[T] for T^{jk} = (g0+1) Y^{jk} (g0+1) + g^k X^j (g0+1)/2 - (g0+1) X^j g^k/2 ; X or Y may be NULL (= 0) */
static cx a_func_R(cx X[4][4][4], cx Y[4][4][4][4]) {
  cx PM[4][4], s = 0; a_gamma(0, PM); for (int i = 0; i < 4; i++) PM[i][i] += 1;
  for (int j = 1; j <= 3; j++) for (int k = 1; k <= 3; k++) for (int l = 1; l <= 3; l++) {
    int e = a_eps(j, k, l); if (!e) continue;
    cx T[4][4]; memset(T, 0, sizeof T);
    if (Y) { cx W[4][4]; a_mul(PM, Y[j][k], W); a_mul(W, PM, W); for (int r = 0; r < 4; r++) for (int c = 0; c < 4; c++) T[r][c] += W[r][c]; }
    if (X) {
      cx Gk[4][4], W1[4][4], W2[4][4]; a_gamma(k, Gk);
      a_mul(Gk, X[j], W1); a_mul(W1, PM, W1); a_mul(PM, X[j], W2); a_mul(W2, Gk, W2);
      for (int r = 0; r < 4; r++) for (int c = 0; c < 4; c++) T[r][c] += 0.5 * W1[r][c] - 0.5 * W2[r][c];
    }
    /* Sigma^l P+ : Sigma^l = diag(sigma_l, sigma_l), P+ = (1+g0)/2 keeps the upper block */
    cx SP[4][4]; memset(SP, 0, sizeof SP);
    if (l == 1) { SP[0][1] = 1; SP[1][0] = 1; } else if (l == 2) { SP[0][1] = -I; SP[1][0] = I; } else { SP[0][0] = 1; SP[1][1] = -1; }
    cx W[4][4]; a_mul(SP, T, W); s += (double)e * a_tr(W);
  }
  return s;
}
static cx a_R_gamma(void) { cx X[4][4][4]; for (int mu = 0; mu < 4; mu++) a_gamma(mu, X[mu]); return a_func_R(X, NULL); }

/* ---- one piece ---- */
enum { OPA_A, OPA_U, OPA_L, OPA_LMU, OPA_NULL };
/* 0 = the definition. Bit 0: U instead of L on intermediate elements of I[G]; bit 1: U instead of L on G when G' != G (the term
 * then vanishes). Deliberately WRONG variants: tests/test_oracle_a.py uses them to show that the infrared pin tells L from U. */
static int a_variant = 0;
enum { EL_CHORDV, EL_FREEV, EL_LINE, EL_INS };
typedef struct {
  int type, nch, chord[AL];                       /* own chords (graph chord indices) */
  int nel; struct { int kind, chord, slot, child; } el[AMAXEL];
  int nslot; struct { int line, ins, child, sgn; unsigned eps; } slot[AMAXSLOT];
  int nchild; const AVal *cval[AMAXSEG]; int ctype[AMAXSEG];
  double beta[AMAXSLOT][AMAXSLOT], At[AMAXSLOT], Aq[AMAXSLOT], U, V;
  int op, Lglobal; cx Rg;
  cx acc[2][ANG];                                  /* sum over configurations, by output and total grade */
} APiece;

static double a_det(int n, double M[AL][AL]) {      /* Laplace expansion along the first row */
  if (n == 1) return M[0][0];
  double d = 0;
  for (int c = 0; c < n; c++) {
    double S[AL][AL];
    for (int i = 1; i < n; i++) for (int j = 0, k = 0; j < n; j++) if (j != c) S[i - 1][k++] = M[i][j];
    d += ((c & 1) ? -1.0 : 1.0) * M[0][c] * a_det(n - 1, S);
  }
  return d;
}
static void a_scalars(const AGraph *g, APiece *p, const double *z) {
  int n = p->nch; double A[AL][AL], Inv[AL][AL];
  for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) A[i][j] = 0;
  for (int s = 0; s < p->nslot; s++) if (!p->slot[s].ins)
    for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) if ((p->slot[s].eps >> i & 1) && (p->slot[s].eps >> j & 1)) A[i][j] += z[p->slot[s].line];
  for (int i = 0; i < n; i++) A[i][i] += z[2 * g->L + p->chord[i]];
  p->U = a_det(n, A);
  for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) {   /* inverse = transposed cofactors / det */
    if (n == 1) { Inv[0][0] = 1 / A[0][0]; continue; }
    double S[AL][AL];
    for (int r = 0, rr = 0; r < n; r++) if (r != j) { for (int c = 0, cc = 0; c < n; c++) if (c != i) S[rr][cc++] = A[r][c]; rr++; }
    Inv[i][j] = (((i + j) & 1) ? -1.0 : 1.0) * a_det(n - 1, S) / p->U;
  }
  for (int s = 0; s < p->nslot; s++) for (int u = 0; u < p->nslot; u++) {
    double b = 0;
    for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) if ((p->slot[s].eps >> i & 1) && (p->slot[u].eps >> j & 1)) b += Inv[i][j];
    p->beta[s][u] = b;
  }
  p->V = 0;
  for (int s = 0; s < p->nslot; s++) {
    double x = 0, q = 0;
    for (int u = 0; u < p->nslot; u++) if (!p->slot[u].ins) { x += z[p->slot[u].line] * p->beta[s][u]; q += z[p->slot[u].line] * p->beta[s][u] * p->slot[u].sgn; }
    p->At[s] = 1 - x; p->Aq[s] = 0.5 * (p->slot[s].sgn - q);
    if (!p->slot[s].ins) p->V += z[p->slot[s].line] * x;
  }
}

static void a_gmul(const double *x, const double *y, double *out) {   /* graded product, truncated */
  double r[ANG];
  for (int c = 0; c < ANG; c++) { r[c] = 0; for (int i = 0; i <= c; i++) r[c] += x[i] * y[c - i]; }
  memcpy(out, r, sizeof r);
}

/* leaf of the walk: all elements consumed, no kappa open; gm = graded multiplier collected from children and own pairs */
static void a_leaf(APiece *p, const ATen *T, const double *gm, int usedq) {
  cx out[2] = {0, 0};
  if (p->type == 0) { cx G0[4][4], W[4][4]; a_gamma(0, G0); out[0] = a_tr(T->m[0]) / 4; a_mul(G0, T->m[0], W); out[1] = a_tr(W) / 4; }
  else if (!usedq) {
    cx X[4][4][4]; memcpy(X, T->m, sizeof X);          /* the one open axis is mu */
    if (p->op == OPA_NULL) out[0] = 0;
    else if (p->op == OPA_L) out[0] = a_func_L(X);
    else if (p->op == OPA_U) out[0] = a_func_UV(X);
    else if (p->op == OPA_LMU) out[0] = a_func_L(X) - a_func_UV(X);
    else out[0] = a_func_R(X, NULL) / p->Rg - a_func_L(X);
  } else {
    int amu = at_find(T, AX_MU, -1), anu = at_find(T, AX_NU, -1);
    cx Y[4][4][4][4];
    for (int j = 0; j < 4; j++) for (int k = 0; k < 4; k++) memcpy(Y[j][k], T->m[((size_t)j << (2 * amu)) | ((size_t)k << (2 * anu))], sizeof(cx) * 16);
    out[0] = a_func_R(NULL, Y) / p->Rg;
  }
  for (int o = 0; o < 2; o++) for (int c = 0; c < ANG; c++) p->acc[o][c] += out[o] * gm[c];
}

static void a_walk(APiece *p, int ei, const ATen *T, const double *gm, int npairs, int nopen, int usedq) {
  if (ei == p->nel) { if (nopen == 0) a_leaf(p, T, gm, usedq); return; }
  int left = 0; for (int k = ei; k < p->nel; k++) if (p->el[k].kind == EL_LINE || p->el[k].kind == EL_INS) left++;
  if (nopen > left) return;                             /* the open kappa's can no longer all be paired */
  int kind = p->el[ei].kind;
  if (kind == EL_CHORDV || kind == EL_FREEV) {
    double g2[ANG]; memcpy(g2, gm, sizeof g2);
    if (p->el[ei].child >= 0) a_gmul(gm, p->cval[p->el[ei].child]->v[0], g2);       /* V-child: point vertex times its scalar */
    ATen t2;
    if (kind == EL_FREEV) t2 = at_open(T, AX_MU, 0, 1.0);
    else { int ax = at_find(T, AX_CHORD, p->el[ei].chord); t2 = ax < 0 ? at_open(T, AX_CHORD, p->el[ei].chord, 1.0) : at_close(T, ax, 1.0); }
    a_walk(p, ei + 1, &t2, g2, npairs, nopen, usedq); free(t2.m);
    return;
  }
  int s = p->el[ei].slot, ins = kind == EL_INS;
  const AVal *cv = ins ? p->cval[p->el[ei].child] : NULL;
  double gb[ANG]; if (ins) a_gmul(gm, cv->v[1], gb); else memcpy(gb, gm, sizeof gb);   /* multiplier of the momentum-dependent part */
  cx E[4][4], G0[4][4]; a_gamma(0, G0);
  /* (1) the part without kappa and q: line (A_t pslash + m); insertion a*1 and b*A_t pslash */
  for (int r = 0; r < 4; r++) for (int c = 0; c < 4; c++) E[r][c] = p->At[s] * G0[r][c] + ((!ins && r == c) ? 1.0 : 0.0);
  { ATen t2 = at_left(T, E); a_walk(p, ei + 1, &t2, gb, npairs, nopen, usedq); free(t2.m); }
  if (ins) { double ga[ANG]; a_gmul(gm, cv->v[0], ga); a_walk(p, ei + 1, T, ga, npairs, nopen, usedq); }
  /* (2) kappaslash: open a new index (total own grade is bounded by L-1, O6) ... */
  if (npairs + nopen + 1 <= p->Lglobal - 1) { ATen t2 = at_open(T, AX_KAPPA, s, 1.0); a_walk(p, ei + 1, &t2, gb, npairs, nopen + 1, usedq); free(t2.m); }
  /* ... or pair with an open kappa of slot u: (-1/2) beta_us g_{rho sigma}; one more own grade */
  for (int ax = 0; ax < T->nax; ax++) if (T->kind[ax] == AX_KAPPA) {
    ATen t2 = at_close(T, ax, -0.5 * p->beta[T->id[ax]][s]);
    double g2[ANG]; g2[0] = 0; for (int c = 1; c < ANG; c++) g2[c] = gb[c - 1];
    a_walk(p, ei + 1, &t2, g2, npairs + 1, nopen - 1, usedq); free(t2.m);
  }
  /* (3) the q-linear part A'_t qslash: once, only under operator A */
  if (p->op == OPA_A && !usedq) { ATen t2 = at_open(T, AX_NU, 0, p->Aq[s]); a_walk(p, ei + 1, &t2, gb, npairs, nopen, 1); free(t2.m); }
}

/* value of forest element H (index into segs, or -1 for G) of forest F under the term's G' = gp */
static void a_element(const AGraph *g, const ASeg *segs, int nseg, unsigned F, int H, int gp, const double *z, AVal *out) {
  ASeg me; if (H < 0) { me.lo = 0; me.hi = 2 * g->L; me.type = 1; } else me = segs[H];
  /* maximal elements of F strictly inside me */
  int kids[AMAXSEG], nk = 0;
  for (int i = 0; i < nseg; i++) {
    if (!(F >> i & 1) || i == H || !a_inside(&segs[i], &me)) continue;
    int maximal = 1;
    for (int j = 0; j < nseg; j++) if ((F >> j & 1) && j != i && j != H && a_inside(&segs[j], &me) && a_inside(&segs[i], &segs[j])) maximal = 0;
    if (maximal) kids[nk++] = i;
  }
  AVal kv[AMAXSEG];
  for (int k = 0; k < nk; k++) a_element(g, segs, nseg, F, kids[k], gp, z, &kv[k]);
  /* operator (O1) */
  APiece *p = (APiece *)calloc(1, sizeof(APiece));
  int inI = H < 0 || (me.type == 1 && me.lo <= g->e && g->e <= me.hi);
  if (H == gp) p->op = OPA_A;
  else if (!inI) p->op = OPA_U;
  else if (gp < 0) p->op = OPA_U;                                          /* G' = G: every proper element lies strictly inside G' */
  else if (H >= 0 && a_inside(&me, &segs[gp])) p->op = OPA_U;              /* strictly inside G' (H != G') */
  else p->op = H < 0 ? OPA_LMU : OPA_L;                                    /* G' strictly inside H */
  if (a_variant & 1) { if (p->op == OPA_L) p->op = OPA_U; }               /* negative controls of the IR pin (oracle_a_set_variant) */
  if ((a_variant & 2) && p->op == OPA_LMU) p->op = OPA_NULL;
  p->type = me.type; p->Lglobal = g->L; p->Rg = a_R_gamma(); p->nchild = nk;
  for (int k = 0; k < nk; k++) { p->cval[k] = &kv[k]; p->ctype[k] = segs[kids[k]].type; }
  /* geometry: own chords, path-ordered elements, momentum slots */
  int local[AL];
  for (int i = 0; i < g->L; i++) {
    local[i] = -1;
    if (g->a[i] < me.lo || g->b[i] > me.hi) continue;
    int same = 0; for (int k = 0; k < nk; k++) if (segs[kids[k]].lo <= g->a[i] && g->b[i] <= segs[kids[k]].hi) same = 1;
    if (!same) { local[i] = p->nch; p->chord[p->nch++] = i; }
  }
  int freepos = -1;
  if (me.type == 1) { if (me.lo <= g->e && g->e <= me.hi) freepos = g->e; else for (int x = me.lo; x <= me.hi; x++) if (g->other[x] < me.lo || g->other[x] > me.hi) freepos = x; }
  for (int pos = me.lo; pos <= me.hi;) {
    int c = -1; for (int k = 0; k < nk; k++) if (segs[kids[k]].lo <= pos && pos <= segs[kids[k]].hi) c = k;
    int n = p->nel++;
    p->el[n].child = c; p->el[n].slot = -1; p->el[n].chord = -1;
    if (c >= 0 && p->ctype[c] == 0) {                                    /* S-child: insertion; its momentum is that of the line before it */
      int s = p->nslot++; p->slot[s].ins = 1; p->slot[s].child = c; p->slot[s].line = segs[kids[c]].lo - 1;
      p->el[n].kind = EL_INS; p->el[n].slot = s; pos = segs[kids[c]].hi + 1;
    } else if (c >= 0) {                                                 /* V-child: one vertex */
      if (segs[kids[c]].lo <= freepos && freepos <= segs[kids[c]].hi) p->el[n].kind = EL_FREEV;
      else { p->el[n].kind = EL_CHORDV; for (int x = segs[kids[c]].lo; x <= segs[kids[c]].hi; x++) if (x != g->e && (g->other[x] < segs[kids[c]].lo || g->other[x] > segs[kids[c]].hi)) for (int i = 0; i < g->L; i++) if (g->a[i] == x || g->b[i] == x) p->el[n].chord = local[i]; }
      pos = segs[kids[c]].hi + 1;
    } else {
      if (pos == freepos) p->el[n].kind = EL_FREEV;
      else { p->el[n].kind = EL_CHORDV; for (int i = 0; i < g->L; i++) if (g->a[i] == pos || g->b[i] == pos) p->el[n].chord = local[i]; }
      pos++;
    }
    if (pos <= me.hi) { int s = p->nslot++; p->slot[s].ins = 0; p->slot[s].child = -1; p->slot[s].line = pos - 1; int m = p->nel++; p->el[m].kind = EL_LINE; p->el[m].slot = s; p->el[m].child = -1; p->el[m].chord = -1; }
  }
  for (int s = 0; s < p->nslot; s++) {
    int t = p->slot[s].line; p->slot[s].eps = 0; p->slot[s].sgn = t < g->e ? -1 : 1;
    for (int j = 0; j < p->nch; j++) if (g->a[p->chord[j]] <= t && t < g->b[p->chord[j]]) p->slot[s].eps |= 1u << j;
  }
  a_scalars(g, p, z);
  /* numerator: walk over all configurations */
  ATen T0 = at_new(0); memset(T0.m[0], 0, sizeof(cx) * 16); for (int i = 0; i < 4; i++) T0.m[0][i][i] = 1;
  double g0[ANG] = {1, 0, 0, 0, 0, 0};
  a_walk(p, 0, &T0, g0, 0, 0, 0); free(T0.m);
  double pref = 1; for (int i = 0; i < p->nch; i++) pref *= -0.25;
  memset(out, 0, sizeof *out);
  for (int o = 0; o < 2; o++) for (int c = 0; c < ANG; c++) out->v[o][c] = pref * creal(p->acc[o][c]);
  out->U = p->U; out->V = p->V;
  for (int k = 0; k < nk; k++) { out->U *= kv[k].U; out->V += kv[k].V; }
  free(p);
}

/* ================= exported ================= */
void oracle_a_set_variant(int v) { a_variant = v; }
typedef struct { int32_t loops, ext_pos, chord_a[5], chord_b[5]; } oracle_a_graph;

/* terms of the forest-like formula in canonical order (forests by ascending bitmask over the subgraphs sorted by (lo,hi);
 * within a forest G' = G first, then the V-type members containing e): forest[], gprime[] (-1 = G), sign[]; returns the count.
 * seg_lo/seg_hi/seg_type receive the subgraphs, *nseg their number. Any output may be NULL. */
int oracle_a_terms(const oracle_a_graph *og, int32_t *nseg_out, int32_t *seg_lo, int32_t *seg_hi, int32_t *seg_type, uint32_t *forest, int32_t *gprime, int32_t *sign) {
  AGraph g; int a[AL], b[AL];
  for (int i = 0; i < og->loops && i < AL; i++) { a[i] = og->chord_a[i]; b[i] = og->chord_b[i]; }
  if (a_graph(&g, og->loops, og->ext_pos, a, b)) return -1;
  ASeg segs[AMAXSEG]; int nseg = a_subgraphs(&g, segs), n = 0;
  if (nseg_out) *nseg_out = nseg;
  for (int i = 0; i < nseg; i++) { if (seg_lo) seg_lo[i] = segs[i].lo; if (seg_hi) seg_hi[i] = segs[i].hi; if (seg_type) seg_type[i] = segs[i].type; }
  for (unsigned F = 0; F < (1u << nseg); F++) {
    if (!a_is_forest(segs, nseg, F)) continue;
    int sg = (__builtin_popcount(F) & 1) ? -1 : 1;
    if (forest) forest[n] = F; if (gprime) gprime[n] = -1; if (sign) sign[n] = sg; n++;
    for (int i = 0; i < nseg; i++) if ((F >> i & 1) && segs[i].type == 1 && segs[i].lo <= g.e && g.e <= segs[i].hi) { if (forest) forest[n] = F; if (gprime) gprime[n] = i; if (sign) sign[n] = sg; n++; }
  }
  return n;
}

/* f(z) at n points (z: n x 3L by line index); terms_out (may be NULL): n x nterm signed term values in the order of oracle_a_terms */
int oracle_a_eval(const oracle_a_graph *og, uint64_t n, const double *z, double *f_out, double *terms_out) {
  AGraph g; int a[AL], b[AL];
  for (int i = 0; i < og->loops && i < AL; i++) { a[i] = og->chord_a[i]; b[i] = og->chord_b[i]; }
  if (a_graph(&g, og->loops, og->ext_pos, a, b)) return -1;
  ASeg segs[AMAXSEG]; int nseg = a_subgraphs(&g, segs);
  int nterm = oracle_a_terms(og, NULL, NULL, NULL, NULL, NULL, NULL, NULL);
  uint32_t *forest = (uint32_t *)malloc(sizeof(uint32_t) * nterm); int32_t *gprime = (int32_t *)malloc(4 * nterm), *sign = (int32_t *)malloc(4 * nterm);
  oracle_a_terms(og, NULL, NULL, NULL, NULL, forest, gprime, sign);
  const int L = g.L, M = 3 * L;
  static const double FACT[6] = {1, 1, 2, 6, 24, 120};
  double *tv = terms_out ? terms_out : (double *)malloc(sizeof(double) * n * nterm);
#pragma omp parallel for schedule(dynamic, 1) collapse(2)
  for (int64_t i = 0; i < (int64_t)n; i++) for (int t = 0; t < nterm; t++) {
    AVal v; a_element(&g, segs, nseg, forest[t], -1, gprime[t], z + (size_t)i * M, &v);
    double ft = 0, Vp = 1;
    for (int c = L - 1; c >= 0; c--) { Vp *= v.V; ft += sign[t] * FACT[L - c - 1] * v.v[0][c] / (v.U * v.U * Vp); }
    tv[(size_t)i * nterm + t] = ft;
  }
  if (f_out) for (uint64_t i = 0; i < n; i++) { double f = 0; for (int t = 0; t < nterm; t++) f += tv[i * nterm + t]; f_out[i] = f; }
  if (!terms_out) free(tv);
  free(forest); free(gprime); free(sign);
  return 0;
}
