/* oracle/qed_sampler.h — TEST INFRASTRUCTURE (CPU oracle).
 *
 * The non-adaptive Hepp-sector sampler of PAPER.md:69-78, Eq.(1):
 *     p(z) = C * prod_{l=2..M} (z_{j_l}/z_{j_{l-1}})^{Deg({j_l..j_M})} / (z_1 ... z_M)
 * on the sector z_{j_1} >= ... >= z_{j_M}; Deg(s) > 0 on proper non-empty subsets of lines
 * (PAPER.md:78). The paper does not print Deg ("quite complicated", two versions elsewhere);
 * DESIGN.md reading S5 is implemented here. Random stream: Philox4x32-10, the
 * public counter-based generator, written out by hand (S1), or MRG32k3a (S1b).
 *
 * Bit-exactness contract (S2-S4): every floating-point operation below is a single
 * IEEE-754 binary64 add/mul/div in the order written; compile with -ffp-contract=off.
 */
#ifndef QED_SAMPLER_H
#define QED_SAMPLER_H
#include "qed_piece.h"
#include <math.h>

/* ---------------- Philox4x32-10 ---------------- */
static void philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int r = 0; r < 10; r++) {
    uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0, hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}
/* uniform in (0,1), exact in binary64 (52 random bits): ((x>>6)*2^26 + (y>>6) + 0.5) * 2^-52 */
static double u01_from_words(uint32_t x, uint32_t y) {
  return ((double)(x >> 6) * 67108864.0 + (double)(y >> 6) + 0.5) * (1.0 / 4503599627370496.0);
}
/* uniform number r of sample idx of diagram diag_id: Philox block r/2, words (0,1) or (2,3) */
static double sample_uniform(uint64_t idx, uint32_t diag_id, uint64_t seed, int r) {
  uint32_t ctr[4] = {(uint32_t)idx, (uint32_t)(idx >> 32), (uint32_t)(r >> 1), diag_id};
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)}, w[4];
  philox4x32_10(ctr, key, w);
  return (r & 1) ? u01_from_words(w[2], w[3]) : u01_from_words(w[0], w[1]);
}

/* ---------------- MRG32k3a ("Calc 1"; P. L'Ecuyer, Operations Research 47 (1999) 159, Table III) ----------------
 * Two order-3 linear recurrences, m1 = 2^32 - 209, m2 = 2^32 - 22853:
 *     x1_n = (1403580 x1_{n-2} -  810728 x1_{n-3}) mod m1,     x2_n = (527612 x2_{n-1} - 1370589 x2_{n-3}) mod m2,
 * output number n: w_n = (x1_n - x2_n) mod m1. The state holds (x_{n-3}, x_{n-2}, x_{n-1}) of both components.
 * How the method uses it is a READING (S1b; the paper names the generator only): the initial state is
 * (1 + seed_lo mod (m-1), 1 + seed_hi mod (m-1), 12345) in both components (seed_lo = seed_hi = 12344 gives L'Ecuyer's
 * reference state, all 12345); sample idx (< 2^38) of diagram diag_id (< 2^20) owns the 64 outputs from position
 * (diag_id * 2^38 + idx) * 64 on, and uniform number r of the sample is made from outputs 2r and 2r+1 of those, with the same
 * 52-bit construction as for Philox. Positions are reached by plain skipping here: state_n = A^n state_0 with the 3x3 companion
 * matrices, A^n by square-and-multiply at every call (slow, obviously right).
 * Pins (tests/test_oracle_rng.py): the published jump matrices A^(2^76), A^(2^127) of both components (recurrences, moduli, matrix
 * power), stepping = skipping. The output combination (x1 - x2) mod m1 and the seeding have no published number at hand: for
 * them "parity unpinned" (restated with Python integers in the test only). */
#define MRG_M1 4294967087ull
#define MRG_M2 4294944443ull
typedef struct { uint64_t s1[3], s2[3]; } Mrg;
static uint64_t mrg_next(Mrg *g) {
  uint64_t x1 = ((1403580ull * g->s1[1]) % MRG_M1 + ((MRG_M1 - 810728ull) * g->s1[0]) % MRG_M1) % MRG_M1;
  uint64_t x2 = ((527612ull * g->s2[2]) % MRG_M2 + ((MRG_M2 - 1370589ull) * g->s2[0]) % MRG_M2) % MRG_M2;
  g->s1[0] = g->s1[1]; g->s1[1] = g->s1[2]; g->s1[2] = x1;
  g->s2[0] = g->s2[1]; g->s2[1] = g->s2[2]; g->s2[2] = x2;
  return (x1 + MRG_M1 - x2) % MRG_M1;
}
static void mrg_matmul(const uint64_t A[3][3], const uint64_t B[3][3], uint64_t m, uint64_t out[3][3]) {
  uint64_t T[3][3];
  for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) {
    uint64_t acc = 0;
    for (int k = 0; k < 3; k++) acc = (acc + (A[i][k] * B[k][j]) % m) % m;     /* entries < 2^32: the products fit 64 bits */
    T[i][j] = acc;
  }
  memcpy(out, T, sizeof T);
}
/* companion matrix of component comp (0, 1): (x_{n-3}, x_{n-2}, x_{n-1})^T -> (x_{n-2}, x_{n-1}, x_n)^T */
static void mrg_companion(int comp, uint64_t A[3][3]) {
  uint64_t A1[3][3] = {{0, 1, 0}, {0, 0, 1}, {MRG_M1 - 810728ull, 1403580ull, 0}};
  uint64_t A2[3][3] = {{0, 1, 0}, {0, 0, 1}, {MRG_M2 - 1370589ull, 0, 527612ull}};
  memcpy(A, comp ? A2 : A1, sizeof A1);
}
/* A^n mod m of component comp */
static void mrg_matpow(int comp, uint64_t n, uint64_t out[3][3]) {
  uint64_t m = comp ? MRG_M2 : MRG_M1, B[3][3], R[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}};
  mrg_companion(comp, B);
  for (; n; n >>= 1) { if (n & 1) mrg_matmul(B, R, m, R); mrg_matmul(B, B, m, B); }
  memcpy(out, R, sizeof R);
}
static void mrg_skip(Mrg *g, uint64_t n) {
  for (int comp = 0; comp < 2; comp++) {
    uint64_t P[3][3], m = comp ? MRG_M2 : MRG_M1, *s = comp ? g->s2 : g->s1, t[3];
    mrg_matpow(comp, n, P);
    for (int i = 0; i < 3; i++) { t[i] = 0; for (int k = 0; k < 3; k++) t[i] = (t[i] + (P[i][k] * s[k]) % m) % m; }
    for (int i = 0; i < 3; i++) s[i] = t[i];
  }
}
static Mrg mrg_seed(uint64_t seed) {
  uint64_t lo = (uint32_t)seed, hi = (uint32_t)(seed >> 32);
  Mrg g = {{1 + lo % (MRG_M1 - 1), 1 + hi % (MRG_M1 - 1), 12345}, {1 + lo % (MRG_M2 - 1), 1 + hi % (MRG_M2 - 1), 12345}};
  return g;
}
/* uniform number r of sample idx of diagram diag_id from the MRG32k3a stream */
static double sample_uniform_mrg(uint64_t idx, uint32_t diag_id, uint64_t seed, int r) {
  Mrg g = mrg_seed(seed);
  mrg_skip(&g, (((uint64_t)diag_id << 38) + idx) * 64 + 2 * (uint64_t)r);
  uint64_t a = mrg_next(&g), b = mrg_next(&g);
  return u01_from_words((uint32_t)a, (uint32_t)b);
}

/* ---------------- deterministic pow: t = u^(1/Deg) = det_exp2(det_log2(u)*invDeg) ---------------- */
static double det_log2(double u) {
  uint64_t bits; memcpy(&bits, &u, 8);
  int ex = (int)((bits >> 52) & 0x7FF) - 1023;
  bits = (bits & 0x000FFFFFFFFFFFFFull) | 0x3FF0000000000000ull;
  double m; memcpy(&m, &bits, 8);                 /* m in [1,2) */
  if (m > 1.4142135623730951) { m = m * 0.5; ex += 1; }
  double s = (m - 1.0) / (m + 1.0), s2 = s * s;
  /* ln m = 2 s (1 + s^2/3 + s^4/5 + ... + s^22/23), |s| <= 0.1716 */
  double P = 1.0 / 23.0;
  P = P * s2 + 1.0 / 21.0; P = P * s2 + 1.0 / 19.0; P = P * s2 + 1.0 / 17.0; P = P * s2 + 1.0 / 15.0;
  P = P * s2 + 1.0 / 13.0; P = P * s2 + 1.0 / 11.0; P = P * s2 + 1.0 / 9.0;  P = P * s2 + 1.0 / 7.0;
  P = P * s2 + 1.0 / 5.0;  P = P * s2 + 1.0 / 3.0;  P = P * s2 + 1.0;
  double lnm = (2.0 * s) * P;
  return (double)ex + lnm * 1.4426950408889634;   /* log2(e) */
}
static double det_exp2(double y) {
  if (y < -1020.0) return 0.0;
  double n = floor(y + 0.5), r = y - n, w = r * 0.6931471805599453; /* ln 2 */
  /* e^w, |w| <= 0.3466, Taylor to degree 14 */
  double P = 1.0 / 87178291200.0;
  P = P * w + 1.0 / 6227020800.0; P = P * w + 1.0 / 479001600.0; P = P * w + 1.0 / 39916800.0;
  P = P * w + 1.0 / 3628800.0;    P = P * w + 1.0 / 362880.0;    P = P * w + 1.0 / 40320.0;
  P = P * w + 1.0 / 5040.0;       P = P * w + 1.0 / 720.0;       P = P * w + 1.0 / 120.0;
  P = P * w + 1.0 / 24.0;         P = P * w + 1.0 / 6.0;         P = P * w + 0.5;
  P = P * w + 1.0;                P = P * w + 1.0;
  uint64_t bits = (uint64_t)((int64_t)n + 1023) << 52;
  double sc; memcpy(&sc, &bits, 8);
  return P * sc;
}
static double det_pow(double u, double inv_deg) { return det_exp2(det_log2(u) * inv_deg); }

/* ---------------- Deg(s) (S5) ---------------- */
/* I-closure: s plus every photon whose connecting electron path lies in s */
static unsigned i_closure(const Graph *g, unsigned s) {
  for (int i = 0; i < g->L; i++) {
    int all = 1;
    for (int t = g->a[i]; t < g->b[i]; t++) if (!(s >> t & 1)) all = 0;
    if (all) s |= 1u << (2 * g->L + i);
  }
  return s;
}
/* cycle rank of the line set s restricted to the piece graph of h (children contracted to points) */
static int piece_loops(const Graph *g, const Geom *h, unsigned s) {
  int parent[MAXPOS + MAXCHILD], touched[MAXPOS + MAXCHILD];
  int nn = MAXPOS + MAXCHILD;
  for (int i = 0; i < nn; i++) { parent[i] = i; touched[i] = 0; }
  int nedge = 0;
#define NODE(pos) (pos_child(h, (pos)) >= 0 ? MAXPOS + pos_child(h, (pos)) : (pos))
#define FIND(x, r) { r = (x); while (parent[r] != r) r = parent[r]; }
  for (int k = 0; k < h->nline + h->nch; k++) {
    int u, v, idx;
    if (k < h->nline) { int t = h->line[k]; idx = t; u = NODE(t); v = NODE(t + 1); }
    else { int i = h->chord[k - h->nline]; idx = 2 * g->L + i; u = NODE(g->a[i]); v = NODE(g->b[i]); }
    if (!(s >> idx & 1)) continue;
    nedge++; touched[u] = touched[v] = 1;
    int ru, rv; FIND(u, ru); FIND(v, rv);
    if (ru != rv) parent[ru] = rv;
  }
  int nv = 0, nc = 0;
  for (int i = 0; i < nn; i++) if (touched[i]) { nv++; if (parent[i] == i) nc++; }
#undef NODE
#undef FIND
  return nedge - nv + nc;
}

typedef struct {
  int M;
  double *deg;     /* 2^M, entries for proper non-empty masks */
  double *invdeg;  /* 1.0/deg */
  double *Z;       /* 2^M sector-sum table, Z[0]=1 */
  double C;        /* normalisation of Eq.(1) */
  int rng;         /* 0 = Philox4x32-10, 1 = MRG32k3a (oracle_set_generator) */
  /* defensive mixture (S5b, a READING: the paper has one density): with probability alpha the
   * point is drawn from the second Eq.(1) density `alt` (other Deg floors), and the density of the point is the mixture
   * (1 - alpha) p_this + alpha p_alt, so that a weight f/p is bounded by the better of the two channels. NULL = off. */
  const void *alt; double alpha;
} SamplerTab;

/* Deg(s) = clamp(|sbar| - |e(sbar)|/2 - 2 max_F sum_H loops_H(sbar∩H), floor, cap); sbar=full -> floor_ir: the sets whose I-closure
 * is the whole graph are the soft-photon sets; the infrared pin (tests/test_oracle_a.py) measures one power of the
 * scale over a nested PAIR of such limits, so their exponent must stay near 1/2 while the UV-type sets can take 1 (S5) */
static void build_deg(const Graph *g, const Sub *subs, int nsub, const uint32_t *forests, int nforest,
                      double dfloor, double dcap, double dfloor_ir, SamplerTab *tab) {
  int M = g->M; unsigned full = (1u << M) - 1;
  tab->M = M;
  tab->deg = (double *)calloc((size_t)1 << M, sizeof(double));
  tab->invdeg = (double *)calloc((size_t)1 << M, sizeof(double));
  tab->Z = (double *)calloc((size_t)1 << M, sizeof(double));
  /* pieces of every forest (+G) */
  int npieces_tot = 0;
  Geom *pieces = (Geom *)malloc(sizeof(Geom) * (size_t)nforest * (MAXSUB + 1));
  int *first = (int *)malloc(sizeof(int) * (nforest + 1));
  for (int f = 0; f < nforest; f++) {
    first[f] = npieces_tot;
    Sub ch[MAXSUB];
    int nc = forest_children(subs, nsub, forests[f], 0, 2 * g->L, ch, NULL);
    /* G = [0,2L] itself is never in subs, so "strictly inside" excludes nothing wrongly */
    geom_build(g, 0, 2 * g->L, 1, nc, ch, &pieces[npieces_tot++]);
    for (int i = 0; i < nsub; i++) if (forests[f] >> i & 1) {
      nc = forest_children(subs, nsub, forests[f], subs[i].lo, subs[i].hi, ch, NULL);
      geom_build(g, subs[i].lo, subs[i].hi, subs[i].type, nc, ch, &pieces[npieces_tot++]);
    }
  }
  first[nforest] = npieces_tot;
  unsigned emask = (1u << (2 * g->L)) - 1;
  for (unsigned s = 1; s < full; s++) {
    unsigned sb = i_closure(g, s);
    double d;
    if (sb == full) d = dfloor_ir;
    else {
      int best = 0;
      for (int f = 0; f < nforest; f++) {
        int tot = 0;
        for (int k = first[f]; k < first[f + 1]; k++) tot += piece_loops(g, &pieces[k], sb);
        if (tot > best) best = tot;
      }
      d = (double)__builtin_popcount(sb) - 0.5 * (double)__builtin_popcount(sb & emask) - 2.0 * (double)best;
      if (d < dfloor) d = dfloor;
      if (d > dcap) d = dcap;
    }
    tab->deg[s] = d; tab->invdeg[s] = 1.0 / d;
  }
  free(pieces); free(first);
  /* sector sums (S2): ascending masks, inner sum ascending line index, one multiply by invdeg */
  tab->Z[0] = 1.0;
  for (unsigned s = 1; s < full; s++) {
    double acc = 0.0;
    for (int x = 0; x < M; x++) if (s >> x & 1) acc = acc + tab->Z[s & ~(1u << x)];
    tab->Z[s] = acc * tab->invdeg[s];
  }
  double tot = 0.0;
  for (int x = 0; x < M; x++) tot = tot + tab->Z[full & ~(1u << x)];
  tab->Z[full] = tot;
  tab->C = 1.0 / tot;
}
static void free_samplertab(SamplerTab *t) { free(t->deg); free(t->invdeg); free(t->Z); }

/* ---------------- one sample point (S3) ---------------- */
/* out: z[M] (by line index), order[M] (j_1..j_M), returns p(z) */
static double draw_point(const SamplerTab *tab0, uint64_t idx, uint32_t diag_id, uint64_t seed, double *z, int *order) {
  int M = tab0->M; unsigned mask = (1u << M) - 1;
  double r[MAXM], rl = 1.0, pu = 1.0, pq = 1.0;
  /* mixture: uniform number 2(M-1) of the sample picks the channel; `tab` draws the point, `oth` only contributes its density */
  const SamplerTab *tab = tab0, *oth = NULL;
  if (tab0->alt) {
    double uc = tab0->rng ? sample_uniform_mrg(idx, diag_id, seed, 2 * (M - 1)) : sample_uniform(idx, diag_id, seed, 2 * (M - 1));
    if (uc < tab0->alpha) { tab = (const SamplerTab *)tab0->alt; oth = tab0; } else oth = (const SamplerTab *)tab0->alt;
  }
  for (int l = 0; l < M; l++) {
    int x = -1;
    if (l == M - 1) { x = __builtin_ctz(mask); }
    else {
      double u = tab0->rng ? sample_uniform_mrg(idx, diag_id, seed, l) : sample_uniform(idx, diag_id, seed, l);
      double total = 0.0;
      for (int y = 0; y < M; y++) if (mask >> y & 1) total = total + tab->Z[mask & ~(1u << y)];
      double target = u * total, cum = 0.0;
      int last = -1;
      for (int y = 0; y < M; y++) if (mask >> y & 1) {
        cum = cum + tab->Z[mask & ~(1u << y)]; last = y;
        if (target < cum) { x = y; break; }
      }
      if (x < 0) x = last;
    }
    if (l >= 1) {
      double u = tab0->rng ? sample_uniform_mrg(idx, diag_id, seed, (M - 1) + (l - 1)) : sample_uniform(idx, diag_id, seed, (M - 1) + (l - 1));
      double lg = det_log2(u) * tab->invdeg[mask];   /* mask = S_l before removing x; t = u^(1/Deg) = det_pow(u, invdeg) */
      double t = det_exp2(lg);
      rl = rl * t; pu = pu * u;
      if (oth) pq = pq * det_exp2(lg * oth->deg[mask]);   /* t^Deg_other: the other channel's factor of Eq.(1) at this point */
    }
    r[l] = rl; order[l] = x;
    mask &= ~(1u << x);
  }
  double S = 0.0;
  for (int l = 0; l < M; l++) S = S + r[l];
  double pz = 1.0;
  for (int l = 0; l < M; l++) { double zz = r[l] / S; z[order[l]] = zz; pz = pz * zz; }
  double p_drawn = (tab->C * pu) / pz;
  if (!oth) return p_drawn;
  double p_other = (oth->C * pq) / pz;
  double p_main = tab == tab0 ? p_drawn : p_other, p_alt = tab == tab0 ? p_other : p_drawn;
  return (1.0 - tab0->alpha) * p_main + tab0->alpha * p_alt;
}

/* density of a given point (S6; tests only): sort descending, ties lower index first */
static double density_at(const SamplerTab *tab, const double *z) {
  int M = tab->M, ord[MAXM];
  for (int i = 0; i < M; i++) ord[i] = i;
  for (int i = 1; i < M; i++) for (int j = i; j > 0 && z[ord[j - 1]] < z[ord[j]]; j--) { int t = ord[j]; ord[j] = ord[j - 1]; ord[j - 1] = t; }
  unsigned mask = (1u << M) - 1;
  double lp = log(tab->C);
  for (int l = 0; l < M; l++) {
    if (l >= 1) lp += tab->deg[mask] * log(z[ord[l]] / z[ord[l - 1]]);
    lp -= log(z[ord[l]]);
    mask &= ~(1u << ord[l]);
  }
  return exp(lp);
}
/* density the points are drawn with: Eq.(1), or the mixture of the two Eq.(1) densities */
static double density_mix_at(const SamplerTab *tab, const double *z) {
  if (!tab->alt) return density_at(tab, z);
  return (1.0 - tab->alpha) * density_at(tab, z) + tab->alpha * density_at((const SamplerTab *)tab->alt, z);
}
#endif
