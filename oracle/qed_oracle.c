/* oracle/qed_oracle.c — TEST INFRASTRUCTURE: the CPU oracle for the CUDA path in
 * paper_1905_08007_b200/. Plain, slow, written from the paper (arXiv:1905.08007, PAPER.md) and
 * the readings listed in DESIGN.md. It shares no code with the CUDA path and is only to be
 * used by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs.
 *
 * What it computes: for one Feynman graph without lepton loops,
 *   (i)  sample points z on the simplex from the Hepp-sector density Eq.(1)   [qed_sampler.h]
 *   (ii) the subtracted Feynman-parametric integrand f(z) = sum over the forest-like formula
 *        of products of operators A, U, L applied to UV-divergent subgraphs     [qed_tables.h, qed_eval_impl.h]
 *   (iii) the Monte Carlo sums of w=f/p and w^2.
 * Pins: see tests/test_oracle_*.py (A1^(2)=1/2 pointwise and integrated, the 2-loop value
 * -0.344166, diagram counts 3213 and Table 1 N_diag, Dirichlet closed forms, Philox known
 * answers, projector identities) and tests/test_oracle_a.py: every term of every 1-, 2- and 3-loop
 * graph (and of some 4-loop graphs) against Oracle-A (qed_oracle_a.c: the definition evaluated per
 * point with explicit matrices, pairings and traces, its own forests and operator assignment), the
 * infrared pin that tells the operator L from U, hand-written term lists, the oracle-only 3-loop sum.
 * Parity status: L=1,2 pinned by the paper's values; L=3 pinned by Oracle-A, the infrared/UV scaling
 * pins and (softly) the literature value; the branches that first appear at L>=3 (L on intermediate
 * elements of I[G], nested forests, several S-children) are covered by those pins: swapping OP_L for
 * OP_U in op_of() fails four CPU tests. L=4,5 VALUES are "parity unpinned" by the paper (no per-graph
 * numbers are printed) — structural pins and Oracle-A at 4 loops apply.
 */
#include "qed_combi.h"
#include "qed_piece.h"
#include "qed_sampler.h"
#include "qed_tables.h"
#ifdef _OPENMP
#include <omp.h>
#endif

#define NGRADE 6
#define MAXGEOM 512
#define MAXNODE 1024

typedef struct { Geom h; int sub; uint32_t childmask; PieceTable *tab[4]; } GeomEntry;
typedef struct { int geom, op, nchild, child[MAXCHILD]; } Node;
typedef struct { int root, sign, gprime; uint32_t forest; } TermEntry;

struct oracle_diagram {
  Graph g; int id;
  int nsub; Sub subs[MAXSUB];
  int nforest; uint32_t forests[MAXFOREST];
  int nterm; TermEntry terms[MAXTERM];
  int ngeom; GeomEntry *geoms;
  int nnode; Node *nodes;
  SamplerTab stab;
  int have_tables;
  long n_monomials;
};
typedef struct oracle_diagram oracle_diagram;

#define REAL double
#define FN(x) x##_d
#include "qed_eval_impl.h"
#undef REAL
#undef FN
#define REAL __float128
#define FN(x) x##_q
#include "qed_eval_impl.h"
#undef REAL
#undef FN

/* ---------- term trees ---------- */
static int op_of(const oracle_diagram *d, int H /* sub index or -1 */, int gprime) {
  const Graph *g = &d->g;
  if (H == gprime) return OP_A;
  int inI = (H < 0) || (d->subs[H].type == 1 && d->subs[H].lo <= g->e && g->e <= d->subs[H].hi);
  int inside_gp = 0; /* H strictly inside G' */
  if (H >= 0) {
    if (gprime < 0) inside_gp = 1;
    else inside_gp = (d->subs[gprime].lo <= d->subs[H].lo && d->subs[H].hi <= d->subs[gprime].hi && H != gprime);
  }
  if (!inI || inside_gp) return OP_U;
  if (H < 0) return OP_LMU; /* H = G, G' != G */
  return OP_L;
}
static int get_geom(oracle_diagram *d, int H, uint32_t F) {
  int lo = H < 0 ? 0 : d->subs[H].lo, hi = H < 0 ? 2 * d->g.L : d->subs[H].hi, type = H < 0 ? 1 : d->subs[H].type;
  Sub ch[MAXSUB]; int idx[MAXSUB];
  int nc = forest_children(d->subs, d->nsub, F, lo, hi, ch, idx);
  uint32_t cm = 0; for (int c = 0; c < nc; c++) cm |= 1u << idx[c];
  for (int k = 0; k < d->ngeom; k++) if (d->geoms[k].sub == H && d->geoms[k].childmask == cm) return k;
  GeomEntry *ge = &d->geoms[d->ngeom];
  memset(ge, 0, sizeof *ge);
  ge->sub = H; ge->childmask = cm;
  geom_build(&d->g, lo, hi, type, nc, ch, &ge->h);
  return d->ngeom++;
}
static int build_node(oracle_diagram *d, int H, uint32_t F, int gprime) {
  Node nd; memset(&nd, 0, sizeof nd);
  nd.geom = get_geom(d, H, F); nd.op = op_of(d, H, gprime);
  int lo = H < 0 ? 0 : d->subs[H].lo, hi = H < 0 ? 2 * d->g.L : d->subs[H].hi;
  Sub ch[MAXSUB]; int idx[MAXSUB];
  nd.nchild = forest_children(d->subs, d->nsub, F, lo, hi, ch, idx);
  for (int c = 0; c < nd.nchild; c++) nd.child[c] = build_node(d, idx[c], F, gprime);
  for (int k = 0; k < d->nnode; k++) {
    const Node *o = &d->nodes[k];
    if (o->geom == nd.geom && o->op == nd.op && o->nchild == nd.nchild && memcmp(o->child, nd.child, sizeof(int) * nd.nchild) == 0) return k;
  }
  d->nodes[d->nnode] = nd;
  return d->nnode++;
}

/* ================= exported API (host pointers only) ================= */
typedef struct { int32_t loops, ext_pos, chord_a[5], chord_b[5]; } oracle_graph;

int oracle_graph_count(int L) { return (L < 1 || L > MAXL) ? -1 : graph_count(L); }
int oracle_graph_get(int L, int idx, oracle_graph *out) {
  Graph g; if (L < 1 || L > MAXL || graph_by_index(L, idx, &g) != 0) return -1;
  memset(out, 0, sizeof *out); out->loops = L; out->ext_pos = g.e;
  for (int i = 0; i < L; i++) { out->chord_a[i] = g.a[i]; out->chord_b[i] = g.b[i]; }
  return 0;
}
/* all valid graphs of order L in canonical order; out must hold oracle_graph_count(L) entries */
int oracle_graph_list(int L, oracle_graph *out) {
  if (L < 1 || L > MAXL) return -1;
  int n = graph_count(L);
  int *le = (int *)malloc(sizeof(int) * n), *la = (int *)malloc(sizeof(int) * n * MAXL), *lb = (int *)malloc(sizeof(int) * n * MAXL);
  EnumCtx c; memset(&c, 0, sizeof c); c.want_idx = -1; c.target_e = -1; c.list_e = le; c.list_a = la; c.list_b = lb;
  enum_run(&c, L);
  for (int i = 0; i < n; i++) { memset(&out[i], 0, sizeof out[i]); out[i].loops = L; out[i].ext_pos = le[i]; for (int k = 0; k < L; k++) { out[i].chord_a[k] = la[i * MAXL + k]; out[i].chord_b[k] = lb[i * MAXL + k]; } }
  free(le); free(la); free(lb);
  return n;
}
static int to_graph(const oracle_graph *og, Graph *g) {
  int a[MAXL], b[MAXL];
  if (og->loops < 1 || og->loops > MAXL) return -1;
  for (int i = 0; i < og->loops; i++) { a[i] = og->chord_a[i]; b[i] = og->chord_b[i]; }
  return graph_init(g, og->loops, og->ext_pos, a, b);
}
int oracle_graph_validate(const oracle_graph *og) { Graph g; return to_graph(og, &g); }
int oracle_graph_id(const oracle_graph *og) { Graph g; if (to_graph(og, &g)) return -1; return graph_canonical_id(&g); }
int oracle_graph_class(const oracle_graph *og, int *k, int *m, int *n) { Graph g; if (to_graph(og, &g)) return -1; graph_class(&g, k, m, n); return 0; }
int oracle_graph_mirror(const oracle_graph *og, oracle_graph *out) {
  Graph g, r; if (to_graph(og, &g) || graph_mirror(&g, &r)) return -1;
  memset(out, 0, sizeof *out); out->loops = r.L; out->ext_pos = r.e;
  for (int i = 0; i < r.L; i++) { out->chord_a[i] = r.a[i]; out->chord_b[i] = r.b[i]; }
  return 0;
}

/* level 0: combinatorics + sampler tables; level 1: + integrand tables. max_grade_prune: 1 = skip the
 * top own grade of pieces under A and (L-U) (it vanishes identically, O4), 0 = compute it */
int oracle_prepare_diagram(const oracle_graph *og, double deg_floor, double deg_cap, double deg_floor_ir, int level, int prune, oracle_diagram **out) {
  oracle_diagram *d = (oracle_diagram *)calloc(1, sizeof *d);
  if (to_graph(og, &d->g)) { free(d); return -1; }
  d->id = graph_canonical_id(&d->g);
  d->nsub = enum_subgraphs(&d->g, d->subs);
  d->nforest = enum_forests(d->subs, d->nsub, d->forests);
  Term terms[MAXTERM];
  d->nterm = enum_terms(&d->g, d->subs, d->nsub, d->forests, d->nforest, terms);
  build_deg(&d->g, d->subs, d->nsub, d->forests, d->nforest, deg_floor, deg_cap, deg_floor_ir > 0 ? deg_floor_ir : deg_floor, &d->stab);
  d->geoms = (GeomEntry *)calloc(MAXGEOM, sizeof(GeomEntry));
  d->nodes = (Node *)calloc(MAXNODE, sizeof(Node));
  for (int t = 0; t < d->nterm; t++) {
    d->terms[t].forest = terms[t].forest; d->terms[t].gprime = terms[t].gprime; d->terms[t].sign = terms[t].sign;
    d->terms[t].root = build_node(d, -1, terms[t].forest, terms[t].gprime);
  }
  if (level >= 1) {
    /* which (geom, op) tables are needed */
    int need[MAXGEOM][4]; memset(need, 0, sizeof need);
    for (int k = 0; k < d->nnode; k++) need[d->nodes[k].geom][d->nodes[k].op] = 1;
    int jobs[MAXGEOM * 4][2], njob = 0;
    for (int k = 0; k < d->ngeom; k++) for (int op = 0; op < 4; op++) if (need[k][op]) { jobs[njob][0] = k; jobs[njob][1] = op; njob++; }
    for (int j = 0; j < njob; j++) {   /* each table build is parallel inside (qed_tables.h) */
      int k = jobs[j][0], op = jobs[j][1];
      PieceTable *t = (PieceTable *)calloc(1, sizeof(PieceTable));
      int mg = -1;
      int has_ins = 0;
      for (int c = 0; c < d->geoms[k].h.nchild; c++) if (d->geoms[k].h.child_type[c] == 0) has_ins = 1;
      if (prune && !has_ins && (op == OP_A || op == OP_LMU)) mg = d->geoms[k].h.nch - 1;
      build_piece_table(&d->geoms[k].h, op, mg, t);
      d->geoms[k].tab[op] = t;
    }
    for (int j = 0; j < njob; j++) d->n_monomials += d->geoms[jobs[j][0]].tab[jobs[j][1]]->n;
    d->have_tables = 1;
  }
  *out = d;
  return 0;
}
void oracle_free_diagram(oracle_diagram *d) {
  if (!d) return;
  for (int k = 0; k < d->ngeom; k++) for (int op = 0; op < 4; op++) if (d->geoms[k].tab[op]) { free(d->geoms[k].tab[op]->mono); free(d->geoms[k].tab[op]); }
  if (d->stab.alt) { free_samplertab((SamplerTab *)d->stab.alt); free((void *)d->stab.alt); }
  free(d->geoms); free(d->nodes); free_samplertab(&d->stab); free(d);
}
/* info[0..7] = id, M, nsub, nforest, nterm, ngeom, nnode, n_monomials */
int oracle_diagram_info(const oracle_diagram *d, int64_t *info) {
  info[0] = d->id; info[1] = d->g.M; info[2] = d->nsub; info[3] = d->nforest; info[4] = d->nterm; info[5] = d->ngeom; info[6] = d->nnode; info[7] = d->n_monomials;
  return 0;
}
int oracle_get_subgraphs(const oracle_diagram *d, int32_t *lo, int32_t *hi, int32_t *type) {
  for (int i = 0; i < d->nsub; i++) { lo[i] = d->subs[i].lo; hi[i] = d->subs[i].hi; type[i] = d->subs[i].type; }
  return d->nsub;
}
int oracle_get_forests(const oracle_diagram *d, uint32_t *f) { for (int i = 0; i < d->nforest; i++) f[i] = d->forests[i]; return d->nforest; }
int oracle_get_terms(const oracle_diagram *d, uint32_t *forest, int32_t *gprime, int32_t *sign) {
  for (int i = 0; i < d->nterm; i++) { forest[i] = d->terms[i].forest; gprime[i] = d->terms[i].gprime; sign[i] = d->terms[i].sign; }
  return d->nterm;
}
int oracle_get_sampler_tables(const oracle_diagram *d, double *deg, double *Z, double *C) {
  size_t n = (size_t)1 << d->g.M;
  if (deg) memcpy(deg, d->stab.deg, n * sizeof(double));
  if (Z) memcpy(Z, d->stab.Z, n * sizeof(double));
  if (C) *C = d->stab.C;
  return 0;
}
/* sample points first..first+n-1: z[n*M] by line index, p[n], order[n*M] (the Hepp sector j_1..j_M) */
int oracle_sample_points(const oracle_diagram *d, uint64_t first, uint64_t n, uint64_t seed, double *z, double *p, int32_t *order) {
  int M = d->g.M;
#pragma omp parallel for schedule(static)
  for (int64_t i = 0; i < (int64_t)n; i++) {
    int ord[MAXM];
    p[i] = draw_point(&d->stab, first + (uint64_t)i, (uint32_t)d->id, seed, z + (size_t)i * M, ord);
    if (order) for (int l = 0; l < M; l++) order[(size_t)i * M + l] = ord[l];
  }
  return 0;
}
int oracle_density(const oracle_diagram *d, uint64_t n, const double *z, double *p) {
  for (uint64_t i = 0; i < n; i++) p[i] = density_mix_at(&d->stab, z + i * d->g.M);
  return 0;
}
/* integrand at given points. f64 / fwide (the wide value rounded to double) / abs64 (round-off scale) /
 * terms64 (n*nterm) may each be NULL */
int oracle_eval_z(const oracle_diagram *d, uint64_t n, const double *z, double *f64, double *fwide, double *abs64, double *terms64) {
  if (!d->have_tables) return -2;
  int M = d->g.M;
#pragma omp parallel for schedule(dynamic, 16)
  for (int64_t i = 0; i < (int64_t)n; i++) {
    if (f64 || abs64 || terms64) {
      double a, f = eval_integrand_d(d, z + (size_t)i * M, terms64 ? terms64 + (size_t)i * d->nterm : NULL, &a);
      if (f64) f64[i] = f;
      if (abs64) abs64[i] = a;
    }
    if (fwide) {
      __float128 zq[MAXM]; for (int k = 0; k < M; k++) zq[k] = z[(size_t)i * M + k];
      fwide[i] = (double)eval_integrand_q(d, zq, NULL, NULL);
    }
  }
  return 0;
}
/* Monte Carlo sums over sample indices first..first+n-1 (O7). mode 0: binary64 values;
 * mode 1: wide values; mode 2: binary64 unless the truth flag |f64-fwide|>1e-10|fwide| is set, then wide.
 * sums are accumulated in __float128 so that the oracle's own summation error is irrelevant. */
int oracle_integrate(const oracle_diagram *d, uint64_t first, uint64_t n, uint64_t seed, int mode, double *sum, double *sumsq, uint64_t *nflag) {
  if (!d->have_tables) return -2;
  int M = d->g.M;
  __float128 S1 = 0, S2 = 0; uint64_t NF = 0;
#pragma omp parallel
  {
    __float128 s1 = 0, s2 = 0; uint64_t nf = 0;
#pragma omp for schedule(dynamic, 256)
    for (int64_t i = 0; i < (int64_t)n; i++) {
      double z[MAXM]; int ord[MAXM];
      double p = draw_point(&d->stab, first + (uint64_t)i, (uint32_t)d->id, seed, z, ord);
      double f;
      if (mode == 0) f = eval_integrand_d(d, z, NULL, NULL);
      else {
        __float128 zq[MAXM]; for (int k = 0; k < M; k++) zq[k] = z[k];
        double fw = (double)eval_integrand_q(d, zq, NULL, NULL);
        if (mode == 1) f = fw;
        else { double fd = eval_integrand_d(d, z, NULL, NULL); if (fabs(fd - fw) > 1e-10 * fabs(fw)) { f = fw; nf++; } else f = fd; }
      }
      double w = f / p;
      s1 += w; s2 += (__float128)w * w;
    }
#pragma omp critical
    { S1 += s1; S2 += s2; NF += nf; }
  }
  *sum = (double)S1; *sumsq = (double)S2; if (nflag) *nflag = NF;
  return 0;
}
int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ---- small hooks for the pins ---- */
void oracle_philox(const uint32_t *ctr, const uint32_t *key, uint32_t *out) { philox4x32_10(ctr, key, out); }
double oracle_u01(uint32_t x, uint32_t y) { return u01_from_words(x, y); }
double oracle_sample_uniform(uint64_t idx, uint32_t diag, uint64_t seed, int r) { return sample_uniform(idx, diag, seed, r); }
double oracle_sample_uniform_mrg(uint64_t idx, uint32_t diag, uint64_t seed, int r) { return sample_uniform_mrg(idx, diag, seed, r); }
/* raw MRG32k3a: state6 = (x1_{n-3}, x1_{n-2}, x1_{n-1}, x2_{n-3}, x2_{n-2}, x2_{n-1}); skips `skip` outputs, then writes nout outputs w_n */
void oracle_mrg32k3a(const uint64_t *state6, uint64_t skip, int nout, uint64_t *out) {
  Mrg g; for (int i = 0; i < 3; i++) { g.s1[i] = state6[i]; g.s2[i] = state6[3 + i]; }
  mrg_skip(&g, skip);
  for (int i = 0; i < nout; i++) out[i] = mrg_next(&g);
}
/* A^(2^e * mult) mod m of component comp (0, 1), row-major into out9 */
void oracle_mrg_matpow(int comp, int e, uint64_t mult, uint64_t *out9) {
  uint64_t P[3][3], m = comp ? MRG_M2 : MRG_M1; mrg_matpow(comp, mult, P);
  for (int i = 0; i < e; i++) mrg_matmul(P, P, m, P);
  for (int i = 0; i < 9; i++) out9[i] = P[i / 3][i % 3];
}
/* defensive mixture (S5b): with probability alpha a point is drawn from a second Eq.(1) density with the Deg floors
 * (deg_floor2, deg_floor_ir2) and the same cap; alpha = 0 switches it off */
int oracle_set_mixture(oracle_diagram *d, double alpha, double deg_floor2, double deg_cap2, double deg_floor_ir2) {
  if (!(alpha >= 0.0 && alpha < 1.0)) return -1;
  if (d->stab.alt) { free_samplertab((SamplerTab *)d->stab.alt); free((void *)d->stab.alt); d->stab.alt = NULL; }
  d->stab.alpha = 0.0;
  if (alpha == 0.0) return 0;
  if (!(deg_floor2 > 0.0 && deg_cap2 >= deg_floor2)) return -1;
  SamplerTab *t = (SamplerTab *)calloc(1, sizeof *t);
  build_deg(&d->g, d->subs, d->nsub, d->forests, d->nforest, deg_floor2, deg_cap2, deg_floor_ir2 > 0 ? deg_floor_ir2 : deg_floor2, t);
  d->stab.alt = t; d->stab.alpha = alpha;
  return 0;
}
/* generator of the sampler of an existing diagram: 0 = Philox4x32-10 (default), 1 = MRG32k3a */
int oracle_set_generator(oracle_diagram *d, int kind) { if (kind < 0 || kind > 1) return -1; d->stab.rng = kind; return 0; }
double oracle_det_pow(double u, double inv_deg) { return det_pow(u, inv_deg); }
double oracle_det_log2(double u) { return det_log2(u); }
double oracle_det_exp2(double y) { return det_exp2(y); }
/* operator functionals applied to user-supplied X[4][4][4] (re,im interleaved) and Y[4][4][4][4]: out = {L, U_V, A} */
int oracle_functionals(const double *Xri, const double *Yri, double *out_ri) {
  cplx X[4][4][4], Y[4][4][4][4];
  for (int i = 0; i < 64; i++) ((cplx *)X)[i] = Xri[2 * i] + I * Xri[2 * i + 1];
  for (int i = 0; i < 256; i++) ((cplx *)Y)[i] = Yri ? Yri[2 * i] + I * Yri[2 * i + 1] : 0;
  cplx l = func_L(X), u = func_UV(X), a = (func_R_X(X) + func_R_Y(Y)) / R_gamma() - l;
  out_ri[0] = creal(l); out_ri[1] = cimag(l); out_ri[2] = creal(u); out_ri[3] = cimag(u); out_ri[4] = creal(a); out_ri[5] = cimag(a);
  return 0;
}
int oracle_dense_gamma(int mu, double *ri) { cplx G[4][4]; dense_gamma(mu, G); for (int i = 0; i < 16; i++) { ri[2 * i] = creal(((cplx *)G)[i]); ri[2 * i + 1] = cimag(((cplx *)G)[i]); } return 0; }
/* graded value(s) of one node (by term root or node index) at a point, binary64: out[2*NGRADE], plus U product and V sum */
int oracle_node_value(const oracle_diagram *d, int node, const double *z, double *out, double *UV) {
  if (!d->have_tables || node < 0 || node >= d->nnode) return -2;
  GeomVal_d *gvs = (GeomVal_d *)calloc(d->ngeom, sizeof(GeomVal_d));
  NodeVal_d *nvs = (NodeVal_d *)calloc(d->nnode, sizeof(NodeVal_d));
  eval_node_d(d, node, z, gvs, nvs);
  for (int o = 0; o < 2; o++) for (int c = 0; c < NGRADE; c++) out[o * NGRADE + c] = nvs[node].v[o][c];
  UV[0] = nvs[node].Uprod; UV[1] = nvs[node].Vsum;
  free(gvs); free(nvs);
  return 0;
}
/* node table: for node k -> geom sub index (-1 = G), op, children */
int oracle_get_nodes(const oracle_diagram *d, int32_t *sub, int32_t *op, int32_t *nchild, int32_t *children /* MAXCHILD each */) {
  for (int k = 0; k < d->nnode; k++) { sub[k] = d->geoms[d->nodes[k].geom].sub; op[k] = d->nodes[k].op; nchild[k] = d->nodes[k].nchild; for (int c = 0; c < MAXCHILD; c++) children[k * MAXCHILD + c] = c < d->nodes[k].nchild ? d->nodes[k].child[c] : -1; }
  return d->nnode;
}
int oracle_get_term_roots(const oracle_diagram *d, int32_t *root) { for (int t = 0; t < d->nterm; t++) root[t] = d->terms[t].root; return d->nterm; }
