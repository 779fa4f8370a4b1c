/* oracle/qed_eval_impl.h — TEST INFRASTRUCTURE (CPU oracle).
 * Per-point evaluation of the subtracted integrand, generic in the real type.
 * Include with REAL (double or __float128) and FN(name) (name mangling) defined.
 *
 * DESIGN.md O2 (scalars of a piece), O5 (piece value), O6 (term and integrand value):
 *   A    = sum_{own lines t} z_t eps_t eps_t^T + diag(z_gamma)
 *   U    = det A,  beta_tu = eps_t^T A^-1 eps_u
 *   x_t  = sum_{own lines u} z_u beta_tu            ( = 1 - A_t )
 *   A'_t = 1/2 [ s_t - sum_{own lines u} z_u beta_tu s_u ]
 *   V    = sum_{own lines u} z_u x_u                (m = 1)
 *   f    = sum_terms sign * sum_{c<L} (L-c-1)! N_c / ( (prod_H U_H)^2 (sum_H V_H)^(L-c) )
 */

typedef struct { REAL U, V, beta[MAXSLOT][MAXSLOT], x[MAXSLOT], aq[MAXSLOT]; int done; } FN(GeomVal);
typedef struct { REAL v[2][NGRADE], Uprod, Vsum; int done; } FN(NodeVal);

static void FN(eval_geom)(const Graph *g, const Geom *h, const REAL *z, FN(GeomVal) *gv) {
  int n = h->nch;
  REAL A[MAXL][MAXL], Inv[MAXL][MAXL];
  for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) { A[i][j] = 0; Inv[i][j] = (i == j) ? 1 : 0; }
  for (int s = 0; s < h->nslot; s++) if (h->slot[s].kind == SLOT_LINE) {
    unsigned e = h->slot[s].eps; REAL zt = z[h->slot[s].line];
    for (int i = 0; i < n; i++) if (e >> i & 1) for (int j = 0; j < n; j++) if (e >> j & 1) A[i][j] += zt;
  }
  for (int i = 0; i < n; i++) A[i][i] += z[2 * g->L + h->chord[i]];
  /* Gauss-Jordan with partial pivoting: determinant and inverse */
  REAL det = 1;
  for (int c = 0; c < n; c++) {
    int piv = c; REAL best = A[c][c] < 0 ? -A[c][c] : A[c][c];
    for (int r = c + 1; r < n; r++) { REAL v = A[r][c] < 0 ? -A[r][c] : A[r][c]; if (v > best) { best = v; piv = r; } }
    if (piv != c) { for (int k = 0; k < n; k++) { REAL t = A[c][k]; A[c][k] = A[piv][k]; A[piv][k] = t; t = Inv[c][k]; Inv[c][k] = Inv[piv][k]; Inv[piv][k] = t; } det = -det; }
    REAL p = A[c][c]; det *= p;
    for (int k = 0; k < n; k++) { A[c][k] /= p; Inv[c][k] /= p; }
    for (int r = 0; r < n; r++) if (r != c) { REAL f = A[r][c]; if (f != 0) for (int k = 0; k < n; k++) { A[r][k] -= f * A[c][k]; Inv[r][k] -= f * Inv[c][k]; } }
  }
  gv->U = det;
  for (int s = 0; s < h->nslot; s++) for (int u = 0; u < h->nslot; u++) {
    REAL b = 0;
    for (int i = 0; i < n; i++) if (h->slot[s].eps >> i & 1) for (int j = 0; j < n; j++) if (h->slot[u].eps >> j & 1) b += Inv[i][j];
    gv->beta[s][u] = b;
  }
  REAL V = 0;
  for (int s = 0; s < h->nslot; s++) {
    REAL x = 0, q = 0;
    for (int u = 0; u < h->nslot; u++) if (h->slot[u].kind == SLOT_LINE) {
      REAL zb = z[h->slot[u].line] * gv->beta[s][u];
      x += zb; q += zb * (REAL)h->slot[u].sgn;
    }
    gv->x[s] = x; gv->aq[s] = ((REAL)h->slot[s].sgn - q) / 2;
  }
  for (int u = 0; u < h->nslot; u++) if (h->slot[u].kind == SLOT_LINE) V += z[h->slot[u].line] * gv->x[u];
  gv->V = V; gv->done = 1;
}

static void FN(graded_mul)(REAL *acc, const REAL *b) { /* acc <- acc (*) b, truncated at NGRADE */
  REAL r[NGRADE];
  for (int c = 0; c < NGRADE; c++) { REAL s = 0; for (int i = 0; i <= c; i++) s += acc[i] * b[c - i]; r[c] = s; }
  for (int c = 0; c < NGRADE; c++) acc[c] = r[c];
}

static void FN(eval_node)(const struct oracle_diagram *d, int ni, const REAL *z, FN(GeomVal) *gvs, FN(NodeVal) *nvs) {
  const Node *nd = &d->nodes[ni]; FN(NodeVal) *nv = &nvs[ni];
  if (nv->done) return;
  const GeomEntry *ge = &d->geoms[nd->geom]; const Geom *h = &ge->h;
  FN(GeomVal) *gv = &gvs[nd->geom];
  if (!gv->done) FN(eval_geom)(&d->g, h, z, gv);
  nv->Uprod = gv->U; nv->Vsum = gv->V;
  for (int c = 0; c < nd->nchild; c++) {
    FN(eval_node)(d, nd->child[c], z, gvs, nvs);
    nv->Uprod *= nvs[nd->child[c]].Uprod; nv->Vsum += nvs[nd->child[c]].Vsum;
  }
  const PieceTable *tab = ge->tab[nd->op];
  int npat = 1 << h->nchild;
  REAL (*N)[32][NGRADE] = (REAL(*)[32][NGRADE])calloc(2, sizeof(REAL[32][NGRADE]));
  for (int k = 0; k < tab->n; k++) {
    const Monomial *m = &tab->mono[k];
    REAL prod = 1;
    for (int f = 0; f < m->nfac; f++) {
      int i = m->fac[f].i, j = m->fac[f].j;
      switch (m->fac[f].kind) {
        case F_DPLUS: prod *= (2 - gv->x[i]); break;      /* 1 + A_t */
        case F_DMINUS: prod *= gv->x[i]; break;            /* 1 - A_t */
        case F_BETA: prod *= gv->beta[i][j]; break;
        case F_AQ: prod *= gv->aq[i]; break;
        case F_AT: prod *= (1 - gv->x[i]); break;          /* A_t */
      }
    }
    for (int o = 0; o < tab->nout; o++) N[o][m->pattern][m->grade] += (REAL)m->coef[o] * prod;
  }
  if (h->type == 1 && (nd->op == OP_U || nd->op == OP_LMU))     /* these tables hold 12*coefficient (qed_tables.h func_UV12) */
    for (int pat = 0; pat < npat; pat++) for (int c = 0; c < NGRADE; c++) N[0][pat][c] /= 12;
  for (int o = 0; o < 2; o++) for (int c = 0; c < NGRADE; c++) nv->v[o][c] = 0;
  for (int o = 0; o < tab->nout; o++)
    for (int pat = 0; pat < npat; pat++) {
      REAL G[NGRADE]; int any = 0;
      for (int c = 0; c < NGRADE; c++) { G[c] = N[o][pat][c]; if (G[c] != 0) any = 1; }
      if (!any) continue;
      for (int c = 0; c < h->nchild; c++) {
        const FN(NodeVal) *cv = &nvs[nd->child[c]];
        if (h->child_type[c] == 1) FN(graded_mul)(G, cv->v[0]);
        else FN(graded_mul)(G, (pat >> c & 1) ? cv->v[1] : cv->v[0]);
      }
      for (int c = 0; c < NGRADE; c++) nv->v[o][c] += G[c];
    }
  free(N);
  nv->done = 1;
}

/* integrand at a point; term_out (may be NULL) receives the signed value of every term; abs_out the
 * sum of |sign * grade contribution| over all terms and grades (round-off scale) */
static REAL FN(eval_integrand)(const struct oracle_diagram *d, const REAL *z, REAL *term_out, REAL *abs_out) {
  FN(GeomVal) *gvs = (FN(GeomVal) *)malloc(sizeof(FN(GeomVal)) * d->ngeom);
  FN(NodeVal) *nvs = (FN(NodeVal) *)malloc(sizeof(FN(NodeVal)) * d->nnode);
  for (int i = 0; i < d->ngeom; i++) gvs[i].done = 0;
  for (int i = 0; i < d->nnode; i++) nvs[i].done = 0;
  int L = d->g.L;
  static const double FACT[6] = {1, 1, 2, 6, 24, 120};
  REAL f = 0, asum = 0;
  for (int t = 0; t < d->nterm; t++) {
    int root = d->terms[t].root;
    FN(eval_node)(d, root, z, gvs, nvs);
    const FN(NodeVal) *nv = &nvs[root];
    REAL U2 = nv->Uprod * nv->Uprod, ft = 0, Vp = 1; /* Vp = Vsum^(L-c), built from c=L-1 downwards */
    for (int c = L - 1; c >= 0; c--) {
      Vp *= nv->Vsum;
      REAL contrib = (REAL)(d->terms[t].sign * FACT[L - c - 1]) * nv->v[0][c] / (U2 * Vp);
      ft += contrib; asum += contrib < 0 ? -contrib : contrib;
    }
    if (term_out) term_out[t] = ft;
    f += ft;
  }
  if (abs_out) *abs_out = asum;
  free(gvs); free(nvs);
  return f;
}
