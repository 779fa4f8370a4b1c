// host_prepare.cpp — host-side preparation of one diagram: term trees, unique pieces and nodes,
// numerator tables, and the device blob (device_layout.h). Not on the timed path.
// Product code (libmcqed.so); shares nothing with oracle/.
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <functional>
#include <memory>
#include <thread>

#include "coef_gen.hpp"
#include "diagram.hpp"

// =====================================================================================
//                                   host preparation
// =====================================================================================
namespace {

struct NodeKey { int geom, op; std::vector<int> kids; bool operator==(const NodeKey &o) const { return geom == o.geom && op == o.op && kids == o.kids; } };

struct Builder {
  mc_diagram &d;
  std::vector<mq::Piece> pieces;                 // one per geom
  std::vector<std::pair<int, uint32_t>> geomKey; // (sub index or -1, child mask)
  std::vector<NodeKey> nodeKeys;
  explicit Builder(mc_diagram &dd_) : d(dd_) {}

  mq::Segment segOf(int sub) const { return sub < 0 ? mq::Segment{0, 2 * d.g.L, true} : d.ft.subs[sub]; }

  int opOf(int H, int gprime) const {
    if (H == gprime) return MQ_OP_A;
    const bool inI = H < 0 || (d.ft.subs[H].vertexLike && d.ft.subs[H].has(d.g.e));
    const bool insideGp = H >= 0 && (gprime < 0 || (d.ft.subs[H].within(d.ft.subs[gprime]) && H != gprime));
    if (!inI || insideGp) return MQ_OP_U;
    return H < 0 ? MQ_OP_LMU : MQ_OP_L;
  }
  int geomOf(int H, uint32_t F) {
    auto kids = d.ft.childrenOf(F, segOf(H));
    uint32_t cm = 0; for (int k : kids) cm |= 1u << k;
    for (size_t i = 0; i < geomKey.size(); i++) if (geomKey[i].first == H && geomKey[i].second == cm) return (int)i;
    std::vector<mq::Segment> ks; for (int k : kids) ks.push_back(d.ft.subs[k]);
    mq::Piece p; p.build(d.g, segOf(H), ks);
    pieces.push_back(p); geomKey.emplace_back(H, cm);
    return (int)pieces.size() - 1;
  }
  int nodeOf(int H, uint32_t F, int gprime) {
    NodeKey k; k.geom = geomOf(H, F); k.op = opOf(H, gprime);
    for (int c : d.ft.childrenOf(F, segOf(H))) k.kids.push_back(nodeOf(c, F, gprime));
    for (size_t i = 0; i < nodeKeys.size(); i++) if (nodeKeys[i] == k) return (int)i;
    nodeKeys.push_back(k);
    return (int)nodeKeys.size() - 1;
  }
};

}  // namespace

int mq_prepare_host(const mc_graph *graph, const mc_forests *uf, const mc_options *opts, bool use_gpu, mc_diagram **out) {
  if (!graph || !out) return MC_EINVAL;
  std::unique_ptr<mc_diagram> d(new mc_diagram);
  d->opt = opts ? *opts : mc_options{1.0, 1e30, 2.8e4, 1e-2, 0u, 0.5, 0.0, 0.0, 0.0};
  if (!(d->opt.deg_floor > 0) || !(d->opt.deg_cap >= d->opt.deg_floor) || !(d->opt.cond_max > 0)) return MC_EINVAL;
  if (!(d->opt.mix_alpha >= 0.0 && d->opt.mix_alpha < 1.0)) return MC_EINVAL;
  if (d->opt.mix_alpha > 0.0 && !(d->opt.deg_floor2 > 0 && d->opt.deg_cap >= d->opt.deg_floor2)) return MC_EINVAL;
  if (!d->g.build(graph->loops, graph->ext_pos, graph->chord_a, graph->chord_b)) return MC_EINVAL;
  d->id = d->g.canonicalId();
  if (d->id < 0) return MC_EINVAL;
  d->ft.enumerate(d->g);
  if (uf) {   // user forests must agree with the enumeration
    if (uf->n_sub != (int)d->ft.subs.size() || uf->n_forest != (int)d->ft.forests.size()) return MC_EINVAL;
    for (int i = 0; i < uf->n_sub; i++) if (uf->seg_lo[i] != d->ft.subs[i].lo || uf->seg_hi[i] != d->ft.subs[i].hi) return MC_EINVAL;
    for (int i = 0; i < uf->n_forest; i++) if (uf->forest_mask[i] != d->ft.forests[i]) return MC_EINVAL;
  }
  d->st.build(d->g, d->ft, d->opt.deg_floor, d->opt.deg_cap, d->opt.deg_floor_ir);
  if (d->opt.mix_alpha > 0.0) d->st2.build(d->g, d->ft, d->opt.deg_floor2, d->opt.deg_cap, d->opt.deg_floor_ir2);

  // ---- term trees -> unique pieces (geoms) and nodes ----
  Builder B(*d);
  std::vector<int> roots;
  for (auto &t : d->ft.terms) roots.push_back(B.nodeOf(-1, t.forest, t.gprime));
  const int ngeom0 = (int)B.pieces.size(), nnode0 = (int)B.nodeKeys.size();
  if (ngeom0 > MQ_MAXGEOM || nnode0 > MQ_MAXNODE) return MC_ELIMIT;
  // geoms sorted by segment length (children first), then lo, then child mask
  std::vector<int> gorder(ngeom0);
  for (int i = 0; i < ngeom0; i++) gorder[i] = i;
  std::sort(gorder.begin(), gorder.end(), [&](int a, int b) {
    const auto &pa = B.pieces[a].seg, &pb = B.pieces[b].seg;
    if (pa.hi - pa.lo != pb.hi - pb.lo) return pa.hi - pa.lo < pb.hi - pb.lo;
    if (pa.lo != pb.lo) return pa.lo < pb.lo;
    return B.geomKey[a].second < B.geomKey[b].second;
  });
  std::vector<int> gnew(ngeom0);
  for (int i = 0; i < ngeom0; i++) gnew[gorder[i]] = i;
  // tables: (geom, op) pairs in geom order; nodes sorted by (geom, op)
  std::vector<int> norder(nnode0);
  for (int i = 0; i < nnode0; i++) norder[i] = i;
  std::stable_sort(norder.begin(), norder.end(), [&](int a, int b) {
    int ga = gnew[B.nodeKeys[a].geom], gb = gnew[B.nodeKeys[b].geom];
    if (ga != gb) return ga < gb;
    return B.nodeKeys[a].op < B.nodeKeys[b].op;
  });
  std::vector<int> nnew(nnode0);
  for (int i = 0; i < nnode0; i++) nnew[norder[i]] = i;

  d->geoms.resize(ngeom0);
  for (int gi = 0; gi < ngeom0; gi++) {
    const mq::Piece &p = B.pieces[gorder[gi]];
    DevGeom G; std::memset(&G, 0, sizeof G);
    G.nch = (int)p.ownChord.size(); G.nslot = (int)p.slots.size(); G.nchild = (int)p.kids.size(); G.nS = p.nS;
    if (G.nslot > MQ_MAXSLOT || G.nchild > MQ_MAXCHILD || (1 << G.nS) > MQ_MAXPAT) return MC_ELIMIT;
    for (int i = 0; i < G.nch; i++) G.chord_zline[i] = 2 * d->g.L + p.ownChord[i];
    for (int s = 0; s < G.nslot; s++) {
      G.slot[s].kind = p.slots[s].insertion ? MQ_SLOT_INS : MQ_SLOT_LINE;
      G.slot[s].zline = (int8_t)p.slots[s].line; G.slot[s].sgn = (int8_t)p.slots[s].sgn;
      G.slot[s].child = (int8_t)p.slots[s].child; G.slot[s].eps = p.slots[s].eps;
    }
    for (int c = 0; c < G.nchild; c++) { G.child_type[c] = p.kids[c].vertexLike ? 1 : 0; G.child_patbit[c] = (int8_t)p.patbit[c]; }
    d->geoms[gi] = G;
  }
  // nodes + tables
  const bool no_tables = d->opt.flags & 2u;
  d->nodes.resize(nnode0);
  std::vector<mq::TableBuild> builds;
  unsigned hw = std::thread::hardware_concurrency();
  int nthreads = hw ? (int)hw : 4;
  if (const char *env = std::getenv("MCQED_PREPARE_THREADS")) nthreads = std::max(1, atoi(env));
  for (int ni = 0; ni < nnode0; ni++) {
    const NodeKey &k = B.nodeKeys[norder[ni]];
    const int gi = gnew[k.geom];
    const mq::Piece &p = B.pieces[k.geom];
    if (d->tables.empty() || d->tables.back().geom != gi || d->tables.back().op != k.op) {
      DevTable T; std::memset(&T, 0, sizeof T);
      T.geom = gi; T.op = k.op; T.nout = p.seg.vertexLike ? 1 : 2; T.first_node = ni; T.nnode = 0;
      d->tables.push_back(T);
      builds.push_back(no_tables ? mq::TableBuild{} : mq::buildTable(p, k.op, nthreads, d->g.L - 1, use_gpu ? mq_count_units_gpu : nullptr));
    }
    d->tables.back().nnode++;
    DevNode N; std::memset(&N, 0, sizeof N);
    N.table = (int)d->tables.size() - 1; N.geom = gi; N.nchild = (int)k.kids.size(); N.nout = p.seg.vertexLike ? 1 : 2;
    for (int c = 0; c < N.nchild; c++) N.child[c] = nnew[k.kids[c]];
    int loops_inside = 0;
    for (int i = 0; i < d->g.L; i++) if (p.seg.has(d->g.ca[i]) && p.seg.has(d->g.cb[i])) loops_inside++;
    N.ngr = std::min(MQ_NGRADE, loops_inside + 1);
    N.val_off = d->nodeval_len; d->nodeval_len += N.nout * N.ngr;
    d->nodes[ni] = N;
  }
  if (d->nodeval_len > MQ_MAXNODEVAL) return MC_ELIMIT;
  for (size_t ti = 0; ti < d->tables.size(); ti++) {
    DevGeom &G = d->geoms[d->tables[ti].geom];
    if (G.ntable == 0) G.first_table = (int)ti;
    G.ntable++;
  }
  for (size_t t = 0; t < d->ft.terms.size(); t++) d->terms.push_back({nnew[roots[t]], d->ft.terms[t].sign});
  // layout of the per-point scalar array of every piece (only what its tables can reference)
  for (auto &G : d->geoms) {
    bool needAq = false;
    for (int ti = G.first_table; ti < G.first_table + G.ntable; ti++) needAq |= d->tables[ti].op == MQ_OP_A;
    int o = G.nslot;
    G.off_at = G.nS > 0 ? o : -1; if (G.nS > 0) o += G.nslot;
    G.off_aq = needAq ? o : -1; if (needAq) o += G.nslot;
    G.off_bt = o; o += G.nslot * (G.nslot - 1) / 2;
    G.scal_len = o;
    d->max_scal_len = std::max(d->max_scal_len, o);
  }

  // ---- blob ----
  auto words = [](size_t bytes) { return (int64_t)((bytes + 7) / 8); };
  DevHeader H; std::memset(&H, 0, sizeof H);
  H.L = d->g.L; H.M = d->g.M; H.diag_id = d->id; H.ngeom = ngeom0; H.ntable = (int)d->tables.size(); H.nnode = nnode0; H.nterm = (int)d->terms.size();
  H.nodeval_len = d->nodeval_len; H.max_scal_len = d->max_scal_len; H.wl = MQ_WL; H.C = d->st.C; H.cond_max = d->opt.cond_max;
  int64_t off = words(sizeof(DevHeader));
  const int64_t nZ = (int64_t)1 << d->g.M;
  H.off_Z = off; off += nZ; H.off_invdeg = off; off += nZ;
  H.off_geom = off; off += words(sizeof(DevGeom) * d->geoms.size());
  H.off_table = off; off += words(sizeof(DevTable) * d->tables.size());
  H.off_node = off; off += words(sizeof(DevNode) * d->nodes.size());
  H.off_term = off; off += words(sizeof(DevTerm) * d->terms.size());
  if (d->opt.mix_alpha > 0.0) {
    H.mix_alpha = d->opt.mix_alpha; H.C2 = d->st2.C;
    H.off_Z2 = off; off += nZ; H.off_invdeg2 = off; off += nZ; H.off_deg1 = off; off += nZ; H.off_deg2 = off; off += nZ;
  }
  // MRG32k3a (mc_options.flags bit 2, S1b): the powers A^(2^k), k < 64, of the companion matrices of
  // x1_n = (1403580 x1_{n-2} - 810728 x1_{n-3}) mod m1 and x2_n = (527612 x2_{n-1} - 1370589 x2_{n-3}) mod m2, acting on
  // (x_{n-3}, x_{n-2}, x_{n-1}); the kernels reach a sample's position in the sequence with one matrix-vector product per set bit
  std::vector<uint32_t> mrg_pow;
  if (d->opt.flags & 4u) {
    if (d->id >= (1 << 20)) return MC_ELIMIT;
    const uint64_t mod[2] = {4294967087ull, 4294944443ull};
    mrg_pow.resize(2 * 64 * 9);
    for (int comp = 0; comp < 2; comp++) {
      const uint64_t m = mod[comp];
      uint64_t A[3][3] = {{0, 1, 0}, {0, 0, 1}, {0, 0, 0}};
      if (comp == 0) { A[2][0] = m - 810728ull; A[2][1] = 1403580ull; } else { A[2][0] = m - 1370589ull; A[2][2] = 527612ull; }
      for (int k = 0; k < 64; k++) {
        for (int i = 0; i < 9; i++) mrg_pow[(size_t)(comp * 64 + k) * 9 + i] = (uint32_t)A[i / 3][i % 3];
        uint64_t Q[3][3];
        for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) {
          uint64_t acc = 0;
          for (int t = 0; t < 3; t++) acc = (acc + A[i][t] * A[t][j] % m) % m;
          Q[i][j] = acc;
        }
        std::memcpy(A, Q, sizeof A);
      }
    }
    H.rng = 1; H.off_mrg = off; off += words(sizeof(uint32_t) * mrg_pow.size());
  }
  // streams: a sequence of entries of MQ_WL same-shape families (device_layout.h). The kernels stage the stream through
  // shared memory in chunks of MQ_CHUNK_WORDS (bulk async copies), so (i) the stream starts on a 16-byte boundary,
  // (ii) no entry straddles a chunk boundary (a PAD header, c = 7, fills the rest of a chunk), (iii) coefficients
  // start on a 16-byte boundary (read as double2), (iv) the stream is consumed strictly in order: tables are laid
  // out in the order the evaluator visits them.
  if (off & 1) off++;
  std::vector<uint64_t> streams;
  const int64_t stream_base = off;
  for (size_t ti = 0; ti < d->tables.size(); ti++) {
    DevTable &T = d->tables[ti]; const mq::TableBuild &tb = builds[ti];
    T.stream_off = stream_base + (int64_t)streams.size(); T.n_monomials = tb.n_stored;
    const int ns = d->geoms[T.geom].nslot;
    const DevGeom &GG = d->geoms[T.geom];
    auto tri = [&](int a, int b) { if (a > b) std::swap(a, b); return GG.off_bt + a * ns - a * (a + 1) / 2 + (b - a - 1); };
    std::vector<const mq::Family *> order;
    for (auto &f : tb.fams) order.push_back(&f);
    // shape-major, so that MQ_WL consecutive families share their static code; inside a shape by (output, pattern): the
    // evaluator accumulates a run of equal (output, pattern, grade) in registers
    std::stable_sort(order.begin(), order.end(), [](const mq::Family *a, const mq::Family *b) {
      if (a->c != b->c) return a->c < b->c;
      if (a->kd != b->kd) return a->kd < b->kd;
      if (a->out != b->out) return a->out < b->out;
      return a->pattern < b->pattern;
    });
    auto index_bytes = [&](const mq::Family &f, std::vector<uint8_t> &idx) -> bool {
      idx.clear();
      const int n2 = 2 * f.c;
      for (int i = 0; i < n2; i++) for (int j = i + 1; j < n2; j++) idx.push_back((uint8_t)tri(f.paired[i], f.paired[j]));
      for (uint8_t sl : f.inner) idx.push_back(sl);                            // r_t lives at S[t]
      for (uint8_t sc : f.scal) {
        const int kind = sc >> 4, slot = sc & 15;
        const int base = kind == MQ_SC_R ? 0 : kind == MQ_SC_AT ? GG.off_at : GG.off_aq;
        if (base < 0) return false;                                            // a table references a scalar its piece does not carry
        idx.push_back((uint8_t)(base + slot));
      }
      return true;
    };
    int nentries = 0;
    std::vector<size_t> entry_at;                                              // stream position of every entry header of this table
    std::vector<int> entry_shape;
    for (size_t at0 = 0; at0 < order.size();) {
      const mq::Family &f0 = *order[at0];
      int nm = 1;                                                              // members of this entry (same shape), the rest is VOID
      while (nm < MQ_WL && at0 + nm < order.size() && order[at0 + nm]->c == f0.c && order[at0 + nm]->kd == f0.kd) nm++;
      std::vector<uint8_t> idx[MQ_WL];
      int idxw = 1;                                                            // the kernel always reads two index words per member
      for (int m = 0; m < MQ_WL; m++) {
        if (!index_bytes(m < nm ? *order[at0 + m] : f0, idx[m])) return MC_ELIMIT;
        if (m >= nm) idx[m].resize((size_t)(f0.c * (2 * f0.c - 1) + f0.kd));   // VOID member: no scalar factors
        idxw = std::max(idxw, (int)words(idx[m].size()));
      }
      const size_t ncf = f0.coef.size();
      const int64_t need = MQ_WL + (int64_t)MQ_WL * idxw + (int64_t)MQ_WL * (int64_t)ncf;    // even: coefficients stay 16-byte aligned
      if (need > MQ_CHUNK_WORDS) return MC_ELIMIT;
      const int64_t in_chunk = (int64_t)streams.size() % MQ_CHUNK_WORDS;
      if (in_chunk + need > MQ_CHUNK_WORDS) {                                  // PAD to the chunk boundary
        const int64_t rest = MQ_CHUNK_WORDS - in_chunk;
        streams.push_back(mq_pack_family(7, 0, 0, 0, 0, (int)(rest - 1), 0u));
        streams.resize(streams.size() + (size_t)(rest - 1), 0ull);
      }
      entry_at.push_back(streams.size()); entry_shape.push_back(f0.c * 8 + f0.kd);
      for (int m = 0; m < MQ_WL; m++) {
        const mq::Family &f = m < nm ? *order[at0 + m] : f0;
        if (f.coef.size() != ncf || MQ_WL * ncf > 0xFFFF) return MC_ELIMIT;
        streams.push_back(mq_pack_family(f.c, f.kd, f.pattern, m < nm ? (int)f.scal.size() : 0, f.out, idxw, (uint32_t)(MQ_WL * ncf), m < nm ? 0 : 1));
      }
      for (int m = 0; m < MQ_WL; m++) {
        const size_t at = streams.size();
        streams.resize(at + idxw, 0ull);
        std::memcpy(streams.data() + at, idx[m].data(), idx[m].size());
      }
      const size_t unit = f0.kd >= 1 ? 2 : 1, nunit = ncf / unit, at = streams.size();
      streams.resize(at + MQ_WL * ncf, 0ull);
      for (int m = 0; m < nm; m++) {
        const double *src = order[at0 + m]->coef.data();
        for (size_t u = 0; u < nunit; u++) std::memcpy(streams.data() + at + (u * MQ_WL + m) * unit, src + u * unit, sizeof(double) * unit);
      }
      at0 += nm; nentries++;
    }
    // run lengths: bits 48..63 of every header word = entries from this one to the end of its run of equal shape (c, kd);
    // the kernels take the shape switch once per run (mcqed_kernels.cuh run_loop)
    for (size_t i = entry_at.size(); i-- > 0;) {
      const uint64_t run = (i + 1 < entry_at.size() && entry_shape[i + 1] == entry_shape[i]) ? (streams[entry_at[i + 1]] >> 48) + 1 : 1;
      if (run > 0xFFFF) return MC_ELIMIT;
      for (int m = 0; m < MQ_WL; m++) streams[entry_at[i] + m] |= run << 48;
    }
    T.nfam = nentries;
    T.stream_words = stream_base + (int64_t)streams.size() - T.stream_off;
    d->n_stored += tb.n_stored; d->n_nonzero += tb.n_nonzero;
  }
  {                                                                            // close the last chunk
    const int64_t in_chunk = (int64_t)streams.size() % MQ_CHUNK_WORDS;
    if (in_chunk || streams.empty()) {
      const int64_t rest = MQ_CHUNK_WORDS - in_chunk;
      streams.push_back(mq_pack_family(7, 0, 0, 0, 0, (int)(rest - 1), 0u));
      streams.resize(streams.size() + (size_t)(rest - 1), 0ull);
    }
  }
  H.off_stream = stream_base; H.stream_chunks = (int64_t)streams.size() / MQ_CHUNK_WORDS;
  off += (int64_t)streams.size();
  H.total_words = off;
  d->blob.assign((size_t)off, 0ull);
  std::memcpy(d->blob.data(), &H, sizeof H);
  std::memcpy(d->blob.data() + H.off_Z, d->st.Z.data(), sizeof(double) * nZ);
  std::memcpy(d->blob.data() + H.off_invdeg, d->st.invdeg.data(), sizeof(double) * nZ);
  std::memcpy(d->blob.data() + H.off_geom, d->geoms.data(), sizeof(DevGeom) * d->geoms.size());
  std::memcpy(d->blob.data() + H.off_table, d->tables.data(), sizeof(DevTable) * d->tables.size());
  std::memcpy(d->blob.data() + H.off_node, d->nodes.data(), sizeof(DevNode) * d->nodes.size());
  std::memcpy(d->blob.data() + H.off_term, d->terms.data(), sizeof(DevTerm) * d->terms.size());
  if (!mrg_pow.empty()) std::memcpy(d->blob.data() + H.off_mrg, mrg_pow.data(), sizeof(uint32_t) * mrg_pow.size());
  if (d->opt.mix_alpha > 0.0) {
    std::memcpy(d->blob.data() + H.off_Z2, d->st2.Z.data(), sizeof(double) * nZ);
    std::memcpy(d->blob.data() + H.off_invdeg2, d->st2.invdeg.data(), sizeof(double) * nZ);
    std::memcpy(d->blob.data() + H.off_deg1, d->st.deg.data(), sizeof(double) * nZ);
    std::memcpy(d->blob.data() + H.off_deg2, d->st2.deg.data(), sizeof(double) * nZ);
  }
  if (!streams.empty()) std::memcpy(d->blob.data() + stream_base, streams.data(), sizeof(uint64_t) * streams.size());
  d->have_tables = !no_tables;
  *out = d.release();
  return MC_OK;
}

