// mcqed_api.cpp — the C ABI of include/mcqed.h: argument checks, device upload, launch sequencing.
// Product code (libmcqed.so); shares nothing with oracle/. No CPU fallback: every device entry
// point fails with MC_ECUDA if CUDA is unusable.
#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstring>
#include <new>

#include "diagram.hpp"

namespace {
std::atomic<unsigned long long> g_launches{0};

int to_device(mc_diagram *d) {
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return MC_ECUDA;
  if (!d->have_tables) return MC_EINVAL;
  const size_t bytes = d->blob.size() * 8;
  if (cudaMalloc(&d->d_blob, bytes) != cudaSuccess) return MC_ENOMEM;
  if (cudaMemcpy(d->d_blob, d->blob.data(), bytes, cudaMemcpyHostToDevice) != cudaSuccess) return MC_ECUDA;
  if (cudaMalloc(&d->ws.partial, sizeof(double) * 3 * mqk::MAXGRID * 4) != cudaSuccess) return MC_ENOMEM;
  if (cudaMalloc(&d->ws.lost_list, sizeof(unsigned long long) * mqk::LOSTCAP) != cudaSuccess) return MC_ENOMEM;
  if (cudaMalloc(&d->ws.flag_list, sizeof(unsigned long long) * mqk::CHUNK) != cudaSuccess) return MC_ENOMEM;
  if (cudaMalloc(&d->ws.counters, sizeof(unsigned long long) * 4) != cudaSuccess) return MC_ENOMEM;
  if (cudaMemset(d->ws.counters, 0, sizeof(unsigned long long) * 4) != cudaSuccess) return MC_ECUDA;
  if (mq_config_f64(d) != 0 || mq_config_dd(d) != 0 || mq_config_qd(d) != 0) return MC_ECUDA;
  d->on_device = true;
  return MC_OK;
}
}  // namespace

#define MQ_CK(x) do { if ((x) != cudaSuccess) return MC_ECUDA; } while (0)

extern "C" {

int mc_prepare_diagram_host(const mc_graph *graph, const mc_forests *forests, const mc_options *opts, mc_diagram **out) {
  try { return mq_prepare_host(graph, forests, opts, false, out); } catch (const std::bad_alloc &) { return MC_ENOMEM; } catch (...) { return MC_EINVAL; }
}
int mc_prepare_diagram(const mc_graph *graph, const mc_forests *forests, const mc_options *opts, mc_diagram **out) {
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return MC_ECUDA;   // fail loudly: no CPU fallback
  mc_diagram *d = nullptr;
  int rc;
  try { rc = mq_prepare_host(graph, forests, opts, true, &d); } catch (const std::bad_alloc &) { rc = MC_ENOMEM; } catch (...) { rc = MC_EINVAL; }
  if (rc != MC_OK) return rc;
  rc = to_device(d);
  if (rc != MC_OK) { mc_free_diagram(d); return rc; }
  *out = d;
  return MC_OK;
}
void mc_free_diagram(mc_diagram *d) {
  if (!d) return;
  if (d->d_blob) cudaFree(d->d_blob);
  if (d->ws.partial) cudaFree(d->ws.partial);
  if (d->ws.flag_list) cudaFree(d->ws.flag_list);
  if (d->ws.lost_list) cudaFree(d->ws.lost_list);
  if (d->ws.counters) cudaFree(d->ws.counters);
  delete d;
}
int mc_diagram_info(const mc_diagram *d, int32_t *k, int32_t *m, int32_t *n, int32_t *n_terms, int64_t *flop_per_sample, int64_t *table_bytes) {
  if (!d) return MC_EINVAL;
  int kk, mm, nn; d->g.classKMN(kk, mm, nn);
  if (k) *k = kk;
  if (m) *m = mm;
  if (n) *n = nn;
  if (n_terms) *n_terms = (int32_t)d->terms.size();
  // 2 flop per non-zero numerator monomial (one FMA in the nested evaluation) + ~600 flop per piece (a4) + ~3000 (a1-a3) + 12 per term grade (a6)
  if (flop_per_sample) *flop_per_sample = 2 * d->n_nonzero + 600 * (int64_t)d->geoms.size() + 3000 + 12 * (int64_t)d->terms.size() * d->g.L;
  if (table_bytes) *table_bytes = (int64_t)d->blob.size() * 8;
  return MC_OK;
}
int mc_diagram_id(const mc_diagram *d, int32_t *id) { if (!d || !id) return MC_EINVAL; *id = d->id; return MC_OK; }
int mc_diagram_subgraphs(const mc_diagram *d, int32_t *lo, int32_t *hi, int32_t *type, int32_t cap) {
  if (!d) return MC_EINVAL;
  int n = (int)d->ft.subs.size();
  for (int i = 0; i < n && i < cap; i++) { if (lo) lo[i] = d->ft.subs[i].lo; if (hi) hi[i] = d->ft.subs[i].hi; if (type) type[i] = d->ft.subs[i].vertexLike ? 1 : 0; }
  return n;
}
int mc_diagram_forests(const mc_diagram *d, uint32_t *mask, int32_t cap) {
  if (!d) return MC_EINVAL;
  int n = (int)d->ft.forests.size();
  for (int i = 0; i < n && i < cap; i++) if (mask) mask[i] = d->ft.forests[i];
  return n;
}
int mc_diagram_terms(const mc_diagram *d, uint32_t *forest, int32_t *gprime, int32_t *sign, int32_t cap) {
  if (!d) return MC_EINVAL;
  int n = (int)d->ft.terms.size();
  for (int i = 0; i < n && i < cap; i++) { if (forest) forest[i] = d->ft.terms[i].forest; if (gprime) gprime[i] = d->ft.terms[i].gprime; if (sign) sign[i] = d->ft.terms[i].sign; }
  return n;
}
int mc_diagram_sampler_tables(const mc_diagram *d, double *deg, double *Z, double *C) {
  if (!d) return MC_EINVAL;
  size_t n = (size_t)1 << d->g.M;
  if (deg) std::memcpy(deg, d->st.deg.data(), n * sizeof(double));
  if (Z) std::memcpy(Z, d->st.Z.data(), n * sizeof(double));
  if (C) *C = d->st.C;
  return MC_OK;
}
int mc_diagram_set_flags(mc_diagram *d, uint32_t flags) {
  if (!d) return MC_EINVAL;
  d->opt.flags = (d->opt.flags & ~1u) | (flags & 1u);
  return MC_OK;
}
int mc_diagram_set_precision(mc_diagram *d, double cond_max, double amin_min, double dd_cond_max, double w_abs_tol) {
  if (!d || !(cond_max > 0) || !(dd_cond_max >= 1.0) || !(w_abs_tol >= 0) || !(amin_min <= 1.0)) return MC_EINVAL;
  d->opt.cond_max = cond_max; d->opt.amin_min = amin_min; d->dd_cond_max = dd_cond_max; d->w_abs_tol = w_abs_tol;
  return MC_OK;
}
int64_t mc_diagram_blob(const mc_diagram *d, uint64_t *out, int64_t cap) {
  if (!d) return MC_EINVAL;
  int64_t n = (int64_t)d->blob.size();
  if (out) std::memcpy(out, d->blob.data(), sizeof(uint64_t) * (size_t)std::min(n, cap));
  return n;
}

// MRG32k3a stream (mc_options.flags bit 2): a sample owns 64 outputs of the sequence and a diagram 2^38 samples (S1b)
static bool rng_range_ok(const mc_diagram *d, uint64_t first, uint64_t n) {
  return !(d->opt.flags & 4u) || (first <= (1ull << 38) && n <= (1ull << 38) - first);
}

int mc_integrate(const mc_diagram *d, uint64_t first_sample, uint64_t n_samples, uint64_t seed, void *cuda_stream,
                 double *out_sum, double *out_sumsq, unsigned long long *out_n_flagged, unsigned long long *out_n_dropped) {
  if (!d || !d->on_device || !rng_range_ok(d, first_sample, n_samples)) return MC_EINVAL;
  mq_stream st = (mq_stream)cuda_stream;
  const bool no_dd = d->opt.flags & 1u;
  for (uint64_t done = 0; done < n_samples; done += mqk::CHUNK) {
    const uint64_t n = std::min<uint64_t>(mqk::CHUNK, n_samples - done);
    const int g1 = (int)std::min<uint64_t>((uint64_t)d->grid_f64, (n + mqk::PTS_F64 - 1) / mqk::PTS_F64);
    mq_launch_integrate_f64(d, g1, first_sample + done, n, seed, d->prec(no_dd), st);
    int g2 = 0, g3 = 0;
    if (!no_dd) {     // second tier (double-double) and third tier (quad-double, only what the second could not resolve)
      g2 = d->grid_dd; mq_launch_integrate_dd(d, seed, st);
      g3 = d->grid_qd; mq_launch_integrate_qd(d, seed, st);
      g_launches += 2;
    }
    mq_launch_finish(d, g1, g2, g3, out_sum, out_sumsq, out_n_flagged, out_n_dropped, st);
    g_launches += 2;
  }
  MQ_CK(cudaGetLastError());
  return MC_OK;
}

int mc_integrate_host(const mc_diagram *d, uint64_t first_sample, uint64_t n_samples, uint64_t seed, void *cuda_stream,
                      double *sum, double *sumsq, unsigned long long *n_flagged, unsigned long long *n_dropped) {
  if (!d || !d->on_device) return MC_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  struct Out { double s, s2; unsigned long long nf, nd; } *dev = nullptr, host{0, 0, 0, 0};
  MQ_CK(cudaMallocAsync((void **)&dev, sizeof(Out), st));
  int rc = cudaMemsetAsync(dev, 0, sizeof(Out), st) == cudaSuccess ? MC_OK : MC_ECUDA;      // every exit below frees dev
  if (rc == MC_OK) rc = mc_integrate(d, first_sample, n_samples, seed, cuda_stream, &dev->s, &dev->s2, &dev->nf, &dev->nd);
  if (rc == MC_OK && cudaMemcpyAsync(&host, dev, sizeof(Out), cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = MC_ECUDA;
  if (cudaFreeAsync(dev, st) != cudaSuccess && rc == MC_OK) rc = MC_ECUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess && rc == MC_OK) rc = MC_ECUDA;
  if (rc != MC_OK) return rc;
  if (sum) *sum = host.s;
  if (sumsq) *sumsq = host.s2;
  if (n_flagged) *n_flagged = host.nf;
  if (n_dropped) *n_dropped = host.nd;
  return MC_OK;
}

int mc_integrate_static(const mc_diagram *d, uint64_t first_sample, uint64_t n_samples, uint64_t seed, void *cuda_stream,
                        double *out_sum, double *out_sumsq, unsigned long long *out_n_flagged, unsigned long long *out_n_dropped) {
  if (!d || !d->on_device || !rng_range_ok(d, first_sample, n_samples)) return MC_EINVAL;
  if (n_samples > (uint64_t)MC_STATIC_MAX_SAMPLES) return MC_ETOOBIG;       // the static flagged list has one slot per sample
  if (n_samples == 0) return MC_OK;
  if (mq_static_integrate_f64(d, first_sample, n_samples, seed, d->prec(true), out_sum, out_sumsq, out_n_flagged, out_n_dropped, (mq_stream)cuda_stream) != 0) return MC_ECUDA;
  g_launches += 3;
  return MC_OK;
}

int mc_eval_points(const mc_diagram *d, uint64_t first_sample, uint64_t n, uint64_t seed, void *cuda_stream,
                   double *z_out, int32_t *order_out, double *p_out, double *f_out, double *f64_out, double *cond_out, uint8_t *flag_out) {
  if (!d || !d->on_device || !rng_range_ok(d, first_sample, n)) return MC_EINVAL;
  mq_stream st = (mq_stream)cuda_stream;
  const bool no_dd = d->opt.flags & 1u;
  const int M = d->g.M;
  for (uint64_t done = 0; done < n; done += mqk::CHUNK) {
    const uint64_t m = std::min<uint64_t>(mqk::CHUNK, n - done);
    const int g1 = (int)std::min<uint64_t>(mqk::MAXGRID, (m + mqk::PTS_EVAL - 1) / mqk::PTS_EVAL);
    const bool list = f_out && !no_dd;
    mq_launch_reset(d, st);
    mq_launch_eval_points(d, g1, first_sample + done, m, seed, d->prec(no_dd),
                          z_out ? z_out + done * M : nullptr, order_out ? order_out + done * M : nullptr, p_out ? p_out + done : nullptr,
                          f_out ? f_out + done : nullptr, f64_out ? f64_out + done : nullptr, cond_out ? cond_out + done : nullptr,
                          flag_out ? flag_out + done : nullptr, list, st);
    g_launches += 2;
    if (list) {
      mq_launch_eval_points_dd(d, first_sample + done, seed, f_out + done, st);
      mq_launch_eval_points_qd(d, first_sample + done, seed, f_out + done, st);
      g_launches += 2;
    }
    mq_launch_reset(d, st);
    g_launches++;
  }
  MQ_CK(cudaGetLastError());
  return MC_OK;
}

int mc_eval_z(const mc_diagram *d, uint64_t n, const double *z_in, void *cuda_stream, double *f64_out, double *fdd_out, double *cond_out, double *aux_out) {
  if (!d || !d->on_device || !z_in) return MC_EINVAL;
  if (n == 0) return MC_OK;
  mq_stream st = (mq_stream)cuda_stream;
  const int g1 = (int)std::min<uint64_t>(mqk::MAXGRID, (n + mqk::PTS_EVAL - 1) / mqk::PTS_EVAL);
  const int g2 = (int)std::min<uint64_t>(mqk::MAXGRID, (n + mqk::PTS_DD - 1) / mqk::PTS_DD);
  if (f64_out || cond_out || aux_out) { mq_launch_eval_z_f64(d, g1, n, z_in, f64_out, cond_out, aux_out, st); g_launches++; }
  if (fdd_out) { mq_launch_eval_z_dd(d, g2, n, z_in, fdd_out, st); g_launches++; }
  MQ_CK(cudaGetLastError());
  return MC_OK;
}

int mc_eval_z_qd(const mc_diagram *d, uint64_t n, const double *z_in, void *cuda_stream, double *fqd_out) {
  if (!d || !d->on_device || !z_in || !fqd_out) return MC_EINVAL;
  if (n == 0) return MC_OK;
  mq_launch_eval_z_qd(d, n, z_in, fqd_out, (mq_stream)cuda_stream);
  g_launches++;
  MQ_CK(cudaGetLastError());
  return MC_OK;
}

int mc_eval_z_interval(const mc_diagram *d, uint64_t n, const double *z_in, void *cuda_stream, double *lo_out, double *hi_out) {
  if (!d || !d->on_device || !z_in || !lo_out || !hi_out) return MC_EINVAL;
  if (n == 0) return MC_OK;
  if (mq_launch_eval_z_iv(d, n, z_in, lo_out, hi_out, (mq_stream)cuda_stream) != 0) return MC_ECUDA;
  g_launches++;
  return MC_OK;
}

// ---- batched path ----
int mc_batch_create(const mc_diagram *const *diagrams, int32_t n_diagrams, uint64_t max_samples_per_call, mc_batch **out) {
  if (!diagrams || n_diagrams < 1 || !out || max_samples_per_call < 1 || max_samples_per_call > (1ull << 30)) return MC_EINVAL;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return MC_ECUDA;
  mc_batch *b = new (std::nothrow) mc_batch;
  if (!b) return MC_ENOMEM;
  for (int i = 0; i < n_diagrams; i++) {
    if (!diagrams[i] || !diagrams[i]->on_device) { delete b; return MC_EINVAL; }
    b->diags.push_back(diagrams[i]);
    b->scal_len = std::max(b->scal_len, diagrams[i]->max_scal_len);
  }
  const size_t P = mqk::PTS_F64, nd = (size_t)n_diagrams;
  b->cap = (uint32_t)((max_samples_per_call + P - 1) / P * P);
  b->lostcap = std::max<uint32_t>(1024u, b->cap / 8);
  const size_t ipd = b->cap / P, idd = (size_t)b->cap / mqk::PTS_DD + 1, iqd = (size_t)b->lostcap + 1;
  // carve one allocation (every array 256-byte aligned)
  size_t off = 0;
  auto take = [&](size_t bytes) { const size_t o = off; off += (bytes + 255) & ~(size_t)255; return o; };
  const size_t o_dg = take(nd * sizeof(mqk::BatchDiag)), o_cnt = take(nd * ipd * 4), o_raw = take(nd * b->cap * 4), o_list = take(nd * b->cap * 4),
               o_lost = take(nd * b->lostcap * 4), o_nf = take(nd * 8), o_nl = take(nd * 8), o_ndp = take(nd * 8), o_dds = take((nd + 1) * 4),
               o_qds = take((nd + 1) * 4), o_p1 = take(nd * ipd * 32), o_p2 = take(nd * idd * 32), o_p3 = take(nd * iqd * 32), o_q = take(32),
               o_fs = take((nd + 1) * 4), o_vf = take(nd * 8), o_vn = take(nd * 4);
  if (cudaMalloc(&b->d_mem, off) != cudaSuccess) { delete b; return MC_ENOMEM; }
  if (cudaMemset(b->d_mem, 0, off) != cudaSuccess) { mc_batch_free(b); return MC_ECUDA; }
  char *base = (char *)b->d_mem;
  std::vector<mqk::BatchDiag> dg(nd);
  for (size_t i = 0; i < nd; i++) { dg[i].blob = diagrams[i]->d_blob; dg[i].pr = diagrams[i]->prec(false); }
  if (cudaMemcpy(base + o_dg, dg.data(), nd * sizeof(mqk::BatchDiag), cudaMemcpyHostToDevice) != cudaSuccess) { mc_batch_free(b); return MC_ECUDA; }
  mqk::BatchView &v = b->view;
  v.dg = (const mqk::BatchDiag *)(base + o_dg); v.nd = n_diagrams; v.cap = b->cap; v.ipd = 0;
  v.item_cnt = (uint32_t *)(base + o_cnt); v.flag_raw = (uint32_t *)(base + o_raw); v.flag_list = (uint32_t *)(base + o_list);
  v.lost_list = (uint32_t *)(base + o_lost); v.lostcap = b->lostcap;
  v.nflag = (unsigned long long *)(base + o_nf); v.nlost = (unsigned long long *)(base + o_nl); v.ndrop = (unsigned long long *)(base + o_ndp);
  v.dd_start = (uint32_t *)(base + o_dds); v.qd_start = (uint32_t *)(base + o_qds);
  v.part_f64 = (double *)(base + o_p1); v.part_dd = (double *)(base + o_p2); v.part_qd = (double *)(base + o_p3);
  v.queue = (unsigned long long *)(base + o_q);
  v.f64_start = nullptr; v.v_first = nullptr; v.v_n = nullptr;
  b->d_f64_start = (uint32_t *)(base + o_fs); b->d_v_first = (uint64_t *)(base + o_vf); b->d_v_n = (uint32_t *)(base + o_vn);
  b->smem_f64 = mq_batch_smem_f64(b->scal_len); b->smem_dd = mq_batch_smem_dd(b->scal_len); b->smem_qd = mq_batch_smem_qd(b->scal_len);
  if (mq_batch_config_f64(b->smem_f64, &b->grid_f64) != 0 || mq_batch_config_dd(b->smem_dd, &b->grid_dd) != 0 || mq_batch_config_qd(b->smem_qd, &b->grid_qd) != 0) {
    mc_batch_free(b); return MC_ECUDA;
  }
  *out = b;
  return MC_OK;
}
void mc_batch_free(mc_batch *b) {
  if (!b) return;
  if (b->d_mem) cudaFree(b->d_mem);
  delete b;
}
namespace {
// one pass of the three tiers over the sample ranges described by v (uniform: first, n; per diagram: v.f64_start / v_first / v_n)
void batch_pass(mc_batch *b, const mqk::BatchView &v, uint64_t items, uint64_t first, uint64_t n, uint64_t seed, uint32_t flags, mq_stream st,
                double *out_sum, double *out_sumsq, unsigned long long *out_n_flagged, unsigned long long *out_n_dropped) {
  const bool no_dd = flags & 1u, no_qd = flags & 2u;
  mq_launch_batch_f64(v, (int)std::min<uint64_t>((uint64_t)b->grid_f64, items), b->smem_f64, first, n, seed, b->scal_len, no_dd ? 1 : 0, st);
  mq_launch_batch_compact(v, st);
  g_launches += 2;
  if (!no_dd) {
    mq_launch_batch_ranges(v, 1, st);
    mq_launch_batch_dd(v, b->grid_dd, b->smem_dd, first, seed, b->scal_len, st);
    g_launches += 2;
    if (!no_qd) {
      mq_launch_batch_ranges(v, 2, st);
      mq_launch_batch_qd(v, b->grid_qd, b->smem_qd, first, seed, b->scal_len, st);
      g_launches += 2;
    }
  }
  mq_launch_batch_finish(v, no_dd ? 1 : no_qd ? 2 : 3, out_sum, out_sumsq, out_n_flagged, out_n_dropped, st);
  g_launches++;
}
}  // namespace

int mc_batch_integrate(mc_batch *b, uint64_t first_sample, uint64_t n_samples, uint64_t seed, uint32_t flags, void *cuda_stream,
                       double *out_sum, double *out_sumsq, unsigned long long *out_n_flagged, unsigned long long *out_n_dropped) {
  if (!b) return MC_EINVAL;
  for (const mc_diagram *d : b->diags) if (!rng_range_ok(d, first_sample, n_samples)) return MC_EINVAL;
  mq_stream st = (mq_stream)cuda_stream;
  for (uint64_t done = 0; done < n_samples; done += b->cap) {
    const uint64_t n = std::min<uint64_t>(b->cap, n_samples - done);
    mqk::BatchView v = b->view;
    v.ipd = (uint32_t)((n + mqk::PTS_F64 - 1) / mqk::PTS_F64);
    batch_pass(b, v, (uint64_t)v.ipd * v.nd, first_sample + done, n, seed, flags, st, out_sum, out_sumsq, out_n_flagged, out_n_dropped);
  }
  MQ_CK(cudaGetLastError());
  return MC_OK;
}

int mc_batch_integrate_counts(mc_batch *b, const uint64_t *first_sample, const uint64_t *n_samples, uint64_t seed, uint32_t flags, void *cuda_stream,
                              double *out_sum, double *out_sumsq, unsigned long long *out_n_flagged, unsigned long long *out_n_dropped) {
  if (!b || !first_sample || !n_samples) return MC_EINVAL;
  cudaStream_t cst = (cudaStream_t)cuda_stream;
  const size_t nd = b->diags.size();
  uint64_t longest = 0;
  for (size_t d = 0; d < nd; d++) { longest = std::max(longest, n_samples[d]); if (!rng_range_ok(b->diags[d], first_sample[d], n_samples[d])) return MC_EINVAL; }
  std::vector<uint32_t> start(nd + 1), vn(nd);
  std::vector<uint64_t> vf(nd);
  for (uint64_t done = 0; done < longest; done += b->cap) {        // diagrams whose range is longer than the capacity take several passes
    uint64_t items = 0;
    for (size_t d = 0; d < nd; d++) {
      const uint64_t left = n_samples[d] > done ? n_samples[d] - done : 0, n = std::min<uint64_t>(b->cap, left);
      start[d] = (uint32_t)items; vn[d] = (uint32_t)n; vf[d] = first_sample[d] + done;
      items += (n + mqk::PTS_F64 - 1) / mqk::PTS_F64;
    }
    if (items > 0xFFFFFFFFull) return MC_EINVAL;
    start[nd] = (uint32_t)items;
    if (items == 0) continue;
    MQ_CK(cudaMemcpyAsync(b->d_f64_start, start.data(), (nd + 1) * 4, cudaMemcpyHostToDevice, cst));
    MQ_CK(cudaMemcpyAsync(b->d_v_first, vf.data(), nd * 8, cudaMemcpyHostToDevice, cst));
    MQ_CK(cudaMemcpyAsync(b->d_v_n, vn.data(), nd * 4, cudaMemcpyHostToDevice, cst));
    MQ_CK(cudaStreamSynchronize(cst));                              // the host vectors are reused by the next pass
    mqk::BatchView v = b->view;
    v.ipd = 0; v.f64_start = b->d_f64_start; v.v_first = b->d_v_first; v.v_n = b->d_v_n;
    batch_pass(b, v, items, 0, 0, seed, flags, (mq_stream)cuda_stream, out_sum, out_sumsq, out_n_flagged, out_n_dropped);
  }
  MQ_CK(cudaGetLastError());
  return MC_OK;
}

/* N_j ~ sigma_j / sqrt(cost_j): the split of a total cost budget that minimises sum_j sigma_j^2 / N_j (Neyman allocation with
 * unequal costs); every diagram gets at least n_min samples. sigma_j = the per-sample standard deviation of the weight. */
int mc_allocate_samples(const double *sigma, const double *cost, int32_t n_diagrams, double budget, uint64_t n_min, uint64_t *n_out) {
  if (!sigma || !cost || !n_out || n_diagrams < 1 || !(budget > 0)) return MC_EINVAL;
  double norm = 0;
  for (int j = 0; j < n_diagrams; j++) { if (!(cost[j] > 0) || !(sigma[j] >= 0)) return MC_EINVAL; norm += sigma[j] * std::sqrt(cost[j]); }
  for (int j = 0; j < n_diagrams; j++) {
    const double n = norm > 0 ? budget * sigma[j] / (std::sqrt(cost[j]) * norm) : budget / (cost[j] * n_diagrams);
    n_out[j] = std::max<uint64_t>(n_min, (uint64_t)std::llround(n));
  }
  return MC_OK;
}

int mc_batch_integrate_host(mc_batch *b, uint64_t first_sample, uint64_t n_samples, uint64_t seed, uint32_t flags, void *cuda_stream,
                            double *sum, double *sumsq, unsigned long long *n_flagged, unsigned long long *n_dropped) {
  if (!b) return MC_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t nd = b->diags.size();
  char *dev = nullptr;
  MQ_CK(cudaMallocAsync((void **)&dev, nd * 32, st));
  double *ds = (double *)dev, *ds2 = ds + nd; unsigned long long *dnf = (unsigned long long *)(ds2 + nd), *dnd = dnf + nd;
  // every exit after the allocation goes through the free below
  int rc = cudaMemsetAsync(dev, 0, nd * 32, st) == cudaSuccess ? MC_OK : MC_ECUDA;
  if (rc == MC_OK) rc = mc_batch_integrate(b, first_sample, n_samples, seed, flags, cuda_stream, ds, ds2, dnf, dnd);
  auto back = [&](void *dst, const void *src) { if (rc == MC_OK && dst && cudaMemcpyAsync(dst, src, nd * 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) rc = MC_ECUDA; };
  back(sum, ds); back(sumsq, ds2); back(n_flagged, dnf); back(n_dropped, dnd);
  if (cudaFreeAsync(dev, st) != cudaSuccess && rc == MC_OK) rc = MC_ECUDA;
  if (cudaStreamSynchronize(st) != cudaSuccess && rc == MC_OK) rc = MC_ECUDA;
  return rc;
}

unsigned long long mc_kernel_launch_count(void) { return g_launches.load(); }

int mc_fp64_peak(int iters, void *cuda_stream, double *flops, double *ms) {
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return MC_ECUDA;
  if (mq_fp64_peak(iters, (mq_stream)cuda_stream, flops, ms) != 0) return MC_ECUDA;
  g_launches += 2;
  return MC_OK;
}

const char *mc_strerror(int code) {
  switch (code) {
    case MC_OK: return "ok";
    case MC_EINVAL: return "invalid argument or not a valid 1PI vertex graph";
    case MC_ENOMEM: return "out of memory";
    case MC_ECUDA: return "CUDA error or no CUDA device (this library has no CPU fallback)";
    case MC_ELIMIT: return "graph exceeds a compiled-in limit";
    case MC_ETOOBIG: return "n_samples exceeds MC_STATIC_MAX_SAMPLES, the capacity of the static scratch of mc_integrate_static (split the range)";
  }
  return "unknown error";
}
const char *mc_version(void) { return "mcqed-b200 0.1 (sm_100a)"; }

}  // extern "C"
