// diagram.hpp — the object behind mc_diagram* and the host-callable launchers of the kernels.
// Product code (libmcqed.so); shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <vector>

#include "../../include/mcqed.h"
#include "device_layout.h"
#include "host_model.hpp"

namespace mqk {
// binary64 tier: a lane carries NP_F64 sample points (pt2_arith.cuh: every loaded table coefficient feeds NP_F64 FMAs)
#ifndef MQ_NP
#define MQ_NP 4
#endif
#ifndef MQ_TPB_F64
#define MQ_TPB_F64 128
#endif
#ifndef MQ_MINB_F64
#define MQ_MINB_F64 2
#endif
#ifndef MQ_TPB_DD
#define MQ_TPB_DD 128
#endif
constexpr int NP_F64 = MQ_NP;    // 1, 2 or 4
constexpr int TPB_F64 = MQ_TPB_F64, TPB_DD = MQ_TPB_DD, TPB_EVAL = 128;
// warp split (mcqed_kernels.cuh): W warps share one group of points. Measured on B200 before the lane split existed
// (profiles/r1_summary.md): W = 2 doubles the resident warps but is slower than W = 1 (binary64 11.9 % vs 13.5 % of peak on a
// subtraction-free graph; double-double 2.6e5 vs 4.2e5 points/s on a 12-term graph), so W = 1; the lane split (MQ_WL lanes of a
// warp per point, device_layout.h) is what doubles the resident warps now.
constexpr int W_F64 = 1, W_DD = 1;
constexpr int PTS_F64 = TPB_F64 / (W_F64 * MQ_WL) * NP_F64, PTS_DD = TPB_DD / (W_DD * MQ_WL), PTS_EVAL = TPB_EVAL / (W_F64 * MQ_WL) * NP_F64;   // points per CTA (MQ_WL lanes share NP points)
constexpr uint64_t CHUNK = 1ull << 22;     // samples per launch (bounds the flagged-index list)
constexpr int MAXGRID = 148 * 32;
// precision policy of one diagram as the kernels see it (O8; include/mcqed.h mc_diagram_set_precision)
struct MqPrec { double cond_max, amin_min, dd_cond_max, w_abs_tol; };
constexpr uint64_t LOSTCAP = CHUNK / 8;   // capacity of the list of points handed from double-double to quad-double
}  // namespace mqk

struct McWorkspace {
  double *partial = nullptr;               // [3][MAXGRID][4] per-block compensated partial sums (f64, dd, qd pass)
  unsigned long long *lost_list = nullptr; // [LOSTCAP] points the double-double pass could not resolve
  unsigned long long *flag_list = nullptr; // [CHUNK] sample indices flagged in the current chunk
  unsigned long long *counters = nullptr;  // [4]: flagged in chunk, dropped, handed to quad-double, -
};

struct mc_diagram {
  mq::VertexGraph g;
  mq::ForestTerms ft;
  mq::SamplerTables st, st2;               // st2: the second channel of the defensive mixture (empty when off)
  mc_options opt{};
  double dd_cond_max = 1e26, w_abs_tol = 1e-10;   // mc_diagram_set_precision
  mqk::MqPrec prec(bool no_dd) const {    // no_dd: nothing but non-finite points is handed on
    return no_dd ? mqk::MqPrec{1e300, -1.0, dd_cond_max, w_abs_tol} : mqk::MqPrec{opt.cond_max, opt.amin_min, dd_cond_max, w_abs_tol};
  }
  int id = -1;
  std::vector<uint64_t> blob;              // host copy of the device blob (device_layout.h)
  std::vector<DevGeom> geoms; std::vector<DevTable> tables; std::vector<DevNode> nodes; std::vector<DevTerm> terms;
  int64_t n_stored = 0, n_nonzero = 0;
  int max_scal_len = 0, nodeval_len = 0;
  bool have_tables = false;
  // device side
  uint64_t *d_blob = nullptr;
  McWorkspace ws;
  bool on_device = false;
  int grid_f64 = 0, grid_dd = 0, grid_qd = 0;
  size_t smem_f64 = 0, smem_dd = 0, smem_eval = 0, smem_qd = 0;
};

// the object behind mc_batch*: a set of prepared diagrams integrated together by one persistent launch per precision tier
namespace mqk {
struct BatchDiag {
  const uint64_t *blob;
  MqPrec pr;
};
struct BatchView {
  const BatchDiag *dg;             // [nd]
  int nd; uint32_t cap;            // diagrams; capacity (points per diagram per call, multiple of PTS_F64)
  uint32_t ipd;                    // binary64 items per diagram in this call (uniform calls: every diagram gets the same range)
  // per-diagram sample ranges (mc_batch_integrate_counts; nullptr in a uniform call): first item, first sample index, samples
  const uint32_t *f64_start;       // [nd+1]
  const uint64_t *v_first;         // [nd]
  const uint32_t *v_n;             // [nd]
  uint32_t *item_cnt;              // [nd*cap/PTS_F64] flagged points of a binary64 item
  uint32_t *flag_raw;              // [nd*cap] item-local lists (relative sample indices), entry b*PTS_F64+k of diagram d
  uint32_t *flag_list;             // [nd*cap] compacted, ascending
  uint32_t *lost_list;             // [nd*lostcap] handed from double-double to quad-double
  uint32_t lostcap;
  unsigned long long *nflag, *nlost, *ndrop;   // [nd]
  uint32_t *dd_start, *qd_start;   // [nd+1] first item of diagram d in the double-double / quad-double pass
  double *part_f64, *part_dd, *part_qd;        // [items][4]
  unsigned long long *queue;       // [4] heads of the three work queues
};
}  // namespace mqk
struct mc_batch {
  std::vector<const mc_diagram *> diags;
  uint32_t cap = 0, lostcap = 0;           // points per diagram per call (multiple of PTS_F64); quad-double list capacity
  int scal_len = 0;                        // max over the diagrams: fixes the shared-memory layout of the batch kernels
  int grid_f64 = 0, grid_dd = 0, grid_qd = 0;
  size_t smem_f64 = 0, smem_dd = 0, smem_qd = 0;
  void *d_mem = nullptr;                   // one device allocation holding every array of BatchView
  uint32_t *d_f64_start = nullptr; uint64_t *d_v_first = nullptr; uint32_t *d_v_n = nullptr;   // inside d_mem (per-diagram ranges)
  mqk::BatchView view{};                   // the kernel argument (pointers into d_mem)
};

// host preparation (host_prepare.cpp)
// use_gpu: count the gamma-string paths of the numerator tables with the CUDA kernel of prep_kernel.cu
int mq_prepare_host(const mc_graph *graph, const mc_forests *uf, const mc_options *opts, bool use_gpu, mc_diagram **out);
int mq_count_units_gpu(const MqCountUnit *units, size_t nunits, int32_t *counts, size_t nints);

// launchers (kern_f64.cu / kern_dd.cu); every one returns a cudaError_t cast to int
typedef struct CUstream_st *mq_stream;
int mq_config_f64(mc_diagram *d);
int mq_config_dd(mc_diagram *d);
int mq_config_qd(mc_diagram *d);
void mq_launch_integrate_qd(const mc_diagram *d, uint64_t seed, mq_stream st);
void mq_launch_eval_points_qd(const mc_diagram *d, uint64_t first, uint64_t seed, double *f_out, mq_stream st);
void mq_launch_eval_z_qd(const mc_diagram *d, uint64_t n, const double *z_in, double *fqd_out, mq_stream st);
void mq_launch_integrate_f64(const mc_diagram *d, int grid, uint64_t first, uint64_t n, uint64_t seed, mqk::MqPrec pr, mq_stream st);
void mq_launch_integrate_dd(const mc_diagram *d, uint64_t seed, mq_stream st);
void mq_launch_finish(const mc_diagram *d, int nb1, int nb2, int nb3, double *out_sum, double *out_sumsq, unsigned long long *out_nflag, unsigned long long *out_ndrop, mq_stream st);
void mq_launch_reset(const mc_diagram *d, mq_stream st);
void mq_launch_eval_points(const mc_diagram *d, int grid, uint64_t first, uint64_t n, uint64_t seed, mqk::MqPrec pr,
                           double *z_out, int32_t *order_out, double *p_out, double *f_out, double *f64_out, double *cond_out,
                           uint8_t *flag_out, bool list_flagged, mq_stream st);
void mq_launch_eval_points_dd(const mc_diagram *d, uint64_t first, uint64_t seed, double *f_out, mq_stream st);
void mq_launch_eval_z_f64(const mc_diagram *d, int grid, uint64_t n, const double *z_in, double *f64_out, double *cond_out, double *aux_out, mq_stream st);
void mq_launch_eval_z_dd(const mc_diagram *d, int grid, uint64_t n, const double *z_in, double *fdd_out, mq_stream st);
int mq_fp64_peak(int iters, mq_stream st, double *flops, double *ms);
// interval tier (kern_iv.cu): enclosure [lo, hi] of the integrand at given points
int mq_launch_eval_z_iv(const mc_diagram *d, uint64_t n, const double *z_in, double *lo_out, double *hi_out, mq_stream st);
// binary64 tier with the scratch in a file-scope device array (kern_f64.cu); allocates nothing
int mq_static_integrate_f64(const mc_diagram *d, uint64_t first, uint64_t n, uint64_t seed, mqk::MqPrec pr,
                            double *out_sum, double *out_sumsq, unsigned long long *out_nflag, unsigned long long *out_ndrop, mq_stream st);
// batched path (kern_f64.cu / kern_dd.cu / kern_qd.cu)
size_t mq_batch_smem_f64(int scal_len); size_t mq_batch_smem_dd(int scal_len); size_t mq_batch_smem_qd(int scal_len);
int mq_batch_config_f64(size_t smem, int *grid); int mq_batch_config_dd(size_t smem, int *grid); int mq_batch_config_qd(size_t smem, int *grid);
void mq_launch_batch_f64(const mqk::BatchView &bv, int grid, size_t smem, uint64_t first, uint64_t n, uint64_t seed, int scal_len, int no_dd, mq_stream st);
void mq_launch_batch_compact(const mqk::BatchView &bv, mq_stream st);
void mq_launch_batch_ranges(const mqk::BatchView &bv, int tier, mq_stream st);
void mq_launch_batch_dd(const mqk::BatchView &bv, int grid, size_t smem, uint64_t first, uint64_t seed, int scal_len, mq_stream st);
void mq_launch_batch_qd(const mqk::BatchView &bv, int grid, size_t smem, uint64_t first, uint64_t seed, int scal_len, mq_stream st);
void mq_launch_batch_finish(const mqk::BatchView &bv, int tiers, double *out_sum, double *out_sumsq, unsigned long long *out_nflag, unsigned long long *out_ndrop, mq_stream st);
