/* include/mcqed.h — C ABI of libmcqed.so: the data-parallel Monte Carlo hot path of
 * S. Volkov, "Numerical calculation of 5-loop QED contributions to the electron anomalous magnetic
 * moment" (arXiv:1905.08007; PAPER.md), hand-written CUDA for sm_100a.
 *
 * The path (PAPER.md:9-13 items (i)-(iii)): for one Feynman graph without lepton loops
 * and per sample point
 *   a1-a3  draw z on the simplex from the graph's own Hepp-sector density, Eq.(1),
 *          with a Philox4x32-10 counter stream;
 *   a4     build the loop matrix of every piece of every forest term and derive U, B_ij/U, the
 *          scalar currents and V in binary64;
 *   a5-a6  evaluate the Feynman-parametric integrand together with every subtraction term of the
 *          forest-like formula so that IR and UV divergences cancel point by point;
 *   a7     weight by f/p and accumulate sum and sum of squares;
 *   a8     re-evaluate points flagged for round-off in double-double.
 * Every step runs in CUDA kernels of this library; there is no CPU fallback: every entry point
 * that touches the device returns MC_ECUDA when no CUDA device / driver is usable.
 *
 * Conventions. All functions return 0 (MC_OK) or a negative error code; nothing throws across the
 * boundary. Global state: the launch counter behind mc_kernel_launch_count and the static scratch of
 * mc_integrate_static, nothing else. A handle (mc_diagram, mc_batch) owns device scratch that every
 * device call on it writes (partial sums, flagged lists, counters): introspection calls may run concurrently,
 * but at most ONE device call (mc_integrate*, mc_eval_*, mc_batch_integrate*) per handle may be in flight at a
 * time — calls on one stream are ordered and safe, calls on the same handle from two streams or threads race on
 * the scratch and return wrong sums without an error. Distinct handles are independent.
 * "HOST" / "DEVICE" says where a pointer must live. Line index convention (R1): electron line t (joining path
 * positions t,t+1) has index t, photon i (chords sorted by their first end) has index 2L+i; M=3L.
 */
#ifndef MCQED_H
#define MCQED_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define MC_OK 0
#define MC_EINVAL (-1)  /* not a valid graph (no perfect matching, chord on the external vertex, a line not
                           covered => not 1PI), bad argument, user forests disagree with the enumeration */
#define MC_ENOMEM (-2)
#define MC_ECUDA (-3)   /* CUDA runtime error or no device */
#define MC_ELIMIT (-4)  /* graph exceeds a compiled-in limit */
#define MC_ETOOBIG (-5) /* n_samples exceeds the capacity of the static scratch of mc_integrate_static */

typedef struct mc_diagram mc_diagram; /* opaque; owns its host and device tables */

/* A vertex graph without lepton loops: an open electron path with positions
 * 0..2*loops; position ext_pos carries the external photon; the other positions are joined in
 * pairs by `loops` photon chords. HOST, caller-owned, read during the call only. */
typedef struct {
  int32_t loops;                  /* L, 1..5 */
  int32_t ext_pos;                /* e, 1..2L-1 */
  int32_t chord_a[5], chord_b[5]; /* chord ends, any order; must form a perfect matching of the positions != e */
} mc_graph;

/* Optional cross-check of the UV-divergent subgraphs and forests. NULL => the
 * library enumerates them itself. If given, they must equal the library's own enumeration
 * (subgraphs ascending (lo,hi); forests = ascending bitmasks over the subgraphs, the empty forest
 * included), else MC_EINVAL. HOST. */
typedef struct {
  int32_t n_sub; const int32_t *seg_lo, *seg_hi;
  int32_t n_forest; const uint32_t *forest_mask;
} mc_forests;

/* NULL => defaults {1.0, 1e30, 2.8e4, 1e-2, 0, 0.5, 0, 0, 0}. deg_floor/deg_cap clamp Deg(s) of Eq.(1) (S5); deg_floor_ir is the
 * value of Deg on the sets whose I-closure is the whole graph, the soft-photon sets (<= 0: same as deg_floor).
 * cond_max, amin_min: thresholds of the relative acceptance test of the binary64 tier; the full precision policy
 *   (relative or absolute acceptance, three tiers) is stated at mc_diagram_set_precision.
 * flags bit 0: never run the double-double pass (only non-finite points are then flagged; they contribute 0).
 * flags bit 1: build no numerator tables (introspection of the combinatorics only; host handles).
 * flags bit 2: the random stream is MRG32k3a (the generator of the paper's "Calc 1") instead of Philox4x32-10
 *   (PAPER.md:94): the initial state is (1 + seed_lo mod (m-1), 1 + seed_hi mod (m-1), 12345) in both components, sample index i
 *   of diagram id owns the 64 outputs from position (id * 2^38 + i) * 64 of the sequence, and uniform number r of the sample is
 *   made from outputs 2r, 2r+1 with the 52-bit construction used for Philox (S1b). Calls with disjoint sample ranges stay
 *   independent and additive. Fixed at prepare time (mc_diagram_set_flags cannot change it); sample indices must stay below 2^38
 *   (MC_EINVAL beyond) and the diagram id below 2^20 (MC_ELIMIT). */
typedef struct {
  double deg_floor, deg_cap, cond_max, amin_min; uint32_t flags; double deg_floor_ir;
  /* Defensive mixture (S5b; a READING: the paper has one density). mix_alpha in (0, 1): with
   * probability mix_alpha (decided by uniform number 2(M-1) of the sample) the point is drawn from a SECOND Eq.(1) density built with
   * the floors (deg_floor2, deg_floor_ir2; <= 0: same as deg_floor2) and the same cap, and the density every weight is divided by is
   * (1 - mix_alpha) p_first(z) + mix_alpha p_second(z): a weight is bounded by the better of the two channels. 0 = off (default). */
  double mix_alpha, deg_floor2, deg_floor_ir2;
} mc_options;

/* Host-side preparation of one diagram (not on the timed path): validates the graph, enumerates
 * subgraphs/forests/terms (forest-like formula, O1), builds Deg and the sector-sum table
 * (Eq.(1)), the numerator tables of every piece, and uploads them to the current CUDA device.
 * *out is owned by the caller and released with mc_free_diagram. */
int mc_prepare_diagram(const mc_graph *graph, const mc_forests *forests, const mc_options *opts, mc_diagram **out);

/* Same as mc_prepare_diagram but builds host tables only (no CUDA call): for introspection and CPU
 * tests of the host logic. Such a handle is rejected (MC_EINVAL) by mc_integrate / mc_eval_points. */
int mc_prepare_diagram_host(const mc_graph *graph, const mc_forests *forests, const mc_options *opts, mc_diagram **out);

void mc_free_diagram(mc_diagram *);

/* Class (k,m,n) of PAPER.md:104; number of formula terms; algorithmic flop per sample point
 * (2 per stored numerator monomial + the a1-a4,a6 estimate of DESIGN.md §5); device table bytes.
 * Any output pointer may be NULL. HOST. */
int mc_diagram_info(const mc_diagram *, int32_t *k, int32_t *m, int32_t *n, int32_t *n_terms,
                    int64_t *flop_per_sample, int64_t *table_bytes);

/* Canonical index of the graph among the valid graphs of its loop order (ascending e, then
 * lexicographic sorted chord list; A19) — it is the 4th Philox counter word. */
int mc_diagram_id(const mc_diagram *, int32_t *id);

/* Introspection (HOST outputs, caller-allocated, any may be NULL; returns the count):
 * subgraphs (lo,hi,type 0=S/1=V), forests (bitmasks), terms (forest, gprime index or -1, sign). */
int mc_diagram_subgraphs(const mc_diagram *, int32_t *lo, int32_t *hi, int32_t *type, int32_t cap);
int mc_diagram_forests(const mc_diagram *, uint32_t *mask, int32_t cap);
int mc_diagram_terms(const mc_diagram *, uint32_t *forest, int32_t *gprime, int32_t *sign, int32_t cap);
/* Sampler tables of Eq.(1): deg and Z have 2^M entries, C is the normalisation. HOST outputs. */
int mc_diagram_sampler_tables(const mc_diagram *, double *deg, double *Z, double *C);

/* Changes the run-time flag bits of mc_options.flags on an existing handle (bit 0: skip the double-double
 * pass). Used by bench.py to time the binary64 kernel alone. HOST. */
int mc_diagram_set_flags(mc_diagram *, uint32_t flags);

/* Precision policy of an existing handle (O8; "interval arithmetic ... with different precisions":
 * the paper gives no thresholds). Every tier carries next to f a running bound a on the sum of |monomial| (it sees the
 * cancellation between terms, pieces, families, pairings and inside a coefficient block), amin = the smallest |A_t| and
 * xmin = the smallest pivot ratio / g_t of the point. A tier's value is ACCEPTED if
 *   (relative) a <= cond * |f| * min(1, amin, xmin) and min(amin, xmin) >= inner_min, with (cond, inner_min) = (cond_max, amin_min)
 *              in binary64 (cond_max = 2.8e4 = 1e-10 / unit: the round-off model unit * a / min(1, amin, xmin) is below 1e-10 |f|)
 *              and (dd_cond_max, 1/dd_cond_max) in double-double, or
 *   (absolute) unit * a <= w_abs_tol * p * min(1, xmin), unit = 32 ulp of the tier's arithmetic (64 in double-double): the
 *              round-off bound on the WEIGHT w = f/p is below w_abs_tol. The Monte Carlo sums need absolute accuracy of the
 *              weights; deep in the corners of the simplex the subtracted integrand loses all relative precision while f/p
 *              is 1e-20 and smaller.
 * Otherwise the point goes to the next tier (binary64 -> double-double -> quad-double). Defaults: cond_max = 2.8e4, amin_min =
 * 1e-2 (mc_options); dd_cond_max = 1e26; w_abs_tol = 1e-10 (0 switches the absolute criterion off). A batch copies the
 * values when it is created. HOST. MC_EINVAL on cond_max <= 0, dd_cond_max < 1, w_abs_tol < 0. */
int mc_diagram_set_precision(mc_diagram *, double cond_max, double amin_min, double dd_cond_max, double w_abs_tol);

/* Host copy of the device table blob (layout: csrc/device_layout.h), for format tests. Returns the
 * number of 8-byte words; copies min(words, cap) words into out (may be NULL). HOST. */
int64_t mc_diagram_blob(const mc_diagram *, uint64_t *out, int64_t cap);

/* The hot path. Processes sample indices first_sample .. first_sample+n_samples-1 of this diagram
 * (the Philox counter is the sample index, so calls with disjoint ranges are independent and
 * additive: that is also the checkpoint/resume story). Asynchronous on `cuda_stream`
 * (a cudaStream_t; NULL = legacy default stream). out_* are DEVICE pointers, one element each,
 * accumulated into (+=): sum of w=f/p, sum of w^2, number of points re-evaluated in double-double (those
 * double-double cannot resolve either go on to quad-double), number of points dropped because some z
 * underflowed or even the quad-double value was non-finite (their w is 0). */
int mc_integrate(const mc_diagram *, uint64_t first_sample, uint64_t n_samples, uint64_t seed, void *cuda_stream,
                 double *out_sum, double *out_sumsq, unsigned long long *out_n_flagged, unsigned long long *out_n_dropped);

/* Same computation with HOST outputs: allocates nothing persistent, copies the four results back
 * and synchronises the stream. For end-to-end use without touching device memory. */
int mc_integrate_host(const mc_diagram *, uint64_t first_sample, uint64_t n_samples, uint64_t seed, void *cuda_stream,
                      double *sum, double *sumsq, unsigned long long *n_flagged, unsigned long long *n_dropped);

/* The binary64 tier of mc_integrate (steps a1-a7) for callers that cannot allocate: code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc. Same kernels and launch configuration as mc_integrate on
 * a handle with flags bit 0 set (no double-double pass: only points with a non-finite value or an underflowed coordinate are
 * flagged; they contribute 0 and are counted in out_n_flagged), so the results are the same numbers. The per-call scratch
 * (per-block partial sums, the flagged-index list, counters) lives in a file-scope `static __device__` array of the library
 * instead of device memory owned by the handle: every GPU that loads the library holds MC_STATIC_SCRATCH_BYTES (0.65 MiB)
 * until the process exits. The call makes no cudaMalloc / cudaFree / allocating library call. The first call on a device
 * resolves the array's device address (cudaGetSymbolAddress, once per device, with that device current): make it outside
 * stream capture. n_samples must not exceed MC_STATIC_MAX_SAMPLES (the flagged list holds one entry per sample in the worst
 * case): MC_ETOOBIG otherwise, nothing launched; split longer ranges into several calls (results are additive).
 * Every call on a device shares the one array, which keeps the last call's contents (the counters are cleared on the stream
 * at the start of each call): calls whose kernels can overlap on the GPU (different streams, threads or processes sharing the
 * context) race on it and give wrong sums without an error; calls on one stream are ordered and safe.
 * out_* are DEVICE pointers, one element each, accumulated into (+=), any may be NULL. Asynchronous on cuda_stream.
 * Errors: MC_EINVAL (NULL or host-only handle), MC_ETOOBIG, MC_ECUDA. */
#define MC_STATIC_MAX_SAMPLES 65536
#define MC_STATIC_SCRATCH_BYTES (256 + 32 * 148 * 32 + 8 * MC_STATIC_MAX_SAMPLES)
int mc_integrate_static(const mc_diagram *, uint64_t first_sample, uint64_t n_samples, uint64_t seed, void *cuda_stream,
                        double *out_sum, double *out_sumsq, unsigned long long *out_n_flagged, unsigned long long *out_n_dropped);

/* Batched form of the hot path: the same computation as mc_integrate for EVERY diagram of a set, with one
 * persistent kernel launch per precision tier for the whole set instead of four launches per diagram. The
 * paper's workload is a sum over thousands of graphs (Table 1 :112-124): per-diagram launches
 * leave the GPU idle in the tail of every launch (a point costs up to milliseconds in double-double), a set-wide
 * work queue has one tail per call. Work items are CTA-loads of points of one diagram; results do not depend on
 * which CTA ran which item (per-item compensated partial sums, added in item order).
 *   mc_batch_create: diagrams = HOST array of n_diagrams device-prepared handles (they must outlive the batch);
 *     max_samples_per_call bounds n_samples of one pass (longer calls are split); allocates the device work space
 *     (about 8 bytes per diagram and sample of one pass).
 *   mc_batch_integrate: sample indices first_sample .. first_sample+n_samples-1 of every diagram (each with its own
 *     diagram id in the Philox counter, as in mc_integrate). out_* are DEVICE arrays of n_diagrams elements,
 *     accumulated into (+=); any may be NULL. flags bit 0: skip the double-double / quad-double passes (flagged
 *     points then contribute 0; used to time the binary64 kernel alone); bit 1: skip the quad-double pass only (its
 *     points contribute 0 and are counted as dropped). Asynchronous on cuda_stream.
 *   mc_batch_integrate_host: same with HOST output arrays (n_diagrams each; overwritten, not accumulated);
 *     synchronises the stream.
 * Errors: MC_EINVAL (NULL / host-only handle, n_diagrams < 1, max_samples_per_call 0 or > 2^30), MC_ENOMEM, MC_ECUDA. */
typedef struct mc_batch mc_batch;
int mc_batch_create(const mc_diagram *const *diagrams, int32_t n_diagrams, uint64_t max_samples_per_call, mc_batch **out);
int mc_batch_integrate(mc_batch *, uint64_t first_sample, uint64_t n_samples, uint64_t seed, uint32_t flags, void *cuda_stream,
                       double *out_sum, double *out_sumsq, unsigned long long *out_n_flagged, unsigned long long *out_n_dropped);
int mc_batch_integrate_host(mc_batch *, uint64_t first_sample, uint64_t n_samples, uint64_t seed, uint32_t flags, void *cuda_stream,
                            double *sum, double *sumsq, unsigned long long *n_flagged, unsigned long long *n_dropped);
void mc_batch_free(mc_batch *);

/* Sample allocation across the graphs of a set (the deliverable is a sum over thousands of graphs whose
 * individual errors differ by orders of magnitude; the paper does not disclose its allocation).
 *   mc_batch_integrate_counts: as mc_batch_integrate, but diagram j processes sample indices first_sample[j] ..
 *     first_sample[j] + n_samples[j] - 1 (HOST arrays of n_diagrams elements; n_samples[j] may be 0; ranges longer than the
 *     batch capacity are split into passes). The arrays are copied to the device at the start of every pass (synchronises
 *     the stream once per pass); outputs as in mc_batch_integrate (DEVICE, accumulated into).
 *   mc_allocate_samples: the split of a cost budget sum_j n_j cost_j = budget that minimises sum_j sigma_j^2 / n_j:
 *     n_j ~ sigma_j / sqrt(cost_j), at least n_min each. sigma_j: per-sample standard deviation of the weight of diagram j (from
 *     a pilot pass), cost_j: cost per sample in any unit (e.g. flop_per_sample of mc_diagram_info). HOST arrays. */
int mc_batch_integrate_counts(mc_batch *, const uint64_t *first_sample, const uint64_t *n_samples, uint64_t seed, uint32_t flags,
                              void *cuda_stream, double *out_sum, double *out_sumsq, unsigned long long *out_n_flagged,
                              unsigned long long *out_n_dropped);
int mc_allocate_samples(const double *sigma, const double *cost, int32_t n_diagrams, double budget, uint64_t n_min, uint64_t *n_out);

/* Parity hook: per-point values for comparison with the oracle. DEVICE outputs, any may be NULL:
 * z_out n*M (row = point, column = line index), order_out n*M (the Hepp sector j_1..j_M),
 * p_out n (density), f_out n (value used by mc_integrate: binary64, or double-double rounded to
 * binary64 if re-evaluated), f64_out n (plain binary64 value), cond_out n (a/|f|), flag_out n: 0 = accepted by the
 * relative bound, 1 = re-evaluated in double-double (or beyond), 2 = precision loss detected but accepted by the absolute
 * bound on the weight (mc_diagram_set_precision). */
int mc_eval_points(const mc_diagram *, uint64_t first_sample, uint64_t n, uint64_t seed, void *cuda_stream,
                   double *z_out, int32_t *order_out, double *p_out, double *f_out, double *f64_out,
                   double *cond_out, uint8_t *flag_out);

/* Integrand at caller-supplied points (DEVICE z_in n*M): f64_out, fdd_out (double-double evaluation
 * rounded to binary64), cond_out (a/|f|, a = the running bound on the sum of |monomial|), aux_out n*2 (amin = min |A_t|;
 * xmin = min over pieces of pivot/diagonal ratio and g_t = 1 + A_t); any output may be NULL. */
int mc_eval_z(const mc_diagram *, uint64_t n, const double *z_in, void *cuda_stream,
              double *f64_out, double *fdd_out, double *cond_out, double *aux_out);

/* Integrand at caller-supplied points in the third precision tier (quad-double, ~212 bits), rounded to binary64.
 * DEVICE z_in n*M, DEVICE fqd_out n. */
int mc_eval_z_qd(const mc_diagram *, uint64_t n, const double *z_in, void *cuda_stream, double *fqd_out);

/* Integrand at caller-supplied points in binary64 INTERVAL arithmetic with directed rounding (the paper controls
 * round-off by interval arithmetic): [lo_out[i], hi_out[i]] contains the true value of the subtracted integrand at the binary64
 * coordinates z_in[i] (table coefficients are exact), whatever the cancellation between the terms; (-inf, +inf) when an interval
 * division met 0. The width tells how much binary64 can be trusted at the point; the library's own precision decision uses the
 * cheaper bound of mc_diagram_set_precision, this call is the rigorous cross-check (about the cost of a double-double evaluation).
 * DEVICE z_in n*M, DEVICE lo_out, hi_out n. */
int mc_eval_z_interval(const mc_diagram *, uint64_t n, const double *z_in, void *cuda_stream, double *lo_out, double *hi_out);

/* Number of kernels this library has launched in the calling process (for gpu_launches in bench.py). */
unsigned long long mc_kernel_launch_count(void);

/* FP64 FMA throughput micro-benchmark: runs `iters` dependent-chain rounds of 8
 * independent DFMA chains per thread on all SMs and returns achieved FLOP/s in *flops (HOST). */
int mc_fp64_peak(int iters, void *cuda_stream, double *flops, double *ms);

const char *mc_strerror(int code);
const char *mc_version(void);
#ifdef __cplusplus
}
#endif
#endif
