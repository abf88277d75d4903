/*
 * nss.h — C ABI of libnss.so: the B200 (sm_100a) hot path of "Parallel Nested Slice Sampling for
 * Gravitational Wave Parameter Estimation" (arxiv 2509.24949; /root/reference/PAPER.md).
 *
 * One batched nested-slice-sampling replacement step whose every chain step
 * evaluates a heterodyned / relative-binning frequency-domain GW log-likelihood (PAPER.md:33, 39,
 * 49), plus the on-device nested-sampling bookkeeping and a full-frequency-grid likelihood.
 * The paper prints no equations; the operations are defined by SURVEY.md §8(c) O1..O16 (restated
 * in DESIGN.md §3), cited per call below.
 *
 * Conventions
 *  - Every call returns 0 on success or a negative NSS_E* code; nothing throws or aborts.
 *  - "device" pointers are CUDA device pointers on the device the handle was created on
 *    (e.g. torch tensor.data_ptr()); "host" pointers are ordinary host memory.
 *  - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *  - All floating point is IEEE fp64.  Row-major everywhere.
 *  - One handle serves one stream at a time (not re-entrant).  Single GPU.  There is NO CPU
 *    fallback: without a CUDA device every compute call returns NSS_ECUDA.
 *  - Ownership: nss_create deep-copies everything it needs (the caller may free psd/data when it
 *    returns); the handle owns its device tables and scratch; every output buffer is allocated by
 *    the caller; the library never frees caller memory.
 */
#ifndef NSS_H
#define NSS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define NSS_NSLOT 11      /* canonical parameter slots, O2 */
#define NSS_MAXDET 4

/* canonical slot order (O2): 0 Mc [Msun, detector frame], 1 q = m2/m1 in (0,1], 2 chi1z, 3 chi2z,
 * 4 dL [Mpc], 5 tc [s], 6 phic [rad], 7 iota, 8 psi, 9 ra, 10 dec.
 * Physical domain: Mc > 0, 0 < q <= 1, |chi| < 1, dL > 0, everything finite; outside it the
 * log-likelihood is -inf (not an error). */

enum {
  NSS_OK = 0,
  NSS_EINVAL = -1,    /* bad sizes, lo >= hi, PSD <= 0, n_delete >= n_live, fiducial outside domain,
                         survivor below a supplied logLstar, NULL pointer */
  NSS_ENOMEM = -2,    /* host or device allocation failed */
  NSS_ECUDA = -3,     /* a CUDA call failed (no device, launch error); see nss_last_cuda_error */
  NSS_ECHOL = -4,     /* non-positive Cholesky pivot of the live-point covariance */
  NSS_ECAP = -5,      /* nss_result arrays too small */
  NSS_ENOTCONV = -6,  /* nss_run hit max_iter; the results written are still valid */
  NSS_ELIMIT = -7     /* a size beyond the fixed capacity of an entry point that does not allocate (*_static) */
};

enum { NSS_KIND_RB = 0, NSS_KIND_FULL = 1, NSS_KIND_GAUSS = 2 };

typedef struct nss_handle nss_handle; /* opaque */

typedef struct {
  double vertex_m[3], xarm[3], yarm[3];   /* Earth-fixed frame; arms are unit vectors (O4) */
} nss_detector;

typedef struct {
  int32_t d;                       /* sampled dimensions, 1..11                                  */
  int32_t param_index[NSS_NSLOT];  /* sampled dim j -> canonical slot (kinds 0, 1)               */
  double  theta_fixed[NSS_NSLOT];  /* canonical values for unsampled slots                       */
  double  lo[NSS_NSLOT], hi[NSS_NSLOT]; /* uniform prior box per sampled dim, lo < hi (A22)      */
  int32_t n_det;                   /* 1..4 (kinds 0, 1)                                          */
  nss_detector det[NSS_MAXDET];
  double  gmst;                    /* Greenwich sidereal angle [rad]                             */
  int32_t n_freq;                  /* grid f_k = f_min + k*df, k = 0..n_freq-1                   */
  double  f_min, df;
  const double *psd;               /* host, [n_det][n_freq], one-sided, > 0                      */
  const double *data;              /* host, [n_det][n_freq][2] = complex128 (re, im)             */
  double  theta_fid[NSS_NSLOT];    /* canonical heterodyne reference, kind 0       */
  int32_t n_bins;                  /* B, 1 <= B <= n_freq-1, kind 0                              */
  int32_t kind;                    /* NSS_KIND_*                                                 */
  double  gauss_mu[NSS_NSLOT], gauss_sigma[NSS_NSLOT]; /* per sampled dim, kind 2 (O16)          */
} nss_config;

/* Setup (heterodyne reference fixed in advance, excluded from quoted runtimes).
 * Host: validates, chooses the bin edges (O8), evaluates the fiducial waveform (O3, O4), builds the
 * per-(detector, bin) summary data A0, A1, B0, B1 and <d,d> (O9), packs the device tables and
 * uploads them.  Synchronous. */
int nss_create(const nss_config *cfg, nss_handle **out);
int nss_destroy(nss_handle *h);

/* Batched log-likelihood (O10 relative binning, O7 full grid or O16 Gaussian, by cfg.kind).
 * theta_dev: device [N][d] sampled coordinates; logL_dev: device [N].  Evaluates any theta (inside
 * the prior box or not); outside the physical domain or non-finite -> -inf.  N = 0 is a no-op.
 * Asynchronous on the stream. */
int nss_loglike_batch(nss_handle *h, const double *theta_dev, int64_t N, double *logL_dev,
                      void *cuda_stream);

/* Variant selector for nss_loglike_batch (profiling / tests): 0 = automatic (default),
 * 1 = one thread per point, 2 = one sub-warp (8 or 32 lanes) per point. */
int nss_set_loglike_variant(nss_handle *h, int32_t variant);

/* Warps that run one slice chain (K3): 0 = automatic, else 1, 2, 4 or 8.  A chain is one CTA of G warps; every
 * sub-warp of `lanes` lanes evaluates one bracket test, so a round evaluates the next G * 32/lanes tests of
 * the sequential algorithm speculatively; the decisions, positions and evaluation count are those of the
 * sequential algorithm for every G and every lane count (tests/test_gpu_sampler.py). */
int nss_set_chain_warps(nss_handle *h, int32_t warps);

/* NEXT-2 (covariance-tuned slices are "troublesome for the wrapped phase and polarization angle"):
 * flags_host[j] != 0 makes sampled dimension j periodic in the slice sampler: a candidate's coordinate is mapped back
 * into [lo_j, hi_j) as y - W floor((y - lo_j)/W), W = hi_j - lo_j, and takes no part in the prior-box test (default and
 * NULL: hard inclusive walls in every dimension, reading A16).  Host array of d flags, copied.  The likelihood should
 * be periodic in that coordinate over the box (phi_c over 2 pi, psi over pi, ra over 2 pi); the evidence is valid either way.
 * The tuning follows the geometry too (reading R7; "better tuning that respects the geometry of the
 * parameter space"): in nss_tune and in every iteration a periodic coordinate is unwrapped around its circular mean
 * (x' = x - W rint((x - mu_c)/W), mu_c from atan2 of the summed sines and cosines of 2 pi (x - lo)/W) before mean,
 * covariance and Cholesky factor are formed, so a population that straddles the seam is tuned with the width it has on
 * the circle; a population that does not reach across the seam, and any non-periodic coordinate, is tuned as before. */
int nss_set_periodic(nss_handle *h, const int32_t *flags_host);

/* Diagnostics of the most recent nss_replace_step / nss_iterate (read from the control block that call fetched):
 * rounds run by all chains together, and candidates evaluated including the speculative ones the sequential
 * algorithm did not need (the evaluation count n_evals never includes those). */
int nss_last_chain_diag(nss_handle *h, int64_t *rounds_host, int64_t *evaluated_host);

/* Lanes that evaluate one candidate in K3 (relative binning only): 0 = automatic, else 8, 16 or 32 (a width
 * whose table was not built, e.g. 8 lanes with more than 256 bins, falls back to the automatic choice). */
int nss_set_chain_lanes(nss_handle *h, int32_t lanes);

/* Single-warp chains (nss_set_chain_warps 1, or the automatic choice for many chains) packed per CTA of K3: the warps of
 * a CTA share one shared-memory copy of the record table and take chains from a device counter as they finish.
 * 0 = automatic, else 1 .. 8.  Like the two setters above it changes the schedule only, never a result. */
int nss_set_chain_pack(nss_handle *h, int32_t chains_per_cta);

/* One NS iteration (O12): select the n_delete lowest logL (ascending, ties by lower slot), tune the
 * slice directions from the covariance of the full live set (Cholesky), run one chain per deleted
 * point (start = uniformly chosen survivor; n_repeats x {direction, stepping-out, shrinkage} under
 * logL > logLstar inside the prior box), overwrite the deleted slots in place.
 * live_dev [n_live][d] and logL_dev [n_live] are updated in place.  logLstar = NaN: the threshold is
 * the highest deleted logL; otherwise the supplied value is used and every survivor must have
 * logL >= logLstar (NSS_EINVAL if not) — the teacher-forced form used for trajectory parity.
 * Random numbers: Philox4x32-10, key = seed, counter = (block, step, chain, iteration) (O11).
 * Outputs: dead_theta_dev [n_delete][d], dead_logL_dev [n_delete], dead_idx_dev [n_delete]
 * (ascending logL); *logLstar_host, *n_evals_host (sequential-algorithm likelihood evaluations).
 * Synchronises the stream before returning. */
int nss_replace_step(nss_handle *h, double *live_dev, double *logL_dev, int32_t n_live,
                     int32_t n_delete, double logLstar, int32_t n_repeats, uint64_t seed,
                     uint32_t iteration, double *dead_theta_dev, double *dead_logL_dev,
                     int32_t *dead_idx_dev, double *logLstar_host, int64_t *n_evals_host,
                     void *cuda_stream);

/* One COMPLETE NS iteration = every row of the hot path with one host
 * synchronisation: nss_replace_step's work (delete select, tuning, chains, replace; threshold
 * selected internally), then the evidence bookkeeping of the deleted batch (O12.2) and the live
 * evidence / stop test (O14).  This is the loop body of nss_run and the "step" bench.py times.
 * state: logX, logZ in/out (start a run with 0, -inf); the rest out. */
typedef struct {
  double  logX, logZ;              /* in/out: log prior volume, log evidence of the dead points  */
  double  logZ_live;               /* out: logX + logsumexp(logL_live) - ln n after the step     */
  double  logLstar;                /* out: threshold of this iteration                           */
  int64_t n_evals;                 /* out: sequential-algorithm likelihood evaluations           */
  int32_t converged;               /* out: logZ_live - logZ < stop_dlogz                         */
  int32_t pad_;
} nss_iter_state;

int nss_iterate(nss_handle *h, double *live_dev, double *logL_dev, int32_t n_live, int32_t n_delete,
                int32_t n_repeats, uint64_t seed, uint32_t iteration, double stop_dlogz,
                double *dead_theta_dev /*[n_delete][d]*/, double *dead_logL_dev /*[n_delete]*/,
                double *dead_logw_dev /*[n_delete]*/, int32_t *dead_idx_dev /*[n_delete]*/,
                nss_iter_state *state_host, void *cuda_stream);

/* The same iteration with HOST buffers (pinned memory recommended): live/logL are copied to the
 * device, the iteration runs, and live, logL and the dead rows are copied back, all queued on the stream
 * inside the call, which waits once at the end.  On NSS_ECHOL the live set comes back unchanged (the
 * chains did not run) and state_host is untouched.  bench.py's end-to-end (`e2e`) leg. */
int nss_iterate_host(nss_handle *h, double *live_host, double *logL_host, int32_t n_live,
                     int32_t n_delete, int32_t n_repeats, uint64_t seed, uint32_t iteration,
                     double stop_dlogz, double *dead_theta_host, double *dead_logL_host,
                     double *dead_logw_host, int32_t *dead_idx_host, nss_iter_state *state_host,
                     void *cuda_stream);

/* Host-buffer form of nss_loglike_batch: theta_host [N][d] -> logL_host [N]; H2D copy, kernel and
 * D2H copy on the stream, synchronised before returning. */
int nss_loglike_batch_host(nss_handle *h, const double *theta_host, int64_t N, double *logL_host,
                           void *cuda_stream);

/* Test hook: if set (device pointers, may be NULL to clear), the next nss_replace_step calls also
 * write trace_dev [n_delete][n_repeats][3] = (left expansions, right expansions, accepted shrink
 * index or -1) and margin_dev [n_delete] = min |logL - logLstar| over the chain's bracket tests. */
int nss_set_trace(nss_handle *h, int32_t *trace_dev, double *margin_dev);

/* K4 bookkeeping kernels on their own (O12.1, O12.3, O12.2). */
int nss_select_lowest(nss_handle *h, const double *logL_dev, int32_t n_live, int32_t n_delete,
                      int32_t *dead_idx_dev /*[n_delete] ascending logL, ties by slot*/,
                      int32_t *surv_idx_dev /*[n_live-n_delete] ascending slot, may be NULL*/,
                      double *logLstar_host, void *cuda_stream);

/* The delete-select of nss_select_lowest (O12.1: the n_delete lowest logL in ascending order, ties by the lower slot,
 * the survivors in ascending slot order, the threshold L* = the highest deleted logL) for callers that cannot let this
 * library allocate device memory.  Who that is: a process whose GPU memory has been handed over wholesale to a pool
 * (PyTorch's caching allocator, a job that pre-reserves its whole HBM budget), where a cudaMalloc issued from inside a
 * library fails with "out of memory" although the pool has plenty free; a sampler loop that shares the GPU with other
 * streams and cannot take the device-wide stall cudaMalloc / cudaFree bring with them; and code that must prove, after
 * start-up, that no later call can fail for want of memory.  Every other entry point here needs an nss_handle, and both
 * nss_create and the handle's first use of the sampler allocate; this one needs no handle at all.
 *
 * Its work space (partial counts, ranks, a spare survivor list: 1 114 144 bytes) is a fixed array inside libnss.so's
 * device image, so every GPU that loads the library carries it until the process exits, used or not, and the size is
 * capped: n_live <= NSS_SELECT_STATIC_MAX_LIVE, else NSS_ELIMIT and nothing is launched (larger live sets need the
 * sample sort of nss_select_lowest, whose work space grows with n_live).  The call issues no cudaMalloc, cudaFree or
 * other allocating routine; it launches two kernels on the stream and returns without waiting for them.
 *
 * logL_dev: device [n_live], read only.  dead_idx_dev: device [n_delete], out.  surv_idx_dev: device
 * [n_live - n_delete], out, or NULL if not wanted.  logLstar_dev: DEVICE [1], out, or NULL (a host slot would need a
 * synchronising copy; read it with your own copy when you need it).  Works on the CURRENT device; all pointers must
 * belong to it.  Returns NSS_EINVAL for NULL / inconsistent sizes (as nss_select_lowest), NSS_ELIMIT, NSS_ECUDA.
 *
 * First use on a device: the first call made while that device is current looks up the array's device address
 * (cudaGetSymbolAddress) and remembers it; make that first call during start-up, before any stream capture begins.
 * Sharing: there is ONE array per device and every call uses it, whatever the stream or thread.  Calls must not
 * overlap on the GPU: two in flight at once (two streams, or two host threads on one device) overwrite each other's
 * counts and both results are garbage; order them on one stream or with events.  The array keeps what the last call
 * wrote, which is harmless: each call overwrites every word it later reads, so nothing has to be cleared in between. */
#define NSS_SELECT_STATIC_MAX_LIVE 8192
int nss_select_lowest_static(const double *logL_dev, int32_t n_live, int32_t n_delete,
                             int32_t *dead_idx_dev /*[n_delete]*/, int32_t *surv_idx_dev /*[n_live-n_delete] or NULL*/,
                             double *logLstar_dev /*device [1] or NULL*/, void *cuda_stream);

int nss_tune(nss_handle *h, const double *live_dev, int32_t n_live, double *mean_dev /*[d]*/,
             double *chol_dev /*[d][d] lower, row-major*/, void *cuda_stream);
/* logw_j = logX + ln(1 - e^{-1/m_j}), m_j = n_live - j; logX -= sum 1/m_j; logZ = logaddexp(...).
 * state_host[2] = {logX, logZ} in/out. */
int nss_evidence_update(nss_handle *h, const double *dead_logL_dev, int32_t n_live, int32_t n_delete,
                        double *logw_dev /*[n_delete]*/, double *state_host, void *cuda_stream);
/* Initial live points (O13): uniform in the box from the Philox stream, then their logL. */
int nss_init_live(nss_handle *h, int32_t n_live, uint64_t seed, double *live_dev, double *logL_dev,
                  void *cuda_stream);
/* Philox test hook: out_dev [n][4] uint32 = Philox4x32-10(key = seed, counter = ctr_dev[i][4]). */
int nss_philox(nss_handle *h, uint64_t seed, const uint32_t *ctr_dev, int64_t n, uint32_t *out_dev,
               void *cuda_stream);

/* NEXT-4, reading R6: equal-weight posterior samples.  PAPER.md:59-63 quotes the number of "equal weight
 * samples" in brackets beside the Kish ESS and does not define them.  Reading: row i (weight p_i ~ exp(logL_i + logw_i))
 * is kept iff u_i < p_i / max_j p_j, u_i the [0, 1) uniform of Philox counter (0, i mod 2^32, i div 2^32, 0xFFFFFFFD)
 * under key `seed`; rows with logL + logw = -inf are never kept.  logL_dev, logw_dev: device [n]; idx_dev: device [n] or
 * NULL, receives the kept row indices in ascending order; *n_equal_host = their number.  Synchronous. */
int nss_resample_equal(nss_handle *h, const double *logL_dev, const double *logw_dev, int64_t n, uint64_t seed,
                       int64_t *idx_dev, int64_t *n_equal_host, void *cuda_stream);

typedef struct {
  double  logZ, logZ_err, H;       /* evidence, its replica s.d. (O15), information             */
  int32_t n_iter;
  int64_t n_dead, n_evals;         /* rows written; sequential-algorithm likelihood evaluations  */
  double *dead_theta;              /* host [cap][d]   caller-allocated                           */
  double *dead_logL;               /* host [cap]                                                 */
  double *dead_logL_birth;         /* host [cap]                                                 */
  double *dead_logw;               /* host [cap]      log prior-volume weight                    */
  int64_t cap;                     /* >= n_iter*n_delete + n_live                                */
  double  gpu_ms;                  /* device time of the run (CUDA events), setup excluded       */
  double  ess;                     /* Kish effective sample size (sum p)^2 / sum p^2 of the posterior weights
                                      p_i ~ exp(logL_i + logw_i) over all rows (O15; the paper's Table 1b metric) */
  int64_t n_equal;                 /* equal-weight posterior rows (reading R6; the bracketed count of PAPER.md:59-63) */
  int64_t *equal_idx;              /* host [cap] or NULL: if given, receives the n_equal kept row indices, ascending  */
} nss_result;

/* Full run (O13, O14): initial live points, NS iterations until logZ_live - logZ < stop_dlogz
 * (default -3.0) or max_iter, then the live points are appended (ascending logL, weight X/n).
 * Everything stays on the device; results are copied to the caller's host arrays at the end.  The host queues one
 * iteration ahead: the stop test sets a device flag, the kernels of an iteration queued past it return at once, and the
 * flag reaches the host through a pinned slot ("the entire end-to-end algorithm can then run in GPU memory").
 * logZ_err (200 stochastic-compression replicas, O15), ess and n_equal (the rows nss_resample_equal keeps, same seed) are
 * reduced on the device.  Returns NSS_OK, NSS_ENOTCONV
 * (max_iter reached, results valid), NSS_ECAP (out->cap too small: needs n_iter * n_delete + n_live rows), NSS_ECHOL,
 * NSS_EINVAL, NSS_ENOMEM or NSS_ECUDA.  Synchronous: returns after the stream has drained.
 * `out` is read as well as written: zero the whole nss_result first (memset / = {0}), then set the four array pointers
 * and cap.  equal_idx in particular MUST be NULL unless it points to cap int64 slots — nss_run copies n_equal indices
 * through any non-NULL value, so a field left uninitialised is a wild write. */
int nss_run(nss_handle *h, int32_t n_live, int32_t n_delete, int32_t n_repeats, uint64_t seed,
            double stop_dlogz, int32_t max_iter, nss_result *out, void *cuda_stream);

/* Host-side strain of one detector on an arbitrary frequency list (O3, O4), the routine nss_create
 * uses for the fiducial waveform; out [n][2].  Used by bench.py to synthesise injections. */
int nss_waveform(const double *theta_canon /*[11]*/, const nss_detector *det, double gmst,
                 const double *freqs, int32_t n, double *out);

/* Read back the setup tables (tests): bin-edge grid indices [B+1] and summary data
 * [n_det][B][6] = (A0re, A0im, A1re, A1im, B0, B1) as defined in O9 (unscaled). */
int nss_get_tables(nss_handle *h, int32_t *edge_idx_host, double *summary_host, double *dd_host);

/* Register-resident DFMA chain on every SM for ~`ms` milliseconds: measured fp64 FMA throughput,
 * the roofline denominator.  *tflops_host = 2 * FMA/s / 1e12. */
int nss_fp64_peak(double ms, double *tflops_host, void *cuda_stream);

/* on != 0: from now on the library records a CUDA event pair around every K3 (slice-sampling chains) launch on the
 * caller's stream.  Off by default: the event in front of K3 keeps its prologue from overlapping the kernel before it
 * (programmatic dependent launch). */
int nss_set_chain_timing(nss_handle *h, int32_t on);
/* Device time [ms] of the most recent K3 launch from that event pair (bench.py's roofline for the dominant kernel);
 * NSS_EINVAL unless nss_set_chain_timing(h, 1) was called before that launch. */
int nss_last_chain_ms(nss_handle *h, double *ms_host);

/* Kernel launches issued by this handle since creation (bench.py's gpu_launches). */
int64_t nss_launch_count(const nss_handle *h);

const char *nss_strerror(int code);
const char *nss_last_cuda_error(void);
int nss_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NSS_H */
