/*
 * sanitize_main.c — driver for the sanitizer build of the ORACLE (test infrastructure, not the product).
 *
 * tests/test_oracle_sampler.py::test_oracle_is_clean_under_address_and_undefined_sanitizers compiles
 *     gcc -std=c99 -O1 -g -fsanitize=address,undefined -fno-sanitize-recover=all -ffp-contract=off -fopenmp \
 *         oracle/nss_oracle.c oracle/sanitize_main.c -lm
 * and runs the result ("-fsanitize=address,undefined on the oracle").  The driver walks every
 * entry point of nss_oracle.c on tiny problems of all three kinds (relative binning, full grid, Gaussian):
 * create, batch likelihood, one replacement step with traces, a whole run, the periodic wrap, the resampler.
 * It checks nothing numerically (the pins do that); it exists so that an out-of-bounds index, a read of
 * uninitialised heap, a leak or undefined arithmetic in the oracle aborts a test.
 */
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>

typedef struct orc_problem orc_problem;
orc_problem *orc_create(int d, const int *param_index, const double *theta_fixed, const double *lo, const double *hi, int n_det,
                        const double *det_flat, double gmst, int n_freq, double f_min, double df, const double *psd,
                        const double *data, const double *theta_fid, int n_bins, int kind, const double *gauss_mu,
                        const double *gauss_sigma);
void orc_destroy(orc_problem *p);
void orc_set_periodic(orc_problem *p, const int *flags);
void orc_waveform(const double *th, const double *det9, double gmst, const double *f, int n, double *out);
void orc_loglike_batch(const orc_problem *p, const double *theta, int64_t N, double *out, int nthreads);
void orc_init_live(const orc_problem *p, int n, uint64_t seed, double *live, double *logL, int nthreads);
int orc_replace_step(const orc_problem *p, double *live, double *logL, int n, int k, double logLstar_in, int n_repeats,
                     uint64_t seed, uint32_t iteration, double *dead_theta, double *dead_logL, int *dead_idx,
                     double *logLstar_out, int64_t *n_evals_out, int32_t *trace, double *margin, int nthreads);
int orc_run(const orc_problem *p, int n, int k, int n_repeats, uint64_t seed, double stop_dlogz, int max_iter, int64_t cap,
            double *dead_theta, double *dead_logL, double *dead_logL_birth, double *dead_logw, double *scal, int nthreads);
int64_t orc_resample_equal(const double *logL, const double *logw, int64_t n, uint64_t seed, int64_t *idx_out);
void orc_get_summary(const orc_problem *p, double *out);
void orc_get_edges(const orc_problem *p, int *idx, double *f);

static int exercise(orc_problem *p, int d, int n, int k, int n_repeats, int periodic_dim)
{
  double *live = malloc(sizeof(double) * n * d), *logL = malloc(sizeof(double) * n);
  double *dth = malloc(sizeof(double) * k * d), *dl = malloc(sizeof(double) * k), *margin = malloc(sizeof(double) * k);
  int *didx = malloc(sizeof(int) * k);
  int32_t *trace = malloc(sizeof(int32_t) * k * n_repeats * 3);
  double Lstar;
  int64_t ne;
  orc_init_live(p, n, 3, live, logL, 2);
  int rc = orc_replace_step(p, live, logL, n, k, NAN, n_repeats, 3, 0, dth, dl, didx, &Lstar, &ne, trace, margin, 2);
  if (periodic_dim >= 0) {
    int flags[11] = {0};
    flags[periodic_dim] = 1;
    orc_set_periodic(p, flags);
    rc |= orc_replace_step(p, live, logL, n, k, NAN, n_repeats, 3, 1, dth, dl, didx, &Lstar, &ne, trace, margin, 2);
    orc_set_periodic(p, NULL);
  }
  const int64_t cap = (int64_t)k * 40 + n;
  double *rt = malloc(sizeof(double) * cap * d), *rl = malloc(sizeof(double) * cap), *rb = malloc(sizeof(double) * cap),
         *rw = malloc(sizeof(double) * cap), scal[6];
  const int rrc = orc_run(p, n, k, n_repeats, 5, -3.0, 40, cap, rt, rl, rb, rw, scal, 2);
  if (rrc >= 0) {
    const int64_t nd = (int64_t)scal[4];
    int64_t *idx = malloc(sizeof(int64_t) * nd);
    const int64_t ne_q = orc_resample_equal(rl, rw, nd, 5, idx);
    if (ne_q < 0 || ne_q > nd) rc |= 8;
    free(idx);
  } else rc |= 4;
  free(live); free(logL); free(dth); free(dl); free(margin); free(didx); free(trace);
  free(rt); free(rl); free(rb); free(rw);
  return rc;
}

int main(void)
{
  const int nf = 257, ndet = 2, B = 7;
  const double fmin = 20.0, df = 0.5;
  const double det[18] = {-2.16141492636e6, -3.83469517889e6, 4.60035022664e6, -0.22389266154, 0.79983062746, 0.55690487831,
                          -0.91397818574, 0.02609403989, -0.40492342125,
                          0, 0, 0, 1, 0, 0, 0, 1, 0};
  double th[11] = {30.0, 0.8, 0.1, -0.05, 400.0, 0.0, 1.0, 0.6, 0.8, 1.5, -0.5};
  double *f = malloc(sizeof(double) * nf), *psd = malloc(sizeof(double) * ndet * nf), *data = malloc(sizeof(double) * ndet * nf * 2);
  for (int k = 0; k < nf; ++k) f[k] = fmin + k * df;
  for (int a = 0; a < ndet; ++a) {
    orc_waveform(th, det + 9 * a, 0.3, f, nf, data + (size_t)a * nf * 2);
    for (int k = 0; k < nf; ++k) psd[a * nf + k] = 1e-46;
  }
  const int pidx[4] = {0, 1, 5, 6};
  const double lo[4] = {25.0, 0.5, -0.05, 0.0}, hi[4] = {35.0, 1.0, 0.05, 6.283185307179586};
  int bad = 0;
  for (int kind = 0; kind < 2; ++kind) {
    orc_problem *p = orc_create(4, pidx, th, lo, hi, ndet, det, 0.3, nf, fmin, df, psd, data, th, B, kind, NULL, NULL);
    if (!p) { fprintf(stderr, "orc_create failed (kind %d)\n", kind); return 2; }
    if (kind == 0) {
      double summ[2 * 7 * 6], ef[8];
      int ei[8];
      orc_get_summary(p, summ);
      orc_get_edges(p, ei, ef);
    }
    bad |= exercise(p, 4, 24, kind == 0 ? 12 : 23, 3, 3);
    orc_destroy(p);
  }
  {
    const double glo[3] = {-1, -1, -1}, ghi[3] = {1, 1, 1}, mu[3] = {0, 0.1, -0.2}, sg[3] = {0.1, 0.2, 0.1};
    orc_problem *p = orc_create(3, NULL, NULL, glo, ghi, 0, NULL, 0.0, 0, 0.0, 0.0, NULL, NULL, NULL, 0, 2, mu, sg);
    if (!p) return 2;
    bad |= exercise(p, 3, 40, 1, 4, 0);
    bad |= exercise(p, 3, 40, 20, 4, -1);
    orc_destroy(p);
  }
  /* rejected inputs must free what they allocated */
  if (orc_create(4, pidx, th, hi, lo, ndet, det, 0.3, nf, fmin, df, psd, data, th, B, 0, NULL, NULL)) bad |= 16;
  psd[5] = 0.0;
  if (orc_create(4, pidx, th, lo, hi, ndet, det, 0.3, nf, fmin, df, psd, data, th, B, 0, NULL, NULL)) bad |= 16;
  free(f); free(psd); free(data);
  printf("sanitize_main: %s (%d)\n", bad ? "FAILED" : "ok", bad);
  return bad ? 1 : 0;
}
