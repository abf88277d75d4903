// nss_setup.cu — L0 host setup (untimed) and handle lifetime.
//
// nss_create: validate -> bin edges (O8) -> fiducial waveform on the full grid (O3, O4) ->
// summary data A0/A1/B0/B1 per (detector, bin) and <d,d> (O9) -> pack device tables -> upload.
#include <math.h>
#include <string.h>

#include <complex>
#include <new>
#include <vector>

#include "nss_internal.cuh"

thread_local char g_nss_cuda_err[256] = "";

int nss_cuda_fail(cudaError_t e, const char *where)
{
  snprintf(g_nss_cuda_err, sizeof(g_nss_cuda_err), "%s: %s", where, cudaGetErrorString(e));
  cudaGetLastError();
  return NSS_ECUDA;
}

extern "C" const char *nss_last_cuda_error(void) { return g_nss_cuda_err; }

extern "C" const char *nss_strerror(int code)
{
  switch (code) {
    case NSS_OK: return "ok";
    case NSS_EINVAL: return "invalid argument";
    case NSS_ENOMEM: return "out of memory";
    case NSS_ECUDA: return "CUDA error (see nss_last_cuda_error)";
    case NSS_ECHOL: return "non-positive Cholesky pivot of the live-point covariance";
    case NSS_ECAP: return "result arrays too small";
    case NSS_ENOTCONV: return "max_iter reached before the stop rule (results valid)";
    case NSS_ELIMIT: return "size beyond the fixed capacity of a *_static entry point (NSS_SELECT_STATIC_MAX_LIVE live points)";
    default: return "unknown error";
  }
}

extern "C" int nss_version(void) { return 1; }

using cplx = std::complex<double>;

namespace {

void detector_tensor(const nss_detector &det, double *D6, double *rc)
{
  const double *x = det.xarm, *y = det.yarm;
  D6[0] = 0.5 * (x[0] * x[0] - y[0] * y[0]);
  D6[1] = 0.5 * (x[0] * x[1] - y[0] * y[1]);
  D6[2] = 0.5 * (x[0] * x[2] - y[0] * y[2]);
  D6[3] = 0.5 * (x[1] * x[1] - y[1] * y[1]);
  D6[4] = 0.5 * (x[1] * x[2] - y[1] * y[2]);
  D6[5] = 0.5 * (x[2] * x[2] - y[2] * y[2]);
  for (int c = 0; c < 3; ++c) rc[c] = det.vertex_m[c] / nssp::kC;
}

// complex amplitude (without f^-7/6) and arrival-time offset of one detector
void det_amplitude(const nssp::Intrinsic &I, const double *th, double gmst, const double *D6, const double *rc,
                   cplx &amp, double &tau)
{
  nssp::Sky S;
  nssp::sky_frame(gmst, th[9], th[10], th[8], S);
  double fp, fc;
  nssp::antenna(S, D6, rc, fp, fc, tau);
  const double ci = I.cos_iota;
  amp = I.amp * cplx(fp * 0.5 * (1.0 + ci * ci), -fc * ci);
}

void host_waveform(const double *th, const double *D6, const double *rc, double gmst, const double *f, int n,
                   cplx *out)
{
  nssp::Intrinsic I;
  nssp::intrinsic(th, I);
  cplx amp;
  double tau;
  det_amplitude(I, th, gmst, D6, rc, amp, tau);
  for (int k = 0; k < n; ++k) {
    double g[nssp::kNB];
    nssp::basis(f[k], g);
    double ph = I.c_const;
    for (int j = 0; j < nssp::kNB; ++j) ph += I.c[j] * g[j];
    ph += f[k] * (I.tc + tau);
    double s, c;
    nssp::sincos_turns(ph, &s, &c);
    const double x = cbrt(f[k]);
    const double f76 = 1.0 / (f[k] * sqrt(x));          // f^-7/6 = 1 / (f * f^(1/6))
    out[k] = amp * f76 * cplx(c, -s);
  }
}

// O8: equal increments of a power-law dephasing measure, snapped to the grid, strictly increasing
std::vector<int32_t> choose_edges(int n, double f_min, double df, int B)
{
  const double f_max = f_min + (n - 1) * df;
  static const double gam[5] = {-5.0 / 3.0, -2.0 / 3.0, 1.0, 5.0 / 3.0, 7.0 / 3.0};
  std::vector<double> del(n);
  for (int k = 0; k < n; ++k) {
    const double f = f_min + k * df;
    double s = 0.0;
    for (double g : gam) s += (g > 0 ? 1.0 : -1.0) * pow(f / (g > 0 ? f_max : f_min), g);
    del[k] = s;
  }
  std::vector<int32_t> ie(B + 1);
  int cur = 0;                       // del is monotone: a forward scan finds the nearest grid point
  for (int e = 0; e <= B; ++e) {
    const double target = del[0] + ((double)e / (double)B) * (del[n - 1] - del[0]);
    while (cur + 1 < n && fabs(del[cur + 1] - target) < fabs(del[cur] - target)) ++cur;
    ie[e] = cur;
  }
  ie[0] = 0;
  ie[B] = n - 1;
  for (int e = 1; e <= B; ++e) ie[e] = ie[e] < ie[e - 1] + 1 ? ie[e - 1] + 1 : ie[e];
  ie[B] = n - 1;
  for (int e = B - 1; e >= 0; --e) ie[e] = ie[e] > ie[e + 1] - 1 ? ie[e + 1] - 1 : ie[e];
  return ie;
}

inline int per_of(int round, int per) { return round == 0 ? 2 : per; }

template <class T>
int upload(const std::vector<T> &v, T **dptr, size_t *bytes)
{
  *bytes = v.size() * sizeof(T);
  if (v.empty()) { *dptr = nullptr; return NSS_OK; }
  cudaError_t e = cudaMalloc((void **)dptr, *bytes);
  if (e != cudaSuccess) { nss_cuda_fail(e, "cudaMalloc(table)"); return e == cudaErrorMemoryAllocation ? NSS_ENOMEM : NSS_ECUDA; }
  NSS_CUDA(cudaMemcpy(*dptr, v.data(), *bytes, cudaMemcpyHostToDevice));
  return NSS_OK;
}

}  // namespace

extern "C" int nss_waveform(const double *theta_canon, const nss_detector *det, double gmst, const double *freqs,
                            int32_t n, double *out)
{
  if (!theta_canon || !det || !freqs || !out || n < 0) return NSS_EINVAL;
  if (!nssp::domain_ok(theta_canon)) return NSS_EINVAL;
  double D6[6], rc[3];
  detector_tensor(*det, D6, rc);
  std::vector<cplx> h(n);
  host_waveform(theta_canon, D6, rc, gmst, freqs, n, h.data());
  for (int k = 0; k < n; ++k) { out[2 * k] = h[k].real(); out[2 * k + 1] = h[k].imag(); }
  return NSS_OK;
}

extern "C" int nss_destroy(nss_handle *h)
{
  if (!h) return NSS_OK;
  cudaSetDevice(h->device);
  cudaFree(h->d_rec); cudaFree(h->d_soa[0]); cudaFree(h->d_soa[1]); cudaFree(h->d_soa[2]);
  cudaFree(h->d_surv_idx); cudaFree(h->d_dead_idx); cudaFree(h->d_rank); cudaFree(h->d_rank_part); cudaFree(h->d_tune_scratch); cudaFree(h->d_ctl);
  if (h->h_ctl) cudaFreeHost(h->h_ctl);
  cudaFree(h->d_mean); cudaFree(h->d_chol); cudaFree(h->d_birth); cudaFree(h->d_stage);
  cudaFree(h->d_run);
  if (h->h_run) cudaFreeHost(h->h_run);
  if (h->ev_ctl[0]) cudaEventDestroy(h->ev_ctl[0]);
  if (h->ev_ctl[1]) cudaEventDestroy(h->ev_ctl[1]);
  if (h->ev_run[0]) cudaEventDestroy(h->ev_run[0]);
  if (h->ev_run[1]) cudaEventDestroy(h->ev_run[1]);
  if (h->ev_k3[0]) cudaEventDestroy(h->ev_k3[0]);
  if (h->ev_k3[1]) cudaEventDestroy(h->ev_k3[1]);
  delete h;
  return NSS_OK;
}

extern "C" int nss_create(const nss_config *cfg, nss_handle **out)
{
  if (!cfg || !out) return NSS_EINVAL;
  *out = nullptr;
  if (cfg->d < 1 || cfg->d > NSS_NSLOT) return NSS_EINVAL;
  if (cfg->kind < 0 || cfg->kind > 2) return NSS_EINVAL;
  for (int j = 0; j < cfg->d; ++j)
    if (!(cfg->lo[j] < cfg->hi[j]) || !isfinite(cfg->lo[j]) || !isfinite(cfg->hi[j])) return NSS_EINVAL;
  const int kind = cfg->kind;
  if (kind == NSS_KIND_GAUSS) {
    for (int j = 0; j < cfg->d; ++j)
      if (!(cfg->gauss_sigma[j] > 0.0) || !isfinite(cfg->gauss_mu[j])) return NSS_EINVAL;
  } else {
    if (cfg->n_det < 1 || cfg->n_det > NSS_MAXDET || cfg->n_freq < 2 || !cfg->psd || !cfg->data) return NSS_EINVAL;
    if (!(cfg->df > 0.0) || !(cfg->f_min > 0.0)) return NSS_EINVAL;
    bool seen[NSS_NSLOT] = {false};
    for (int j = 0; j < cfg->d; ++j) {
      const int s = cfg->param_index[j];
      if (s < 0 || s >= NSS_NSLOT || seen[s]) return NSS_EINVAL;
      seen[s] = true;
    }
    const size_t nn = (size_t)cfg->n_det * cfg->n_freq;
    for (size_t k = 0; k < nn; ++k)
      if (!(cfg->psd[k] > 0.0) || !isfinite(cfg->psd[k])) return NSS_EINVAL;
    if (kind == NSS_KIND_RB) {
      if (cfg->n_bins < 1 || cfg->n_bins > cfg->n_freq - 1) return NSS_EINVAL;
      if (!nssp::domain_ok(cfg->theta_fid)) return NSS_EINVAL;
    }
  }

  int dev_id = 0;
  NSS_CUDA(cudaGetDevice(&dev_id));
  cudaDeviceProp prop;
  NSS_CUDA(cudaGetDeviceProperties(&prop, dev_id));

  nss_handle *h = new (std::nothrow) nss_handle();
  if (!h) return NSS_ENOMEM;
  h->device = dev_id;
  h->n_sm = prop.multiProcessorCount;
  NssDev &P = h->dev;
  memset(&P, 0, sizeof(P));
  P.d = cfg->d; P.kind = kind; P.n_det = kind == NSS_KIND_GAUSS ? 0 : cfg->n_det;
  P.n_freq = kind == NSS_KIND_GAUSS ? 0 : cfg->n_freq;
  P.gmst = cfg->gmst;
  for (int j = 0; j < NSS_NSLOT; ++j) P.slot_src[j] = -1;
  for (int j = 0; j < NSS_NSLOT; ++j) {
    P.param_index[j] = j < cfg->d ? (kind == NSS_KIND_GAUSS ? j : cfg->param_index[j]) : 0;
    if (j < cfg->d) P.slot_src[P.param_index[j]] = j;
    P.theta_fixed[j] = cfg->theta_fixed[j];
    P.lo[j] = j < cfg->d ? cfg->lo[j] : 0.0;
    P.hi[j] = j < cfg->d ? cfg->hi[j] : 0.0;
    P.gauss_mu[j] = j < cfg->d ? cfg->gauss_mu[j] : 0.0;
    P.gauss_isig[j] = (j < cfg->d && kind == NSS_KIND_GAUSS) ? 1.0 / cfg->gauss_sigma[j] : 0.0;
  }
  if (kind == NSS_KIND_GAUSS) { *out = h; return NSS_OK; }

  const int n = cfg->n_freq, nd = cfg->n_det;
  const double df = cfg->df;
  for (int a = 0; a < nd; ++a) detector_tensor(cfg->det[a], P.D6[a], P.rc[a]);
  std::vector<double> f(n);
  for (int k = 0; k < n; ++k) f[k] = cfg->f_min + k * df;
  const cplx *data = reinterpret_cast<const cplx *>(cfg->data);

  double DD = 0.0;
  for (int a = 0; a < nd; ++a)
    for (int k = 0; k < n; ++k) DD += 4.0 * df * std::norm(data[(size_t)a * n + k]) / cfg->psd[(size_t)a * n + k];
  h->DD = DD;
  P.half_DD = 0.5 * DD;

  // ---- record tables ---------------------------------------------------------------------------------
  // Both likelihoods are evaluated in the same form.  With the detector waveform written as
  //     h(f) = A f^-7/6 z(f),  z = exp(-2 pi i phi(f)),  A = complex amplitude of the point (no f dependence),
  // and h0 = A0 f^-7/6 z0 the heterodyne reference (kind 0) or A0 = z0 = 1 (kind 1), the ratio is
  // r = (A/A0) (z/z0), |r| = |A/A0| at every frequency, and per detector
  //     <d,h> = Re( conj(A/A0) T ),       T = sum_rec W_rec conj(z/z0)_rec
  //     <h,h> = |A/A0|^2 ( hh0 + sum_b V_b X_b ),   X_b = Re( (z/z0)_b conj (z/z0)_{b+1} ).
  // kind 0 (O10): records are the bin edges; collecting r0 = (r_b + r_b+1)/2, r1 = (r_b+1 - r_b)/dF per edge,
  //     W_e = [e < B](A0_e/2 - A1_e/dF_e) + [e > 0](A0_e-1/2 + A1_e-1/dF_e-1),  V_b = B0_b/2,  hh0 = sum_b B0_b/2;
  //     the B1 term, 2 B1_b Re(r0 conj r1) = B1_b (|r_b+1|^2 - |r_b|^2)/dF, vanishes because |r| is constant.
  // kind 1 (O7): records are the grid frequencies; W_k = (4 df/S_k) d_k f_k^-7/6, no cross term,
  //     hh0 = sum_k (4 df/S_k) f_k^-7/3;  logL = sum_det(<d,h> - <h,h>/2) - DD/2 as for kind 0.
  int rc_up = NSS_OK;
  std::vector<double> rf;                    // record frequencies
  std::vector<double> W;                     // [nd][n_rec][2]
  std::vector<double> V;                     // [nd][n_rec]: V of the bin ending at this record (0 for record 0)
  int n_rec = 0;
  if (kind == NSS_KIND_FULL) {
    n_rec = n;
    rf = f;
    W.assign((size_t)nd * n * 2, 0.0);
    for (int a = 0; a < nd; ++a) {
      P.inv_a0[a][0] = 1.0; P.inv_a0[a][1] = 0.0;
      double hh = 0.0;
      for (int k = 0; k < n; ++k) {
        const double w = 4.0 * df / cfg->psd[(size_t)a * n + k];
        const double f76 = 1.0 / (f[k] * sqrt(cbrt(f[k])));
        const cplx dk = data[(size_t)a * n + k];
        W[((size_t)a * n + k) * 2] = w * f76 * dk.real();
        W[((size_t)a * n + k) * 2 + 1] = w * f76 * dk.imag();
        hh += w * f76 * f76;
      }
      P.hh0[a] = hh;
    }
    P.cross = 0;
  } else {
    const int B = cfg->n_bins, E = B + 1;
    P.n_bins = B; P.n_edges = E;
    h->edge_idx = choose_edges(n, cfg->f_min, df, B);
    // fiducial
    nssp::Intrinsic I0;
    nssp::intrinsic(cfg->theta_fid, I0);
    for (int j = 0; j < nssp::kNB; ++j) P.c_fid[j] = I0.c[j];
    P.c_const_fid = I0.c_const; P.tc_fid = I0.tc;
    h->summary.assign((size_t)nd * B * 6, 0.0);
    std::vector<cplx> h0(n);
    for (int a = 0; a < nd; ++a) {
      cplx amp0; double tau0;
      det_amplitude(I0, cfg->theta_fid, cfg->gmst, P.D6[a], P.rc[a], amp0, tau0);
      if (!(std::abs(amp0) > 0.0)) { nss_destroy(h); return NSS_EINVAL; }   // fiducial invisible in this detector
      const cplx inv = 1.0 / amp0;
      P.inv_a0[a][0] = inv.real(); P.inv_a0[a][1] = inv.imag();
      P.tau_fid[a] = tau0;
      host_waveform(cfg->theta_fid, P.D6[a], P.rc[a], cfg->gmst, f.data(), n, h0.data());
      for (int b = 0; b < B; ++b) {
        const int k0 = h->edge_idx[b];
        const int k1 = b == B - 1 ? h->edge_idx[B] + 1 : h->edge_idx[b + 1];     // last bin owns its right edge (A8)
        const double fbar = 0.5 * (f[h->edge_idx[b]] + f[h->edge_idx[b + 1]]);
        cplx a0 = 0, a1 = 0; double b0 = 0, b1 = 0;
        for (int k = k0; k < k1; ++k) {
          const double w = 4.0 * df / cfg->psd[(size_t)a * n + k];
          const cplx dh = data[(size_t)a * n + k] * std::conj(h0[k]) * w;
          const double hh = std::norm(h0[k]) * w;
          a0 += dh; a1 += dh * (f[k] - fbar);
          b0 += hh; b1 += hh * (f[k] - fbar);
        }
        double *s = &h->summary[((size_t)a * B + b) * 6];
        s[0] = a0.real(); s[1] = a0.imag(); s[2] = a1.real(); s[3] = a1.imag(); s[4] = b0; s[5] = b1;
      }
    }
    n_rec = E;
    rf.resize(E);
    for (int e = 0; e < E; ++e) rf[e] = f[h->edge_idx[e]];
    W.assign((size_t)nd * E * 2, 0.0);
    V.assign((size_t)nd * E, 0.0);
    for (int a = 0; a < nd; ++a) {
      double hh = 0.0;
      for (int b = 0; b < B; ++b) {
        const double *s = &h->summary[((size_t)a * B + b) * 6];
        const double idF = 1.0 / (rf[b + 1] - rf[b]);
        double *wl = &W[((size_t)a * E + b) * 2], *wr = &W[((size_t)a * E + b + 1) * 2];
        wl[0] += 0.5 * s[0] - s[2] * idF; wl[1] += 0.5 * s[1] - s[3] * idF;
        wr[0] += 0.5 * s[0] + s[2] * idF; wr[1] += 0.5 * s[1] + s[3] * idF;
        V[(size_t)a * E + b + 1] = 0.5 * s[4];
        hh += 0.5 * s[4];
      }
      P.hh0[a] = hh;
    }
    P.cross = 1;
  }
  {
    const int cr = P.cross, per = 2 + cr;
    P.n_rec = n_rec;
    // (1) AoS records for the thread-per-point kernel: g0..g7, f, pad, then per detector (Wr, Wi[, V])
    const int rs = (10 + per * nd + 1) & ~1;
    std::vector<double> rec((size_t)n_rec * rs, 0.0);
    for (int e = 0; e < n_rec; ++e) {
      double *r = &rec[(size_t)e * rs];
      nssp::basis(rf[e], r);
      r[8] = rf[e];
      for (int a = 0; a < nd; ++a) {
        r[10 + per * a] = W[((size_t)a * n_rec + e) * 2];
        r[11 + per * a] = W[((size_t)a * n_rec + e) * 2 + 1];
        if (cr) r[12 + per * a] = V[(size_t)a * n_rec + e];
      }
    }
    P.rec_rs = rs;
    rc_up = upload(rec, &h->d_rec, &h->rec_bytes);
    P.rec = h->d_rec;
    // (2) sub-warp layouts, round major, for L = 8, 16, 32 lanes per point: lane l owns records l*m+1 .. l*m+m
    //     (rounds 1..m) and evaluates record l*m in round 0 (the left edge of its first bin; its W counts for
    //     lane 0 only).  Records past the end repeat the last one with zero weights.  L < 32 (several points
    //     per warp) is built while it keeps m <= 32.
    for (int li = 0; li < 3; ++li) {
      const int L = 8 << li;
      const int m = n_rec > 1 ? (n_rec - 1 + L - 1) / L : 1;
      if (L < 32 && (kind != NSS_KIND_RB || m > 32)) continue;
      P.soa_m[li] = m;
      const size_t r0_sz = (size_t)(9 + 2 * nd) * L, round_sz = (size_t)(9 + per * nd) * L;
      std::vector<double> soa(r0_sz + (size_t)m * round_sz, 0.0);
      for (int l = 0; l < L; ++l) {
        for (int j = 0; j <= m; ++j) {
          double *te = j == 0 ? soa.data() : soa.data() + r0_sz + (size_t)(j - 1) * round_sz;
          const int e0 = l * m + j;
          const int e = e0 < n_rec ? e0 : n_rec - 1;
          double g[nssp::kNB];
          nssp::basis(rf[e], g);
          for (int c = 0; c < 8; ++c) te[c * L + l] = g[c];
          te[8 * L + l] = rf[e];
          if (e0 >= n_rec || (j == 0 && l != 0)) continue;
          for (int a = 0; a < nd; ++a) {
            te[(9 + per_of(j, per) * a) * L + l] = W[((size_t)a * n_rec + e) * 2];
            te[(10 + per_of(j, per) * a) * L + l] = W[((size_t)a * n_rec + e) * 2 + 1];
            if (cr && j > 0) te[(11 + per * a) * L + l] = V[(size_t)a * n_rec + e];
          }
        }
      }
      if (rc_up == NSS_OK) rc_up = upload(soa, &h->d_soa[li], &h->soa_bytes[li]);
      P.soa[li] = h->d_soa[li];
    }
  }
  if (rc_up != NSS_OK) { nss_destroy(h); return rc_up; }
  *out = h;
  return NSS_OK;
}

extern "C" int nss_get_tables(nss_handle *h, int32_t *edge_idx_host, double *summary_host, double *dd_host)
{
  if (!h) return NSS_EINVAL;
  if (dd_host) *dd_host = h->DD;
  if (h->dev.kind != NSS_KIND_RB) return (edge_idx_host || summary_host) ? NSS_EINVAL : NSS_OK;
  if (edge_idx_host) memcpy(edge_idx_host, h->edge_idx.data(), h->edge_idx.size() * sizeof(int32_t));
  if (summary_host) memcpy(summary_host, h->summary.data(), h->summary.size() * sizeof(double));
  return NSS_OK;
}

extern "C" int nss_set_loglike_variant(nss_handle *h, int32_t variant)
{
  if (!h || variant < 0 || variant > 2) return NSS_EINVAL;
  h->loglike_variant = variant;
  return NSS_OK;
}

extern "C" int64_t nss_launch_count(const nss_handle *h) { return h ? h->launches : 0; }
