// nss_loglike_dev.cuh — device functions of the likelihood kernels (K1 relative binning, K2 full grid).
//
// Shared by the batch kernels (nss_loglike.cu) and the persistent slice-sampling kernel
// (nss_sampler.cu), where one warp evaluates one point co-operatively.
#pragma once
#include "nss_internal.cuh"

namespace nssk {

using nssp::kNB;

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---- TMA (1-D bulk) staging of a table into shared memory -----------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes)
{
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_LOOP:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE;\n\t"
      "bra WAIT_LOOP;\n\t"
      "DONE:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst_smem, const void *src_gmem, uint32_t bytes, uint64_t *bar)
{
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
// one thread stages `bytes` (multiple of 16) from global to shared in <= 32 KB bulk copies
__device__ __forceinline__ void stage_table(void *dst_smem, const void *src, uint32_t bytes, uint64_t *bar)
{
  mbar_expect_tx(bar, bytes);
  const uint32_t piece = 32768u;
  for (uint32_t off = 0; off < bytes; off += piece) {
    const uint32_t nb = bytes - off < piece ? bytes - off : piece;
    bulk_g2s((char *)dst_smem + off, (const char *)src + off, nb, bar);
  }
}

// ---- per-point quantities -------------------------------------------------------------------------
__device__ __forceinline__ void canon_from_sampled(const NssDev &P, const double *theta, double *th)
{
#pragma unroll
  for (int j = 0; j < NSS_NSLOT; ++j) th[j] = P.theta_fixed[j];
#pragma unroll
  for (int j = 0; j < NSS_NSLOT; ++j)
    if (j < P.d) {
      const int s = P.param_index[j];
      const double v = theta[j];
#pragma unroll
      for (int t = 0; t < NSS_NSLOT; ++t)
        if (t == s) th[t] = v;
    }
}

// heterodyned point: phase difference to the fiducial (turns) and complex amplitude ratio per detector
template <int NDET>
struct RbPoint {
  double dc[kNB];
  double dconst;
  double ft[NDET];            // coefficient of F_e: (tc + tau_det) - (tc_fid + tau_fid_det)
  double ar[NDET], ai[NDET];  // amplitude ratio
};

template <int NDET>
__device__ __forceinline__ void rb_point(const NssDev &P, const double *th, RbPoint<NDET> &R)
{
  nssp::Intrinsic I;
  nssp::intrinsic(th, I);
#pragma unroll
  for (int j = 0; j < kNB; ++j) R.dc[j] = I.c[j] - P.c_fid[j];
  R.dconst = I.c_const - P.c_const_fid;
  nssp::Sky S;
  nssp::sky_frame(P.gmst, th[9], th[10], th[8], S);
  const double ci = I.cos_iota;
  const double pp = 0.5 * (1.0 + ci * ci) * I.amp, pc = -ci * I.amp;
#pragma unroll
  for (int a = 0; a < NDET; ++a) {
    double fp, fc, tau;
    nssp::antenna(S, P.D6[a], P.rc[a], fp, fc, tau);
    const double hr = fp * pp, hi = fc * pc;                      // amp * (F+ (1+c^2)/2 - i Fx c)
    R.ar[a] = hr * P.inv_a0[a][0] - hi * P.inv_a0[a][1];
    R.ai[a] = hr * P.inv_a0[a][1] + hi * P.inv_a0[a][0];
    R.ft[a] = (I.tc - P.tc_fid) + (tau - P.tau_fid[a]);
  }
}

// bin contribution from the waveform ratio at the bin's two edges (pre-scaled terms q[0..5], see nss_setup.cu)
__device__ __forceinline__ double bin_term(double q0, double q1, double q2, double q3, double q4, double q5,
                                           double r0r, double r0i, double r1r, double r1i)
{
  const double sr = r1r + r0r, si = r1i + r0i, tr = r1r - r0r, ti = r1i - r0i;
  double lin = q0 * sr;
  lin = fma(q1, si, lin);
  lin = fma(q2, tr, lin);
  lin = fma(q3, ti, lin);
  const double ss = fma(sr, sr, si * si);
  const double st = fma(sr, tr, si * ti);
  return fma(q4, ss, fma(q5, st, lin));
}

// ---- K1, one thread per point: records streamed from `rec` (shared or global), all lanes read the
// same address (broadcast) --------------------------------------------------------------------------
template <int NDET>
__device__ __forceinline__ double rb_loglike_thread(const NssDev &P, const double *__restrict__ rec,
                                                    const RbPoint<NDET> &R)
{
  const int E = P.n_edges, rs = P.rb_rs;
  double pr[NDET], pi[NDET], acc[NDET];
#pragma unroll
  for (int a = 0; a < NDET; ++a) { pr[a] = 0.0; pi[a] = 0.0; acc[a] = 0.0; }
  for (int e = 0; e < E; ++e) {
    const double2 *r2 = reinterpret_cast<const double2 *>(rec + (size_t)e * rs);
    const double2 g01 = r2[0], g23 = r2[1], g45 = r2[2], g67 = r2[3], fx = r2[4];
    double ph = R.dconst;
    ph = fma(R.dc[0], g01.x, ph); ph = fma(R.dc[1], g01.y, ph);
    ph = fma(R.dc[2], g23.x, ph); ph = fma(R.dc[3], g23.y, ph);
    ph = fma(R.dc[4], g45.x, ph); ph = fma(R.dc[5], g45.y, ph);
    ph = fma(R.dc[6], g67.x, ph); ph = fma(R.dc[7], g67.y, ph);
#pragma unroll
    for (int a = 0; a < NDET; ++a) {
      double s, c;
      nssp::sincos_turns(fma(fx.x, R.ft[a], ph), &s, &c);
      const double rr = fma(R.ar[a], c, R.ai[a] * s);
      const double ri = fma(R.ai[a], c, -R.ar[a] * s);
      const double2 q01 = r2[5 + 3 * a], q23 = r2[6 + 3 * a], q45 = r2[7 + 3 * a];
      acc[a] += bin_term(q01.x, q01.y, q23.x, q23.y, q45.x, q45.y, pr[a], pi[a], rr, ri);
      pr[a] = rr; pi[a] = ri;
    }
  }
  double tot = 0.0;
#pragma unroll
  for (int a = 0; a < NDET; ++a) tot += acc[a];
  return tot - P.half_DD;
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;       // butterfly: every lane ends with the same bits
}

// ---- K1, one warp per point: lane l owns bins [l*m, l*m+m); `tab` = warp layout (shared or global)
template <int NDET>
__device__ __forceinline__ double rb_loglike_warp(const NssDev &P, const double *__restrict__ tab,
                                                  const RbPoint<NDET> &R)
{
  const int lane = threadIdx.x & 31, m = P.rb_m;
  const double *te = tab + lane;
  const double *tb = tab + (size_t)9 * (m + 1) * 32 + lane;
  double pr[NDET], pi[NDET], acc[NDET];
#pragma unroll
  for (int a = 0; a < NDET; ++a) { pr[a] = 0.0; pi[a] = 0.0; acc[a] = 0.0; }
  for (int j = 0; j <= m; ++j) {
    double ph = R.dconst;
#pragma unroll
    for (int c = 0; c < kNB; ++c) ph = fma(R.dc[c], te[((size_t)c * (m + 1) + j) * 32], ph);
    const double F = te[((size_t)8 * (m + 1) + j) * 32];
#pragma unroll
    for (int a = 0; a < NDET; ++a) {
      double s, c;
      nssp::sincos_turns(fma(F, R.ft[a], ph), &s, &c);
      const double rr = fma(R.ar[a], c, R.ai[a] * s);
      const double ri = fma(R.ai[a], c, -R.ar[a] * s);
      if (j > 0) {
        const double *q = tb + ((size_t)(a * 6) * m + (j - 1)) * 32;
        const size_t st = (size_t)m * 32;
        acc[a] += bin_term(q[0], q[st], q[2 * st], q[3 * st], q[4 * st], q[5 * st], pr[a], pi[a], rr, ri);
      }
      pr[a] = rr; pi[a] = ri;
    }
  }
  double tot = 0.0;
#pragma unroll
  for (int a = 0; a < NDET; ++a) tot += acc[a];
  return warp_sum(tot) - P.half_DD;
}

// ---- K2, full grid, one warp per point: lanes stride over frequencies, 128-bit loads -----------------
template <int NDET>
__device__ __forceinline__ double full_loglike_warp(const NssDev &P, const double *th)
{
  nssp::Intrinsic I;
  nssp::intrinsic(th, I);
  nssp::Sky S;
  nssp::sky_frame(P.gmst, th[9], th[10], th[8], S);
  const double ci = I.cos_iota;
  const double pp = 0.5 * (1.0 + ci * ci) * I.amp, pc = -ci * I.amp;
  double hr[NDET], hi[NDET], ft[NDET], acc[NDET];
#pragma unroll
  for (int a = 0; a < NDET; ++a) {
    double fp, fc, tau;
    nssp::antenna(S, P.D6[a], P.rc[a], fp, fc, tau);
    hr[a] = fp * pp; hi[a] = fc * pc; ft[a] = I.tc + tau; acc[a] = 0.0;
  }
  const int lane = threadIdx.x & 31, n = P.n_freq, rs = P.full_rs;
  for (int k = lane; k < n; k += 32) {
    const double2 *r2 = reinterpret_cast<const double2 *>(P.full_rec + (size_t)k * rs);
    const double2 g01 = __ldg(r2), g23 = __ldg(r2 + 1), g45 = __ldg(r2 + 2), g67 = __ldg(r2 + 3), fx = __ldg(r2 + 4);
    double ph = I.c_const;
    ph = fma(I.c[0], g01.x, ph); ph = fma(I.c[1], g01.y, ph);
    ph = fma(I.c[2], g23.x, ph); ph = fma(I.c[3], g23.y, ph);
    ph = fma(I.c[4], g45.x, ph); ph = fma(I.c[5], g45.y, ph);
    ph = fma(I.c[6], g67.x, ph); ph = fma(I.c[7], g67.y, ph);
    const double *rd = P.full_rec + (size_t)k * rs + 10;
#pragma unroll
    for (int a = 0; a < NDET; ++a) {
      double s, c;
      nssp::sincos_turns(fma(fx.x, ft[a], ph), &s, &c);
      const double ar = hr[a] * fx.y, ai = hi[a] * fx.y;         // amplitude * f^-7/6
      const double mr = fma(ar, c, ai * s), mi = fma(ai, c, -ar * s);
      const double dr = __ldg(rd + 3 * a) - mr, di = __ldg(rd + 3 * a + 1) - mi;
      acc[a] = fma(__ldg(rd + 3 * a + 2), fma(dr, dr, di * di), acc[a]);
    }
  }
  double tot = 0.0;
#pragma unroll
  for (int a = 0; a < NDET; ++a) tot += acc[a];
  return -0.5 * warp_sum(tot);
}

// O16 Gaussian test likelihood on sampled coordinates
__device__ __forceinline__ double gauss_loglike(const NssDev &P, const double *theta)
{
  double s = 0.0;
  bool ok = true;
#pragma unroll
  for (int j = 0; j < NSS_NSLOT; ++j)
    if (j < P.d) {
      ok = ok && isfinite(theta[j]);
      const double z = (theta[j] - P.gauss_mu[j]) * P.gauss_isig[j];
      s = fma(z, z, s);
    }
  return ok ? -0.5 * s : -INFINITY;
}

// One warp evaluates logL of sampled coordinates theta (identical in all lanes); every lane returns
// the same bits.  `tab` = warp-layout RB table (shared or global), ignored for other kinds.
template <int NDET>
__device__ __forceinline__ double loglike_warp(const NssDev &P, const double *__restrict__ tab, const double *theta)
{
  if (P.kind == NSS_KIND_GAUSS) return gauss_loglike(P, theta);
  double th[NSS_NSLOT];
  canon_from_sampled(P, theta, th);
  if (!nssp::domain_ok(th)) return -INFINITY;
  if (P.kind == NSS_KIND_RB) {
    RbPoint<NDET> R;
    rb_point<NDET>(P, th, R);
    return rb_loglike_warp<NDET>(P, tab, R);
  }
  return full_loglike_warp<NDET>(P, th);
}

}  // namespace nssk
