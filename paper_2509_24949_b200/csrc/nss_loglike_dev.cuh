// nss_loglike_dev.cuh — device functions of the likelihood kernels (K1 relative binning, K2 full grid).
//
// Shared by the batch kernels (nss_loglike.cu) and the slice-sampling kernel (nss_sampler.cu), where one
// warp evaluates one point co-operatively: the canonical parameter vector sits in a per-warp shared-memory
// scratch, the transcendental part of the per-point setup is spread over lanes (same instruction, different
// argument) and broadcast by shuffles, and lanes own contiguous slices of the bins.
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

__device__ __forceinline__ double shfl_d(double v, int src) { return __shfl_sync(0xffffffffu, v, src); }

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;       // butterfly: every lane ends with the same bits
}

// ---- per-point quantities -------------------------------------------------------------------------
// canonical vector from sampled coordinates held in memory (global or shared): slot t takes
// theta[slot_src[t]] if sampled, else the fixed value.  All indices are uniform.
__device__ __forceinline__ void canon_from_mem(const NssDev &P, const double *__restrict__ theta, double *th)
{
#pragma unroll
  for (int t = 0; t < NSS_NSLOT; ++t) {
    const int s = P.slot_src[t];
    th[t] = s >= 0 ? theta[s] : P.theta_fixed[t];
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
__device__ __forceinline__ void rb_finish_point(const NssDev &P, const nssp::Intrinsic &I, const nssp::Sky &S, RbPoint<NDET> &R)
{
#pragma unroll
  for (int j = 0; j < kNB; ++j) R.dc[j] = I.c[j] - P.c_fid[j];
  R.dconst = I.c_const - P.c_const_fid;
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

// one thread does everything (batch kernel, one thread per point)
template <int NDET>
__device__ __forceinline__ void rb_point(const NssDev &P, const double *th, RbPoint<NDET> &R)
{
  nssp::Intrinsic I;
  nssp::intrinsic(th, I);
  nssp::Sky S;
  nssp::sky_frame(P.gmst, th[9], th[10], th[8], S);
  rb_finish_point<NDET>(P, I, S, R);
}

// One warp, same th[] in every lane.  The transcendental calls are spread over lanes and broadcast:
//   sincos: lane 0 gmst - ra, 1 dec, 2 psi, 3 iota          (one call instead of four)
//   log   : lane 0 pi G Mc / c^3, lane 1 eta                 (u = (pi M)^(1/3) via ln u = ln(.)/3 - ln(eta)/5)
//   exp   : lane 0 u, lane 1 1/u, lane 2 (G Mc/c^3)^(5/6)
// Every lane ends with identical bits (all inputs of the replicated arithmetic come from one lane).
__device__ __forceinline__ void point_setup_warp(const NssDev &P, const double *th, nssp::Intrinsic &I, nssp::Sky &S)
{
  const int lane = threadIdx.x & 31;
  const double q = th[1];
  const double m1 = 1.0 / (1.0 + q), m2 = q * m1;
  const double eta = q * m1 * m1;
  // stage 1: four angles
  const double ang = lane == 0 ? P.gmst - th[9] : lane == 1 ? th[10] : lane == 2 ? th[8] : th[7];
  double sn, cs;
  sincos(ang, &sn, &cs);
  const double sg = shfl_d(sn, 0), cg = shfl_d(cs, 0), sd = shfl_d(sn, 1), cd = shfl_d(cs, 1), sp = shfl_d(sn, 2),
               cp = shfl_d(cs, 2), ci = shfl_d(cs, 3);
  nssp::sky_from_sincos(sg, cg, sd, cd, sp, cp, S);
  // stage 2: two logarithms
  const double mcs = th[0] * nssp::kGMsun;                       // G Mc / c^3 [s]
  const double lg = log(lane == 0 ? nssp::kPi * mcs : eta);
  const double ln_pimc = shfl_d(lg, 0), ln_eta = shfl_d(lg, 1);
  const double lnu = ln_pimc * (1.0 / 3.0) - 0.2 * ln_eta;       // ln (pi M)^(1/3), M = Mc eta^(-3/5)
  // stage 3: three exponentials
  const double ln_mcs = ln_pimc - 1.1447298858494001741;         // ln(pi)
  const double ex = exp(lane == 0 ? lnu : lane == 1 ? -lnu : (5.0 / 6.0) * ln_mcs);
  const double u = shfl_d(ex, 0), iu = shfl_d(ex, 1), mc56 = shfl_d(ex, 2);
  nssp::intrinsic_from(th, eta, m1, m2, u, iu, lnu, mc56, ci, I);
}

template <int NDET>
__device__ __forceinline__ void rb_point_warp(const NssDev &P, const double *th, RbPoint<NDET> &R)
{
  nssp::Intrinsic I;
  nssp::Sky S;
  point_setup_warp(P, th, I, S);
  rb_finish_point<NDET>(P, I, S, R);
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

// ---- K1, one warp per point: lane l owns bins [l*m, l*m+m) and edges [l*m, l*m+m].
// `tab` = warp layout (shared or global), edge-round major so every offset inside a round is an immediate:
//   round 0 : [9][32]                      g0..g7, F of edge l*m
//   round j : [9][32] then [NDET*6][32]    edge l*m+j, then the six pre-scaled terms of bin l*m+j-1, j = 1..m
template <int NDET>
__device__ __forceinline__ int rb_warp_table_doubles(int m) { return (9 + m * (9 + 6 * NDET)) * 32; }

template <int NDET>
__device__ __forceinline__ double rb_loglike_warp(const NssDev &P, const double *__restrict__ tab,
                                                  const RbPoint<NDET> &R)
{
  const int lane = threadIdx.x & 31, m = P.rb_m;
  const double *t = tab + lane;
  double pr[NDET], pi[NDET], acc[NDET];
  {
    double ph = R.dconst;
#pragma unroll
    for (int c = 0; c < kNB; ++c) ph = fma(R.dc[c], t[c * 32], ph);
    const double F = t[8 * 32];
#pragma unroll
    for (int a = 0; a < NDET; ++a) {
      double s, c;
      nssp::sincos_turns(fma(F, R.ft[a], ph), &s, &c);
      pr[a] = fma(R.ar[a], c, R.ai[a] * s);
      pi[a] = fma(R.ai[a], c, -R.ar[a] * s);
      acc[a] = 0.0;
    }
  }
  t += 9 * 32;
  for (int j = 1; j <= m; ++j, t += (9 + 6 * NDET) * 32) {
    double ph = R.dconst;
#pragma unroll
    for (int c = 0; c < kNB; ++c) ph = fma(R.dc[c], t[c * 32], ph);
    const double F = t[8 * 32];
#pragma unroll
    for (int a = 0; a < NDET; ++a) {
      double s, c;
      nssp::sincos_turns(fma(F, R.ft[a], ph), &s, &c);
      const double rr = fma(R.ar[a], c, R.ai[a] * s);
      const double ri = fma(R.ai[a], c, -R.ar[a] * s);
      const double *q = t + (9 + 6 * a) * 32;
      acc[a] += bin_term(q[0], q[32], q[64], q[96], q[128], q[160], pr[a], pi[a], rr, ri);
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
  nssp::Sky S;
  point_setup_warp(P, th, I, S);
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

// O16 Gaussian test likelihood on sampled coordinates (memory operand; uniform indices)
__device__ __forceinline__ double gauss_loglike(const NssDev &P, const double *__restrict__ theta)
{
  double s = 0.0;
  bool ok = true;
#pragma unroll
  for (int j = 0; j < NSS_NSLOT; ++j)
    if (j < P.d) {
      const double x = theta[j];
      ok = ok && isfinite(x);
      const double z = (x - P.gauss_mu[j]) * P.gauss_isig[j];
      s = fma(z, z, s);
    }
  return ok ? -0.5 * s : -INFINITY;
}

// One warp evaluates logL of the sampled coordinates `theta` (memory the whole warp can read: global or the
// warp's shared scratch); every lane returns the same bits.  `tab` = warp-layout RB table (shared or
// global), ignored for other kinds.
template <int NDET, int KIND>
__device__ __forceinline__ double loglike_warp(const NssDev &P, const double *__restrict__ tab, const double *__restrict__ theta)
{
  if (KIND == NSS_KIND_GAUSS) return gauss_loglike(P, theta);
  double th[NSS_NSLOT];
  canon_from_mem(P, theta, th);
  if (!nssp::domain_ok(th)) return -INFINITY;
  if (KIND == NSS_KIND_RB) {
    RbPoint<NDET> R;
    rb_point_warp<NDET>(P, th, R);
    return rb_loglike_warp<NDET>(P, tab, R);
  }
  return full_loglike_warp<NDET>(P, th);
}

}  // namespace nssk
