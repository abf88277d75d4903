// nss_loglike_dev.cuh — device functions of the likelihood kernels (K1 relative binning, K2 full grid).
//
// Shared by the batch kernels (nss_loglike.cu) and the slice-sampling kernel (nss_sampler.cu), where one
// warp evaluates one point co-operatively: the per-point setup is spread over lanes (same instruction stream,
// different argument or coefficient per lane) and broadcast through a per-warp shared-memory scratch, and
// lanes own contiguous slices of the records (bin edges or grid frequencies).
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

// A point relative to the reference (nss_setup.cu "record tables"): phase difference in turns
// phi(f) = dconst + sum_j dc_j g_j(f) + f ft_det, and the complex amplitude ratio A/A0 per detector.
template <int NDET>
struct RbPoint {
  double dc[kNB];
  double dconst;
  double ft[NDET];            // coefficient of f: (tc + tau_det) - (tc_fid + tau_fid_det)
  double ar[NDET], ai[NDET];  // amplitude ratio
};

// one thread does everything (batch kernel, one thread per point)
template <int NDET>
__device__ __forceinline__ void rb_point(const NssDev &P, const double *th, RbPoint<NDET> &R)
{
  nssp::Intrinsic I;
  nssp::intrinsic(th, I);
  nssp::Sky S;
  nssp::sky_frame(P.gmst, th[9], th[10], th[8], S);
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

// ---- a SUB-WARP of LANES lanes (8 or 32) per point: the per-point setup is spread over lanes ----------------
// A warp holds 32/LANES sub-warps that run in lockstep, each on its own point, so every instruction of the
// per-point setup is shared by 32/LANES points.
// Per-CTA constants in shared memory (filled once per kernel by sub_consts_init):
//   coef[9][8] : lane j < 8 builds phase coefficient j as  K A_j(eta, beta, ln u) exp(p_j ln u) - c_fid_j,
//                A_j = t0 + t1 eta + t2 eta^2 + t3 eta^3 + t4 beta + t5 ln u;  rows: t0..t5, p, q, c_fid.
//                Coefficient 4 (K P5, no power of u) is cheap and computed by every lane; lane 4 builds
//                (G Mc/c^3)^(5/6) = exp(q_4 ln(G Mc/c^3)) instead (t0 = 1, no K).
//   det[12][4] : per detector D6[0..5], rc[0..2], inv_a0 re, im, tau_fid
//   dom[2][12] : open interval (lo, hi) of the physical domain per canonical slot (O2); +-inf where free,
//                so the test also rejects non-finite values
// Per-sub-warp scratch (kSubScratchDoubles): canonical parameters [12], then two broadcast rounds.
constexpr int kSubConstDoubles = 9 * 8 + 12 * 4 + 2 * 12;
constexpr int kSubScratchDoubles = 52;        // [0..11] theta (canonical), [12..27] stage 1, [28..47] stage 2

struct SubCtx {
  const double *tab;      // sub-warp-layout record table (shared or global)
  const double *consts;   // kSubConstDoubles, shared
  double *scr;            // kSubScratchDoubles, shared, private to the sub-warp
};

template <int LANES>
__host__ __device__ constexpr int lanes_index() { return LANES == 8 ? 0 : LANES == 16 ? 1 : 2; }

template <int LANES>
__device__ __forceinline__ double sub_sum(double v)
{
#pragma unroll
  for (int o = LANES / 2; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;       // butterfly inside the sub-warp: every lane of it ends with the same bits
}

__device__ __forceinline__ void sub_consts_init(const NssDev &P, double *consts)
{
  const double pi = nssp::kPi;
  for (int i = threadIdx.x; i < kSubConstDoubles; i += blockDim.x) {
    double v = 0.0;
    if (i < 72) {
      const int k = i >> 3, j = i & 7;
      // rows t0..t5 of A_j (O3 regrouped by power of f, nss_physics.cuh: intrinsic_from)
      if (k == 0)
        v = j == 0 ? 1.0 : j == 1 ? 3715.0 / 756.0 : j == 2 ? -16.0 * pi : j == 3 ? 15293365.0 / 508032.0
          : j == 4 ? 1.0
          : j == 5 ? 11583231236531.0 / 4694215680.0 - 640.0 / 3.0 * pi * pi - 6848.0 / 21.0 * nssp::kEuler
                       - 6848.0 / 21.0 * 1.3862943611198906188
          : j == 6 ? -6848.0 / 63.0 : pi * (77096675.0 / 254016.0);
      else if (k == 1)
        v = j == 1 ? 55.0 / 9.0 : j == 3 ? 27145.0 / 504.0
          : j == 5 ? -15737765635.0 / 3048192.0 + 2255.0 / 12.0 * pi * pi : j == 7 ? pi * (378515.0 / 1512.0) : 0.0;
      else if (k == 2)
        v = j == 3 ? 3085.0 / 72.0 : j == 5 ? 76055.0 / 1728.0 : j == 7 ? -pi * (74045.0 / 756.0) : 0.0;
      else if (k == 3)
        v = j == 5 ? -127825.0 / 1296.0 : 0.0;
      else if (k == 4)
        v = j == 2 ? 4.0 : 0.0;
      else if (k == 5)
        v = j == 5 ? -6848.0 / 21.0 : 0.0;
      else if (k == 6)         // power of u = (pi M)^(1/3)
        v = j == 0 ? -5.0 : j == 1 ? -3.0 : j == 2 ? -2.0 : j == 3 ? -1.0 : j == 5 ? 1.0 : j == 6 ? 1.0 : j == 7 ? 2.0 : 0.0;
      else if (k == 7)         // power of G Mc / c^3
        v = j == 4 ? 5.0 / 6.0 : 0.0;
      else
        v = j != 4 ? P.c_fid[j] : 0.0;
    } else if (i < 120) {
      const int k = (i - 72) >> 2, a = (i - 72) & 3;
      v = k < 6 ? P.D6[a][k] : k < 9 ? P.rc[a][k - 6] : k < 11 ? P.inv_a0[a][k - 9] : P.tau_fid[a];
    } else {
      const int hi = (i - 120) / 12, t = (i - 120) % 12;
      // O2: Mc > 0, 0 < q <= 1, |chi| < 1, d_L > 0
      if (!hi) v = (t == 0 || t == 1 || t == 4) ? 0.0 : (t == 2 || t == 3) ? -1.0 : -INFINITY;
      else v = t == 1 ? 1.0000000000000002 : (t == 2 || t == 3) ? 1.0 : INFINITY;
    }
    consts[i] = v;
  }
}

// The canonical parameters of the sub-warp's point are in X.scr[0..10].  Returns false (in every lane of the
// sub-warp) if the point is outside the physical domain or not finite; R is then meaningless but harmless.
// Stage 1 (one instruction stream each, a different argument per lane):
//   1/x   : lane 0: 1 + q, 1: q, 2: d_L
//   ln x  : lane 0: pi G Mc/c^3, 1: q, 2: 1 + q
//   sincos: lane 0: gmst - ra, 1: dec, 2: psi, 3: iota
// broadcast through the scratch; stage 2: lane j < 8 builds one coefficient (one exp), lane a < NDET the antenna
// response of detector a; broadcast again.  Every lane of the sub-warp ends with identical bits.
template <int NDET, int LANES>
__device__ __forceinline__ bool rb_point_sub(const NssDev &P, const SubCtx &X, RbPoint<NDET> &R)
{
  const int lane = threadIdx.x & 31, sl = lane & (LANES - 1);
  const double2 *s2 = reinterpret_cast<const double2 *>(X.scr);
  // domain test: lane sl checks slots sl, sl + LANES, ...
  bool ok = true;
#pragma unroll
  for (int t0 = 0; t0 < NSS_NSLOT; t0 += LANES) {
    const int t = t0 + sl < NSS_NSLOT ? t0 + sl : NSS_NSLOT - 1;
    const double v = X.scr[t];
    ok = ok && (v > X.consts[120 + t]) && (v < X.consts[132 + t]);
  }
  const unsigned bal = __ballot_sync(0xffffffffu, ok);
  const unsigned sub_mask = (LANES == 32 ? 0xffffffffu : ((1u << LANES) - 1u)) << (lane & ~(LANES - 1));
  ok = (bal & sub_mask) == sub_mask;
  const double2 t01 = s2[0], t23 = s2[1], t45 = s2[2], t67 = s2[3], t89 = s2[4];
  const double th10 = X.scr[10];
  const double q = t01.y, opq = 1.0 + q;
  const double mcs = t01.x * nssp::kGMsun;                       // G Mc / c^3 [s]
  {
    const double xr = sl == 0 ? opq : sl == 1 ? q : sl == 2 ? t45.x : 1.0;
    const double xl = sl == 0 ? nssp::kPi * mcs : sl == 1 ? q : sl == 2 ? opq : 1.0;
    const double xa = sl == 0 ? P.gmst - t89.y : sl == 1 ? th10 : sl == 2 ? t89.x : t67.y;
    const double rc = 1.0 / xr, lg = log(xl);
    double sn, cs;
    nssp::sincos_turns_dev(xa * 0.15915494309189533577, &sn, &cs);
    if (sl < 4) { X.scr[12 + sl] = rc; X.scr[16 + sl] = lg; X.scr[20 + sl] = sn; X.scr[24 + sl] = cs; }
  }
  __syncwarp();
  const double2 r01 = s2[6], r23 = s2[7], l01 = s2[8], l23 = s2[9], sn01 = s2[10], sn23 = s2[11], cs01 = s2[12], cs23 = s2[13];
  const double m1 = r01.x, iq = r01.y, idL = r23.x;
  const double ln_pimc = l01.x, ln_eta = l01.y - 2.0 * l23.x;
  const double ci = cs23.y;
  nssp::Sky S;
  nssp::sky_from_sincos(sn01.x, cs01.x, sn01.y, cs01.y, sn23.x, cs23.x, S);
  const double m2 = q * m1, eta = m2 * m1;
  const double lnu = ln_pimc * (1.0 / 3.0) - 0.2 * ln_eta;       // ln (pi M)^(1/3), M = Mc eta^(-3/5)
  const double ln_mcs = ln_pimc - 1.1447298858494001741;         // - ln(pi)
  const double K = (3.0 / (256.0 * nssp::kPi)) * (opq * opq * iq);     // 3/(128 eta)/(2 pi), turns
  const double beta = (113.0 / 12.0 * m1 * m1 + 6.25 * eta) * t23.x + (113.0 / 12.0 * m2 * m2 + 6.25 * eta) * t23.y;
  {
    // coefficient lane
    const int j = sl & 7;
    const double *cf = X.consts + j;
    const double E = exp(fma(cf[6 * 8], lnu, cf[7 * 8] * ln_mcs));
    double A = cf[3 * 8];
    A = fma(A, eta, cf[2 * 8]);
    A = fma(A, eta, cf[1 * 8]);
    A = fma(A, eta, cf[0]);
    A = fma(cf[4 * 8], beta, A);
    A = fma(cf[5 * 8], lnu, A);
    const double val = fma((j == 4 ? 1.0 : K) * A, E, -cf[8 * 8]);
    // detector lane
    const double *dt = X.consts + 72 + ((sl & 3) < NDET ? (sl & 3) : 0);
    double D6[6], rcv[3];
#pragma unroll
    for (int k = 0; k < 6; ++k) D6[k] = dt[4 * k];
#pragma unroll
    for (int k = 0; k < 3; ++k) rcv[k] = dt[4 * (6 + k)];
    double fp, fc, tau;
    nssp::antenna(S, D6, rcv, fp, fc, tau);
    const double hr = fp * (0.5 * (1.0 + ci * ci)), hi = -fc * ci;     // F+ (1+c^2)/2 - i Fx c
    const double i0r = dt[4 * 9], i0i = dt[4 * 10];
    const double ar = hr * i0r - hi * i0i, ai = hr * i0i + hi * i0r;
    const double ft = (t45.y - P.tc_fid) + (tau - dt[4 * 11]);
    if (sl < 8) X.scr[28 + sl] = val;
    if (sl < NDET) { X.scr[36 + 3 * sl] = ar; X.scr[37 + 3 * sl] = ai; X.scr[38 + 3 * sl] = ft; }
  }
  __syncwarp();
  {
    const double2 c01 = s2[14], c23 = s2[15], c45 = s2[16], c67 = s2[17];
    // coefficient 4 = K P5 (ln f term): computed here, its lane built (G Mc/c^3)^(5/6)
    const double kp5 = K * (nssp::kPi * (38645.0 / 756.0) - nssp::kPi * (65.0 / 9.0) * eta);
    R.dc[0] = c01.x; R.dc[1] = c01.y; R.dc[2] = c23.x; R.dc[3] = c23.y;
    R.dc[4] = kp5 - P.c_fid[4]; R.dc[5] = c45.y; R.dc[6] = c67.x; R.dc[7] = c67.y;
    const double mc56 = c45.x;
    const double amp = 0.45643546458763842789 /* sqrt(5/24) */ * 0.46619407703541166 /* pi^(-2/3) */ * mc56 * nssp::kC
                     * (idL * (1.0 / nssp::kMpc));
#pragma unroll
    for (int a = 0; a < NDET; ++a) {
      R.ar[a] = X.scr[36 + 3 * a] * amp;
      R.ai[a] = X.scr[37 + 3 * a] * amp;
      R.ft[a] = X.scr[38 + 3 * a];
    }
    // c_const = (-phic - pi/4)/(2 pi) + K P5 (1 + 3 (ln u - ln v_lso))
    R.dconst = fma(kp5, 1.0 + 3.0 * (lnu + 0.89587973461402748), (-t67.x - 0.25 * nssp::kPi) * 0.15915494309189533577)
             - P.c_const_fid;
  }
  return ok;
}

// ---- record loops ------------------------------------------------------------------------------------------
// accumulators of one detector: T = sum W conj(z), Q = sum V X, and the previous record's (cos, sin)
struct DetAcc {
  double tr, ti, q, pc, ps;
};

template <bool CROSS>
__device__ __forceinline__ void rec_term(DetAcc &A, double wr, double wi, double v, double c, double s)
{
  A.tr = fma(wr, c, A.tr); A.tr = fma(-wi, s, A.tr);
  A.ti = fma(wr, s, A.ti); A.ti = fma(wi, c, A.ti);
  if (CROSS) {
    A.q = fma(v, fma(c, A.pc, s * A.ps), A.q);
    A.pc = c; A.ps = s;
  }
}

// logL from the accumulators of one thread
template <int NDET>
__device__ __forceinline__ double finish_logl(const NssDev &P, const RbPoint<NDET> &R, const DetAcc *A)
{
  double part = 0.0, cst = P.half_DD;
#pragma unroll
  for (int a = 0; a < NDET; ++a) {
    const double h2 = 0.5 * fma(R.ar[a], R.ar[a], R.ai[a] * R.ai[a]);
    part += fma(R.ar[a], A[a].tr, R.ai[a] * A[a].ti) - h2 * A[a].q;
    cst = fma(h2, P.hh0[a], cst);
  }
  return part - cst;
}

// one thread per point: `count` records streamed from `rec` (shared memory, all lanes read the same address)
template <int NDET, bool CROSS>
__device__ __forceinline__ void records_thread(const double *__restrict__ rec, int rs, int count, const RbPoint<NDET> &R,
                                               DetAcc *A)
{
  constexpr int PER = CROSS ? 3 : 2;
#pragma unroll 2
  for (int e = 0; e < count; ++e) {
    const double *r = rec + (size_t)e * rs;
    const double2 *r2 = reinterpret_cast<const double2 *>(r);
    const double2 g01 = r2[0], g23 = r2[1], g45 = r2[2], g67 = r2[3];
    const double F = r[8];
    double ph = R.dconst;
    ph = fma(R.dc[0], g01.x, ph); ph = fma(R.dc[1], g01.y, ph);
    ph = fma(R.dc[2], g23.x, ph); ph = fma(R.dc[3], g23.y, ph);
    ph = fma(R.dc[4], g45.x, ph); ph = fma(R.dc[5], g45.y, ph);
    ph = fma(R.dc[6], g67.x, ph); ph = fma(R.dc[7], g67.y, ph);
#pragma unroll
    for (int a = 0; a < NDET; ++a) {
      double s, c;
      nssp::sincos_turns_dev(fma(F, R.ft[a], ph), &s, &c);
      rec_term<CROSS>(A[a], r[10 + PER * a], r[11 + PER * a], CROSS ? r[12 + PER * a] : 0.0, c, s);
    }
  }
}

// a sub-warp per point: lane l (of LANES) evaluates record l*m in round 0 and records l*m+1 .. l*m+m in rounds
// 1..m (layout in nss_setup.cu); every offset inside a round is an immediate and the reads are conflict-free
// (the sub-warps of a warp read the same words: broadcast).
template <int NDET, bool CROSS, int LANES>
__device__ __forceinline__ int sub_table_doubles(int m) { return ((9 + 2 * NDET) + m * (9 + (CROSS ? 3 : 2) * NDET)) * LANES; }

template <int NDET, bool CROSS, int LANES>
__device__ __forceinline__ double records_sub(const NssDev &P, const double *__restrict__ tab, const RbPoint<NDET> &R)
{
  constexpr int PER = CROSS ? 3 : 2;
  const int sl = threadIdx.x & (LANES - 1), m = P.soa_m[lanes_index<LANES>()];
  const double *t = tab + sl;
  DetAcc A[NDET];
  {
    double ph = R.dconst;
#pragma unroll
    for (int c = 0; c < kNB; ++c) ph = fma(R.dc[c], t[c * LANES], ph);
    const double F = t[8 * LANES];
#pragma unroll
    for (int a = 0; a < NDET; ++a) {
      double s, c;
      nssp::sincos_turns_dev(fma(F, R.ft[a], ph), &s, &c);
      const double wr = t[(9 + 2 * a) * LANES], wi = t[(10 + 2 * a) * LANES];
      A[a].tr = fma(wr, c, -wi * s);
      A[a].ti = fma(wr, s, wi * c);
      A[a].q = 0.0; A[a].pc = c; A[a].ps = s;
    }
  }
  t += (9 + 2 * NDET) * LANES;
  // The sub-warp's warp is often alone on its SM sub-partition (a DFMA result takes 8 cycles, the pipe accepts one
  // warp DFMA per ~2.2): two records are in flight per iteration and the phase is a two-chain sum.
  auto phase_of = [&](const double *tt, double &F) {
    double pa = fma(R.dc[0], tt[0], R.dconst), pb = R.dc[4] * tt[4 * LANES];
#pragma unroll
    for (int c = 1; c < 4; ++c) { pa = fma(R.dc[c], tt[c * LANES], pa); pb = fma(R.dc[4 + c], tt[(4 + c) * LANES], pb); }
    F = tt[8 * LANES];
    return pa + pb;
  };
  constexpr int STRIDE = (9 + PER * NDET) * LANES;
  if (CROSS) {
    // relative binning: the table is in shared memory
#pragma unroll 2
    for (int j = 1; j <= m; ++j, t += STRIDE) {
      double F;
      const double ph = phase_of(t, F);
#pragma unroll
      for (int a = 0; a < NDET; ++a) {
        double s, c;
        nssp::sincos_turns_dev(fma(F, R.ft[a], ph), &s, &c);
        const double *w = t + (9 + PER * a) * LANES;
        rec_term<CROSS>(A[a], w[0], w[LANES], w[2 * LANES], c, s);
      }
    }
  } else {
    // full grid: the table is read from L2, so the loop is software-pipelined: the loads and the phase of record
    // j+1 are issued while the sincos polynomials of record j run (2.4x faster than the plain loop on B200)
    double Fn, phn = phase_of(t, Fn);
#pragma unroll 2
    for (int j = 1; j <= m; ++j, t += STRIDE) {
      const double ph = phn, F = Fn;
      if (j < m) phn = phase_of(t + STRIDE, Fn);
#pragma unroll
      for (int a = 0; a < NDET; ++a) {
        double s, c;
        nssp::sincos_turns_dev(fma(F, R.ft[a], ph), &s, &c);
        const double *w = t + (9 + PER * a) * LANES;
        rec_term<CROSS>(A[a], w[0], w[LANES], 0.0, c, s);
      }
    }
  }
  double part = 0.0, cst = P.half_DD;
#pragma unroll
  for (int a = 0; a < NDET; ++a) {
    const double h2 = 0.5 * fma(R.ar[a], R.ar[a], R.ai[a] * R.ai[a]);
    part += fma(R.ar[a], A[a].tr, R.ai[a] * A[a].ti) - h2 * A[a].q;
    cst = fma(h2, P.hh0[a], cst);
  }
  return sub_sum<LANES>(part) - cst;
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

// Every sub-warp of the warp evaluates logL of the canonical parameters in its X.scr[0..10] (written by the
// caller, followed by __syncwarp()); every lane of a sub-warp returns the same bits.  `want` says whether this
// sub-warp needs a value at all: the warp returns early when none of its sub-warps does.  The whole warp must
// call this together.
template <int NDET, int KIND, int LANES>
__device__ __forceinline__ double loglike_sub(const NssDev &P, const SubCtx &X, bool want)
{
  if (!__any_sync(0xffffffffu, want)) return -INFINITY;
  RbPoint<NDET> R;
  const bool ok = rb_point_sub<NDET, LANES>(P, X, R);
  const double l = records_sub<NDET, KIND == NSS_KIND_RB, LANES>(P, X.tab, R);
  return ok ? l : -INFINITY;
}

}  // namespace nssk
