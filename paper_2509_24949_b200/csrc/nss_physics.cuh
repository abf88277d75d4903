// nss_physics.cuh — waveform / detector-response arithmetic of the CUDA path (host setup + kernels).
//
// TaylorF2 3.5PN phase + 1.5PN spin-orbit, Newtonian amplitude (BASELINE.json
// configs) and the detector response (O4), arranged for the kernels:
//
//   phase in TURNS   Psi(f)/(2 pi) = sum_{j<8} c_j g_j(f) + c_const + f * tc
//   basis            g = f^-5/3, f^-1, f^-2/3, f^-1/3, ln f, f^1/3, f^1/3 ln f, f^2/3
//
// so a kernel evaluates the phase at a tabulated frequency with 8 FMAs against theta-dependent
// coefficients, plus one FMA per detector for the arrival-time term f*(tc + dt_det).
// This file shares nothing with oracle/ (which evaluates the defining formula directly).
#pragma once
#include <math.h>
#include <stdint.h>

#if defined(__CUDACC__)
#define NSS_HD __host__ __device__ __forceinline__
#else
#define NSS_HD inline
#endif

namespace nssp {

constexpr double kGMsun = 4.925490947641267e-6;   // G Msun / c^3 [s]   (O1)
constexpr double kMpc = 3.085677581491367e22;     // [m]
constexpr double kC = 299792458.0;                // [m/s]
constexpr double kEuler = 0.5772156649015329;
constexpr double kPi = 3.14159265358979323846;
constexpr int kNB = 8;                             // phase basis functions (above)
constexpr int kNSlot = 11;

struct Intrinsic {
  double c[kNB];     // phase coefficients, turns
  double c_const;    // frequency-independent phase, turns
  double tc;         // coefficient of f, turns/Hz = seconds
  double amp;        // Newtonian amplitude A (multiplies f^-7/6), O3
  double cos_iota;
};

NSS_HD bool domain_ok(const double *th)
{
  bool ok = true;
#pragma unroll
  for (int j = 0; j < kNSlot; ++j) ok = ok && isfinite(th[j]);
  ok = ok && (th[0] > 0.0) && (th[1] > 0.0) && (th[1] <= 1.0);
  ok = ok && (fabs(th[2]) < 1.0) && (fabs(th[3]) < 1.0) && (th[4] > 0.0);
  return ok;
}

// O3: PN coefficients regrouped by power of f.  v = u f^(1/3), u = (pi M)^(1/3).
// Inputs: eta, m1 = m_1/M, m2 = m_2/M, u, iu = 1/u, lnu = ln u, mc56 = (G Mc/c^3)^(5/6), ci = cos(iota).
NSS_HD void intrinsic_from(const double *th, double eta, double m1, double m2, double u, double iu, double lnu, double mc56,
                           double ci, Intrinsic &I)
{
  const double chi1 = th[2], chi2 = th[3], dL = th[4];
  const double K = 3.0 / (128.0 * eta) / (2.0 * kPi);          // turns
  const double eta2 = eta * eta;
  const double beta = (113.0 / 12.0 * m1 * m1 + 6.25 * eta) * chi1 + (113.0 / 12.0 * m2 * m2 + 6.25 * eta) * chi2;
  const double phi2 = 3715.0 / 756.0 + 55.0 / 9.0 * eta;
  const double phi3 = -16.0 * kPi + 4.0 * beta;
  const double phi4 = 15293365.0 / 508032.0 + 27145.0 / 504.0 * eta + 3085.0 / 72.0 * eta2;
  const double P5 = kPi * (38645.0 / 756.0 - 65.0 / 9.0 * eta);
  const double Q6 = 11583231236531.0 / 4694215680.0 - 640.0 / 3.0 * kPi * kPi - 6848.0 / 21.0 * kEuler
                  + eta * (-15737765635.0 / 3048192.0 + 2255.0 / 12.0 * kPi * kPi)
                  + 76055.0 / 1728.0 * eta2 - 127825.0 / 1296.0 * eta2 * eta;
  const double phi7 = kPi * (77096675.0 / 254016.0 + 378515.0 / 1512.0 * eta - 74045.0 / 756.0 * eta2);
  const double iu2 = iu * iu;
  const double ln_vlso = -0.89587973461402748;                  // -ln(6)/2
  const double ln4 = 1.3862943611198906188;
  I.c[0] = K * iu2 * iu2 * iu;                                  // f^-5/3
  I.c[1] = K * phi2 * iu2 * iu;                                 // f^-1
  I.c[2] = K * phi3 * iu2;                                      // f^-2/3
  I.c[3] = K * phi4 * iu;                                       // f^-1/3
  I.c[4] = K * P5;                                              // ln f      (3 ln v = 3 ln u + ln f)
  I.c[5] = K * u * (Q6 - 6848.0 / 21.0 * (ln4 + lnu));          // f^1/3
  I.c[6] = -K * u * (6848.0 / 63.0);                            // f^1/3 ln f
  I.c[7] = K * phi7 * u * u;                                    // f^2/3
  I.c_const = (-th[6] - 0.25 * kPi) / (2.0 * kPi) + K * P5 * (1.0 + 3.0 * (lnu - ln_vlso));
  I.tc = th[5];
  I.amp = 0.45643546458763842789 /* sqrt(5/24) */ * 0.46619407703541166 /* pi^(-2/3) */ * mc56 * kC / (dL * kMpc);
  I.cos_iota = ci;
}

// everything in one thread (host setup, one-thread-per-point kernel)
NSS_HD void intrinsic(const double *th, Intrinsic &I)
{
  const double Mc = th[0], q = th[1];
  const double m1 = 1.0 / (1.0 + q), m2 = q * m1;
  const double eta = q * m1 * m1;
  const double M = Mc * pow(eta, -0.6) * kGMsun;
  const double u = cbrt(kPi * M);
  intrinsic_from(th, eta, m1, m2, u, 1.0 / u, log(u), pow(Mc * kGMsun, 5.0 / 6.0), cos(th[7]), I);
}

// polarisation basis of O4 (independent of the detector)
struct Sky {
  double X[3], Y[3], n[3];
};

NSS_HD void sky_from_sincos(double sg, double cg, double sd, double cd, double sp, double cp, Sky &S)
{
  S.X[0] = -cp * sg - sp * cg * sd;
  S.X[1] = -cp * cg + sp * sg * sd;
  S.X[2] = sp * cd;
  S.Y[0] = sp * sg - cp * cg * sd;
  S.Y[1] = sp * cg + cp * sg * sd;
  S.Y[2] = cp * cd;
  S.n[0] = cd * cg;          // cos(ra - gmst) = cos g
  S.n[1] = -cd * sg;         // sin(ra - gmst) = -sin g
  S.n[2] = sd;
}

NSS_HD void sky_frame(double gmst, double ra, double dec, double psi, Sky &S)
{
  double sg, cg, sd, cd, sp, cp;
  sincos(gmst - ra, &sg, &cg);
  sincos(dec, &sd, &cd);
  sincos(psi, &sp, &cp);
  sky_from_sincos(sg, cg, sd, cd, sp, cp, S);
}

// D6 = symmetric detector tensor (xx, xy, xz, yy, yz, zz) of D = (x x^T - y y^T)/2; rc = vertex / c
NSS_HD void antenna(const Sky &S, const double *D6, const double *rc, double &fp, double &fc, double &tau)
{
  const double DX0 = D6[0] * S.X[0] + D6[1] * S.X[1] + D6[2] * S.X[2];
  const double DX1 = D6[1] * S.X[0] + D6[3] * S.X[1] + D6[4] * S.X[2];
  const double DX2 = D6[2] * S.X[0] + D6[4] * S.X[1] + D6[5] * S.X[2];
  const double DY0 = D6[0] * S.Y[0] + D6[1] * S.Y[1] + D6[2] * S.Y[2];
  const double DY1 = D6[1] * S.Y[0] + D6[3] * S.Y[1] + D6[4] * S.Y[2];
  const double DY2 = D6[2] * S.Y[0] + D6[4] * S.Y[1] + D6[5] * S.Y[2];
  fp = (S.X[0] * DX0 + S.X[1] * DX1 + S.X[2] * DX2) - (S.Y[0] * DY0 + S.Y[1] * DY1 + S.Y[2] * DY2);
  fc = 2.0 * (S.X[0] * DY0 + S.X[1] * DY1 + S.X[2] * DY2);
  tau = -(rc[0] * S.n[0] + rc[1] * S.n[1] + rc[2] * S.n[2]);
}

// basis values at one frequency
NSS_HD void basis(double f, double *g)
{
  const double x = cbrt(f), lf = log(f);
  const double ix = 1.0 / x, ix2 = ix * ix;
  g[0] = ix2 * ix2 * ix;
  g[1] = 1.0 / f;
  g[2] = ix2;
  g[3] = ix;
  g[4] = lf;
  g[5] = x;
  g[6] = x * lf;
  g[7] = x * x;
}

// sin / cos of an angle given in turns.
// Device: t = q/4 + r with q = rint(4t) taken from the low word of 4t + 1.5*2^52 (exact for |t| < 2^29)
// and r = t - q/4 exact, |r| <= 1/8; sin(2 pi r)/r and cos(2 pi r) are degree-6 polynomials in r^2
// (Chebyshev-node fits on [0, 1/64]: relative error 4e-17 / absolute error 1e-16 before rounding); the
// quadrant swaps and negates through the sign bit.  17 fp64-pipe instructions and ~10 integer ones, no
// conversion (XU) instructions; a non-finite t gives NaNs.
#if defined(__CUDACC__)
// coefficients in the constant bank: an fp64 instruction takes them as c[bank][offset] operands, whereas
// immediates are re-materialised into uniform registers (two UMOV each) inside every loop body
static __constant__ double kSinT[7] = {0x1.921fb54442d18p+2, -0x1.4abbce625be41p+5, 0x1.466bc677587f8p+6, -0x1.32d2cce2e5b19p+6,
                                       0x1.50782fda12d96p+5, -0x1.e30071afc3e59p+3, 0x1.e3f38399551bfp+1};
static __constant__ double kCosT[7] = {1.0, -0x1.3bd3cc9be458bp+4, 0x1.03c1f081b0780p+6, -0x1.55d3c7dbfd139p+6,
                                       0x1.e1f4fb60281f6p+5, -0x1.a6c9c1be9eb49p+4, 0x1.f3dbcea61b1a4p+2};

__device__ __forceinline__ void sincos_turns_dev(double t, double *s, double *c)
{
  const double kMagic = 6755399441055744.0;            // 1.5 * 2^52
  const double tq = fma(t, 4.0, kMagic);
  const int q = __double2loint(tq);
  const double r = fma(tq - kMagic, -0.25, t);
  const double y = r * r;
  double ps = kSinT[6], pc = kCosT[6];
#pragma unroll
  for (int k = 5; k >= 0; --k) {
    ps = fma(ps, y, kSinT[k]);
    pc = fma(pc, y, kCosT[k]);
  }
  ps *= r;
  const bool sw = q & 1;
  const double a = sw ? pc : ps, b = sw ? ps : pc;     // quadrant 1, 3: sin <- cos, cos <- sin
  const int ah = __double2hiint(a) ^ ((q << 30) & 0x80000000);          // sin < 0 in quadrants 2, 3
  const int bh = __double2hiint(b) ^ (((q + 1) << 30) & 0x80000000);    // cos < 0 in quadrants 1, 2
  *s = __hiloint2double(ah, __double2loint(a));
  *c = __hiloint2double(bh, __double2loint(b));
}
#endif

NSS_HD void sincos_turns(double t, double *s, double *c)
{
#if defined(__CUDA_ARCH__)
  sincos_turns_dev(t, s, c);
#else
  const double fr = t - rint(t);
  sincos(2.0 * kPi * fr, s, c);
#endif
}

}  // namespace nssp
