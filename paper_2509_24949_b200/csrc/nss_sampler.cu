// nss_sampler.cu — K3 slice-sampling chains (slice directions included), K4 on-device NS bookkeeping, and the host
// driver behind nss_replace_step / nss_run (O11-O15).
#include <math.h>
#include <string.h>

#include <algorithm>
#include <mutex>
#include <vector>

#include "nss_loglike_dev.cuh"

namespace {

constexpr double kSliceW = 2.0;       // A14
constexpr int kMaxExpand = 32;        // A15
constexpr int kMaxShrink = 64;        // A15
constexpr uint32_t kIterInit = 0xFFFFFFFFu, kIterErr = 0xFFFFFFFEu, kStepStart = 0xFFFFFFFFu;
constexpr double kTwoM53 = 1.0 / 9007199254740992.0;

// ---- O11: Philox4x32-10, counter = (block, step, chain, iteration), key = seed ------------------------
__host__ __device__ __forceinline__ void philox_round(uint32_t &c0, uint32_t &c1, uint32_t &c2, uint32_t &c3, uint32_t k0,
                                                      uint32_t k1)
{
#if defined(__CUDA_ARCH__)
  const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
  const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
#else
  const uint64_t p0 = (uint64_t)0xD2511F53u * c0, p1 = (uint64_t)0xCD9E8D57u * c2;
  const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0, hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
#endif
  const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
  c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
}

__host__ __device__ __forceinline__ void philox4x32_10(uint64_t seed, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                       uint32_t *w)
{
  uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    philox_round(c0, c1, c2, c3, k0, k1);
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  w[0] = c0; w[1] = c1; w[2] = c2; w[3] = c3;
}

__host__ __device__ __forceinline__ void draw53(uint64_t seed, uint32_t block, uint32_t step, uint32_t chain, uint32_t it,
                                                uint64_t &ka, uint64_t &kb)
{
  uint32_t w[4];
  philox4x32_10(seed, block, step, chain, it, w);
  ka = ((uint64_t)(w[0] >> 5) << 26) + (uint64_t)(w[1] >> 6);
  kb = ((uint64_t)(w[2] >> 5) << 26) + (uint64_t)(w[3] >> 6);
}

__device__ __forceinline__ double uniform_a(uint64_t seed, uint32_t block, uint32_t step, uint32_t chain, uint32_t it)
{
  uint64_t ka, kb;
  draw53(seed, block, step, chain, it, ka, kb);
  return (double)ka * kTwoM53;
}

__global__ void k_philox(uint64_t seed, const uint32_t *__restrict__ ctr, int64_t n, uint32_t *__restrict__ out)
{
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint32_t w[4];
  philox4x32_10(seed, ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], w);
  out[4 * i] = w[0]; out[4 * i + 1] = w[1]; out[4 * i + 2] = w[2]; out[4 * i + 3] = w[3];
}

// ---- O13: initial live points ---------------------------------------------------------------------------
__global__ void k_init_live(const __grid_constant__ NssDev P, int n, uint64_t seed, double *__restrict__ live)
{
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int d = P.d;
  if (idx >= n * d) return;
  const int i = idx / d, j = idx - i * d;
  uint64_t ka, kb;
  draw53(seed, (uint32_t)(j >> 1), 0u, (uint32_t)i, kIterInit, ka, kb);
  const double u = (double)((j & 1) ? kb : ka) * kTwoM53;
  live[idx] = __dadd_rn(P.lo[j], __dmul_rn(P.hi[j] - P.lo[j], u));   // unfused: same bits as the oracle
}

// ---- K4 bookkeeping (O12.1 - O12.3, O14) as block-level device functions ------------------------------------------
// They run either as kernels of their own (the test hooks nss_select_lowest / nss_tune / nss_evidence_update, the
// initial stop test of nss_run) or inside the two fused kernels of an iteration: k4_front (rank + tune in parallel
// blocks, then selection tail + evidence in whichever block finishes last) and the epilogue of K3 (live evidence).
constexpr int kOneCta = 1024;
constexpr int kMaxDevices = 64;          // device ordinals the per-device tables below cover
constexpr int kRankElems = 256;          // live points ranked per block: 4 threads per point, each scanning a quarter of every tile

struct __align__(16) K4Smem {         // rank_block reads rank.tile two doubles per load
  union {
    struct { double tile[1024]; int cnt4[4 * kRankElems]; } rank;
    struct { double part[kOneCta]; double mean[NSS_NSLOT]; double cov[NSS_NSLOT * NSS_NSLOT]; double Lc[NSS_NSLOT * NSS_NSLOT]; double muc[NSS_NSLOT]; } tune;
    struct { double red[32]; double warp_tot[32]; int iwarp_tot[32]; } red;
  };
  unsigned ticket;
};

// K4.1 (O12.1): rank_i = #{ j : logL_j < logL_i  or (logL_j == logL_i and j < i) }, by counting: exact and stable (ties by
// slot).  The n x n comparisons are cut into blocks of kRankElems live points x one segment of J slots (4 threads per
// point, a quarter of the segment each; the segment is staged in shared memory and read two values per load by
// broadcast); a block writes the partial counts part[segment][i] and rank_finish adds them.  The kernel is bound by
// instruction issue (~2.5 instructions per comparison), so the segments are short (J ~ 256, at most kRankMaxSeg of
// them) to spread the work over every SM: ~3 us at n_live = 1000 .. 5000, ~0.5 ms at 65536 (where one
// iteration of chains takes > 10 ms).
constexpr int kRankMaxSeg = 32;
__host__ __device__ inline int rank_segments(int n) { const int s = (n + 255) / 256; return s < 1 ? 1 : s < kRankMaxSeg ? s : kRankMaxSeg; }
__host__ __device__ inline int rank_seg_len(int n) { const int nseg = rank_segments(n); return (((n + nseg - 1) / nseg) + 7) & ~7; }

__device__ __forceinline__ void rank_block(const double *__restrict__ logL, int n, int be, int sg, int nseg, int32_t *__restrict__ part,
                                           K4Smem &sm)
{
  const int e = threadIdx.x & (kRankElems - 1), seg4 = threadIdx.x >> 8;
  const int i = be * kRankElems + e;
  const double Li = i < n ? logL[i] : INFINITY;
  const double *tile = sm.rank.tile;
  const int J = rank_seg_len(n), j0 = sg * J, j1 = min(n, j0 + J);
  int cnt = 0;
  for (int base = j0; base < j1; base += 1024) {
    const int len = min(1024, j1 - base);
    __syncthreads();
    if ((int)threadIdx.x < len) sm.rank.tile[threadIdx.x] = logL[base + threadIdx.x];
    __syncthreads();
    const int q = ((len + 3) / 4 + 1) & ~1;                // quarter of the tile per thread, even so that pairs stay aligned
    const int t0 = min(len, seg4 * q), t1 = min(len, t0 + q);
    const int split = max(t0, min(t1, i - base));          // tile positions before slot i count on <=, the rest on <
    int t = t0;
    for (; t < split && (t & 1); ++t) cnt += tile[t] <= Li;
    for (; t + 1 < split; t += 2) { const double2 v = *reinterpret_cast<const double2 *>(tile + t); cnt += (int)(v.x <= Li) + (int)(v.y <= Li); }
    for (; t < split; ++t) cnt += tile[t] <= Li;
    for (; t < t1 && (t & 1); ++t) cnt += tile[t] < Li;
    for (; t + 1 < t1; t += 2) { const double2 v = *reinterpret_cast<const double2 *>(tile + t); cnt += (int)(v.x < Li) + (int)(v.y < Li); }
    for (; t < t1; ++t) cnt += tile[t] < Li;
  }
  __syncthreads();
  sm.rank.cnt4[seg4 * kRankElems + e] = cnt;
  __syncthreads();
  if (seg4 == 0 && i < n)
    part[(size_t)sg * n + i] = sm.rank.cnt4[e] + sm.rank.cnt4[kRankElems + e] + sm.rank.cnt4[2 * kRankElems + e] + sm.rank.cnt4[3 * kRankElems + e];
  __syncthreads();
}

// one block: rank_i = sum of the partial counts; dead_idx[rank] = i for rank < k
__device__ __forceinline__ void rank_finish(const int32_t *__restrict__ part, int n, int k, int nseg, int32_t *__restrict__ rank,
                                            int32_t *__restrict__ dead_idx)
{
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    int c = 0;
#pragma unroll 8                              // independent L2 loads: keep several in flight
    for (int sg = 0; sg < nseg; ++sg) c += __ldcg(part + (size_t)sg * n + i);
    rank[i] = c;
    if (c < k) dead_idx[c] = i;
  }
  __syncthreads();
}

// K4.2: survivor compaction (ascending slot), gather of the dead rows, threshold.  Returns (to every thread) whether a
// survivor lies below a supplied threshold.
__device__ __forceinline__ int finish_select_block(const double *__restrict__ live, const double *__restrict__ logL,
                                                   const double *__restrict__ birth, int n, int k, int d, double Lstar_in,
                                                   const int32_t *__restrict__ rank, const int32_t *__restrict__ dead_idx,
                                                   int32_t *__restrict__ surv_idx, double *__restrict__ dead_theta,
                                                   double *__restrict__ dead_logL, double *__restrict__ dead_birth,
                                                   double *__restrict__ state, K4Smem &sm)
{
  int *warp_tot = sm.red.iwarp_tot;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const double Lstar = isnan(Lstar_in) ? logL[dead_idx[k - 1]] : Lstar_in;
  const int chunk = (n + kOneCta - 1) / kOneCta;
  const int i0 = min(n, tid * chunk), i1 = min(n, i0 + chunk);
  int cnt = 0;
  bool bad = false;
  for (int i = i0; i < i1; ++i)
    if (rank[i] >= k) { ++cnt; bad = bad || (logL[i] < Lstar); }
  int incl = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  __syncthreads();
  if (lane == 31) warp_tot[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    int v = warp_tot[lane], s = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int u = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += u;
    }
    warp_tot[lane] = s - v;
  }
  __syncthreads();
  int pos = warp_tot[wid] + incl - cnt;
  if (surv_idx)
    for (int i = i0; i < i1; ++i)
      if (rank[i] >= k) surv_idx[pos++] = i;
  for (int j = tid; j < k; j += kOneCta) {
    const int slot = dead_idx[j];
    if (dead_logL) dead_logL[j] = logL[slot];
    if (dead_birth) dead_birth[j] = birth ? birth[slot] : -INFINITY;
    if (dead_theta) {
#pragma unroll 11                             // independent L2 loads of one row
      for (int a = 0; a < d; ++a) dead_theta[(size_t)j * d + a] = live[(size_t)slot * d + a];
    }
  }
  if (tid == 0 && state) state[3] = Lstar;
  return __syncthreads_or(bad ? 1 : 0);
}

__device__ __forceinline__ double block_sum(double v, double *red)
{
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  v = nssk::warp_sum(v);
  __syncthreads();
  if (lane == 0) red[wid] = v;
  __syncthreads();
  double s = 0.0;
  const int nw = blockDim.x >> 5;
  for (int w = 0; w < nw; ++w) s += red[w];     // fixed order: deterministic
  return s;
}

// K4.3 (O12.3): mean, covariance (two-pass, 1/(n-1)), lower Cholesky, by T co-resident blocks (T <= kTuneMaxBlocks; they
// are the first blocks of their grid, so they are scheduled together).  Block b owns the rows [b n/T, (b+1) n/T): column
// sums, then — after a counter barrier among the T blocks — the d(d+1)/2 centred products of its rows; inside a block
// the rows are split over thread groups (thread = (row group, column) or (row group, pair)) and added in a fixed order,
// and the blocks' partial sums are added in block order, so the result is deterministic.  The block that finishes last
// factors the matrix: *chol_fail = 1 if a pivot is <= 0 (reading R5: no relative epsilon), else 0.
constexpr int kTuneMaxBlocks = 32;
constexpr int kTuneProdOff = NSS_NSLOT, kTuneCircOff = NSS_NSLOT + NSS_NSLOT * (NSS_NSLOT + 1) / 2;
constexpr int kTunePartDoubles = kTuneCircOff + 2 * NSS_NSLOT;     // per block: column sums, products, circular sums (S, C)
// NEXT-2, second half (reading R7): sampled dimensions whose bit is set in `mask` are periodic with
// period W over [lo, lo + W): before the moments they are unwrapped around their circular mean,
//   mu_c = lo + W atan2(sum sin phi, sum cos phi)/(2 pi) (mod W),  phi = 2 pi (x - lo)/W,   x' = x - W rint((x - mu_c)/W).
// mask == 0: nothing changes (no extra pass, no extra barrier, the same bits as before).
struct TunePer {
  int32_t mask, pad_;
  double lo[NSS_NSLOT], W[NSS_NSLOT];
};
// One block per 1024 live points (about one row per thread in the column sums, ~70 in the products): a single block, with
// no barrier between blocks, up to 2047 rows.
__host__ __device__ inline int tune_blocks_for(int n) { const int t = n / 1024; return t < 2 ? 1 : t > kTuneMaxBlocks ? kTuneMaxBlocks : t; }
// The barrier among the tuning blocks is a spin on a counter, so all T of them must get an SM while the others wait.  A
// 1024-thread CTA of these kernels always fits an empty SM (__launch_bounds__), the rank blocks beside them and any other
// stream's CTAs finish without waiting for anybody here, so T <= number of SMs is enough for the last tuning block to be
// scheduled eventually.  On a B200 (148 SMs) the cap never binds; on a small MIG slice it does (and T, hence the order
// of the partial sums, then differs from a full device's in the last bits).
inline int tune_blocks_on(const nss_handle *h, int n) { const int t = tune_blocks_for(n); return t > h->n_sm ? (h->n_sm < 1 ? 1 : h->n_sm) : t; }

__device__ __forceinline__ void tune_block(const double *__restrict__ live, int n, int d, int b, int T, double *__restrict__ scratch,
                                           uint32_t *__restrict__ counters /*[3]*/, double *__restrict__ mean_out,
                                           double *__restrict__ chol_out, int32_t *__restrict__ chol_fail, const TunePer &tp,
                                           K4Smem &sm)
{
  double *part = sm.tune.part, *mean = sm.tune.mean, *cov = sm.tune.cov, *sLc = sm.tune.Lc, *muc = sm.tune.muc;
  const int tid = threadIdx.x;
  const int r0 = (int)((long long)n * b / T), r1 = (int)((long long)n * (b + 1) / T);
  const int np = d * (d + 1) / 2;
  const bool any_per = tp.mask != 0;
  if (any_per) {
    // R7, pass 0: circular sums of the periodic coordinates (thread = (row group, column), fixed-order tree as below),
    // a barrier among the blocks, then every block forms the same circular means from the same partial sums
    const int ng = kOneCta / d, j = tid % d, g = tid / d;
    const bool pj = g < ng && ((tp.mask >> j) & 1);
    double S = 0.0, C = 0.0;
    if (pj) {
      const double lo = tp.lo[j], W = tp.W[j];
      for (int i = r0 + g; i < r1; i += ng) {
        double sn, cs;
        sincos(2.0 * nssp::kPi * ((live[(size_t)i * d + j] - lo) / W), &sn, &cs);
        S += sn; C += cs;
      }
    }
    int top = 1;
    while (2 * top < ng) top *= 2;
    for (int pass = 0; pass < 2; ++pass) {
      __syncthreads();
      part[tid] = pass ? C : S;
      __syncthreads();
      for (int step = top; step >= 1; step >>= 1) {
        if (g < step && g + step < ng) part[tid] += part[tid + step * d];
        __syncthreads();
      }
      if (tid < d) scratch[b * kTunePartDoubles + kTuneCircOff + pass * NSS_NSLOT + tid] = part[tid];
    }
    if (T > 1) {
      __threadfence();
      __syncthreads();
      if (tid == 0) {
        atomicAdd(&counters[2], 1u);
        while (*(volatile uint32_t *)&counters[2] < (uint32_t)T) {}
      }
      __syncthreads();
      __threadfence();
    } else __syncthreads();
    if (tid < d) {
      double m = 0.0;
      if ((tp.mask >> tid) & 1) {
        double St = 0.0, Ct = 0.0;
        for (int q = 0; q < T; ++q) {
          St += __ldcg(scratch + q * kTunePartDoubles + kTuneCircOff + tid);
          Ct += __ldcg(scratch + q * kTunePartDoubles + kTuneCircOff + NSS_NSLOT + tid);
        }
        double a = atan2(St, Ct);
        if (a < 0.0) a += 2.0 * nssp::kPi;
        m = tp.lo[tid] + tp.W[tid] * (a / (2.0 * nssp::kPi));
      }
      muc[tid] = m;
    }
    __syncthreads();
  }
  // the value the moments see: the nearest image of a periodic coordinate to its circular mean (itself, bit for bit, when that is 0 periods away)
  auto val = [&](int i, int j) -> double {
    const double v = live[(size_t)i * d + j];
    if (!any_per || !((tp.mask >> j) & 1)) return v;
    const double W = tp.W[j];
    return __dsub_rn(v, __dmul_rn(W, rint((v - muc[j]) / W)));
  };
  {
    const int ng = kOneCta / d, j = tid % d, g = tid / d;
    double s = 0.0;
    if (g < ng) {
#pragma unroll 8                              // the rows come from L2: keep several loads in flight (same order of additions)
      for (int i = r0 + g; i < r1; i += ng) s += val(i, j);
    }
    part[tid] = s;
    __syncthreads();
    int top = 1;
    while (2 * top < ng) top *= 2;
    for (int step = top; step >= 1; step >>= 1) {           // pairwise tree over the row groups: fixed order, deterministic
      if (g < step && g + step < ng) part[tid] += part[tid + step * d];
      __syncthreads();
    }
    if (tid < d) scratch[b * kTunePartDoubles + tid] = part[tid];
    if (T > 1) {                                // every block needs every block's column sums
      __threadfence();
      __syncthreads();
      if (tid == 0) {
        atomicAdd(&counters[0], 1u);
        while (*(volatile uint32_t *)&counters[0] < (uint32_t)T) {}
      }
      __syncthreads();
      __threadfence();
    } else __syncthreads();
    if (tid < d) {
      double t = 0.0;
      for (int q = 0; q < T; ++q) t += __ldcg(scratch + q * kTunePartDoubles + tid);
      mean[tid] = t / n;
    }
    __syncthreads();
  }
  int a = 0, bb = 0;
  {
    const int ng = kOneCta / np, p = tid % np, g = tid / np;
    int rem = p;                              // pair index p -> (a, bb), bb <= a, row-major lower triangle
    while (rem > a) { rem -= a + 1; ++a; }
    bb = rem;
    double s = 0.0;
    if (g < ng) {
      const double ma = mean[a], mb = mean[bb];
#pragma unroll 8
      for (int i = r0 + g; i < r1; i += ng) s = fma(val(i, a) - ma, val(i, bb) - mb, s);
    }
    __syncthreads();
    part[tid] = s;
    __syncthreads();
    int top = 1;
    while (2 * top < ng) top *= 2;
    for (int step = top; step >= 1; step >>= 1) {
      if (g < step && g + step < ng) part[tid] += part[tid + step * np];
      __syncthreads();
    }
    if (tid < np) scratch[b * kTunePartDoubles + kTuneProdOff + tid] = part[tid];
  }
  if (T > 1) {                                  // the block that finishes last adds the partial products and factors
    __threadfence();
    __syncthreads();
    if (tid == 0) sm.ticket = atomicAdd(&counters[1], 1u);
    __syncthreads();
    if (sm.ticket != (unsigned)T - 1u) return;
    __threadfence();
  } else __syncthreads();
  if (tid < np) {
    double t = 0.0;
    for (int q = 0; q < T; ++q) t += __ldcg(scratch + q * kTunePartDoubles + kTuneProdOff + tid);
    cov[a * d + bb] = t / (n - 1);
    cov[bb * d + a] = t / (n - 1);
  }
  __syncthreads();
  // Cholesky by the first warp, column by column: lane i owns row i.  Every element is the same sum in the same
  // order as the row-by-row definition (s = cov_ij - sum_{m<j} L_im L_jm), only the rows of a column run side by side.
  if (tid < 32) {
    const int i = tid;
    for (int q = tid; q < d * d; q += 32) sLc[q] = 0.0;
    __syncwarp();
    bool ok = true;
    for (int j = 0; j < d; ++j) {
      double sacc = 0.0;
      if (i >= j && i < d) {
        sacc = cov[i * d + j];
        for (int m = 0; m < j; ++m) sacc -= sLc[i * d + m] * sLc[j * d + m];
      }
      const double piv = __shfl_sync(0xffffffffu, sacc, j);
      if (!(piv > 0.0)) { ok = false; break; }              // uniform: every lane sees the same pivot
      const double ljj = sqrt(piv);
      if (i == j) sLc[j * d + j] = ljj;
      else if (i > j && i < d) sLc[i * d + j] = sacc / ljj;
      __syncwarp();
    }
    if (tid == 0) *chol_fail = ok ? 0 : 1;
    __syncwarp();
    for (int q = tid; q < d * d; q += 32) chol_out[q] = sLc[q];
    if (mean_out)
      for (int q = tid; q < d; q += 32) mean_out[q] = mean[q];
  }
  __syncthreads();
}

__device__ __forceinline__ double block_max(double v, double *red)
{
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
  __syncthreads();
  if (lane == 0) red[wid] = v;
  __syncthreads();
  double m = -INFINITY;
  const int nw = blockDim.x >> 5;
  for (int w = 0; w < nw; ++w) m = fmax(m, red[w]);
  return m;
}

__device__ __forceinline__ double logaddexp_d(double a, double b)
{
  if (a == -INFINITY) return b;
  if (b == -INFINITY) return a;
  const double m = fmax(a, b);
  return m + log(exp(a - m) + exp(b - m));
}

// K4.4 (O12.2): log-weights of the dead points, logX shrinkage, logZ accumulation; one block of any size (multiple of 32)
__device__ __forceinline__ void evidence_block(const double *__restrict__ dead_logL, int n, int k, double *__restrict__ logw,
                                               double logX0, double logZ0, double *__restrict__ state, K4Smem &sm)
{
  double *red = sm.red.red, *warp_tot = sm.red.warp_tot;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const int nt = blockDim.x, chunk = (k + nt - 1) / nt;
  const int j0 = min(k, tid * chunk), j1 = min(k, j0 + chunk);
  double part = 0.0;
  for (int j = j0; j < j1; ++j) part += 1.0 / (double)(n - j);
  double incl = part;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const double v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  __syncthreads();
  if (tid < 32) warp_tot[tid] = 0.0;
  __syncthreads();
  if (lane == 31) warp_tot[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    double v = warp_tot[lane], s = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const double u = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += u;
    }
    warp_tot[lane] = s - v;
  }
  __syncthreads();
  double S = warp_tot[wid] + incl - part;       // sum_{i<j0} 1/m_i
  double mx = -INFINITY;
  for (int j = j0; j < j1; ++j) {
    const double im = 1.0 / (double)(n - j);
    const double lw = (logX0 - S) + log(-expm1(-im));
    logw[j] = lw;
    mx = fmax(mx, dead_logL[j] + lw);
    S += im;
  }
  const double total = block_sum(part, red);
  mx = block_max(mx, red);
  double se = 0.0;
  if (mx > -INFINITY)
    for (int j = j0; j < j1; ++j) se += exp(dead_logL[j] + logw[j] - mx);
  se = block_sum(se, red);
  if (tid == 0) {
    state[0] = logX0 - total;
    state[1] = mx > -INFINITY ? logaddexp_d(logZ0, mx + log(se)) : logZ0;
  }
  __syncthreads();
}

// ---- K4.1 for many live points: ranks by a sample sort ---------------------------------------------------------------
// Counting ranks costs n^2 comparisons (0.5 ms at n = 65536).  Above kRankDirectMax live points the ranks come from a
// sample sort instead — the same total order (logL ascending, ties by slot), so the same bits:
//   k4s_splitters  one block: S = 4 NB strided samples ordered by counting; every 4th is a splitter (NB - 1 of them)
//   k4s_bucket     every key finds its bucket (binary search among the splitters) and takes a place in it
//   k4s_offsets    one block: exclusive prefix sum of the bucket sizes
//   k4s_scatter    keys grouped by bucket (order inside a bucket arbitrary)
//   k4s_rank       rank = bucket offset + number of smaller keys in the bucket (~n / NB comparisons per key); a thread takes
//                  one grouped key, so the lanes of a warp scan the same bucket and their loads coalesce
// Splitters are (logL, slot) pairs, so even a population of equal values splits evenly.
constexpr int kRankDirectMax = 8192;
constexpr int kSplitMaxBuckets = 512;
__host__ __device__ inline int split_buckets(int n) { return n <= 131072 ? 256 : kSplitMaxBuckets; }

struct SplitBufs {           // carved out of the handle's rank scratch (n x kRankMaxSeg int32)
  double *gv;                // [n] grouped keys: value
  int32_t *gi;               // [n] grouped keys: slot
  int32_t *gb;               // [n] bucket of the grouped key
  int32_t *eb, *epos;        // [n] bucket of slot i and its place in the bucket
  double *spv;               // [NB - 1] splitters: value
  int32_t *spi;              // [NB - 1] splitters: slot
  int32_t *cnt, *off;        // [NB] bucket sizes, [NB + 1] offsets
};

__device__ __forceinline__ bool key_less(double a, int ia, double b, int ib) { return a < b || (a == b && ia < ib); }

__global__ void __launch_bounds__(kOneCta) k4s_splitters(const double *__restrict__ logL, int n, int NB, SplitBufs B, const NssCtl *ctl, int reset)
{
  __shared__ double sv[4 * kSplitMaxBuckets];
  __shared__ int si[4 * kSplitMaxBuckets];
  if (!reset && (ctl->flags[2] | ctl->flags[0])) return;
  const int S = 4 * NB;
  for (int t = threadIdx.x; t < S; t += kOneCta) {
    const int i = (int)((long long)t * n / S);
    sv[t] = logL[i]; si[t] = i;
  }
  for (int t = threadIdx.x; t < NB; t += kOneCta) B.cnt[t] = 0;
  __syncthreads();
  for (int t = threadIdx.x; t < S; t += kOneCta) {
    const double v = sv[t];
    const int i = si[t];
    int r = 0;
    for (int u = 0; u < S; ++u) r += key_less(sv[u], si[u], v, i) ? 1 : 0;
    if ((r & 3) == 0 && r > 0) { B.spv[r / 4 - 1] = v; B.spi[r / 4 - 1] = i; }     // ranks 4, 8, ...: the NB - 1 splitters
  }
}

__global__ void __launch_bounds__(256) k4s_bucket(const double *__restrict__ logL, int n, int NB, SplitBufs B, const NssCtl *ctl, int reset)
{
  __shared__ double sv[kSplitMaxBuckets];
  __shared__ int si[kSplitMaxBuckets];
  if (!reset && (ctl->flags[2] | ctl->flags[0])) return;
  for (int t = threadIdx.x; t < NB - 1; t += blockDim.x) { sv[t] = B.spv[t]; si[t] = B.spi[t]; }
  __syncthreads();
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const double v = logL[i];
  int lo = 0, hi = NB - 1;                       // bucket = number of splitters <= key
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (key_less(v, i, sv[mid], si[mid])) hi = mid; else lo = mid + 1;
  }
  B.eb[i] = lo;
  B.epos[i] = atomicAdd(&B.cnt[lo], 1);
}

__global__ void __launch_bounds__(kOneCta) k4s_offsets(int NB, SplitBufs B, const NssCtl *ctl, int reset)
{
  __shared__ int s[kOneCta];
  if (!reset && (ctl->flags[2] | ctl->flags[0])) return;
  const int t = threadIdx.x;
  s[t] = t < NB ? B.cnt[t] : 0;
  __syncthreads();
  for (int o = 1; o < kOneCta; o <<= 1) {        // inclusive scan
    const int v = t >= o ? s[t - o] : 0;
    __syncthreads();
    s[t] += v;
    __syncthreads();
  }
  if (t < NB) B.off[t + 1] = s[t];
  if (t == 0) B.off[0] = 0;
}

__global__ void __launch_bounds__(256) k4s_scatter(const double *__restrict__ logL, int n, SplitBufs B, const NssCtl *ctl, int reset)
{
  if (!reset && (ctl->flags[2] | ctl->flags[0])) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int b = B.eb[i], j = B.off[b] + B.epos[i];
  B.gv[j] = logL[i]; B.gi[j] = i; B.gb[j] = b;
}

__global__ void __launch_bounds__(256) k4s_rank(int n, int k, SplitBufs B, int32_t *__restrict__ rank, int32_t *__restrict__ dead_idx,
                                                 const NssCtl *ctl, int reset)
{
  if (!reset && (ctl->flags[2] | ctl->flags[0])) return;
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  const double v = B.gv[j];
  const int i = B.gi[j], b = B.gb[j];
  const int t0 = B.off[b], t1 = B.off[b + 1];
  int c = t0;
  for (int t = t0; t < t1; ++t) c += key_less(B.gv[t], B.gi[t], v, i) ? 1 : 0;
  rank[i] = c;
  if (c < k) dead_idx[c] = i;
}

// ---- stand-alone kernels (test hooks; the final ordering of the live points in nss_run) -------------------------------
__global__ void __launch_bounds__(kOneCta) k4_rank(const double *__restrict__ logL, int n, int nseg, int32_t *__restrict__ part)
{
  __shared__ K4Smem sm;
  rank_block(logL, n, blockIdx.x / nseg, blockIdx.x % nseg, nseg, part, sm);
}

// surv_idx == NULL: only the ordering (rank, dead_idx) is wanted
__global__ void __launch_bounds__(kOneCta) k4_finish_select(const double *__restrict__ logL, int n, int k, int nseg,
                                                            const int32_t *__restrict__ part, int32_t *__restrict__ rank,
                                                            int32_t *__restrict__ dead_idx, int32_t *__restrict__ surv_idx,
                                                            double *__restrict__ state)
{
  __shared__ K4Smem sm;
  if (nseg > 0) rank_finish(part, n, k, nseg, rank, dead_idx);     // nseg == 0: ranks and dead list come from the sample sort
  if (surv_idx) finish_select_block(nullptr, logL, nullptr, n, k, 0, NAN, rank, dead_idx, surv_idx, nullptr, nullptr, nullptr, state, sm);
}

__global__ void __launch_bounds__(kOneCta) k4_tune(const double *__restrict__ live, int n, int d, int T, double *__restrict__ scratch,
                                                   NssCtl *ctl, double *__restrict__ mean_out, double *__restrict__ chol_out,
                                                   const TunePer tp)
{
  __shared__ K4Smem sm;
  tune_block(live, n, d, blockIdx.x, T, scratch, ctl->tune_cnt, mean_out, chol_out, &ctl->flags[0], tp, sm);
  // Leave the two counters at zero, as k4_front's last block does: an iteration queued next on this handle (nss_iterate,
  // nss_replace_step: no k_begin in front of them) starts its own tuning blocks from them.  The block holding the last
  // ticket is the only one still running tune_block's tail, and every other block has passed the barrier on counters[0]
  // before it took its ticket, so nobody reads them any more.
  if (T > 1 && threadIdx.x == 0 && sm.ticket == (unsigned)T - 1u) { ctl->tune_cnt[0] = 0; ctl->tune_cnt[1] = 0; ctl->tune_cnt[2] = 0; }
}

__global__ void __launch_bounds__(kOneCta) k4_evidence(const double *__restrict__ dead_logL, int n, int k, double *__restrict__ logw,
                                                       double *__restrict__ state)
{
  __shared__ K4Smem sm;
  const double logX0 = state[0], logZ0 = state[1];
  __syncthreads();
  evidence_block(dead_logL, n, k, logw, logX0, logZ0, state, sm);
}

// ---- K4.5 (O14): live evidence and stop test ------------------------------------------------------------------
__global__ void __launch_bounds__(kOneCta) k4_live_evidence(const double *__restrict__ logL, int n, double stop_dlogz, int check,
                                                            double *__restrict__ state, int32_t *__restrict__ flags)
{
  __shared__ double red[32];
  double mx = -INFINITY;
  for (int i = threadIdx.x; i < n; i += kOneCta) mx = fmax(mx, logL[i]);
  mx = block_max(mx, red);
  double se = 0.0;
  if (mx > -INFINITY)
    for (int i = threadIdx.x; i < n; i += kOneCta) se += exp(logL[i] - mx);
  se = block_sum(se, red);
  if (threadIdx.x == 0) {
    const double lzl = mx > -INFINITY ? state[0] + mx + log(se) - log((double)n) : -INFINITY;
    state[2] = lzl;
    if (check && (lzl - state[1] < stop_dlogz)) flags[2] = 1;
  }
}

// ---- the front of an NS iteration in ONE launch ---------------------------------------------------------------------
// blocks 0 .. T-1 tune (a3: mean, covariance, Cholesky), the others rank the live points (a1) beside them; the rank block
// that finishes last adds the partial ranks, compacts the survivors, gathers the dead rows, fixes the threshold (a1) and
// does the evidence bookkeeping of the deleted batch (a2: it needs only the dead logL it has just gathered); the block
// that finishes last of all publishes the flags and resets the counters.  `reset` = a stand-alone iteration (nss_iterate, nss_replace_step): flags and,
// on request, state and counters are re-initialised; otherwise (nss_run's loop, queued one iteration ahead of the host) an
// iteration queued after convergence or after a Cholesky failure does nothing.
struct FrontArgs {
  const double *live, *logL, *birth;
  int32_t n, k, d, T, nseg;
  double Lstar_in;
  int32_t *rank_part, *rank, *dead_idx, *surv_idx;
  double *dead_theta, *dead_logL, *dead_birth;
  double *dead_logw;            // not NULL: the evidence bookkeeping of the deleted batch (a2) follows the selection
  double *tune_scratch, *mean, *chol;
  TunePer per;                  // periodic coordinates are unwrapped around their circular mean before the moments (R7)
  NssCtl *ctl;
  int32_t reset, set_state, zero_evals;
  double logX, logZ;
};

__global__ void __launch_bounds__(kOneCta) k4_front(const FrontArgs A)
{
  __shared__ K4Smem sm;
  // K3 is launched with programmatic stream serialization: let its CTAs start their prologue (table staging, constants)
  // on the SMs this small grid leaves free; they wait (griddepcontrol.wait) for this grid to finish before reading anything
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  NssCtl *ctl = A.ctl;
  if (!A.reset && (ctl->flags[2] | ctl->flags[0])) return;
  const int b = blockIdx.x;
  if (b < A.T) {
    tune_block(A.live, A.n, A.d, b, A.T, A.tune_scratch, ctl->tune_cnt, A.mean, A.chol, &ctl->chol_now, A.per, sm);
  } else {
    // nseg == 0: the ranks and the dead list are there already (sample sort, many live points) and this is the only block
    // behind the tuning blocks; else the rank block that finishes last runs the selection tail (it does not wait for the
    // tuning blocks)
    if (A.nseg > 0) {
      rank_block(A.logL, A.n, (b - A.T) / A.nseg, (b - A.T) % A.nseg, A.nseg, A.rank_part, sm);
      __threadfence();
      __syncthreads();
      if (threadIdx.x == 0) sm.ticket = atomicAdd(&ctl->rank_done, 1u);
      __syncthreads();
    }
    if (A.nseg == 0 || sm.ticket == gridDim.x - A.T - 1u) {
      __threadfence();
      if (A.nseg > 0) rank_finish(A.rank_part, A.n, A.k, A.nseg, A.rank, A.dead_idx);
      const int bad = finish_select_block(A.live, A.logL, A.birth, A.n, A.k, A.d, A.Lstar_in, A.rank, A.dead_idx, A.surv_idx, A.dead_theta,
                                          A.dead_logL, A.dead_birth, ctl->state, sm);
      if (threadIdx.x == 0) ctl->sel_bad = bad;
      // a2 (O12.2).  A stand-alone iteration takes logX, logZ from the arguments, nss_run's loop from the control block.
      const double logX0 = (A.reset && A.set_state) ? A.logX : ctl->state[0], logZ0 = (A.reset && A.set_state) ? A.logZ : ctl->state[1];
      __syncthreads();
      if (A.dead_logw) evidence_block(A.dead_logL, A.n, A.k, A.dead_logw, logX0, logZ0, ctl->state, sm);
      else if (threadIdx.x == 0 && A.reset && A.set_state) { ctl->state[0] = logX0; ctl->state[1] = logZ0; }
      if (threadIdx.x == 0 && A.reset && A.set_state) ctl->state[2] = 0.0;
    }
  }
  // the block that finishes last of all publishes the flags and resets the counters
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) sm.ticket = atomicAdd(&ctl->front_done, 1u);
  __syncthreads();
  if (sm.ticket != gridDim.x - 1 || threadIdx.x != 0) return;
  __threadfence();
  ctl->front_done = 0; ctl->rank_done = 0; ctl->chains_done = 0; ctl->chain_next = 0; ctl->tune_cnt[0] = 0; ctl->tune_cnt[1] = 0; ctl->tune_cnt[2] = 0;
  const int chol_fail = *(volatile int32_t *)&ctl->chol_now;
  ctl->flags[1] = *(volatile int32_t *)&ctl->sel_bad;
  if (A.reset) {
    ctl->flags[0] = chol_fail; ctl->flags[2] = 0; ctl->flags[3] = 0;
    if (A.zero_evals) { ctl->nevals = 0ull; ctl->nrounds = 0ull; ctl->nexec = 0ull; }
  } else if (chol_fail) ctl->flags[0] = 1;
}

// ---- O15: evidence-error replicas (stochastic compression), one CTA per replica -------------------------------
// ln t_j = ln(u+_j)/m_j with m_j = n - (j mod k); logX_j = sum_{i<j} ln t_i; w_j = X_j (1 - t_j);
// lZ = logsumexp_j(logL_j + ln w_j) (+) [logX_end + logsumexp(live logL) - ln n].  The prefix sum is split over
// the threads (chunk sums, one block scan, then each thread walks its chunk), the draws are regenerated in the
// second pass (Philox counter = (0, j, replica, 0xFFFFFFFE)).
constexpr int kErrReplicas = 200;
__global__ void __launch_bounds__(256) k_evidence_error(const double *__restrict__ dead_logL, long long n_dead, int n, int k,
                                                        uint64_t seed, const double *__restrict__ live_logL,
                                                        double *__restrict__ lZ_out)
{
  __shared__ double red[32];
  __shared__ double warp_tot[8];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const uint32_t rpl = blockIdx.x;
  const long long chunk = (n_dead + blockDim.x - 1) / blockDim.x;
  const long long j0 = min(n_dead, (long long)tid * chunk), j1 = min(n_dead, j0 + chunk);
  auto lnt = [&](long long j) {
    uint64_t ka, kb;
    draw53(seed, 0u, (uint32_t)j, rpl, kIterErr, ka, kb);
    return log((double)(ka + 1) * kTwoM53) / (double)(n - (int)(j % k));
  };
  double part = 0.0;
  for (long long j = j0; j < j1; ++j) part += lnt(j);
  double incl = part;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const double v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  if (lane == 31) warp_tot[wid] = incl;
  __syncthreads();
  double lX = incl - part;
  for (int q = 0; q < wid; ++q) lX += warp_tot[q];
  double mx = -INFINITY, se = 0.0;
  for (long long j = j0; j < j1; ++j) {
    const double lt = lnt(j);
    const double a = dead_logL[j] + lX + log1p(-exp(lt));
    if (a > mx) { se = se * exp(mx - a) + 1.0; mx = a; }
    else if (a > -INFINITY) se += exp(a - mx);
    lX += lt;
  }
  const double M = block_max(mx, red);
  const double tot = block_sum(M > -INFINITY && mx > -INFINITY ? se * exp(mx - M) : 0.0, red);
  const double lX_end = block_sum(part, red);
  // live term
  double lm = -INFINITY;
  for (int i = tid; i < n; i += blockDim.x) lm = fmax(lm, live_logL[i]);
  lm = block_max(lm, red);
  double ls = 0.0;
  if (lm > -INFINITY)
    for (int i = tid; i < n; i += blockDim.x) ls += exp(live_logL[i] - lm);
  ls = block_sum(ls, red);
  if (tid == 0) {
    const double lz_dead = M > -INFINITY ? M + log(tot) : -INFINITY;
    const double lz_live = lm > -INFINITY ? lX_end + lm + log(ls) - log((double)n) : -INFINITY;
    lZ_out[rpl] = logaddexp_d(lz_dead, lz_live);
  }
}

// ---- O15 / NEXT-4: Kish effective sample size of the posterior weights, one CTA -----------------------------------
// a_i = logL_i + logw_i over the dead rows, and logL_i + logX_end - ln n over the final live points;
// ESS = (sum e^(a_i - amax))^2 / sum e^(2 (a_i - amax)).  out[0] = ESS.
__global__ void __launch_bounds__(kOneCta) k_kish_ess(const double *__restrict__ dead_logL, const double *__restrict__ dead_logw,
                                                      long long n_dead, const double *__restrict__ live_logL, int n,
                                                      const double *__restrict__ state, double *__restrict__ out)
{
  __shared__ double red[32];
  const double lw_live = state[0] - log((double)n);
  double mx = -INFINITY;
  for (long long i = threadIdx.x; i < n_dead; i += kOneCta) mx = fmax(mx, dead_logL[i] + dead_logw[i]);
  for (int i = threadIdx.x; i < n; i += kOneCta) mx = fmax(mx, live_logL[i] + lw_live);
  mx = block_max(mx, red);
  double s1 = 0.0, s2 = 0.0;
  if (mx > -INFINITY) {
    for (long long i = threadIdx.x; i < n_dead; i += kOneCta) {
      const double a = dead_logL[i] + dead_logw[i];
      if (a > -INFINITY) { const double p = exp(a - mx); s1 += p; s2 = fma(p, p, s2); }
    }
    for (int i = threadIdx.x; i < n; i += kOneCta) {
      const double a = live_logL[i] + lw_live;
      if (a > -INFINITY) { const double p = exp(a - mx); s1 += p; s2 = fma(p, p, s2); }
    }
  }
  s1 = block_sum(s1, red);
  s2 = block_sum(s2, red);
  if (threadIdx.x == 0) out[0] = s2 > 0.0 ? s1 * s1 / s2 : 0.0;
}

// ---- NEXT-4 / reading R6: equal-weight posterior samples, one CTA --------------------------------------------------
// Row i (posterior weight p_i ~ exp(logL_i + logw_i)) is kept iff u_i < p_i / max_j p_j, with u_i the [0, 1) uniform of
// Philox counter (0, i mod 2^32, i div 2^32, 0xFFFFFFFD): an equally weighted sample of the posterior whose expected size
// is sum p / max p (PAPER.md:59-63 quotes such a count in brackets beside the Kish ESS and does not define it).
// out[0] = number kept (as a double: exact below 2^53); idx_out (optional) = the kept rows in ascending order.
constexpr uint32_t kIterEqual = 0xFFFFFFFDu;
__global__ void __launch_bounds__(kOneCta) k_resample_equal(const double *__restrict__ logL, const double *__restrict__ logw,
                                                            long long n, uint64_t seed, long long *__restrict__ idx_out,
                                                            double *__restrict__ out)
{
  __shared__ double red[32];
  __shared__ long long wtot[32];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  double mx = -INFINITY;
  for (long long i = tid; i < n; i += kOneCta) mx = fmax(mx, logL[i] + logw[i]);
  mx = block_max(mx, red);
  const long long chunk = (n + kOneCta - 1) / kOneCta;
  const long long i0 = min(n, (long long)tid * chunk), i1 = min(n, i0 + chunk);
  auto keep = [&](long long i) {
    const double a = logL[i] + logw[i];
    if (!(a > -INFINITY)) return false;
    return uniform_a(seed, 0u, (uint32_t)(i & 0xFFFFFFFFll), (uint32_t)(i >> 32), kIterEqual) < exp(a - mx);
  };
  long long cnt = 0;
  if (mx > -INFINITY)
    for (long long i = i0; i < i1; ++i) cnt += keep(i) ? 1 : 0;
  long long incl = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const long long v = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += v;
  }
  __syncthreads();
  if (lane == 31) wtot[wid] = incl;
  __syncthreads();
  long long pos = incl - cnt, total = 0;
  for (int q = 0; q < kOneCta / 32; ++q) {
    if (q < wid) pos += wtot[q];
    total += wtot[q];
  }
  if (idx_out && mx > -INFINITY)
    for (long long i = i0; i < i1; ++i)
      if (keep(i)) idx_out[pos++] = i;
  if (tid == 0) out[0] = (double)total;
}

// logw of the final live points, logX - ln n (O14), written on the device so that host and device rows are the same bits
__global__ void k_fill_live_logw(double *__restrict__ p, int n, const double *__restrict__ state)
{
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = state[0] - log((double)n);
}

__global__ void k_fill(double *__restrict__ p, int n, double v)
{
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = v;
}

__global__ void k_gather_rows(const double *__restrict__ live, const double *__restrict__ logL, const double *__restrict__ birth,
                              const int32_t *__restrict__ order, int n, int d, double *__restrict__ out_theta,
                              double *__restrict__ out_logL, double *__restrict__ out_birth)
{
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n) return;
  const int slot = order[j];
  out_logL[j] = logL[slot];
  out_birth[j] = birth[slot];
  for (int a = 0; a < d; ++a) out_theta[(size_t)j * d + a] = live[(size_t)slot * d + a];
}

// ---- a5: the slice direction of one (chain, step) by one thread ---------------------------------------------------
// z ~ N(0, I_d) by Box-Muller (one Philox block per pair: counter (1 + pair, step, chain, iteration)),
// n = z/|z|, v = w L n with L the Cholesky factor of the live-point covariance (O12.4a); sL and out in shared memory.
__device__ __forceinline__ void draw_direction(int d, const double *__restrict__ sL, uint64_t seed, uint32_t it, uint32_t ch, uint32_t s,
                                               double *__restrict__ out)
{
  double z[NSS_NSLOT + 1];
#pragma unroll
  for (int b = 0; b < (NSS_NSLOT + 1) / 2; ++b)
    if (2 * b < d) {
      uint64_t ka, kb;
      draw53(seed, (uint32_t)(1 + b), s, ch, it, ka, kb);
      const double r = sqrt(-2.0 * log((double)(ka + 1) * kTwoM53));
      double sn, cs;
      sincospi(2.0 * ((double)kb * kTwoM53), &sn, &cs);
      z[2 * b] = r * cs;
      z[2 * b + 1] = r * sn;
    }
  double nz = 0.0;
#pragma unroll
  for (int j = 0; j < NSS_NSLOT; ++j)
    if (j < d) nz += z[j] * z[j];
  nz = sqrt(nz);
#pragma unroll
  for (int j = 0; j < NSS_NSLOT; ++j)
    if (j < d) z[j] = z[j] / nz;
#pragma unroll
  for (int i = 0; i < NSS_NSLOT; ++i)
    if (i < d) {
      double a = 0.0;
#pragma unroll
      for (int j = 0; j < NSS_NSLOT; ++j)
        if (j <= i) a += sL[i * d + j] * z[j];
      out[i] = kSliceW * a;
    }
}

// ---- K3: slice-sampling chains (O12.4, O12.5) -------------------------------------------------------------------
// A chain is run by a GROUP of G warps (G = 1, 2, 4 or 8).  Every bracket test is one likelihood evaluation by
// ONE SUB-WARP of LANES lanes (8 for relative binning: four candidates per warp share every instruction of the
// per-point setup; 32 otherwise), so a group evaluates C = G * 32/LANES candidates per round: the next C tests of
// the sequential algorithm under the assumption that each of them fails — which is what they do most of the time:
//     [left end l, if the left side is still stepping out] [right end r, likewise]
//     [shrinkage proposals t_kk, t_kk+1, ... from the bracket those two tests would leave]
// The proposals that follow a rejection depend only on the rejected proposals (bracket <- t on the side of
// sign(t)) and on counter-based Philox draws, never on logL, so they are known in advance.  After the round
// every warp replays the sequential decisions on the shared results and discards whatever the sequential
// algorithm would not have evaluated (shrinkage proposals speculated across an expansion; proposals after
// the accepted one).  Decisions, positions and the evaluation count are those of the sequential oracle.
// The chain position x and direction v are spread over the lanes of every sub-warp (lane j holds x_j, v_j, and
// x_{j+LANES}, v_{j+LANES} when LANES < d).
// NEXT-2 (R4): a periodic coordinate is mapped back into its box, y - W floor((y - lo)/W), every
// operation rounded once (the oracle does the same with contraction off), and takes no part in the box test
__device__ __forceinline__ double wrap_periodic(double y, double lo, double hi)
{
  const double W = __dsub_rn(hi, lo);
  const double kf = floor(__ddiv_rn(__dsub_rn(y, lo), W));
  return __dsub_rn(y, __dmul_rn(W, kf));
}

struct ChainArgs {
  double *live;                 // [n][d] in/out
  double *logL;                 // [n]    in/out
  double *birth;                // [n]    in/out, may be NULL
  int32_t n, k, n_repeats;
  uint64_t seed;
  uint32_t iteration;
  const int32_t *surv_idx, *dead_idx;
  const double *chol;           // [d][d] lower Cholesky factor of the live-point covariance (k4_front)
  NssCtl *ctl;                  // state[3] = L*; flags (any set -> do nothing); evaluation counters; chains_done
  int32_t *trace;               // optional [k][n_repeats][3]
  double *margin;               // optional [k]
  int32_t G;                    // warps per chain
  int32_t live_evidence;        // the CTA that finishes the last chain computes logZ_live and the stop test (a11, O14)
  double stop_dlogz;
};

constexpr int kChainWarps = 8;          // largest group; a CTA is ONE group (G warps), one chain at a time
constexpr int kDirChunk = 32;           // slice directions drawn at a time by a group (one lane of its first warp each)
constexpr int kChainThreads = kChainWarps * 32;

__device__ __forceinline__ void group_sync(int G)
{
  if (G == 1) __syncwarp(); else __syncthreads();        // the CTA is the group
}

// Registers: a lone warp needs the instruction-level parallelism of two records x three detectors in flight, and the
// register file is per SM sub-partition (16384 registers: two warps above 170 registers per thread, three up to 168, four
// up to 128).  Capping the kernel at 168, 144 or 128 registers (no spills) costs 35 - 100 % per warp on B200 and loses
// more than the extra resident warps return, for 500 chains and for 2500 (profiles/r02_k3_experiments.md): it may use 255.
#define NSS_K3_BOUNDS __launch_bounds__(kChainThreads, 1)
template <int NDET, int KIND, int LANES, bool RESIDENT>
__global__ void NSS_K3_BOUNDS k3_slice(const __grid_constant__ NssDev P, const ChainArgs A)
{
  constexpr int NSUB = 32 / LANES;                              // candidates per warp
  constexpr int NC = (NSS_NSLOT + LANES - 1) / LANES;           // coordinates per lane
  constexpr int kSlots = kChainWarps * NSUB;                    // most candidates per round
  extern __shared__ __align__(128) unsigned char smem_raw[];    // [record table if RESIDENT][C sub-warp scratches]
  __shared__ __align__(8) uint64_t bar;
  __shared__ double sV[kChainWarps][NSS_NSLOT + 1];                // direction of the current step, one copy per warp
  __shared__ double sRes[2][kSlots];                               // double-buffered: logL of every candidate slot
  __shared__ double sX[kChainWarps][NSS_NSLOT + 1];                // chain position, one copy per warp (lane-level box tests)
  __shared__ double sLo[NSS_NSLOT + 1], sHi[NSS_NSLOT + 1];        // prior box, (-inf, +inf) for the unused coordinates
  __shared__ __align__(16) double sConst[nssk::kSubConstDoubles];
  __shared__ unsigned sLast;
  __shared__ double sChol[NSS_NSLOT * NSS_NSLOT];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int sl = lane & (LANES - 1), sub = lane / LANES;
  nssk::SubCtx X;
  constexpr int LI = nssk::lanes_index<LANES>();
  X.tab = P.soa[LI];
  X.consts = sConst;
  const size_t tab_bytes = RESIDENT ? nssk::sub_table_doubles<NDET, KIND == NSS_KIND_RB, LANES>(P.soa_m[LI]) * sizeof(double) : 0;
  X.scr = reinterpret_cast<double *>(smem_raw + tab_bytes) + (size_t)(warp * NSUB + sub) * nssk::kSubScratchDoubles;
  if (RESIDENT) {
    if (threadIdx.x == 0) {
      nssk::mbar_init(&bar, 1);
      nssk::stage_table(smem_raw, P.soa[LI], (uint32_t)tab_bytes, &bar);
    }
  }
  const int d = P.d;
  for (int t = threadIdx.x; t <= NSS_NSLOT; t += blockDim.x) {
    const bool wall = t < d && !P.periodic[t];
    sLo[t] = wall ? P.lo[t] : -INFINITY;
    sHi[t] = wall ? P.hi[t] : INFINITY;
  }
  if (lane <= NSS_NSLOT) { sX[warp][lane] = 0.0; sV[warp][lane] = 0.0; }
  if (KIND != NSS_KIND_GAUSS) {
    nssk::sub_consts_init(P, sConst);
    for (int t = sl; t < 12; t += LANES) X.scr[t] = t < NSS_NSLOT ? P.theta_fixed[t] : 0.0;   // unsampled slots never change
  }
  __syncthreads();
  if (RESIDENT) {
    nssk::mbar_wait(&bar, 0);
    X.tab = reinterpret_cast<const double *>(smem_raw);
  }
  // Everything above is independent of the kernels in front (programmatic dependent launch: it overlaps their tails);
  // everything below reads what k4_front wrote.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  NssCtl *ctl = A.ctl;
  if (ctl->flags[0] | ctl->flags[1] | ctl->flags[2]) return;      // Cholesky failure, threshold violation, or converged
  for (int t = threadIdx.x; t < d * d; t += blockDim.x) sChol[t] = A.chol[t];
  __syncthreads();
  // A CTA is one group of G warps (G > 1), or W = blockDim/32 single-warp groups that share the record table (G == 1);
  // single-warp groups take their chains from a device counter, so a warp that finishes early starts the next chain
  const int G = A.G, C = G * NSUB;
  const int w = warp & (G - 1);                          // warp in the group
  const int gbase = (warp - w) * NSUB;                   // first candidate slot of the group in sRes
  // a5: the group's slice directions, kDirChunk steps at a time: [kDirChunk][NSS_NSLOT] per group, behind the scratches
  double *sDir = reinterpret_cast<double *>(smem_raw + tab_bytes) + (size_t)(blockDim.x >> 5) * NSUB * nssk::kSubScratchDoubles
               + (size_t)((warp - w) / G) * kDirChunk * NSS_NSLOT;
  const int gl = w * 32 + lane;                          // lane in the group
  const int cs = w * NSUB + sub;                         // candidate slot of this sub-warp in the group
  const double Lstar = ctl->state[3];
  const uint32_t it = A.iteration;
  const int ns = A.n - A.k;
  bool own[NC];
  int dst_idx[NC];                                       // where coordinate j goes in the likelihood's input
  double lo_j[NC], hi_j[NC];
  bool per[NC];                                          // the coordinate wraps instead of hitting a wall
#pragma unroll
  for (int c = 0; c < NC; ++c) {
    const int j = sl + c * LANES;
    own[c] = j < d;
    lo_j[c] = own[c] ? P.lo[j] : 0.0;
    hi_j[c] = own[c] ? P.hi[j] : 0.0;
    dst_idx[c] = own[c] ? (KIND == NSS_KIND_GAUSS ? j : P.param_index[j]) : 0;
    per[c] = own[c] && P.periodic[j] != 0;
  }
  int par = 0;
  // lane j < d owns coordinate j of the per-warp position copy sX (walls and period of that coordinate in registers)
  const bool lper = lane < d && P.periodic[lane < NSS_NSLOT ? lane : 0] != 0;
  const double llo = lane < d ? P.lo[lane < NSS_NSLOT ? lane : 0] : 0.0, lhi = lane < d ? P.hi[lane < NSS_NSLOT ? lane : 0] : 0.0;

  for (int ch = blockIdx.x;; ch += gridDim.x) {
    if (G == 1) {
      if (lane == 0) ch = (int)atomicAdd(&ctl->chain_next, 1u);
      ch = __shfl_sync(0xffffffffu, ch, 0);
    }
    if (ch >= A.k) break;
    const uint32_t chain = (uint32_t)ch;
    // a4: start from a uniformly chosen survivor
    int si = (int)floor(uniform_a(A.seed, 0u, kStepStart, chain, it) * (double)ns);
    si = si > ns - 1 ? ns - 1 : si;
    const int slot = A.surv_idx[si];
    double xj[NC];
#pragma unroll
    for (int c = 0; c < NC; ++c) xj[c] = own[c] ? A.live[(size_t)slot * d + sl + c * LANES] : 0.0;
    __syncwarp();
    for (int j = lane; j < d; j += 32) sX[warp][j] = A.live[(size_t)slot * d + j];
    __syncwarp();
    double lx = A.logL[slot];
    long long evals = 0;
    int rounds = 0, nexec = 0;
    double margin = INFINITY, margin_l = INFINITY;        // bracket-end tests (uniform) / this lane's proposals

    // uniforms of a step: lane 0 -> bracket offset (block 0); lane 1+i -> shrinkage proposal ubase+i (block 64+ubase+i).
    // Drawn one step ahead, so that the Philox rounds are off the critical path of the step that uses them.
    double unext = uniform_a(A.seed, lane == 0 ? 0u : (uint32_t)(63 + lane), 0u, chain, it);
    {
      for (int s = 0; s < A.n_repeats; ++s) {
        // a5: the directions of the next kDirChunk steps, one lane of the group's first warp each (they depend on the
        // Cholesky factor and on counter-based draws only)
        if ((s & (kDirChunk - 1)) == 0) {
          group_sync(G);                                 // every warp of the group has taken the last direction of the chunk before
          if (gl < kDirChunk && s + gl < A.n_repeats) draw_direction(d, sChol, A.seed, it, chain, (uint32_t)(s + gl), sDir + gl * NSS_NSLOT);
          group_sync(G);
        }
        __syncwarp();
        if (lane < d) sV[warp][lane] = sDir[(s & (kDirChunk - 1)) * NSS_NSLOT + lane];
        __syncwarp();
        const double *vrow = sV[warp];
        double vj[NC];
#pragma unroll
        for (int c = 0; c < NC; ++c) vj[c] = own[c] ? vrow[sl + c * LANES] : 0.0;
        double ulane = unext;
        unext = uniform_a(A.seed, lane == 0 ? 0u : (uint32_t)(63 + lane), (uint32_t)(s + 1), chain, it);
        int ubase = 0;
        const double u0 = nssk::shfl_d(ulane, 0);
        double l = -u0, r = 1.0 - u0;
        int nl = 0, nr = 0, kk = 0, acc = -1;
        bool ldone = false, rdone = false, done = false;
        while (!done) {
          // ---- the next tests of the sequential algorithm, one per lane, assuming each of them fails ------------
          if (kk - ubase > 15) {                         // keep at least 16 proposals' uniforms in the lanes
            ubase = kk;
            ulane = uniform_a(A.seed, (uint32_t)(63 + ubase + lane), (uint32_t)s, chain, it);
          }
          int nside = (ldone ? 0 : 1) + (rdone ? 0 : 1);
          int nshr = 31 - (kk - ubase);                  // proposals whose uniforms are at hand
          nshr = nshr < kMaxShrink - kk ? nshr : kMaxShrink - kk;
          nshr = nshr < 32 - nside ? nshr : 32 - nside;
          nshr = nshr < 2 * C ? nshr : 2 * C;            // no point in listing far more tests than can be evaluated
          const int nt = nside + nshr;
          double my_t = (lane == 0 && !ldone) ? l : r;   // lanes < nside: the bracket ends
          double my_ls = l, my_rs = r;                   // the bracket after this lane's test has failed
          {
            // The proposals are a serial recurrence (each bracket follows from the rejection of the proposal before), so
            // the walk is on the critical path of the round: the first kWalk steps run with a fixed trip count (uniforms
            // fetched up front, no branches; steps past nshr compute values no lane keeps), the rest in a plain loop.
            constexpr int kWalk = 8;
            double ls = l, rs = r;
            double uk[kWalk];
#pragma unroll
            for (int j = 0; j < kWalk; ++j) uk[j] = nssk::shfl_d(ulane, (kk - ubase + j + 1) & 31);
            const int mine = lane - nside;                 // this lane's proposal in the list (if 0 <= mine < nshr)
#pragma unroll
            for (int j = 0; j < kWalk; ++j) {
              const double t = __dadd_rn(ls, __dmul_rn(rs - ls, uk[j]));
              const bool neg = t < 0.0;
              ls = neg ? t : ls;
              rs = neg ? rs : t;
              if (mine == j) { my_t = t; my_ls = ls; my_rs = rs; }
            }
            for (int j = kWalk; j < nshr; ++j) {
              const double u = nssk::shfl_d(ulane, kk - ubase + j + 1);
              const double t = __dadd_rn(ls, __dmul_rn(rs - ls, u));
              if (t < 0.0) ls = t; else rs = t;
              if (mine == j) { my_t = t; my_ls = ls; my_rs = rs; }
            }
          }
          // box test (inclusive) of the lane's own test: y = x + t v, every coordinate
          int inb_i = lane < nt;                         // branch-free: every coordinate, then one AND
#pragma unroll
          for (int j = 0; j < NSS_NSLOT; ++j) {
            const double y = __dadd_rn(sX[warp][j], __dmul_rn(my_t, vrow[j]));
            inb_i &= (int)(y >= sLo[j]) & (int)(y <= sHi[j]);
          }
          const bool inb = inb_i != 0;
          const unsigned M = __ballot_sync(0xffffffffu, inb);      // tests inside the box, in sequential order
          // ---- evaluate: the cs-th test inside the box goes to candidate slot cs -------------------------------
          const bool have = cs < __popc(M);
          ++rounds;
          nexec += min(C, __popc(M));
          int e = 0;                                     // lane holding the test of slot cs: the one with cs set bits of M below it
          const int below = __popc(M & ((1u << lane) - 1u));
          {
#pragma unroll
            for (int q = 0; q < NSUB; ++q) {
              const unsigned hit = __ballot_sync(0xffffffffu, inb && below == w * NSUB + q);
              if (sub == q && hit) e = __ffs(hit) - 1;
            }
          }
          const double tc = nssk::shfl_d(my_t, e);
#pragma unroll
          for (int c = 0; c < NC; ++c)
            if (own[c]) {
              double y = __dadd_rn(xj[c], __dmul_rn(tc, vj[c]));
              if (per[c]) y = wrap_periodic(y, lo_j[c], hi_j[c]);
              X.scr[dst_idx[c]] = y;
            }
          __syncwarp();
          double ly;
          if (KIND == NSS_KIND_GAUSS) ly = have ? nssk::gauss_loglike(P, X.scr) : -INFINITY;
          else ly = nssk::loglike_sub<NDET, KIND, LANES>(P, X, have);
          if (sl == 0) sRes[par][gbase + cs] = ly;
          group_sync(G);
          const double *res = sRes[par] + gbase;
          par ^= 1;
          // ---- replay the sequential decisions: tests outside the box fail without an evaluation, tests inside
          // take the next result; the first test whose result is not there yet ends the round -------------------
          int rank = 0, ti = 0;
          bool expanded = false, stop = false;
          if (!ldone) {
            const bool in = (M >> ti) & 1u; ++ti;
            bool pass = false;
            if (in) { const double v = res[rank++]; ++evals; margin = fmin(margin, fabs(v - Lstar)); pass = v > Lstar; }
            if (pass) { l -= 1.0; ++nl; expanded = true; ldone = nl >= kMaxExpand; } else ldone = true;
          }
          if (ti < nside) {                              // the right end was listed this round
            const bool in = (M >> ti) & 1u; ++ti;
            if (in && rank >= C) stop = true;            // C = 1 and the left end took the only slot
            else {
              bool pass = false;
              if (in) { const double v = res[rank++]; ++evals; margin = fmin(margin, fabs(v - Lstar)); pass = v > Lstar; }
              if (pass) { r += 1.0; ++nr; expanded = true; rdone = nr >= kMaxExpand; } else rdone = true;
            }
          }
          if (ldone && rdone && !expanded && !stop) {
            // shrinkage, all listed proposals at once: lane i holds proposal i - nside.  A proposal outside the box
            // fails for free; one inside has the result of slot `below` if below < C, else it is not known yet.
            const bool shr = lane >= nside && lane < nt;
            const bool has = inb && below < C;
            const double vi = has ? res[has ? below : 0] : -INFINITY;
            const unsigned mU = __ballot_sync(0xffffffffu, shr && inb && below >= C);
            const unsigned mP = __ballot_sync(0xffffffffu, shr && has && vi > Lstar);
            const unsigned mH = __ballot_sync(0xffffffffu, shr && has);
            const int firstU = mU ? __ffs(mU) - 1 : 32, firstP = mP ? __ffs(mP) - 1 : 32;
            const bool accepted = firstP < firstU;
            int end = firstU < firstP ? firstU : firstP;   // proposals [nside, end) failed
            end = end < nt ? end : nt;
            const unsigned upto = accepted ? (firstP == 31 ? 0xffffffffu : ((1u << (firstP + 1)) - 1u))
                                           : (end >= 32 ? 0xffffffffu : ((1u << end) - 1u));
            evals += __popc(mH & upto);
            if (shr && has && ((upto >> lane) & 1u)) margin_l = fmin(margin_l, fabs(vi - Lstar));
            if (accepted) {
              const double tj = nssk::shfl_d(my_t, firstP);
              lx = nssk::shfl_d(vi, firstP);
#pragma unroll
              for (int c = 0; c < NC; ++c) {
                xj[c] = __dadd_rn(xj[c], __dmul_rn(tj, vj[c]));
                if (per[c]) xj[c] = wrap_periodic(xj[c], lo_j[c], hi_j[c]);
              }
              if (lane < d) {                            // d <= NSS_NSLOT < 32: one coordinate per lane
                double y = __dadd_rn(sX[warp][lane], __dmul_rn(tj, vrow[lane]));
                if (lper) y = wrap_periodic(y, llo, lhi);
                sX[warp][lane] = y;
              }
              acc = kk + (firstP - nside); done = true;
            } else {
              const int nrej = end - nside;
              if (nrej > 0) {
                l = nssk::shfl_d(my_ls, end - 1);
                r = nssk::shfl_d(my_rs, end - 1);
                kk += nrej;
              }
              if (kk >= kMaxShrink) done = true;
            }
          }
          __syncwarp();
        }
        if (A.trace && gl == 0) {
          int32_t *tr = A.trace + ((size_t)ch * A.n_repeats + s) * 3;
          tr[0] = nl; tr[1] = nr; tr[2] = acc;
        }
      }
    }
    double margin_all = fmin(margin, margin_l);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) margin_all = fmin(margin_all, __shfl_xor_sync(0xffffffffu, margin_all, o));
    // a10: replace the deleted slot in place
    if (w == 0 && sub == 0) {
      const int dst = A.dead_idx[ch];
#pragma unroll
      for (int c = 0; c < NC; ++c)
        if (own[c]) A.live[(size_t)dst * d + sl + c * LANES] = xj[c];
      if (sl == 0) {
        A.logL[dst] = lx;
        if (A.birth) A.birth[dst] = Lstar;
        if (A.margin) A.margin[ch] = margin_all;
        atomicAdd(&ctl->nevals, (unsigned long long)evals);
        atomicAdd(&ctl->nrounds, (unsigned long long)rounds);
        atomicAdd(&ctl->nexec, (unsigned long long)nexec);
      }
    }
    // a11 (O14) as epilogue: the CTA that finishes the last chain of the iteration computes
    // logZ_live = logX + logsumexp(logL) - ln n over the updated live set and applies the stop test
    if (A.live_evidence) {
      __threadfence();
      group_sync(G);
      unsigned last = 0;
      if (gl == 0) last = atomicAdd(&ctl->chains_done, 1u);
      if (G == 1) last = __shfl_sync(0xffffffffu, last, 0);
      else {
        if (gl == 0) sLast = last;
        __syncthreads();
        last = sLast;
      }
      if (last == (unsigned)A.k - 1u) {
        __threadfence();
        double *red = sRes[0] + gbase;
        const int GT = 32 * G;
        double mx = -INFINITY;
        for (int i = gl; i < A.n; i += GT) mx = fmax(mx, __ldcg(A.logL + i));
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
        group_sync(G);
        if (lane == 0) red[w] = mx;
        group_sync(G);
        mx = red[0];
        for (int q = 1; q < G; ++q) mx = fmax(mx, red[q]);
        group_sync(G);
        double se = 0.0;
        if (mx > -INFINITY)
          for (int i = gl; i < A.n; i += GT) se += exp(__ldcg(A.logL + i) - mx);
        se = nssk::warp_sum(se);
        if (lane == 0) red[w] = se;
        group_sync(G);
        if (gl == 0) {
          double tot = 0.0;
          for (int q = 0; q < G; ++q) tot += red[q];          // fixed order: deterministic
          const double lzl = mx > -INFINITY ? ctl->state[0] + mx + log(tot) - log((double)A.n) : -INFINITY;
          ctl->state[2] = lzl;
          if (lzl - ctl->state[1] < A.stop_dlogz) ctl->flags[2] = 1;
        }
      }
    }
  }
}

template <int NDET, int KIND, int LANES, bool RESIDENT>
int launch_chains_k(nss_handle *h, ChainArgs &A, size_t tab_bytes, cudaStream_t st)
{
  auto kern = k3_slice<NDET, KIND, LANES, RESIDENT>;
  int G = h->chain_warps;
  if (G != 1 && G != 2 && G != 4 && G != 8) {
    // automatic (measured on B200: profiles/r02_config5_microbench.md, third table): a chain is a serial process, so few chains want
    // wide speculation, but once there are about as many warps as SM sub-partitions (4 per SM) the kernel turns
    // throughput-bound and every speculative evaluation costs time
    const long long S = 4LL * h->n_sm;
    G = LANES == 8 ? 1 : (A.k * 8LL <= S ? 4 : A.k <= S ? 2 : 1);
  }
  A.G = G;
  // G > 1: one chain per CTA, the block scheduler balances the SMs.  G == 1: W single-warp chains per CTA share one copy of
  // the record table, and the warps of a persistent grid take chains from a device counter until none is left.
  int W = 1;
  if (G == 1) {
    W = h->chain_pack >= 1 && h->chain_pack <= kChainWarps ? h->chain_pack : (A.k > 4LL * h->n_sm ? 4 : 1);
  }
  const size_t smem = tab_bytes + (size_t)W * G * (32 / LANES) * nssk::kSubScratchDoubles * sizeof(double)
                    + (size_t)W * kDirChunk * NSS_NSLOT * sizeof(double);
  {
    // The dynamic shared memory limit is an attribute of (function, device) shared by every handle and host thread of the
    // process: it is only ever raised, under a lock, and remembered per device (one table per instantiation).
    static std::mutex mu;
    static size_t smem_set[kMaxDevices] = {0};
    if (h->device < 0 || h->device >= kMaxDevices) return NSS_EINVAL;
    std::lock_guard<std::mutex> lock(mu);
    if (smem > smem_set[h->device]) {
      NSS_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      smem_set[h->device] = smem;
    }
  }
  unsigned grid = (unsigned)A.k;
  if (G == 1) {
    // resident CTAs per SM: depends on the instantiation, W and this handle's table size, so it is cached in the handle
    const void *kp = reinterpret_cast<const void *>(kern);
    if (h->occ_kern != kp || h->occ_W != W || h->occ_smem != smem) {
      int nb = 0;
      NSS_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, kern, 32 * W, smem));
      h->occ_kern = kp; h->occ_W = W; h->occ_smem = smem; h->occ_per_sm = nb > 0 ? nb : 1;
    }
    const long long slots = (long long)h->occ_per_sm * h->n_sm, need = (A.k + W - 1) / W;
    grid = (unsigned)(need < slots ? need : slots);
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(32u * G * W); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;      // the prologue (table staging) overlaps the kernels in front
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  // An event in front of K3 separates it from k4_front in the stream (the programmatic launch then overlaps nothing: ~5 us
  // per iteration on B200), so the pair is recorded only on request (nss_set_chain_timing)
  if (h->chain_timing) NSS_CUDA(cudaEventRecord(h->ev_k3[0], st));
  NSS_CUDA(cudaLaunchKernelEx(&cfg, kern, h->dev, A));
  if (h->chain_timing) NSS_CUDA(cudaEventRecord(h->ev_k3[1], st));
  h->ev_k3_valid = h->chain_timing;
  return NSS_OK;
}

template <int NDET>
int launch_chains(nss_handle *h, ChainArgs &A, cudaStream_t st)
{
  const NssDev &P = h->dev;
  if (!h->ev_k3[0]) {
    NSS_CUDA(cudaEventCreate(&h->ev_k3[0]));
    NSS_CUDA(cudaEventCreate(&h->ev_k3[1]));
  }
  int rc;
  if (P.kind == NSS_KIND_RB) {
    // lanes per candidate: 8 shares the per-point setup among four candidates per warp (fewest instructions per
    // evaluation: best when the chains alone fill the SM sub-partitions), 16 halves the latency of a round
    int L = h->chain_lanes;
    if (!(L == 8 || L == 16 || L == 32) || !P.soa[L == 8 ? 0 : L == 16 ? 1 : 2]) {
      const bool many = A.k > 4LL * h->n_sm;             // more chains than SM sub-partitions: fewest instructions wins
      L = (many && P.soa[0]) ? 8 : P.soa[1] ? 16 : P.soa[0] ? 8 : 32;
    }
    const int li = L == 8 ? 0 : L == 16 ? 1 : 2;
    const size_t bytes = (size_t)((9 + 2 * NDET) + P.soa_m[li] * (9 + 3 * NDET)) * L * sizeof(double);
    const bool fits = bytes <= 64 * 1024;                // several CTAs per SM keep their own copy
    if (L == 8)
      rc = fits ? launch_chains_k<NDET, NSS_KIND_RB, 8, true>(h, A, bytes, st) : launch_chains_k<NDET, NSS_KIND_RB, 8, false>(h, A, 0, st);
    else if (L == 16)
      rc = fits ? launch_chains_k<NDET, NSS_KIND_RB, 16, true>(h, A, bytes, st) : launch_chains_k<NDET, NSS_KIND_RB, 16, false>(h, A, 0, st);
    else
      rc = fits ? launch_chains_k<NDET, NSS_KIND_RB, 32, true>(h, A, bytes, st) : launch_chains_k<NDET, NSS_KIND_RB, 32, false>(h, A, 0, st);
  } else if (P.kind == NSS_KIND_FULL) {
    rc = launch_chains_k<NDET, NSS_KIND_FULL, 32, false>(h, A, 0, st);
  } else {
    rc = launch_chains_k<1, NSS_KIND_GAUSS, 32, false>(h, A, 0, st);
  }
  if (rc) return rc;
  h->launches += 1;
  NSS_CUDA(cudaGetLastError());
  return NSS_OK;
}

// start of a stand-alone hook call: clear the flags (and the evaluation counter), optionally load logX / logZ
__global__ void k_begin(NssCtl *ctl, int set_state, double logX, double logZ, int zero_evals)
{
  if (threadIdx.x < 4) ctl->flags[threadIdx.x] = 0;
  if (threadIdx.x == 0) {
    ctl->front_done = 0; ctl->rank_done = 0; ctl->sel_bad = 0; ctl->chains_done = 0; ctl->chain_next = 0; ctl->chol_now = 0; ctl->tune_cnt[0] = 0; ctl->tune_cnt[1] = 0; ctl->tune_cnt[2] = 0;
    if (set_state) { ctl->state[0] = logX; ctl->state[1] = logZ; ctl->state[2] = 0.0; ctl->state[3] = 0.0; }
    if (zero_evals) { ctl->nevals = 0ull; ctl->nrounds = 0ull; ctl->nexec = 0ull; }
  }
}

int begin_iteration(nss_handle *h, int set_state, double logX, double logZ, int zero_evals, cudaStream_t st)
{
  k_begin<<<1, 32, 0, st>>>(h->d_ctl, set_state, logX, logZ, zero_evals);
  h->launches += 1;
  NSS_CUDA(cudaGetLastError());
  return NSS_OK;
}

// one copy of the control block into the pinned mirror, then wait for the stream
int fetch_ctl(nss_handle *h, cudaStream_t st)
{
  NSS_CUDA(cudaMemcpyAsync(h->h_ctl, h->d_ctl, sizeof(NssCtl), cudaMemcpyDeviceToHost, st));
  NSS_CUDA(cudaStreamSynchronize(st));
  return NSS_OK;
}

int ensure_scratch(nss_handle *h, int n)
{
  if (h->scratch_n >= n && h->d_flags) return NSS_OK;
  cudaFree(h->d_surv_idx); cudaFree(h->d_dead_idx); cudaFree(h->d_rank); cudaFree(h->d_rank_part); cudaFree(h->d_birth);
  h->d_surv_idx = h->d_dead_idx = h->d_rank = h->d_rank_part = nullptr; h->d_birth = nullptr;
  NSS_CUDA(cudaMalloc(&h->d_surv_idx, sizeof(int32_t) * n));
  NSS_CUDA(cudaMalloc(&h->d_dead_idx, sizeof(int32_t) * n));
  NSS_CUDA(cudaMalloc(&h->d_rank, sizeof(int32_t) * n));
  NSS_CUDA(cudaMalloc(&h->d_rank_part, sizeof(int32_t) * (size_t)n * kRankMaxSeg));
  NSS_CUDA(cudaMalloc(&h->d_birth, sizeof(double) * n));
  if (!h->d_flags) {
    NSS_CUDA(cudaMalloc(&h->d_ctl, sizeof(NssCtl)));
    NSS_CUDA(cudaMemset(h->d_ctl, 0, sizeof(NssCtl)));
    NSS_CUDA(cudaMallocHost(&h->h_ctl, 2 * sizeof(NssCtl)));     // [1] is nss_run's second slot
    NSS_CUDA(cudaEventCreateWithFlags(&h->ev_ctl[0], cudaEventDisableTiming));
    NSS_CUDA(cudaEventCreateWithFlags(&h->ev_ctl[1], cudaEventDisableTiming));
    NSS_CUDA(cudaMalloc(&h->d_mean, sizeof(double) * NSS_NSLOT));
    NSS_CUDA(cudaMalloc(&h->d_chol, sizeof(double) * NSS_NSLOT * NSS_NSLOT));
    NSS_CUDA(cudaMalloc(&h->d_tune_scratch, sizeof(double) * kTuneMaxBlocks * kTunePartDoubles));
    h->d_state = h->d_ctl->state;             // addresses inside the device block (not dereferenced on the host)
    h->d_nevals = &h->d_ctl->nevals;
    h->d_flags = h->d_ctl->flags;
  }
  h->scratch_n = n;
  return NSS_OK;
}

// the periodic sampled dimensions of the handle (nss_set_periodic) in the form the tuning blocks take
TunePer tune_per_of(const nss_handle *h)
{
  TunePer tp;
  tp.mask = 0; tp.pad_ = 0;
  for (int j = 0; j < NSS_NSLOT; ++j) {
    const bool on = j < h->dev.d && h->dev.periodic[j] != 0;
    if (on) tp.mask |= 1 << j;
    tp.lo[j] = on ? h->dev.lo[j] : 0.0;
    tp.W[j] = on ? h->dev.hi[j] - h->dev.lo[j] : 1.0;
  }
  return tp;
}

// ranks (and the k lowest slots in ascending order) of n > kRankDirectMax values by the sample sort above, five small launches
int launch_sample_rank(nss_handle *h, const double *logL, int n, int k, int32_t *rank, int32_t *dead_idx, int reset, cudaStream_t st)
{
  const int NB = split_buckets(n);
  unsigned char *base = reinterpret_cast<unsigned char *>(h->d_rank_part);       // n x kRankMaxSeg int32 = 128 n bytes
  SplitBufs B;
  B.gv = reinterpret_cast<double *>(base);
  B.spv = B.gv + n;
  int32_t *ip = reinterpret_cast<int32_t *>(B.spv + kSplitMaxBuckets);
  B.gi = ip; B.gb = ip + n; B.eb = ip + 2 * (size_t)n; B.epos = ip + 3 * (size_t)n;
  B.spi = ip + 4 * (size_t)n; B.cnt = B.spi + kSplitMaxBuckets; B.off = B.cnt + kSplitMaxBuckets;
  const unsigned nb = (unsigned)((n + 255) / 256);
  k4s_splitters<<<1, kOneCta, 0, st>>>(logL, n, NB, B, h->d_ctl, reset);
  k4s_bucket<<<nb, 256, 0, st>>>(logL, n, NB, B, h->d_ctl, reset);
  k4s_offsets<<<1, kOneCta, 0, st>>>(NB, B, h->d_ctl, reset);
  k4s_scatter<<<nb, 256, 0, st>>>(logL, n, B, h->d_ctl, reset);
  k4s_rank<<<nb, 256, 0, st>>>(n, k, B, rank, dead_idx, h->d_ctl, reset);
  h->launches += 5;
  NSS_CUDA(cudaGetLastError());
  return NSS_OK;
}

// The device part of one NS iteration (no host synchronisation), two launches:
//   k4_front      a1 rank/select, a2 evidence (if dead_logw), a3 tune, flag and counter reset
//   k3_slice      a4 - a10 (the slice directions a5 are drawn by the chain's own lanes), and a11's live evidence + stop test
//                 as epilogue (if live_evidence)
// `reset`: a stand-alone iteration (flags cleared; logX / logZ loaded and counters zeroed on request).
int enqueue_iteration(nss_handle *h, double *live, double *logL, double *birth, int n, int k, double Lstar_in, int n_repeats,
                      uint64_t seed, uint32_t iteration, double *dead_theta, double *dead_logL, double *dead_birth,
                      int32_t *dead_idx, double *dead_logw, int reset, int set_state, double logX, double logZ, int zero_evals,
                      int live_evidence, double stop_dlogz, cudaStream_t st)
{
  const int d = h->dev.d;
  FrontArgs F;
  F.live = live; F.logL = logL; F.birth = birth; F.n = n; F.k = k; F.d = d; F.Lstar_in = Lstar_in;
  F.T = tune_blocks_on(h, n); F.nseg = n > kRankDirectMax ? 0 : rank_segments(n);
  if (F.nseg == 0) {                                     // many live points: the ranks come from a sample sort (five more launches)
    const int rc = launch_sample_rank(h, logL, n, k, h->d_rank, dead_idx, reset, st);
    if (rc) return rc;
  }
  F.rank_part = h->d_rank_part; F.rank = h->d_rank; F.dead_idx = dead_idx; F.surv_idx = h->d_surv_idx; F.tune_scratch = h->d_tune_scratch;
  F.dead_theta = dead_theta; F.dead_logL = dead_logL; F.dead_birth = dead_birth; F.dead_logw = dead_logw;
  F.mean = h->d_mean; F.chol = h->d_chol; F.ctl = h->d_ctl; F.per = tune_per_of(h);
  F.reset = reset; F.set_state = set_state; F.zero_evals = zero_evals; F.logX = logX; F.logZ = logZ;
  k4_front<<<F.T + (F.nseg ? ((n + kRankElems - 1) / kRankElems) * F.nseg : 1), kOneCta, 0, st>>>(F);
  h->launches += 1;
  NSS_CUDA(cudaGetLastError());
  ChainArgs A;
  A.live = live; A.logL = logL; A.birth = birth; A.n = n; A.k = k; A.n_repeats = n_repeats; A.seed = seed;
  A.iteration = iteration; A.surv_idx = h->d_surv_idx; A.dead_idx = dead_idx; A.chol = h->d_chol; A.ctl = h->d_ctl;
  A.trace = h->trace_dev; A.margin = h->margin_dev; A.G = 1; A.live_evidence = live_evidence; A.stop_dlogz = stop_dlogz;
  switch (h->dev.n_det) {
    case 0: case 1: return launch_chains<1>(h, A, st);
    case 2: return launch_chains<2>(h, A, st);
    case 3: return launch_chains<3>(h, A, st);
    default: return launch_chains<4>(h, A, st);
  }
}

}  // namespace

extern "C" int nss_last_chain_ms(nss_handle *h, double *ms_host)
{
  if (!h || !ms_host || !h->ev_k3_valid) return NSS_EINVAL;
  NSS_CUDA(cudaEventSynchronize(h->ev_k3[1]));
  float ms = 0.f;
  NSS_CUDA(cudaEventElapsedTime(&ms, h->ev_k3[0], h->ev_k3[1]));
  *ms_host = ms;
  return NSS_OK;
}

extern "C" int nss_last_chain_diag(nss_handle *h, int64_t *rounds_host, int64_t *evaluated_host)
{
  if (!h || !h->h_ctl) return NSS_EINVAL;
  if (rounds_host) *rounds_host = (int64_t)h->h_ctl->nrounds;
  if (evaluated_host) *evaluated_host = (int64_t)h->h_ctl->nexec;
  return NSS_OK;
}

extern "C" int nss_set_chain_warps(nss_handle *h, int32_t warps)
{
  if (!h || !(warps == 0 || warps == 1 || warps == 2 || warps == 4 || warps == 8)) return NSS_EINVAL;
  h->chain_warps = warps;
  return NSS_OK;
}

extern "C" int nss_set_chain_lanes(nss_handle *h, int32_t lanes)
{
  if (!h || !(lanes == 0 || lanes == 8 || lanes == 16 || lanes == 32)) return NSS_EINVAL;
  h->chain_lanes = lanes;
  return NSS_OK;
}

extern "C" int nss_set_chain_timing(nss_handle *h, int32_t on)
{
  if (!h) return NSS_EINVAL;
  h->chain_timing = on != 0;
  if (!on) h->ev_k3_valid = 0;
  return NSS_OK;
}

extern "C" int nss_set_chain_pack(nss_handle *h, int32_t chains_per_cta)
{
  if (!h || chains_per_cta < 0 || chains_per_cta > kChainWarps) return NSS_EINVAL;
  h->chain_pack = chains_per_cta;
  return NSS_OK;
}

extern "C" int nss_set_periodic(nss_handle *h, const int32_t *flags_host)
{
  if (!h) return NSS_EINVAL;
  for (int j = 0; j < NSS_NSLOT; ++j) h->dev.periodic[j] = (flags_host && j < h->dev.d) ? (flags_host[j] != 0) : 0;
  return NSS_OK;
}

extern "C" int nss_set_trace(nss_handle *h, int32_t *trace_dev, double *margin_dev)
{
  if (!h) return NSS_EINVAL;
  h->trace_dev = trace_dev;
  h->margin_dev = margin_dev;
  return NSS_OK;
}

extern "C" int nss_philox(nss_handle *h, uint64_t seed, const uint32_t *ctr_dev, int64_t n, uint32_t *out_dev, void *cuda_stream)
{
  if (!h || n < 0 || (n > 0 && (!ctr_dev || !out_dev))) return NSS_EINVAL;
  if (n == 0) return NSS_OK;
  NSS_CUDA(cudaSetDevice(h->device));
  k_philox<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)cuda_stream>>>(seed, ctr_dev, n, out_dev);
  h->launches += 1;
  NSS_CUDA(cudaGetLastError());
  return NSS_OK;
}

extern "C" int nss_init_live(nss_handle *h, int32_t n_live, uint64_t seed, double *live_dev, double *logL_dev, void *cuda_stream)
{
  if (!h || n_live < 1 || !live_dev || !logL_dev) return NSS_EINVAL;
  NSS_CUDA(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int tot = n_live * h->dev.d;
  k_init_live<<<(tot + 255) / 256, 256, 0, st>>>(h->dev, n_live, seed, live_dev);
  h->launches += 1;
  NSS_CUDA(cudaGetLastError());
  return nss_launch_loglike(h, live_dev, n_live, logL_dev, st);
}

extern "C" int nss_select_lowest(nss_handle *h, const double *logL_dev, int32_t n_live, int32_t n_delete, int32_t *dead_idx_dev,
                                 int32_t *surv_idx_dev, double *logLstar_host, void *cuda_stream)
{
  if (!h || !logL_dev || !dead_idx_dev || n_live < 2 || n_delete < 1 || n_delete >= n_live) return NSS_EINVAL;
  NSS_CUDA(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = ensure_scratch(h, n_live);
  if (rc) return rc;
  rc = begin_iteration(h, 0, 0.0, 0.0, 0, st);
  if (rc) return rc;
  const int nseg = n_live > kRankDirectMax ? 0 : rank_segments(n_live);
  if (nseg == 0) {
    rc = launch_sample_rank(h, logL_dev, n_live, n_delete, h->d_rank, dead_idx_dev, 1, st);
    if (rc) return rc;
  } else {
    k4_rank<<<((n_live + kRankElems - 1) / kRankElems) * nseg, kOneCta, 0, st>>>(logL_dev, n_live, nseg, h->d_rank_part);
    h->launches += 1;
  }
  k4_finish_select<<<1, kOneCta, 0, st>>>(logL_dev, n_live, n_delete, nseg, h->d_rank_part, h->d_rank, dead_idx_dev,
                                          surv_idx_dev ? surv_idx_dev : h->d_surv_idx, h->d_state);
  h->launches += 1;
  NSS_CUDA(cudaGetLastError());
  rc = fetch_ctl(h, st);
  if (rc) return rc;
  if (logLstar_host) *logLstar_host = h->h_ctl->state[3];
  return NSS_OK;
}

extern "C" int nss_tune(nss_handle *h, const double *live_dev, int32_t n_live, double *mean_dev, double *chol_dev, void *cuda_stream)
{
  if (!h || !live_dev || !chol_dev || n_live < 2) return NSS_EINVAL;
  NSS_CUDA(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = ensure_scratch(h, n_live);
  if (rc) return rc;
  rc = begin_iteration(h, 0, 0.0, 0.0, 0, st);
  if (rc) return rc;
  const int T = tune_blocks_on(h, n_live);
  k4_tune<<<T, kOneCta, 0, st>>>(live_dev, n_live, h->dev.d, T, h->d_tune_scratch, h->d_ctl, mean_dev, chol_dev, tune_per_of(h));
  h->launches += 1;
  NSS_CUDA(cudaGetLastError());
  rc = fetch_ctl(h, st);
  if (rc) return rc;
  return h->h_ctl->flags[0] ? NSS_ECHOL : NSS_OK;
}

extern "C" int nss_evidence_update(nss_handle *h, const double *dead_logL_dev, int32_t n_live, int32_t n_delete, double *logw_dev,
                                   double *state_host, void *cuda_stream)
{
  if (!h || !dead_logL_dev || !logw_dev || !state_host || n_delete < 1 || n_delete >= n_live) return NSS_EINVAL;
  NSS_CUDA(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = ensure_scratch(h, n_live);
  if (rc) return rc;
  rc = begin_iteration(h, 1, state_host[0], state_host[1], 0, st);
  if (rc) return rc;
  k4_evidence<<<1, kOneCta, 0, st>>>(dead_logL_dev, n_live, n_delete, logw_dev, h->d_state);
  h->launches += 1;
  NSS_CUDA(cudaGetLastError());
  rc = fetch_ctl(h, st);
  if (rc) return rc;
  state_host[0] = h->h_ctl->state[0];
  state_host[1] = h->h_ctl->state[1];
  return NSS_OK;
}

extern "C" int nss_replace_step(nss_handle *h, double *live_dev, double *logL_dev, int32_t n_live, int32_t n_delete, double logLstar,
                                int32_t n_repeats, uint64_t seed, uint32_t iteration, double *dead_theta_dev, double *dead_logL_dev,
                                int32_t *dead_idx_dev, double *logLstar_host, int64_t *n_evals_host, void *cuda_stream)
{
  if (!h || !live_dev || !logL_dev || !dead_theta_dev || !dead_logL_dev || !dead_idx_dev) return NSS_EINVAL;
  if (n_live < 2 || n_delete < 1 || n_delete >= n_live || n_repeats < 0) return NSS_EINVAL;
  NSS_CUDA(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = ensure_scratch(h, n_live);
  if (rc) return rc;
  rc = enqueue_iteration(h, live_dev, logL_dev, nullptr, n_live, n_delete, logLstar, n_repeats, seed, iteration, dead_theta_dev,
                         dead_logL_dev, nullptr, dead_idx_dev, nullptr, /*reset*/ 1, /*set_state*/ 0, 0.0, 0.0, /*zero_evals*/ 1,
                         /*live_evidence*/ 0, 0.0, st);
  if (rc) return rc;
  rc = fetch_ctl(h, st);
  if (rc) return rc;
  if (logLstar_host) *logLstar_host = h->h_ctl->state[3];
  if (n_evals_host) *n_evals_host = (int64_t)h->h_ctl->nevals;
  if (h->h_ctl->flags[1]) return NSS_EINVAL;
  if (h->h_ctl->flags[0]) return NSS_ECHOL;
  return NSS_OK;
}

extern "C" int nss_resample_equal(nss_handle *h, const double *logL_dev, const double *logw_dev, int64_t n, uint64_t seed,
                                  int64_t *idx_dev, int64_t *n_equal_host, void *cuda_stream)
{
  if (!h || n < 0 || !n_equal_host || (n > 0 && (!logL_dev || !logw_dev))) return NSS_EINVAL;
  *n_equal_host = 0;
  if (n == 0) return NSS_OK;
  NSS_CUDA(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = ensure_scratch(h, 2);
  if (rc) return rc;
  static_assert(sizeof(long long) == sizeof(int64_t), "int64_t rows");
  k_resample_equal<<<1, kOneCta, 0, st>>>(logL_dev, logw_dev, (long long)n, seed, (long long *)idx_dev, h->d_tune_scratch);
  h->launches += 1;
  NSS_CUDA(cudaGetLastError());
  double cnt = 0.0;
  NSS_CUDA(cudaMemcpyAsync(&cnt, h->d_tune_scratch, sizeof(double), cudaMemcpyDeviceToHost, st));
  NSS_CUDA(cudaStreamSynchronize(st));
  *n_equal_host = (int64_t)cnt;
  return NSS_OK;
}

namespace {
int ensure_stage(nss_handle *h, size_t bytes)
{
  if (h->stage_bytes >= bytes && h->d_stage) return NSS_OK;
  cudaFree(h->d_stage);
  h->d_stage = nullptr; h->stage_bytes = 0;
  cudaError_t e = cudaMalloc((void **)&h->d_stage, bytes);
  if (e != cudaSuccess) { nss_cuda_fail(e, "cudaMalloc(stage)"); return e == cudaErrorMemoryAllocation ? NSS_ENOMEM : NSS_ECUDA; }
  h->stage_bytes = bytes;
  return NSS_OK;
}
size_t align256(size_t b) { return (b + 255) & ~(size_t)255; }
}  // namespace

extern "C" int nss_iterate(nss_handle *h, double *live_dev, double *logL_dev, int32_t n_live, int32_t n_delete, int32_t n_repeats,
                           uint64_t seed, uint32_t iteration, double stop_dlogz, double *dead_theta_dev, double *dead_logL_dev,
                           double *dead_logw_dev, int32_t *dead_idx_dev, nss_iter_state *state_host, void *cuda_stream)
{
  if (!h || !live_dev || !logL_dev || !dead_theta_dev || !dead_logL_dev || !dead_logw_dev || !dead_idx_dev || !state_host)
    return NSS_EINVAL;
  if (n_live < 2 || n_delete < 1 || n_delete >= n_live || n_repeats < 0) return NSS_EINVAL;
  NSS_CUDA(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = ensure_scratch(h, n_live);
  if (rc) return rc;
  rc = enqueue_iteration(h, live_dev, logL_dev, nullptr, n_live, n_delete, NAN, n_repeats, seed, iteration, dead_theta_dev,
                         dead_logL_dev, nullptr, dead_idx_dev, dead_logw_dev, /*reset*/ 1, /*set_state*/ 1, state_host->logX,
                         state_host->logZ, /*zero_evals*/ 1, /*live_evidence*/ 1, stop_dlogz, st);
  if (rc) return rc;
  rc = fetch_ctl(h, st);
  if (rc) return rc;
  const NssCtl &c = *h->h_ctl;
  if (c.flags[0]) return NSS_ECHOL;
  state_host->logX = c.state[0]; state_host->logZ = c.state[1]; state_host->logZ_live = c.state[2]; state_host->logLstar = c.state[3];
  state_host->n_evals = (int64_t)c.nevals;
  state_host->converged = c.flags[2];
  return NSS_OK;
}

extern "C" int nss_iterate_host(nss_handle *h, double *live_host, double *logL_host, int32_t n_live, int32_t n_delete,
                                int32_t n_repeats, uint64_t seed, uint32_t iteration, double stop_dlogz, double *dead_theta_host,
                                double *dead_logL_host, double *dead_logw_host, int32_t *dead_idx_host, nss_iter_state *state_host,
                                void *cuda_stream)
{
  if (!h || !live_host || !logL_host || !dead_theta_host || !dead_logL_host || !dead_logw_host || !dead_idx_host || !state_host)
    return NSS_EINVAL;
  if (n_live < 2 || n_delete < 1 || n_delete >= n_live || n_repeats < 0) return NSS_EINVAL;
  NSS_CUDA(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t d = (size_t)h->dev.d, n = (size_t)n_live, k = (size_t)n_delete;
  const size_t o_live = 0, o_logL = o_live + align256(n * d * 8), o_dth = o_logL + align256(n * 8),
               o_dl = o_dth + align256(k * d * 8), o_dw = o_dl + align256(k * 8), o_di = o_dw + align256(k * 8),
               total = o_di + align256(k * 4);
  int rc = ensure_stage(h, total);
  if (rc) return rc;
  unsigned char *b = h->d_stage;
  double *live = (double *)(b + o_live), *logL = (double *)(b + o_logL), *dth = (double *)(b + o_dth), *dl = (double *)(b + o_dl),
         *dw = (double *)(b + o_dw);
  int32_t *di = (int32_t *)(b + o_di);
  // everything is queued on the stream — inputs in, the iteration, the control block and the results out — and the
  // host waits once (on a Cholesky failure the live set comes back unchanged and the dead rows are those selected)
  NSS_CUDA(cudaMemcpyAsync(live, live_host, n * d * 8, cudaMemcpyHostToDevice, st));
  NSS_CUDA(cudaMemcpyAsync(logL, logL_host, n * 8, cudaMemcpyHostToDevice, st));
  rc = ensure_scratch(h, n_live);
  if (rc) return rc;
  rc = enqueue_iteration(h, live, logL, nullptr, n_live, n_delete, NAN, n_repeats, seed, iteration, dth, dl, nullptr, di, dw,
                         /*reset*/ 1, /*set_state*/ 1, state_host->logX, state_host->logZ, /*zero_evals*/ 1, /*live_evidence*/ 1,
                         stop_dlogz, st);
  if (rc) return rc;
  NSS_CUDA(cudaMemcpyAsync(h->h_ctl, h->d_ctl, sizeof(NssCtl), cudaMemcpyDeviceToHost, st));
  NSS_CUDA(cudaMemcpyAsync(live_host, live, n * d * 8, cudaMemcpyDeviceToHost, st));
  NSS_CUDA(cudaMemcpyAsync(logL_host, logL, n * 8, cudaMemcpyDeviceToHost, st));
  NSS_CUDA(cudaMemcpyAsync(dead_theta_host, dth, k * d * 8, cudaMemcpyDeviceToHost, st));
  NSS_CUDA(cudaMemcpyAsync(dead_logL_host, dl, k * 8, cudaMemcpyDeviceToHost, st));
  NSS_CUDA(cudaMemcpyAsync(dead_logw_host, dw, k * 8, cudaMemcpyDeviceToHost, st));
  NSS_CUDA(cudaMemcpyAsync(dead_idx_host, di, k * 4, cudaMemcpyDeviceToHost, st));
  NSS_CUDA(cudaStreamSynchronize(st));
  const NssCtl &c = *h->h_ctl;
  if (c.flags[0]) return NSS_ECHOL;
  state_host->logX = c.state[0]; state_host->logZ = c.state[1]; state_host->logZ_live = c.state[2]; state_host->logLstar = c.state[3];
  state_host->n_evals = (int64_t)c.nevals;
  state_host->converged = c.flags[2];
  return NSS_OK;
}

extern "C" int nss_loglike_batch_host(nss_handle *h, const double *theta_host, int64_t N, double *logL_host, void *cuda_stream)
{
  if (!h || N < 0) return NSS_EINVAL;
  if (N == 0) return NSS_OK;
  if (!theta_host || !logL_host) return NSS_EINVAL;
  NSS_CUDA(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t d = (size_t)h->dev.d, o_out = align256((size_t)N * d * 8);
  int rc = ensure_stage(h, o_out + align256((size_t)N * 8));
  if (rc) return rc;
  double *th = (double *)h->d_stage, *out = (double *)(h->d_stage + o_out);
  NSS_CUDA(cudaMemcpyAsync(th, theta_host, (size_t)N * d * 8, cudaMemcpyHostToDevice, st));
  rc = nss_launch_loglike(h, th, N, out, st);
  if (rc) return rc;
  NSS_CUDA(cudaMemcpyAsync(logL_host, out, (size_t)N * 8, cudaMemcpyDeviceToHost, st));
  NSS_CUDA(cudaStreamSynchronize(st));
  return NSS_OK;
}

extern "C" int nss_run(nss_handle *h, int32_t n_live, int32_t n_delete, int32_t n_repeats, uint64_t seed, double stop_dlogz,
                       int32_t max_iter, nss_result *out, void *cuda_stream)
{
  if (!h || !out || !out->dead_theta || !out->dead_logL || !out->dead_logL_birth || !out->dead_logw) return NSS_EINVAL;
  if (n_live < 2 || n_delete < 1 || n_delete >= n_live || n_repeats < 0 || max_iter < 0) return NSS_EINVAL;
  if (out->cap < n_live) return NSS_ECAP;
  NSS_CUDA(cudaSetDevice(h->device));
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int n = n_live, k = n_delete, d = h->dev.d;
  int rc = ensure_scratch(h, n);
  if (rc) return rc;
  const int64_t cap = out->cap;
  // one device block, kept by the handle between runs: live, logL, the dead buffers and the replica evidences
  const size_t o_live = 0, o_logL = o_live + align256(sizeof(double) * (size_t)n * d), o_dth = o_logL + align256(sizeof(double) * n),
               o_dl = o_dth + align256(sizeof(double) * (size_t)cap * d), o_db = o_dl + align256(sizeof(double) * cap),
               o_dw = o_db + align256(sizeof(double) * cap), o_err = o_dw + align256(sizeof(double) * cap),
               o_eq = o_err + align256(sizeof(double) * (kErrReplicas + 2)),
               total = o_eq + (out->equal_idx ? align256(sizeof(int64_t) * cap) : 0);
  if (h->run_bytes < total) {
    cudaFree(h->d_run);
    h->d_run = nullptr; h->run_bytes = 0;
    cudaError_t e = cudaMalloc((void **)&h->d_run, total);
    if (e != cudaSuccess) { nss_cuda_fail(e, "cudaMalloc(run)"); return e == cudaErrorMemoryAllocation ? NSS_ENOMEM : NSS_ECUDA; }
    h->run_bytes = total;
  }
  if (!h->ev_run[0]) {
    NSS_CUDA(cudaEventCreate(&h->ev_run[0]));
    NSS_CUDA(cudaEventCreate(&h->ev_run[1]));
  }
  unsigned char *rb = h->d_run;
  double *live = (double *)(rb + o_live), *logL = (double *)(rb + o_logL), *dth = (double *)(rb + o_dth), *dl = (double *)(rb + o_dl),
         *db = (double *)(rb + o_db), *dw = (double *)(rb + o_dw), *derr = (double *)(rb + o_err);
  long long *deq = out->equal_idx ? (long long *)(rb + o_eq) : nullptr;
  cudaEvent_t e0 = h->ev_run[0], e1 = h->ev_run[1];
  // every exit, the error exits included, leaves the stream drained (an iteration may still be queued)
  auto cleanup = [&]() { cudaStreamSynchronize(st); };
#define RUN_CUDA(x)                                                           \
  do {                                                                        \
    cudaError_t e__ = (x);                                                    \
    if (e__ != cudaSuccess) { cleanup(); return nss_cuda_fail(e__, #x); }     \
  } while (0)

  RUN_CUDA(cudaEventRecord(e0, st));
  rc = begin_iteration(h, 1, 0.0, -INFINITY, 1, st);
  if (rc) { cleanup(); return rc; }
  rc = nss_init_live(h, n, seed, live, logL, st);
  if (rc) { cleanup(); return rc; }
  k_fill<<<(n + 255) / 256, 256, 0, st>>>(h->d_birth, n, -INFINITY);
  h->launches += 1;
  int t = 0;
  int64_t n_dead = 0;
  int result = NSS_OK;
  // The loop runs one iteration ahead of the host: the stop test of iteration t (the epilogue of its K3 sets flags[2] on
  // the device) is read from a pinned slot while iteration t+1 is already queued.  Both kernels of an iteration return
  // at once when flags[2] (or the Cholesky flag) is set, so an iteration queued past the end of the run changes nothing.
  auto stage = [&](int tt) -> int {
    if (tt == 0) {                                       // logZ_live of the initial live set (no stop test before iteration 0)
      k4_live_evidence<<<1, kOneCta, 0, st>>>(logL, n, stop_dlogz, 0, h->d_state, h->d_flags);
      h->launches += 1;
    }
    NSS_CUDA(cudaMemcpyAsync(&h->h_ctl[tt & 1], h->d_ctl, sizeof(NssCtl), cudaMemcpyDeviceToHost, st));
    NSS_CUDA(cudaEventRecord(h->ev_ctl[tt & 1], st));
    return NSS_OK;
  };
  rc = stage(0);
  if (rc) { cleanup(); return rc; }
  for (;;) {
    const bool room = n_dead + k + n <= cap, more = t < max_iter;
    if (room && more) {
      rc = enqueue_iteration(h, live, logL, h->d_birth, n, k, NAN, n_repeats, seed, (uint32_t)t, dth + (size_t)n_dead * d, dl + n_dead,
                             db + n_dead, h->d_dead_idx, dw + n_dead, /*reset*/ 0, 0, 0.0, 0.0, 0, /*live_evidence*/ 1, stop_dlogz, st);
      if (rc) { cleanup(); return rc; }
      rc = stage(t + 1);
      if (rc) { cleanup(); return rc; }
    }
    RUN_CUDA(cudaEventSynchronize(h->ev_ctl[t & 1]));
    const NssCtl &c = h->h_ctl[t & 1];
    if (c.flags[0]) { result = NSS_ECHOL; break; }
    if (c.flags[2]) break;                               // converged before iteration t: what was queued for it did nothing
    if (!more) { result = NSS_ENOTCONV; break; }
    if (!room) { result = NSS_ECAP; break; }
    n_dead += k;
    ++t;
  }
  if (result == NSS_OK || result == NSS_ENOTCONV) {
    // O14: append the live points in ascending logL
    const int nseg = n > kRankDirectMax ? 0 : rank_segments(n);
    if (nseg == 0) {
      rc = launch_sample_rank(h, logL, n, n, h->d_rank, h->d_dead_idx, 1, st);
      if (rc) { cleanup(); return rc; }
    } else {
      k4_rank<<<((n + kRankElems - 1) / kRankElems) * nseg, kOneCta, 0, st>>>(logL, n, nseg, h->d_rank_part);
      h->launches += 1;
    }
    k4_finish_select<<<1, kOneCta, 0, st>>>(logL, n, n, nseg, h->d_rank_part, h->d_rank, h->d_dead_idx, nullptr, nullptr);
    k_gather_rows<<<(n + 255) / 256, 256, 0, st>>>(live, logL, h->d_birth, h->d_dead_idx, n, d, dth + (size_t)n_dead * d, dl + n_dead,
                                                   db + n_dead);
    h->launches += 2;
    const int64_t n_it_dead = n_dead;
    n_dead += n;
    // O15: the replica evidences, the Kish ESS and the equal-weight rows on the device (one CTA per replica; one CTA each)
    k_fill_live_logw<<<(n + 255) / 256, 256, 0, st>>>(dw + n_it_dead, n, h->d_state);
    k_evidence_error<<<kErrReplicas, 256, 0, st>>>(dl, n_it_dead, n, k, seed, logL, derr);
    k_kish_ess<<<1, kOneCta, 0, st>>>(dl, dw, n_it_dead, logL, n, h->d_state, derr + kErrReplicas);
    k_resample_equal<<<1, kOneCta, 0, st>>>(dl, dw, (long long)n_dead, seed, deq, derr + kErrReplicas + 1);
    h->launches += 4;
    // results: device -> one pinned staging block (asynchronous copies whatever memory the caller's arrays are in) -> caller
    const size_t nd = (size_t)n_dead;
    const size_t s_th = 0, s_l = s_th + align256(sizeof(double) * nd * d), s_b = s_l + align256(sizeof(double) * nd),
                 s_w = s_b + align256(sizeof(double) * nd), s_misc = s_w + align256(sizeof(double) * nd),
                 s_eq = s_misc + align256(sizeof(double) * (kErrReplicas + 2 + 4 + 1)),
                 s_total = s_eq + (deq ? align256(sizeof(int64_t) * nd) : 0);
    if (h->h_run_bytes < s_total) {
      if (h->h_run) cudaFreeHost(h->h_run);
      h->h_run = nullptr; h->h_run_bytes = 0;
      cudaError_t e = cudaMallocHost((void **)&h->h_run, s_total + s_total / 2);     // room to grow: pinning is slow
      if (e != cudaSuccess) { cleanup(); nss_cuda_fail(e, "cudaMallocHost(run)"); return NSS_ENOMEM; }
      h->h_run_bytes = s_total + s_total / 2;
    }
    unsigned char *hb = h->h_run;
    double *lz_rep = (double *)(hb + s_misc);            // [kErrReplicas] replicas, then Kish ESS, equal-weight rows
    double *state = lz_rep + kErrReplicas + 2;           // logX, logZ, logZ_live, L*
    unsigned long long *ne_p = (unsigned long long *)(state + 4);
    RUN_CUDA(cudaMemcpyAsync(hb + s_th, dth, sizeof(double) * nd * d, cudaMemcpyDeviceToHost, st));
    RUN_CUDA(cudaMemcpyAsync(hb + s_l, dl, sizeof(double) * nd, cudaMemcpyDeviceToHost, st));
    RUN_CUDA(cudaMemcpyAsync(hb + s_b, db, sizeof(double) * nd, cudaMemcpyDeviceToHost, st));
    RUN_CUDA(cudaMemcpyAsync(hb + s_w, dw, sizeof(double) * nd, cudaMemcpyDeviceToHost, st));
    RUN_CUDA(cudaMemcpyAsync(lz_rep, derr, sizeof(double) * (kErrReplicas + 2), cudaMemcpyDeviceToHost, st));
    RUN_CUDA(cudaMemcpyAsync(state, h->d_state, sizeof(double) * 4, cudaMemcpyDeviceToHost, st));
    RUN_CUDA(cudaMemcpyAsync(ne_p, h->d_nevals, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    if (deq) RUN_CUDA(cudaMemcpyAsync(hb + s_eq, deq, sizeof(int64_t) * nd, cudaMemcpyDeviceToHost, st));
    RUN_CUDA(cudaEventRecord(e1, st));
    RUN_CUDA(cudaStreamSynchronize(st));
    memcpy(out->dead_theta, hb + s_th, sizeof(double) * nd * d);
    memcpy(out->dead_logL, hb + s_l, sizeof(double) * nd);
    memcpy(out->dead_logL_birth, hb + s_b, sizeof(double) * nd);
    memcpy(out->dead_logw, hb + s_w, sizeof(double) * nd);
    const unsigned long long ne = *ne_p;
    float ms = 0.f;
    RUN_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    out->gpu_ms = ms;
    const double logX = state[0], logZ = state[1], logZ_live = state[2];
    auto lae = [](double a, double b) {
      if (a == -INFINITY) return b;
      if (b == -INFINITY) return a;
      const double m = a > b ? a : b;
      return m + log(exp(a - m) + exp(b - m));
    };
    const double logZf = lae(logZ, logZ_live);
    // O15: information and replica evidence error (host post-processing)
    double H = 0.0;
    for (int64_t i = 0; i < n_dead; ++i)
      if (out->dead_logL[i] > -INFINITY) H += exp(out->dead_logL[i] + out->dead_logw[i] - logZf) * (out->dead_logL[i] - logZf);
    const int R = kErrReplicas;
    double sum = 0.0, sum2 = 0.0;
    for (int rpl = 0; rpl < R; ++rpl) { sum += lz_rep[rpl]; sum2 += lz_rep[rpl] * lz_rep[rpl]; }
    const double mu = sum / R;
    double var = sum2 / R - mu * mu;
    var = var < 0 ? 0 : var;
    out->logZ = logZf; out->logZ_err = sqrt(var * R / (R - 1)); out->H = H;
    out->ess = lz_rep[kErrReplicas];
    out->n_equal = (int64_t)lz_rep[kErrReplicas + 1];
    if (out->equal_idx && out->n_equal > 0) memcpy(out->equal_idx, hb + s_eq, sizeof(int64_t) * (size_t)out->n_equal);
    out->n_iter = t; out->n_dead = n_dead; out->n_evals = (int64_t)ne + n;
  }
#undef RUN_CUDA
  cleanup();
  return result;
}

// ---- nss_select_lowest_static: the delete-select (a1, O12.1) for callers that must not allocate ---------------------------
// The counting select needs work space beside its inputs and outputs: the partial counts of every (segment, live point)
// pair, the ranks, and a survivor list when the caller does not want one.  nss_select_lowest keeps that space in the handle
// and grows it with cudaMalloc; this entry point keeps it in the image of the library instead, so neither creating a handle
// nor the call itself asks the CUDA allocator for anything.  See include/nss.h for who needs that and what it costs.
//
// Layout of the array, in 32-bit words (kSelStaticLive = NSS_SELECT_STATIC_MAX_LIVE = the largest n the counting select
// serves, kRankDirectMax):
//   [0, 32 n_max)            partial counts, [segment][live point] with the call's own n as the row length
//   [32 n_max, 33 n_max)     ranks
//   [33 n_max, 34 n_max)     survivor list when surv_idx_dev is NULL
//   then 4 doubles           the {logX, logZ, logZ_live, L*} block the selection tail writes L* into
constexpr int kSelStaticLive = NSS_SELECT_STATIC_MAX_LIVE;
static_assert(kSelStaticLive == kRankDirectMax, "the static select serves exactly the sizes the counting ranks serve");
constexpr size_t kSelStaticWords = (size_t)(kRankMaxSeg + 2) * kSelStaticLive + 8;
static __device__ __align__(256) int32_t g_sel_static[kSelStaticWords];       // 1 114 144 bytes on every device that loads libnss.so

namespace {

// The tail of the counting select on the static work space: partial counts -> ranks and dead list, survivor compaction,
// threshold.  Same device functions, in the same order, as k4_finish_select; the threshold also goes to the caller's slot.
__global__ void __launch_bounds__(kOneCta) k4_finish_select_static(const double *__restrict__ logL, int n, int k, int nseg,
                                                                   const int32_t *__restrict__ part, int32_t *__restrict__ rank,
                                                                   int32_t *__restrict__ dead_idx, int32_t *__restrict__ surv_idx,
                                                                   double *__restrict__ state, double *__restrict__ logLstar_out)
{
  __shared__ K4Smem sm;
  rank_finish(part, n, k, nseg, rank, dead_idx);
  finish_select_block(nullptr, logL, nullptr, n, k, 0, NAN, rank, dead_idx, surv_idx, nullptr, nullptr, nullptr, state, sm);
  if (threadIdx.x == 0 && logLstar_out) *logLstar_out = state[3];      // written by thread 0 just above
}

// In host code `g_sel_static` is only a handle for the runtime, not an address a kernel can use: the device address is
// asked for once per device (with that device current) and remembered.
constexpr int kSelStaticMaxDevices = 64;
int32_t *g_sel_static_dev[kSelStaticMaxDevices];
std::mutex g_sel_static_mu;

int sel_static_base(int32_t **base)
{
  int dev = -1;
  NSS_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kSelStaticMaxDevices) return NSS_EINVAL;
  std::lock_guard<std::mutex> lock(g_sel_static_mu);
  if (!g_sel_static_dev[dev]) {
    void *p = nullptr;
    NSS_CUDA(cudaGetSymbolAddress(&p, g_sel_static));
    if (!p) return NSS_ECUDA;
    g_sel_static_dev[dev] = static_cast<int32_t *>(p);
  }
  *base = g_sel_static_dev[dev];
  return NSS_OK;
}

}  // namespace

extern "C" int nss_select_lowest_static(const double *logL_dev, int32_t n_live, int32_t n_delete, int32_t *dead_idx_dev,
                                        int32_t *surv_idx_dev, double *logLstar_dev, void *cuda_stream)
{
  if (!logL_dev || !dead_idx_dev || n_live < 2 || n_delete < 1 || n_delete >= n_live) return NSS_EINVAL;
  if (n_live > kSelStaticLive) return NSS_ELIMIT;
  int32_t *base = nullptr;
  const int rc = sel_static_base(&base);
  if (rc) return rc;
  int32_t *part = base, *rank = base + (size_t)kRankMaxSeg * kSelStaticLive, *surv = rank + kSelStaticLive;
  double *state = reinterpret_cast<double *>(surv + kSelStaticLive);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // Nothing in the work space has to start at zero: both kernels write every word they (or the next kernel) later read —
  // part[sg][i] for every sg < nseg, i < n; rank[i] for every i < n; state[3] — so what an earlier call left is never seen.
  const int nseg = rank_segments(n_live);
  k4_rank<<<((n_live + kRankElems - 1) / kRankElems) * nseg, kOneCta, 0, st>>>(logL_dev, n_live, nseg, part);
  k4_finish_select_static<<<1, kOneCta, 0, st>>>(logL_dev, n_live, n_delete, nseg, part, rank, dead_idx_dev,
                                                 surv_idx_dev ? surv_idx_dev : surv, state, logLstar_dev);
  NSS_CUDA(cudaGetLastError());
  return NSS_OK;
}
