// nss_loglike.cu — batch likelihood kernels behind nss_loglike_batch.
//
//  k1_rb_thread : relative binning, ONE THREAD per point.  The AoS edge/bin table is staged into shared
//                 memory by TMA bulk copies (when it fits) and read by broadcast; a persistent grid-stride
//                 loop over points.  Highest throughput for large N (no per-point redundancy, no shuffles).
//  k1_rb_warp   : relative binning, ONE WARP per point (lanes own contiguous bin slices, warp-shuffle
//                 reduction).  For small N, and the form the slice sampler uses.
//  k2_full_warp : full frequency grid, one warp per point, 128-bit coalesced loads of data/PSD records.
//  k_gauss      : O16 test likelihood.
#include "nss_loglike_dev.cuh"

namespace {

constexpr int kThreads = 256;
constexpr size_t kSmemMax = 227 * 1024;

template <int NDET, bool RESIDENT>
__global__ void __launch_bounds__(kThreads) k1_rb_thread(const __grid_constant__ NssDev P, const double *__restrict__ theta,
                                                         int64_t N, double *__restrict__ out)
{
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar;
  const double *rec = P.rb_rec;
  if (RESIDENT) {
    if (threadIdx.x == 0) {
      nssk::mbar_init(&bar, 1);
      nssk::stage_table(smem_raw, P.rb_rec, (uint32_t)((size_t)P.n_edges * P.rb_rs * sizeof(double)), &bar);
    }
    __syncthreads();
    nssk::mbar_wait(&bar, 0);
    rec = reinterpret_cast<const double *>(smem_raw);
  }
  const int d = P.d;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
    double th[NSS_NSLOT];
    nssk::canon_from_mem(P, theta + i * d, th);
    double l = -INFINITY;
    if (nssp::domain_ok(th)) {
      nssk::RbPoint<NDET> R;
      nssk::rb_point<NDET>(P, th, R);
      l = nssk::rb_loglike_thread<NDET>(P, rec, R);
    }
    out[i] = l;
  }
}

template <int NDET, bool RESIDENT>
__global__ void __launch_bounds__(kThreads) k1_rb_warp(const __grid_constant__ NssDev P, const double *__restrict__ theta,
                                                       int64_t N, double *__restrict__ out)
{
  extern __shared__ __align__(128) unsigned char smem_raw[];
  __shared__ __align__(8) uint64_t bar;
  const double *tab = P.rb_soa;
  if (RESIDENT) {
    if (threadIdx.x == 0) {
      nssk::mbar_init(&bar, 1);
      const size_t bytes = (size_t)(9 * (P.rb_m + 1) + 6 * NDET * P.rb_m) * 32 * sizeof(double);
      nssk::stage_table(smem_raw, P.rb_soa, (uint32_t)bytes, &bar);
    }
    __syncthreads();
    nssk::mbar_wait(&bar, 0);
    tab = reinterpret_cast<const double *>(smem_raw);
  }
  const int d = P.d, lane = threadIdx.x & 31;
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarp = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t i = warp0; i < N; i += nwarp) {
    const double l = nssk::loglike_warp<NDET, NSS_KIND_RB>(P, tab, theta + i * d);
    if (lane == 0) out[i] = l;
  }
}

template <int NDET>
__global__ void __launch_bounds__(kThreads) k2_full_warp(const __grid_constant__ NssDev P, const double *__restrict__ theta,
                                                         int64_t N, double *__restrict__ out)
{
  const int d = P.d, lane = threadIdx.x & 31;
  const int64_t warp0 = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int64_t nwarp = ((int64_t)gridDim.x * blockDim.x) >> 5;
  for (int64_t i = warp0; i < N; i += nwarp) {
    const double l = nssk::loglike_warp<NDET, NSS_KIND_FULL>(P, nullptr, theta + i * d);
    if (lane == 0) out[i] = l;
  }
}

__global__ void __launch_bounds__(kThreads) k_gauss(const __grid_constant__ NssDev P, const double *__restrict__ theta,
                                                    int64_t N, double *__restrict__ out)
{
  const int d = P.d;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < N; i += (int64_t)gridDim.x * blockDim.x) {
    out[i] = nssk::gauss_loglike(P, theta + i * d);
  }
}

template <class K>
int set_smem(K kernel, size_t bytes)
{
  if (bytes > 48 * 1024) NSS_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
  return NSS_OK;
}

template <int NDET>
int launch_rb(nss_handle *h, const double *theta, int64_t N, double *logL, cudaStream_t st)
{
  const NssDev &P = h->dev;
  int variant = h->loglike_variant;
  if (variant == 0) variant = N >= (int64_t)h->n_sm * 512 ? 1 : 2;
  if (variant == 1) {
    const size_t bytes = (size_t)P.n_edges * P.rb_rs * sizeof(double);
    const bool resident = bytes + 1024 <= kSmemMax;
    const size_t smem = resident ? bytes : 0;
    int per_sm = resident ? (int)(kSmemMax / (bytes + 1024)) : 4;
    per_sm = per_sm > 3 ? 3 : per_sm;
    int64_t want = (N + kThreads - 1) / kThreads;
    const int64_t cap = (int64_t)h->n_sm * per_sm;
    const int grid = (int)(want < cap ? want : cap);
    if (resident) {
      int rc = set_smem(k1_rb_thread<NDET, true>, smem);
      if (rc) return rc;
      k1_rb_thread<NDET, true><<<grid, kThreads, smem, st>>>(P, theta, N, logL);
    } else {
      k1_rb_thread<NDET, false><<<grid, kThreads, 0, st>>>(P, theta, N, logL);
    }
  } else {
    const size_t bytes = (size_t)(9 * (P.rb_m + 1) + 6 * NDET * P.rb_m) * 32 * sizeof(double);
    const bool resident = bytes + 1024 <= 200 * 1024;
    const size_t smem = resident ? bytes : 0;
    int per_sm = resident ? (int)(kSmemMax / (bytes + 1024)) : 8;
    per_sm = per_sm > 8 ? 8 : per_sm;
    int64_t want = (N * 32 + kThreads - 1) / kThreads;
    const int64_t cap = (int64_t)h->n_sm * per_sm;
    const int grid = (int)(want < cap ? want : cap);
    if (resident) {
      int rc = set_smem(k1_rb_warp<NDET, true>, smem);
      if (rc) return rc;
      k1_rb_warp<NDET, true><<<grid, kThreads, smem, st>>>(P, theta, N, logL);
    } else {
      k1_rb_warp<NDET, false><<<grid, kThreads, 0, st>>>(P, theta, N, logL);
    }
  }
  return NSS_OK;
}

template <int NDET>
int launch_full(nss_handle *h, const double *theta, int64_t N, double *logL, cudaStream_t st)
{
  int64_t want = (N * 32 + kThreads - 1) / kThreads;
  const int64_t cap = (int64_t)h->n_sm * 8;
  const int grid = (int)(want < cap ? want : cap);
  k2_full_warp<NDET><<<grid, kThreads, 0, st>>>(h->dev, theta, N, logL);
  return NSS_OK;
}

}  // namespace

int nss_launch_loglike(nss_handle *h, const double *theta, int64_t N, double *logL, cudaStream_t st)
{
  const NssDev &P = h->dev;
  int rc = NSS_OK;
  if (P.kind == NSS_KIND_GAUSS) {
    int64_t want = (N + kThreads - 1) / kThreads;
    const int64_t cap = (int64_t)h->n_sm * 8;
    k_gauss<<<(int)(want < cap ? want : cap), kThreads, 0, st>>>(P, theta, N, logL);
  } else if (P.kind == NSS_KIND_RB) {
    switch (P.n_det) {
      case 1: rc = launch_rb<1>(h, theta, N, logL, st); break;
      case 2: rc = launch_rb<2>(h, theta, N, logL, st); break;
      case 3: rc = launch_rb<3>(h, theta, N, logL, st); break;
      default: rc = launch_rb<4>(h, theta, N, logL, st); break;
    }
  } else {
    switch (P.n_det) {
      case 1: rc = launch_full<1>(h, theta, N, logL, st); break;
      case 2: rc = launch_full<2>(h, theta, N, logL, st); break;
      case 3: rc = launch_full<3>(h, theta, N, logL, st); break;
      default: rc = launch_full<4>(h, theta, N, logL, st); break;
    }
  }
  if (rc) return rc;
  h->launches += 1;
  NSS_CUDA(cudaGetLastError());
  return NSS_OK;
}

extern "C" int nss_loglike_batch(nss_handle *h, const double *theta_dev, int64_t N, double *logL_dev, void *cuda_stream)
{
  if (!h || N < 0) return NSS_EINVAL;
  if (N == 0) return NSS_OK;
  if (!theta_dev || !logL_dev) return NSS_EINVAL;
  NSS_CUDA(cudaSetDevice(h->device));
  return nss_launch_loglike(h, theta_dev, N, logL_dev, (cudaStream_t)cuda_stream);
}

// ---- fp64 FMA peak: register-resident DFMA chains on every SM -----------------------------------------
namespace {
__global__ void __launch_bounds__(256) k_dfma_peak(double *sink, int iters, double a, double b)
{
  double x0 = threadIdx.x * 1e-3, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  const double s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
  if (s == 123.456) sink[0] = s;
}
}  // namespace

extern "C" int nss_fp64_peak(double ms, double *tflops_host, void *cuda_stream)
{
  if (!tflops_host || !(ms > 0)) return NSS_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int dev = 0;
  NSS_CUDA(cudaGetDevice(&dev));
  cudaDeviceProp prop;
  NSS_CUDA(cudaGetDeviceProperties(&prop, dev));
  double *sink = nullptr;
  NSS_CUDA(cudaMalloc(&sink, sizeof(double)));
  cudaEvent_t e0, e1;
  NSS_CUDA(cudaEventCreate(&e0));
  NSS_CUDA(cudaEventCreate(&e1));
  const int grid = prop.multiProcessorCount * 8;
  int iters = 2000;
  float t = 0.f;
  double best = 0.0;
  for (int rep = 0; rep < 6; ++rep) {
    NSS_CUDA(cudaEventRecord(e0, st));
    k_dfma_peak<<<grid, 256, 0, st>>>(sink, iters, 0.999999, 1e-9);
    NSS_CUDA(cudaEventRecord(e1, st));
    NSS_CUDA(cudaEventSynchronize(e1));
    NSS_CUDA(cudaEventElapsedTime(&t, e0, e1));
    const double fma_count = (double)grid * 256.0 * (double)iters * 16.0 * 8.0;
    const double tf = 2.0 * fma_count / (t * 1e-3) / 1e12;
    if (rep > 0 && tf > best) best = tf;
    if (rep == 0 && t > 0.f) {                 // calibrate the iteration count to ~ms per launch
      double scale = ms / (double)t;
      if (scale > 50) scale = 50;
      iters = (int)(iters * scale) + 1;
    }
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
  *tflops_host = best;
  return NSS_OK;
}
