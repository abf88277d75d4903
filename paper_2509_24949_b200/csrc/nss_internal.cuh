// nss_internal.cuh — handle, device-side problem description and launch helpers (CUDA path only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/nss.h"
#include "nss_physics.cuh"

// Device-side problem description, passed to kernels by value (__grid_constant__).
struct NssDev {
  int32_t d, n_det, kind, n_bins, n_edges, n_freq;
  int32_t param_index[NSS_NSLOT];   // sampled dim j -> canonical slot
  int32_t slot_src[NSS_NSLOT];      // canonical slot t -> sampled dim, or -1 (fixed)
  double theta_fixed[NSS_NSLOT];
  double lo[NSS_NSLOT], hi[NSS_NSLOT];
  int32_t periodic[NSS_NSLOT];      // sampled dim j wraps in [lo_j, hi_j) in the slice sampler (nss_set_periodic)
  double gauss_mu[NSS_NSLOT], gauss_isig[NSS_NSLOT];
  double D6[NSS_MAXDET][6];   // symmetric detector tensors (O4)
  double rc[NSS_MAXDET][3];   // vertex / c [s]
  double gmst;
  // heterodyne reference (kind 0); for the full grid (kind 1) the reference is the identity:
  // c_fid = c_const_fid = tc_fid = tau_fid = 0, inv_a0 = (1, 0)
  double c_fid[nssp::kNB], c_const_fid, tc_fid;
  double inv_a0[NSS_MAXDET][2];   // 1 / (complex amplitude of the fiducial waveform per detector)
  double tau_fid[NSS_MAXDET];
  double half_DD;                 // 1/2 sum_det <d,d>
  double hh0[NSS_MAXDET];         // <h,h> = |A|^2 (hh0 + sum_b V_b X_b)   (nss_setup.cu: "record tables")
  // record tables (device pointers owned by the handle); a record is a bin edge (kind 0) or a grid frequency (kind 1)
  int32_t n_rec;
  int32_t cross;          // 1: records carry the cross-term weight V (kind 0), 0: they do not (kind 1)
  const double *rec;      // AoS [n_rec][rec_rs]: g0..g7, f, pad, then per det (Wr, Wi[, V])
  int32_t rec_rs;
  // sub-warp layouts for L = 8, 16, 32 lanes per point (index 0, 1, 2; NULL if not built), round major:
  // [9 + 2 n_det][L], then m x [9 + (2 + cross) n_det][L]; m = rounds after round 0 = ceil((n_rec - 1)/L);
  // lane l owns records l*m+1 .. l*m+m
  const double *soa[3];
  int32_t soa_m[3];
};

// device control block of an NS iteration; one pinned host mirror per handle (a single small D2H copy per sync)
struct NssCtl {
  double state[4];             // logX, logZ, logZ_live, Lstar
  unsigned long long nevals;
  unsigned long long nrounds, nexec;   // K3 diagnostics: rounds run by all chains, candidates evaluated (incl. speculative)
  int32_t flags[4];            // [0] Cholesky error, [1] threshold violation, [2] stop rule reached
  // work distribution inside an iteration (device only)
  uint32_t front_done;         // blocks of k4_front that have finished (the last one publishes the flags)
  uint32_t rank_done;          // ranking blocks of k4_front that have finished (the last one does the selection tail)
  int32_t sel_bad;             // a survivor below a supplied threshold (selection tail -> flags[1])
  uint32_t tune_cnt[3];        // counters of the tuning blocks of k4_front: column sums published, products published, circular sums published (R7)
  uint32_t chains_done;        // chains finished (the CTA that finishes the last one runs the live-evidence epilogue)
  uint32_t chain_next;         // next chain to start (K3 with single-warp groups: warps fetch chains as they finish)
  int32_t chol_now;            // Cholesky status of the tuning block of the iteration being set up
};

struct nss_handle {
  NssDev dev;
  int device;
  int n_sm;
  int loglike_variant;
  int chain_warps;          // warps per slice chain: 0 = automatic, else 1, 2, 4 or 8
  int chain_lanes;          // lanes per candidate in the slice kernel: 0 = automatic, else 8, 16 or 32
  int chain_pack;           // single-warp chains per CTA (they share the record table): 0 = automatic, else 1 .. 8
  int64_t launches;
  // host copies kept for nss_get_tables
  std::vector<int32_t> edge_idx;
  std::vector<double> summary;     // [n_det][B][6]
  double DD;
  // device allocations
  double *d_rec, *d_soa[3];
  size_t rec_bytes, soa_bytes[3];
  // sampler scratch (grown on demand)
  int32_t scratch_n;
  int32_t *d_surv_idx, *d_dead_idx, *d_rank, *d_rank_part, *d_flags;   // flags: [0] chol error, [1] threshold violation, [2] done
  double *d_mean, *d_chol, *d_tune_scratch, *d_state;                      // state: logX, logZ, logZ_live, Lstar
  unsigned long long *d_nevals;
  NssCtl *d_ctl, *h_ctl;       // d_state, d_nevals, d_flags point into d_ctl; h_ctl is pinned, two slots
  cudaEvent_t ev_ctl[2];       // nss_run: the copy into slot i has landed
  double *d_birth;
  int32_t *trace_dev;
  double *margin_dev;
  // device staging for the host-buffer entry points (grown on demand)
  unsigned char *d_stage;
  size_t stage_bytes;
  // device block and events of nss_run, kept between runs
  unsigned char *d_run;
  size_t run_bytes;
  unsigned char *h_run;        // pinned staging block of nss_run's results (the caller's arrays may be pageable)
  size_t h_run_bytes;
  cudaEvent_t ev_run[2];
  // CUDA events recorded around the most recent K3 (slice chains) launch: nss_last_chain_ms
  cudaEvent_t ev_k3[2];
  int ev_k3_valid;
  int chain_timing;            // record the event pair around K3 (nss_set_chain_timing); off by default
  // resident CTAs per SM of the K3 instantiation launched last with packed single-warp chains (occupancy query cached
  // per kernel, warps per CTA and dynamic shared memory: the latter depends on this handle's table)
  const void *occ_kern;
  int occ_W, occ_per_sm;
  size_t occ_smem;
};

extern thread_local char g_nss_cuda_err[256];
int nss_cuda_fail(cudaError_t e, const char *where);
#define NSS_CUDA(x)                                              \
  do {                                                           \
    cudaError_t e__ = (x);                                       \
    if (e__ != cudaSuccess) return nss_cuda_fail(e__, #x);       \
  } while (0)

// launchers implemented in nss_loglike.cu
int nss_launch_loglike(nss_handle *h, const double *theta, int64_t N, double *logL, cudaStream_t st);
// sampler entry points implemented in nss_sampler.cu use the device functions of nss_loglike_dev.cuh
