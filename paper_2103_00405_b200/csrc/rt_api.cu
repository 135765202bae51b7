// rt_api.cu -- host side of the C ABI declared in include/rt.h: validation, dependency-list
// construction, device store, launch planning.  Every step of the simulation itself runs in the
// kernels of rt_bundle.cuh / rt_thread.cuh; there is no CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <mutex>
#include <new>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/rt.h"
#include "rt_bundle.cuh"
#include "rt_fast.cuh"
#include "rt_thread.cuh"

using rt::u64;

#ifndef RT_BLOCK_SMEM
#define RT_BLOCK_SMEM 256
#endif
#ifndef RT_BLOCK_GLOBAL
#define RT_BLOCK_GLOBAL 512
#endif
#ifndef RT_BLOCK_FAST
#define RT_BLOCK_FAST 256
#endif
namespace {

// Threads per CTA of the bundle kernel (stream warps + 1 walker warp).  Measured on B200: with
// the state in shared memory the pass is issue-bound and every extra warp only lengthens the
// barriers and the block argmin (cfg4: 256 threads 4.47 us, 384: 4.49, 512: 4.70, 192: 5.35);
// with the state streamed from HBM more threads keep more bytes in flight (cfg5a: 512 threads
// 55.7 us, 384: 58.2, 256: 65.4).
constexpr int kBlockSmem = RT_BLOCK_SMEM;
constexpr int kBlockGlobal = RT_BLOCK_GLOBAL;
constexpr int kBlockFast = RT_BLOCK_FAST;                      // candidate-first kernel (rt_fast.cuh)
constexpr size_t kSmemStateBytesFast = 203 * 1024;             // (its static shared memory is larger)
constexpr int kThreadKernelMaxM = 64; // one-thread-per-trajectory path: M, N at most this
constexpr int kMinPairsPerCta = 256;  // do not spread a trajectory thinner than this
constexpr int kBigDeg = 64;           // species read by more reactions than this get a block-offset table
constexpr int kTargetBlocks = 256;    // ... with about this many reaction blocks
constexpr size_t kSmemStateBytes = 210 * 1024;   // dynamic shared memory the (T,P,a) state may take

#define CU_TRY(expr)                                                         \
  do {                                                                       \
    cudaError_t e_ = (expr);                                                 \
    if (e_ != cudaSuccess) {                                                 \
      if (getenv("RT_DEBUG"))                                                \
        fprintf(stderr, "rt: %s -> %s\n", #expr, cudaGetErrorString(e_));    \
      return e_ == cudaErrorMemoryAllocation ? RT_ERR_OOM : RT_ERR_CUDA;     \
    }                                                                        \
  } while (0)

struct DevBuf {
  void *p = nullptr;
  size_t bytes = 0;
  int ensure(size_t want) {
    if (want <= bytes) return RT_OK;
    if (p) cudaFree(p);
    p = nullptr;
    bytes = 0;
    cudaError_t e = cudaMalloc(&p, want);
    if (e != cudaSuccess) { p = nullptr; return e == cudaErrorMemoryAllocation ? RT_ERR_OOM : RT_ERR_CUDA; }
    bytes = want;
    return RT_OK;
  }
  void release() { if (p) cudaFree(p); p = nullptr; bytes = 0; }
};

}  // namespace

struct rt_model {
  int device = 0;
  int num_sms = 0;
  rt::NetDev net{};
  uint32_t nnz_r = 0, nnz_v = 0;
  int max_sigma = 1;
  // device copies of the network
  DevBuf d_react_ptr, d_react_species, d_react_sigma, d_stoich_ptr, d_stoich_species, d_stoich_v,
      d_rate, d_srow, d_sp_rec, d_sp_big, d_big_off, d_dep;
  // per-bundle state
  DevBuf d_T, d_P, d_a, d_n, d_X, d_exch, d_err;
  // rate schedule (time-dependent rates)
  DevBuf d_sched_t, d_sched_f, d_sched_mask, d_lambda;
  bool rate_exp = false;     // exponential rates c_k exp(lambda_k t) are set
  int sched_n = 0;
  bool sched_has_mask = false;
  // staging for the host-pointer API
  DevBuf d_x0, d_xout, d_res, d_trace_mu, d_trace_t, d_T0, d_P0, d_n0;
  // options
  int refresh_mode = 0, opt_bundle_ctas = 0, opt_ensemble_path = 0, opt_state_mode = 0, opt_x_replicas = 0, opt_prefetch = 7, opt_formulation = 0;
  int opt_exchange = 0, opt_pipeline = 1, opt_l2_persist = 1, opt_tiny = 1;
  rt::TinyNet tiny{};        // dense copy of a network small enough for rt_tiny_kernel
  bool tiny_ok = false;
  int last_tiny = 0;
  size_t l2_persist_max = 0, l2_window_max = 0;   // device limits for persisting L2 lines / window size
  bool l2_limit_set = false;
  int last_fast = 0;
  int max_clusters[rt::kMaxClusterCtas + 1] = {};   // co-resident clusters per cluster size (0 = not asked yet, -1 = none)
  int last_cluster = 0;
  // info
  int64_t kernel_launches = 0;
  int last_S = 0, last_B = 0, last_path = 0, last_state_smem = 0, last_block = 0;
  size_t n_big = 0;
  unsigned char *noalloc_scratch = nullptr;   // device address of the static scratch array (rt_noalloc_prepare)
};

namespace {

int validate(const rt_network *net, int *max_sigma_out) {
  if (!net) return RT_ERR_NULL;
  if (!net->react_ptr || !net->stoich_ptr || !net->rate) return RT_ERR_NULL;
  const int64_t N = net->n_species, M = net->n_reactions;
  if (N < 1 || M < 1) return RT_ERR_BAD_NETWORK;
  if (net->react_ptr[0] != 0 || net->stoich_ptr[0] != 0) return RT_ERR_BAD_NETWORK;
  for (int64_t k = 0; k < M; ++k)
    if (net->react_ptr[k + 1] < net->react_ptr[k] || net->stoich_ptr[k + 1] < net->stoich_ptr[k])
      return RT_ERR_BAD_NETWORK;
  const int64_t nr = net->react_ptr[M], nv = net->stoich_ptr[M];
  if ((nr > 0 && (!net->react_species || !net->react_sigma)) ||
      (nv > 0 && (!net->stoich_species || !net->stoich_v)))
    return RT_ERR_NULL;
  if (nr >= (int64_t)0xffffffffll || nv >= (int64_t)0xffffffffll) return RT_ERR_UNSUPPORTED;
  int max_sigma = 1;
  bool unsupported = false;
  std::vector<int32_t> row;
  for (int64_t k = 0; k < M; ++k) {
    if (!std::isfinite(net->rate[k]) || net->rate[k] < 0.0) return RT_ERR_BAD_NETWORK;
    const int64_t rb = net->react_ptr[k], re = net->react_ptr[k + 1];
    for (int64_t e = rb; e < re; ++e) {
      const int32_t j = net->react_species[e], s = net->react_sigma[e];
      if (j < 0 || j >= N || s < 1) return RT_ERR_BAD_NETWORK;
      if (s > 3) unsupported = true;
      max_sigma = std::max(max_sigma, (int)std::min(s, 4));
      for (int64_t f = rb; f < e; ++f)
        if (net->react_species[f] == j) return RT_ERR_BAD_NETWORK;     // G18: A+A must be sigma=2
    }
    const int64_t sb = net->stoich_ptr[k], se = net->stoich_ptr[k + 1];
    for (int64_t e = sb; e < se; ++e) {
      const int32_t j = net->stoich_species[e], v = net->stoich_v[e];
      if (j < 0 || j >= N || v == 0) return RT_ERR_BAD_NETWORK;
      for (int64_t f = sb; f < e; ++f)
        if (net->stoich_species[f] == j) return RT_ERR_BAD_NETWORK;
      if (v < 0) {   // may not remove more than the reaction requires
        int32_t sigma = 0;
        for (int64_t f = rb; f < re; ++f)
          if (net->react_species[f] == j) sigma = net->react_sigma[f];
        if ((int64_t)v < -(int64_t)sigma) return RT_ERR_BAD_NETWORK;
      }
    }
  }
  if (unsupported) return RT_ERR_UNSUPPORTED;
  if (max_sigma_out) *max_sigma_out = max_sigma;
  return RT_OK;
}

template <typename T>
int upload(DevBuf &buf, const std::vector<T> &host) {
  const size_t bytes = std::max<size_t>(host.size() * sizeof(T), 16);
  int rc = buf.ensure(bytes);
  if (rc != RT_OK) return rc;
  if (!host.empty()) CU_TRY(cudaMemcpy(buf.p, host.data(), host.size() * sizeof(T), cudaMemcpyHostToDevice));
  return RT_OK;
}

// Checkpoint a single trajectory resumes from (device pointers); all null = fresh start.
struct StartDev {
  double t0 = 0.0;
  const double *T0 = nullptr, *P0 = nullptr;
  const uint32_t *n0 = nullptr;
};

// How one launch is shaped: B bundles of S CTAs; smem = the (T,P,a) state lives in shared memory.
// cluster = each bundle is one thread-block cluster and exchanges through distributed shared memory.
// fast = the candidate-first kernel of rt_fast.cuh (on-chip state, dependency refresh, constant rates).
struct Plan { int S, B, G; int pairs_per_cta; int cnt_pad; bool smem; bool cluster; bool fast; };

// stream threads of the kernel that keeps the state in shared memory
int stream_threads(bool fast) {
  return fast ? kBlockFast - 32 * rt::kFastHelperWarps : kBlockSmem - 32 * rt::kWalkerWarps;
}
size_t smem_budget(bool fast) { return fast ? kSmemStateBytesFast : kSmemStateBytes; }
// slots per shared-memory state array: a CTA's reactions padded to whole scan batches
int padded_count(int pairs_per_cta, bool fast) {
  const int batch = rt::kScanBatch * stream_threads(fast);
  return (2 * pairs_per_cta + batch - 1) / batch * batch;
}
size_t smem_state_bytes(int pairs_per_cta, bool fast) {
  size_t slots = (size_t)padded_count(pairs_per_cta, fast);
  if (fast) slots = slots / stream_threads(true) * (stream_threads(true) + 1);   // padded rows (rt_fast.cuh sidx)
  return slots * 3 * sizeof(double);
}

// The bundle kernel for a launch shape (FULL = refresh_mode 1; rate: 0 constant, 1 schedule, 2 exponential).
const void *bundle_kernel(bool smem, bool full, int rate, bool cluster, bool fast = false) {
  using namespace rt;
  if (fast) return cluster ? (const void *)rt_fast_kernel<kBlockFast, true> : (const void *)rt_fast_kernel<kBlockFast, false>;
  if (smem && cluster)
    return full        ? (const void *)rt_bundle_kernel<kBlockSmem, true, true, 0, true>
           : rate == 1 ? (const void *)rt_bundle_kernel<kBlockSmem, true, false, 1, true>
           : rate == 2 ? (const void *)rt_bundle_kernel<kBlockSmem, true, false, 2, true>
                       : (const void *)rt_bundle_kernel<kBlockSmem, true, false, 0, true>;
  if (smem)
    return full        ? (const void *)rt_bundle_kernel<kBlockSmem, true, true, 0>
           : rate == 1 ? (const void *)rt_bundle_kernel<kBlockSmem, true, false, 1>
           : rate == 2 ? (const void *)rt_bundle_kernel<kBlockSmem, true, false, 2>
                       : (const void *)rt_bundle_kernel<kBlockSmem, true, false, 0>;
  return full        ? (const void *)rt_bundle_kernel<kBlockGlobal, false, true, 0>
         : rate == 1 ? (const void *)rt_bundle_kernel<kBlockGlobal, false, false, 1>
         : rate == 2 ? (const void *)rt_bundle_kernel<kBlockGlobal, false, false, 2>
                     : (const void *)rt_bundle_kernel<kBlockGlobal, false, false, 0>;
}

// Clusters of S CTAs (one per SM: the state fills shared memory) that can be co-resident; the GPC
// structure decides (B200: 74 of 2, 33 of 4, 15 of 8, 7 of 16).  Asked once per size.
int max_active_clusters(rt_model *m, int S) {
  if (S < 2 || S > rt::kMaxClusterCtas) return 0;
  if (m->max_clusters[S] == 0) {
    const void *kern = bundle_kernel(true, false, 0, true);     // (the same count holds for rt_fast_kernel:
    int n = 0;                                                   //  one CTA per SM either way)
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(S); cfg.blockDim = dim3(kBlockSmem); cfg.dynamicSmemBytes = kSmemStateBytes;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = S; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemStateBytes) != cudaSuccess ||
        cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) != cudaSuccess ||
        cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess) {
      cudaGetLastError();
      n = 0;
    }
    m->max_clusters[S] = n > 0 ? n : -1;
  }
  return std::max(m->max_clusters[S], 0);
}

Plan plan_bundles_for(rt_model *m, u64 n_traj, bool fast);

Plan plan_bundles(rt_model *m, u64 n_traj) {
  // the candidate-first kernel covers the default configuration: on-chip state, dependency refresh,
  // constant rates, one copy of X
  const bool fast = m->opt_pipeline != 0 && m->refresh_mode == 0 && m->sched_n == 0 && !m->rate_exp &&
                    m->opt_x_replicas <= 1 && m->opt_state_mode != 1;
  Plan pl = plan_bundles_for(m, n_traj, fast);
  // (its static shared memory is larger: at the capacity edge only the plain kernel still fits)
  if (fast && !pl.smem) pl = plan_bundles_for(m, n_traj, false);
  return pl;
}

Plan plan_bundles_for(rt_model *m, u64 n_traj, bool fast) {
  const int pairs_total = m->net.M_pad / 2;
  const int sms = m->num_sms;
  // fewest CTAs whose share of the state still fits in shared memory
  const int batch = rt::kScanBatch * stream_threads(fast);
  const int pairs_fit = std::max(1, (int)((smem_budget(fast) - (fast ? 64 * 3 * sizeof(double) : 0)) /
                                          (3 * sizeof(double)) / batch * batch / 2));
  const int s_fit = (pairs_total + pairs_fit - 1) / pairs_fit;
  const int s_thin = std::max(1, (pairs_total + kMinPairsPerCta - 1) / kMinPairsPerCta);
  const bool may_cluster = m->opt_exchange != 1 && m->opt_state_mode != 1;
  int S, B = 0;
  bool cluster = false, force_l2 = false;
  if (m->opt_bundle_ctas > 0) {
    S = std::min(m->opt_bundle_ctas, sms);
  } else if (n_traj <= 1) {
    S = std::min(sms, s_thin);                          // one trajectory: the whole chip ...
    // ... unless ONE cluster holds the state: its exchange through distributed shared memory costs
    // ~0.25 us instead of ~1.2 us through L2 (profiles/r2_exchange_floor.md), which outweighs the
    // longer pass of fewer, fuller CTAs.
    const int sc = std::min(rt::kMaxClusterCtas, s_thin);
    if (may_cluster && sc >= 2 && sc >= s_fit && max_active_clusters(m, sc) >= 1) S = sc;
    // Through L2 every lane of the exchange warp polls ceil(S / 32) slots: with the pass hidden behind
    // the exchange (candidate-first kernel) 128 CTAs with 4 slots per lane beat 148 with 5 (cfg4: 3.16
    // against 3.23 us per firing; 119..128 alike, 129 already slower), if the state still fits.
    else if (fast && m->opt_state_mode != 1 && S == sms && S % 32 != 0 && S / 32 * 32 >= s_fit) S = S / 32 * 32;
  } else {
    S = (int)std::max<u64>(1, (u64)sms / n_traj);       // many: as many bundles as fit ...
    if (m->opt_state_mode != 1 && S < s_fit && s_fit <= sms) S = s_fit;   // ... with on-chip state
    S = std::min(S, s_thin);
    if (m->opt_state_mode != 1 && S >= s_fit && S >= 2) {
      // Ensemble throughput = trajectories in flight / time per firing.  Model (measured on B200 with
      // the candidate-first kernel, profiles/r2_fast_kernel.md): a firing costs ~1.9 us of latency
      // chain + 0.13 us per 1000 reactions of a CTA, + 1.0 us when the exchange crosses L2.  Clusters
      // exchange faster but tile the chip worse (7 clusters of 16 = 112 SMs, against 12 L2 bundles of
      // 12 = 144 SMs): cfg5b runs 3.1e6 trajectory-steps/s as 12 x 12 through L2, 2.3e6 as 7 x 16.
      // In flight = n_traj / rounds, rounds = ceil(n_traj / bundles).
      double best = 0.0;
      int best_S = S;
      bool best_cluster = false;
      const int s_hi = std::min(std::min(s_thin, sms), std::max(S, 2 * rt::kMaxClusterCtas));
      for (int c = std::max(2, s_fit); c <= s_hi; ++c) {
        const double t_cta = 1.9 + 0.13 * (2.0 * pairs_total / c / 1000.0);
        for (int cl = 0; cl < 2; ++cl) {
          if (cl && (!may_cluster || c > rt::kMaxClusterCtas)) continue;
          const u64 bundles = cl ? (u64)max_active_clusters(m, c) : (u64)(sms / c);
          if (bundles == 0) continue;
          const u64 bb = std::min<u64>(n_traj, bundles);
          const double in_flight = (double)n_traj / (double)((n_traj + bb - 1) / bb);
          const double thr = in_flight / (t_cta + (cl ? 0.0 : 1.0));
          if (thr > best) { best = thr; best_S = c; best_cluster = cl != 0; }
        }
      }
      S = best_S;
      force_l2 = !best_cluster;
    }
  }
  S = std::max(std::min(S, rt::kMaxBundleCtas), 1);
  Plan pl;
  pl.S = S;
  pl.pairs_per_cta = (pairs_total + S - 1) / S;
  pl.smem = m->opt_state_mode != 1 && smem_state_bytes(pl.pairs_per_cta, fast) <= smem_budget(fast);
  pl.fast = fast && pl.smem;
  pl.cnt_pad = padded_count(pl.pairs_per_cta, pl.fast);
  if (may_cluster && !force_l2 && pl.smem && S >= 2 && S <= rt::kMaxClusterCtas) {
    B = (int)std::min<u64>(std::max<u64>(n_traj, 1), (u64)max_active_clusters(m, S));
    cluster = B >= 1;
  }
  pl.cluster = cluster;
  pl.B = cluster ? B : (int)std::min<u64>(std::max<u64>(n_traj, 1), (u64)(sms / S));
  pl.G = std::min(S, m->opt_x_replicas > 0 ? m->opt_x_replicas : 1);      // X replicas: spread the per-firing reads/atomics of hot species
  while (pl.G > 1 && (size_t)pl.B * pl.G * (size_t)m->net.N * 8 > ((size_t)64 << 20)) pl.G /= 2;
  return pl;
}

int ensure_state(rt_model *m, const Plan &pl) {
  const size_t Mp = (size_t)m->net.M_pad, N = (size_t)m->net.N, B = (size_t)pl.B;
  int rc;
  if ((rc = m->d_T.ensure(B * Mp * 8)) != RT_OK) return rc;
  if ((rc = m->d_P.ensure(B * Mp * 8)) != RT_OK) return rc;
  if ((rc = m->d_a.ensure(B * Mp * 8)) != RT_OK) return rc;
  if ((rc = m->d_n.ensure(B * Mp * 4)) != RT_OK) return rc;
  if ((rc = m->d_X.ensure(B * (size_t)pl.G * N * 8)) != RT_OK) return rc;
  if ((rc = m->d_exch.ensure(B * 2 * (size_t)pl.S * rt::kSlotStride * 8)) != RT_OK) return rc;
  if ((rc = m->d_err.ensure(16)) != RT_OK) return rc;
  return RT_OK;
}

int launch_bundles(rt_model *m, const long long *x0_dev, u64 seed, u64 traj_first, u64 n_traj,
                   u64 max_firings, double t_end, long long *x_out_dev, rt_result *res_dev,
                   int32_t *trace_mu_dev, double *trace_t_dev, u64 trace_cap, cudaStream_t st,
                   const StartDev &start = StartDev()) {
  const Plan pl = plan_bundles(m, n_traj);
  int rc = ensure_state(m, pl);
  if (rc != RT_OK) return rc;
  CU_TRY(cudaMemsetAsync(m->d_exch.p, 0, (size_t)pl.B * 2 * pl.S * rt::kSlotStride * 8, st));
  rt::BundleParams p{};
  p.net = m->net;
  p.T = (double *)m->d_T.p; p.P = (double *)m->d_P.p; p.a = (double *)m->d_a.p;
  p.n = (uint32_t *)m->d_n.p; p.X = (u64 *)m->d_X.p;
  p.exch = (u64 *)m->d_exch.p;
  p.S = pl.S; p.B = pl.B; p.G = pl.G; p.pairs_per_cta = pl.pairs_per_cta; p.cnt_pad = pl.cnt_pad;
  p.x0 = x0_dev; p.seed = seed; p.traj_first = traj_first; p.n_traj = n_traj;
  p.max_firings = max_firings; p.t_end = t_end;
  p.T0 = start.T0; p.P0 = start.P0; p.n0 = start.n0; p.t0 = start.t0;
  p.x_out = x_out_dev; p.res = res_dev;
  p.trace_mu = trace_mu_dev; p.trace_t = trace_t_dev;
  p.trace_cap = (trace_mu_dev || trace_t_dev) ? trace_cap : 0;
  p.refresh_mode = m->refresh_mode;
  p.prefetch = m->opt_prefetch;
  p.formulation = m->opt_formulation;
  if (m->sched_n > 0 && (m->refresh_mode != 0 || m->opt_formulation != 0 || start.T0)) return RT_ERR_UNSUPPORTED;
  if (m->rate_exp && (m->refresh_mode != 0 || m->opt_formulation != 0 || m->sched_n > 0)) return RT_ERR_UNSUPPORTED;
  p.rate_lambda = (const double *)m->d_lambda.p;
  p.sched_n = m->sched_n;
  p.sched_t = (const double *)m->d_sched_t.p;
  p.sched_f = (const double *)m->d_sched_f.p;
  p.sched_mask = m->sched_has_mask ? (const unsigned char *)m->d_sched_mask.p : nullptr;
  p.err = (int *)m->d_err.p;
  void *args[] = {&p};
  const int rate = m->sched_n > 0 ? 1 : m->rate_exp ? 2 : 0;   // (never with refresh_mode 1: checked above)
  const void *kern = bundle_kernel(pl.smem, m->refresh_mode != 0, rate, pl.cluster, pl.fast);
  const size_t dyn = pl.smem ? smem_state_bytes(pl.pairs_per_cta, pl.fast) : 0;
  if (dyn) CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
  const int block = pl.fast ? kBlockFast : pl.smem ? kBlockSmem : kBlockGlobal;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(pl.S * pl.B); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = dyn; cfg.stream = st;
  cudaLaunchAttribute at[2];
  if (pl.cluster) {
    // One cluster per bundle: the hardware co-schedules its CTAs, and bundles never wait for one
    // another, so no cooperative launch is needed.
    if (pl.S > 8) CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = pl.S; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  } else {
    // Cooperative launch: the CTAs of a bundle spin on one another, so all must be co-resident.
    at[0].id = cudaLaunchAttributeCooperative;
    at[0].val.cooperative = 1;
  }
  cfg.attrs = at; cfg.numAttrs = 1;
  if (m->l2_limit_set && (pl.smem || !m->opt_l2_persist)) {   // (give the set-aside part of L2 back to everybody;
                                                               //  lines made persisting earlier would stay so)
    cudaCtxResetPersistingL2Cache();
    cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, 0);
    cudaGetLastError();
    m->l2_limit_set = false;
  }
  if (!pl.smem && m->opt_l2_persist && m->l2_persist_max > 0 && m->l2_window_max > 0) {
    // State streamed from HBM (cfg5a): T is read AND written every firing, 16 of the 32 bytes per
    // reaction.  Keep as much of it as the device allows as persisting lines in the 126 MB L2
    // (access-policy window on this launch only); P, a and the rest of T stream past it.
    if (!m->l2_limit_set) {
      cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, m->l2_persist_max);
      cudaGetLastError();
      m->l2_limit_set = true;
    }
    const size_t bytes = std::min((size_t)pl.B * (size_t)m->net.M_pad * sizeof(double), m->l2_window_max);
    void *base = m->opt_l2_persist == 2 ? m->d_a.p : m->d_T.p;      // (2: keep a instead, for comparison)
    at[1].id = cudaLaunchAttributeAccessPolicyWindow;
    at[1].val.accessPolicyWindow.base_ptr = base;
    at[1].val.accessPolicyWindow.num_bytes = bytes;
    // (measured on cfg5a: 55.0 us per firing without the window, 42.1 us with every line of T
    // persisting; a partial window is worse than none -- 58 us at half the set-aside)
    at[1].val.accessPolicyWindow.hitRatio = (float)std::min(1.0, (double)m->l2_persist_max / (double)bytes);
    at[1].val.accessPolicyWindow.hitProp = cudaAccessPropertyPersisting;
    at[1].val.accessPolicyWindow.missProp = cudaAccessPropertyStreaming;
    cfg.numAttrs = 2;
  }
  CU_TRY(cudaLaunchKernelExC(&cfg, kern, args));
  m->last_block = block;
  m->kernel_launches += 1;
  m->last_S = pl.S; m->last_B = pl.B; m->last_path = 2; m->last_state_smem = pl.smem ? 1 : 0;
  m->last_cluster = pl.cluster ? 1 : 0;
  m->last_fast = pl.fast ? 1 : 0;
  return RT_OK;
}

template <int BLOCK>
int launch_thread_kernel(rt_model *m, const rt::ThreadParams &p, size_t smem, cudaStream_t st) {
  CU_TRY(cudaFuncSetAttribute(rt::rt_thread_kernel<BLOCK>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)smem));
  const unsigned grid = (unsigned)((p.n_traj + BLOCK - 1) / BLOCK);
  rt::rt_thread_kernel<BLOCK><<<grid, BLOCK, smem, st>>>(p);
  CU_TRY(cudaGetLastError());
  m->kernel_launches += 1;
  m->last_path = 1;
  return RT_OK;
}

bool thread_path_fits(const rt_model *m) {
  return m->net.M <= kThreadKernelMaxM && m->net.N <= kThreadKernelMaxM &&
         rt::thread_kernel_smem(m->net.M, m->net.N, m->nnz_r, m->nnz_v, 32) <= 200 * 1024;
}

int launch_threads(rt_model *m, const long long *x0_dev, u64 seed, u64 traj_first, u64 n_traj,
                   u64 max_firings, double t_end, long long *x_out_dev, rt_result *res_dev,
                   cudaStream_t st, const StartDev &start = StartDev(), double *T_out = nullptr,
                   double *P_out = nullptr, uint32_t *n_out = nullptr) {
  rt::ThreadParams p{};
  p.T0 = start.T0; p.P0 = start.P0; p.n0 = start.n0; p.t0 = start.t0;
  p.T_out = T_out; p.P_out = P_out; p.n_out = n_out;
  p.net = m->net; p.nnz_r = m->nnz_r; p.nnz_v = m->nnz_v;
  p.x0 = x0_dev; p.seed = seed; p.traj_first = traj_first; p.n_traj = n_traj;
  p.max_firings = max_firings; p.t_end = t_end; p.x_out = x_out_dev; p.res = res_dev;
  m->last_tiny = 0;
  if (m->tiny_ok && m->opt_tiny) {
    rt::TinyParams q{};
    q.net = m->tiny; q.net.xmax = m->net.xmax;
    q.x0 = x0_dev; q.seed = seed; q.traj_first = traj_first; q.n_traj = n_traj;
    q.max_firings = max_firings; q.t_end = t_end; q.x_out = x_out_dev; q.res = res_dev;
    q.T0 = start.T0; q.P0 = start.P0; q.n0 = start.n0; q.t0 = start.t0;
    q.T_out = T_out; q.P_out = P_out; q.n_out = n_out;
    if (n_traj >= (u64)m->num_sms * 2048)
      rt::rt_tiny_kernel<128><<<(unsigned)((n_traj + 127) / 128), 128, 0, st>>>(q);
    else
      rt::rt_tiny_kernel<32><<<(unsigned)((n_traj + 31) / 32), 32, 0, st>>>(q);
    CU_TRY(cudaGetLastError());
    m->kernel_launches += 1;
    m->last_path = 1;
    m->last_tiny = 1;
    return RT_OK;
  }
  // Smallest CTA that still fills the chip: more CTAs -> finer balance over the 148 SMs.
  const size_t s32 = rt::thread_kernel_smem(m->net.M, m->net.N, m->nnz_r, m->nnz_v, 32);
  const size_t s128 = rt::thread_kernel_smem(m->net.M, m->net.N, m->nnz_r, m->nnz_v, 128);
  if (n_traj >= (u64)m->num_sms * 2048 && s128 <= 48 * 1024)
    return launch_thread_kernel<128>(m, p, s128, st);
  return launch_thread_kernel<32>(m, p, s32, st);
}

int check_limits(u64 max_firings, double t_end) {
  if (std::isnan(t_end) || t_end < 0.0) return RT_ERR_BAD_ARG;
  if (max_firings == 0 && std::isinf(t_end)) return RT_ERR_BAD_ARG;
  return RT_OK;
}

int check_x0(const rt_model *m, const int64_t *x0) {
  for (int32_t j = 0; j < m->net.N; ++j)
    if (x0[j] < 0 || x0[j] > m->net.xmax) return RT_ERR_BAD_ARG;
  return RT_OK;
}

int finish(rt_model *m, cudaStream_t st) {
  CU_TRY(cudaStreamSynchronize(st));
  if (m->d_err.p) {
    int err = 0;
    CU_TRY(cudaMemcpy(&err, m->d_err.p, sizeof(int), cudaMemcpyDeviceToHost));
    if (err) { cudaMemset(m->d_err.p, 0, sizeof(int)); return RT_ERR_CUDA; }
  }
  return RT_OK;
}

}  // namespace

extern "C" {

int rt_validate_network(const rt_network *net) { return validate(net, nullptr); }

int rt_create(const rt_network *net, int device, rt_model **out) {
  if (!out) return RT_ERR_NULL;
  *out = nullptr;
  int max_sigma = 1;
  int rc = validate(net, &max_sigma);
  if (rc != RT_OK) return rc;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0 || device < 0 || device >= ndev) {
    cudaGetLastError();
    return RT_ERR_CUDA;
  }
  CU_TRY(cudaSetDevice(device));
  rt_model *m = new (std::nothrow) rt_model();
  if (!m) return RT_ERR_OOM;
  m->device = device;
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) { delete m; return RT_ERR_CUDA; }
  m->num_sms = prop.multiProcessorCount;
  if (!prop.cooperativeLaunch) { delete m; return RT_ERR_CUDA; }
  m->l2_persist_max = (size_t)prop.persistingL2CacheMaxSize;
  m->l2_window_max = (size_t)prop.accessPolicyMaxWindowSize;

  const int32_t N = net->n_species, M = net->n_reactions;
  const size_t nr = (size_t)net->react_ptr[M], nv = (size_t)net->stoich_ptr[M];
  std::vector<uint32_t> rp(M + 1), sp(M + 1);
  for (int32_t k = 0; k <= M; ++k) { rp[k] = (uint32_t)net->react_ptr[k]; sp[k] = (uint32_t)net->stoich_ptr[k]; }
  std::vector<int32_t> rs(net->react_species, net->react_species + nr),
      rg(net->react_sigma, net->react_sigma + nr), ss(net->stoich_species, net->stoich_species + nv),
      sv(net->stoich_v, net->stoich_v + nv);
  std::vector<double> rate(net->rate, net->rate + M);
  for (double &c : rate) c += 0.0;     // -0.0 -> +0.0: a_k is then never -0.0 (same results: a_k = 0 either way)
  // ---- the smallest networks also get a dense by-value table for the register-resident kernel
  if (M <= rt::kTinyM && N <= rt::kTinyN) {
    bool ok = true;
    rt::TinyNet &tn = m->tiny;
    tn.M = M; tn.N = N;
    for (int k = 0; k < rt::kTinyM; ++k) {
      tn.rate[k] = k < M ? rate[k] : 0.0;
      for (int e = 0; e < 2; ++e) { tn.r_j[k][e] = -1; tn.r_s[k][e] = 1; }
      for (int j = 0; j < rt::kTinyN; ++j) tn.v[k][j] = 0;
      if (k >= M) continue;
      if (rp[k + 1] - rp[k] > 2) { ok = false; break; }
      for (uint32_t e = rp[k]; e < rp[k + 1]; ++e) { tn.r_j[k][e - rp[k]] = rs[e]; tn.r_s[k][e - rp[k]] = rg[e]; }
      for (uint32_t e = sp[k]; e < sp[k + 1]; ++e) tn.v[k][ss[e]] = sv[e];
    }
    m->tiny_ok = ok;
  }
  // ---- dependency graph, two-hop: stoich row of mu -> species -> reactions that
  // have the species as a reactant.  Entries of one species ascend in k (counting sort over the
  // reactant CSR, which is ordered by reaction) and carry what a refresh needs.
  std::vector<uint32_t> dp((size_t)N + 1, 0u);
  for (size_t e = 0; e < nr; ++e) dp[(size_t)rs[e] + 1] += 1u;
  for (int32_t j = 0; j < N; ++j) dp[j + 1] += dp[j];
  std::vector<int32_t> dep(8 * std::max<size_t>(nr, 1), 0);      // 32-byte entries
  {
    std::vector<uint32_t> cursor(dp.begin(), dp.end() - 1);
    for (int32_t k = 0; k < M; ++k) {
      const uint32_t rb = rp[k], re = rp[k + 1];
      const bool has = rb < re;                  // (rs / rg are empty when no reaction has reactants)
      const int32_t j1 = has ? rs[rb] : -1, s1 = has ? rg[rb] : 0;
      const int32_t j2 = (re - rb >= 2) ? rs[rb + 1] : -1, s2 = (re - rb >= 2) ? rg[rb + 1] : 0;
      const int32_t flags = s1 | (s2 << 8) | ((re - rb > 2) ? 0x10000 : 0);
      for (uint32_t e = rb; e < re; ++e) {
        const size_t at = 8 * (size_t)cursor[rs[e]]++;
        dep[at] = k; dep[at + 1] = j1; dep[at + 2] = j2; dep[at + 3] = flags;
        memcpy(&dep[at + 4], &rate[k], sizeof(double));
      }
    }
  }
  std::vector<uint32_t> sp_rec(2 * (size_t)N);
  std::vector<int32_t> sp_big((size_t)N, -1);
  int blk_shift = 0;
  while (((int64_t)M >> blk_shift) > kTargetBlocks) ++blk_shift;
  const int n_blk = (int)(((int64_t)M + (1ll << blk_shift) - 1) >> blk_shift) + 1;   // + the odd pad
  size_t n_big = 0;
  for (int32_t j = 0; j < N; ++j) {
    sp_rec[2 * (size_t)j] = dp[j];
    sp_rec[2 * (size_t)j + 1] = dp[j + 1];
    if (dp[j + 1] - dp[j] > (uint32_t)kBigDeg) sp_big[j] = (int32_t)n_big++;
  }
  std::vector<uint32_t> big_off(std::max<size_t>(n_big * (size_t)(n_blk + 1), 1), 0u);
  for (int32_t j = 0; j < N; ++j) {
    if (sp_big[j] < 0) continue;
    uint32_t *off = big_off.data() + (size_t)sp_big[j] * (size_t)(n_blk + 1);
    uint32_t i = dp[j];
    for (int bq = 0; bq <= n_blk; ++bq) {      // off[bq] = first entry with k >= bq << blk_shift
      const int64_t kmin = (int64_t)bq << blk_shift;
      while (i < dp[j + 1] && (int64_t)dep[8 * (size_t)i] < kmin) ++i;
      off[bq] = i;
    }
  }
  // ELL copy of the stoich rows: up to 4 x (j, v, lo, hi), 64 bytes per reaction
  std::vector<int32_t> srow(16 * (size_t)M);
  for (int32_t k = 0; k < M; ++k) {
    int32_t *row = srow.data() + 16 * (size_t)k;
    for (int e = 0; e < 4; ++e) { row[4 * e] = -1; row[4 * e + 1] = 0; row[4 * e + 2] = 0; row[4 * e + 3] = 0; }
    const uint32_t sb = sp[k], se = sp[k + 1];
    if (se - sb > 4) { row[0] = -2; continue; }
    for (uint32_t e = sb; e < se; ++e) {
      const int32_t j = ss[e];
      int32_t *q = row + 4 * (e - sb);
      q[0] = j; q[1] = sv[e];
      if (sp_big[j] >= 0) { q[2] = sp_big[j]; q[3] = (int32_t)0xffffffffu; }
      else { q[2] = (int32_t)dp[j]; q[3] = (int32_t)dp[j + 1]; }
    }
  }
  rc = RT_OK;
  if (rc == RT_OK) rc = upload(m->d_react_ptr, rp);
  if (rc == RT_OK) rc = upload(m->d_react_species, rs);
  if (rc == RT_OK) rc = upload(m->d_react_sigma, rg);
  if (rc == RT_OK) rc = upload(m->d_stoich_ptr, sp);
  if (rc == RT_OK) rc = upload(m->d_stoich_species, ss);
  if (rc == RT_OK) rc = upload(m->d_stoich_v, sv);
  if (rc == RT_OK) rc = upload(m->d_rate, rate);
  if (rc == RT_OK) rc = upload(m->d_srow, srow);
  if (rc == RT_OK) rc = upload(m->d_sp_rec, sp_rec);
  if (rc == RT_OK) rc = upload(m->d_sp_big, sp_big);
  if (rc == RT_OK) rc = upload(m->d_big_off, big_off);
  if (rc == RT_OK) rc = upload(m->d_dep, dep);
  if (rc == RT_OK) rc = m->d_err.ensure(16);
  if (rc == RT_OK && cudaMemset(m->d_err.p, 0, 16) != cudaSuccess) rc = RT_ERR_CUDA;
  if (rc != RT_OK) { rt_destroy(m); return rc; }

  m->nnz_r = (uint32_t)nr; m->nnz_v = (uint32_t)nv; m->max_sigma = max_sigma;
  rt::NetDev &d = m->net;
  d.N = N; d.M = M; d.M_pad = (M + 1) & ~1;
  d.react_ptr = (const uint32_t *)m->d_react_ptr.p;
  d.react_species = (const int32_t *)m->d_react_species.p;
  d.react_sigma = (const int32_t *)m->d_react_sigma.p;
  d.stoich_ptr = (const uint32_t *)m->d_stoich_ptr.p;
  d.stoich_species = (const int32_t *)m->d_stoich_species.p;
  d.stoich_v = (const int32_t *)m->d_stoich_v.p;
  d.rate = (const double *)m->d_rate.p;
  d.srow = (const int32_t *)m->d_srow.p;
  d.sp_rec = (const uint32_t *)m->d_sp_rec.p;
  d.sp_big = (const int32_t *)m->d_sp_big.p;
  d.big_off = (const uint32_t *)m->d_big_off.p;
  d.dep = (const int32_t *)m->d_dep.p;
  d.n_blk = n_blk; d.blk_shift = blk_shift; d.big_deg = kBigDeg;
  m->n_big = n_big;
  d.xmax = max_sigma <= 2 ? ((1ll << 31) - 1) : ((1ll << 21) - 1);
  *out = m;
  return RT_OK;
}

int rt_run_dev(rt_model *m, const int64_t *x0_dev, uint64_t seed, uint64_t trajectory,
               uint64_t max_firings, double t_end, int64_t *x_out_dev, rt_result *res_dev,
               int32_t *trace_mu_dev, double *trace_t_dev, uint64_t trace_cap, void *stream) {
  if (!m || !x0_dev || !res_dev) return RT_ERR_NULL;
  int rc = check_limits(max_firings, t_end);
  if (rc != RT_OK) return rc;
  CU_TRY(cudaSetDevice(m->device));
  return launch_bundles(m, (const long long *)x0_dev, seed, trajectory, 1, max_firings, t_end,
                        (long long *)x_out_dev, res_dev, trace_mu_dev, trace_t_dev, trace_cap,
                        (cudaStream_t)stream);
}

// Body of rt_run / rt_run_resume (host pointers).  resume: start from (t0, T0, P0, n0).
static int run_host(rt_model *m, const int64_t *x0, bool resume, double t0, const double *T0, const double *P0,
             const uint64_t *n0, uint64_t seed, uint64_t trajectory, uint64_t max_firings, double t_end,
             int64_t *x_out, rt_result *res, uint64_t *fire_count_out, double *T_out, double *P_out,
             int32_t *trace_mu, double *trace_t, uint64_t trace_cap) {
  if (!m || !x0 || !res) return RT_ERR_NULL;
  if (resume && (!T0 || !P0 || !n0)) return RT_ERR_NULL;
  int rc = check_limits(max_firings, t_end);
  if (rc != RT_OK) return rc;
  if ((rc = check_x0(m, x0)) != RT_OK) return rc;
  const size_t N = (size_t)m->net.N, M = (size_t)m->net.M;
  if (resume) {
    if (!std::isfinite(t0) || t0 < 0.0 || t0 > t_end) return RT_ERR_BAD_ARG;
    for (size_t k = 0; k < M; ++k)
      if (std::isnan(T0[k]) || std::isnan(P0[k]) || n0[k] > 0xffffffffull) return RT_ERR_BAD_ARG;
  }
  CU_TRY(cudaSetDevice(m->device));
  if (!trace_mu && !trace_t) trace_cap = 0;
  if ((rc = m->d_x0.ensure(N * 8)) != RT_OK) return rc;
  if ((rc = m->d_xout.ensure(N * 8)) != RT_OK) return rc;
  if ((rc = m->d_res.ensure(sizeof(rt_result))) != RT_OK) return rc;
  if (trace_cap) {
    if ((rc = m->d_trace_mu.ensure(trace_cap * 4)) != RT_OK) return rc;
    if ((rc = m->d_trace_t.ensure(trace_cap * 8)) != RT_OK) return rc;
  }
  cudaStream_t st = 0;
  StartDev start;
  if (resume) {
    std::vector<uint32_t> n32(M);
    for (size_t k = 0; k < M; ++k) n32[k] = (uint32_t)n0[k];
    if ((rc = m->d_T0.ensure(M * 8)) != RT_OK) return rc;
    if ((rc = m->d_P0.ensure(M * 8)) != RT_OK) return rc;
    if ((rc = m->d_n0.ensure(M * 4)) != RT_OK) return rc;
    CU_TRY(cudaMemcpy(m->d_T0.p, T0, M * 8, cudaMemcpyHostToDevice));
    CU_TRY(cudaMemcpy(m->d_P0.p, P0, M * 8, cudaMemcpyHostToDevice));
    CU_TRY(cudaMemcpy(m->d_n0.p, n32.data(), M * 4, cudaMemcpyHostToDevice));
    start.t0 = t0;
    start.T0 = (const double *)m->d_T0.p; start.P0 = (const double *)m->d_P0.p;
    start.n0 = (const uint32_t *)m->d_n0.p;
  }
  CU_TRY(cudaMemcpyAsync(m->d_x0.p, x0, N * 8, cudaMemcpyHostToDevice, st));
  CU_TRY(cudaMemsetAsync(m->d_res.p, 0, sizeof(rt_result), st));
  // "ensemble_path" = 1 sends a resumed single trajectory of a tiny network through the
  // one-thread-per-trajectory kernel (which records no trace)
  const bool threads = resume && m->opt_ensemble_path == 1;
  if (threads) {
    if (!thread_path_fits(m) || m->opt_formulation != 0 || m->sched_n > 0 || m->rate_exp || trace_cap)
      return RT_ERR_UNSUPPORTED;
    const Plan pl = plan_bundles(m, 1);
    if ((rc = ensure_state(m, pl)) != RT_OK) return rc;
    rc = launch_threads(m, (const long long *)m->d_x0.p, seed, trajectory, 1, max_firings, t_end,
                        (long long *)m->d_xout.p, (rt_result *)m->d_res.p, st, start,
                        (double *)m->d_T.p, (double *)m->d_P.p, (uint32_t *)m->d_n.p);
  } else {
    rc = launch_bundles(m, (const long long *)m->d_x0.p, seed, trajectory, 1, max_firings, t_end,
                        (long long *)m->d_xout.p, (rt_result *)m->d_res.p,
                        trace_cap ? (int32_t *)m->d_trace_mu.p : nullptr,
                        trace_cap ? (double *)m->d_trace_t.p : nullptr, trace_cap, st, start);
  }
  if (rc != RT_OK) return rc;
  if ((rc = finish(m, st)) != RT_OK) return rc;
  CU_TRY(cudaMemcpy(res, m->d_res.p, sizeof(rt_result), cudaMemcpyDeviceToHost));
  if (x_out) CU_TRY(cudaMemcpy(x_out, m->d_xout.p, N * 8, cudaMemcpyDeviceToHost));
  const size_t nrec = (size_t)std::min<uint64_t>(res->firings, trace_cap);
  if (trace_mu && nrec) CU_TRY(cudaMemcpy(trace_mu, m->d_trace_mu.p, nrec * 4, cudaMemcpyDeviceToHost));
  if (trace_t && nrec) CU_TRY(cudaMemcpy(trace_t, m->d_trace_t.p, nrec * 8, cudaMemcpyDeviceToHost));
  if (T_out) CU_TRY(cudaMemcpy(T_out, m->d_T.p, M * 8, cudaMemcpyDeviceToHost));
  if (P_out) CU_TRY(cudaMemcpy(P_out, m->d_P.p, M * 8, cudaMemcpyDeviceToHost));
  if (fire_count_out) {
    std::vector<uint32_t> n32(M);
    CU_TRY(cudaMemcpy(n32.data(), m->d_n.p, M * 4, cudaMemcpyDeviceToHost));
    for (size_t k = 0; k < M; ++k) fire_count_out[k] = n32[k];
  }
  return res->status;
}

int rt_run(rt_model *m, const int64_t *x0, uint64_t seed, uint64_t trajectory,
           uint64_t max_firings, double t_end, int64_t *x_out, rt_result *res,
           uint64_t *fire_count_out, double *T_out, double *P_out,
           int32_t *trace_mu, double *trace_t, uint64_t trace_cap) {
  return run_host(m, x0, false, 0.0, nullptr, nullptr, nullptr, seed, trajectory, max_firings, t_end,
                  x_out, res, fire_count_out, T_out, P_out, trace_mu, trace_t, trace_cap);
}

int rt_run_resume(rt_model *m, const int64_t *x0, double t0, const double *T0, const double *P0,
                  const uint64_t *fire_count0, uint64_t seed, uint64_t trajectory,
                  uint64_t max_firings, double t_end, int64_t *x_out, rt_result *res,
                  uint64_t *fire_count_out, double *T_out, double *P_out,
                  int32_t *trace_mu, double *trace_t, uint64_t trace_cap) {
  return run_host(m, x0, true, t0, T0, P0, fire_count0, seed, trajectory, max_firings, t_end,
                  x_out, res, fire_count_out, T_out, P_out, trace_mu, trace_t, trace_cap);
}

int rt_ensemble_dev(rt_model *m, const int64_t *x0_dev, uint64_t seed, uint64_t traj_first,
                    uint64_t n_traj, uint64_t max_firings, double t_end, int64_t *x_out_dev,
                    rt_result *res_dev, void *stream) {
  if (!m || !x0_dev || !res_dev) return RT_ERR_NULL;
  int rc = check_limits(max_firings, t_end);
  if (rc != RT_OK) return rc;
  if (n_traj == 0) return RT_OK;
  CU_TRY(cudaSetDevice(m->device));
  // (the thread kernel implements the plain (T,P) form with constant rates only)
  bool use_threads = thread_path_fits(m) && m->opt_formulation == 0 && m->sched_n == 0 && !m->rate_exp;
  if (m->opt_ensemble_path == 1) {
    if (!thread_path_fits(m)) return RT_ERR_BAD_ARG;
    // the thread kernel implements the plain (T,P) form with constant rates only
    if (m->opt_formulation != 0 || m->sched_n > 0 || m->rate_exp) return RT_ERR_UNSUPPORTED;
    use_threads = true;
  } else if (m->opt_ensemble_path == 2) {
    use_threads = false;
  }
  if (use_threads)
    return launch_threads(m, (const long long *)x0_dev, seed, traj_first, n_traj, max_firings, t_end,
                          (long long *)x_out_dev, res_dev, (cudaStream_t)stream);
  return launch_bundles(m, (const long long *)x0_dev, seed, traj_first, n_traj, max_firings, t_end,
                        (long long *)x_out_dev, res_dev, nullptr, nullptr, 0, (cudaStream_t)stream);
}

int rt_ensemble(rt_model *m, const int64_t *x0, uint64_t seed, uint64_t traj_first,
                uint64_t n_traj, uint64_t max_firings, double t_end, int64_t *x_out,
                rt_result *res) {
  if (!m || !x0 || !res) return RT_ERR_NULL;
  int rc = check_limits(max_firings, t_end);
  if (rc != RT_OK) return rc;
  if ((rc = check_x0(m, x0)) != RT_OK) return rc;
  if (n_traj == 0) return RT_OK;
  CU_TRY(cudaSetDevice(m->device));
  const size_t N = (size_t)m->net.N;
  if ((rc = m->d_x0.ensure(N * 8)) != RT_OK) return rc;
  if ((rc = m->d_res.ensure(n_traj * sizeof(rt_result))) != RT_OK) return rc;
  if (x_out && (rc = m->d_xout.ensure(n_traj * N * 8)) != RT_OK) return rc;
  cudaStream_t st = 0;
  CU_TRY(cudaMemcpyAsync(m->d_x0.p, x0, N * 8, cudaMemcpyHostToDevice, st));
  CU_TRY(cudaMemsetAsync(m->d_res.p, 0, n_traj * sizeof(rt_result), st));
  rc = rt_ensemble_dev(m, (const int64_t *)m->d_x0.p, seed, traj_first, n_traj, max_firings, t_end,
                       x_out ? (int64_t *)m->d_xout.p : nullptr, (rt_result *)m->d_res.p, st);
  if (rc != RT_OK) return rc;
  if ((rc = finish(m, st)) != RT_OK) return rc;
  CU_TRY(cudaMemcpy(res, m->d_res.p, n_traj * sizeof(rt_result), cudaMemcpyDeviceToHost));
  if (x_out) CU_TRY(cudaMemcpy(x_out, m->d_xout.p, n_traj * N * 8, cudaMemcpyDeviceToHost));
  for (uint64_t i = 0; i < n_traj; ++i)
    if (res[i].status != RT_OK) return res[i].status;
  return RT_OK;
}

int rt_sync(rt_model *m, void *stream) {
  if (!m) return RT_ERR_NULL;
  CU_TRY(cudaSetDevice(m->device));
  return finish(m, (cudaStream_t)stream);
}

int rt_set_rate_schedule(rt_model *m, int32_t n_break, const double *t_break, const double *factor,
                         const uint8_t *mask) {
  if (!m) return RT_ERR_NULL;
  if (n_break < 0 || n_break > (1 << 20)) return RT_ERR_BAD_ARG;
  if (n_break == 0) { m->sched_n = 0; m->sched_has_mask = false; return RT_OK; }
  if (!t_break || !factor) return RT_ERR_NULL;
  for (int32_t i = 0; i < n_break; ++i) {
    if (!std::isfinite(t_break[i]) || t_break[i] < 0.0 || !std::isfinite(factor[i]) || factor[i] < 0.0)
      return RT_ERR_BAD_ARG;
    if (i > 0 && !(t_break[i] > t_break[i - 1])) return RT_ERR_BAD_ARG;
  }
  CU_TRY(cudaSetDevice(m->device));
  int rc;
  if ((rc = upload(m->d_sched_t, std::vector<double>(t_break, t_break + n_break))) != RT_OK) return rc;
  if ((rc = upload(m->d_sched_f, std::vector<double>(factor, factor + n_break))) != RT_OK) return rc;
  m->sched_has_mask = mask != nullptr;
  if (mask && (rc = upload(m->d_sched_mask, std::vector<uint8_t>(mask, mask + m->net.M))) != RT_OK) return rc;
  m->sched_n = n_break;
  return RT_OK;
}

int rt_set_rate_exponent(rt_model *m, const double *lambda) {
  if (!m) return RT_ERR_NULL;
  if (!lambda) { m->rate_exp = false; return RT_OK; }
  const size_t M = (size_t)m->net.M;
  std::vector<double> lam((size_t)m->net.M_pad, 0.0);
  bool any = false;
  for (size_t k = 0; k < M; ++k) {
    if (!std::isfinite(lambda[k])) return RT_ERR_BAD_ARG;
    lam[k] = lambda[k];
    any = any || lambda[k] != 0.0;
  }
  CU_TRY(cudaSetDevice(m->device));
  int rc = upload(m->d_lambda, lam);
  if (rc != RT_OK) return rc;
  m->rate_exp = any;         // all zero: constant rates, the default kernel
  return RT_OK;
}

int rt_set_option(rt_model *m, const char *name, int64_t value) {
  if (!m || !name) return RT_ERR_NULL;
  if (!strcmp(name, "refresh_mode")) {
    if (value != 0 && value != 1) return RT_ERR_BAD_ARG;
    m->refresh_mode = (int)value;
  } else if (!strcmp(name, "bundle_ctas")) {
    if (value < 0 || value > 1024) return RT_ERR_BAD_ARG;
    m->opt_bundle_ctas = (int)value;
  } else if (!strcmp(name, "ensemble_path")) {
    if (value < 0 || value > 2) return RT_ERR_BAD_ARG;
    m->opt_ensemble_path = (int)value;
  } else if (!strcmp(name, "formulation")) {
    if (value < 0 || value > 1) return RT_ERR_BAD_ARG;
    m->opt_formulation = (int)value;
  } else if (!strcmp(name, "prefetch")) {
    if (value < 0 || value > 7) return RT_ERR_BAD_ARG;
    m->opt_prefetch = (int)value;
  } else if (!strcmp(name, "x_replicas")) {
    if (value < 0 || value > 64) return RT_ERR_BAD_ARG;
    m->opt_x_replicas = (int)value;
  } else if (!strcmp(name, "state_mode")) {
    if (value < 0 || value > 1) return RT_ERR_BAD_ARG;
    m->opt_state_mode = (int)value;
  } else if (!strcmp(name, "tiny_kernel")) {
    if (value < 0 || value > 1) return RT_ERR_BAD_ARG;
    m->opt_tiny = (int)value;
  } else if (!strcmp(name, "l2_persist")) {
    if (value < 0 || value > 2) return RT_ERR_BAD_ARG;
    m->opt_l2_persist = (int)value;
  } else if (!strcmp(name, "pipeline")) {
    if (value < 0 || value > 1) return RT_ERR_BAD_ARG;
    m->opt_pipeline = (int)value;
  } else if (!strcmp(name, "exchange")) {
    if (value < 0 || value > 1) return RT_ERR_BAD_ARG;
    m->opt_exchange = (int)value;
  } else {
    return RT_ERR_BAD_ARG;
  }
  return RT_OK;
}

int rt_get_info(const rt_model *m, const char *name, int64_t *value) {
  if (!m || !name || !value) return RT_ERR_NULL;
  if (!strcmp(name, "kernel_launches")) *value = m->kernel_launches;
  else if (!strcmp(name, "bundle_ctas")) *value = m->last_S;
  else if (!strcmp(name, "bundles")) *value = m->last_B;
  else if (!strcmp(name, "block_threads")) *value = m->last_block;
  else if (!strcmp(name, "ensemble_path")) *value = m->last_path;
  else if (!strcmp(name, "num_sms")) *value = m->num_sms;
  else if (!strcmp(name, "dep_entries")) *value = m->nnz_r;
  else if (!strcmp(name, "max_sigma")) *value = m->max_sigma;
  else if (!strcmp(name, "state_in_smem")) *value = m->last_state_smem;
  else if (!strcmp(name, "cluster_exchange")) *value = m->last_cluster;
  else if (!strcmp(name, "pipeline")) *value = m->last_fast;
  else if (!strcmp(name, "tiny_kernel")) *value = m->last_tiny;
  else if (!strcmp(name, "l2_persist")) *value = (m->opt_l2_persist && m->l2_persist_max > 0 && m->l2_window_max > 0) ? m->opt_l2_persist : 0;
  else if (!strcmp(name, "hub_species")) *value = (int64_t)m->n_big;
  else return RT_ERR_BAD_ARG;
  return RT_OK;
}

void rt_destroy(rt_model *m) {
  if (!m) return;
  cudaSetDevice(m->device);
  if (m->l2_limit_set) {
    cudaDeviceSynchronize();
    cudaCtxResetPersistingL2Cache();
    cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, 0);
    cudaGetLastError();
  }
  DevBuf *bufs[] = {&m->d_react_ptr, &m->d_react_species, &m->d_react_sigma, &m->d_stoich_ptr,
                    &m->d_stoich_species, &m->d_stoich_v, &m->d_rate, &m->d_srow,
                    &m->d_sp_rec, &m->d_sp_big, &m->d_big_off, &m->d_dep,
                    &m->d_T, &m->d_P, &m->d_a, &m->d_n, &m->d_X, &m->d_exch, &m->d_err,
                    &m->d_x0, &m->d_xout, &m->d_res, &m->d_trace_mu, &m->d_trace_t,
                    &m->d_T0, &m->d_P0, &m->d_n0,
                    &m->d_sched_t, &m->d_sched_f, &m->d_sched_mask, &m->d_lambda};
  for (DevBuf *b : bufs) b->release();
  delete m;
}

const char *rt_strerror(int code) {
  switch (code) {
    case RT_OK: return "ok";
    case RT_ERR_NULL: return "null pointer argument";
    case RT_ERR_BAD_NETWORK: return "invalid reaction network";
    case RT_ERR_BAD_ARG: return "invalid argument";
    case RT_ERR_UNSUPPORTED: return "unsupported network (sigma > 3 or too many entries)";
    case RT_ERR_OVERFLOW: return "species count left the supported range";
    case RT_ERR_CUDA: return "CUDA error or in-kernel barrier timeout";
    case RT_ERR_OOM: return "out of memory";
    case RT_ERR_SCRATCH:
      return "no-allocation entry point: rt_noalloc_prepare not called for this model, or the run "
             "needs more than RT_NOALLOC_SCRATCH_BYTES of scratch";
    default: return "unknown error code";
  }
}

}  // extern "C"

// ---- no-allocation entry point (include/rt.h: rt_noalloc_prepare / rt_run_dev_noalloc) ---------
// The bundle kernels' scratch -- T, P, a, n, X and the exchange slots, which rt_run_dev keeps in
// cudaMalloc'ed buffers (ensure_state) -- carved out of one file-scope array in device memory.
// Every context that loads this module holds the array until it is destroyed.  In HOST code the
// name below is only a handle for cudaGetSymbolAddress, never a device address.
static __device__ __align__(256) unsigned char g_noalloc_scratch[RT_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int kNoallocMaxDevices = 64;
std::mutex g_noalloc_mu;
unsigned char *g_noalloc_ptr[kNoallocMaxDevices] = {};   // the array's device address, per device

struct ScratchLayout { size_t T, P, a, n, X, exch, exch_bytes, total; };

ScratchLayout scratch_layout(const rt_model *m, const Plan &pl) {
  auto up = [](size_t x) { return (x + 255) & ~(size_t)255; };
  const size_t Mp = (size_t)m->net.M_pad, N = (size_t)m->net.N, B = (size_t)pl.B;
  ScratchLayout L{};
  size_t at = 0;
  L.T = at; at += up(B * Mp * 8);
  L.P = at; at += up(B * Mp * 8);
  L.a = at; at += up(B * Mp * 8);
  L.n = at; at += up(B * Mp * 4);
  L.X = at; at += up(B * (size_t)pl.G * N * 8);
  L.exch = at;
  L.exch_bytes = B * 2 * (size_t)pl.S * rt::kSlotStride * 8;
  at += up(L.exch_bytes);
  L.total = at;
  return L;
}

}  // namespace

extern "C" {

int rt_noalloc_prepare(rt_model *m, uint64_t *need_bytes) {
  if (!m) return RT_ERR_NULL;
  if (m->device < 0 || m->device >= kNoallocMaxDevices) return RT_ERR_UNSUPPORTED;
  CU_TRY(cudaSetDevice(m->device));
  {
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[m->device]) {         // once per device, with that device current
      unsigned char *ptr = nullptr;
      CU_TRY(cudaGetSymbolAddress((void **)&ptr, g_noalloc_scratch));
      if (!ptr) return RT_ERR_CUDA;
      g_noalloc_ptr[m->device] = ptr;
    }
    m->noalloc_scratch = g_noalloc_ptr[m->device];
  }
  const Plan pl = plan_bundles(m, 1);        // (also asks the occupancy questions the plan caches)
  const ScratchLayout L = scratch_layout(m, pl);
  if (need_bytes) *need_bytes = (uint64_t)L.total;
  if (L.total > (size_t)RT_NOALLOC_SCRATCH_BYTES) return RT_ERR_SCRATCH;
  // load the kernel this plan launches now, outside the caller's no-allocation region
  const int rate = m->sched_n > 0 ? 1 : m->rate_exp ? 2 : 0;
  if (rate != 0 && (m->refresh_mode != 0 || m->opt_formulation != 0)) return RT_OK;   // (the run reports it)
  const void *kern = bundle_kernel(pl.smem, m->refresh_mode != 0, rate, pl.cluster, pl.fast);
  cudaFuncAttributes fa;
  CU_TRY(cudaFuncGetAttributes(&fa, kern));
  return RT_OK;
}

int rt_run_dev_noalloc(rt_model *m, const int64_t *x0_dev, uint64_t seed, uint64_t trajectory,
                       uint64_t max_firings, double t_end, int64_t *x_out_dev, rt_result *res_dev,
                       int32_t *trace_mu_dev, double *trace_t_dev, uint64_t trace_cap, void *stream) {
  if (!m || !x0_dev || !res_dev) return RT_ERR_NULL;
  int rc = check_limits(max_firings, t_end);
  if (rc != RT_OK) return rc;
  if (!m->noalloc_scratch) return RT_ERR_SCRATCH;
  if (m->sched_n > 0 && (m->refresh_mode != 0 || m->opt_formulation != 0)) return RT_ERR_UNSUPPORTED;
  if (m->rate_exp && (m->refresh_mode != 0 || m->opt_formulation != 0 || m->sched_n > 0)) return RT_ERR_UNSUPPORTED;
  CU_TRY(cudaSetDevice(m->device));
  cudaStream_t st = (cudaStream_t)stream;
  const Plan pl = plan_bundles(m, 1);
  const ScratchLayout L = scratch_layout(m, pl);
  if (L.total > (size_t)RT_NOALLOC_SCRATCH_BYTES) return RT_ERR_SCRATCH;
  unsigned char *base = m->noalloc_scratch;
  // the array keeps the last call's contents: the exchange slots must start at zero (their tags
  // would otherwise match a new round); everything else is written by the kernel before it is read
  CU_TRY(cudaMemsetAsync(base + L.exch, 0, L.exch_bytes, st));
  rt::BundleParams p{};
  p.net = m->net;
  p.T = (double *)(base + L.T); p.P = (double *)(base + L.P); p.a = (double *)(base + L.a);
  p.n = (uint32_t *)(base + L.n); p.X = (u64 *)(base + L.X);
  p.exch = (u64 *)(base + L.exch);
  p.S = pl.S; p.B = pl.B; p.G = pl.G; p.pairs_per_cta = pl.pairs_per_cta; p.cnt_pad = pl.cnt_pad;
  p.x0 = (const long long *)x0_dev; p.seed = seed; p.traj_first = trajectory; p.n_traj = 1;
  p.max_firings = max_firings; p.t_end = t_end;
  p.x_out = (long long *)x_out_dev; p.res = res_dev;
  p.trace_mu = trace_mu_dev; p.trace_t = trace_t_dev;
  p.trace_cap = (trace_mu_dev || trace_t_dev) ? trace_cap : 0;
  p.refresh_mode = m->refresh_mode;
  p.prefetch = m->opt_prefetch;
  p.formulation = m->opt_formulation;
  p.rate_lambda = (const double *)m->d_lambda.p;
  p.sched_n = m->sched_n;
  p.sched_t = (const double *)m->d_sched_t.p;
  p.sched_f = (const double *)m->d_sched_f.p;
  p.sched_mask = m->sched_has_mask ? (const unsigned char *)m->d_sched_mask.p : nullptr;
  p.err = (int *)m->d_err.p;                 // (16 bytes owned by the model since rt_create)
  void *args[] = {&p};
  const int rate = m->sched_n > 0 ? 1 : m->rate_exp ? 2 : 0;
  const void *kern = bundle_kernel(pl.smem, m->refresh_mode != 0, rate, pl.cluster, pl.fast);
  const size_t dyn = pl.smem ? smem_state_bytes(pl.pairs_per_cta, pl.fast) : 0;
  if (dyn) CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dyn));
  const int block = pl.fast ? kBlockFast : pl.smem ? kBlockSmem : kBlockGlobal;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(pl.S * pl.B); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = dyn; cfg.stream = st;
  cudaLaunchAttribute at[1];
  if (pl.cluster) {
    if (pl.S > 8) CU_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = pl.S; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  } else {
    at[0].id = cudaLaunchAttributeCooperative;
    at[0].val.cooperative = 1;
  }
  cfg.attrs = at; cfg.numAttrs = 1;
  CU_TRY(cudaLaunchKernelExC(&cfg, kern, args));
  m->last_block = block;
  m->kernel_launches += 1;
  m->last_S = pl.S; m->last_B = pl.B; m->last_path = 2; m->last_state_smem = pl.smem ? 1 : 0;
  m->last_cluster = pl.cluster ? 1 : 0;
  m->last_fast = pl.fast ? 1 : 0;
  return RT_OK;
}

}  // extern "C"
