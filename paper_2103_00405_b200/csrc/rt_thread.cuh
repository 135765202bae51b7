// rt_thread.cuh -- ensemble kernel for small networks: ONE THREAD = ONE TRAJECTORY
// (north_star subsystem 5; the paper's Fig.1 workload is exactly this regime: 10 000 Lotka
// trajectories side by side).  The network (a few CSR rows) is staged once per
// CTA in shared memory; every thread keeps its whole state (T, P, a, n per reaction, X per
// species) in shared memory, laid out [item][thread] so that a warp's accesses to item i hit
// 32 different banks.  No thread ever talks to another: each lane loops over its own firings
// to its own t_end / max_firings.  Every propensity is recomputed each firing (M is tiny), in
// exactly the operation order of the bundle kernel, so the two paths give identical results.
#pragma once
#include "rt_device.cuh"
#include "../../include/rt.h"

namespace rt {

struct ThreadParams {
  NetDev net;
  uint32_t nnz_r, nnz_v;
  const long long *x0;
  u64 seed, traj_first, n_traj, max_firings;
  double t_end;
  long long *x_out;      // [n_traj][N] or nullptr
  rt_result *res;        // [n_traj]
  // single trajectory through this kernel (rt_run_resume with ensemble_path = 1): checkpoint to
  // start from and final per-reaction state; all nullptr for ensembles
  const double *T0, *P0;
  const uint32_t *n0;
  double t0;
  double *T_out, *P_out;
  uint32_t *n_out;
};

// Shared-memory bytes: network copy + BLOCK * (3*8*M + 4*M + 8*N).
__host__ __device__ inline size_t thread_kernel_smem(int M, int N, uint32_t nnz_r, uint32_t nnz_v,
                                                     int block) {
  size_t net = (size_t)M * 8 + 2 * (size_t)(M + 1) * 4 + 2 * (size_t)nnz_r * 4 + 2 * (size_t)nnz_v * 4;
  net = (net + 15) & ~(size_t)15;
  return net + (size_t)block * ((size_t)M * 28 + (size_t)N * 8);
}

template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) rt_thread_kernel(const ThreadParams p) {
  extern __shared__ __align__(16) unsigned char smem[];
  const NetDev &net = p.net;
  const int M = net.M, N = net.N, tid = threadIdx.x;
  const double INF = __longlong_as_double(0x7ff0000000000000ll);

  // ---- carve shared memory: network first, then per-thread state [item][BLOCK]
  double *s_rate = reinterpret_cast<double *>(smem);
  uint32_t *s_rp = reinterpret_cast<uint32_t *>(s_rate + M);
  uint32_t *s_sp = s_rp + (M + 1);
  int32_t *s_rs = reinterpret_cast<int32_t *>(s_sp + (M + 1));
  int32_t *s_rg = s_rs + p.nnz_r;
  int32_t *s_ss = s_rg + p.nnz_r;
  int32_t *s_sv = s_ss + p.nnz_v;
  size_t off = (size_t)M * 8 + 2 * (size_t)(M + 1) * 4 + 2 * (size_t)p.nnz_r * 4 + 2 * (size_t)p.nnz_v * 4;
  off = (off + 15) & ~(size_t)15;
  double *sT = reinterpret_cast<double *>(smem + off);
  double *sP = sT + (size_t)M * BLOCK;
  double *sA = sP + (size_t)M * BLOCK;
  long long *sX = reinterpret_cast<long long *>(sA + (size_t)M * BLOCK);
  uint32_t *sN = reinterpret_cast<uint32_t *>(sX + (size_t)N * BLOCK);

  for (int i = tid; i < M; i += BLOCK) s_rate[i] = net.rate[i];
  for (int i = tid; i <= M; i += BLOCK) { s_rp[i] = net.react_ptr[i]; s_sp[i] = net.stoich_ptr[i]; }
  for (uint32_t i = tid; i < p.nnz_r; i += BLOCK) { s_rs[i] = net.react_species[i]; s_rg[i] = net.react_sigma[i]; }
  for (uint32_t i = tid; i < p.nnz_v; i += BLOCK) { s_ss[i] = net.stoich_species[i]; s_sv[i] = net.stoich_v[i]; }
  __syncthreads();

  const u64 it = (u64)blockIdx.x * BLOCK + tid;
  if (it >= p.n_traj) return;
  const u64 traj = p.traj_first + it;

#define ST(arr, i) arr[(size_t)(i) * BLOCK + tid]
  for (int j = 0; j < N; ++j) ST(sX, j) = p.x0[j];
  for (int k = 0; k < M; ++k) {
    ST(sT, k) = p.T0 ? p.T0[k] : 0.0;
    ST(sP, k) = p.T0 ? p.P0[k] : exp_draw(p.seed, traj, (uint32_t)k, 0u);
    ST(sN, k) = p.T0 ? p.n0[k] : 0u;
  }
  double t = p.t0;
  u64 fired = 0;
  int stop = 0, status = RT_OK;

  for (;;) {
    // a-1, a-2, a-3: propensities, waiting times, argmin (lowest k on ties: strict <, k ascending)
    double delta = INF;
    int mu = 0;
    for (int k = 0; k < M; ++k) {
      double a = s_rate[k];
      for (uint32_t e = s_rp[k]; e < s_rp[k + 1]; ++e)
        a = __dmul_rn(a, __ll2double_rn(binom(ST(sX, s_rs[e]), s_rg[e])));
      ST(sA, k) = a;
      const double d = waiting_time(ST(sP, k), ST(sT, k), a);
      if (d < delta) { delta = d; mu = k; }
    }
    // a-4
    if (delta == INF) { stop = RT_STOP_ABSORBED; break; }
    if (p.t_end < INF && __dadd_rn(t, delta) > p.t_end) {
      const double rest = __dsub_rn(p.t_end, t);
      for (int k = 0; k < M; ++k) ST(sT, k) = __dadd_rn(ST(sT, k), __dmul_rn(ST(sA, k), rest));
      t = p.t_end;
      stop = RT_STOP_T_END;
      break;
    }
    // a-5
    t = __dadd_rn(t, delta);
    for (int k = 0; k < M; ++k) ST(sT, k) = __dadd_rn(ST(sT, k), __dmul_rn(ST(sA, k), delta));
    // a-6: nothing is written if any count of the row would leave [0, xmax] (as in the bundle kernel)
    for (uint32_t e = s_sp[mu]; e < s_sp[mu + 1]; ++e) {
      const long long x = ST(sX, s_ss[e]) + (long long)s_sv[e];
      if (x < 0 || x > net.xmax) status = RT_ERR_OVERFLOW;
    }
    if (status == RT_OK)
      for (uint32_t e = s_sp[mu]; e < s_sp[mu + 1]; ++e) ST(sX, s_ss[e]) += (long long)s_sv[e];
    // a-7
    const uint32_t c = ST(sN, mu) + 1u;
    ST(sN, mu) = c;
    ST(sP, mu) = __dadd_rn(ST(sP, mu), exp_draw(p.seed, traj, (uint32_t)mu, c));
    fired += 1;
    if (status != RT_OK) break;
    if (p.max_firings != 0 && fired == p.max_firings) { stop = RT_STOP_MAX_FIRINGS; break; }
  }

  if (p.x_out)
    for (int j = 0; j < N; ++j) p.x_out[it * (u64)N + (u64)j] = ST(sX, j);
  if (p.T_out && it == 0)
    for (int k = 0; k < M; ++k) { p.T_out[k] = ST(sT, k); p.P_out[k] = ST(sP, k); p.n_out[k] = ST(sN, k); }
  rt_result res;
  res.t = t; res.firings = fired; res.stop = stop; res.status = status;
  p.res[it] = res;
#undef ST
}


// ---- rt_tiny_kernel: the same one-thread-per-trajectory scheme for the smallest networks (at most
// kTinyM reactions of at most two reactants over at most kTinyN species: BASELINE configs 1 and 2),
// with the whole state -- T, P, a, n, X -- in REGISTERS (loops over k and j fully unrolled; the
// network comes as a dense by-value table in the kernel's constant bank, indexed by the uniform or
// per-thread reaction number).  Same operations in the same order as rt_thread_kernel, so the two
// give identical results; what goes away is every shared-memory access, every CSR pointer chase,
// and the three exact divisions of a step become independent instruction streams.
constexpr int kTinyM = 4, kTinyN = 4;
struct TinyNet {
  int M, N;
  double rate[kTinyM];
  int r_j[kTinyM][2];          // reactant species in CSR order (-1: none)
  int r_s[kTinyM][2];          //   and their sigma
  int v[kTinyM][kTinyN];       // net stoichiometry, dense
  long long xmax;
};
struct TinyParams {
  TinyNet net;
  const long long *x0;
  u64 seed, traj_first, n_traj, max_firings;
  double t_end;
  long long *x_out;
  rt_result *res;
  const double *T0, *P0;
  const uint32_t *n0;
  double t0;
  double *T_out, *P_out;
  uint32_t *n_out;
};

__device__ __forceinline__ long long tiny_x(const long long (&X)[kTinyN], int j) {
  long long x = X[0];
#pragma unroll
  for (int i = 1; i < kTinyN; ++i) x = (j == i) ? X[i] : x;
  return x;
}

template <int BLOCK>
__global__ void __launch_bounds__(BLOCK) rt_tiny_kernel(const TinyParams p) {
  const TinyNet &net = p.net;
  const int M = net.M, N = net.N;
  const double INF = __longlong_as_double(0x7ff0000000000000ll);
  const u64 it = (u64)blockIdx.x * BLOCK + threadIdx.x;
  if (it >= p.n_traj) return;
  const u64 traj = p.traj_first + it;

  long long X[kTinyN];
  double T[kTinyM], P[kTinyM], A[kTinyM];
  uint32_t n[kTinyM];
#pragma unroll
  for (int j = 0; j < kTinyN; ++j) X[j] = j < N ? p.x0[j] : 0;
#pragma unroll
  for (int k = 0; k < kTinyM; ++k) {
    T[k] = 0.0; P[k] = 0.0; A[k] = 0.0; n[k] = 0u;
    if (k < M) {
      T[k] = p.T0 ? p.T0[k] : 0.0;
      P[k] = p.T0 ? p.P0[k] : exp_draw(p.seed, traj, (uint32_t)k, 0u);
      n[k] = p.T0 ? p.n0[k] : 0u;
    }
  }
  double t = p.t0;
  u64 fired = 0;
  int stop = 0, status = RT_OK;

  for (;;) {
    // a-1, a-2, a-3: propensities, waiting times, argmin (lowest k on ties: strict <, k ascending)
    double d[kTinyM];
#pragma unroll
    for (int k = 0; k < kTinyM; ++k) {
      d[k] = INF;
      if (k < M) {
        double a = net.rate[k];
        if (net.r_j[k][0] >= 0) a = __dmul_rn(a, __ll2double_rn(binom(tiny_x(X, net.r_j[k][0]), net.r_s[k][0])));
        if (net.r_j[k][1] >= 0) a = __dmul_rn(a, __ll2double_rn(binom(tiny_x(X, net.r_j[k][1]), net.r_s[k][1])));
        A[k] = a;
        d[k] = waiting_time(P[k], T[k], a);      // (an approximate-quotient filter as in scan_filtered was
      }                                          //  measured SLOWER here: the divisions overlap anyway)
    }
    double delta = INF;
    int mu = 0;
#pragma unroll
    for (int k = 0; k < kTinyM; ++k)
      if (d[k] < delta) { delta = d[k]; mu = k; }
    // a-4
    if (delta == INF) { stop = RT_STOP_ABSORBED; break; }
    if (p.t_end < INF && __dadd_rn(t, delta) > p.t_end) {
      const double rest = __dsub_rn(p.t_end, t);
#pragma unroll
      for (int k = 0; k < kTinyM; ++k) if (k < M) T[k] = __dadd_rn(T[k], __dmul_rn(A[k], rest));
      t = p.t_end;
      stop = RT_STOP_T_END;
      break;
    }
    // a-5
    t = __dadd_rn(t, delta);
#pragma unroll
    for (int k = 0; k < kTinyM; ++k) if (k < M) T[k] = __dadd_rn(T[k], __dmul_rn(A[k], delta));
    // a-6: nothing is written if any count of the row would leave [0, xmax]
    long long xn[kTinyN];
    bool bad = false;
#pragma unroll
    for (int j = 0; j < kTinyN; ++j) {
      xn[j] = X[j] + (long long)net.v[mu][j];
      bad = bad || (j < N && (xn[j] < 0 || xn[j] > net.xmax));
    }
    if (bad) status = RT_ERR_OVERFLOW;
    else {
#pragma unroll
      for (int j = 0; j < kTinyN; ++j) X[j] = xn[j];
    }
    // a-7
    uint32_t c = 0u;
#pragma unroll
    for (int k = 0; k < kTinyM; ++k) if (k == mu) { n[k] += 1u; c = n[k]; }
    const double e_new = exp_draw(p.seed, traj, (uint32_t)mu, c);
#pragma unroll
    for (int k = 0; k < kTinyM; ++k) if (k == mu) P[k] = __dadd_rn(P[k], e_new);
    fired += 1;
    if (status != RT_OK) break;
    if (p.max_firings != 0 && fired == p.max_firings) { stop = RT_STOP_MAX_FIRINGS; break; }
  }

  if (p.x_out)
#pragma unroll
    for (int j = 0; j < kTinyN; ++j) if (j < N) p.x_out[it * (u64)N + (u64)j] = X[j];
  if (p.T_out && it == 0) {
#pragma unroll
    for (int k = 0; k < kTinyM; ++k) if (k < M) { p.T_out[k] = T[k]; p.P_out[k] = P[k]; p.n_out[k] = n[k]; }
  }
  rt_result res;
  res.t = t; res.firings = fired; res.stop = stop; res.status = status;
  p.res[it] = res;
}

}  // namespace rt
