// rt_bundle.cuh -- persistent "bundle" kernel: a group of S CTAs (the paper's bundle =
// "a batch of blocks" holding one trajectory) simulates one trajectory after
// another; B bundles run side by side.  One launch covers every firing of every trajectory, so
// launch latency never sits between firings.
//
// Every CTA owns a fixed contiguous range [k0, k1) of reactions.  Its (T, P, a) triples live
//   * in SHARED MEMORY for the whole trajectory when the range fits (STATE_SMEM: M up to
//     ~1.3e6 on 148 SMs) -- the per-firing pass then never leaves the SM;
//   * in global memory otherwise (structure-of-arrays fp64, 16-byte vector accesses,
//     24 B read + 8 B written per reaction per firing -- the HBM-streaming regime).
//
// One firing costs ONE grid-wide exchange.  Between two exchanges a CTA runs, concurrently:
//   stream warps:  T_k += a_k * dt_prev      internal-time increment of the PREVIOUS firing (Eq.15)
//                  dt_k = (P_k - T_k) / a_k  waiting time for THIS firing (Eq.24), +inf if a_k = 0
//                  thread-local lexicographic min (Eq.25, ties to the lowest k)
//   walker warp:   X += v_mu (Eq.5): every CTA knows mu after the exchange and applies the
//                  update itself to the one L2-resident copy of X (versioned words, atomicMax:
//                  see rt_device.cuh), so no CTA ever waits for another's write; redraw of
//                  P_mu (Eq.26); then the dependency walk: 64-byte stoich row of
//                  mu (with the dependency ranges of its species) -> dense 32-byte dependency
//                  entries (k, reactants, sigma, c_k) -> new a_k for the k in [k0, k1).
// The stream uses the OLD a_k, which is exactly the propensity that held during the elapsed
// interval, so T is right for every k; only the waiting times of the refreshed reactions (and
// of mu) are stale.  After one CTA barrier the new a_k / P_mu are stored; a refreshed reaction
// joins the reduction as a fresh candidate, and only a thread whose own proposal was refreshed
// (or fired) re-scans its reactions (read-only); the block argmin follows.  While the exchange
// runs, the walker warp pre-walks the runner-up, the likeliest next winner (see Spec).
// The CTA partials are combined by an all-gather through L2 (one 16-byte slot per CTA,
// self-validating words, double-buffered), which doubles as the per-firing bundle barrier.
#pragma once
#include "rt_device.cuh"
#include "../../include/rt.h"

namespace rt {

constexpr int kListCap = 256;       // refreshed reactions a CTA stages per round
constexpr int kWalkerWarps = 1;
constexpr int kMaxBundleCtas = 160; // CTAs that may share one trajectory (5 exchange slots per lane)
#ifndef RT_SLOT_STRIDE
#define RT_SLOT_STRIDE 128
#endif
// u64 words between exchange slots: 1 KiB, so that the slots every CTA polls spread over as many L2
// slices instead of queueing on a few.  Measured (tests/helpers/exchange_floor.cu with this stride,
// 148 CTAs): 16 B..128 B apart 2.3-3.2 us per round (posters share lines), 256 B 1.23 us, 1 KiB
// 1.02 us, 4 KiB 1.06 us; in the kernel cfg4 3.26 -> 3.23 us, cfg5b +1.5 %.
constexpr int kSlotStride = RT_SLOT_STRIDE;

struct BundleParams {
  NetDev net;
  double *T, *P, *a;      // [B][M_pad]   (STATE_SMEM: written once, at the end of a trajectory)
  uint32_t *n;            // [B][M_pad]   firings per reaction
  u64 *X;                 // [B][G][N]    versioned counts (rt_device.cuh); CTA r uses replica r % G
  int G;                  //              so that no more than S/G CTAs hammer one L2 line
  u64 *exch;              // [B][2][S][kSlotStride] exchange slots (2 words used), zeroed before launch
  int S, B;
  int pairs_per_cta;
  int cnt_pad;            // STATE_SMEM: slots per array (the CTA's reactions padded to a whole number
                          // of scan batches; padding slots hold a = T = 0, P = 1)
  const long long *x0;    // [N]
  // checkpoint to resume from (rt_run_resume; single trajectory): nullptr = fresh start
  const double *T0, *P0;  // [M]
  const uint32_t *n0;     // [M]
  double t0;              // real time of the checkpoint (0 for a fresh start)
  u64 seed, traj_first, n_traj, max_firings;
  double t_end;
  long long *x_out;       // [n_traj][N] or nullptr
  rt_result *res;         // [n_traj]
  int32_t *trace_mu;      // first trajectory of the launch only; may be nullptr
  double *trace_t;
  u64 trace_cap;
  int prefetch;           // walker prefetches its candidate's walk data during the exchange
  int formulation;        // 0: (T, P) internal-time form; 1: residual (Table 3) form, kept as
                          //    T_k = -R_k with P_k = 0 (same operations, one array less to read)
  int refresh_mode;       // 0 dependency walk, 1 recompute every a_k (the paper's GPU scheme)
  // time-dependent rates (Eq.28, piecewise constant): c_k(t) = c_k * sched_f[i] for t in
  // [sched_t[i], sched_t[i+1]) for the channels with sched_mask[k] != 0 (all if nullptr)
  int sched_n;
  const double *sched_t, *sched_f;
  const unsigned char *sched_mask;
  // smoothly time-dependent rates (Eq.28): c_k(t) = c_k exp(rate_lambda[k] t), [M_pad]
  const double *rate_lambda;
  int *err;               // set to 1 on a barrier timeout
};

constexpr long long kSpinLimitCycles = 6000000000ll;   // ~3 s: a barrier that long is a bug

template <int BLOCK>
struct BundleCtx {
  Cand warp_part[BLOCK / 32];
  Cand win;
  int second_k;           // runner-up of the exchange (reaction index, or 0x7fffffff)
  int abort_local;        // a count left [0, xmax] (identical in every CTA: all replicate X)
  int list_n;             // staged refreshes of this round
  int more;               // walker has entries left for another round
  int any_odd;            // some a_k of this CTA is outside the filter's safe range (sticky)
  int n_stale;            // global-memory state: threads whose candidate must be re-scanned
  int p_k;                // reaction whose P was redrawn (or -1), and its new value
  double p_val;
  // cluster bundles: every peer's (dt, k) lands here by st.async, double-buffered by generation
  // parity; cl_bar[b] counts the 16 * S bytes of generation parity b
  alignas(16) u64 cl_slot[2][kMaxClusterCtas][2];
  alignas(8) u64 cl_bar[2];
};

// ---- filtered scan (state in shared memory) ----------------------------------------------------
// The argmin needs the correctly rounded quotient of only ONE of a thread's reactions: the others
// are ruled out by an approximate quotient q~ = (float)(r * rcp.approx(a)).  rcp.approx.ftz.f64
// (MUFU.RCP64H) is good to 2^-19.9 relative on normal inputs (measured over 4e9 values);
// with the multiply's and the conversion's rounding q~ is within 2^-19.5 of the true quotient.
// A reaction whose q~ exceeds (1 + 2^-16) times the thread's smallest q~ has a correctly rounded
// quotient strictly above that reaction's, so it can neither win nor tie.  If a second reaction
// of the thread is within the tolerance, or the smallest q~ is outside [2^-100, 2^100] (which
// also catches negative residuals, zeros and NaNs), or some a_k of this CTA is outside the range
// where the bound holds (`any_odd`), the thread divides exactly (__ddiv_rn) and compares
// lexicographically -- so the result is always bit-identical to dividing everything.
// a_k = 0 needs no test: rcp gives +inf, the product +inf or NaN, neither is ever the smallest.
// Per reaction the pass issues ~16 instructions instead of ~45: the pass is issue-bound.
constexpr float kFilterTol = 0x1.0p-16f;
constexpr int kScanBatch = 4;     // reactions in flight per thread; state padded to kScanBatch * NT
__device__ __forceinline__ double rcp_approx(double x) {
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  return y;
}
// a_k values for which the error bound of the filter is not established (non-zero only)
__device__ __forceinline__ bool filter_unsafe(double a) {
  const unsigned ea = ((unsigned)__double2hiint(a) >> 20) & 0x7ffu;
  return (ea - 100u >= 1847u) && ((__double_as_longlong(a) << 1) != 0ll);
}

// ---- smooth time-dependent rates (Eq.28, :224-231): c_k(s) = c_k exp(lambda_k s) -------
// The stored a_k is the time-independent part b_k = c_k h_k; the propensity at time t is
// a_k(t) = b_k exp(lambda_k t).  Channel k's own equation of Eq.28,
//   P_k - T_k = int_t^{t+d} a_k(s) ds = a_k(t) (exp(lambda_k d) - 1) / lambda_k,
// is solved in closed form, dt_k = log1p(lambda_k (P_k - T_k) / a_k(t)) / lambda_k (+inf when the
// argument is <= -1: a decaying channel whose remaining integral is smaller than its residual),
// and the clocks advance by T_k += a_k(t) expm1(lambda_k d) / lambda_k.  lambda_k = 0 is the
// constant-rate formula.  One rounded operation per step, in the order DESIGN.md fixes.
struct RateExp {
  const double *lam;     // [M_pad] lambda_k (0 in the padding)
  double t_now;          // real time now (start of the interval being searched)
  double t_prev;         // real time at the start of the interval that just elapsed (length dprev)
};
__device__ __noinline__ double waiting_time_exp(double P, double T, double b, double lam, double t) {
  const double INF = __longlong_as_double(0x7ff0000000000000ll);
  if (lam == 0.0) return waiting_time(P, T, b);
  const double a = __dmul_rn(b, exp(__dmul_rn(lam, t)));
  if (!(a > 0.0)) return INF;
  double r = __dsub_rn(P, T);
  r = r < 0.0 ? 0.0 : r;
  const double x = __ddiv_rn(__dmul_rn(lam, r), a);
  return x > -1.0 ? __ddiv_rn(log1p(x), lam) : INF;
}
__device__ __noinline__ double advance_exp(double T, double b, double lam, double t0, double d) {
  if (lam == 0.0) return __dadd_rn(T, __dmul_rn(b, d));
  const double a = __dmul_rn(b, exp(__dmul_rn(lam, t0)));
  const double e = __ddiv_rn(expm1(__dmul_rn(lam, d)), lam);
  return __dadd_rn(T, __dmul_rn(a, e));
}
template <bool EXPR>
__device__ __forceinline__ double wt(double P, double T, double a, int k, const RateExp &rx) {
  return EXPR ? waiting_time_exp(P, T, a, __ldg(rx.lam + k), rx.t_now) : waiting_time(P, T, a);
}

template <int NT, bool UPDATE>
__device__ __forceinline__ Cand scan_filtered(int tid, int k0, int cnt_pad, double *__restrict__ sT,
                                              const double *__restrict__ sP,
                                              const double *__restrict__ sA, double dprev, bool any_odd,
                                              bool &defer) {
  constexpr int U = kScanBatch;
  const float FINF = __int_as_float(0x7f800000);
  float m1 = FINF, m2 = FINF;
  int i1 = tid;
  for (int i = tid; i < cnt_pad; i += U * NT) {
    double a[U], t[U], pk[U];
#pragma unroll
    for (int u = 0; u < U; ++u) { a[u] = sA[i + u * NT]; t[u] = sT[i + u * NT]; pk[u] = sP[i + u * NT]; }
    if (UPDATE) {
#pragma unroll
      for (int u = 0; u < U; ++u) {
        t[u] = __dadd_rn(t[u], __dmul_rn(a[u], dprev));
        sT[i + u * NT] = t[u];
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const float q = __double2float_rn(__dmul_rn(__dsub_rn(pk[u], t[u]), rcp_approx(a[u])));
      m2 = fminf(m2, fmaxf(q, m1));          // NaN (0 * inf) is dropped by fminf / fmaxf
      if (q < m1) { m1 = q; i1 = i + u * NT; }
    }
  }
  Cand best;
  best.dt = __longlong_as_double(0x7ff0000000000000ll);
  best.k = 0x7fffffff;
  const float thr = m1 * (1.0f + kFilterTol);
  if (!any_odd && m1 >= 0x1.0p-100f && m1 <= 0x1.0p100f && m2 > thr) {   // common case: one division
    best.dt = waiting_time(sP[i1], sT[i1], sA[i1]);
    best.k = k0 + i1;
  } else if (UPDATE) {
    // Not decidable by the filter.  In the first pass that is nearly always the thread that owns
    // the reaction that just fired (its residual is ~0 until P is redrawn) -- which re-scans
    // anyway once the new values are stored.  Leave every such case to the re-scan.
    defer = true;
  } else {
    const bool all = any_odd || !(m1 >= 0x1.0p-100f && m1 <= 0x1.0p100f);
    for (int i = tid; i < cnt_pad; i += NT) {             // near tie (or odd values): a second,
      const double a = sA[i], pk = sP[i], t = sT[i];      // read-only pass divides what is close
      const float q = __double2float_rn(__dmul_rn(__dsub_rn(pk, t), rcp_approx(a)));
      if (all || q <= thr) {
        const double d = waiting_time(pk, t, a);
        if (d < best.dt) { best.dt = d; best.k = k0 + i; }
      }
    }
  }
  return best;
}

// The same filter over state streamed from global memory (HBM regime, cfg5a): 4 pairs of
// reactions per thread and iteration, i.e. twelve 16-byte loads (192 B) in flight per thread
// before any is used, and ~1/3 of the instructions of dividing everything, so that the pass is
// bound by the memory system and not by issue slots.  Padding reactions (k >= M) hold a = 0.
// RESID: residual form -- P is identically 0 and is not read (24 instead of 32 bytes per reaction).
template <int NT, bool UPDATE, bool RESID>
__device__ __forceinline__ Cand scan_filtered_global(int tid, int k0, int k1, double *T, double *P,
                                                     double *A, double dprev, bool any_odd, bool &defer) {
  constexpr int U = 4;
  const float FINF = __int_as_float(0x7f800000);
  double2 *T2 = reinterpret_cast<double2 *>(T);
  const double2 *P2 = reinterpret_cast<const double2 *>(P);
  const double2 *A2 = reinterpret_cast<const double2 *>(A);
  const int q0 = k0 >> 1, q1 = k1 >> 1;
  float m1 = FINF, m2 = FINF;
  int i1 = k0;
  for (int q = q0 + tid; q < q1; q += U * NT) {
    double2 tt[U], pp[U], aa[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int qu = q + u * NT;
      if (qu < q1) {
        tt[u] = __ldcg(T2 + qu); aa[u] = __ldcg(A2 + qu);
        pp[u] = RESID ? make_double2(0.0, 0.0) : __ldcg(P2 + qu);
      } else {                                   // P - T = 1, a = 0: q~ = +inf
        tt[u] = make_double2(RESID ? -1.0 : 0.0, RESID ? -1.0 : 0.0);
        pp[u] = make_double2(RESID ? 0.0 : 1.0, RESID ? 0.0 : 1.0);
        aa[u] = make_double2(0.0, 0.0);
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int qu = q + u * NT;
      if (UPDATE) {
        tt[u].x = __dadd_rn(tt[u].x, __dmul_rn(aa[u].x, dprev));
        tt[u].y = __dadd_rn(tt[u].y, __dmul_rn(aa[u].y, dprev));
        if (qu < q1) __stcg(T2 + qu, tt[u]);
      }
      float qf = __double2float_rn(__dmul_rn(__dsub_rn(pp[u].x, tt[u].x), rcp_approx(aa[u].x)));
      m2 = fminf(m2, fmaxf(qf, m1));
      if (qf < m1) { m1 = qf; i1 = 2 * qu; }
      qf = __double2float_rn(__dmul_rn(__dsub_rn(pp[u].y, tt[u].y), rcp_approx(aa[u].y)));
      m2 = fminf(m2, fmaxf(qf, m1));
      if (qf < m1) { m1 = qf; i1 = 2 * qu + 1; }
    }
  }
  Cand best;
  best.dt = __longlong_as_double(0x7ff0000000000000ll);
  best.k = 0x7fffffff;
  const float thr = m1 * (1.0f + kFilterTol);
  const bool decided = !any_odd && m1 >= 0x1.0p-100f && m1 <= 0x1.0p100f && m2 > thr;
  if (decided) {
    best.dt = waiting_time(RESID ? 0.0 : __ldcg(P + i1), __ldcg(T + i1), __ldcg(A + i1));
    best.k = i1;
  } else if (UPDATE) {
    defer = true;                               // left to the re-scan (see scan_filtered)
  } else {
    const bool all = any_odd || !(m1 >= 0x1.0p-100f && m1 <= 0x1.0p100f);
    for (int q = q0 + tid; q < q1; q += NT) {
      const double2 t2 = __ldcg(T2 + q), p2 = __ldcg(P2 + q), a2 = __ldcg(A2 + q);
      float qf = __double2float_rn(__dmul_rn(__dsub_rn(p2.x, t2.x), rcp_approx(a2.x)));
      if (all || qf <= thr) {
        const double d = waiting_time(p2.x, t2.x, a2.x);
        if (d < best.dt) { best.dt = d; best.k = 2 * q; }
      }
      qf = __double2float_rn(__dmul_rn(__dsub_rn(p2.y, t2.y), rcp_approx(a2.y)));
      if (all || qf <= thr) {
        const double d = waiting_time(p2.y, t2.y, a2.y);
        if (d < best.dt) { best.dt = d; best.k = 2 * q + 1; }
      }
    }
  }
  return best;
}

// The per-firing pass of one thread over the reactions it owns.  UPDATE: also apply the
// internal-time increment T_k += a_k * dprev (first pass); otherwise read-only (re-scan).
// FULL: recompute a_k from X for every k (refresh_mode 1).
// Ownership: STATE_SMEM -- local index i = tid, tid+NT, ...; global state -- pair q0+tid, +NT, ...
// EXPR: exponential time-dependent rates (plain loops with the closed-form solve; no filter).
template <int NT, bool SMEM, bool UPDATE, bool EXPR = false>
__device__ __forceinline__ Cand scan_own(const NetDev &net, const u64 *X, int tid, int k0, int k1,
                                         double *sT, const double *sP, double *sA,
                                         double *T, double *P, double *A, double dprev, bool full,
                                         int cnt_pad, bool any_odd, bool &defer, bool resid = false,
                                         const RateExp &rx = RateExp()) {
  Cand best;
  best.dt = __longlong_as_double(0x7ff0000000000000ll);
  best.k = 0x7fffffff;
  if (!EXPR && SMEM && !full) return scan_filtered<NT, UPDATE>(tid, k0, cnt_pad, sT, sP, sA, dprev, any_odd, defer);
  if (!EXPR && !SMEM && !full)
    return resid ? scan_filtered_global<NT, UPDATE, true>(tid, k0, k1, T, P, A, dprev, any_odd, defer)
                 : scan_filtered_global<NT, UPDATE, false>(tid, k0, k1, T, P, A, dprev, any_odd, defer);
  if (SMEM) {
    const int cnt = k1 - k0;
#pragma unroll 4
    for (int i = tid; i < cnt; i += NT) {
      double a = sA[i], t = sT[i];
      const double pk = sP[i];
      if (UPDATE) {
        t = EXPR ? advance_exp(t, a, __ldg(rx.lam + k0 + i), rx.t_prev, dprev) : __dadd_rn(t, __dmul_rn(a, dprev));
        sT[i] = t;
        if (full) {
          a = (k0 + i < net.M) ? propensity(net, X, k0 + i) : 0.0;
          sA[i] = a;
        }
      }
      const double d = wt<EXPR>(pk, t, a, k0 + i, rx);
      if (d < best.dt) { best.dt = d; best.k = k0 + i; }
    }
  } else {
    // State streamed from global memory (HBM regime): 4 pairs of reactions per thread and
    // iteration, i.e. twelve 16-byte loads (192 B) in flight per thread before any is used.
    double2 *T2 = reinterpret_cast<double2 *>(T);
    double2 *P2 = reinterpret_cast<double2 *>(P);
    double2 *A2 = reinterpret_cast<double2 *>(A);
    constexpr int U = 4;
    const int q0 = k0 >> 1, q1 = k1 >> 1;
    for (int q = q0 + tid; q < q1; q += U * NT) {
      double2 tt[U], pp[U], aa[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int qu = q + u * NT;
        if (qu < q1) { tt[u] = __ldcg(T2 + qu); pp[u] = __ldcg(P2 + qu); aa[u] = __ldcg(A2 + qu); }
        else { tt[u] = make_double2(0.0, 0.0); pp[u] = tt[u]; aa[u] = tt[u]; }   // a = 0: no candidate
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int qu = q + u * NT;
        if (UPDATE && qu < q1) {
          if (EXPR) {
            tt[u].x = advance_exp(tt[u].x, aa[u].x, __ldg(rx.lam + 2 * qu), rx.t_prev, dprev);
            tt[u].y = advance_exp(tt[u].y, aa[u].y, __ldg(rx.lam + 2 * qu + 1), rx.t_prev, dprev);
          } else {
            tt[u].x = __dadd_rn(tt[u].x, __dmul_rn(aa[u].x, dprev));
            tt[u].y = __dadd_rn(tt[u].y, __dmul_rn(aa[u].y, dprev));
          }
          __stcg(T2 + qu, tt[u]);
          if (full) {
            aa[u].x = (2 * qu < net.M) ? propensity(net, X, 2 * qu) : 0.0;
            aa[u].y = (2 * qu + 1 < net.M) ? propensity(net, X, 2 * qu + 1) : 0.0;
            __stcg(A2 + qu, aa[u]);
          }
        }
        double d = (qu < q1) ? wt<EXPR>(pp[u].x, tt[u].x, aa[u].x, 2 * qu, rx) : best.dt;
        if (d < best.dt) { best.dt = d; best.k = 2 * qu; }
        d = (qu < q1) ? wt<EXPR>(pp[u].y, tt[u].y, aa[u].y, 2 * qu + 1, rx) : best.dt;
        if (d < best.dt) { best.dt = d; best.k = 2 * qu + 1; }
      }
    }
  }
  return best;
}

// Thread (0 .. NT-1) that owns reaction k in scan_own's assignment.
template <int NT, bool SMEM>
__device__ __forceinline__ int owner_thread(int k, int k0) {
  return SMEM ? (k - k0) % NT : ((k - k0) >> 1) % NT;
}



// One dependency entry (32 bytes, see NetDev::dep).
struct DepEnt {
  int4 d;      // k, j1, j2 or -1, sigma1 | sigma2 << 8 | general << 16
  double c;    // c_k
};
__device__ __forceinline__ DepEnt load_dep(const NetDev &net, uint32_t idx) {
  const char *base = reinterpret_cast<const char *>(net.dep) + (size_t)idx * 32;
  DepEnt e;
  e.d = __ldg(reinterpret_cast<const int4 *>(base));
  e.c = __ldg(reinterpret_cast<const double *>(base + 16));
  return e;
}

// Effective rate constant of reaction k under the rate schedule: one rounded product c_k * f.
template <bool SCHED>
__device__ __forceinline__ double eff_rate(const BundleParams &p, int k, double c, double fac) {
  if (SCHED && (p.sched_mask == nullptr || __ldg(p.sched_mask + k))) return __dmul_rn(c, fac);
  return c;
}
__device__ __forceinline__ double propensity_eff(const BundleParams &p, const u64 *X, int k, double fac) {
  return propensity_csr(eff_rate<true>(p, k, __ldg(p.net.rate + k), fac), p.net.react_ptr, p.net.react_species,
                        p.net.react_sigma, X, k);
}

// New propensity of the reaction of entry d = (k, j1, j2, sigma1 | sigma2 << 8 | general << 16)
// with rate c: same operation order as propensity().
__device__ __forceinline__ double propensity_dep(const NetDev &net, const u64 *X, const int4 d, double c) {
  if (d.w & 0x10000)                                    // more than two reactants (rare)
    return propensity_csr(c, net.react_ptr, net.react_species, net.react_sigma, X, d.x);
  const long long x1 = x_load(X, d.y);
  const long long x2 = x_load(X, d.z >= 0 ? d.z : d.y);
  double a = __dmul_rn(c, __ll2double_rn(binom(x1, d.w & 0xff)));
  if (d.z >= 0) a = __dmul_rn(a, __ll2double_rn(binom(x2, (d.w >> 8) & 0xff)));
  return a;
}

// Up to four dependency ranges walked as one flat index space, 128 entries per step so that
// the loads of a whole step (typically of the whole firing) are in flight together.
struct Ranges {
  uint32_t lo[4];
  uint32_t end[4];   // inclusive prefix sums of the range lengths
};

// Scan: visits flat indices [f, end[3]) of rg and compacts the entries with k in [k0, k1) into
// (list_d, list_a = c_k).  Cheap per entry, so the many entries of other CTAs' reactions cost
// little.  Returns true when the staging list filled up (f then tells where to resume).
__device__ __forceinline__ bool walk_scan(const NetDev &net, const Ranges &rg, uint32_t &f, int k0,
                                          int k1, int lane, int &n, int4 *list_d, double *list_a) {
  const uint32_t total = rg.end[3];
  while (f < total) {
    if (n + 128 > kListCap) return true;
    DepEnt ent[4];
    bool in[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const uint32_t fi = f + (uint32_t)(u * 32 + lane);
      const bool valid = fi < total;
      const int e = (fi >= rg.end[0]) + (fi >= rg.end[1]) + (fi >= rg.end[2]);
      const uint32_t beg = e == 0 ? 0u : e == 1 ? rg.end[0] : e == 2 ? rg.end[1] : rg.end[2];
      const uint32_t lo = e == 0 ? rg.lo[0] : e == 1 ? rg.lo[1] : e == 2 ? rg.lo[2] : rg.lo[3];
      ent[u] = load_dep(net, valid ? lo + (fi - beg) : rg.lo[0]);   // idle lanes: a line others load too
      in[u] = valid && ent[u].d.x >= k0 && ent[u].d.x < k1;
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const unsigned m = __ballot_sync(0xffffffffu, in[u]);
      if (in[u]) {
        const int pos = n + __popc(m & ((1u << lane) - 1u));
        list_d[pos] = ent[u].d;
        list_a[pos] = ent[u].c;
      }
      n += __popc(m);
    }
    f += 128u;
  }
  return false;
}

// Finish: new a_k for the n compacted entries (X loads of 32 entries in flight together).
template <bool SCHED>
__device__ __forceinline__ void walk_finish(const BundleParams &p, double fac, const u64 *X, int lane,
                                            int n, const int4 *list_d, int *list_k, double *list_a) {
  __syncwarp();
  for (int i = lane; i < n; i += 32) {
    const int4 d = list_d[i];
    list_k[i] = d.x;
    list_a[i] = propensity_dep(p.net, X, d, eff_rate<SCHED>(p, d.x, list_a[i], fac));
  }
}

// Dependency range of a species given its (lo, hi) or, for hubs, (row of big_off, 0xffffffff):
// hubs are narrowed to the reaction blocks touching [k0, k1).
__device__ __forceinline__ void narrow_range(const NetDev &net, uint32_t &lo, uint32_t &hi, int k0, int k1) {
  if (hi == 0xffffffffu) {
    const uint32_t *off = net.big_off + (size_t)lo * (size_t)(net.n_blk + 1);
    lo = __ldg(off + (k0 >> net.blk_shift));
    hi = __ldg(off + ((k1 - 1) >> net.blk_shift) + 1);
  }
}

// X_j += v for one changed species at firing number `ver` (>= 1).  Returns the new count, or
// -1 if it would leave [0, xmax] (nothing is written then).  `apply` = false: only compute.
__device__ __forceinline__ long long x_peek(const u64 *Xv, int j, int v, u64 ver, long long xmax, bool &done) {
  const u64 w = __ldcg(Xv + j);
  done = x_version(w) == ver;                  // another CTA has already applied this firing
  const long long x = done ? x_count(w) : x_count(w) + (long long)v;
  return (x < 0 || x > xmax) ? -1 : x;
}

// Walker-warp state that outlives a firing: what it has prepared for this CTA's candidate.
struct Spec {
  int pf_k;          // candidate whose walk data was last prefetched into L2
  int k;             // candidate whose redraw is precomputed (lane 0), or -1
  uint32_t n;        //   its new firing count
  double P;          //   its new internal firing time P_k + E(seed, traj, k, n)
  const double *sP;  // shared-memory P (nullptr: state in global memory)
  const double *P_glob;
  int k0, k1;
  u64 seed, traj;
  // pre-walk: the dependency entries of reaction pw_k that fall in [k0, k1), compacted in shared
  // memory (pw_d, pw_c) ahead of time; pw_ent = its stoich row (lanes 0..3).  Network data only,
  // so it stays valid until another reaction is pre-walked.
  int k2;            // runner-up of the last exchange: the likeliest next winner
  int pw_k, pw_n;
  int4 pw_ent;
  int4 *pw_d;
  double *pw_c;
};

// All-gather of the S CTA partials of a bundle (one warp; every lane holds this CTA's partial in
// `c`): through distributed shared memory when the bundle is one cluster, else through the exchange
// slots in L2.  Doubles as the per-firing bundle barrier.  On return every lane holds the
// bundle-wide winner in `c` (c.k == -2: timeout) and the runner-up in `c2`.
// `between` runs after this CTA has posted and before it waits (work hidden behind the exchange).
// DEFER2: `c2` comes back as each lane's contribution to the runner-up; the caller reduces it
// (warp_lexmin) after it has published the winner, off the critical path of the firing.
struct NoWork { __device__ __forceinline__ void operator()() const {} };
template <bool CLUSTER, typename Between = NoWork, bool DEFER2 = false>
__device__ __forceinline__ void exchange_partials(const BundleParams &p, u64 (*cl_slot)[kMaxClusterCtas][2],
                                                  u64 *cl_bar, u64 *exch, int r, uint32_t gen, int lane,
                                                  Cand &c, Cand &c2, Between between = Between()) {
  c2.dt = __longlong_as_double(0x7ff0000000000000ll); c2.k = 0x7fffffff;
  if (CLUSTER && p.S > 1) {
    // One thread-block cluster = one bundle: lane l stores this CTA's partial into slot r of
    // peer l (st.async: the store also completes 16 bytes on the peer's mbarrier), then every
    // CTA waits for its own 16 * S bytes.  No global memory on the path.
    const uint32_t par = gen & 1u, ph = (gen >> 1) & 1u;
    const uint32_t bar = smem_addr(&cl_bar[par]);
    if (lane == 0) mbar_arrive_expect_tx(bar, 16u * (uint32_t)p.S);
    if (lane < p.S)
      st_async_v2(mapa_u32(smem_addr(&cl_slot[par][r][0]), (uint32_t)lane),
                  (u64)__double_as_longlong(c.dt), (u64)(uint32_t)c.k, mapa_u32(bar, (uint32_t)lane));
    between();
    const long long t0 = clock64();
    bool timed_out = false;
    while (!mbar_try_wait(bar, ph))
      if (clock64() - t0 > kSpinLimitCycles) { atomicExch(p.err, 1); timed_out = true; break; }
    Cand s;
    s.dt = __longlong_as_double(0x7ff0000000000000ll); s.k = 0x7fffffff;
    if (lane < p.S) {
      s.dt = __longlong_as_double((long long)cl_slot[par][lane][0]);
      s.k = (int)(uint32_t)cl_slot[par][lane][1];
    }
    c = warp_lexmin(s);
    if (s.k == c.k) { s.dt = __longlong_as_double(0x7ff0000000000000ll); s.k = 0x7fffffff; }
    c2 = DEFER2 ? s : warp_lexmin(s);           // runner-up: best of everything but the winner
    if (__any_sync(0xffffffffu, timed_out)) c.k = -2;
  } else if (p.S > 1) {
    const uint32_t tag = gen + 1u;
    const u64 par = (u64)(((gen >> 1) & 1u) ^ 1u) << 63;     // never matches zeroed memory
    u64 *buf = exch + (size_t)(gen & 1u) * (size_t)p.S * kSlotStride;
    if (lane == 0)
      st_relaxed_v2(buf + (size_t)kSlotStride * r, (u64)__double_as_longlong(c.dt) | par,
                    ((u64)tag << 32) | (u64)(uint32_t)c.k);
    between();
    c.dt = __longlong_as_double(0x7ff0000000000000ll);
    c.k = 0x7fffffff;
    const long long t0 = clock64();
    // Lane l gathers slots l, l+32, ...: all of its loads are in flight together, so the
    // all-gather completes one L2 round trip after the last CTA has posted.
    constexpr int kMaxPer = kMaxBundleCtas / 32;
    unsigned pending = 0;
    for (int i = 0; i < kMaxPer; ++i) if (lane + 32 * i < p.S) pending |= 1u << i;
    while (pending) {
      u64 w0[kMaxPer], w1[kMaxPer];
#pragma unroll
      for (int i = 0; i < kMaxPer; ++i)
        if (pending & (1u << i)) ld_relaxed_v2(buf + (size_t)kSlotStride * (lane + 32 * i), w0[i], w1[i]);
#pragma unroll
      for (int i = 0; i < kMaxPer; ++i)
        if ((pending & (1u << i)) && (uint32_t)(w1[i] >> 32) == tag && (w0[i] >> 63) == (par >> 63)) {
          pending &= ~(1u << i);
          const double dt = __longlong_as_double((long long)(w0[i] & 0x7fffffffffffffffull));
          const int k = (int)(uint32_t)(w1[i] & 0x7fffffffu);
          if (cand_less(dt, k, c)) { c2 = c; c.dt = dt; c.k = k; }
          else if (cand_less(dt, k, c2)) { c2.dt = dt; c2.k = k; }
        }
      if (pending && clock64() - t0 > kSpinLimitCycles) { atomicExch(p.err, 1); c.k = -2; break; }
    }
    const bool timed_out = __any_sync(0xffffffffu, c.k == -2);
    const Cand mine_best = c;
    c = warp_lexmin(c);
    // runner-up = best of everything but the winner: the likeliest winner of the next firing
    c2 = (mine_best.k == c.k) ? c2 : mine_best;
    if (!DEFER2) c2 = warp_lexmin(c2);
    if (timed_out) c.k = -2;
  }
}

// Named barriers of the kernel: 0 = __syncthreads; 1 = the stream warps among themselves; 2 = warp 0
// hands the winner to the walker warp; 3 = the walker's staged refreshes are ready (kBarStaged);
// 4 = the stream warps' partials are ready for the walker (kBarParts).
constexpr int kBarStaged = 3, kBarParts = 4;
template <int COUNT> __device__ __forceinline__ void named_sync(int id) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "n"(COUNT) : "memory");
}
template <int COUNT> __device__ __forceinline__ void named_arrive(int id) {
  __threadfence_block();
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "n"(COUNT) : "memory");
}

// Pre-walk of the runner-up k2 (walker warp): row -> ranges -> this CTA's dependency entries, into
// pw_d / pw_c.  Network data only, so it stays valid until another reaction is pre-walked.
__device__ __forceinline__ void prewalk(const BundleParams &p, Spec &spec, int lane);

// Block-wide lexmin of the thread candidates, then all-gather of the S CTA partials (exchange_partials,
// which is also the per-firing bundle barrier).  Every thread returns the
// bundle-wide winner.  win.k == -2 signals a timeout.
// FREE: the walker warp runs ahead of the stream warps (see the kernel): it does not post a partial
// and pre-walks BEFORE it waits for the stream warps' partials.
template <int BLOCK, bool PREWALK, bool CLUSTER, bool FREE>
__device__ __forceinline__ Cand bundle_argmin(const BundleParams &p, BundleCtx<BLOCK> &ctx,
                                              u64 *exch, const uint32_t *nfire, int r,
                                              uint32_t &gen, Cand mine, Spec &spec) {
  constexpr int NT = BLOCK - 32 * kWalkerWarps;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool walker = warp == BLOCK / 32 - 1;
  if (!walker) {
    mine = warp_lexmin(mine);
    if (lane == 0) ctx.warp_part[warp] = mine;
  }
  if (FREE) {
    if (walker) {
      if (PREWALK && (p.prefetch & 4)) prewalk(p, spec, lane);
      named_sync<BLOCK>(kBarParts);
    } else {
      named_sync<NT>(1);
      named_arrive<BLOCK>(kBarParts);
    }
  } else {
    __syncthreads();
  }
  if (warp == 0) {
    Cand c = ctx.warp_part[lane];                 // NT / 32 <= 32 partials
    if (lane >= NT / 32) { c.dt = __longlong_as_double(0x7ff0000000000000ll); c.k = 0x7fffffff; }
    c = warp_lexmin(c);
    Cand c2;                                      // this lane's second-best slot (runner-up search)
    c2.dt = __longlong_as_double(0x7ff0000000000000ll); c2.k = 0x7fffffff;
    exchange_partials<CLUSTER>(p, ctx.cl_slot, ctx.cl_bar, exch, r, gen, lane, c, c2);
    if (lane == 0) { ctx.win = c; ctx.second_k = (c2.dt < __longlong_as_double(0x7ff0000000000000ll)) ? c2.k : 0x7fffffff; }
  } else if (walker) {
    // Walker warp, idle during the exchange.  If this CTA's candidate wins (it usually stays the
    // candidate for many firings before it does), this CTA must redraw P_k (Philox + log, the
    // longest serial piece of a firing) and every CTA will need the candidate's stoich row and
    // the dependency entries of its species, all DRAM-cold (each reaction fires rarely).
    // Do the redraw now, speculatively, and pull the rest into L2 -- once per candidate.
    Cand c = ctx.warp_part[lane];
    if (lane >= NT / 32) { c.dt = __longlong_as_double(0x7ff0000000000000ll); c.k = 0x7fffffff; }
    c = warp_lexmin(c);
    if (!FREE && PREWALK && (p.prefetch & 4)) prewalk(p, spec, lane);
    if (c.k < p.net.M && c.k != spec.k && lane == 0 && (p.prefetch & 2)) {
      const uint32_t n1 = nfire[c.k] + 1u;
      if (p.formulation) {
        spec.P = -exp_draw(spec.seed, spec.traj, (uint32_t)c.k, n1);       // residual form: T_k = -E
      } else {
        const double pold = spec.sP ? spec.sP[c.k - spec.k0] : __ldcg(spec.P_glob + c.k);
        spec.P = __dadd_rn(pold, exp_draw(spec.seed, spec.traj, (uint32_t)c.k, n1));
      }
      spec.n = n1;
      spec.k = c.k;
    }
    if (c.k != spec.pf_k && c.k < p.net.M && (p.prefetch & 1)) {
      spec.pf_k = c.k;
      int4 ent = make_int4(-1, 0, 0, 0);
      if (lane < 4) ent = __ldg(reinterpret_cast<const int4 *>(p.net.srow) + (size_t)c.k * 4 + lane);
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int j = __shfl_sync(0xffffffffu, ent.x, e);
        const uint32_t lo = (uint32_t)__shfl_sync(0xffffffffu, ent.z, e);
        const uint32_t hi = (uint32_t)__shfl_sync(0xffffffffu, ent.w, e);
        if (j >= 0 && hi != 0xffffffffu)            // hubs stay hot by themselves
          for (uint32_t i = lo + 4u * lane; i < hi; i += 128u)
            prefetch_l2(reinterpret_cast<const char *>(p.net.dep) + (size_t)i * 32);
      }
    }
  }
  gen += 1u;
  // The stream warps leave as soon as warp 0 has the winner; the walker warp, which may still
  // be busy with its speculative work, pairs with warp 0 on a barrier of its own.
  if (warp == 0) asm volatile("bar.arrive 2, 64;" ::: "memory");
  if (walker) { asm volatile("bar.sync 2, 64;" ::: "memory"); spec.k2 = ctx.second_k; }
  else asm volatile("bar.sync 1, %0;" ::"r"(NT) : "memory");
  return ctx.win;
}

__device__ __forceinline__ void prewalk(const BundleParams &p, Spec &spec, int lane) {
  if (spec.k2 == spec.pw_k || spec.k2 >= p.net.M || spec.k1 <= spec.k0) return;
  const int k2 = spec.k2;
  int4 ent = make_int4(-1, 0, 0, 0);
  if (lane < 4) ent = __ldg(reinterpret_cast<const int4 *>(p.net.srow) + (size_t)k2 * 4 + lane);
  spec.pw_k = -1;
  if (__shfl_sync(0xffffffffu, ent.x, 0) == -2) return;     // more than 4 changed species: CSR walk
  uint32_t lo = 0, hi = 0;
  if (ent.x >= 0) { lo = (uint32_t)ent.z; hi = (uint32_t)ent.w; narrow_range(p.net, lo, hi, spec.k0, spec.k1); }
  Ranges rg;
  uint32_t acc = 0;
#pragma unroll
  for (int e = 0; e < 4; ++e) {
    rg.lo[e] = __shfl_sync(0xffffffffu, lo, e);
    acc += __shfl_sync(0xffffffffu, hi - lo, e);
    rg.end[e] = acc;
  }
  uint32_t f = 0;
  int n = 0;
  if (!walk_scan(p.net, rg, f, spec.k0, spec.k1, lane, n, spec.pw_d, spec.pw_c)) {
    spec.pw_k = k2; spec.pw_n = n; spec.pw_ent = ent;
  }
}


// Fenced barrier over the CTAs of a bundle (start and end of a trajectory): all earlier global
// writes of every CTA are visible to all later reads of every CTA.  Uses the exchange slots and
// generation counter of bundle_argmin.  Returns false on a timeout.
template <int BLOCK, bool CLUSTER>
__device__ __noinline__ bool bundle_barrier(u64 *exch, int S, int r, uint32_t gen, int *err) {
  __threadfence();
  if (CLUSTER) {                                  // the bundle is one cluster: hardware barrier
    cluster_barrier();
    __threadfence();
    return true;
  }
  __syncthreads();
  bool ok = true;
  if (threadIdx.x < 32 && S > 1) {
    const int lane = threadIdx.x;
    const uint32_t tag = gen + 1u;
    const u64 par = (u64)(((gen >> 1) & 1u) ^ 1u) << 63;
    u64 *buf = exch + (size_t)(gen & 1u) * (size_t)S * kSlotStride;
    if (lane == 0) st_relaxed_v2(buf + (size_t)kSlotStride * r, par | 0x7ff0000000000000ull, ((u64)tag << 32) | 0x7fffffffull);
    const long long t0 = clock64();
    for (int s = lane; s < S; s += 32) {
      u64 w0, w1;
      for (;;) {
        ld_relaxed_v2(buf + (size_t)kSlotStride * s, w0, w1);
        if ((uint32_t)(w1 >> 32) == tag && (w0 >> 63) == (par >> 63)) break;
        if (clock64() - t0 > kSpinLimitCycles) { atomicExch(err, 1); ok = false; break; }
      }
      if (!ok) break;
    }
  }
  ok = __syncthreads_and(ok ? 1 : 0) != 0;
  __threadfence();
  return ok;
}

// FULL = refresh_mode 1 (recompute every a_k each firing, the paper's own GPU scheme) is a separate
// instantiation so that its code stays out of the instruction stream of the default kernel.
// RATE = 1: a piecewise-constant rate schedule is set; RATE = 2: exponential rates c_k exp(lambda_k t)
// (time-dependent rates, Eq.28): also their own instantiations.
// CLUSTER: the launch makes each bundle one thread-block cluster (S <= kMaxClusterCtas): the
// exchange goes through distributed shared memory and `exch` is not used.
template <int BLOCK, bool SMEM, bool FULL, int RATE, bool CLUSTER = false>
__global__ void __launch_bounds__(BLOCK, 1) rt_bundle_kernel(const BundleParams p) {
  constexpr bool SCHED = RATE == 1, EXPR = RATE == 2;
  constexpr int NT = BLOCK - 32 * kWalkerWarps;      // stream threads; the last warp walks
  // FREE: the walker warp only ANNOUNCES its staged refreshes (bar.arrive) and runs ahead into the
  // pre-walk of the likely next winner while the stream warps apply them, re-scan and reduce; the
  // stream warps never wait for it except for the refreshes themselves.
  constexpr bool FREE = SMEM && !FULL;
  __shared__ BundleCtx<BLOCK> ctx;
  __shared__ int list_k[kListCap];
  __shared__ int4 list_d[kListCap];
  __shared__ int4 pw_d[SMEM ? kListCap : 1];
  __shared__ double pw_c[SMEM ? kListCap : 1];
  __shared__ double list_a[kListCap];
  __shared__ unsigned char dirty[BLOCK];
  __shared__ int mybest_k[BLOCK];                    // reaction each stream thread proposes (-3: undecided)
  __shared__ Cand redo[SMEM ? 1 : BLOCK];            // global-memory state: cooperative re-scan results
  __shared__ short stale_list[SMEM ? 1 : BLOCK];
  extern __shared__ __align__(16) unsigned char dyn_smem[];
  const NetDev &net = p.net;
  const int tid = threadIdx.x, lane = tid & 31;
  const bool is_walker = tid >= NT;
  const int b = blockIdx.x / p.S, r = blockIdx.x % p.S;
  const int M = net.M, N = net.N;
  const double INF = __longlong_as_double(0x7ff0000000000000ll);
  const bool resid = p.formulation != 0;

  double *T = p.T + (size_t)b * net.M_pad;
  double *P = p.P + (size_t)b * net.M_pad;
  double *A = p.a + (size_t)b * net.M_pad;
  uint32_t *nfire = p.n + (size_t)b * net.M_pad;
  const int xg = r % p.G;                                      // X replica of this CTA
  u64 *X = p.X + ((size_t)b * p.G + xg) * (size_t)N;
  u64 *exch = p.exch + (size_t)b * 2 * p.S * kSlotStride;

  const int pairs_total = net.M_pad / 2;
  const int q0 = min(r * p.pairs_per_cta, pairs_total);
  const int q1 = min(q0 + p.pairs_per_cta, pairs_total);
  const int k0 = 2 * q0, k1 = 2 * q1;
  double *sT = reinterpret_cast<double *>(dyn_smem);
  const int cnt_pad = p.cnt_pad;
  double *sP = sT + (SMEM ? cnt_pad : 0);
  double *sA = sP + (SMEM ? cnt_pad : 0);

  uint32_t gen = 0;   // exchange generation, identical in every CTA of the bundle
  Spec spec;
  spec.pf_k = -1; spec.k = -1; spec.n = 0u; spec.P = 0.0;
  spec.k2 = 0x7fffffff; spec.pw_k = -1; spec.pw_n = 0; spec.pw_ent = make_int4(-1, 0, 0, 0);
  spec.pw_d = pw_d; spec.pw_c = pw_c; spec.k1 = 0;
  spec.sP = nullptr; spec.P_glob = nullptr; spec.k0 = 0; spec.seed = p.seed; spec.traj = 0;
  dirty[tid] = 0;
  if (tid == 0) { ctx.abort_local = 0; ctx.list_n = 0; ctx.more = 0; ctx.p_k = -1; ctx.any_odd = 0; }
  if (CLUSTER && tid == 0) {     // (peers touch them only after the first bundle_barrier)
    mbar_init(smem_addr(&ctx.cl_bar[0]), 1u);
    mbar_init(smem_addr(&ctx.cl_bar[1]), 1u);
    mbar_fence_init();
  }
  __syncthreads();
  Cand none; none.dt = INF; none.k = 0x7fffffff;

  for (u64 it = (u64)b; it < p.n_traj; it += (u64)p.B) {
    const u64 traj = p.traj_first + it;
    spec.k = -1; spec.traj = traj; spec.sP = SMEM ? sP : nullptr; spec.P_glob = P; spec.k0 = k0; spec.k1 = k1;
    spec.k2 = 0x7fffffff;
    const bool tracing = (it == 0) && p.trace_cap > 0 && r == 0;

    // ---- a-0: X = x0 (slices, version 0), then T = 0, P = E(k,0), a = a(X0), n = 0 for the own range
    for (int j = (r / p.G) * BLOCK + tid; j < N; j += ((p.S - xg + p.G - 1) / p.G) * BLOCK)
      __stcg(X + j, x_pack(0ull, p.x0[j]));
    if (!bundle_barrier<BLOCK, CLUSTER>(exch, p.S, r, gen, p.err)) return;
    if (!CLUSTER) gen += 1u;     // (a cluster's gen counts exchanges only: it is the mbarrier phase)
    for (int k = k0 + tid; k < (SMEM ? k0 + cnt_pad : k1); k += BLOCK) {
      double a0 = 0.0, p0 = 1.0;     // padding: a = 0, P - T = 1 > 0, so its q~ is +inf, never NaN
      double t_init = 0.0, p_init = 1.0;
      uint32_t n_init = 0u;
      if (k < k1 && k < M) {
        a0 = propensity(net, X, k);
        if (filter_unsafe(a0)) ctx.any_odd = 1;
        if (p.T0) {                                   // resume: the checkpointed internal times
          t_init = __ldg(p.T0 + k); p_init = __ldg(p.P0 + k); n_init = __ldg(p.n0 + k);
        } else {
          p0 = exp_draw(p.seed, traj, (uint32_t)k, 0u);
          t_init = resid ? -p0 : 0.0; p_init = resid ? 0.0 : p0;            // residual form: T = -R
        }
      } else if (resid) { t_init = -1.0; p_init = 0.0; }
      if (SMEM) { sT[k - k0] = t_init; sP[k - k0] = p_init; sA[k - k0] = a0; }
      else { __stcg(T + k, t_init); __stcg(P + k, p_init); __stcg(A + k, a0); }
      if (k < k1) nfire[k] = n_init;
    }
    __syncthreads();

    double t = p.t0, dprev = 0.0;
    RateExp rx;                          // (EXPR only)
    rx.lam = p.rate_lambda; rx.t_now = t; rx.t_prev = t;
    u64 fired = 0;
    int mu_prev = -1, stop = 0, status = RT_OK;
    bool finishing = false;
    double fac = 1.0, fac_next = 1.0;   // rate schedule: current factor, factor after the breakpoint
    int seg = 0;                        //   breakpoints passed
    bool rate_change = false;           //   this pass ends at a breakpoint: recompute every a_k
    constexpr bool full = FULL;

    for (;;) {   // one iteration per firing, plus one closing pass
      // walker-warp state of this firing (uniform over the warp)
      Ranges rg;
#pragma unroll
      for (int e = 0; e < 4; ++e) { rg.lo[e] = 0; rg.end[e] = 0; }
      uint32_t w_f = 0;         // flat position inside rg
      int w_e = 0, w_ne = 0;    // CSR rows (more than 4 changed species): species cursor / count
      uint32_t w_e0 = 0;
      bool w_csr = false;
      int pre_n = -1;           // >= 0: the pre-walk hit, list_k / list_a already hold pre_n refreshes
      Cand best = none;
      Cand extra = none;        // fresh waiting times of refreshed reactions this thread stored

      if (is_walker && lane == 0) ctx.p_k = -1;   // (re)set below by the owner of the fired reaction
      if (is_walker && mu_prev >= 0) {
        // ===== walker warp: discrete updates of the previous firing (a-6, a-7, a-8) =====
        const bool owner = (mu_prev >= k0 && mu_prev < k1);
        uint32_t c_old = 0; double p_old = 0.0;
        const bool have_spec = (spec.k == mu_prev);          // lane 0: redraw precomputed
        if (owner && lane == 0 && !have_spec) {
          c_old = nfire[mu_prev];
          p_old = SMEM ? sP[mu_prev - k0] : __ldcg(P + mu_prev);
        }
        const bool hit = SMEM && !full && spec.pw_k == mu_prev;   // (pre-walk: shared-memory state only)      // pre-walked while the exchange ran
        int4 ent = spec.pw_ent;                 // lane e < 4: (j, v, lo, hi) of the e-th changed species
        if (!hit) {
          ent = make_int4(-1, 0, 0, 0);
          if (lane < 4) ent = __ldg(reinterpret_cast<const int4 *>(net.srow) + (size_t)mu_prev * 4 + lane);
        }
        w_csr = __shfl_sync(0xffffffffu, ent.x, 0) == -2;
        if (hit) {
          // One L2 round trip: the X words of the changed species and of the reactants of the
          // first 32 pre-walked entries are loaded together; a word that does not yet carry this
          // firing's version is brought up to date locally (X_j + v_j).
          const bool active = ent.x >= 0;
          const bool has0 = lane < spec.pw_n;
          int4 d0 = make_int4(0, 0, -1, 0);
          double c0 = 0.0;
          u64 w1 = 0, w2 = 0;
          if (has0) {
            d0 = pw_d[lane]; c0 = pw_c[lane];
            w1 = __ldcg(X + d0.y);
            w2 = __ldcg(X + (d0.z >= 0 ? d0.z : d0.y));
          }
          bool done = false;
          long long xn = 0;
          if (active) xn = x_peek(X, ent.x, ent.y, fired, net.xmax, done);
          const bool bad = __any_sync(0xffffffffu, active && xn < 0);
          if (bad) { if (lane == 0) ctx.abort_local = 1; }
          else if (active && !done) atomicMax(X + ent.x, x_pack(fired, xn));
          long long x1 = x_count(w1), x2 = x_count(w2);
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int je = __shfl_sync(0xffffffffu, ent.x, e);
            const long long ve = (long long)__shfl_sync(0xffffffffu, ent.y, e);
            if (je == d0.y && x_version(w1) != fired) x1 += ve;
            if (je == d0.z && x_version(w2) != fired) x2 += ve;
          }
          __syncwarp();
          if (has0) {
            c0 = eff_rate<SCHED>(p, d0.x, c0, fac);
            double a = __dmul_rn(c0, __ll2double_rn(binom(x1, d0.w & 0xff)));
            if (d0.z >= 0) a = __dmul_rn(a, __ll2double_rn(binom(x2, (d0.w >> 8) & 0xff)));
            if (d0.w & 0x10000)                                     // > 2 reactants: after the update
              a = propensity_csr(c0, net.react_ptr, net.react_species, net.react_sigma, X, d0.x);
            list_k[lane] = d0.x;
            list_a[lane] = a;
          }
          for (int i = lane + 32; i < spec.pw_n; i += 32) {        // more than 32: plain path
            const int4 d = pw_d[i];
            list_k[i] = d.x;
            list_a[i] = propensity_dep(net, X, d, eff_rate<SCHED>(p, d.x, pw_c[i], fac));
          }
          pre_n = spec.pw_n;
        } else if (!w_csr) {
          // a-6: X += v_mu (Eq.5); nothing is written if any count would leave [0, xmax]
          const bool active = ent.x >= 0;
          bool done = false;
          long long xn = 0;
          uint32_t lo = 0, hi = 0;
          if (active && !full && k1 > k0) {        // (hub: two loads, in flight with the X word)
            lo = (uint32_t)ent.z; hi = (uint32_t)ent.w;
            narrow_range(net, lo, hi, k0, k1);
          }
          if (active) xn = x_peek(X, ent.x, ent.y, fired, net.xmax, done);
          const bool bad = __any_sync(0xffffffffu, active && xn < 0);
          if (bad) { if (lane == 0) ctx.abort_local = 1; }
          else if (active && !done) atomicMax(X + ent.x, x_pack(fired, xn));
          uint32_t acc = 0;
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            rg.lo[e] = __shfl_sync(0xffffffffu, lo, e);
            acc += __shfl_sync(0xffffffffu, hi - lo, e);
            rg.end[e] = acc;
          }
        } else {
          // rows with more than 4 changed species: plain CSR walk (rare, correctness path)
          w_e0 = __ldg(net.stoich_ptr + mu_prev);
          w_ne = (int)(__ldg(net.stoich_ptr + mu_prev + 1) - w_e0);
          bool bad_l = false;
          for (int e = lane; e < w_ne; e += 32) {
            bool done;
            bad_l |= x_peek(X, __ldg(net.stoich_species + w_e0 + e), __ldg(net.stoich_v + w_e0 + e),
                            fired, net.xmax, done) < 0;
          }
          if (__any_sync(0xffffffffu, bad_l)) {
            if (lane == 0) ctx.abort_local = 1;
          } else {
            for (int e = lane; e < w_ne; e += 32) {
              bool done;
              const int j = __ldg(net.stoich_species + w_e0 + e);
              const long long xn = x_peek(X, j, __ldg(net.stoich_v + w_e0 + e), fired, net.xmax, done);
              if (!done) atomicMax(X + j, x_pack(fired, xn));
            }
          }
          if (full || k1 <= k0) w_ne = 0;
        }
        if (lane == 0) {
          if (owner) {                           // a-7: new internal firing time of mu (Eq.26)
            if (have_spec) {
              nfire[mu_prev] = spec.n;
              ctx.p_val = spec.P;
            } else {
              nfire[mu_prev] = c_old + 1u;
              const double e_new = exp_draw(p.seed, traj, (uint32_t)mu_prev, c_old + 1u);
              ctx.p_val = resid ? -e_new : __dadd_rn(p_old, e_new);
            }
            ctx.p_k = mu_prev;
            spec.k = -1;
          }
          if (tracing && fired - 1 < p.trace_cap) {   // a-8
            if (p.trace_mu) p.trace_mu[fired - 1] = mu_prev;
            if (p.trace_t) p.trace_t[fired - 1] = t;
          }
        }
        __syncwarp();                            // this warp's X updates precede its reads below
      }
      if (full && mu_prev >= 0) __syncthreads(); // full recompute reads the new X in the stream

      bool first_round = true;
      for (;;) {   // rounds: one, unless this CTA has more than kListCap refreshes
        if (is_walker) {
          // ===== walker warp: dependency walk (a-1 for k in D(mu) that fall in [k0, k1)) =====
          int n = 0;
          bool more = false;
          if (pre_n >= 0) {
            n = first_round ? pre_n : 0;
          } else if (!w_csr) {
            more = walk_scan(net, rg, w_f, k0, k1, lane, n, list_d, list_a);
          } else {
            while (w_e < w_ne) {
              if (w_f == 0) {                    // entering species w_e: fetch its range
                const int j = __ldg(net.stoich_species + w_e0 + w_e);
                const uint2 rec = __ldg(reinterpret_cast<const uint2 *>(net.sp_rec) + j);
                uint32_t lo = rec.x, hi = rec.y;
                if (hi - lo > (uint32_t)net.big_deg) { lo = (uint32_t)__ldg(net.sp_big + j); hi = 0xffffffffu; }
                narrow_range(net, lo, hi, k0, k1);
                rg.lo[0] = lo;
                rg.end[0] = rg.end[1] = rg.end[2] = rg.end[3] = hi - lo;
              }
              more = walk_scan(net, rg, w_f, k0, k1, lane, n, list_d, list_a);
              if (more) break;
              w_e += 1;
              w_f = 0;
            }
          }
          if (pre_n < 0) walk_finish<SCHED>(p, fac, X, lane, n, list_d, list_k, list_a);
          if (lane == 0) { ctx.list_n = n; ctx.more = more ? 1 : 0; }
          if (FREE && !more && !(SCHED && rate_change)) {      // run ahead (see FREE)
            named_arrive<BLOCK>(kBarStaged);
            break;
          }
        } else if (first_round) {
          // ===== stream warps: a-5 of the previous firing fused with a-2/a-3 of this one =====
          bool defer = false;
          best = scan_own<NT, SMEM, true, EXPR>(net, X, tid, k0, k1, sT, sP, sA, T, P, A, dprev, full, cnt_pad,
                                                ctx.any_odd != 0, defer, resid, rx);
          mybest_k[tid] = defer ? -3 : best.k;
          if (defer) dirty[tid] = 1;
        }
        if (FREE) named_sync<BLOCK>(kBarStaged); else __syncthreads();
        // ----- apply the staged refreshes; mark the owning threads for a re-scan
        const int n = ctx.list_n;
        const bool more = ctx.more != 0;
        // A refreshed reaction invalidates its owner's proposal only if it IS that proposal (the
        // proposal is the minimum over the owner's other, unchanged reactions as well).  Then the
        // owner re-scans; otherwise the new waiting time simply joins the reduction as one more
        // candidate.  The reaction that fired (new P) always sends its owner to the re-scan.
        const int pk_now = ctx.p_k;
        for (int i = tid; i < n && !(FREE && is_walker); i += (FREE ? NT : BLOCK)) {
          const int k = list_k[i];
          const double a_new = list_a[i];
          if (SMEM) sA[k - k0] = a_new; else __stcg(A + k, a_new);
          if (filter_unsafe(a_new)) ctx.any_odd = 1;
          const int o = owner_thread<NT, SMEM>(k, k0);
          if (mybest_k[o] == k || mybest_k[o] == -3 || k == pk_now) {
            dirty[o] = 1;
          } else {
            const double d = wt<EXPR>(SMEM ? sP[k - k0] : __ldcg(P + k),
                                      SMEM ? sT[k - k0] : __ldcg(T + k), a_new, k, rx);
            if (cand_less(d, k, extra)) { extra.dt = d; extra.k = k; }
          }
        }
        if (tid == 0) {
          if (first_round && pk_now >= 0) {
            if (resid) { if (SMEM) sT[pk_now - k0] = ctx.p_val; else __stcg(T + pk_now, ctx.p_val); }
            else { if (SMEM) sP[pk_now - k0] = ctx.p_val; else __stcg(P + pk_now, ctx.p_val); }
            dirty[owner_thread<NT, SMEM>(pk_now, k0)] = 1;
          }
          ctx.n_stale = 0;
        }
        if (FREE && !more && !(SCHED && rate_change)) named_sync<NT>(1);   // (the walker is not here)
        else __syncthreads();
        if (!more) break;
        first_round = false;
      }
      if (SCHED && rate_change) {
        // the pass above brought every T_k to the breakpoint with the old rates; now switch
        rate_change = false;
        fac = fac_next;
        for (int k = k0 + tid; k < k1; k += BLOCK)
          if (k < M) {
            const double a_new = propensity_eff(p, X, k, fac);
            if (SMEM) sA[k - k0] = a_new; else __stcg(A + k, a_new);
            if (filter_unsafe(a_new)) ctx.any_odd = 1;
          }
        dirty[tid] = 0;
        __syncthreads();
        if (!is_walker) {
          bool defer = false;
          best = scan_own<NT, SMEM, false>(net, X, tid, k0, k1, sT, sP, sA, T, P, A, 0.0, false, cnt_pad,
                                           ctx.any_odd != 0, defer, resid);
        }
      } else if (SMEM) {
        // re-scan (read-only) with the new a_k, P_mu.  Stale threads are few (usually one, in the
        // CTA that owns the fired reaction, which is then the last to post), so the thread's warp
        // shares its reactions: one exact division per lane instead of a serial pass.
        if (!is_walker) {
          unsigned stale_mask = __ballot_sync(0xffffffffu, dirty[tid] != 0);
          if (dirty[tid]) dirty[tid] = 0;
          if (cnt_pad <= 32 * NT) {
            while (stale_mask) {
              const int L = __ffs(stale_mask) - 1;
              stale_mask &= stale_mask - 1;
              const int i = (tid - lane + L) + lane * NT;      // lane j: the thread's j-th reaction
              Cand c = none;
              if (i < cnt_pad) { c.dt = wt<EXPR>(sP[i], sT[i], sA[i], min(k0 + i, net.M_pad - 1), rx); c.k = k0 + i; }
              c = warp_lexmin(c);
              if (lane == L) best = c;
            }
          } else if (stale_mask & (1u << lane)) {
            bool defer = false;
            best = scan_own<NT, SMEM, false, EXPR>(net, X, tid, k0, k1, sT, sP, sA, T, P, A, 0.0, false, cnt_pad,
                                                   ctx.any_odd != 0, defer, false, rx);
          }
        }
      } else {
        // State in global memory: one thread re-reading its ~130 strided reactions is a chain of
        // DRAM latencies (17 us on cfg5a).  The whole CTA shares the work instead: each warp takes
        // one stale thread's reactions, 32 pairs at a time.
        const bool was_stale = !is_walker && dirty[tid];
        if (was_stale) { dirty[tid] = 0; stale_list[atomicAdd(&ctx.n_stale, 1)] = (short)tid; }
        __syncthreads();
        const int n_stale = ctx.n_stale;
        if (n_stale > 0) {
          const double2 *T2 = reinterpret_cast<const double2 *>(T);
          const double2 *P2 = reinterpret_cast<const double2 *>(P);
          const double2 *A2 = reinterpret_cast<const double2 *>(A);
          for (int sidx = tid >> 5; sidx < n_stale; sidx += BLOCK / 32) {
            const int d = stale_list[sidx];
            Cand c = none;
            for (int q = (k0 >> 1) + d + lane * NT; q < (k1 >> 1); q += 32 * NT) {
              const double2 t2 = __ldcg(T2 + q), p2 = __ldcg(P2 + q), a2 = __ldcg(A2 + q);
              double w = wt<EXPR>(p2.x, t2.x, a2.x, 2 * q, rx);
              if (cand_less(w, 2 * q, c)) { c.dt = w; c.k = 2 * q; }
              w = wt<EXPR>(p2.y, t2.y, a2.y, 2 * q + 1, rx);
              if (cand_less(w, 2 * q + 1, c)) { c.dt = w; c.k = 2 * q + 1; }
            }
            c = warp_lexmin(c);
            if (lane == 0) redo[d] = c;
          }
          __syncthreads();
          if (was_stale) best = redo[tid];
        }
      }
      if (cand_less(extra.dt, extra.k, best)) best = extra;
      if (ctx.abort_local) { status = RT_ERR_OVERFLOW; stop = 0; break; }
      if (finishing) break;

      // ---- a-3 argmin over the bundle
      const Cand win = bundle_argmin<BLOCK, SMEM, CLUSTER, FREE>(p, ctx, exch, nfire, r, gen, best, spec);
      if (win.k == -2) return;

      // ---- a-4 stop tests, identical in every thread of every CTA of the bundle
      const double delta = win.dt;
      if (SCHED) {
        // Eq.28 with piecewise-constant c_k(t): a step that would cross the next breakpoint is cut
        // there -- T_k += a_k (b - t), t = b, no firing -- and the rates switch.
        const double tb = (seg < p.sched_n && __ldg(p.sched_t + seg) <= p.t_end) ? __ldg(p.sched_t + seg) : INF;
        if (tb < INF && (delta == INF || __dadd_rn(t, delta) > tb)) {
          dprev = __dsub_rn(tb, t);
          t = tb;
          mu_prev = -1;
          fac_next = __ldg(p.sched_f + seg);
          seg += 1;
          rate_change = true;
          continue;
        }
      }
      if (delta == INF) { stop = RT_STOP_ABSORBED; break; }
      if (p.t_end < INF && __dadd_rn(t, delta) > p.t_end) {
        dprev = __dsub_rn(p.t_end, t);           // closing pass: T_k += a_k * (t_end - t), no firing
        rx.t_prev = t; rx.t_now = p.t_end;
        t = p.t_end;
        mu_prev = -1;
        stop = RT_STOP_T_END;
        finishing = true;
        continue;
      }
      if (fired >= kXMaxVersion) { status = RT_ERR_OVERFLOW; break; }   // firing counter exhausted
      rx.t_prev = t;
      t = __dadd_rn(t, delta);
      rx.t_now = t;
      fired += 1;
      mu_prev = win.k;
      dprev = delta;
      if (p.max_firings != 0 && fired == p.max_firings) {
        stop = RT_STOP_MAX_FIRINGS;              // closing pass applies this firing's updates
        finishing = true;
      }
    }

    // ---- trajectory done: every CTA's X updates are visible bundle-wide after the fenced barrier
    if (!bundle_barrier<BLOCK, CLUSTER>(exch, p.S, r, gen, p.err)) return;
    if (!CLUSTER) gen += 1u;
    dirty[tid] = 0;
    if (SMEM)
      for (int k = k0 + tid; k < k1; k += BLOCK) {
        __stcg(T + k, sT[k - k0]); __stcg(P + k, sP[k - k0]); __stcg(A + k, sA[k - k0]);
      }
    if (p.x_out)
      for (int j = r * BLOCK + tid; j < N; j += p.S * BLOCK)
        p.x_out[it * (u64)N + (u64)j] = x_load(X, j);
    if (r == 0 && tid == 0) {
      rt_result res;
      res.t = t; res.firings = fired; res.stop = stop; res.status = status;
      p.res[it] = res;
    }
    if (tid == 0) { ctx.abort_local = 0; ctx.p_k = -1; ctx.any_odd = 0; }
    __syncthreads();
  }
}

}  // namespace rt
