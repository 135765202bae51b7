// rt_bundle.cuh -- persistent "bundle" kernel: a group of S CTAs (the paper's bundle =
// "a batch of blocks" holding one trajectory) simulates one trajectory after
// another; B bundles run side by side.  One launch covers every firing of every trajectory, so
// launch latency never sits between firings.
//
// Per firing, each CTA owns a fixed contiguous range of reactions and does ONE streaming pass
// over its (T, P, a) triples (structure-of-arrays fp64, 16-byte vector accesses):
//     T_k += |a_k| * dt_prev            internal-time increment of the PREVIOUS firing (Eq.15)
//     dt_k = (P_k - T_k) / a_k          waiting time for THIS firing (Eq.24), +inf if a_k <= 0
//     thread-local lexicographic min    (Eq.25, ties to the lowest k)
// i.e. 24 B read + 8 B written per reaction per firing.  Reactions whose propensity changes
// (the dependency lists of the fired reaction) are excluded from the stream by
// storing -|a_k| (sign bit = "refresh pending"): the stream still advances their T_k with the
// OLD propensity -- the one that held during the elapsed interval -- and yields +inf for them;
// a fix-up step then recomputes a_k from the new X and contributes their candidates.
// The CTA partials are combined by an all-gather through L2 (one 16-byte slot per CTA,
// self-validating words, double-buffered), which doubles as the per-firing bundle barrier.
#pragma once
#include "rt_device.cuh"
#include "../../include/rt.h"

namespace rt {

struct BundleParams {
  NetDev net;
  double *T, *P, *a;      // [B][M_pad]
  uint32_t *n;            // [B][M_pad]  firings per reaction
  long long *X;           // [B][N]
  u64 *exch;              // [B][2][S][2] exchange slots, zeroed before launch
  uint32_t *xgen;         // [B][32]     X generation counters (128 B apart), zeroed before launch
  int S, B;
  int pairs_per_cta;
  const long long *x0;    // [N]
  u64 seed, traj_first, n_traj, max_firings;
  double t_end;
  long long *x_out;       // [n_traj][N] or nullptr
  rt_result *res;         // [n_traj]
  int32_t *trace_mu;      // first trajectory of the launch only; may be nullptr
  double *trace_t;
  u64 trace_cap;
  int refresh_mode;       // 0 dependency lists, 1 recompute every a_k
  int *err;               // set to 1 on a barrier timeout
};

constexpr long long kSpinLimitCycles = 6000000000ll;   // ~3 s: a barrier that long is a bug

// Spin until the bundle's X generation counter reaches `want` (wrap-safe); gives up after
// kSpinLimitCycles and raises *err (the run is then reported as RT_ERR_CUDA).
__device__ __forceinline__ void wait_xgen(const uint32_t *xgen, uint32_t want, int *err) {
  const long long t0 = clock64();
  while ((int)(ld_acquire_u32(xgen) - want) < 0)
    if (clock64() - t0 > kSpinLimitCycles) { atomicExch(err, 1); break; }
}

// Lower bound of `key` in sorted dep_rxn[lo, hi).
__device__ __forceinline__ uint32_t lower_bound_dep(const int32_t *__restrict__ v, uint32_t lo,
                                                    uint32_t hi, int key) {
  while (lo < hi) {
    const uint32_t mid = (lo + hi) >> 1;
    if (__ldg(v + mid) < key) lo = mid + 1; else hi = mid;
  }
  return lo;
}

// Calls f(k) for every reaction k in [k0, k1) that reads a species changed by reaction mu
// (entries are spread over the threads of the CTA; a reaction reading two changed species is
// visited twice -- both visits do the same idempotent work).
template <int BLOCK, typename F>
__device__ __forceinline__ void for_each_dependent(const NetDev &net, int mu, int k0, int k1, F f) {
  const uint32_t e1 = __ldg(net.stoich_ptr + mu + 1);
  for (uint32_t e = __ldg(net.stoich_ptr + mu); e < e1; ++e) {
    const int j = __ldg(net.stoich_species + e);
    const uint32_t lo = __ldg(net.dep_ptr + j), hi = __ldg(net.dep_ptr + j + 1);
    if (lo == hi) continue;
    const uint32_t s = lower_bound_dep(net.dep_rxn, lo, hi, k0);
    const uint32_t t = lower_bound_dep(net.dep_rxn, s, hi, k1);
    for (uint32_t i = s + threadIdx.x; i < t; i += BLOCK) f(__ldg(net.dep_rxn + i));
  }
}

template <int BLOCK>
struct BundleCtx {
  Cand warp_part[BLOCK / 32];
  Cand win;
  int abort_any;
  int abort_local;
};

// Block-wide lexmin of the thread candidates, then all-gather of the S CTA partials through the
// exchange slots (which is also the bundle barrier).  Every thread returns the bundle-wide
// winner; ctx.abort_any is the OR of every CTA's abort_local.  win.k == -2 signals a timeout.
// fence = true additionally orders all earlier global writes of every CTA before all later
// reads of every CTA (used around X copies; the per-firing call does not need it).
template <int BLOCK>
__device__ __forceinline__ Cand bundle_argmin(const BundleParams &p, BundleCtx<BLOCK> &ctx,
                                              u64 *exch, int r, uint32_t &gen, Cand mine,
                                              bool fence) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  mine = warp_lexmin(mine);
  if (lane == 0) ctx.warp_part[warp] = mine;
  if (fence) __threadfence();
  __syncthreads();
  if (warp == 0) {
    Cand c;
    c.dt = __longlong_as_double(0x7ff0000000000000ll);
    c.k = 0x7fffffff;
    for (int w = lane; w < BLOCK / 32; w += 32)
      if (cand_less(ctx.warp_part[w].dt, ctx.warp_part[w].k, c)) c = ctx.warp_part[w];
    c = warp_lexmin(c);
    int abort_any = ctx.abort_local;
    if (p.S > 1) {
      const uint32_t tag = gen + 1u;
      const u64 par = (u64)(((gen >> 1) & 1u) ^ 1u) << 63;     // never matches zeroed memory
      u64 *buf = exch + (size_t)(gen & 1u) * (size_t)p.S * 2;
      if (lane == 0)
        st_relaxed_v2(buf + 2 * r, (u64)__double_as_longlong(c.dt) | par,
                      ((u64)tag << 32) | ((u64)(abort_any ? 1u : 0u) << 31) | (u64)(uint32_t)c.k);
      c.dt = __longlong_as_double(0x7ff0000000000000ll);
      c.k = 0x7fffffff;
      const long long t0 = clock64();
      for (int s = lane; s < p.S; s += 32) {
        u64 w0, w1;
        for (;;) {
          ld_relaxed_v2(buf + 2 * s, w0, w1);
          if ((uint32_t)(w1 >> 32) == tag && (w0 >> 63) == (par >> 63)) break;
          if (clock64() - t0 > kSpinLimitCycles) { atomicExch(p.err, 1); c.k = -2; break; }
        }
        if (c.k == -2) break;
        const double dt = __longlong_as_double((long long)(w0 & 0x7fffffffffffffffull));
        const int k = (int)(uint32_t)(w1 & 0x7fffffffu);
        abort_any |= (int)((w1 >> 31) & 1u);
        if (cand_less(dt, k, c)) { c.dt = dt; c.k = k; }
      }
      const bool timed_out = __any_sync(0xffffffffu, c.k == -2);
      c = warp_lexmin(c);
      abort_any = __any_sync(0xffffffffu, abort_any != 0);
      if (timed_out) c.k = -2;
    }
    if (lane == 0) { ctx.win = c; ctx.abort_any = abort_any; }
  }
  gen += 1u;
  __syncthreads();
  if (fence) __threadfence();
  return ctx.win;
}

#ifdef RT_PHASE_TIMING
#define PT_DECL long long pt_acc[6] = {0, 0, 0, 0, 0, 0}; long long pt_last = clock64();
#define PT_MARK(i) { long long now_ = clock64(); pt_acc[i] += now_ - pt_last; pt_last = now_; }
#else
#define PT_DECL
#define PT_MARK(i)
#endif

template <int BLOCK>
__global__ void __launch_bounds__(BLOCK, 1) rt_bundle_kernel(const BundleParams p) {
  __shared__ BundleCtx<BLOCK> ctx;
  PT_DECL
  const NetDev &net = p.net;
  const int tid = threadIdx.x;
  const int b = blockIdx.x / p.S, r = blockIdx.x % p.S;
  const int M = net.M, N = net.N;
  const double INF = __longlong_as_double(0x7ff0000000000000ll);

  double *__restrict__ T = p.T + (size_t)b * net.M_pad;
  double *__restrict__ P = p.P + (size_t)b * net.M_pad;
  double *__restrict__ A = p.a + (size_t)b * net.M_pad;
  uint32_t *__restrict__ nfire = p.n + (size_t)b * net.M_pad;
  long long *X = p.X + (size_t)b * N;
  u64 *exch = p.exch + (size_t)b * 2 * p.S * 2;
  uint32_t *xgen = p.xgen + (size_t)b * 32;

  const int pairs_total = net.M_pad / 2;
  const int q0 = min(r * p.pairs_per_cta, pairs_total);
  const int q1 = min(q0 + p.pairs_per_cta, pairs_total);
  const int k0 = 2 * q0, k1 = 2 * q1;
  double2 *__restrict__ T2 = reinterpret_cast<double2 *>(T);
  const double2 *__restrict__ P2 = reinterpret_cast<const double2 *>(P);
  const double2 *__restrict__ A2 = reinterpret_cast<const double2 *>(A);

  uint32_t gen = 0;   // exchange generation, identical in every CTA of the bundle
  uint32_t xg = 0;    // number of X updates this bundle has published in this launch
  if (tid == 0) { ctx.abort_local = 0; ctx.abort_any = 0; }
  __syncthreads();

  for (u64 it = (u64)b; it < p.n_traj; it += (u64)p.B) {
    const u64 traj = p.traj_first + it;
    const bool tracing = (it == 0) && p.trace_cap > 0;

    // ---- a-0: X = x0 (slices), then T = 0, P = E(k,0), a = a(X0), n = 0 for the own range
    for (int j = r * BLOCK + tid; j < N; j += p.S * BLOCK) X[j] = p.x0[j];
    Cand none; none.dt = INF; none.k = 0x7fffffff;
    if (bundle_argmin<BLOCK>(p, ctx, exch, r, gen, none, true).k == -2) return;
    for (int k = k0 + tid; k < k1; k += BLOCK) {
      if (k < M) {
        A[k] = propensity(net, X, k);
        P[k] = exp_draw(p.seed, traj, (uint32_t)k, 0u);
      } else {
        A[k] = 0.0;
        P[k] = 0.0;
      }
      __stcg(T + k, 0.0);
      nfire[k] = 0u;
    }
    __syncthreads();

    double t = 0.0, dprev = 0.0;
    u64 fired = 0;
    int mu_prev = -1, stop = 0, status = RT_OK;

    for (;;) {
      PT_MARK(5)
      // ---- A: discrete updates of the previous firing (a-6, a-7, a-8) and refresh flags
      if (mu_prev >= 0) {
        const bool owner = (mu_prev >= k0 && mu_prev < k1);
        if (owner && tid == 0) {              // a-7: new internal firing time of mu (Eq.26)
          const uint32_t c = nfire[mu_prev] + 1u;
          nfire[mu_prev] = c;
          P[mu_prev] = __dadd_rn(P[mu_prev], exp_draw(p.seed, traj, (uint32_t)mu_prev, c));
        }
        if (owner && tid == 32 % BLOCK) {     // a-6: X += v_mu (Eq.5), then publish generation xg
          wait_xgen(xgen, xg - 1u, p.err);
          const uint32_t e1 = __ldg(net.stoich_ptr + mu_prev + 1);
          for (uint32_t e = __ldg(net.stoich_ptr + mu_prev); e < e1; ++e) {
            long long *xp = X + __ldg(net.stoich_species + e);
            const long long x = __ldcg(xp) + (long long)__ldg(net.stoich_v + e);
            if (x < 0 || x > net.xmax) ctx.abort_local = 1;
            __stcg(xp, x);
          }
          st_release_u32(xgen, xg);
          if (tracing && fired - 1 < p.trace_cap) {   // a-8
            if (p.trace_mu) p.trace_mu[fired - 1] = mu_prev;
            if (p.trace_t) p.trace_t[fired - 1] = t;
          }
        }
        if (p.refresh_mode == 0)
          for_each_dependent<BLOCK>(net, mu_prev, k0, k1, [&](int k) { A[k] = -fabs(A[k]); });
        __syncthreads();
      }
      if (p.refresh_mode != 0 && mu_prev >= 0) {      // full recompute reads the new X everywhere
        if (tid == 0) wait_xgen(xgen, xg, p.err);
        __syncthreads();
      }

      PT_MARK(0)
      // ---- B: the streaming pass (a-5 of the previous firing fused with a-2/a-3 of this one)
      Cand best; best.dt = INF; best.k = 0x7fffffff;
      const bool full = (p.refresh_mode != 0);
      for (int q = q0 + tid; q < q1; q += 2 * BLOCK) {
        const int qb = q + BLOCK;
        const bool hb = qb < q1;
        double2 ta = __ldcg(T2 + q), pa = P2[q], aa = A2[q];
        double2 tb, pb, ab;
        if (hb) { tb = __ldcg(T2 + qb); pb = P2[qb]; ab = A2[qb]; }
        ta.x = __dadd_rn(ta.x, __dmul_rn(fabs(aa.x), dprev));
        ta.y = __dadd_rn(ta.y, __dmul_rn(fabs(aa.y), dprev));
        __stcg(T2 + q, ta);
        if (full) {
          aa.x = (2 * q < M) ? propensity(net, X, 2 * q) : 0.0;
          aa.y = (2 * q + 1 < M) ? propensity(net, X, 2 * q + 1) : 0.0;
          const_cast<double2 *>(A2)[q] = aa;
        }
        double d = waiting_time(pa.x, ta.x, aa.x);
        if (d < best.dt) { best.dt = d; best.k = 2 * q; }
        d = waiting_time(pa.y, ta.y, aa.y);
        if (d < best.dt) { best.dt = d; best.k = 2 * q + 1; }
        if (hb) {
          tb.x = __dadd_rn(tb.x, __dmul_rn(fabs(ab.x), dprev));
          tb.y = __dadd_rn(tb.y, __dmul_rn(fabs(ab.y), dprev));
          __stcg(T2 + qb, tb);
          if (full) {
            ab.x = (2 * qb < M) ? propensity(net, X, 2 * qb) : 0.0;
            ab.y = (2 * qb + 1 < M) ? propensity(net, X, 2 * qb + 1) : 0.0;
            const_cast<double2 *>(A2)[qb] = ab;
          }
          d = waiting_time(pb.x, tb.x, ab.x);
          if (d < best.dt) { best.dt = d; best.k = 2 * qb; }
          d = waiting_time(pb.y, tb.y, ab.y);
          if (d < best.dt) { best.dt = d; best.k = 2 * qb + 1; }
        }
      }

      PT_MARK(1)
      // ---- C: fix-up -- a-1 for the dependents of the previous firing, from the new X
      if (mu_prev >= 0 && p.refresh_mode == 0) {
        if (tid == 0) wait_xgen(xgen, xg, p.err);
        __syncthreads();                       // X generation xg visible; T of pass B visible
        for_each_dependent<BLOCK>(net, mu_prev, k0, k1, [&](int k) {
          const double an = propensity(net, X, k);
          A[k] = an;
          const double d = waiting_time(P[k], __ldcg(T + k), an);
          if (cand_less(d, k, best)) { best.dt = d; best.k = k; }
        });
      }

      PT_MARK(2)
      // ---- D/E: a-3 argmin over the bundle
      const Cand win = bundle_argmin<BLOCK>(p, ctx, exch, r, gen, best, false);
      PT_MARK(3)
      if (win.k == -2) return;

      // ---- F: a-4 stop tests, identical in every thread of every CTA of the bundle
      if (ctx.abort_any) { status = RT_ERR_OVERFLOW; break; }
      const double delta = win.dt;
      if (delta == INF) { stop = RT_STOP_ABSORBED; break; }
      if (p.t_end < INF && __dadd_rn(t, delta) > p.t_end) {
        const double rest = __dsub_rn(p.t_end, t);
        for (int k = k0 + tid; k < k1; k += BLOCK)
          __stcg(T + k, __dadd_rn(__ldcg(T + k), __dmul_rn(fabs(A[k]), rest)));
        t = p.t_end;
        stop = RT_STOP_T_END;
        break;
      }
      t = __dadd_rn(t, delta);
      fired += 1;
      xg += 1u;
      mu_prev = win.k;
      dprev = delta;
      if (p.max_firings != 0 && fired == p.max_firings) {
        // last firing: apply its discrete updates and its internal-time increment now
        const bool owner = (mu_prev >= k0 && mu_prev < k1);
        if (owner && tid == 0) {
          const uint32_t c = nfire[mu_prev] + 1u;
          nfire[mu_prev] = c;
          P[mu_prev] = __dadd_rn(P[mu_prev], exp_draw(p.seed, traj, (uint32_t)mu_prev, c));
        }
        if (owner && tid == 32 % BLOCK) {
          wait_xgen(xgen, xg - 1u, p.err);
          const uint32_t e1 = __ldg(net.stoich_ptr + mu_prev + 1);
          for (uint32_t e = __ldg(net.stoich_ptr + mu_prev); e < e1; ++e) {
            long long *xp = X + __ldg(net.stoich_species + e);
            const long long x = __ldcg(xp) + (long long)__ldg(net.stoich_v + e);
            if (x < 0 || x > net.xmax) ctx.abort_local = 1;
            __stcg(xp, x);
          }
          st_release_u32(xgen, xg);
          if (tracing && fired - 1 < p.trace_cap) {
            if (p.trace_mu) p.trace_mu[fired - 1] = mu_prev;
            if (p.trace_t) p.trace_t[fired - 1] = t;
          }
        }
        for (int k = k0 + tid; k < k1; k += BLOCK)
          __stcg(T + k, __dadd_rn(__ldcg(T + k), __dmul_rn(fabs(A[k]), dprev)));
        stop = RT_STOP_MAX_FIRINGS;
        break;
      }
    }

#ifdef RT_PHASE_TIMING
    if (tid == 0 && (r == 0 || r == p.S - 1 || r == p.S / 2))
      printf("cta %d: A %.0f B %.0f C %.0f D+E %.0f F %.0f cyc/firing\n", r, (double)pt_acc[0] / fired,
             (double)pt_acc[1] / fired, (double)pt_acc[2] / fired, (double)pt_acc[3] / fired,
             (double)pt_acc[5] / fired);
#endif
    // ---- trajectory done: make X visible bundle-wide, collect the overflow flag, write results
    if (bundle_argmin<BLOCK>(p, ctx, exch, r, gen, none, true).k == -2) return;
    if (ctx.abort_any) status = RT_ERR_OVERFLOW;
    if (p.x_out)
      for (int j = r * BLOCK + tid; j < N; j += p.S * BLOCK)
        p.x_out[it * (u64)N + (u64)j] = __ldcg(X + j);
    if (r == 0 && tid == 0) {
      rt_result res;
      res.t = t; res.firings = fired; res.stop = stop; res.status = status;
      p.res[it] = res;
    }
    __syncthreads();
    if (tid == 0) ctx.abort_local = 0;
    __syncthreads();
  }
}

}  // namespace rt
