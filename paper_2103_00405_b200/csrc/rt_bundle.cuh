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
//   walker warp:   X += v_mu on this CTA's PRIVATE replica of X (Eq.5) -- every CTA knows mu
//                  after the exchange, so X never crosses CTAs; redraw of P_mu (Eq.26); then the
//                  dependency walk: stoich row of mu -> species record -> dense
//                  dependency entries (k, reactants, sigma) -> new a_k for the k in [k0, k1).
// The stream uses the OLD a_k, which is exactly the propensity that held during the elapsed
// interval, so T is right for every k; only the waiting times of the refreshed reactions (and
// of mu) are stale.  After one CTA barrier the new a_k / P_mu are stored, the threads that own
// a refreshed reaction re-scan their few reactions (read-only), and the block argmin follows.
// The CTA partials are combined by an all-gather through L2 (one 16-byte slot per CTA,
// self-validating words, double-buffered), which doubles as the per-firing bundle barrier.
#pragma once
#include "rt_device.cuh"
#include "../../include/rt.h"

namespace rt {

constexpr int kListCap = 1024;      // refreshed reactions a CTA stages per round
constexpr int kWalkerWarps = 1;

struct BundleParams {
  NetDev net;
  double *T, *P, *a;      // [B][M_pad]   (STATE_SMEM: written once, at the end of a trajectory)
  uint32_t *n;            // [B][M_pad]   firings per reaction
  long long *X;           // [B][S][N]    one private replica of X per CTA
  u64 *exch;              // [B][2][S][2] exchange slots, zeroed before launch
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
  int refresh_mode;       // 0 dependency walk, 1 recompute every a_k (the paper's GPU scheme)
  int *err;               // set to 1 on a barrier timeout
};

constexpr long long kSpinLimitCycles = 6000000000ll;   // ~3 s: a barrier that long is a bug

template <int BLOCK>
struct BundleCtx {
  Cand warp_part[BLOCK / 32];
  Cand win;
  int abort_local;        // a count left [0, xmax] (identical in every CTA: all replicate X)
  int list_n;             // staged refreshes of this round
  int more;               // walker has entries left for another round
  int p_k;                // reaction whose P was redrawn (or -1), and its new value
  double p_val;
};

// Block-wide lexmin of the thread candidates, then all-gather of the S CTA partials through the
// exchange slots (which is also the bundle barrier).  Every thread returns the bundle-wide
// winner.  win.k == -2 signals a timeout.
template <int BLOCK>
__device__ __forceinline__ Cand bundle_argmin(const BundleParams &p, BundleCtx<BLOCK> &ctx,
                                              u64 *exch, int r, uint32_t &gen, Cand mine) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  mine = warp_lexmin(mine);
  if (lane == 0) ctx.warp_part[warp] = mine;
  __syncthreads();
  if (warp == 0) {
    Cand c = ctx.warp_part[lane];                 // BLOCK / 32 <= 32 partials
    if (lane >= BLOCK / 32) { c.dt = __longlong_as_double(0x7ff0000000000000ll); c.k = 0x7fffffff; }
    c = warp_lexmin(c);
    if (p.S > 1) {
      const uint32_t tag = gen + 1u;
      const u64 par = (u64)(((gen >> 1) & 1u) ^ 1u) << 63;     // never matches zeroed memory
      u64 *buf = exch + (size_t)(gen & 1u) * (size_t)p.S * 2;
      if (lane == 0)
        st_relaxed_v2(buf + 2 * r, (u64)__double_as_longlong(c.dt) | par,
                      ((u64)tag << 32) | (u64)(uint32_t)c.k);
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
        if (cand_less(dt, k, c)) { c.dt = dt; c.k = k; }
      }
      const bool timed_out = __any_sync(0xffffffffu, c.k == -2);
      c = warp_lexmin(c);
      if (timed_out) c.k = -2;
    }
    if (lane == 0) ctx.win = c;
  }
  gen += 1u;
  __syncthreads();
  return ctx.win;
}

#ifdef RT_PHASE_TIMING
#define PT_DECL long long pt_acc[6] = {0, 0, 0, 0, 0, 0}; long long pt_last = clock64();
#define PT_MARK(i) { long long now_ = clock64(); pt_acc[i] += now_ - pt_last; pt_last = now_; }
#else
#define PT_DECL
#define PT_MARK(i)
#endif

// The per-firing pass of one thread over the reactions it owns.  UPDATE: also apply the
// internal-time increment T_k += a_k * dprev (first pass); otherwise read-only (re-scan).
// FULL: recompute a_k from X for every k (refresh_mode 1).
// Ownership: STATE_SMEM -- local index i = tid, tid+NT, ...; global state -- pair q0+tid, +NT, ...
template <int NT, bool SMEM, bool UPDATE>
__device__ __forceinline__ Cand scan_own(const NetDev &net, const long long *X, int tid, int k0, int k1,
                                         double *sT, const double *sP, double *sA,
                                         double *T, double *P, double *A, double dprev, bool full) {
  Cand best;
  best.dt = __longlong_as_double(0x7ff0000000000000ll);
  best.k = 0x7fffffff;
  if (SMEM) {
    const int cnt = k1 - k0;
#pragma unroll 4
    for (int i = tid; i < cnt; i += NT) {
      double a = sA[i], t = sT[i];
      const double pk = sP[i];
      if (UPDATE) {
        t = __dadd_rn(t, __dmul_rn(a, dprev));
        sT[i] = t;
        if (full) {
          a = (k0 + i < net.M) ? propensity(net, X, k0 + i) : 0.0;
          sA[i] = a;
        }
      }
      const double d = waiting_time(pk, t, a);
      if (d < best.dt) { best.dt = d; best.k = k0 + i; }
    }
  } else {
    double2 *T2 = reinterpret_cast<double2 *>(T);
    double2 *P2 = reinterpret_cast<double2 *>(P);
    double2 *A2 = reinterpret_cast<double2 *>(A);
    const int q0 = k0 >> 1, q1 = k1 >> 1;
    for (int q = q0 + tid; q < q1; q += 2 * NT) {
      const int qb = q + NT;
      const bool hb = qb < q1;
      double2 ta = __ldcg(T2 + q), pa = __ldcg(P2 + q), aa = __ldcg(A2 + q);
      double2 tb, pb, ab;
      if (hb) { tb = __ldcg(T2 + qb); pb = __ldcg(P2 + qb); ab = __ldcg(A2 + qb); }
      if (UPDATE) {
        ta.x = __dadd_rn(ta.x, __dmul_rn(aa.x, dprev));
        ta.y = __dadd_rn(ta.y, __dmul_rn(aa.y, dprev));
        __stcg(T2 + q, ta);
        if (full) {
          aa.x = (2 * q < net.M) ? propensity(net, X, 2 * q) : 0.0;
          aa.y = (2 * q + 1 < net.M) ? propensity(net, X, 2 * q + 1) : 0.0;
          __stcg(A2 + q, aa);
        }
      }
      double d = waiting_time(pa.x, ta.x, aa.x);
      if (d < best.dt) { best.dt = d; best.k = 2 * q; }
      d = waiting_time(pa.y, ta.y, aa.y);
      if (d < best.dt) { best.dt = d; best.k = 2 * q + 1; }
      if (hb) {
        if (UPDATE) {
          tb.x = __dadd_rn(tb.x, __dmul_rn(ab.x, dprev));
          tb.y = __dadd_rn(tb.y, __dmul_rn(ab.y, dprev));
          __stcg(T2 + qb, tb);
          if (full) {
            ab.x = (2 * qb < net.M) ? propensity(net, X, 2 * qb) : 0.0;
            ab.y = (2 * qb + 1 < net.M) ? propensity(net, X, 2 * qb + 1) : 0.0;
            __stcg(A2 + qb, ab);
          }
        }
        d = waiting_time(pb.x, tb.x, ab.x);
        if (d < best.dt) { best.dt = d; best.k = 2 * qb; }
        d = waiting_time(pb.y, tb.y, ab.y);
        if (d < best.dt) { best.dt = d; best.k = 2 * qb + 1; }
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



// New propensity of the reaction of dependency entry d = (k, j1, j2, sigma1 | sigma2 << 8 |
// general << 16), same operation order as propensity().  `on` = false turns the entry into a
// harmless dummy (index 0 everywhere) so that the loads of a batch can be issued together.
__device__ __forceinline__ double propensity_dep(const NetDev &net, const long long *X, int4 d, bool on) {
  const int k = on ? d.x : 0, j1 = on ? d.y : 0, j2 = (on && d.z >= 0) ? d.z : 0;
  const double c = __ldg(net.rate + k);
  const long long x1 = X[j1], x2 = X[j2];
  double a = __dmul_rn(c, __ll2double_rn(binom(x1, d.w & 0xff)));
  if (d.z >= 0) a = __dmul_rn(a, __ll2double_rn(binom(x2, (d.w >> 8) & 0xff)));
  if (on && (d.w & 0x10000)) a = propensity(net, X, k);    // more than two reactants (rare)
  return a;
}

// Walker-warp state for one firing, uniform over the warp except my_lo / my_hi.
struct Walk {
  int n_e;               // changed species of the fired reaction
  int e;                 // species being walked
  bool entered;          // (i, hi) hold the range of species e
  uint32_t i, hi;        // dependency entries of species e still to visit
  uint32_t my_lo, my_hi; // lane l: range of species l (l < 32)
  uint32_t e0;           // CSR row start (rows with more than 4 entries)
};

// Dependency range of species j restricted (for hubs: to the reaction blocks touching [k0,k1)).
__device__ __forceinline__ void species_range(const NetDev &net, int j, int k0, int k1,
                                              uint32_t &lo, uint32_t &hi) {
  const uint2 rec = __ldg(reinterpret_cast<const uint2 *>(net.sp_rec) + j);
  lo = rec.x; hi = rec.y;
  if (hi - lo > (uint32_t)net.big_deg && k1 > k0) {
    const uint32_t *off = net.big_off + (size_t)__ldg(net.sp_big + j) * (size_t)(net.n_blk + 1);
    lo = __ldg(off + (k0 >> net.blk_shift));
    hi = __ldg(off + ((k1 - 1) >> net.blk_shift) + 1);
  }
}

template <int BLOCK, bool SMEM>
__global__ void __launch_bounds__(BLOCK, 1) rt_bundle_kernel(const BundleParams p) {
  constexpr int NT = BLOCK - 32 * kWalkerWarps;      // stream threads; the last warp walks
  __shared__ BundleCtx<BLOCK> ctx;
  __shared__ int list_k[kListCap];
  __shared__ double list_a[kListCap];
  __shared__ unsigned char dirty[BLOCK];
  extern __shared__ __align__(16) unsigned char dyn_smem[];
  PT_DECL
  const NetDev &net = p.net;
  const int tid = threadIdx.x, lane = tid & 31;
  const bool is_walker = tid >= NT;
  const int b = blockIdx.x / p.S, r = blockIdx.x % p.S;
  const int M = net.M, N = net.N;
  const double INF = __longlong_as_double(0x7ff0000000000000ll);

  double *T = p.T + (size_t)b * net.M_pad;
  double *P = p.P + (size_t)b * net.M_pad;
  double *A = p.a + (size_t)b * net.M_pad;
  uint32_t *nfire = p.n + (size_t)b * net.M_pad;
  long long *X = p.X + ((size_t)b * p.S + r) * (size_t)N;     // this CTA's replica
  u64 *exch = p.exch + (size_t)b * 2 * p.S * 2;

  const int pairs_total = net.M_pad / 2;
  const int q0 = min(r * p.pairs_per_cta, pairs_total);
  const int q1 = min(q0 + p.pairs_per_cta, pairs_total);
  const int k0 = 2 * q0, k1 = 2 * q1;
  double *sT = reinterpret_cast<double *>(dyn_smem);
  double *sP = sT + (SMEM ? 2 * p.pairs_per_cta : 0);
  double *sA = sP + (SMEM ? 2 * p.pairs_per_cta : 0);

  uint32_t gen = 0;   // exchange generation, identical in every CTA of the bundle
  dirty[tid] = 0;
  if (tid == 0) { ctx.abort_local = 0; ctx.list_n = 0; ctx.more = 0; ctx.p_k = -1; }
  __syncthreads();

  for (u64 it = (u64)b; it < p.n_traj; it += (u64)p.B) {
    const u64 traj = p.traj_first + it;
    const bool tracing = (it == 0) && p.trace_cap > 0 && r == 0;

    // ---- a-0: X replica = x0, then T = 0, P = E(k,0), a = a(X0), n = 0 for the own range
    for (int j = tid; j < N; j += BLOCK) X[j] = p.x0[j];
    __syncthreads();
    for (int k = k0 + tid; k < k1; k += BLOCK) {
      double a0 = 0.0, p0 = 0.0;
      if (k < M) {
        a0 = propensity(net, X, k);
        p0 = exp_draw(p.seed, traj, (uint32_t)k, 0u);
      }
      if (SMEM) { sT[k - k0] = 0.0; sP[k - k0] = p0; sA[k - k0] = a0; }
      else { __stcg(T + k, 0.0); __stcg(P + k, p0); __stcg(A + k, a0); }
      nfire[k] = 0u;
    }
    __syncthreads();

    double t = 0.0, dprev = 0.0;
    u64 fired = 0;
    int mu_prev = -1, stop = 0, status = RT_OK;
    bool finishing = false;
    const bool full = (p.refresh_mode != 0);

    for (;;) {   // one iteration per firing, plus one closing pass
      PT_MARK(5)
      Walk w;
      w.n_e = 0; w.e = 0; w.entered = false; w.i = 0; w.hi = 0; w.my_lo = 0; w.my_hi = 0; w.e0 = 0;
      Cand best; best.dt = INF; best.k = 0x7fffffff;

      if (is_walker && mu_prev >= 0) {
        // ===== walker warp: discrete updates of the previous firing (a-6, a-7, a-8) =====
        const bool owner = (mu_prev >= k0 && mu_prev < k1);
        uint32_t c_old = 0; double p_old = 0.0;
        if (owner && lane == 0) {
          c_old = nfire[mu_prev];
          p_old = SMEM ? sP[mu_prev - k0] : __ldcg(P + mu_prev);
        }
        const int4 row_j = __ldg(reinterpret_cast<const int4 *>(net.srow_j) + mu_prev);
        const int4 row_v = __ldg(reinterpret_cast<const int4 *>(net.srow_v) + mu_prev);
        const bool ell = row_j.x != -2;       // -2: more than 4 entries, use the CSR row instead
        if (ell) {
          w.n_e = (row_v.x != 0) + (row_v.y != 0) + (row_v.z != 0) + (row_v.w != 0);
        } else {
          w.e0 = __ldg(net.stoich_ptr + mu_prev);
          w.n_e = (int)(__ldg(net.stoich_ptr + mu_prev + 1) - w.e0);
        }
        for (int e = lane; e < w.n_e; e += 32) {     // a-6: X += v_mu (Eq.5), entry e by lane e%32
          int j, v;
          if (ell) {
            j = e == 0 ? row_j.x : e == 1 ? row_j.y : e == 2 ? row_j.z : row_j.w;
            v = e == 0 ? row_v.x : e == 1 ? row_v.y : e == 2 ? row_v.z : row_v.w;
          } else {
            j = __ldg(net.stoich_species + w.e0 + e);
            v = __ldg(net.stoich_v + w.e0 + e);
          }
          if (e < 32 && !full) species_range(net, j, k0, k1, w.my_lo, w.my_hi);
          const long long x = X[j] + (long long)v;
          if (x < 0 || x > net.xmax) ctx.abort_local = 1;
          X[j] = x;
        }
        if (lane == 0) {
          if (owner) {                           // a-7: new internal firing time of mu (Eq.26)
            nfire[mu_prev] = c_old + 1u;
            ctx.p_val = __dadd_rn(p_old, exp_draw(p.seed, traj, (uint32_t)mu_prev, c_old + 1u));
            ctx.p_k = mu_prev;
          }
          if (tracing && fired - 1 < p.trace_cap) {   // a-8
            if (p.trace_mu) p.trace_mu[fired - 1] = mu_prev;
            if (p.trace_t) p.trace_t[fired - 1] = t;
          }
        }
        __syncwarp();                            // the replica's new counts are visible warp-wide
      }
      if (full && mu_prev >= 0) __syncthreads(); // full recompute reads the new X in the stream

      PT_MARK(0)
      bool first_round = true;
      for (;;) {   // rounds: one, unless this CTA has more than kListCap refreshes
        if (is_walker) {
          // ===== walker warp: dependency walk (a-1 for k in D(mu) that fall in [k0, k1)) =====
          int n = 0;
          bool more = false;
          if (!full && k1 > k0) {
            while (w.e < w.n_e) {
              if (!w.entered) {
                if (w.e < 32) {
                  w.i = __shfl_sync(0xffffffffu, w.my_lo, w.e);
                  w.hi = __shfl_sync(0xffffffffu, w.my_hi, w.e);
                } else {
                  species_range(net, __ldg(net.stoich_species + w.e0 + w.e), k0, k1, w.i, w.hi);
                }
                w.entered = true;
              }
              while (w.i < w.hi) {
                if (n + 128 > kListCap) { more = true; break; }
                int4 d[4];
                bool in[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                  const uint32_t idx = w.i + (uint32_t)(u * 32 + lane);
                  const bool valid = idx < w.hi;
                  d[u] = __ldg(reinterpret_cast<const int4 *>(net.dep) + (valid ? idx : w.i));
                  in[u] = valid && d[u].x >= k0 && d[u].x < k1;
                }
                double an[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) an[u] = propensity_dep(net, X, d[u], in[u]);
#pragma unroll
                for (int u = 0; u < 4; ++u) {
                  const unsigned m = __ballot_sync(0xffffffffu, in[u]);
                  if (in[u]) {
                    const int pos = n + __popc(m & ((1u << lane) - 1u));
                    list_k[pos] = d[u].x;
                    list_a[pos] = an[u];
                  }
                  n += __popc(m);
                }
                w.i += 128u;
              }
              if (more) break;
              w.e += 1;
              w.entered = false;
            }
          }
          if (lane == 0) { ctx.list_n = n; ctx.more = more ? 1 : 0; }
        } else if (first_round) {
          // ===== stream warps: a-5 of the previous firing fused with a-2/a-3 of this one =====
          best = scan_own<NT, SMEM, true>(net, X, tid, k0, k1, sT, sP, sA, T, P, A, dprev, full);
        }
        PT_MARK(1)
        __syncthreads();
        // ----- apply the staged refreshes; mark the owning threads for a re-scan
        const int n = ctx.list_n;
        const bool more = ctx.more != 0;
        for (int i = tid; i < n; i += BLOCK) {
          const int k = list_k[i];
          if (SMEM) sA[k - k0] = list_a[i]; else __stcg(A + k, list_a[i]);
          dirty[owner_thread<NT, SMEM>(k, k0)] = 1;
        }
        if (tid == 0 && ctx.p_k >= 0) {
          const int k = ctx.p_k;
          if (SMEM) sP[k - k0] = ctx.p_val; else __stcg(P + k, ctx.p_val);
          dirty[owner_thread<NT, SMEM>(k, k0)] = 1;
          ctx.p_k = -1;
        }
        __syncthreads();
        if (!more) break;
        first_round = false;
      }
      PT_MARK(2)
      if (!is_walker && dirty[tid]) {            // re-scan (read-only) with the new a_k, P_mu
        dirty[tid] = 0;
        best = scan_own<NT, SMEM, false>(net, X, tid, k0, k1, sT, sP, sA, T, P, A, 0.0, false);
      }
      if (ctx.abort_local) { status = RT_ERR_OVERFLOW; stop = 0; break; }
      if (finishing) break;

      // ---- a-3 argmin over the bundle
      PT_MARK(3)
      const Cand win = bundle_argmin<BLOCK>(p, ctx, exch, r, gen, best);
      PT_MARK(4)
      if (win.k == -2) return;

      // ---- a-4 stop tests, identical in every thread of every CTA of the bundle
      const double delta = win.dt;
      if (delta == INF) { stop = RT_STOP_ABSORBED; break; }
      if (p.t_end < INF && __dadd_rn(t, delta) > p.t_end) {
        dprev = __dsub_rn(p.t_end, t);           // closing pass: T_k += a_k * (t_end - t), no firing
        t = p.t_end;
        mu_prev = -1;
        stop = RT_STOP_T_END;
        finishing = true;
        continue;
      }
      t = __dadd_rn(t, delta);
      fired += 1;
      mu_prev = win.k;
      dprev = delta;
      if (p.max_firings != 0 && fired == p.max_firings) {
        stop = RT_STOP_MAX_FIRINGS;              // closing pass applies this firing's updates
        finishing = true;
      }
    }

#ifdef RT_PHASE_TIMING
    if (tid == 0 && (r == 0 || r == p.S - 1 || r == p.S / 2))
      printf("cta %d stream thread: updates/sync %.0f  stream %.0f  apply %.0f  rescan %.0f  argmin+exchange %.0f  stop %.0f cyc/firing\n",
             r, (double)pt_acc[0] / fired, (double)pt_acc[1] / fired, (double)pt_acc[2] / fired,
             (double)pt_acc[3] / fired, (double)pt_acc[4] / fired, (double)pt_acc[5] / fired);
    if (tid == NT && (r == 0 || r == p.S - 1 || r == p.S / 2))
      printf("cta %d walker: updates %.0f  walk %.0f  apply %.0f  rescan %.0f  argmin+exchange %.0f  stop %.0f cyc/firing\n",
             r, (double)pt_acc[0] / fired, (double)pt_acc[1] / fired, (double)pt_acc[2] / fired,
             (double)pt_acc[3] / fired, (double)pt_acc[4] / fired, (double)pt_acc[5] / fired);
#endif
    // ---- trajectory done: write the state back (STATE_SMEM), X and the outcome
    __syncthreads();
    dirty[tid] = 0;
    if (SMEM)
      for (int k = k0 + tid; k < k1; k += BLOCK) {
        __stcg(T + k, sT[k - k0]); __stcg(P + k, sP[k - k0]); __stcg(A + k, sA[k - k0]);
      }
    if (p.x_out)
      for (int j = r * BLOCK + tid; j < N; j += p.S * BLOCK)
        p.x_out[it * (u64)N + (u64)j] = X[j];
    if (r == 0 && tid == 0) {
      rt_result res;
      res.t = t; res.firings = fired; res.stop = stop; res.status = status;
      p.res[it] = res;
    }
    if (tid == 0) { ctx.abort_local = 0; ctx.p_k = -1; }
    __syncthreads();
  }
}

}  // namespace rt
