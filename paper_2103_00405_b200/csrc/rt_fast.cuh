// rt_fast.cuh -- "candidate-first" bundle kernel: the per-firing O(M) pass is taken OFF the critical
// path of a firing.  Same algorithm, same arithmetic, same results as rt_bundle_kernel (state in
// shared memory, dependency-graph refresh, constant rates, either formulation); what changes is
// WHEN each piece of a firing's work is done.
//
// In rt_bundle_kernel one firing is  pass over all reactions -> block argmin -> exchange, so the
// exchange (1.2 us through L2, 0.27 us inside a cluster) and the pass (1.3 us) add up.  Here every
// stream thread carries ONE candidate, the reaction the previous pass found to be the thread's
// argmin with a safety margin (below).  After an exchange has named (mu, dt):
//   S1  each thread advances only its candidate, T_c += a_c dt, and divides it exactly;
//   S2  the reactions whose propensity changed (the walker's staged list) are advanced with their
//       OLD a_k, get the new a_k, and join the reduction as fresh candidates;
//   S3  threads whose candidate fired or was refreshed (or that have none) are re-scanned exactly,
//       their warp sharing the work;
//   S4  block argmin -> the exchange warp posts this CTA's partial;
//   S5  WHILE the exchange is in flight the stream warps run the pass: T_k += a_k dt for every
//       reaction not advanced in S1..S3 (per-thread bit masks).  A thread keeps its candidate
//       across firings; its warp re-derives the candidates from approximate quotients when one
//       is void or doubtful, and at least every kRepickPeriod firings.
// Every T_k still receives every increment a_k dt_n, one rounded multiply and one rounded add per
// firing, in firing order: results are bit-identical to dividing everything every firing.
//
// Why a candidate chosen earlier is still the thread's exact argmin: the pass looks
// at the HIGH WORD of q~_k = (P_k - T_k) * rcp.approx(a_k) as an integer key (positive doubles
// order like integers).  Key error: rcp.approx.ftz.f64 2^-19.94 relative
// (tests/test_gpu_kernel_facts.py), truncation < 1 unit; a unit is 2^-20..2^-21 relative, so a key
// is within 3.5 units of the exact quotient's.  One more firing moves every exact quotient of the
// thread by the same dt, except for the rounding of T_k + a_k dt, at most
// 2^-52 (|T_k| + a_k dt) / a_k: the pass checks that P_k - T_k keeps at least 2^-31 of
// max(|P_k|, |T_k|) (kGuardShift; integer test on high words; a_k = 0 exempt), which bounds that
// drift by one unit per reaction per firing.  A thread whose second-smallest key exceeds the
// smallest by more than kQTolUnits = 64 > 2 * 3.5 + 2 * kRepickPeriod therefore keeps a unique
// exact argmin for kRepickPeriod = 24 firings; a refreshed reaction is compared exactly (S2: it
// must stay 2^-13 clear of the candidate, or clearly below it and take over, else the thread
// re-picks); any thread without such a margin has no candidate and is re-scanned exactly every
// firing (S3), as are all threads when some a_k of the CTA is outside the range where the rcp
// bound is established (any_odd).
//
// Warps: NT / 32 stream warps; one exchange warp (reduces the warp partials, posts, gathers,
// publishes the winner, prefetches the CTA candidate's walk data into L2); one walker warp (X
// update, staged refreshes; while the others work it pre-walks the exchange's runner-up AND
// computes that reaction's refreshes speculatively from X as it will be, so that a correct guess
// -- 94..99 % of the firings -- costs no memory round trip at all).  The redraw of P_mu (Philox +
// log) is precomputed by each stream thread for its own candidate and installed by the owner in S1.
#pragma once
#include "rt_bundle.cuh"

namespace rt {

constexpr int kFastHelperWarps = 2;
constexpr int kBarMore = 5, kBarWin = 6;
constexpr int kQTolUnits = 64;       // key margin, in units of the high word's last bit
constexpr int kGuardShift = 29;      // high word of P - T may be at most this many binades below max(|P|, |T|)'s
constexpr int kRepickPeriod = 24;    // a warp re-derives its threads' candidates at least this often

// Per-thread 64-bit slot masks in shared memory, kept as two words so that a bit is set with a
// native 32-bit shared-memory atomic.
__device__ __forceinline__ u64 mask_load(const unsigned (*m)[2], int t) {
  const uint2 v = *reinterpret_cast<const uint2 *>(m[t]);
  return (u64)v.x | ((u64)v.y << 32);
}
__device__ __forceinline__ void mask_store(unsigned (*m)[2], int t, u64 v) {
  *reinterpret_cast<uint2 *>(m[t]) = make_uint2((unsigned)v, (unsigned)(v >> 32));
}
// sets bit `slot` of thread t's mask; true if this call set it
__device__ __forceinline__ bool mask_claim(unsigned (*m)[2], int t, int slot) {
  const unsigned bit = 1u << (slot & 31);
  return (atomicOr(&m[t][slot >> 5], bit) & bit) == 0u;
}

template <int BLOCK>
struct FastCtx {
  Cand warp_part[(BLOCK - 32 * kFastHelperWarps) / 32];
  Cand win;
  u64 second;             // L2 exchange: runner-up tagged with its generation, (gen << 32) | k
  int second_k;           // cluster: runner-up of the exchange (published with the winner)
  int abort_local, list_n, list_buf, more, any_odd;
  alignas(16) u64 cl_slot[2][kMaxClusterCtas][2];
  alignas(8) u64 cl_bar[2];
};

// Shared-memory layout of a CTA's (T, P, a) arrays: reaction li (local index) belongs to stream
// thread li % NT, slot li / NT, and sits at thread + slot * (NT + 1).  The padded row keeps the
// slots of ONE thread in different banks, so that a warp re-scanning a stale thread (S3: lane l
// takes slot l) reads without bank conflicts (with rows of NT they are 32-way: NT is a multiple
// of 32); the pass itself (lane l = thread l, one slot) is conflict-free either way.
template <int NT> __device__ __forceinline__ int sidx(int li) { return li + li / NT; }

// Integer key of the approximate quotient of one reaction; clears guard_ok when the lagged
// candidate argument does not cover it (see the header).
__device__ __forceinline__ int q_key(double pk, double t, double a, bool &guard_ok) {
  const double r = __dsub_rn(pk, t);
  const int hq = __double2hiint(__dmul_rn(r, rcp_approx(a)));
  const int hm = max(__double2hiint(pk) & 0x7fffffff, __double2hiint(t) & 0x7fffffff);
  guard_ok = guard_ok && ((__double2hiint(r) + (kGuardShift << 20) >= hm) || hq >= 0x7ff00000);
  return hq;
}

// S5: the pass of one thread.  Advances the reactions whose bit in `done` is clear, then picks the
// candidate slot for the next firing (-1: none, the thread will be re-scanned exactly).
template <int NT>
__device__ __forceinline__ int pass_and_pick(int tid, int cnt_pad, double *__restrict__ sT,
                                             const double *__restrict__ sP, const double *__restrict__ sA,
                                             double dprev, u64 done, bool any_odd) {
  constexpr int U = kScanBatch;
  int m1 = 0x7fffffff, m2 = 0x7fffffff, s1 = 0;
  bool guard_ok = true;
  int slot = 0;
  constexpr int R = NT + 1;                            // padded row (see sidx)
  for (int i = tid; i < cnt_pad; i += U * R, slot += U) {
    double a[U], t[U], pk[U];
#pragma unroll
    for (int u = 0; u < U; ++u) { a[u] = sA[i + u * R]; t[u] = sT[i + u * R]; pk[u] = sP[i + u * R]; }
#pragma unroll
    for (int u = 0; u < U; ++u)
      if (!((done >> (slot + u)) & 1ull)) {
        t[u] = __dadd_rn(t[u], __dmul_rn(a[u], dprev));
        sT[i + u * R] = t[u];
      }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int q = q_key(pk[u], t[u], a[u], guard_ok);
      m2 = min(m2, max(q, m1));
      if (q < m1) { m1 = q; s1 = slot + u; }
    }
  }
  const bool decided = !any_odd && guard_ok && m1 >= ((1023 - 100) << 20) && m1 <= ((1023 + 100) << 20) &&
                       m2 > m1 + kQTolUnits;
  return decided ? s1 : -1;
}

// S5 of a thread that keeps its candidate: T_k += a_k dt for the reactions not yet advanced, nothing else
// (24 instead of 32 bytes of shared-memory traffic per reaction, a third of the instructions).
template <int NT>
__device__ __forceinline__ void pass_advance(int tid, int cnt_pad, double *__restrict__ sT,
                                             const double *__restrict__ sA, double dprev, u64 done) {
  constexpr int U = kScanBatch;
  int slot = 0;
  constexpr int R = NT + 1;
  for (int i = tid; i < cnt_pad; i += U * R, slot += U) {
    double a[U], t[U];
#pragma unroll
    for (int u = 0; u < U; ++u) { a[u] = sA[i + u * R]; t[u] = sT[i + u * R]; }
#pragma unroll
    for (int u = 0; u < U; ++u)
      if (!((done >> (slot + u)) & 1ull)) sT[i + u * R] = __dadd_rn(t[u], __dmul_rn(a[u], dprev));
  }
}

template <int BLOCK, bool CLUSTER>
__global__ void __launch_bounds__(BLOCK, 1) rt_fast_kernel(const BundleParams p) {
  constexpr int NT = BLOCK - 32 * kFastHelperWarps;   // stream threads
  constexpr int XW = NT / 32;                         // exchange warp
  constexpr int WW = NT / 32 + 1;                     // walker warp
  __shared__ FastCtx<BLOCK> ctx;
  __shared__ int out_k[2][kListCap];                  // staged refreshes (k, new a_k), two buffers:
  __shared__ double out_a[2][kListCap];               //   one published, one being speculated into
  __shared__ int4 list_d[kListCap];
  __shared__ int4 pw_d[kListCap];                     // pre-walked dependency entries of reaction pw_k
  __shared__ double pw_c[kListCap];
  __shared__ __align__(8) unsigned advm[NT][2];       // per stream thread: slots already advanced this firing
  __shared__ __align__(8) unsigned refm[NT][2];       //                    slots whose refresh is claimed
  __shared__ int mybest_k[NT];                        // reaction each stream thread proposes (-3: none)
  __shared__ double dcand[NT];                        //   and its exact waiting time for this firing
  __shared__ unsigned char dirty[NT];                 // the thread's proposal is void: exact re-scan (S3)
  __shared__ unsigned char repick[NT];                // the thread's candidate may have lost its margin
  __shared__ int newcand[NT];                         // a refreshed reaction clearly below the thread's candidate (slot, or -1)
  extern __shared__ __align__(16) unsigned char dyn_smem[];
  const NetDev &net = p.net;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool is_stream = warp < XW, is_xw = warp == XW, is_walker = warp == WW;
  const int b = blockIdx.x / p.S, r = blockIdx.x % p.S;
  const int M = net.M, N = net.N;
  const double INF = __longlong_as_double(0x7ff0000000000000ll);
  const bool resid = p.formulation != 0;

  double *T = p.T + (size_t)b * net.M_pad;
  double *P = p.P + (size_t)b * net.M_pad;
  double *A = p.a + (size_t)b * net.M_pad;
  uint32_t *nfire = p.n + (size_t)b * net.M_pad;
  u64 *X = p.X + (size_t)b * (size_t)N;
  u64 *exch = p.exch + (size_t)b * 2 * p.S * kSlotStride;

  const int pairs_total = net.M_pad / 2;
  const int q0 = min(r * p.pairs_per_cta, pairs_total);
  const int q1 = min(q0 + p.pairs_per_cta, pairs_total);
  const int k0 = 2 * q0, k1 = 2 * q1;
  const int cnt_pad = p.cnt_pad;
  const int nslot = cnt_pad / NT;                     // slots per stream thread (<= 64)
  const int cnt_row = nslot * (NT + 1);               // array length with padded rows (see sidx)
  double *sT = reinterpret_cast<double *>(dyn_smem);
  double *sP = sT + cnt_row;
  double *sA = sP + cnt_row;

  uint32_t gen = 0;
  if (tid == 0) {
    ctx.abort_local = 0; ctx.list_n = 0; ctx.list_buf = 0; ctx.more = 0; ctx.any_odd = 0;
    ctx.second = ~0ull; ctx.second_k = 0x7fffffff;
  }
  if (CLUSTER && tid == 0) {
    mbar_init(smem_addr(&ctx.cl_bar[0]), 1u);
    mbar_init(smem_addr(&ctx.cl_bar[1]), 1u);
    mbar_fence_init();
  }
  if (is_stream) { dirty[tid] = 0; repick[tid] = 0; newcand[tid] = -1; mask_store(advm, tid, 0); mask_store(refm, tid, 0); mybest_k[tid] = -3; }
  __syncthreads();
  Cand none; none.dt = INF; none.k = 0x7fffffff;

  for (u64 it = (u64)b; it < p.n_traj; it += (u64)p.B) {
    const u64 traj = p.traj_first + it;
    const bool tracing = (it == 0) && p.trace_cap > 0 && r == 0;

    // ---- a-0: X = x0 (version 0), then T = 0, P = E(k,0), a = a(X0), n = 0 for the own range
    for (int j = r * BLOCK + tid; j < N; j += p.S * BLOCK) __stcg(X + j, x_pack(0ull, p.x0[j]));
    if (!bundle_barrier<BLOCK, CLUSTER>(exch, p.S, r, gen, p.err)) return;
    if (!CLUSTER) gen += 1u;
    for (int k = k0 + tid; k < k0 + cnt_pad; k += BLOCK) {
      double a0 = 0.0, t_init = 0.0, p_init = 1.0;   // padding: a = 0, P - T = 1: key +inf, never NaN
      uint32_t n_init = 0u;
      if (k < k1 && k < M) {
        a0 = propensity(net, X, k);
        if (filter_unsafe(a0)) ctx.any_odd = 1;
        if (p.T0) {
          t_init = __ldg(p.T0 + k); p_init = __ldg(p.P0 + k); n_init = __ldg(p.n0 + k);
        } else {
          const double e0 = exp_draw(p.seed, traj, (uint32_t)k, 0u);
          t_init = resid ? -e0 : 0.0; p_init = resid ? 0.0 : e0;
        }
      } else if (resid) { t_init = -1.0; p_init = 0.0; }
      const int si = sidx<NT>(k - k0);
      sT[si] = t_init; sP[si] = p_init; sA[si] = a0;
      if (k < k1) nfire[k] = n_init;
    }
    __syncthreads();
    // candidates of the first firing (nothing to advance)
    int cand_slot = -1;
    if (is_stream) {
      cand_slot = pass_and_pick<NT>(tid, cnt_row, sT, sP, sA, 0.0, ~0ull, ctx.any_odd != 0);
      mybest_k[tid] = cand_slot >= 0 ? k0 + tid + cand_slot * NT : -3;
      dirty[tid] = cand_slot < 0;
    }
    __syncthreads();

    double t = p.t0, dprev = 0.0;
    u64 fired = 0;
    int mu_prev = -1, stop = 0, status = RT_OK;
    bool finishing = false;
    int cur = 0;                         // staged-list buffer this firing publishes
    // walker warp: what it has prepared for the likely next winner
    int k2 = 0x7fffffff;                 //   runner-up of the last exchange
    bool want2 = false;                  //   ... still to be fetched from ctx.second (tag tag2)
    uint32_t tag2 = 0u;
    int pw_k = -1, pw_n = 0;             //   pre-walked reaction: its entries in [k0, k1) are in pw_d / pw_c
    int4 pw_ent = make_int4(-1, 0, 0, 0);//   its stoich row (lanes 0..3)
    bool sp_valid = false, sp_bad = false;  // speculative refreshes of pw_k in out_*[1 - cur], computed
    u64 sp_state = 0;                    //   from X after firing number sp_state
    long long sp_xn = 0;                 //   new count of the changed species of lane e < 4
    int pf_k = -1;                       // exchange warp: candidate whose walk data was last prefetched
    int spec_k = -1;                     // stream thread: the precomputed redraw of its candidate:
    uint32_t spec_n = 0u;                //   its new firing count and
    double spec_P = 0.0;                 //   new internal firing time P_k + E(seed, traj, k, n)

    for (;;) {   // one iteration per firing, plus one closing pass
      Cand best = none, extra = none;
      if (is_stream) {
        // ===== S1: advance and divide the candidate; also advance the reaction that fired
        u64 mask = 0;
        if (cand_slot >= 0) {
          const int i = tid + cand_slot * (NT + 1);
          const double a = sA[i];
          const double tn = __dadd_rn(sT[i], __dmul_rn(a, dprev));
          sT[i] = tn;
          best.dt = waiting_time(sP[i], tn, a);
          best.k = k0 + tid + cand_slot * NT;
          mask = 1ull << cand_slot;
        }
        if (mu_prev >= k0 && mu_prev < k1 && (mu_prev - k0) % NT == tid) {
          // a-7: this thread owns the reaction that fired: new internal firing time (Eq.26), as a rule
          // precomputed when the reaction became the thread's candidate (S5)
          const int i = sidx<NT>(mu_prev - k0);
          const u64 bit = 1ull << ((mu_prev - k0) / NT);
          if (spec_k != mu_prev) {
            spec_n = nfire[mu_prev] + 1u;
            const double e_new = exp_draw(p.seed, traj, (uint32_t)mu_prev, spec_n);
            spec_P = resid ? -e_new : __dadd_rn(sP[i], e_new);
          }
          if (resid) {
            sT[i] = spec_P;                              // Table 3: R_mu = ln(1/r), kept as T = -R
          } else {
            if (!(mask & bit)) sT[i] = __dadd_rn(sT[i], __dmul_rn(sA[i], dprev));
            sP[i] = spec_P;
          }
          mask |= bit;
          nfire[mu_prev] = spec_n;
          spec_k = -1;
          dirty[tid] = 1;                                // its proposal (if it was mu) is void
        }
        mask_store(advm, tid, mask);
        dcand[tid] = best.dt;
      } else if (is_walker) {
        // ===== walker warp: a-6 of the firing and its refreshes (a-1)
        int n = 0;
        bool more = false;
        Ranges rg;
#pragma unroll
        for (int e = 0; e < 4; ++e) { rg.lo[e] = 0; rg.end[e] = 0; }
        uint32_t w_f = 0, w_e0 = 0;
        int w_e = 0, w_ne = 0;
        bool w_csr = false, hit = false;
        bool published = false;
        if (mu_prev >= 0) {
          hit = sp_valid && pw_k == mu_prev && sp_state + 1 == fired;
          if (hit) {
            // the refreshes are already in out_*[cur]: publish them at once
            n = pw_n;
            if (lane == 0) {
              if (sp_bad) ctx.abort_local = 1;
              ctx.list_n = n; ctx.list_buf = cur; ctx.more = 0;
            }
            named_arrive<NT + 32>(kBarStaged);
            published = true;
            // X += v_mu (a-6) with the counts known in advance
            if (!sp_bad && lane < 4 && pw_ent.x >= 0) atomicMax(X + pw_ent.x, x_pack(fired, sp_xn));
          }
          if (!hit) {
            int4 ent = make_int4(-1, 0, 0, 0);
            if (lane < 4) ent = __ldg(reinterpret_cast<const int4 *>(net.srow) + (size_t)mu_prev * 4 + lane);
            w_csr = __shfl_sync(0xffffffffu, ent.x, 0) == -2;
            if (!w_csr) {
              const bool active = ent.x >= 0;
              bool done = false;
              long long xn = 0;
              uint32_t lo = 0, hi = 0;
              if (active && k1 > k0) { lo = (uint32_t)ent.z; hi = (uint32_t)ent.w; narrow_range(net, lo, hi, k0, k1); }
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
              if (k1 <= k0) w_ne = 0;
            }
            __syncwarp();                          // this warp's X updates precede its reads below
          }
        }
        // rounds: one, unless this CTA has more than kListCap refreshes
        while (!published) {
          if (mu_prev >= 0) {
            n = 0;
            if (!w_csr) {
              more = walk_scan(net, rg, w_f, k0, k1, lane, n, list_d, out_a[cur]);
            } else {
              more = false;
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
                more = walk_scan(net, rg, w_f, k0, k1, lane, n, list_d, out_a[cur]);
                if (more) break;
                w_e += 1;
                w_f = 0;
              }
            }
            walk_finish<false>(p, 1.0, X, lane, n, list_d, out_k[cur], out_a[cur]);
          }
          if (lane == 0) { ctx.list_n = n; ctx.list_buf = cur; ctx.more = more ? 1 : 0; }
          if (!more) { named_arrive<NT + 32>(kBarStaged); break; }
          named_sync<NT + 32>(kBarStaged);
          named_sync<NT + 32>(kBarMore);           // the stream warps have consumed this round
        }
      }

      if (is_xw && lane == 0 && mu_prev >= 0 && tracing && fired - 1 < p.trace_cap) {   // a-8
        if (p.trace_mu) p.trace_mu[fired - 1] = mu_prev;
        if (p.trace_t) p.trace_t[fired - 1] = t;
      }

      if (is_stream) {
        for (;;) {
          named_sync<NT + 32>(kBarStaged);
          // ===== S2: apply the staged refreshes
          const int n = ctx.list_n;
          const bool more = ctx.more != 0;
          const int *lk = out_k[ctx.list_buf];
          const double *la = out_a[ctx.list_buf];
          for (int i = tid; i < n; i += NT) {
            const int k = lk[i];
            const double a_new = la[i];
            const int o = (k - k0) % NT, slot = (k - k0) / NT, li = o + slot * (NT + 1);   // li: index in shared memory
            const int ob = mybest_k[o];
            const double t_old = sT[li], a_old = sA[li], pk = sP[li];
            if (!mask_claim(refm, o, slot)) continue;         // (a reaction reading two changed species is listed twice)
            // T_k += a_k dt with the OLD a_k, once: S1 has advanced exactly the owner's candidate and mu
            double tk = t_old;
            if (ob != k && k != mu_prev) {
              tk = __dadd_rn(t_old, __dmul_rn(a_old, dprev));
              sT[li] = tk;
              atomicOr(&advm[o][slot >> 5], 1u << (slot & 31));
            }
            sA[li] = a_new;
            if (filter_unsafe(a_new)) ctx.any_odd = 1;
            // A refreshed reaction invalidates its owner's proposal only if it IS that proposal;
            // otherwise its new waiting time joins the reduction as one more candidate.
            if (ob == k || ob == -3 || k == mu_prev) {
              dirty[o] = 1;
            } else {
              const double d = waiting_time(pk, tk, a_new);
              if (cand_less(d, k, extra)) { extra.dt = d; extra.k = k; }
              // The owner keeps its candidate while every other reaction of it stays clear of it (2^-13
              // relative: 256 key units).  A refreshed reaction clearly BELOW the candidate simply becomes
              // the candidate (everything else is above the old one); anything in between, a second such
              // reaction, or one outside the cancellation guard sends the owner to a full re-pick.
              const double dc = dcand[o];
              if (!(d > __dmul_rn(dc, 1.0 + 0x1.0p-13))) {
                const bool guard = __double2hiint(__dsub_rn(pk, tk)) + (kGuardShift << 20) >=
                                   max(__double2hiint(pk) & 0x7fffffff, __double2hiint(tk) & 0x7fffffff);
                if (d < __dmul_rn(dc, 1.0 - 0x1.0p-13) && d > 0.0 && guard && atomicCAS(&newcand[o], -1, slot) == -1) {}
                else repick[o] = 1;
              }
            }
          }
          if (!more) { named_sync<NT>(1); break; }
          named_sync<NT + 32>(kBarMore);
        }
        // ===== S3: exact re-scan of the threads without a valid candidate; the warp shares the work
        unsigned stale_mask = __ballot_sync(0xffffffffu, dirty[tid] != 0);
        const int n_stale = __popc(stale_mask);
        bool pick = dirty[tid] != 0 || repick[tid] != 0 || cand_slot < 0;
        if (dirty[tid]) dirty[tid] = 0;
        // Lane l takes slots l and l + 32 of the stale thread: advance, integer keys (as in the pass),
        // then exact divisions only for the slots whose key is within kQTolUnits of the smallest --
        // no other slot can hold the exact minimum.  Keys are not trusted (everything is divided) when
        // the smallest is outside [2^-100, 2^100] (zero or negative residuals, NaN) or under any_odd.
        int sq0 = 0x7fffffff, sq1 = 0x7fffffff, sm1 = 0x7fffffff;   // (kept for S5: the keys, their minimum,
        Cand swin = none;                                            //  the exact winner, the stale lane)
        int sL = -1;
        bool sguard = true;
        while (stale_mask) {
          const int L = __ffs(stale_mask) - 1;
          stale_mask &= stale_mask - 1;
          const int th = tid - lane + L;
          const u64 m = mask_load(advm, th);
          const int j0 = lane, j1 = lane + 32;
          const bool h0 = j0 < nslot, h1 = j1 < nslot;
          const int i0 = th + j0 * (NT + 1), i1 = th + j1 * (NT + 1);     // (shared memory)
          const int kk0 = k0 + th + j0 * NT, kk1 = kk0 + 32 * NT;        // (reactions)
          double a0 = 0.0, p0 = 1.0, t0 = 0.0, a1 = 0.0, p1 = 1.0, t1 = 0.0;
          if (h0) { a0 = sA[i0]; p0 = sP[i0]; t0 = sT[i0]; }
          if (h1) { a1 = sA[i1]; p1 = sP[i1]; t1 = sT[i1]; }
          if (h0 && !((m >> j0) & 1ull)) { t0 = __dadd_rn(t0, __dmul_rn(a0, dprev)); sT[i0] = t0; }
          if (h1 && !((m >> j1) & 1ull)) { t1 = __dadd_rn(t1, __dmul_rn(a1, dprev)); sT[i1] = t1; }
          sguard = true;
          sq0 = q_key(p0, t0, a0, sguard);
          sq1 = q_key(p1, t1, a1, sguard);
          sm1 = __reduce_min_sync(0xffffffffu, min(sq0, sq1));
          const bool trust = ctx.any_odd == 0 && sm1 >= ((1023 - 100) << 20) && sm1 <= ((1023 + 100) << 20);
          const int lim = trust ? sm1 + kQTolUnits : 0x7fffffff;
          Cand c = none;
          if (h0 && sq0 <= lim) { c.dt = waiting_time(p0, t0, a0); c.k = kk0; }
          if (h1 && sq1 <= lim) {
            const double d = waiting_time(p1, t1, a1);
            if (cand_less(d, kk1, c)) { c.dt = d; c.k = kk1; }
          }
          c = warp_lexmin(c);
          __syncwarp();
          swin = c; sL = L;
          if (!trust) sguard = false;
          if (lane == L) { best = c; mask_store(advm, tid, ~0ull); }
        }
        if (cand_less(extra.dt, extra.k, best)) best = extra;
        // ===== S4: block argmin -> exchange warp
        if (!finishing) {
          best = warp_lexmin(best);
          if (lane == 0) ctx.warp_part[warp] = best;
          named_arrive<NT + 32>(kBarParts);
        }
        // ===== S5: the pass, while the exchange is in flight
        // A thread keeps its candidate (and only advances) unless the candidate is void or may have
        // lost its margin; every kRepickPeriod firings the warp re-derives all of them, which bounds
        // the age of a candidate (the lag argument of the header needs age * 2 + 7 < kQTolUnits units).
        if (n_stale == 1) {
          // The re-scan decides the stale thread's new candidate as the pass would: the exact winner,
          // if every other key is clear of the smallest and the cancellation guard holds.
          const int wslot = (swin.k - k0 - (tid - lane + sL)) / NT;      // slot of the winner
          const int e0 = (wslot == lane) ? 0x7fffffff : sq0;
          const int e1 = (wslot == lane + 32) ? 0x7fffffff : sq1;
          const int sm2 = __reduce_min_sync(0xffffffffu, min(e0, e1));
          const bool ok = __all_sync(0xffffffffu, sguard) && swin.k < M && sm2 > sm1 + kQTolUnits;
          if (lane == sL && ok && !repick[tid]) {
            cand_slot = wslot;
            mybest_k[tid] = swin.k;
            pick = false;
            newcand[tid] = -1;                       // (the re-scan has seen every refreshed reaction)
          }
        }
        if (!pick && newcand[tid] >= 0) {            // (S2) a refreshed reaction took over as the candidate
          cand_slot = newcand[tid];
          mybest_k[tid] = k0 + tid + cand_slot * NT;
        }
        newcand[tid] = -1;
        pick = pick || (((unsigned)fired + (unsigned)warp) % kRepickPeriod == 0u);
        if (__any_sync(0xffffffffu, pick)) {
          cand_slot = pass_and_pick<NT>(tid, cnt_row, sT, sP, sA, dprev, mask_load(advm, tid), ctx.any_odd != 0);
          mybest_k[tid] = cand_slot >= 0 ? k0 + tid + cand_slot * NT : -3;
          if (cand_slot < 0) dirty[tid] = 1;
        } else {
          pass_advance<NT>(tid, cnt_row, sT, sA, dprev, mask_load(advm, tid));
        }
        repick[tid] = 0;
        mask_store(advm, tid, 0);
        mask_store(refm, tid, 0);
        // If the candidate fires, this thread must redraw its P_k: Philox + log, the longest serial piece
        // of a firing.  Do it now, off the critical path, once per candidate.
        if (cand_slot >= 0 && mybest_k[tid] != spec_k && (p.prefetch & 2)) {
          spec_k = mybest_k[tid];
          spec_n = nfire[spec_k] + 1u;
          const double e_new = exp_draw(p.seed, traj, (uint32_t)spec_k, spec_n);
          spec_P = resid ? -e_new : __dadd_rn(sP[sidx<NT>(spec_k - k0)], e_new);
        }
      } else if (is_xw) {
        if (!finishing) named_sync<NT + 32>(kBarParts);
      }
      if (ctx.abort_local) { status = RT_ERR_OVERFLOW; stop = 0; break; }
      if (finishing) break;

      // ---- a-3 argmin over the bundle
      Cand win;
      if (is_xw) {
        Cand c = none;
        if (lane < XW) c = ctx.warp_part[lane];
        c = warp_lexmin(c);
        const Cand mine = c;
        Cand c2;
        // Through L2 the runner-up is reduced after the winner is out: only the walker wants it, and
        // later (cfg4 3.16 -> 3.12 us, cfg5b +3 %).  In a cluster the walker is the busiest warp of
        // the firing and would wait for it: there it is published together with the winner.
        constexpr bool kDefer2 = !CLUSTER;
        exchange_partials<CLUSTER, NoWork, kDefer2>(p, ctx.cl_slot, ctx.cl_bar, exch, r, gen, lane, c, c2);
        if (lane == 0) ctx.win = c;
        if (!kDefer2 && lane == 0) ctx.second_k = (c2.dt < INF) ? c2.k : 0x7fffffff;
        named_arrive<BLOCK>(kBarWin);
        win = c;
        if (kDefer2) {
          c2 = warp_lexmin(c2);
          if (lane == 0)
            *reinterpret_cast<volatile u64 *>(&ctx.second) =
                ((u64)gen << 32) | (u64)(uint32_t)((c2.dt < INF) ? c2.k : 0x7fffffff);
        }
        // every CTA will need the candidate's stoich row and the dependency entries of its species,
        // all DRAM-cold (each reaction fires rarely): pull them into L2, once per candidate
        if (mine.k != pf_k && mine.k < M && (p.prefetch & 1)) {
          pf_k = mine.k;
          int4 ent = make_int4(-1, 0, 0, 0);
          if (lane < 4) ent = __ldg(reinterpret_cast<const int4 *>(net.srow) + (size_t)mine.k * 4 + lane);
#pragma unroll
          for (int e = 0; e < 4; ++e) {
            const int j = __shfl_sync(0xffffffffu, ent.x, e);
            const uint32_t lo = (uint32_t)__shfl_sync(0xffffffffu, ent.z, e);
            const uint32_t hi = (uint32_t)__shfl_sync(0xffffffffu, ent.w, e);
            if (j >= 0 && hi != 0xffffffffu)
              for (uint32_t i = lo + 4u * lane; i < hi; i += 128u)
                prefetch_l2(reinterpret_cast<const char *>(net.dep) + (size_t)i * 32);
          }
        }
      } else {
        if (is_walker) {
          // ===== walker: prepare the likely next winner k2 while the others reduce and exchange
          // (1) its dependency entries in [k0, k1) (network data): row -> ranges -> entries
          if (want2) {                   // (written by the exchange warp right after the last winner)
            u64 v;
            do { v = *reinterpret_cast<volatile u64 *>(&ctx.second); } while ((uint32_t)(v >> 32) != tag2);
            k2 = (int)(uint32_t)v;
            want2 = false;
          }
          if ((p.prefetch & 4) && k2 != pw_k && k2 < M && k1 > k0) {
            pw_k = -1;
            int4 ent = make_int4(-1, 0, 0, 0);
            if (lane < 4) ent = __ldg(reinterpret_cast<const int4 *>(net.srow) + (size_t)k2 * 4 + lane);
            if (__shfl_sync(0xffffffffu, ent.x, 0) != -2) {
              uint32_t lo = 0, hi = 0;
              if (ent.x >= 0) { lo = (uint32_t)ent.z; hi = (uint32_t)ent.w; narrow_range(net, lo, hi, k0, k1); }
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
              if (!walk_scan(net, rg, f, k0, k1, lane, n, pw_d, pw_c)) { pw_k = k2; pw_n = n; pw_ent = ent; }
            }
          }
          // (2) its refreshes, computed from X as it will be after it fires: X now (this warp's own
          // updates of every firing so far precede these loads: __syncwarp) plus its own v.  Another
          // CTA of the bundle may already be one firing ahead (the exchange needs this CTA's exchange
          // warp, not this warp): a word of version fired + 1 already holds that firing's change,
          // which is k2's own if the guess is right (and if it is wrong the result is never used).
          sp_valid = false;
          if ((p.prefetch & 4) && pw_k >= 0 && pw_k == k2) {
            __syncwarp();
            int cj[4], cv[4];
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              cj[e] = __shfl_sync(0xffffffffu, pw_ent.x, e);
              cv[e] = __shfl_sync(0xffffffffu, pw_ent.y, e);
            }
            bool bad = false, general = false;
            sp_xn = 0;
            if (lane < 4 && pw_ent.x >= 0) {
              const u64 w = __ldcg(X + pw_ent.x);
              sp_xn = x_count(w) + (x_version(w) <= fired ? (long long)pw_ent.y : 0ll);
              bad = sp_xn < 0 || sp_xn > net.xmax;
            }
            int *ok = out_k[1 - cur];
            double *oa = out_a[1 - cur];
            for (int i = lane; i < pw_n; i += 32) {
              const int4 d = pw_d[i];
              if (d.w & 0x10000) { general = true; continue; }   // > 2 reactants: not speculated
              const u64 w1 = __ldcg(X + d.y);
              const u64 w2 = __ldcg(X + (d.z >= 0 ? d.z : d.y));
              long long x1 = x_count(w1), x2 = x_count(w2);
#pragma unroll
              for (int e = 0; e < 4; ++e) {
                if (cj[e] == d.y && x_version(w1) <= fired) x1 += (long long)cv[e];
                if (cj[e] == d.z && x_version(w2) <= fired) x2 += (long long)cv[e];
              }
              double a = __dmul_rn(pw_c[i], __ll2double_rn(binom(x1, d.w & 0xff)));
              if (d.z >= 0) a = __dmul_rn(a, __ll2double_rn(binom(x2, (d.w >> 8) & 0xff)));
              ok[i] = d.x;
              oa[i] = a;
            }
            sp_bad = __any_sync(0xffffffffu, bad);
            sp_valid = !__any_sync(0xffffffffu, general);
            sp_state = fired;
          }
        }
        named_sync<BLOCK>(kBarWin);
        win = ctx.win;
        if (is_walker) {
          if (CLUSTER) k2 = ctx.second_k;
          else { want2 = true; tag2 = gen; }
        }
      }
      gen += 1u;
      cur ^= 1;
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
      if (fired >= kXMaxVersion) { status = RT_ERR_OVERFLOW; break; }
      t = __dadd_rn(t, delta);
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
    for (int k = k0 + tid; k < k1; k += BLOCK) {
      const int si = sidx<NT>(k - k0);
      __stcg(T + k, sT[si]); __stcg(P + k, sP[si]); __stcg(A + k, sA[si]);
    }
    if (p.x_out)
      for (int j = r * BLOCK + tid; j < N; j += p.S * BLOCK)
        p.x_out[it * (u64)N + (u64)j] = x_load(X, j);
    if (r == 0 && tid == 0) {
      rt_result res;
      res.t = t; res.firings = fired; res.stop = stop; res.status = status;
      p.res[it] = res;
    }
    if (tid == 0) { ctx.abort_local = 0; ctx.any_odd = 0; }
    if (is_stream) { dirty[tid] = 0; repick[tid] = 0; newcand[tid] = -1; mask_store(advm, tid, 0); mask_store(refm, tid, 0); }
    __syncthreads();
  }
}

}  // namespace rt
