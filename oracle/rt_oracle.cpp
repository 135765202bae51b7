// rt_oracle.cpp -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, single-threaded fp64 reference ("oracle") of the next-reaction
// random-time algorithm (NRRTA) of Liu & Wang, arXiv 2103.00405, written from the
// paper and used only to check the CUDA path.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no
// code, header, table or constant generator with paper_2103_00405_b200/.
//
// Build: g++ -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (see oracle/build.py).
// -ffp-contract=off: every product and sum below is one IEEE-754 binary64
// round-to-nearest operation, in exactly the order written.
//
// What each function follows (PAPER.md = /root/reference/PAPER.md, SURVEY = SURVEY.md):
//   binom()          Eq.2, reading G1/G2 (index garbled: h_k = prod_j C(X_j, sigma_jk))
//   propensity()     Eq.1-2: a_k = c_k * prod_j C(X_j, sigma_jk)
//   philox4x32_10()  Salmon et al., SC'11 (counter-based RNG that north_star substitutes
//                    for the paper's CPU Mersenne Twister)
//   exp_draw()       Eq.23: Delta T = ln(1/r), r uniform; reading G5: r in (0,1]
//   nrrta_run()      Eq.15 internal time T_k = int a_k ds;
//                    Eq.24 with a_k constant between firings:
//                       Delta t_k = (P_k - T_k)/a_k;
//                    Eq.25 first arrival wins: Delta t = min_k Delta t_k;
//                    Eq.26 only the fired channel draws a new
//                       internal-time target; Table 1/3 loop shape;
//                    Eq.5 X += v_mu.
//                    Table 2 (the NRRTA listing) lost its body in PAPER.md:258-260; the
//                    (T_k, P_k) bookkeeping is reading G3 of DESIGN.md.
//   nrrta_run_sched()     Eq.28 with piecewise-constant c_k(t)
//   nrrta_run_rate_exp()  Eq.28 with c_k(t) = c_k exp(lambda_k t), solved per channel
//   nrrta_run_residual()  Table 3 in residual-internal-time form (reading G4)
//   Start / oracle_run_from()  the same two loops started from a checkpoint (t, T, P or R, n)
//                    instead of step 0 -- no arithmetic of its own; pinned by the prefix identity
//                    run(n1) + run_from(n2 - n1) == run(n2) and used to build exact finite ties
//   apply_firing()   Eq.5 plus the count bound of reading G2 (Overflow)
//   direct-method cross-check lives in tests/ (it must not share code with this file).
//
// Parity pins (tests/test_oracle_*.py): Philox known-answer vectors and the CUDA toolkit's
// curand_Philox4x32_10; single-channel closed form t_n = sum E_i / c; birth-death
// Poisson law; Kurtz identity Eq.5; invariants; race of exponentials; binomial factor;
// brute-force Gillespie direct method on tiny networks; exact finite ties (reading G6) built from
// rate_k = E(k,0) * 2^-3 and from checkpointed states.  Exact sample paths of the
// large configs are fixed by no number in the paper: oracle<->GPU parity only.

#include <cstdint>
#include <cstddef>
#include <cmath>
#include <limits>
#include <thread>
#include <vector>

namespace {

// ---------------------------------------------------------------- Philox4x32-10
// Salmon, Moraes, Dror, Shaw: "Parallel random numbers: as easy as 1, 2, 3" (SC'11).
// Ten rounds; round multipliers 0xD2511F53 / 0xCD9E8D57; Weyl key increments
// 0x9E3779B9 / 0xBB67AE85.
void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
  uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
  uint32_t k0 = key_in[0], k1 = key_in[1];
  for (int round = 0; round < 10; ++round) {
    const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// E(seed, trajectory, reaction k, draw number n): the n-th unit-exponential internal-time
// increment of channel k (Eq.23: Delta T_k = ln(1/r_k)).
// key = (lo32 seed, hi32 seed); counter = (k, lo32 n, lo32 traj, hi32 traj).
// r = (u53 + 1) * 2^-53 in (0,1]  (reading G5: the paper's closed [0,1] would allow ln(1/0)).
double exp_draw(uint64_t seed, uint64_t traj, uint32_t k, uint32_t n) {
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  const uint32_t ctr[4] = {k, n, (uint32_t)traj, (uint32_t)(traj >> 32)};
  uint32_t w[4];
  philox4x32_10(ctr, key, w);
  const uint64_t u53 = (((uint64_t)w[1] << 32) | (uint64_t)w[0]) >> 11;
  const double r = (double)(u53 + 1) * 0x1.0p-53;   // exact: u53+1 <= 2^53
  return -std::log(r);
}

// C(x, sigma) as an exact integer (reading G2).  x < sigma gives 0.
int64_t binom(int64_t x, int32_t sigma) {
  switch (sigma) {
    case 1: return x;
    case 2: return x * (x - 1) / 2;
    case 3: return (x * (x - 1) / 2) * (x - 2) / 3;
    default: return -1;   // rejected before any run
  }
}

struct Net {
  int32_t N, M;
  const int64_t *react_ptr; const int32_t *react_species, *react_sigma;
  const int64_t *stoich_ptr; const int32_t *stoich_species, *stoich_v;
  const double *rate;
};

// a_k = c_k * prod_j C(X_j, sigma_jk): one rounded multiply per reactant entry, CSR order.
double propensity(const Net &net, const int64_t *X, int32_t k) {
  double a = net.rate[k];
  for (int64_t e = net.react_ptr[k]; e < net.react_ptr[k + 1]; ++e) {
    const int64_t b = binom(X[net.react_species[e]], net.react_sigma[e]);
    a = a * (double)b;
  }
  return a;
}

enum { STOP_T_END = 1, STOP_MAX_FIRINGS = 2, STOP_ABSORBED = 3 };
enum { OK = 0, ERR_BAD = -1, ERR_OVERFLOW = -5 };

// Optional starting point of a run (checkpoint / resume): the state a previous run returned.
// T, P (or R for the residual form) and n may each be NULL = fresh (T = 0, P = E(k, 0), n = 0).
struct Start {
  double t;
  const double *T, *P;
  const uint64_t *n;
};

int64_t count_bound(const Net &net) {
  int32_t smax = 1;
  for (int64_t e = 0; e < net.react_ptr[net.M]; ++e)
    if (net.react_sigma[e] > smax) smax = net.react_sigma[e];
  return smax <= 2 ? (((int64_t)1 << 31) - 1) : (((int64_t)1 << 21) - 1);
}

// Step 6, X += v_mu (Eq.5), with the count bound of reading G2: if any count of the row would
// leave [0, xmax] the whole update is skipped and the run ends with ERR_OVERFLOW (DESIGN.md
// section 2, "Overflow": the firing is counted and traced, its internal-time increment and redraw
// are applied, its change of X is not).
int apply_firing(const Net &net, int64_t *X, int32_t mu, int64_t xmax) {
  for (int64_t e = net.stoich_ptr[mu]; e < net.stoich_ptr[mu + 1]; ++e) {
    const int64_t xj = X[net.stoich_species[e]] + net.stoich_v[e];
    if (xj < 0 || xj > xmax) return ERR_OVERFLOW;
  }
  for (int64_t e = net.stoich_ptr[mu]; e < net.stoich_ptr[mu + 1]; ++e)
    X[net.stoich_species[e]] += net.stoich_v[e];
  return OK;
}

int nrrta_run(const Net &net, const int64_t *x0, const Start *start, uint64_t seed, uint64_t traj,
              uint64_t max_firings, double t_end,
              int64_t *x_out, double *t_out, uint64_t *firings_out, int32_t *stop_out,
              uint64_t *fire_count_out, double *T_out, double *P_out,
              int32_t *trace_mu, double *trace_t, uint64_t trace_cap) {
  const int32_t M = net.M, N = net.N;
  const double INF = std::numeric_limits<double>::infinity();
  const int64_t xmax = count_bound(net);
  for (int64_t e = 0; e < net.react_ptr[M]; ++e)
    if (net.react_sigma[e] < 1 || net.react_sigma[e] > 3) return ERR_BAD;

  std::vector<int64_t> X(x0, x0 + N);
  for (int32_t j = 0; j < N; ++j) if (X[j] < 0 || X[j] > xmax) return ERR_BAD;
  std::vector<double> T(M, 0.0), P(M), a(M), dt(M);
  std::vector<uint32_t> n(M, 0u);

  // step 0: T_k = 0, P_k = first internal firing time of the unit-rate process Y_k -- or the
  // checkpointed values when the run resumes one.
  for (int32_t k = 0; k < M; ++k) P[k] = exp_draw(seed, traj, (uint32_t)k, 0u);
  double t = 0.0;
  if (start) {
    t = start->t;
    if (start->T) for (int32_t k = 0; k < M; ++k) T[k] = start->T[k];
    if (start->P) for (int32_t k = 0; k < M; ++k) P[k] = start->P[k];
    if (start->n) for (int32_t k = 0; k < M; ++k) n[k] = (uint32_t)start->n[k];
  }
  uint64_t fired = 0;
  int32_t stop = 0;
  int rc = OK;

  for (;;) {
    // step 1: every propensity from the current state.
    for (int32_t k = 0; k < M; ++k) a[k] = propensity(net, X.data(), k);
    // step 2: real waiting time of every channel (Eq.24 with constant a_k).
    for (int32_t k = 0; k < M; ++k) {
      if (a[k] > 0.0) {
        double r = P[k] - T[k];
        if (r < 0.0) r = 0.0;          // reading G7: rounding may leave T an ulp past P
        dt[k] = r / a[k];
      } else {
        dt[k] = INF;
      }
    }
    // step 3: first arrival wins (Eq.25); ties to the lowest index (reading G6).
    int32_t mu = 0;
    double delta = dt[0];
    for (int32_t k = 1; k < M; ++k)
      if (dt[k] < delta) { delta = dt[k]; mu = k; }
    if (delta == INF) { stop = STOP_ABSORBED; break; }
    // step 4: never fire past t_end (reading G8); bring the internal clocks to t_end.
    if (t_end < INF && t + delta > t_end) {
      const double rest = t_end - t;
      for (int32_t k = 0; k < M; ++k) { const double inc = a[k] * rest; T[k] = T[k] + inc; }
      t = t_end;
      stop = STOP_T_END;
      break;
    }
    // step 5: advance real time and every internal time (Eq.15), a_k of step 1.
    t = t + delta;
    for (int32_t k = 0; k < M; ++k) { const double inc = a[k] * delta; T[k] = T[k] + inc; }
    // step 6: X += v_mu (Eq.5).
    rc = apply_firing(net, X.data(), mu, xmax);
    // step 7: only the fired channel gets a new internal-time target (Eq.26).
    n[mu] += 1u;
    P[mu] = P[mu] + exp_draw(seed, traj, (uint32_t)mu, n[mu]);
    if (fired < trace_cap) {
      if (trace_mu) trace_mu[fired] = mu;
      if (trace_t) trace_t[fired] = t;
    }
    fired += 1;
    if (rc != OK) break;
    if (max_firings != 0 && fired == max_firings) { stop = STOP_MAX_FIRINGS; break; }
  }

  if (x_out) for (int32_t j = 0; j < N; ++j) x_out[j] = X[j];
  if (t_out) *t_out = t;
  if (firings_out) *firings_out = fired;
  if (stop_out) *stop_out = stop;
  if (fire_count_out) for (int32_t k = 0; k < M; ++k) fire_count_out[k] = n[k];
  if (T_out) for (int32_t k = 0; k < M; ++k) T_out[k] = T[k];
  if (P_out) for (int32_t k = 0; k < M; ++k) P_out[k] = P[k];
  return rc;
}


// ---------------------------------------------------------------- residual ("Table 3") form
// PAPER.md Table 3 (:262-272), the memory-lean parallel listing: per channel only the remaining
// real waiting time is kept and rescaled, Delta t_k <- (p_k / a_k)(Delta t_k - Delta t_mu) with
// p_k the previous propensity, and the fired channel draws Delta t_mu = ln(1/r) / a_mu.
// Reading G4: written with the residual INTERNAL time R_k = a_k^old (Delta t_k - Delta t_mu)
// = P_k - T_k it is the same process without the division by a_k = 0:
//     Delta t_k = R_k / a_k,   R_k <- R_k - a_k * Delta t_mu for every k,   R_mu <- ln(1/r).
// Same law as nrrta_run, different rounding (one array instead of two), so sample paths differ
// in the last bits and eventually in the fired sequence: its own parity target.
int nrrta_run_residual(const Net &net, const int64_t *x0, const Start *start, uint64_t seed, uint64_t traj,
                       uint64_t max_firings, double t_end,
                       int64_t *x_out, double *t_out, uint64_t *firings_out, int32_t *stop_out,
                       uint64_t *fire_count_out, double *R_out,
                       int32_t *trace_mu, double *trace_t, uint64_t trace_cap) {
  const int32_t M = net.M, N = net.N;
  const double INF = std::numeric_limits<double>::infinity();
  const int64_t xmax = count_bound(net);
  for (int64_t e = 0; e < net.react_ptr[M]; ++e)
    if (net.react_sigma[e] < 1 || net.react_sigma[e] > 3) return ERR_BAD;
  std::vector<int64_t> X(x0, x0 + N);
  for (int32_t j = 0; j < N; ++j) if (X[j] < 0 || X[j] > xmax) return ERR_BAD;
  std::vector<double> R(M), a(M), dt(M);
  std::vector<uint32_t> n(M, 0u);
  for (int32_t k = 0; k < M; ++k) R[k] = exp_draw(seed, traj, (uint32_t)k, 0u);
  double t = 0.0;
  if (start) {             // resume: start->P holds the checkpointed residuals R_k
    t = start->t;
    if (start->P) for (int32_t k = 0; k < M; ++k) R[k] = start->P[k];
    if (start->n) for (int32_t k = 0; k < M; ++k) n[k] = (uint32_t)start->n[k];
  }
  uint64_t fired = 0;
  int32_t stop = 0;
  int rc = OK;
  for (;;) {
    for (int32_t k = 0; k < M; ++k) a[k] = propensity(net, X.data(), k);
    for (int32_t k = 0; k < M; ++k) {
      if (a[k] > 0.0) {
        double r = R[k];
        if (r < 0.0) r = 0.0;          // reading G7
        dt[k] = r / a[k];
      } else {
        dt[k] = INF;
      }
    }
    int32_t mu = 0;
    double delta = dt[0];
    for (int32_t k = 1; k < M; ++k)
      if (dt[k] < delta) { delta = dt[k]; mu = k; }
    if (delta == INF) { stop = STOP_ABSORBED; break; }
    if (t_end < INF && t + delta > t_end) {
      const double rest = t_end - t;
      for (int32_t k = 0; k < M; ++k) { const double dec = a[k] * rest; R[k] = R[k] - dec; }
      t = t_end;
      stop = STOP_T_END;
      break;
    }
    t = t + delta;
    for (int32_t k = 0; k < M; ++k) { const double dec = a[k] * delta; R[k] = R[k] - dec; }
    rc = apply_firing(net, X.data(), mu, xmax);
    n[mu] += 1u;
    R[mu] = exp_draw(seed, traj, (uint32_t)mu, n[mu]);     // Table 3: a fresh ln(1/r) for mu only
    if (fired < trace_cap) {
      if (trace_mu) trace_mu[fired] = mu;
      if (trace_t) trace_t[fired] = t;
    }
    fired += 1;
    if (rc != OK) break;
    if (max_firings != 0 && fired == max_firings) { stop = STOP_MAX_FIRINGS; break; }
  }
  if (x_out) for (int32_t j = 0; j < N; ++j) x_out[j] = X[j];
  if (t_out) *t_out = t;
  if (firings_out) *firings_out = fired;
  if (stop_out) *stop_out = stop;
  if (fire_count_out) for (int32_t k = 0; k < M; ++k) fire_count_out[k] = n[k];
  if (R_out) for (int32_t k = 0; k < M; ++k) R_out[k] = R[k];
  return rc;
}


// ---------------------------------------------------------------- time-dependent rates
// PAPER.md section 6, Eq.28 (:224-231): with rates c_k(s) that depend on time, channel k fires when
//     h_k * int_t^{t+dt_k} c_k(s) ds = P_k - T_k,        h_k = prod_j C(X_j, sigma_jk),
// and "the integral can be calculated analytically for well behaved time-dependent reaction
// rates" (:229).  The family built here is piecewise-constant modulation: c_k(s) = c_k * f_i for
// s in [b_i, b_{i+1}) (f = 1 before b_0) for the channels selected by `mask` (all if NULL), the
// others keep c_k.  The integral is then piecewise linear, so between two breakpoints the step
// is Eq.24 unchanged, and a step that would cross the next breakpoint b is cut there:
// T_k += a_k (b - t) for every k, t = b, no firing, rates switch to the next factor.
// The effective rate is one rounded product RN(c_k * f_i), then Eq.1-2 as before.
double propensity_eff(const Net &net, const int64_t *X, int32_t k, double f, const uint8_t *mask) {
  double a = net.rate[k];
  if (mask == nullptr || mask[k]) a = a * f;
  for (int64_t e = net.react_ptr[k]; e < net.react_ptr[k + 1]; ++e) {
    const int64_t b = binom(X[net.react_species[e]], net.react_sigma[e]);
    a = a * (double)b;
  }
  return a;
}

int nrrta_run_sched(const Net &net, const int64_t *x0, uint64_t seed, uint64_t traj,
                    uint64_t max_firings, double t_end,
                    int32_t n_break, const double *t_break, const double *factor, const uint8_t *mask,
                    int64_t *x_out, double *t_out, uint64_t *firings_out, int32_t *stop_out,
                    uint64_t *fire_count_out, double *T_out, double *P_out,
                    int32_t *trace_mu, double *trace_t, uint64_t trace_cap) {
  const int32_t M = net.M, N = net.N;
  const double INF = std::numeric_limits<double>::infinity();
  const int64_t xmax = count_bound(net);
  for (int64_t e = 0; e < net.react_ptr[M]; ++e)
    if (net.react_sigma[e] < 1 || net.react_sigma[e] > 3) return ERR_BAD;
  for (int32_t i = 0; i < n_break; ++i) {
    if (!(t_break[i] >= 0.0) || !(factor[i] >= 0.0) || factor[i] == INF || t_break[i] == INF) return ERR_BAD;
    if (i > 0 && !(t_break[i] > t_break[i - 1])) return ERR_BAD;
  }
  std::vector<int64_t> X(x0, x0 + N);
  for (int32_t j = 0; j < N; ++j) if (X[j] < 0 || X[j] > xmax) return ERR_BAD;
  std::vector<double> T(M, 0.0), P(M), a(M), dt(M);
  std::vector<uint32_t> n(M, 0u);
  for (int32_t k = 0; k < M; ++k) P[k] = exp_draw(seed, traj, (uint32_t)k, 0u);
  double t = 0.0, f = 1.0;
  int32_t seg = 0;                      // breakpoints already passed
  uint64_t fired = 0;
  int32_t stop = 0;
  int rc = OK;
  for (;;) {
    for (int32_t k = 0; k < M; ++k) a[k] = propensity_eff(net, X.data(), k, f, mask);
    for (int32_t k = 0; k < M; ++k) {
      if (a[k] > 0.0) {
        double r = P[k] - T[k];
        if (r < 0.0) r = 0.0;
        dt[k] = r / a[k];
      } else {
        dt[k] = INF;
      }
    }
    int32_t mu = 0;
    double delta = dt[0];
    for (int32_t k = 1; k < M; ++k)
      if (dt[k] < delta) { delta = dt[k]; mu = k; }
    // the next breakpoint (if it lies within the run) cuts the step
    const double tb = (seg < n_break && t_break[seg] <= t_end) ? t_break[seg] : INF;
    if (tb < INF && (delta == INF || t + delta > tb)) {
      const double rest = tb - t;
      for (int32_t k = 0; k < M; ++k) { const double inc = a[k] * rest; T[k] = T[k] + inc; }
      t = tb;
      f = factor[seg];
      seg += 1;
      continue;
    }
    if (delta == INF) { stop = STOP_ABSORBED; break; }
    if (t_end < INF && t + delta > t_end) {
      const double rest = t_end - t;
      for (int32_t k = 0; k < M; ++k) { const double inc = a[k] * rest; T[k] = T[k] + inc; }
      t = t_end;
      stop = STOP_T_END;
      break;
    }
    t = t + delta;
    for (int32_t k = 0; k < M; ++k) { const double inc = a[k] * delta; T[k] = T[k] + inc; }
    rc = apply_firing(net, X.data(), mu, xmax);
    n[mu] += 1u;
    P[mu] = P[mu] + exp_draw(seed, traj, (uint32_t)mu, n[mu]);
    if (fired < trace_cap) {
      if (trace_mu) trace_mu[fired] = mu;
      if (trace_t) trace_t[fired] = t;
    }
    fired += 1;
    if (rc != OK) break;
    if (max_firings != 0 && fired == max_firings) { stop = STOP_MAX_FIRINGS; break; }
  }
  if (x_out) for (int32_t j = 0; j < N; ++j) x_out[j] = X[j];
  if (t_out) *t_out = t;
  if (firings_out) *firings_out = fired;
  if (stop_out) *stop_out = stop;
  if (fire_count_out) for (int32_t k = 0; k < M; ++k) fire_count_out[k] = n[k];
  if (T_out) for (int32_t k = 0; k < M; ++k) T_out[k] = T[k];
  if (P_out) for (int32_t k = 0; k < M; ++k) P_out[k] = P[k];
  return rc;
}

// ---------------------------------------------------------------- smooth time-dependent rates
// PAPER.md section 6, Eq.28 (:224-231) with a rate that varies smoothly in time, the case the paper
// means by "the integral can be calculated analytically for well behaved time-dependent reaction
// rates" (:229): the exponential family c_k(s) = c_k * exp(lambda_k * s), per-channel lambda_k
// (decay < 0, growth > 0, 0 = constant).  With h_k = prod_j C(X_j, sigma_jk) constant between
// firings and a_k(t) = c_k h_k exp(lambda_k t) the propensity at the start of the step,
//     int_t^{t+d} c_k(s) h_k ds = a_k(t) * (exp(lambda_k d) - 1) / lambda_k,
// so channel k's own equation of Eq.28, P_k - T_k = that integral, has the closed-form solution
//     dt_k = log1p(lambda_k (P_k - T_k) / a_k(t)) / lambda_k,
// which is +inf when lambda_k (P_k - T_k) / a_k(t) <= -1 (a decaying channel whose whole remaining
// integral a_k(t)/|lambda_k| is smaller than its residual never fires again), and the internal
// clocks advance by T_k += a_k(t) * (expm1(lambda_k d) / lambda_k)  (Eq.15 with Eq.1 inside).
// lambda_k = 0 takes the constant-rate formulas of nrrta_run literally, so a run with every
// lambda_k = 0 is nrrta_run bit for bit.  Operation order, each step one rounded operation:
//     b_k = c_k * prod binom (as propensity());  g = exp(lambda_k * t);  a = b_k * g;
//     x = (lambda_k * r) / a;  dt_k = log1p(x) / lambda_k;
//     e = expm1(lambda_k * d) / lambda_k;  T_k = T_k + a * e.
int nrrta_run_rate_exp(const Net &net, const int64_t *x0, const double *lambda, const Start *start,
                       uint64_t seed, uint64_t traj, uint64_t max_firings, double t_end,
                       int64_t *x_out, double *t_out, uint64_t *firings_out, int32_t *stop_out,
                       uint64_t *fire_count_out, double *T_out, double *P_out,
                       int32_t *trace_mu, double *trace_t, uint64_t trace_cap) {
  const int32_t M = net.M, N = net.N;
  const double INF = std::numeric_limits<double>::infinity();
  const int64_t xmax = count_bound(net);
  for (int64_t e = 0; e < net.react_ptr[M]; ++e)
    if (net.react_sigma[e] < 1 || net.react_sigma[e] > 3) return ERR_BAD;
  for (int32_t k = 0; k < M; ++k) if (!std::isfinite(lambda[k])) return ERR_BAD;
  std::vector<int64_t> X(x0, x0 + N);
  for (int32_t j = 0; j < N; ++j) if (X[j] < 0 || X[j] > xmax) return ERR_BAD;
  std::vector<double> T(M, 0.0), P(M), a(M), dt(M);
  std::vector<uint32_t> n(M, 0u);
  for (int32_t k = 0; k < M; ++k) P[k] = exp_draw(seed, traj, (uint32_t)k, 0u);
  double t = 0.0;
  if (start) {
    t = start->t;
    if (start->T) for (int32_t k = 0; k < M; ++k) T[k] = start->T[k];
    if (start->P) for (int32_t k = 0; k < M; ++k) P[k] = start->P[k];
    if (start->n) for (int32_t k = 0; k < M; ++k) n[k] = (uint32_t)start->n[k];
  }
  uint64_t fired = 0;
  int32_t stop = 0;
  int rc = OK;
  // T_k += int_t^{t+d} a_k(s) ds for every k, a[] = propensities at the start t of the interval
  auto advance = [&](double d) {
    for (int32_t k = 0; k < M; ++k) {
      double e = d;
      if (lambda[k] != 0.0) { const double ld = lambda[k] * d; e = std::expm1(ld) / lambda[k]; }
      const double inc = a[k] * e;
      T[k] = T[k] + inc;
    }
  };
  for (;;) {
    // step 1: instantaneous propensities a_k(t) = c_k h_k exp(lambda_k t)
    for (int32_t k = 0; k < M; ++k) {
      a[k] = propensity(net, X.data(), k);
      if (lambda[k] != 0.0) { const double lt = lambda[k] * t; a[k] = a[k] * std::exp(lt); }
    }
    // step 2: each channel's own solution of Eq.28
    for (int32_t k = 0; k < M; ++k) {
      if (a[k] > 0.0) {
        double r = P[k] - T[k];
        if (r < 0.0) r = 0.0;
        if (lambda[k] != 0.0) {
          const double lr = lambda[k] * r;
          const double x = lr / a[k];
          dt[k] = (x > -1.0) ? std::log1p(x) / lambda[k] : INF;
        } else {
          dt[k] = r / a[k];
        }
      } else {
        dt[k] = INF;
      }
    }
    int32_t mu = 0;
    double delta = dt[0];
    for (int32_t k = 1; k < M; ++k)
      if (dt[k] < delta) { delta = dt[k]; mu = k; }
    if (delta == INF) { stop = STOP_ABSORBED; break; }
    if (t_end < INF && t + delta > t_end) {
      advance(t_end - t);
      t = t_end;
      stop = STOP_T_END;
      break;
    }
    advance(delta);
    t = t + delta;
    rc = apply_firing(net, X.data(), mu, xmax);
    n[mu] += 1u;
    P[mu] = P[mu] + exp_draw(seed, traj, (uint32_t)mu, n[mu]);
    if (fired < trace_cap) {
      if (trace_mu) trace_mu[fired] = mu;
      if (trace_t) trace_t[fired] = t;
    }
    fired += 1;
    if (rc != OK) break;
    if (max_firings != 0 && fired == max_firings) { stop = STOP_MAX_FIRINGS; break; }
  }
  if (x_out) for (int32_t j = 0; j < N; ++j) x_out[j] = X[j];
  if (t_out) *t_out = t;
  if (firings_out) *firings_out = fired;
  if (stop_out) *stop_out = stop;
  if (fire_count_out) for (int32_t k = 0; k < M; ++k) fire_count_out[k] = n[k];
  if (T_out) for (int32_t k = 0; k < M; ++k) T_out[k] = T[k];
  if (P_out) for (int32_t k = 0; k < M; ++k) P_out[k] = P[k];
  return rc;
}

}  // namespace

extern "C" {

void oracle_philox4x32_10(const uint32_t *ctr, const uint32_t *key, uint32_t *out) {
  philox4x32_10(ctr, key, out);
}

double oracle_exp_draw(uint64_t seed, uint64_t traj, uint32_t k, uint32_t n) {
  return exp_draw(seed, traj, k, n);
}

int64_t oracle_binom(int64_t x, int32_t sigma) { return binom(x, sigma); }

void oracle_propensities(int32_t N, int32_t M, const int64_t *react_ptr,
                         const int32_t *react_species, const int32_t *react_sigma,
                         const double *rate, const int64_t *X, double *a_out) {
  Net net{N, M, react_ptr, react_species, react_sigma, nullptr, nullptr, nullptr, rate};
  for (int32_t k = 0; k < M; ++k) a_out[k] = propensity(net, X, k);
}

int oracle_run(int32_t N, int32_t M, const int64_t *react_ptr, const int32_t *react_species,
               const int32_t *react_sigma, const int64_t *stoich_ptr,
               const int32_t *stoich_species, const int32_t *stoich_v, const double *rate,
               const int64_t *x0, uint64_t seed, uint64_t traj, uint64_t max_firings,
               double t_end, int64_t *x_out, double *t_out, uint64_t *firings_out,
               int32_t *stop_out, uint64_t *fire_count_out, double *T_out, double *P_out,
               int32_t *trace_mu, double *trace_t, uint64_t trace_cap) {
  Net net{N, M, react_ptr, react_species, react_sigma, stoich_ptr, stoich_species, stoich_v, rate};
  return nrrta_run(net, x0, nullptr, seed, traj, max_firings, t_end, x_out, t_out, firings_out,
                   stop_out, fire_count_out, T_out, P_out, trace_mu, trace_t, trace_cap);
}

// Resume from a checkpoint (t0, T0, P0, n0 = fire counts so far; each array may be NULL = fresh).
// residual != 0: the residual (Table 3) form, P0 = the residuals R_k, T0 unused, R returned in P_out.
int oracle_run_from(int32_t N, int32_t M, const int64_t *react_ptr, const int32_t *react_species,
                    const int32_t *react_sigma, const int64_t *stoich_ptr,
                    const int32_t *stoich_species, const int32_t *stoich_v, const double *rate,
                    const int64_t *x0, double t0, const double *T0, const double *P0,
                    const uint64_t *n0, int32_t residual, uint64_t seed, uint64_t traj,
                    uint64_t max_firings, double t_end, int64_t *x_out, double *t_out,
                    uint64_t *firings_out, int32_t *stop_out, uint64_t *fire_count_out,
                    double *T_out, double *P_out, int32_t *trace_mu, double *trace_t,
                    uint64_t trace_cap) {
  Net net{N, M, react_ptr, react_species, react_sigma, stoich_ptr, stoich_species, stoich_v, rate};
  const Start st{t0, T0, P0, n0};
  if (residual)
    return nrrta_run_residual(net, x0, &st, seed, traj, max_firings, t_end, x_out, t_out,
                              firings_out, stop_out, fire_count_out, P_out, trace_mu, trace_t,
                              trace_cap);
  return nrrta_run(net, x0, &st, seed, traj, max_firings, t_end, x_out, t_out, firings_out,
                   stop_out, fire_count_out, T_out, P_out, trace_mu, trace_t, trace_cap);
}

int oracle_run_sched(int32_t N, int32_t M, const int64_t *react_ptr, const int32_t *react_species,
                     const int32_t *react_sigma, const int64_t *stoich_ptr,
                     const int32_t *stoich_species, const int32_t *stoich_v, const double *rate,
                     const int64_t *x0, uint64_t seed, uint64_t traj, uint64_t max_firings,
                     double t_end, int32_t n_break, const double *t_break, const double *factor,
                     const uint8_t *mask, int64_t *x_out, double *t_out, uint64_t *firings_out,
                     int32_t *stop_out, uint64_t *fire_count_out, double *T_out, double *P_out,
                     int32_t *trace_mu, double *trace_t, uint64_t trace_cap) {
  Net net{N, M, react_ptr, react_species, react_sigma, stoich_ptr, stoich_species, stoich_v, rate};
  return nrrta_run_sched(net, x0, seed, traj, max_firings, t_end, n_break, t_break, factor, mask,
                         x_out, t_out, firings_out, stop_out, fire_count_out, T_out, P_out,
                         trace_mu, trace_t, trace_cap);
}

int oracle_run_rate_exp(int32_t N, int32_t M, const int64_t *react_ptr, const int32_t *react_species,
                        const int32_t *react_sigma, const int64_t *stoich_ptr,
                        const int32_t *stoich_species, const int32_t *stoich_v, const double *rate,
                        const int64_t *x0, const double *lambda, uint64_t seed, uint64_t traj,
                        uint64_t max_firings, double t_end, int64_t *x_out, double *t_out,
                        uint64_t *firings_out, int32_t *stop_out, uint64_t *fire_count_out,
                        double *T_out, double *P_out, int32_t *trace_mu, double *trace_t,
                        uint64_t trace_cap) {
  Net net{N, M, react_ptr, react_species, react_sigma, stoich_ptr, stoich_species, stoich_v, rate};
  return nrrta_run_rate_exp(net, x0, lambda, nullptr, seed, traj, max_firings, t_end, x_out, t_out,
                            firings_out, stop_out, fire_count_out, T_out, P_out, trace_mu, trace_t,
                            trace_cap);
}

int oracle_run_residual(int32_t N, int32_t M, const int64_t *react_ptr, const int32_t *react_species,
                        const int32_t *react_sigma, const int64_t *stoich_ptr,
                        const int32_t *stoich_species, const int32_t *stoich_v, const double *rate,
                        const int64_t *x0, uint64_t seed, uint64_t traj, uint64_t max_firings,
                        double t_end, int64_t *x_out, double *t_out, uint64_t *firings_out,
                        int32_t *stop_out, uint64_t *fire_count_out, double *R_out,
                        int32_t *trace_mu, double *trace_t, uint64_t trace_cap) {
  Net net{N, M, react_ptr, react_species, react_sigma, stoich_ptr, stoich_species, stoich_v, rate};
  return nrrta_run_residual(net, x0, nullptr, seed, traj, max_firings, t_end, x_out, t_out, firings_out,
                            stop_out, fire_count_out, R_out, trace_mu, trace_t, trace_cap);
}

// Independent trajectories traj_first .. traj_first+n_traj-1, each by the single-threaded
// routine above; n_threads > 1 only runs several such instances side by side (one per host
// core) for the timed CPU baseline.  Returns the first non-zero per-trajectory code.
int oracle_ensemble(int32_t N, int32_t M, const int64_t *react_ptr, const int32_t *react_species,
                    const int32_t *react_sigma, const int64_t *stoich_ptr,
                    const int32_t *stoich_species, const int32_t *stoich_v, const double *rate,
                    const int64_t *x0, uint64_t seed, uint64_t traj_first, uint64_t n_traj,
                    uint64_t max_firings, double t_end, int64_t *x_out /*[n_traj*N]*/,
                    double *t_out, uint64_t *firings_out, int32_t *stop_out, int32_t n_threads) {
  Net net{N, M, react_ptr, react_species, react_sigma, stoich_ptr, stoich_species, stoich_v, rate};
  if (n_threads < 1) n_threads = 1;
  std::vector<int> codes(n_traj, 0);
  auto work = [&](uint64_t first, uint64_t step) {
    for (uint64_t i = first; i < n_traj; i += step)
      codes[i] = nrrta_run(net, x0, nullptr, seed, traj_first + i, max_firings, t_end,
                           x_out + (size_t)i * (size_t)N, t_out + i, firings_out + i,
                           stop_out + i, nullptr, nullptr, nullptr, nullptr, nullptr, 0);
  };
  if (n_threads == 1) {
    work(0, 1);
  } else {
    std::vector<std::thread> pool;
    for (int32_t w = 0; w < n_threads; ++w) pool.emplace_back(work, (uint64_t)w, (uint64_t)n_threads);
    for (auto &th : pool) th.join();
  }
  for (uint64_t i = 0; i < n_traj; ++i) if (codes[i] != 0) return codes[i];
  return 0;
}

}  // extern "C"
