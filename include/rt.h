/* rt.h -- C ABI of the B200-native random-time (NRRTA) stochastic simulation hot path.
 *
 * Method: Liu & Wang, "Parallel implementations of random time algorithm for chemical network
 * stochastic simulations", arXiv 2103.00405 (PAPER.md = the extracted text).  One firing is:
 *   a_k   = c_k * prod_j C(X_j, sigma_jk)                 Eq.1-2
 *   dt_k  = (P_k - T_k) / a_k   (+inf if a_k = 0)         Eq.24, a_k constant
 *   mu    = argmin_k dt_k, ties to the lowest k           Eq.25
 *   t    += dt_mu;  T_k += a_k * dt_mu for EVERY k        Eq.15
 *   X    += v_mu                                          Eq.5
 *   P_mu += -ln U, U from Philox4x32-10 keyed by          Eq.23,26
 *           (seed, trajectory, reaction, firing count)
 * Loop shape: Table 1 / Table 3; both a time and a step limit as in the
 * paper's model file.  All arithmetic is IEEE binary64, every operation
 * rounded to nearest separately (no fused multiply-add); DESIGN.md lists the readings taken
 * where the paper is silent or garbled.
 *
 * Conventions.  Every function returns an int: RT_OK (0) or a negative RT_ERR_* code; nothing
 * throws across the boundary.  Pointers are HOST pointers unless the name ends in _dev or the
 * parameter is documented as a device pointer.  The caller owns every array passed in and every
 * output buffer; the library copies what it needs during the call and keeps no caller pointer.
 * Results depend only on (network, x0, seed, trajectory, limits) -- not on the launch shape,
 * on how an ensemble is batched, nor on the propensity refresh mode.
 * A model is not thread-safe: calls on one rt_model must not overlap (different models may).
 * Device-pointer entry points do not validate device data: x0_dev must hold counts in
 * [0, bound] (see below), as the host entry points check for x0.
 */
#ifndef RT_B200_H_
#define RT_B200_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- status codes ------------------------------------------------------------------------ */
#define RT_OK                0
#define RT_ERR_NULL         -1   /* a required pointer is NULL                                   */
#define RT_ERR_BAD_NETWORK  -2   /* rt_network fails validation (see rt_validate_network)        */
#define RT_ERR_BAD_ARG      -3   /* x0 < 0 or above the count bound, t_end NaN or < 0, no limit  */
#define RT_ERR_UNSUPPORTED  -4   /* sigma > 3, or more than 2^32-1 CSR entries                   */
#define RT_ERR_OVERFLOW     -5   /* a species count left [0, bound] during a run                 */
#define RT_ERR_CUDA         -6   /* CUDA runtime error, no device, or an in-kernel barrier timeout */
#define RT_ERR_OOM          -7   /* host or device allocation failed                             */
#define RT_ERR_SCRATCH      -8   /* rt_run_dev_noalloc: rt_noalloc_prepare not called for this model, or
                                    the run needs more than RT_NOALLOC_SCRATCH_BYTES of scratch       */

/* ---- why a trajectory stopped (not errors) ------------------------------------------------- */
#define RT_STOP_T_END        1   /* next firing would pass t_end: t = t_end, nothing fired        */
#define RT_STOP_MAX_FIRINGS  2   /* max_firings reactions fired                                  */
#define RT_STOP_ABSORBED     3   /* every propensity is 0; t stays at the last firing             */

typedef struct rt_model rt_model;   /* opaque; owns the device copy of the network and all state */

/* Reaction network in CSR form (N >= 1 species, M >= 1 reactions, reactant
 * coefficients sigma_jk, net change v_k; sparse matrices).  Row k of the react_*
 * arrays lists the reactant species of reaction k with sigma_jk >= 1; row k of the stoich_*
 * arrays lists the species whose count changes when k fires, with v_jk != 0.  A species may
 * appear at most once per row, and v_jk >= -sigma_jk' must hold (a reaction cannot remove more
 * than it requires, so counts stay >= 0).  rate[k] = c_k, finite and >= 0. */
typedef struct {
  int32_t n_species;               /* N >= 1 */
  int32_t n_reactions;             /* M >= 1 */
  const int64_t *react_ptr;        /* [M+1], react_ptr[0] = 0, non-decreasing                    */
  const int32_t *react_species;    /* [react_ptr[M]] species index in [0, N)                     */
  const int32_t *react_sigma;      /* [react_ptr[M]] 1 <= sigma <= 3                             */
  const int64_t *stoich_ptr;       /* [M+1]                                                      */
  const int32_t *stoich_species;   /* [stoich_ptr[M]]                                            */
  const int32_t *stoich_v;         /* [stoich_ptr[M]] v != 0                                     */
  const double  *rate;             /* [M]                                                        */
} rt_network;

/* Per-trajectory outcome.  24 bytes, no padding surprises: (f64, u64, i32, i32). */
typedef struct {
  double   t;         /* simulated time reached                                                   */
  uint64_t firings;   /* reactions fired                                                          */
  int32_t  stop;      /* RT_STOP_*                                                                */
  int32_t  status;    /* RT_OK or RT_ERR_OVERFLOW for this trajectory                             */
} rt_result;

/* Count bound: species counts must stay in [0, 2^31-1] when every sigma <= 2 and in
 * [0, 2^21-1] when some sigma = 3, so that C(X, sigma) is exact in int64 (G2). */

/* Host-only check of a network (no GPU needed).  RT_OK, RT_ERR_NULL, RT_ERR_BAD_NETWORK
 * (N < 1, M < 1, ptr not starting at 0 / decreasing, species out of range, sigma < 1, v = 0,
 * a species twice in one row, v_jk < -sigma_jk, rate negative / NaN / inf) or RT_ERR_UNSUPPORTED. */
int rt_validate_network(const rt_network *net);

/* Validate, build the species->reactions dependency lists (Gibson & Bruck's dependency graph,
 * PAPER.md:191, stored two-hop: stoich row of mu -> species -> reactions reading that species)
 * and deep-copy everything to `device`.  *out receives the model. */
int rt_create(const rt_network *net, int device, rt_model **out);

/* One trajectory (Table 3 loop).  Runs until max_firings reactions have fired
 * (0 = no firing limit), until the next firing would pass t_end (+inf = no time limit; at least
 * one limit is required), or until absorbed.
 *   x0 [N] initial counts; x_out [N] final counts (may alias nothing; may be NULL).
 *   res: outcome (required).
 *   fire_count_out [M] firings per reaction R_k (Eq.5), T_out/P_out [M] final internal times and
 *   next internal firing times -- each may be NULL.
 *   trace_mu/trace_t [trace_cap]: the fired reaction and the time of each of the first trace_cap
 *   firings (either may be NULL; trace_cap may be 0).
 * Returns RT_ERR_OVERFLOW (also in res->status) if a firing would take a count out of the bound
 * (or after 2^33-2 firings of one trajectory): that firing is counted in res->firings and in the
 * trace, its internal-time increment and redraw are applied, its change of X is not. */
int rt_run(rt_model *m, const int64_t *x0, uint64_t seed, uint64_t trajectory,
           uint64_t max_firings, double t_end,
           int64_t *x_out, rt_result *res,
           uint64_t *fire_count_out, double *T_out, double *P_out,
           int32_t *trace_mu, double *trace_t, uint64_t trace_cap);

/* Checkpoint / resume: continue a trajectory from the state an earlier rt_run (or rt_run_resume)
 * returned -- x0 = its x_out, t0 = its res->t, T0 / P0 / fire_count0 [M] = its T_out / P_out /
 * fire_count_out (all three required; in the residual formulation T0 = -R_k and P0 = 0, exactly as
 * T_out / P_out deliver them).  Nothing is drawn at the start: the internal clocks T_k (Eq.15,
 * PAPER.md:106) and the next internal firing times P_k (Eq.26) ARE the state of
 * the random time-change representation, and later draws are keyed by (seed, trajectory, k,
 * fire count), so rt_run to n1 firings followed by rt_run_resume for n2 - n1 more gives, bit for
 * bit, what rt_run to n2 firings gives.  max_firings, the trace and res->firings count the
 * firings of THIS call; res->t continues from t0; t_end is absolute.
 * Errors as rt_run, plus RT_ERR_NULL (a state array missing), RT_ERR_BAD_ARG (t0 NaN, negative
 * or beyond t_end; NaN in T0 / P0; a fire count >= 2^32) and RT_ERR_UNSUPPORTED (a rate schedule
 * is set: whether a breakpoint at exactly t0 has acted is not part of the state).
 * With "ensemble_path" = 1 a network small enough for it runs on the one-thread-per-trajectory
 * kernel (no trace: RT_ERR_UNSUPPORTED if one is requested). */
int rt_run_resume(rt_model *m, const int64_t *x0, double t0, const double *T0, const double *P0,
                  const uint64_t *fire_count0, uint64_t seed, uint64_t trajectory,
                  uint64_t max_firings, double t_end,
                  int64_t *x_out, rt_result *res,
                  uint64_t *fire_count_out, double *T_out, double *P_out,
                  int32_t *trace_mu, double *trace_t, uint64_t trace_cap);

/* Same trajectory, with x0 / x_out / trace_* DEVICE pointers on m's device and the work
 * enqueued on `stream` (a cudaStream_t, e.g. torch.cuda.current_stream().cuda_stream; NULL = the
 * default stream).  res_dev: device pointer to one rt_result.  The call does not synchronise;
 * device-side failures (overflow, barrier timeout) are reported in res_dev->status and by the
 * next rt_sync.  x_out_dev, trace_*_dev may be NULL. */
int rt_run_dev(rt_model *m, const int64_t *x0_dev, uint64_t seed, uint64_t trajectory,
               uint64_t max_firings, double t_end,
               int64_t *x_out_dev, rt_result *res_dev,
               int32_t *trace_mu_dev, double *trace_t_dev, uint64_t trace_cap, void *stream);

/* ---- no-allocation entry point --------------------------------------------------------------
 * For callers that may not call cudaMalloc (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it).  rt_run_dev keeps the per-trajectory scratch of the bundle kernels
 * (Eq.15/24/26 state T, P, a [M], firing counts n [M], the versioned count words X [N] and the
 * argmin exchange slots of PAPER.md:195-199, :211) in buffers it allocates on first use.
 * rt_run_dev_noalloc is the same launch with that scratch in ONE file-scope array in device memory,
 *   static __device__ __align__(256) unsigned char [RT_NOALLOC_SCRATCH_BYTES]   (4 MiB),
 * which every GPU that loads the library holds until the process exits.  It calls no cudaMalloc,
 * cudaFree or allocating library routine: it enqueues one memset of the exchange slots (they must
 * start at zero; T, P, a, n, X are initialised by the kernel from x0_dev and the Philox stream) and
 * one kernel on `stream`.  Need in bytes, each part rounded up to 256: 3*8*M_pad + 4*M_pad + 8*G*N +
 * 2048*S (M_pad = M rounded up to even; S = CTAs of the bundle, <= 160, two rounds of 1 KiB
 * exchange slots each; G = "x_replicas"), i.e. networks up to about M = 1.3e5: config 3 fits,
 * config 4 does not.
 * THE ARRAY IS SHARED: by every model on the device, every stream and every call.  It keeps the
 * last call's contents, and two calls that overlap on the GPU (different streams, or the same
 * model's rt_run_dev_noalloc twice without stream order) race on it: keep them in stream order.
 *
 * rt_noalloc_prepare: set-up, once per model after its options are set (it MAY allocate: the first
 * call per device loads the kernels and takes the array's device address with
 * cudaGetSymbolAddress).  *need_bytes (may be NULL) receives the scratch the current options need.
 * Returns RT_ERR_SCRATCH if that exceeds RT_NOALLOC_SCRATCH_BYTES, RT_ERR_CUDA on a runtime error.
 *
 * rt_run_dev_noalloc: arguments, results and error reporting exactly as rt_run_dev (bit-identical
 * outputs).  RT_ERR_SCRATCH if the model was not prepared or the launch shape the current options
 * give needs more than RT_NOALLOC_SCRATCH_BYTES; nothing is enqueued then.  State streamed from
 * global memory ("state_mode" = 1) runs without the persisting-L2 window of "l2_persist". */
#define RT_NOALLOC_SCRATCH_BYTES (4u << 20)
int rt_noalloc_prepare(rt_model *m, uint64_t *need_bytes);
int rt_run_dev_noalloc(rt_model *m, const int64_t *x0_dev, uint64_t seed, uint64_t trajectory,
                       uint64_t max_firings, double t_end,
                       int64_t *x_out_dev, rt_result *res_dev,
                       int32_t *trace_mu_dev, double *trace_t_dev, uint64_t trace_cap, void *stream);

/* n_traj independent trajectories traj_first .. traj_first+n_traj-1 from the same x0 (the
 * paper's "bundles").  Row i of the outputs is exactly what
 * rt_run(trajectory = traj_first + i) returns.  x_out [n_traj*N] row-major (may be NULL),
 * res [n_traj].  Returns the first non-OK per-trajectory status, if any. */
int rt_ensemble(rt_model *m, const int64_t *x0, uint64_t seed, uint64_t traj_first,
                uint64_t n_traj, uint64_t max_firings, double t_end,
                int64_t *x_out, rt_result *res);

/* Device-pointer flavour of rt_ensemble (x0_dev [N], x_out_dev [n_traj*N] or NULL,
 * res_dev [n_traj]), enqueued on `stream`, no synchronisation. */
int rt_ensemble_dev(rt_model *m, const int64_t *x0_dev, uint64_t seed, uint64_t traj_first,
                    uint64_t n_traj, uint64_t max_firings, double t_end,
                    int64_t *x_out_dev, rt_result *res_dev, void *stream);

/* Wait for everything enqueued on `stream` by this model; returns RT_ERR_CUDA if a kernel
 * reported a barrier timeout or the runtime reported an error. */
int rt_sync(rt_model *m, void *stream);

/* Time-dependent rates (section 6, Eq.28, :224-231: channel k fires when
 * h_k * int_t^{t+dt_k} c_k(s) ds = P_k - T_k, "calculated analytically for well behaved
 * time-dependent reaction rates").  The family implemented is piecewise-constant modulation:
 *   c_k(s) = c_k * factor[i]  for s in [t_break[i], t_break[i+1])   (factor 1 before t_break[0])
 * for the reactions with mask[k] != 0 (mask == NULL: all reactions); the effective rate is the
 * one rounded product c_k * factor[i].  A step that would cross a breakpoint is cut there
 * (T_k += a_k * (b - t) for every k, t = b, nothing fires) and the rates switch.
 *   t_break [n_break] strictly increasing, finite, >= 0;  factor [n_break] finite, >= 0;
 *   mask [M] or NULL.  n_break = 0 removes the schedule.  The arrays are copied.
 * A factor-0 schedule from t_break[0] = 0 on a mask gives the boundary conditions of the note
 * under PAPER.md Table 2 (:260): the masked channels are forbidden and their internal time is
 * frozen.
 * Applies to rt_run / rt_ensemble (and their _dev forms) through the bundle kernel; not
 * combinable with "refresh_mode" = 1 or "formulation" = 1 (RT_ERR_UNSUPPORTED at run time).
 * Returns RT_ERR_BAD_ARG for an invalid schedule. */
int rt_set_rate_schedule(rt_model *m, int32_t n_break, const double *t_break, const double *factor,
                         const uint8_t *mask);

/* Smoothly time-dependent rates (section 6, Eq.28, :224-231, the case the paper means by
 * "the integral can be calculated analytically for well behaved time-dependent reaction rates"):
 *   c_k(s) = c_k * exp(lambda[k] * s),   lambda [M] finite (decay < 0, growth > 0, 0 = constant).
 * Every channel solves its own equation of Eq.28 in closed form each firing: with a_k(t) =
 * c_k h_k exp(lambda_k t) the propensity now,
 *   dt_k = log1p(lambda_k (P_k - T_k) / a_k(t)) / lambda_k     (+inf if the argument is <= -1),
 *   T_k += a_k(t) * expm1(lambda_k dt_min) / lambda_k           for every k,
 * and lambda_k = 0 takes the constant-rate formulas, so an all-zero lambda is the default path.
 * exp / log1p / expm1 are the CUDA math library's (<= 2 ulp), so sample paths agree with a host
 * implementation in the fired sequence and to ~1e-12 in the times, not to the last bit.
 * lambda == NULL removes it; the array is copied.  Applies to rt_run / rt_run_resume /
 * rt_ensemble (bundle kernel); not combinable with a rate schedule, "refresh_mode" = 1 or
 * "formulation" = 1 (RT_ERR_UNSUPPORTED at run time).  RT_ERR_BAD_ARG for a non-finite lambda. */
int rt_set_rate_exponent(rt_model *m, const double *lambda);

/* Tuning / debug knobs (all optional; results never depend on them, except "formulation").
 *   "refresh_mode"   0 = dependency-graph refresh of a_k (default), 1 = recompute every a_k
 *                    each firing (the paper's own GPU scheme)
 *   "bundle_ctas"    CTAs cooperating on one trajectory; 0 = choose automatically
 *   "ensemble_path"  0 = automatic, 1 = force one-thread-per-trajectory kernel (RT_ERR_BAD_ARG at
 *                    run time if the network is too large for it, RT_ERR_UNSUPPORTED together with
 *                    a rate schedule or "formulation" = 1, which that kernel does not implement),
 *                    2 = force the bundle (CTA-group-per-trajectory) kernel
 *   "state_mode"     0 = keep (T,P,a) in shared memory when a CTA's share fits (default),
 *                    1 = always stream it from global memory (the regime of M > ~1.3e6)
 *   "prefetch"       bit 0: L2 prefetch of the candidate's walk data, bit 1: speculative redraw,
 *                    bit 2: pre-walk of the exchange's runner-up (default 7 = all)
 *   "formulation"    0 = (T_k, P_k) internal-time form (default; the form every parity claim is
 *                    made for), 1 = residual form of PAPER.md Table 3 (R_k = P_k - T_k kept in one
 *                    array: T_out then holds -R_k and P_out zeros).  Same process, different
 *                    rounding: its sample paths match oracle_run_residual, not oracle_run.
 *   "x_replicas"     copies of X per trajectory the CTAs spread their updates over (default 1)
 *   "tiny_kernel"    one-thread-per-trajectory path: 1 = networks of at most 4 reactions (<= 2 reactants
 *                    each) over at most 4 species use the register-resident kernel (default),
 *                    0 = always the general shared-memory kernel.  Same results either way.
 *   "l2_persist"     state streamed from global memory only: 1 = keep T (read and written every
 *                    firing) as persisting lines in L2 through an access-policy window on the launch
 *                    (default; the first such launch raises the device's persisting-L2 limit to its
 *                    maximum), 0 = plain streaming, 2 = keep a instead (for comparison)
 *   "pipeline"       1 = candidate-first kernel (rt_fast.cuh) wherever it applies: state in shared
 *                    memory, "refresh_mode" 0, constant rates, one copy of X (default);
 *                    0 = always the plain bundle kernel (rt_bundle.cuh).  Same results either way.
 *   "exchange"       0 = a bundle of 2..16 CTAs with on-chip state runs as ONE thread-block cluster
 *                    and reduces its per-firing argmin through distributed shared memory (default),
 *                    1 = always exchange through slots in global memory (L2)
 * Returns RT_ERR_BAD_ARG for an unknown name or value. */
int rt_set_option(rt_model *m, const char *name, int64_t value);

/* Introspection for tests and bench.py:
 *   "kernel_launches"  kernels launched by this model so far
 *   "bundle_ctas", "bundles", "block_threads"  shape of the last bundle launch
 *   "ensemble_path"    path taken by the last rt_ensemble call (1 or 2)
 *   "state_in_smem"    1 if the last bundle launch kept (T,P,a) in shared memory
 *   "cluster_exchange" 1 if the last bundle launch ran each bundle as a thread-block cluster
 *   "pipeline"         1 if the last bundle launch used the candidate-first kernel
 *   "tiny_kernel"      1 if the last one-thread-per-trajectory launch used the register-resident kernel
 *   "l2_persist"       the "l2_persist" option in effect (0 if the device has no persisting L2)
 *   "num_sms", "dep_entries", "max_sigma", "hub_species"
 * Unknown name: returns RT_ERR_BAD_ARG and leaves *value alone. */
int rt_get_info(const rt_model *m, const char *name, int64_t *value);

void rt_destroy(rt_model *m);            /* rt_destroy(NULL) is a no-op */

const char *rt_strerror(int code);       /* static string, never NULL */

#ifdef __cplusplus
}
#endif
#endif /* RT_B200_H_ */
