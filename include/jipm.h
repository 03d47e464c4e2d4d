/* jipm.h -- C ABI of the B200-native batched interior-point NLP solver.
 *
 * What it computes: the interior-point iteration of arxiv 2606.26341 section IV applied to a
 * batch of independent parametric NLPs
 *        min f(x,theta)  s.t.  c(x,theta) = 0,  x_L < x < x_U          (eqs 1a-1c)
 * that share f, c and the bounds and differ only in theta and the initial guess (eq 2).
 * General inequalities enter through slack variables.  Each problem runs the barrier
 * iteration (eqs 3-7) with the fallbacks of Table I that this
 * build covers (rows 1-6 and the monotone schedule of row 7: backtracking, second-order correction, watchdog,
 * tiny-step rule, soft and hard feasibility restoration; plus the inertia correction of PAPER.md:114) and a
 * problem slot is refilled from the queue as soon as its problem ends (iteration-level batching,
 * PAPER.md:162-168).
 *
 * Decision vector ("stage order", n entries) and equality vector (m entries) of every family:
 *        x = [ x_0 | u_0 x_1 s_1 | u_1 x_2 s_2 | ... | u_{N-1} x_N s_N ]
 *        c = [ x_0 - xhat0 | dyn_1 g_1 | ... | dyn_N g_N ],  dyn_k = x_k - F(x_{k-1},u_{k-1}),  g_k = h(x_k) - s_k
 * n = (N+1) nx + N nu + N ng,  m = (N+1) nx + N ng;  slacks s >= 0 carry the inequalities h(x_k) >= 0.
 *
 * Conventions: every pointer argument says HOST or DEVICE.  The caller owns all buffers; the library keeps
 * no caller pointer after a call returns.  All work is enqueued on the stream given at create time and
 * jipm_solve_batch returns after that work has completed.  Return value = call-level error code (0 = ok);
 * per-problem outcomes are only in status_out.  There is no CPU fallback: without a CUDA device every
 * compute entry returns JIPM_ERR_CUDA.
 */
#ifndef JIPM_H
#define JIPM_H
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct jipm_solver jipm_solver; /* opaque, owned by the library */

enum { JIPM_OK = 0, JIPM_ERR_ARG = 1, JIPM_ERR_DIM = 2, JIPM_ERR_BOUNDS = 3, JIPM_ERR_CUDA = 4, JIPM_ERR_NOMEM = 5 };
enum { JIPM_FAM_POINTMASS2D = 0, JIPM_FAM_QUAD_TRACK = 1, JIPM_FAM_MULTIQUAD = 2, JIPM_FAM_QUAD_CLUTTER = 3,
       JIPM_FAM_QUAT_NAV = 4 /* the paper's own vehicle: 13-state quaternion quadrotor, rotor speeds */ };
enum { JIPM_ST_NOT_RUN = -1, JIPM_ST_SOLVED = 0, JIPM_ST_MAXITER = 1, JIPM_ST_LOCALLY_INFEASIBLE = 2,
       JIPM_ST_RESTORATION_FAILED = 3, JIPM_ST_RESTO_AT_FEASIBLE_POINT = 4, JIPM_ST_NONFINITE = 5,
       JIPM_ST_TINY_STEP = 6 /* search direction too small to make progress at the smallest mu (Table I row 4) */,
       JIPM_ST_ACCEPTABLE = 7 /* acceptable-level termination (reading AT, off by default): NOT counted as converged */ };

/* Problem family dimensions (BASELINE.json configs). */
typedef struct {
    int32_t horizon_N;   /* control intervals; N+1 state knots */
    int32_t n_agents;    /* 1 except JIPM_FAM_MULTIQUAD */
    int32_t n_obstacles; /* obstacles per knot, 0..254 (ignored by JIPM_FAM_MULTIQUAD: pair constraints) */
    double dt;
} jipm_family_dims;

/* Algorithmic constants.  The paper gives none (it defers to its ref. [7]); the
 * defaults are the readings listed in DESIGN.md "Readings". */
typedef struct {
    double tol, mu_init, kappa_eps, kappa_mu, theta_mu, tau_min, s_max, kappa_sigma;
    double kappa_1, kappa_2, bound_relax_factor, bound_mult_init, lam_init_max, kappa_d;
    double gamma_theta, gamma_phi, eta_phi, delta, s_theta, s_phi, gamma_alpha;
    double theta_max_fact, theta_min_fact, alpha_red, kappa_soc;
    double delta_w_min, delta_w_0, delta_w_max, kappa_w_minus, kappa_w_plus, kappa_w_plus_first;
    double delta_c_bar, kappa_c, residual_ratio_max, rho_resto, kappa_resto, z_reset_threshold;
    /* refinement failure ("pretend singular", reading S-7) and Table I rows 3-5 */
    double residual_ratio_singular, residual_improvement_factor;
    double tiny_step_tol, tiny_step_y_tol, tiny_step_cviol, soft_resto_factor;
    /* adaptive barrier parameter with the switch to the monotone schedule (Table I row 7) */
    double adaptive_red_fact, adaptive_monotone_init, adaptive_sigma_max, adaptive_mu_max_fact;
    /* acceptable-level termination (NEXT-4; an IPOPT feature the paper does not describe: DESIGN.md reading AT) */
    double acceptable_tol, acceptable_dual_inf_tol, acceptable_constr_viol_tol, acceptable_compl_inf_tol;
    int32_t max_iter, max_backtrack, max_soc, refine_min, refine_max, max_mu_updates;
    int32_t init_slacks, enable_restoration;
    int32_t watchdog_trigger, watchdog_trial_max, max_soft_resto_iters;
    int32_t polish_max; /* extra refinement steps (<= this many) taken after the stop rule is met while the residual ratio
                           is above 1e-15 and still shrinking: accuracy of the step only, no decision depends on it */
    int32_t mu_strategy;        /* 0 monotone schedule (default, IPOPT's), 1 adaptive (Mehrotra probing) with the switch */
    int32_t adaptive_red_iters; /* KKT errors remembered by the progress test of the adaptive mode */
    int32_t acceptable_iter;    /* stop after this many consecutive acceptable regular iterations; 0 = off (default) */
} jipm_options;

/* Fill *o with the defaults.  o: HOST.  Returns JIPM_ERR_ARG if o is NULL. */
int jipm_default_options(jipm_options* o);

/* Internal sizes (slacks included) of a family.  n, m, n_theta: HOST out.  JIPM_ERR_DIM on a bad family/dims. */
int jipm_family_sizes(int family, const jipm_family_dims* d, int64_t* n, int64_t* m, int64_t* n_theta);

/* Create a solver for one family.
 *   n, m            must equal jipm_family_sizes (else JIPM_ERR_DIM)
 *   x_L, x_U        HOST [n], +-INFINITY = no bound, shared by all problems; x_L >= x_U on a
 *                   component -> JIPM_ERR_BOUNDS (PAPER.md:63 needs a strict interior).  Copied.
 *   opts            HOST or NULL (defaults).  Copied.
 *   resident_slots  R = problem slots in flight (one CTA per slot); 0 -> library picks (fills the GPU).
 *   cuda_stream     cudaStream_t (e.g. torch.cuda.current_stream().cuda_stream); NULL = default stream.
 * The solver belongs to the CUDA device that is current at this call; later calls switch to it for their duration.
 * Calls on solvers of the same family are serialised inside the library (launch arguments live in one
 * __constant__ block per family instantiation); calls on different families may run concurrently. */
int jipm_create(jipm_solver** out, int family, const jipm_family_dims* d, int64_t n, int64_t m,
                const double* x_L, const double* x_U, const jipm_options* opts, int64_t resident_slots,
                void* cuda_stream);

/* Solve P problems.  Outputs are indexed by problem id (row of the inputs), never by slot;
 * the result of a row does not depend on P, R or row order.
 *   x0       DEVICE [P x n]  initial guess (slack entries are overwritten when opts.init_slacks)
 *   params   DEVICE [P x n_theta]
 *   x_out    DEVICE [P x n];  lam_out DEVICE [P x m] (y_c, sign of eq 4)
 *   zL_out, zU_out  DEVICE [P x n] (0 where no bound) or NULL
 *   status_out, iters_out  DEVICE [P] int32 */
int jipm_solve_batch(jipm_solver* s, int64_t P, const double* x0, const double* params, double* x_out,
                     double* lam_out, double* zL_out, double* zU_out, int32_t* status_out, int32_t* iters_out);

/* Same call with HOST buffers: copies in, solves, copies out (all on the solver's stream).  The device staging
 * buffer is owned by the solver and only grows (no allocation on repeated calls of the same size). */
int jipm_solve_batch_host(jipm_solver* s, int64_t P, const double* x0, const double* params, double* x_out,
                          double* lam_out, double* zL_out, double* zU_out, int32_t* status_out,
                          int32_t* iters_out);

/* Free everything.  NULL is a no-op. */
int jipm_destroy(jipm_solver* s);

/* The same solve (the iteration of PAPER.md:77-150) for callers that must not allocate: no
 * cudaMalloc, cudaFree or allocating library routine is called, no solver object exists.  All device memory the
 * solve needs beyond the caller's buffers -- relaxed bounds, the per-SM slot workspaces of the kernel, queue counter,
 * statistics -- lives in one static device array of JIPM_STATIC_SCRATCH_BYTES that every GPU which loads the library
 * holds until the process exits.
 *   family, d, n, m, x_L, x_U (HOST [n]), opts (HOST or NULL), cuda_stream: as in jipm_create; the library picks R.
 *   P, x0, params, x_out, lam_out, zL_out, zU_out, status_out, iters_out (all DEVICE): as in jipm_solve_batch.
 * Results are bit-identical to jipm_create + jipm_solve_batch with the same arguments.  Returns after the work has
 * completed.  A family whose workspaces do not fit the array (n > 8192, or more than JIPM_STATIC_SCRATCH_BYTES of
 * scratch: C0 and C1 of BASELINE.json fit (C1: 45 MB); workload 5 (81 MB), C3 (198 MB) and C2 (504 MB) do not) -> JIPM_ERR_NOMEM with the sizes in
 * jipm_last_error; nothing is launched.
 * Every call on a device shares the one array, which keeps the previous call's contents (the call clears what must
 * start at zero): calls that overlap on the GPU -- other host threads are serialised by the library, other PROCESSES
 * have their own copy -- would race; no trace, statistics or debug entry applies to this call. */
#define JIPM_STATIC_SCRATCH_BYTES (64u << 20)
int jipm_solve_batch_static(int family, const jipm_family_dims* d, int64_t n, int64_t m, const double* x_L,
                            const double* x_U, const jipm_options* opts, void* cuda_stream, int64_t P,
                            const double* x0, const double* params, double* x_out, double* lam_out,
                            double* zL_out, double* zU_out, int32_t* status_out, int32_t* iters_out);

/* Last error text of the calling thread (static storage, never NULL). */
const char* jipm_last_error(void);

/* ---- statistics of the last jipm_solve_batch (HOST out) ------------------------------------------------
 * stats[0] total IPM iterations, [1] factorisations, [2] KKT solves, [3] derivative evaluations,
 * [4] f/c-only evaluations, [5] slots launched, [6] kernel launches, [7] restoration iterations,
 * [8..14] SM-clock cycles summed over slots spent in: derivative evaluation, factorisations, KKT solves,
 * residuals of (6), trial-point evaluations, whole iterations, Step I (clock64 of each slot's thread 0);
 * [16..20] the same for the factorisation sub-phases: T J, M assembly, control pivots, Phi + stores, D != 0 extras. */
int jipm_last_stats(jipm_solver* s, int64_t* stats, int64_t n_stats);

/* How the solver occupies its device: res[0] = SMs, res[1] = problem slots (CTAs) co-resident per SM for this family.
 * R = resident_slots CTAs are launched per solve, but only res[0] * res[1] run at once; the others start as earlier
 * ones end (they find the queue empty unless R is below that product).  res: HOST out [2]. */
int jipm_residency(jipm_solver* s, int64_t* res);

/* ---- debug / parity-test entries (load a state, step once, compare) ------------------
 * Decision trace: per problem, per iteration JIPM_TRACE_W doubles:
 *   [0] mode (0 regular, 1 restoration) [1] #factorisations [2] delta_w [3] delta_c [4] #refinements
 *   [5] kind (0 newton, 1 soc, 2 ls_fail->resto, 3 ic_fail->resto, 4 terminal) [6] #backtracks [7] #soc
 *   [8] alpha [9] alpha_z [10] f-type? [11] #mu updates [12] E0 at iteration start [13] mu used
 *   [14] theta_k [15] phi_k
 *   [16] watchdog (0 none, 1 started + step taken unconditionally, 2 step taken unconditionally, 3 succeeded,
 *        4 gave up: back at the entry iterate, backtracked from there)
 *   [17] soft restoration (0 none, 1 step accepted by the error reduction, 2 accepted by the original criterion)
 *   [18] tiny step taken? [19] #refinement failures treated as a singular matrix
 *   [20] barrier strategy of the iteration (0 monotone schedule, 1 adaptive rule, 2 monotone phase of the adaptive
 *        strategy) [21] switch taken (0 none, 1 adaptive -> monotone, 2 monotone -> adaptive)
 *   kind [5] also takes 5 = tiny step, 6 = soft restoration step. */
#define JIPM_TRACE_W 22
/* Enable tracing for the next solves: trace DEVICE [P x max_records x JIPM_TRACE_W] (or NULL to disable). */
int jipm_debug_set_trace(jipm_solver* s, double* trace, int64_t max_records);

/* Layout of the debug state vector used by jipm_debug_step: HOST out, offsets in doubles:
 * lay[0]=len, [1]=x, [2]=y, [3]=zL, [4]=zU, [5]=scalars(mu,tau,delta_w_last,theta_min,theta_max,k,status,nfilt),
 * [6]=filter (256 pairs theta,phi), [7]=dx, [8]=dy, [9]=dzL, [10]=dzU (step of the last iteration),
 * [11]=grad f, [12]=c, [13]=J blocks [N][nx][nx+nu], [14]=W blocks [N][nz][nz] then [nx][nx],
 * restoration mode (Step R): [15]=16 scalars (mode, then the parked regular mu, tau, delta_w_last, theta_min,
 * theta_max, #filter entries, theta at entry, zeta), [16]=(p, n) [2m], [17]=(z_p, z_n) [2m], [18]=x_R [n],
 * [19]=restoration filter (256 pairs).  With mode = 1 the fields [1]-[5] hold the restoration iterate and scalars
 * and [6] still holds the REGULAR filter.
 * Line-search memory of the active problem (Table I rows 3-5, 7): [20]=24 scalars (#consecutive shortened steps,
 * watchdog active?, #watchdog trials, watchdog reference theta, phi, grad_phi^T d, alpha, soft phase?, #soft
 * iterations, last step tiny?, tiny flag, adaptive mode free?, upper bound of mu, #remembered KKT errors, the errors [4]), [21]=watchdog entry iterate and direction: x, z_L, z_U, dx, dz_L, dz_U
 * (n + 2m each: the restoration variables follow the n entries), then y, dy (m each). */
int jipm_debug_state_layout(jipm_solver* s, int64_t* lay, int64_t n_lay);

/* Load P states (DEVICE [P x len], regular mode), run n_steps iterations each (stops early on a final
 * status), write the states back in place (step and derivative fields filled from the last iteration). */
int jipm_debug_step(jipm_solver* s, int64_t P, const double* params, double* state, int64_t n_steps);

/* Step I only: initialise P problems from (x0, params) and write their states (DEVICE [P x len]). */
int jipm_debug_init(jipm_solver* s, int64_t P, const double* x0, const double* params, double* state);

/* FP64 FMA microbenchmark (roofline denominator): runs dependent-free DFMA chains on all SMs and returns
 * the achieved TFLOP/s in *tflops (HOST out). */
int jipm_bench_fp64_peak(void* cuda_stream, double* tflops);

#ifdef __cplusplus
}
#endif
#endif /* JIPM_H */
