/* tmpc.h — C ABI of the B200-native batched ADMM-QP hot path of TurboMPC (arxiv/paper_2606_24039).
 *
 * Citations are lines of the paper text with the equation / algorithm they fall in.
 * The library solves, for a batch of B independent stage-structured QPs (eq. 1 / 28-31)
 *
 *     min 1/2 x'Px + q'x + gamma/2 |xi|^2 + lambda |xi|_1   s.t.  Cx = c,  lo <= Gx + delta.xi <= hi,
 *
 * with x = (x_t,u_t)_{t=0..N} (n = nx+nu per stage, T = N+1 stages), P block-tridiagonal (D_t, E_t),
 * C block-bidiagonal (A_init = [I 0], A_t^-, A_t^+), G block-diagonal, by the OSQP-style ADMM of Alg. 3
 * (PAPER.md:207-224): per iteration a solve with the block-tridiagonal S = P + sigma I + A' diag(rho) A
 * (eq. 8), over-relaxation (eq. 10), the (slack-smoothed) projection (eq. 12-15)
 * and the dual update (eq. 16).  tmpc_backward gives implicit-differentiation gradients (Alg. 2, eq. 59-65).
 *
 * Conventions
 *  - every array pointer is DEVICE memory owned by the caller (e.g. torch tensors), contiguous, in the working
 *    dtype of the handle (float for TMPC_F32, double for TMPC_F64); int32 for status.  Layouts are problem-major,
 *    row-major blocks, as written beside each field.  A batch stride of 0 means "one copy shared by the batch".
 *  - the library allocates no device memory: the caller passes a workspace of tmpc_workspace_bytes() bytes to
 *    tmpc_setup; the factor lives there from tmpc_factor until the next tmpc_factor / tmpc_destroy.
 *  - all calls enqueue on the stream given to tmpc_setup and return without synchronising
 *    (tmpc_admm_solve_host is the exception: it takes HOST buffers and synchronises before returning).
 *  - errors: bad arguments / shapes / call order -> a tmpc_status code and nothing is enqueued.  Numerical
 *    trouble never aborts the batch: bits are set in info.status[b] (TMPC_ST_*).
 *  - there is no CPU fallback: without a CUDA device every compute entry point returns TMPC_E_CUDA.
 */
#ifndef TMPC_H_
#define TMPC_H_
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TMPC_MAX_NG 32

typedef struct tmpc_ctx* tmpc_handle; /* opaque; owns nothing the caller passed in */

typedef enum { TMPC_OK = 0, TMPC_E_BADARG, TMPC_E_DIM, TMPC_E_UNSUPPORTED, TMPC_E_STATE, TMPC_E_WORKSPACE, TMPC_E_CUDA,
               TMPC_E_STATIC_LIMIT /* tmpc_admm_solve_static: the problem needs more than TMPC_STATIC_SCRATCH_BYTES of scratch */ } tmpc_status;
typedef enum { TMPC_F32 = 0, TMPC_F64 = 1 } tmpc_dtype;
typedef enum { TMPC_MODEL_NONE = 0, TMPC_MODEL_BICYCLE_IMPLICIT_MIDPOINT = 1, TMPC_MODEL_SRB_HUMANOID_RK4 = 2 } tmpc_model;
typedef enum { TMPC_LIN_SEQUENTIAL = 0, TMPC_LIN_CYCLIC_REDUCTION = 1, TMPC_LIN_AUTO = 2 } tmpc_linsolve;
typedef enum { TMPC_BWD_REFACTOR_REFINE = 0, TMPC_BWD_ADMM_REUSE_FACTOR = 1 } tmpc_bwd_mode;

/* info.status[b] bits */
#define TMPC_ST_PIVOT 1  /* a non-positive or non-finite pivot was met while factoring S (replaced by 1: the problem's result is garbage) */
#define TMPC_ST_NAN 2    /* a non-finite value appeared in the iterate */
/* tmpc_admm_solve flags */
#define TMPC_SOLVE_ZG_GIVEN 1 /* use state.zg / state.xi as passed (resume); default z_g^0 = clip(G x^0, lo, hi) */

typedef struct { /* POD, copied at tmpc_setup */
  int32_t batch, N, nx, nu, ng; /* n_init = nx: the rows x_0 = x_init are implicit (A_init = [I 0]) */
  int32_t dtype;                /* tmpc_dtype */
  int32_t model;                /* tmpc_model, used by tmpc_linearize only */
  int32_t linsolve;             /* tmpc_linsolve */
  double sigma, rho_bar, rho_eq_scale, alpha; /* sigma=1e-6, rho_g=rho_bar, rho_f=rho_eq_scale*rho_bar, alpha in (0,2) */
  double slack_gamma, slack_lambda;           /* gamma_xi and an L1 slack weight lambda >= 0 (0 = the paper's scheme) */
  double eps_active_abs, eps_active_rel;      /* active-set classification of tmpc_backward */
  double wheelbase, dt;                       /* bicycle model */
  double g_lo[TMPC_MAX_NG], g_hi[TMPC_MAX_NG]; /* un-shifted bounds of g_t(x,u) for tmpc_linearize (eq. 38) */
  int32_t g_is_selection;                     /* 1: row r of every G_t is the unit vector e_{g_col[r]} and qp.G is NULL */
  int32_t g_col[TMPC_MAX_NG];
  uint8_t soft_row[TMPC_MAX_NG];              /* per-row delta_xi, same for every stage and problem */
  double model_params[16];                    /* TMPC_MODEL_SRB_HUMANOID_RK4 (eq. 68-69; nx = 12, nu = 6, step `dt`): mass, g[3],
                                                 diag of the body inertia [3], world positions of the left and the right foot [3] + [3] */
} tmpc_config;

typedef struct {
  const void* D; int64_t D_bstride; /* [B|1][T][n][n]   symmetric diagonal blocks of P (eq. 29), full storage            */
  const void* E; int64_t E_bstride; /* [B|1][N][n][n]   block (t+1,t) of P                                               */
  const void* q;                    /* [B][T][n]                                                                         */
  const void* Am; const void* Ap;   /* [B][N][nx][n]    A_t^-, A_t^+ (eq. 36): Am v_t + Ap v_{t+1} = b_t                   */
  const void* b;                    /* [B][N][nx]                                                                        */
  const void* x_init;               /* [B][nx]                                                                           */
  const void* G; int64_t G_bstride; /* [B|1][T][ng][n]  or NULL with g_is_selection (eq. 31)                             */
  const void* lo; const void* hi;   /* [B][T][ng]       +-INFINITY allowed (eq. 38)                                      */
} tmpc_qp; /* tmpc_linearize WRITES Am, Ap, b, G, lo, hi (the caller passes writable buffers there).  D, E, Am, Ap, b and G must be 16-byte
            * aligned (bulk copies of the streamed class, vector stores of tmpc_linearize): TMPC_E_BADARG otherwise. */

typedef struct { /* ADMM state, in/out = warm start (Alg. 3 'Initial guess') */
  void* x;  /* [B][T][n]   */
  void* zg; /* [B][T][ng]  */
  void* yf; /* [B][nx+N*nx] multipliers of (x_0 = x_init ; dynamics rows) */
  void* yg; /* [B][T][ng]  */
  void* xi; /* [B][T][ng]  slack, out (in with TMPC_SOLVE_ZG_GIVEN) */
} tmpc_state;

typedef struct { /* per-problem outputs at the last iterate (eq. 3); any pointer may be NULL */
  void* r_prim; void* r_dual; void* objective; /* [B] working dtype */
  int32_t* status;                             /* [B] TMPC_ST_* bits, OVERWRITTEN by tmpc_admm_solve (no need to zero it): TMPC_ST_PIVOT as
                                                  found by the last tmpc_factor (kept per problem in the workspace), TMPC_ST_NAN from the iterate */
} tmpc_info;

/* Bytes of device workspace tmpc_setup needs for this config. */
tmpc_status tmpc_workspace_bytes(const tmpc_config* cfg, size_t* bytes);
/* Creates a handle. workspace: device memory of >= tmpc_workspace_bytes() bytes, 256-byte aligned, caller-owned and
 * alive until tmpc_destroy.  cuda_stream: a cudaStream_t (NULL = default stream). */
tmpc_status tmpc_setup(const tmpc_config* cfg, void* workspace, size_t bytes, void* cuda_stream, tmpc_handle* out);
/* a1 (eq. 36-38): linearise the built-in model at xbar [B][T][n] against stage_ref [B][T][n]
 * (x_ref,u_ref per stage); writes qp->Am, Ap, b, G, lo, hi.  TMPC_E_UNSUPPORTED for TMPC_MODEL_NONE.
 * TMPC_MODEL_SRB_HUMANOID_RK4 has box bounds on u only (eq. 70d: selection rows, constant bounds): it writes Am, Ap, b and leaves qp->G, lo,
 * hi alone (G may be NULL, stage_ref is not read). */
tmpc_status tmpc_linearize(tmpc_handle h, const void* xbar, const void* stage_ref, tmpc_qp* qp);
/* a2+a3: assemble Theta_t, Phi_t and factor S block by block into the workspace. */
tmpc_status tmpc_factor(tmpc_handle h, const tmpc_qp* qp);
/* a4-a9 (Alg. 3): exactly `iters` ADMM iterations on every problem, no early exit; needs tmpc_factor first.
 * Enqueues one fused kernel for all iterations, or, for the streamed class with more problems than co-resident CTAs,
 * several launches of it over iteration chunks (same arithmetic, bit-identical state), plus the residual kernel (a9)
 * when `info` has a non-NULL pointer.  The state in `st` is complete between calls: a later call with
 * TMPC_SOLVE_ZG_GIVEN continues where this one stopped. */
tmpc_status tmpc_admm_solve(tmpc_handle h, const tmpc_qp* qp, tmpc_state* st, int32_t iters, int32_t flags, tmpc_info* info);
/* f1 — Alg. 3 as the paper runs it: adaptive step size and early termination (eq. 4, 299-303 eq. 17, 380).
 * Every `check_every` iterations (k_rho^iter, paper default 25) and at iteration max_iters each live problem evaluates r_prim, r_dual
 * (eq. 3) and the scales |(Ax, z)|_inf, |(Px, A'y, q, gamma xi, y_g on soft rows)|_inf; a problem that satisfies eq. 4 stops there
 * (its state is final); otherwise, if adapt_rho, rho_new = clip(rho_bar sqrt((r_prim/|.|)/(r_dual/|.|)), [rho_min, rho_max]) replaces
 * its rho_bar when max(rho_new/rho_bar, rho_bar/rho_new) > rho_ratio (paper: 5), and only those problems are re-factorised. */
typedef struct {
  int32_t max_iters;                  /* K_max >= 1 */
  int32_t check_every;                /* k_rho^iter >= 1 */
  int32_t adapt_rho;                  /* 0: termination test only */
  int32_t reserved;
  double eps_abs, eps_rel;            /* eq. 4 */
  double rho_ratio, rho_min, rho_max; /* k_rho^ratio and the clip bounds of eq. 17 (paper: 5, 1e-6, 1e6) */
} tmpc_adaptive;
/* Needs tmpc_factor first (every problem starts from cfg.rho_bar) and, unlike the other calls, SYNCHRONISES: the count of live problems
 * of every round is read back (one round behind the launches, through a pinned page the library allocates once per process) so that the
 * call returns when all have terminated; it returns with the stream idle.  Outputs (DEVICE, [B], any may be NULL): iterations
 * each problem ran, 1 if it met eq. 4, its final rho_bar (working dtype); info as in tmpc_admm_solve, at each problem's last check.
 * Afterwards the factor in the workspace belongs to the per-problem rho_bar values: call tmpc_factor before the next solve.
 * TMPC_E_UNSUPPORTED for cyclic reduction. */
tmpc_status tmpc_admm_solve_adaptive(tmpc_handle h, const tmpc_qp* qp, tmpc_state* st, const tmpc_adaptive* ad, int32_t flags, tmpc_info* info,
                                     int32_t* iters_out, int32_t* converged_out, void* rho_out);
/* f2 — the SQP outer loop of Alg. 1 for the built-in model: per iteration tmpc_linearize at the iterate st.x,
 * tmpc_factor, `admm_iters` iterations of Alg. 3 warm-started there (y carried, z_g re-projected), then the backtracking linesearch of
 * App. D on the l1 merit function with the candidates alpha = 2^-j, j < n_alpha, evaluated in parallel: the largest
 * that satisfies the Armijo condition with eta, else the one with the smallest merit; (x, xi, y) move by alpha along the QP step.
 * A problem stops when eq. 18 holds at its iterate: stationarity, |f|_inf and the bound violation all <= eps_c. */
typedef struct {
  int32_t max_sqp, admm_iters, n_alpha, reserved;   /* n_alpha <= 15 */
  double eps_c, eta;                                /* eq. 18 tolerance; Armijo parameter (paper: 0.4) */
} tmpc_sqp_opts;
/* st.x holds the start iterate and receives the final one (st.yf, st.yg, st.xi likewise); qp->Am, Ap, b, G, lo, hi are written every
 * iteration (as by tmpc_linearize).  Outputs (DEVICE, any may be NULL): SQP iterations per problem [B], eq. 18 met [B], the accepted alpha
 * of every iteration [B][max_sqp] and the eq. 18 quantities of the last test [B][3] (working dtype).  Like tmpc_admm_solve_adaptive the
 * call SYNCHRONISES once per iteration (count of live problems) and leaves the workspace factor unusable for a later tmpc_admm_solve.
 * Both built-in models (for TMPC_MODEL_SRB_HUMANOID_RK4 the equality residual of the merit function is Phi(x_k, u_k) - x_{k+1}, the inequality
 * rows are the handle's selection rows with the caller's constant qp->lo, qp->hi, and stage_ref is not read); TMPC_E_UNSUPPORTED for
 * TMPC_MODEL_NONE and with cyclic reduction. */
tmpc_status tmpc_sqp_solve(tmpc_handle h, tmpc_qp* qp, tmpc_state* st, const void* stage_ref, const tmpc_sqp_opts* o, int32_t* iters_out,
                           int32_t* converged_out, void* alpha_log, void* kkt_out);
/* a10 (Alg. 2, eq. 59-65): dL/dq [B][T][n] and dL/dx_init [B][nx] from dL/dx [B][T][n] (and dL/dxi [B][T][ng] or NULL)
 * at the state st.  dL/dxi is the gradient with respect to the SIGNED slack st.xi that tmpc_admm_solve returns
 * (lo <= Gx + xi <= hi; App. E's xi_A of eq. 54 is |xi| = sign(xi) xi, so eq. 65's S dL/dxi_A is dL/dxi); only its
 * entries on soft-active rows (xi != 0) are read.  REFACTOR_REFINE factors the adjoint-weighted S and runs `iters` refinement sweeps of the
 * active-set KKT system; ADMM_REUSE_FACTOR runs `iters` ADMM iterations on the adjoint QP (eq. 67) with the
 * forward factor.  Overwrites the factor in the workspace in REFACTOR_REFINE mode.  TMPC_E_UNSUPPORTED for handles that use cyclic reduction
 * (TMPC_LIN_CYCLIC_REDUCTION, or AUTO where it picked it). */
tmpc_status tmpc_backward(tmpc_handle h, const tmpc_qp* qp, const tmpc_state* st, const void* dL_dx, const void* dL_dxi,
                          int32_t mode, int32_t iters, void* dL_dq, void* dL_dxinit);
/* eq. 66: dL/dgamma_xi [B] (working dtype, DEVICE) = sum over the soft-active rows of xi_i (G eta_x)_i, from the
 * dL/dq = -eta_x that the preceding tmpc_backward of the same state returned (its row classification is kept in the workspace;
 * TMPC_E_STATE without one). */
tmpc_status tmpc_backward_dgamma(tmpc_handle h, const tmpc_qp* qp, const tmpc_state* st, const void* dL_dq, void* dL_dgamma);
/* Applies the current factor: xt [B][T][n] = S^{-1} eta [B][T][n] (eq. 8).  Test/diagnostic entry. */
tmpc_status tmpc_kkt_solve(tmpc_handle h, const void* eta, void* xt);
/* Same as tmpc_factor + tmpc_admm_solve but every pointer in qp/st/info is HOST memory (pinned for speed); the
 * library stages through `staging` (device, >= tmpc_host_staging_bytes()), copies results back and synchronises. */
tmpc_status tmpc_host_staging_bytes(const tmpc_config* cfg, size_t* bytes);
tmpc_status tmpc_admm_solve_host(tmpc_handle h, const tmpc_qp* host_qp, tmpc_state* host_st, int32_t iters, int32_t flags,
                                 tmpc_info* host_info, void* staging, size_t staging_bytes);
/* Diagnostic: measures a roofline denominator of this GPU at the clocks found with a micro-benchmark kernel.
 * what = TMPC_PEAK_FFMA2 / FFMA / DFMA -> *out in TFLOP/s (independent fused multiply-add chains, 3-register form);
 * TMPC_PEAK_LDS -> *out in GB/s (conflict-free 16-byte shared-memory loads).  scratch: >= 16 bytes of DEVICE memory.
 * Runs `reps` timed launches (+1 warm-up) on cuda_stream, synchronises, returns the best.  HOST pointer `out`. */
#define TMPC_PEAK_FFMA2 0
#define TMPC_PEAK_FFMA 1
#define TMPC_PEAK_DFMA 2
#define TMPC_PEAK_LDS 3
tmpc_status tmpc_measure_peak(int32_t what, void* scratch, void* cuda_stream, int32_t reps, double* out);
/* Allocation-free variant of tmpc_factor + tmpc_admm_solve for callers that cannot allocate device memory (CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): no handle, no caller workspace.  The scratch the kernels need (the block factor of S, the per-problem
 * status word, residual partials) lives in ONE file-scope `static __device__` array of TMPC_STATIC_SCRATCH_BYTES inside the library, which every
 * GPU that loads the library holds until the process exits.  cfg, qp, st, info, iters, flags as in tmpc_setup / tmpc_admm_solve (qp, st, info
 * are DEVICE pointers owned by the caller); the kernels are enqueued on cuda_stream and the call returns without synchronising.
 *  - a problem whose tmpc_workspace_bytes(cfg) exceeds TMPC_STATIC_SCRATCH_BYTES is rejected with TMPC_E_STATIC_LIMIT and nothing is enqueued;
 *    TMPC_LIN_CYCLIC_REDUCTION (and AUTO where it would pick it) returns TMPC_E_UNSUPPORTED;
 *  - the call makes no cudaMalloc / cudaFree / allocating library call (it uses cudaGetSymbolAddress once per device, cudaMemsetAsync and
 *    kernel launches);
 *  - ALL calls on a device share the one array, which keeps the contents of the previous call: the status words are cleared at the start of
 *    every call, everything else is written before it is read.  Two calls that overlap on the GPU (different streams, or different host
 *    threads without ordering) RACE on the array: serialise them on one stream or with events. */
#define TMPC_STATIC_SCRATCH_BYTES (8u << 20)
tmpc_status tmpc_admm_solve_static(const tmpc_config* cfg, const tmpc_qp* qp, tmpc_state* st, int32_t iters, int32_t flags, tmpc_info* info,
                                   void* cuda_stream);
tmpc_status tmpc_destroy(tmpc_handle h);
const char* tmpc_status_string(tmpc_status s);
/* Number of kernels this handle has launched so far (for bench.py's gpu_launches). */
int64_t tmpc_launch_count(tmpc_handle h);

#ifdef __cplusplus
}
#endif
#endif /* TMPC_H_ */
