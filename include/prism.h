/* prism.h - C ABI of the B200-native batched rebalancing solver.
 *
 * What it solves.  For each of A accounts over a shared universe of N instruments, the per-account convex program
 * the paper states as Eq. (1) (Section 4.2), in the concretisation of SURVEY.md 8.0:
 *
 *   minimise   (gamma/2) (w-w_b)' Sigma (w-w_b) - mu'w + kappa ||w-w0||_1
 *              + sum_i [ c_buy (w_i-w0_i)_+ + psi_i((w0_i-w_i)_+) ]            (psi_i: convex piecewise-linear lot penalty)
 *   subject to 1'w = 1,  lo_i <= w_i <= hi_i,  band_lo_g <= sum_{i in g} w_i <= band_hi_g,  ||w-w0||_1 <= tau
 *   Sigma = B diag(f) B' + diag(d)     (factor-structured risk)
 *
 * by a batched ADMM (operator splitting, BASELINE.json:north_star) whose steps are hand-written sm_100a kernels:
 * fp64 factor GEMMs and one fused proximal/projection kernel that holds EVERY nonsmooth and polyhedral term - budget
 * hyperplane, box, exclusions, L1 turnover (buy/sell two-threshold split), group bands, buy cost, lot penalties -
 * together with the dual update, the residuals, the per-account convergence mask and the rho adaptation.  The returned
 * weights are the projection-side iterate: budget, box, exclusions, turnover cap and group bands hold to rounding.
 *
 * Boundary (Fig. 2): problem data in; weights, fixed-vocabulary status codes
 * (Table 14), timings (lanes of Table 4), memory bytes (Table 6) and the
 * external diagnostics of Section 4.4 out.
 *
 * Conventions
 *  - Every pointer inside prism_data and every *_out / w / duals argument is a DEVICE pointer (cudaMalloc'd or a
 *    torch CUDA tensor's data_ptr), 16-byte aligned.  prism_constraint_set, prism_settings, prism_solve_info are
 *    HOST structs.
 *  - Layout of every per-account array: account-major, element (a, i) at [a * N + i] (the N assets of one account
 *    are contiguous).  Lot arrays: element (a, i, l) at [(a * N + i) * PRISM_MAX_LOTS + l].
 *  - Ownership: all data arrays are BORROWED; they must outlive the problem object and must not change during a
 *    call.  The library owns only its workspace.  No hidden host<->device copies of N x A arrays.
 *  - Errors: every call returns an int (0 = PRISM_OK); nothing throws or aborts across the ABI; a per-account
 *    difficulty (iteration cap, NaN, gate failure) is a STATUS, not an error.  prism_last_error() gives the text.
 *  - The turnover scaling D_a of Eq. (1) is the identity in this build (as in every configured
 *    workload); a non-NULL d_t is rejected with PRISM_ERR_INVALID_ARG.
 *  - Domain: lo_a <= hi_a finite per account.  Universes too wide for the cluster-resident projection (N above
 *    ~80,000) take the streaming form, whose per-group constants are accumulated in 2^-60 fixed point: there
 *    hi_a - lo_a <= 4 is required per asset and the sum of the constant trades of one group must stay below 16
 *    (always true for a budget-1 book); wider boxes take the every-asset kernel instead.
 */
#ifndef PRISM_H
#define PRISM_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* the library is built with hidden default visibility: exactly the functions declared here are exported */
#if defined(__GNUC__)
#define PRISM_API __attribute__((visibility("default")))
#else
#define PRISM_API
#endif

#define PRISM_MAX_LOTS 4
#define PRISM_MAX_GROUPS 64
#define PRISM_MAX_FACTORS 128

/* error codes */
enum { PRISM_OK = 0, PRISM_ERR_INVALID_ARG = 1, PRISM_ERR_ALLOC = 2, PRISM_ERR_CUDA = 3, PRISM_ERR_NOT_READY = 4 };

/* status vocabulary, Table 14 */
enum {
  PRISM_STATUS_CERTIFIED = 0,        /* own tolerance met and the external gates pass                            */
  PRISM_STATUS_FEASIBLE = 1,         /* gates pass, tolerance not met (the paper's iteration-capped case, :435)  */
  PRISM_STATUS_TIMEOUT = 2,          /* time_limit_ms reached before the account finished                        */
  PRISM_STATUS_LATE = 3,             /* finished, but after deadline_ms                                           */
  PRISM_STATUS_NO_FEASIBLE = 4,      /* gates fail at exit; NOT a certified-infeasibility claim (:491)           */
  PRISM_STATUS_FAILURE = 5           /* allocation / numerical failure (NaN or Inf seen)                          */
};

/* constraint-set flags: the rule bundles of the burden curve, Table 9 */
enum {
  PRISM_BUDGET = 1, PRISM_BOX = 2, PRISM_EXCLUSION = 4, PRISM_TURNOVER_CAP = 8, PRISM_TURNOVER_PENALTY = 16,
  PRISM_GROUP_BANDS = 32, PRISM_TAX_LOTS = 64, PRISM_BUY_COST = 128, PRISM_BENCHMARK_SHIFT = 256
};

/* form of the fused projection kernel (H4); AUTO picks the first that applies */
enum { PRISM_PROX_AUTO = 0,
       PRISM_PROX_RESIDENT = 1,   /* one thread-block cluster per account, the account resident in shared memory    */
       PRISM_PROX_STREAMING = 2,  /* streaming pass + per-account root kernel: wide universes, no lots / caps        */
       PRISM_PROX_EVERY_ASSET = 3 /* one CTA per account re-reading the account per pass: always applicable         */ };

typedef struct prism_constraint_set {
  uint32_t flags;      /* OR of the flags above; PRISM_BUDGET and PRISM_BOX are mandatory                       */
  int32_t G;           /* number of groups (0 unless PRISM_GROUP_BANDS), <= PRISM_MAX_GROUPS                    */
  int32_t max_lots;    /* lots per asset (0 unless PRISM_TAX_LOTS), <= PRISM_MAX_LOTS                           */
  int32_t prox_form;   /* PRISM_PROX_*; a form that does not apply to the problem is PRISM_ERR_INVALID_ARG      */
} prism_constraint_set;

/* columns of the residual block, one row of PRISM_NRES doubles per account */
enum {
  PRISM_R_BUDGET = 0,   /* |1'w - 1| */
  PRISM_R_BOX = 1,      /* max(||(lo-w)_+||_inf, ||(w-hi)_+||_inf) */
  PRISM_R_EXPOSURE = 2, /* max over groups of band violation */
  PRISM_R_TURNOVER = 3, /* (||w-w0||_1 - tau)_+                                PAPER.md:142 */
  PRISM_R_STAT = 4,     /* stationarity, subgradient-distance form             PAPER.md:146; NaN without duals */
  PRISM_R_COMP = 5,     /* complementarity max_i |lambda_i g_i(w)|             PAPER.md:146; NaN without duals */
  PRISM_R_OBJECTIVE = 6,/* public objective f(w) */
  PRISM_R_PRIMAL = 7,   /* scaled primal residual of the splitting at exit (solver only, else NaN)              */
  PRISM_R_DUAL = 8,     /* scaled dual residual of the splitting at exit   (solver only, else NaN)              */
  PRISM_R_TURNOVER_VALUE = 9, /* ||w-w0||_1                                                                      */
  PRISM_R_RHO = 10,     /* final rho scale c_a (solver only, else NaN)                                           */
  PRISM_R_RESERVED = 11,/* 0, or why the constraint-set precheck returned the account at iteration 0 with w = w0 and status
                           NO_FEASIBLE: 1 box / budget, 2 turnover cap below the forced trades, 3 group bands        */
  PRISM_NRES = 12
};

/* multipliers ("certificate data"): per account 2 + 2 G doubles:
 *   [0] nu (budget), [1] theta >= 0 (turnover cap), [2 .. 2+G) lam_hi >= 0, [2+G .. 2+2G) lam_lo >= 0        */
#define PRISM_NDUAL(G) (2 + 2 * (G))

typedef struct prism_data {
  /* shared universe */
  const void* B;            /* N x k row-major loadings; fp64, or fp32 when B_is_fp32 != 0                       */
  int32_t B_is_fp32;
  const double* f;          /* k   factor variances  > 0                                                        */
  const double* d;          /* N   idiosyncratic variances > 0                                                  */
  const uint8_t* group_id;  /* N   group of each asset in [0, G); NULL when G == 0                               */
  const double* d_t;        /* must be NULL (identity) in this build                                            */
  /* per account, account-major */
  const double* mu;         /* A x N  return input                                                               */
  const double* gamma;      /* A      risk aversion > 0                                                          */
  const double* w0;         /* A x N  current weights                                                            */
  const double* w_b;        /* A x N  benchmark in the risk term, or NULL (=> 0)                                 */
  const double* lo;         /* A      lower bound per account                                                    */
  const double* hi;         /* A      upper bound per account (ignored where hi_full is given)                   */
  const double* hi_full;    /* A x N  per-asset upper bounds (restriction caps), or NULL                         */
  const uint8_t* excl;      /* A x N  1 => w_i = 0 (exclusion), or NULL                                          */
  const double* tau;        /* A      turnover cap, +inf for none; NULL => none                                  */
  const double* kappa;      /* A      L1 transition penalty weight, or NULL (=> 0)                               */
  const double* band_lo;    /* A x G                                                                              */
  const double* band_hi;    /* A x G                                                                              */
  const double* c_buy;      /* A      linear buy cost, or NULL (=> 0)                                            */
  const double* lot_slope;  /* A x N x PRISM_MAX_LOTS ascending sell-penalty slopes, or NULL                     */
  const double* lot_width;  /* A x N x PRISM_MAX_LOTS lot sizes (sum over live lots = sellable amount)           */
  const uint8_t* lot_count; /* A x N  live lots per asset in [0, max_lots]; 0 => no penalty, sells limited by lo */
} prism_data;

enum { PRISM_GEMM_FP64_TENSOR = 0,   /* fp64 on the tensor pipe (DMMA mma.sync.m8n8k4)                              */
       PRISM_GEMM_FP64_FMA = 1,      /* fp64 FMA kernels of the same contract (validation twin)                     */
       PRISM_GEMM_TF32X3 = 3,        /* TF32 tensor path with the 3xTF32 split (fp32-level accuracy, fp32 accumulators):
                                        both GEMMs become HBM-bound instead of fp64-pipe-bound                    */
       PRISM_GEMM_FP32_EXPERIMENT = 2 /* the FMA twins with both operands rounded to fp32 and fp32 accumulation: NOT a
                                        production path - the measurement behind the precision choice: the
                                        Sigma-apply of the external diagnostics stays fp64                         */ };

typedef struct prism_settings {
  double eps_rel;           /* scaled primal/dual tolerance (default 1e-6; BASELINE.json:metric "1e-6 KKT")      */
  double eps_abs;           /* absolute part: converged when r <= eps_abs + eps_rel * scale (default 0)          */
  int32_t max_iter;         /* iteration cap (default 4000)                                                      */
  int32_t check_every;      /* residual / convergence-mask cadence in iterations (default 10)                    */
  int32_t first_check;      /* no residual check before this many iterations (default 40): the first checks of a
                               cold start never pass and a check launch costs more than a plain one          */
  int32_t adapt_rho;        /* 1 => per-account rho adaptation at check iterations (default 1)                   */
  int32_t adapt_start;      /* first iteration at which an account's rho may be adapted (default 200: typical
                               accounts finish before, and adapting them earlier slows them down)               */
  int32_t adapt_every;      /* minimum iterations between two adaptations of one account (default 100)           */
  double alpha;             /* over-relaxation in (0, 2) (default 1.6)                                           */
  double rho_scale;         /* initial c: rho_i = c gamma_a d_i (default 100)                                    */
  int32_t gemm_precision;   /* PRISM_GEMM_* (default PRISM_GEMM_TF32X3, chosen against the tolerance by measurement:
                               DESIGN.md section 5); the external diagnostics are fp64 whatever this says        */
  int32_t profile;          /* 1 => bracket every kernel launch with CUDA events (read with prism_kernel_times);
                               adds event overhead, so never combine with a throughput measurement           */
  double time_limit_ms;     /* 0 => none; accounts unfinished at the limit get PRISM_STATUS_TIMEOUT              */
  double deadline_ms;       /* 0 => none; accounts finishing after it get PRISM_STATUS_LATE                      */
  double prox_window_mult;  /* projection: next live-list window = this x the last movement of the thresholds
                               (default 32)                                                                   */
  int32_t sample_until;     /* streaming form of the projection: plain (non-check) launches of iterations < sample_until,
                               while the group bands are still out of the projection (the first 21 iterations of a cold
                               start), find the thresholds on a SAMPLE of the live assets (every stride-th, scaled) and
                               apply them to all - an inexact prox.  The splitting's only carried state is v, so this
                               perturbs the path of the iteration, not its fixed point; check / final launches are always
                               exact.  0 => never; -1 (default) => 6, or 12 for universes of 65,536 instruments and more (measured on
                               configs[2] / [3] / [4])                                          */
  int32_t reserved0;
  /* warm start - the repeated-run lane (cold rows "pass no previous solution"): previous weights and
     multipliers of the same accounts, e.g. the w_out / duals_out of an earlier call.  Both NULL => cold start.       */
  const double* warm_w;     /* device, A x N, or NULL                                                            */
  const double* warm_duals; /* device, A x PRISM_NDUAL(G), or NULL (=> zero multipliers)                         */
} prism_settings;

typedef struct prism_solve_info {
  double solve_interval_ms; /* CUDA events around the device work: "reported solve interval" lane */
  double wall_ms;           /* host clock around the call incl. final sync: full-call lane        */
  int64_t device_bytes;     /* workspace owned by the problem object: memory class (Table 6)       */
  int32_t iters_max;        /* iterations of the slowest account                                                 */
  int64_t iters_total;      /* sum over accounts of iterations run                                               */
  int32_t n_certified, n_feasible, n_timeout, n_late, n_no_feasible, n_failed;
  int64_t kernel_launches;  /* kernels launched by this call                                                     */
} prism_solve_info;

typedef struct prism_problem prism_problem;

/* Fills *s with the defaults listed above. */
PRISM_API void prism_default_settings(prism_settings* s);

/* Validates shapes and flags, adopts the borrowed device pointers in `data`, allocates ALL workspace once and
 * precomputes what does not depend on the iterate (padded copies of B, the shared Gram matrix U' D^-1 U, q when a
 * benchmark shift is present).  N >= 1, 1 <= k <= PRISM_MAX_FACTORS, accounts >= 1.  Runs on `cuda_stream`
 * (a cudaStream_t, NULL = default stream) and synchronises it.  On failure *out = NULL; PRISM_ERR_ALLOC means
 * the problem object was not allocated (status 5 for every account). */
PRISM_API int prism_problem_create(int64_t N, int32_t k, int32_t accounts, const prism_constraint_set* cs,
                         const prism_data* data, void* cuda_stream, prism_problem** out);

/* Runs the batched solver on `cuda_stream` and synchronises it before returning.  Cold start (default):
 * z = projection of w0, zero duals.  Warm start: see prism_settings.warm_w.
 *   w_out      device, A x N   returned weights
 *   status_out device, A int32 status vocabulary above
 *   iters_out  device, A int32 iterations run per account
 *   resid_out  device, A x PRISM_NRES doubles, or NULL
 *   duals_out  device, A x PRISM_NDUAL(G) doubles, or NULL
 *   info       host, or NULL
 * Re-entrant per problem object; not thread-safe on one object. */
PRISM_API int prism_solve_batch(prism_problem* p, const prism_settings* s, void* cuda_stream, double* w_out,
                      int32_t* status_out, int32_t* iters_out, double* resid_out, double* duals_out,
                      prism_solve_info* info);

/* External-diagnostic semantics: depends only on the problem data and the given w (and
 * multipliers, if any), never on solver state, so it applies to any solver's weights.  Fills columns 0..6 and 9
 * of the residual block (4, 5 are NaN when duals == NULL; 7, 8, 10 are NaN).  Synchronises the stream. */
PRISM_API int prism_residuals(prism_problem* p, const double* w, const double* duals, void* cuda_stream,
                    double* resid_out);

/* ONE application of the fused projection (H4) to caller-given points, outside any iteration - the prox of every
 * nonsmooth / polyhedral term of Eq. (1) in the metric the splitting uses:
 *   z_a = argmin_z  sum_i rho_ai / 2 (z_i - v_ai)^2 + kappa_a |z_i - w0_ai| + c_buy,a (z_i - w0_ai)_+ + psi_ai((w0_ai - z_i)_+)
 *         s.t.  1'z = 1,  lo <= z <= hi (exclusions z_i = 0),  band_lo <= E z <= band_hi,  ||z - w0||_1 <= tau_a
 *   rho_ai = rho_scale * gamma_a * d_i.
 * Solved exactly (the piecewise-linear equations for the multipliers to 2e-15) by the same kernel the iteration
 * launches, from a cold start.  v: device A x N; z_out: device A x N; duals_out: device A x PRISM_NDUAL(G) multipliers
 * of the projection (layout above), or NULL.  Overwrites the solver's iterate (the next prism_solve_batch starts
 * cold anyway).  Synchronises the stream. */
PRISM_API int prism_project(prism_problem* p, const double* v, double rho_scale, void* cuda_stream, double* z_out,
                  double* duals_out);

/* Same solve as prism_solve_batch but with HOST buffers for the per-account data that changes between
 * rebalances (mu, w0) and for the outputs: copies mu and w0 host->device into the problem's borrowed arrays,
 * solves, copies weights / status / iterations / residual block back.  NULL host pointers skip that copy.
 * The other per-account data (bounds, masks, bands, tau, gamma) stays resident from prism_problem_create.
 * This is the end-to-end lane of bench.py ("e2e"). */
PRISM_API int prism_solve_batch_host(prism_problem* p, const prism_settings* s, void* cuda_stream, const double* mu_host,
                           const double* w0_host, double* w_host, int32_t* status_host, int32_t* iters_host,
                           double* resid_host, prism_solve_info* info);

/* Kernel classes of the hot path: H4-H7 fused prox (k_prox_res; for the streaming form both of its
 * kernels), H1 GEMM-1, H2 small solve, H3 GEMM-2 + epilogue, H0/H7 capacitance factorisation, H8/H9 diagnostics,
 * everything else.  PRISM_K_PROX_ROOT is kept for layout stability and stays 0. */
enum { PRISM_K_PROX = 0, PRISM_K_GEMM1 = 1, PRISM_K_SOLVE = 2, PRISM_K_GEMM2 = 3, PRISM_K_FACTOR = 4, PRISM_K_DIAG = 5,
       PRISM_K_OTHER = 6, PRISM_K_PROX_ROOT = 7, PRISM_NKERN = 8 };

/* Device time (ms, CUDA events on the solve stream) and launch count per kernel class of the last
 * prism_solve_batch call that ran with settings.profile = 1.  ms_out, launches_out: host arrays of PRISM_NKERN. */
PRISM_API int prism_kernel_times(const prism_problem* p, double* ms_out, int64_t* launches_out);

/* Factor exposures of caller-given weights through the problem's own GEMM-1 (H1):
 *   T_out[a * k + j] = sum_i B[i][j] w[a * N + i]       w: device A x N, T_out: device A x k.
 * Split-K partials live in the workspace allocated at create.  Synchronises the stream. */
PRISM_API int prism_factor_exposures(prism_problem* p, const double* w, void* cuda_stream, double* T_out);

/* ---- the one entry point that ALLOCATES NOTHING (for CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc).  Same result as prism_factor_exposures, no problem object:
 *   T_out[a * k + j] = sum_i B[i * k + j] X[a * N + i]   B: device N x k row-major (fp64, or fp32 when B_is_fp32),
 *                                                        X: device accounts x N, T_out: device accounts x k.
 * Its split-K partials live in a static __device__ array of PRISM_NOALLOC_SCRATCH_DOUBLES doubles (4 MiB) that every
 * GPU loading the library holds until exit.  Limit: accounts * k <= PRISM_NOALLOC_SCRATCH_DOUBLES, else
 * PRISM_ERR_INVALID_ARG.  Asynchronous on cuda_stream (no synchronisation); calls no cudaMalloc / cudaFree.
 * All calls SHARE the array: calls that overlap on the GPU (different streams, concurrently replayed graphs) race -
 * serialise them.  Nothing has to be cleared between calls (every partial read is written by the same call first).
 * prism_noalloc_init() fetches the array's device address for the current device (cudaGetSymbolAddress); call it
 * once per device before a graph capture - the entry point does the same lazily otherwise. */
#define PRISM_NOALLOC_SCRATCH_DOUBLES 524288
PRISM_API int prism_noalloc_init(void);
PRISM_API int prism_factor_exposures_noalloc(const void* B, int32_t B_is_fp32, const double* X, int64_t N, int32_t k,
                                   int32_t accounts, void* cuda_stream, double* T_out);

/* fp64 yardstick of THIS device: register-resident loops without memory traffic, CUDA-event timed on
 * cuda_stream, best of 5.  tflops_out (host, 2 doubles): [0] tensor pipe (DMMA mma.sync m8n8k4), [1] FMA pipe. */
PRISM_API int prism_fp64_yardstick(prism_problem* p, void* cuda_stream, double* tflops_out);

/* Frees the workspace; never frees borrowed data.  NULL is allowed. */
PRISM_API void prism_problem_destroy(prism_problem* p);

/* The form of the projection kernel this object runs (PRISM_PROX_RESIDENT / _STREAMING / _EVERY_ASSET): what
 * PRISM_PROX_AUTO resolved to. */
PRISM_API int32_t prism_problem_prox_form(const prism_problem* p);

/* Workspace bytes owned by the object (memory class). */
PRISM_API int64_t prism_problem_device_bytes(const prism_problem* p);

/* Thread-local message for the last non-zero return of this thread. */
PRISM_API const char* prism_last_error(void);

/* Build id (the paper records an "evidence build" id). */
PRISM_API const char* prism_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PRISM_H */
