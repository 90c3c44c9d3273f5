// small_args.cuh - argument blocks of the small kernels (small.cuh)
#pragma once
#include "common.cuh"

struct InitArgs {
  int64_t N, ldw; int32_t A, G;
  const double *w0, *gamma;
  const uint8_t* group_id;
  double *v, *gw0, *lamG;
  AccountParams ap;
  double rho_scale;
};

struct SolveArgs {
  int32_t A, kp, nchunk; int64_t ldv;
  const double *Tpart, *Sinv;
  double *V;
  AccountParams ap;
  const int32_t* act; int32_t nact;   // H6: grid = nact, block s solves account act[s] (NULL: identity)
};

// warm start (prism_settings.warm_w / warm_duals): carried state from previous weights and multipliers
struct WarmArgs {
  int64_t N, ldw; int32_t A, G;
  const double *w, *duals;        // A x N; A x NDUAL(G) or NULL
  const double *mu, *gS;          // gS = gamma Sigma (w - w_b)  (A x ldw)
  const double *invd, *gamma, *tau;
  double *v, *lamG;
  AccountParams ap;
};

// constraint-set precheck (k_precheck): necessary conditions for the feasible set of one account to be non-empty
struct PrecheckArgs {
  int64_t N; int32_t A, G, max_lots;
  const double *w0, *lo, *hi, *hi_full, *tau, *band_lo, *band_hi, *lot_width;
  const uint8_t *excl, *lot_count, *group_id;
  double *w_out, *resid, *duals;
  AccountParams ap;
  int32_t* counters;
};
