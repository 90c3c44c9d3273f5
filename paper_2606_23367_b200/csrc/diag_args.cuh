// diag_args.cuh - argument block of the external-diagnostics kernel (diag.cuh)
#pragma once
#include <stdint.h>

struct DiagArgs {
  int64_t N, ldw; int32_t A, G;
  const double *w;            // A x N (ld N)
  const double *gS;           // A x ldw : gamma Sigma (w - w_b)
  const double *duals;        // A x NDUAL(G) or NULL
  const double *mu, *w0, *w_b, *gamma, *lo, *hi, *hi_full, *tau, *kappa, *c_buy, *lot_slope, *lot_width, *band_lo, *band_hi;
  const uint8_t *excl, *lot_count, *group_id;
  double* resid;              // A x PRISM_NRES
  double delta;               // activity threshold (1e-9)
  const int32_t* only_done;   // if non-NULL: skip accounts that are not done (solver's final pass uses NULL)
};

