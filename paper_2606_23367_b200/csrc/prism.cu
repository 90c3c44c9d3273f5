// prism.cu - C ABI (include/prism.h) and the host driver of the batched ADMM.
// The kernels live in the k_*.cu translation units behind the launch wrappers of kernels.h.  No torch types, no CPU
// fallback, no environment variables: everything that steers a solve is in prism_constraint_set / prism_settings.
#include <chrono>
#include <new>
#include <vector>

#include "kernels.h"

#define PRISM_VERSION_STR "prism-b200 r2 (sm_100a; factor GEMMs: 3xTF32 tensor path or fp64 DMMA; fused projection: cluster-resident / streaming pair)"

static const int kMT[] = {2, 4, 7, 8, 13, 16};
static int pick_mt(int k) {
  for (int m : kMT) if (8 * m >= k) return m;
  return -1;
}

extern "C" void prism_default_settings(prism_settings* s) {
  if (!s) return;
  memset(s, 0, sizeof(*s));
  s->eps_rel = 1e-6; s->eps_abs = 0.0; s->max_iter = 4000; s->check_every = 10; s->first_check = 40; s->adapt_rho = 1; s->adapt_start = 200; s->adapt_every = 100; s->sample_until = -1; s->reserved0 = 0;
  s->alpha = 1.6; s->rho_scale = 100.0; s->gemm_precision = PRISM_GEMM_TF32X3; s->profile = 0;
  s->time_limit_ms = 0.0; s->deadline_ms = 0.0; s->prox_window_mult = 32.0; s->warm_w = nullptr; s->warm_duals = nullptr;
}
extern "C" const char* prism_last_error(void) { return g_err; }
int prism_internal_set_error(int code, const char* what, const char* detail) {
  snprintf(g_err, sizeof(g_err), "%s%s%s", what, (detail && detail[0]) ? ": " : "", detail ? detail : "");
  return code;
}
extern "C" const char* prism_version(void) { return PRISM_VERSION_STR; }
extern "C" int64_t prism_problem_device_bytes(const prism_problem* p) { return p ? p->bytes : 0; }
extern "C" int32_t prism_problem_prox_form(const prism_problem* p) {
  return !p ? PRISM_PROX_AUTO : (p->res ? PRISM_PROX_RESIDENT : (p->fast ? PRISM_PROX_STREAMING : PRISM_PROX_EVERY_ASSET));
}

template <typename T>
static int dev_alloc(prism_problem* p, T** ptr, size_t count, bool zero = true) {
  *ptr = nullptr;
  if (count == 0) count = 1;
  cudaError_t e = cudaMalloc((void**)ptr, count * sizeof(T));
  if (e != cudaSuccess) { cudaGetLastError(); return set_err(PRISM_ERR_ALLOC, "cudaMalloc of %s%lld bytes failed", "", (long long)(count * sizeof(T))); }
  if (zero) cudaMemset(*ptr, 0, count * sizeof(T));
  p->bytes += (int64_t)(count * sizeof(T));
  return PRISM_OK;
}
#define ALLOC_TRY(expr) do { int _r = (expr); if (_r != PRISM_OK) { prism_problem_destroy(p); return _r; } } while (0)

extern "C" void prism_problem_destroy(prism_problem* p) {
  if (!p) return;
  void* ptrs[] = {p->Bp, p->Bt, p->Bp_hi, p->Bp_lo, p->Bt_hi, p->Bt_lo, p->Bp32, p->Bt32, p->invd, p->gram, p->q, p->v, p->rt, p->cc, p->xs, p->pxq, p->Tpart, p->V, p->Sinv,
                  p->gw0, p->lamG, p->resid, p->duals, p->status, p->ap.c, p->ap.alpha, p->ap.beta,
                  p->ap.mode, p->ap.bsum, p->ap.done, p->ap.conv, p->ap.iters, p->ap.refactor,
                  p->ap.nadapt, p->ap.win, p->ap.wins, p->ap.slack, p->ap.c_new, p->counters, p->act, p->w_stage, p->i_stage, p->lraw, p->lcomp, p->lcnt, p->cbin, p->chkp, p->lflag};
  for (void* q : ptrs) if (q) cudaFree(q);
  if (p->h_counters) cudaFreeHost(p->h_counters);
  delete p;
}

// ------------------------------------------------------------------------------------------ launch helpers
struct Launcher {
  prism_problem* p;
  cudaStream_t st;
  int mt;
  int gemm_mode;
  int64_t launches = 0;
  bool prof = false;
  cudaError_t err = cudaSuccess;       // first launch error (checked by the caller at its synchronisation points)
  struct Ev { cudaEvent_t a, b; int cls; };
  std::vector<Ev> evs;
  void begin(int cls) {
    if (!prof) return;
    Ev e; e.cls = cls;
    cudaEventCreate(&e.a); cudaEventCreate(&e.b);
    cudaEventRecord(e.a, st);
    evs.push_back(e);
  }
  void end(cudaError_t e, int n = 1) {
    if (prof && !evs.empty()) cudaEventRecord(evs.back().b, st);
    launches += n;
    if (e != cudaSuccess && err == cudaSuccess) err = e;
  }
  // after a stream synchronize: per-class device time and launch counts
  void collect(double* ms, int64_t* cnt) {
    for (int i = 0; i < PRISM_NKERN; ++i) { ms[i] = 0.0; cnt[i] = 0; }
    for (auto& e : evs) {
      float t = 0.f;
      cudaEventElapsedTime(&t, e.a, e.b);
      ms[e.cls] += t; cnt[e.cls] += 1;
      cudaEventDestroy(e.a); cudaEventDestroy(e.b);
    }
    evs.clear();
  }
  // act / nact: the compacted list of active accounts (H6); NULL / A = every account
  void gemm1(const double* X, const int32_t* act, int nact) {
    Gemm1Args a;
    a.Bt = p->Bt; a.ldn = p->ldn; a.X = X; a.ldw = p->ldn; a.Tpart = p->Tpart; a.ldv = p->ldv; a.A = p->A;
    a.chunk = p->chunk; a.Npad = p->ldn; a.act = act; a.nact = nact;
    begin(PRISM_K_GEMM1);
    end(gemm1_launch(gemm_mode, mt, p->nchunk, p->kp, a, tf(), st));
  }
  TfSplit tf() const { return TfSplit{p->Bt_hi, p->Bt_lo, p->Bp_hi, p->Bp_lo, p->Bp32, p->Bt32, p->sm_count}; }
  void gemm2(int mode, const Gemm2Args& a) {
    begin(PRISM_K_GEMM2);
    end(gemm2_launch(gemm_mode, mt, mode, a, tf(), st));
  }
  Gemm2Args g2base() const {
    Gemm2Args a;
    memset(&a, 0, sizeof(a));
    a.Bp = p->Bp; a.kp = p->kp; a.V = p->V; a.ldv = p->ldv; a.N = p->N; a.ldw = p->ldn; a.A = p->A; a.G = 0;     // no consensus rows in the x-update: U = Bp
    a.group_id = nullptr; a.invd = p->invd; a.d = p->d.d; a.gamma = p->d.gamma; a.c = p->ap.c;
    a.v = p->v; a.cc = p->cc; a.rt = p->rt; a.xs = p->xs; a.pxq = p->pxq; a.q = p->q; a.mu = p->d.mu;
    a.relax = 1.0; a.act = nullptr; a.nact = p->A;
    return a;
  }
  // pxq <- gamma Sigma X   (H8: Sigma W = B (F (B'W)) + D o W, fp64)
  void sigma_apply(const double* X) {
    gemm1(X, nullptr, p->A);
    begin(PRISM_K_OTHER);
    end(scale_fs_launch(p->Tpart, p->nchunk, p->A, p->k, p->kp, p->ldv, p->d.f, p->d.gamma, p->V, st));
    Gemm2Args a = g2base();
    a.X = X;
    gemm2(G2_SIGMA, a);
  }
  // q <- -mu - gamma Sigma w_b (benchmark shift); uses rt and pxq as scratch and leaves rt zero
  void build_q() {
    begin(PRISM_K_OTHER);
    end(diff_launch(p->d.w_b, nullptr, p->N, p->ldn, p->A, p->rt, st));
    sigma_apply(p->rt);
    begin(PRISM_K_OTHER);
    end(make_q_launch(p->d.mu, p->pxq, p->N, p->ldn, p->A, p->q, st));
    cudaMemsetAsync(p->rt, 0, (size_t)p->A * p->ldn * sizeof(double), st);
  }
};

// which form of the projection kernel applies (prism.h: PRISM_PROX_*)
static bool stream_applicable(const prism_problem* p) {
  // N % 16: every row of every streamed array is 16-byte aligned (bulk copies)
  return !p->d.lot_count && !p->d.hi_full && p->N < ((int64_t)1 << prox_stream_idx_bits()) && p->N % 16 == 0;
}

// ------------------------------------------------------------------------------------------ create (H0)
extern "C" int prism_problem_create(int64_t N, int32_t k, int32_t accounts, const prism_constraint_set* cs,
                                    const prism_data* data, void* cuda_stream, prism_problem** out) {
  if (out) *out = nullptr;
  if (!out || !cs || !data) return set_err(PRISM_ERR_INVALID_ARG, "null argument%s", "");
  const int A = accounts, G = (cs->flags & PRISM_GROUP_BANDS) ? cs->G : 0;
  if (N < 1 || k < 1 || A < 1) return set_err(PRISM_ERR_INVALID_ARG, "N, k, accounts must be >= 1%s", "");
  if (!(cs->flags & PRISM_BUDGET) || !(cs->flags & PRISM_BOX)) return set_err(PRISM_ERR_INVALID_ARG, "PRISM_BUDGET and PRISM_BOX are mandatory%s", "");
  const int mt = pick_mt(k);
  if (mt < 0 || k > PRISM_MAX_FACTORS) return set_err(PRISM_ERR_INVALID_ARG, "k = %s%lld exceeds PRISM_MAX_FACTORS (128)", "", k);
  if (G < 0 || G > PRISM_MAX_GROUPS || 8 * mt > PRISM_MAX_KPRIME) return set_err(PRISM_ERR_INVALID_ARG, "G = %s%lld out of range", "", G);
  if ((cs->flags & PRISM_GROUP_BANDS) && (G < 1 || !data->group_id || !data->band_lo || !data->band_hi)) return set_err(PRISM_ERR_INVALID_ARG, "group bands need G >= 1, group_id, band_lo, band_hi%s", "");
  if ((cs->flags & PRISM_TAX_LOTS) && (!data->lot_slope || !data->lot_width || !data->lot_count || cs->max_lots < 1 || cs->max_lots > PRISM_MAX_LOTS)) return set_err(PRISM_ERR_INVALID_ARG, "tax lots need lot arrays and 1 <= max_lots <= 4%s", "");
  if (!data->B || !data->f || !data->d || !data->mu || !data->gamma || !data->w0 || !data->lo || !data->hi) return set_err(PRISM_ERR_INVALID_ARG, "missing mandatory data pointer%s", "");
  if (data->d_t) return set_err(PRISM_ERR_INVALID_ARG, "d_t must be NULL: the turnover scaling D_a is the identity in this build%s", "");
  if ((cs->flags & PRISM_BENCHMARK_SHIFT) && !data->w_b) return set_err(PRISM_ERR_INVALID_ARG, "PRISM_BENCHMARK_SHIFT needs w_b%s", "");
  if (cs->prox_form < PRISM_PROX_AUTO || cs->prox_form > PRISM_PROX_EVERY_ASSET) return set_err(PRISM_ERR_INVALID_ARG, "prox_form = %s%lld is not a PRISM_PROX_* value", "", cs->prox_form);

  prism_problem* p = new (std::nothrow) prism_problem();
  if (!p) return set_err(PRISM_ERR_ALLOC, "host allocation failed%s", "");
  memset(p, 0, sizeof(*p));
  p->N = N; p->k = k; p->kp = 8 * mt; p->A = A; p->G = G; p->Kp = p->kp; p->ldv = (p->Kp + 7) / 8 * 8;
  p->flags = cs->flags; p->max_lots = (cs->flags & PRISM_TAX_LOTS) ? cs->max_lots : 0;
  p->d = *data;
  if (!(cs->flags & PRISM_TAX_LOTS)) { p->d.lot_slope = p->d.lot_width = nullptr; p->d.lot_count = nullptr; }
  if (!(cs->flags & PRISM_GROUP_BANDS)) { p->d.group_id = nullptr; p->d.band_lo = p->d.band_hi = nullptr; }
  if (!(cs->flags & PRISM_EXCLUSION)) p->d.excl = nullptr;
  if (!(cs->flags & PRISM_TURNOVER_CAP)) p->d.tau = nullptr;
  if (!(cs->flags & PRISM_TURNOVER_PENALTY)) p->d.kappa = nullptr;
  if (!(cs->flags & PRISM_BUY_COST)) p->d.c_buy = nullptr;
  if (!(cs->flags & PRISM_BENCHMARK_SHIFT)) p->d.w_b = nullptr;
  p->ldn = (N + 31) / 32 * 32;
  int dev = 0;
  cudaGetDevice(&dev);
  cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, dev);
  if (p->sm_count <= 0) { delete p; return set_err(PRISM_ERR_CUDA, "no CUDA device%s", ""); }
  // form of the projection kernel
  {
    int C = 0, SL = 0; size_t sm = 0;
    const bool res_ok = prox_res_geometry(N, G, &C, &SL, &sm);
    const bool str_ok = stream_applicable(p);
    int form = cs->prox_form;
    // AUTO, by measurement on one B200 (kernel table): where both fast forms apply the streaming pair wins once
    // an account needs more than one CTA of the resident form (configs[2]: 65 ms against 78 ms per batch: its streaming
    // pass runs at three CTAs per SM with no wave quantisation), the resident form wins on accounts that fit one CTA
    // (configs[1]: 11.6 against 12.6 ms) and is the only fast form for tax lots, per-asset caps and N % 16 != 0.
    if (form == PRISM_PROX_AUTO) {
      if (res_ok && (C == 1 || !str_ok)) form = PRISM_PROX_RESIDENT;
      else form = str_ok ? PRISM_PROX_STREAMING : (res_ok ? PRISM_PROX_RESIDENT : PRISM_PROX_EVERY_ASSET);
    }
    if ((form == PRISM_PROX_RESIDENT && !res_ok) || (form == PRISM_PROX_STREAMING && !str_ok)) {
      delete p;
      return set_err(PRISM_ERR_INVALID_ARG, "prox_form %s%lld does not apply to this problem (see prism.h)", "", form);
    }
    p->res = form == PRISM_PROX_RESIDENT; p->fast = form == PRISM_PROX_STREAMING;
    if (p->res) { p->res_C = C; p->res_SL = SL; p->res_smem = sm; }
  }
  // split-K chunking of GEMM-1: about two waves of CTAs; three CTAs per SM in one wave for the few-account kernel
  // (gemm_skinny.cuh: 128 threads, no shared memory - its bytes in flight grow with the resident warps)
  const int tilesA = (A + G1_TA - 1) / G1_TA;
  int64_t want = ((A <= 32 ? 3 : 2) * p->sm_count + tilesA - 1) / tilesA;
  const int64_t nst = p->ldn / G1_KS;
  if (want > nst) want = nst;
  if (want < 1) want = 1;
  p->chunk = ((nst + want - 1) / want) * G1_KS;
  p->nchunk = (int)((p->ldn + p->chunk - 1) / p->chunk);
  cudaStream_t st = (cudaStream_t)cuda_stream;

  const size_t AN = (size_t)A * p->ldn;
  ALLOC_TRY(dev_alloc(p, &p->Bp, (size_t)N * p->kp));
  ALLOC_TRY(dev_alloc(p, &p->Bt, (size_t)p->kp * p->ldn));
  ALLOC_TRY(dev_alloc(p, &p->Bp_hi, (size_t)N * p->kp));
  ALLOC_TRY(dev_alloc(p, &p->Bp_lo, (size_t)N * p->kp));
  ALLOC_TRY(dev_alloc(p, &p->Bp32, (size_t)N * p->kp));
  ALLOC_TRY(dev_alloc(p, &p->Bt32, (size_t)p->kp * p->ldn));
  ALLOC_TRY(dev_alloc(p, &p->Bt_hi, (size_t)p->kp * p->ldn));
  ALLOC_TRY(dev_alloc(p, &p->Bt_lo, (size_t)p->kp * p->ldn));
  ALLOC_TRY(dev_alloc(p, &p->invd, (size_t)p->ldn));       // padded with zeros (pair-wise GEMM-2 epilogue)
  ALLOC_TRY(dev_alloc(p, &p->gram, (size_t)p->Kp * p->Kp));
  ALLOC_TRY(dev_alloc(p, &p->v, AN));
  ALLOC_TRY(dev_alloc(p, &p->rt, AN));
  ALLOC_TRY(dev_alloc(p, &p->cc, AN));
  ALLOC_TRY(dev_alloc(p, &p->xs, AN));
  ALLOC_TRY(dev_alloc(p, &p->pxq, AN));
  ALLOC_TRY(dev_alloc(p, &p->Tpart, (size_t)p->nchunk * A * p->ldv));
  ALLOC_TRY(dev_alloc(p, &p->V, (size_t)A * p->ldv));
  ALLOC_TRY(dev_alloc(p, &p->Sinv, (size_t)A * p->Kp * p->Kp));
  ALLOC_TRY(dev_alloc(p, &p->gw0, (size_t)A * (G ? G : 1)));
  ALLOC_TRY(dev_alloc(p, &p->lamG, (size_t)A * (G ? G : 1)));
  ALLOC_TRY(dev_alloc(p, &p->resid, (size_t)A * PRISM_NRES));
  ALLOC_TRY(dev_alloc(p, &p->duals, (size_t)A * PRISM_NDUAL(G)));
  ALLOC_TRY(dev_alloc(p, &p->status, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.c, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.alpha, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.beta, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.mode, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.bsum, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.done, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.conv, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.iters, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.refactor, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.nadapt, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.win, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.wins, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.slack, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->ap.c_new, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->counters, (size_t)4));
  ALLOC_TRY(dev_alloc(p, &p->act, (size_t)A));
  ALLOC_TRY(dev_alloc(p, &p->w_stage, (size_t)A * N));      // staging of the host-buffer lane (prism_solve_batch_host)
  ALLOC_TRY(dev_alloc(p, &p->i_stage, (size_t)A));
  cudaError_t ke = cudaSuccess;
  if (p->res) ke = prox_res_set_attrs(p->d.lot_count != nullptr, p->res_C, p->res_smem);
  if (p->fast) {
    // slices: a few CTAs per resident slot so that the streaming kernel stays bandwidth-bound to the end of the grid
    const int CH = prox_stream_chunk(), NW = prox_stream_warps();
    int64_t target = ((int64_t)4 * 3 * p->sm_count + A - 1) / A;           // CTAs per account wanted
    int64_t sl = (N + target - 1) / target;
    sl = (sl + CH - 1) / CH * CH;
    if (sl < 2 * CH) sl = 2 * CH;
    p->slice_len = sl;
    p->S = (int)((N + sl - 1) / sl);
    p->capw = (int)(sl / NW);
    p->ldc = (int64_t)p->S * sl;
    const int Gb = G > 0 ? G : 1;
    const size_t ent = prox_stream_entry_bytes();
    ALLOC_TRY(dev_alloc(p, (unsigned char**)&p->lraw, (size_t)A * p->ldc * ent, false));
    ALLOC_TRY(dev_alloc(p, (unsigned char**)&p->lcomp, (size_t)A * p->ldc * ent, false));
    ALLOC_TRY(dev_alloc(p, &p->lcnt, (size_t)2 * A * p->S * NW));          // fronts, then backs of the two-level lists
    ALLOC_TRY(dev_alloc(p, &p->cbin, (size_t)2 * A * 2 * Gb));             // bins of the dead assets, then speculative bins
    ALLOC_TRY(dev_alloc(p, &p->chkp, (size_t)A * p->S * 8));
    ALLOC_TRY(dev_alloc(p, &p->lflag, (size_t)A));
    if (ke == cudaSuccess) ke = prox_stream_set_attrs(G, 2 * p->S * NW);
  }
  if (cudaMallocHost((void**)&p->h_counters, 4 * sizeof(int32_t)) != cudaSuccess) { prism_problem_destroy(p); return set_err(PRISM_ERR_ALLOC, "pinned allocation failed%s", ""); }
  if (p->d.w_b) ALLOC_TRY(dev_alloc(p, &p->q, AN));
  if (ke == cudaSuccess) ke = gemm_set_attrs(mt);
  if (ke == cudaSuccess) ke = small_set_attrs(p->Kp);
  if (ke == cudaSuccess && !p->res && !p->fast) ke = prox_generic_set_attrs();
  if (ke != cudaSuccess) { prism_problem_destroy(p); return set_err(PRISM_ERR_CUDA, "kernel attributes: %s", cudaGetErrorString(ke)); }

  Launcher L{p, st, mt, 0};
  L.end(setup_shared_launch(data->B, data->B_is_fp32, data->d, N, k, p->kp, p->ldn, p->Bp, p->Bt, p->invd, st));
  L.end(gram_launch(p->Bt, p->ldn, p->invd, N, p->kp, p->gram, st));
  L.end(split_universe_launch(p->Bp, p->Bt, N, p->kp, p->ldn, p->Bp_hi, p->Bp_lo, p->Bt_hi, p->Bt_lo, p->Bp32, p->Bt32, st));
  if (p->d.w_b) L.build_q();            // q = -mu - gamma Sigma w_b
  cudaError_t e = cudaStreamSynchronize(st);
  if (e == cudaSuccess) e = L.err;
  if (e == cudaSuccess) e = cudaGetLastError();
  if (e != cudaSuccess) { prism_problem_destroy(p); return set_err(PRISM_ERR_CUDA, "setup kernels failed: %s", cudaGetErrorString(e)); }
  *out = p;
  return PRISM_OK;
}

// ------------------------------------------------------------------------------------------ solve (H1-H9)
static ProxArgs make_prox_args(prism_problem* p, const prism_settings& s, double* w_out) {
  ProxArgs a;
  memset(&a, 0, sizeof(a));
  a.N = p->N; a.A = p->A; a.G = p->G; a.kp = p->kp; a.max_lots = p->max_lots; a.ldv = p->ldv;
  a.mu = p->d.mu; a.q = p->q; a.w0 = p->d.w0; a.gamma = p->d.gamma; a.lo = p->d.lo; a.hi = p->d.hi; a.hi_full = p->d.hi_full;
  a.tau = p->d.tau; a.kappa = p->d.kappa; a.c_buy = p->d.c_buy; a.lot_slope = p->d.lot_slope; a.lot_width = p->d.lot_width;
  a.excl = p->d.excl; a.lot_count = p->d.lot_count; a.group_id = p->d.group_id; a.invd = p->invd; a.d = p->d.d;
  a.v = p->v; a.rt = p->rt; a.cc = p->cc; a.xs = p->xs; a.pxq = p->pxq; a.band_lo = p->d.band_lo; a.band_hi = p->d.band_hi;
  a.lamG = p->lamG; a.gw0 = p->gw0;
  a.ap = p->ap; a.w_out = w_out; a.duals = p->duals; a.resid = p->resid; a.counters = p->counters;
  a.eps = s.eps_rel; a.eps_abs = s.eps_abs;
  a.adapt = s.adapt_rho; a.iter = 0; a.ldw = p->ldn;
  // -1 = by measurement: 6 launches; 12 for universes beyond the cluster-resident form's reach, where
  // a pass over a full list costs the root kernel's one CTA per account milliseconds (configs[4]: 22 ms per launch)
  const int sample_auto = (p->fast && p->N >= 65536) ? 12 : 6;
  a.sample_until = s.warm_w ? 0 : (s.sample_until < 0 ? sample_auto : s.sample_until);   // a warm start has its bands in from the first launch
  a.adapt_start = s.adapt_start; a.adapt_every = s.adapt_every < 1 ? 1 : s.adapt_every;
  a.lraw = p->lraw; a.lcomp = p->lcomp; a.lcnt = p->lcnt; a.cbin = p->cbin; a.chkp = p->chkp; a.lflag = p->lflag;
  a.S = p->S; a.capw = p->capw; a.slice_len = p->slice_len; a.ldc = p->ldc;
  a.res_C = p->res_C; a.res_SL = p->res_SL;
  a.win_mult = s.prox_window_mult > 0 ? s.prox_window_mult : 32.0;
  a.band_start = 20;       // band ramp (readings): non-check launches of iterations 0-20 project without the bands
  a.band_wide = 1;
  a.band_ramp = 0;
  a.win_ratio = 16.0;
  return a;
}

static void launch_prox(Launcher& L, ProxArgs& a, int mode, int iter) {
  prism_problem* p = L.p;
  a.iter = iter;
  const bool chk = (mode & (PROX_CHECK | PROX_FINAL)) != 0;       // the final extraction also needs w_out
  L.begin(PRISM_K_PROX);
  if (p->res) L.end(prox_res_launch(p->d.lot_count != nullptr, chk, p->res_C, p->A, p->res_smem, a, mode & ~PROX_CHECK, L.st));
  else if (p->fast) {
    L.end(prox_stream_launch(chk, p->S, p->A, p->G, a, mode, L.st), 2);
    // a check may have decided a rho change for some accounts: their iterate is rewritten for the new rho by a streaming
    // pass of its own (exits at once for every other account)
    if ((mode & PROX_CHECK) && a.adapt) L.end(prox_rescale_launch(p->A, a, L.st));
  }
  else {
    const int grid = p->A < p->sm_count ? p->A : p->sm_count;
    const size_t sm = (size_t)p->N * 20 + 16;
    const bool smem_form = !p->d.lot_count && !p->d.hi_full && sm <= prox_generic_smem_max();
    L.end(prox_generic_launch(grid, p->d.lot_count != nullptr, smem_form, sm, a, mode, L.st));
  }
}

static DiagArgs make_diag_args(prism_problem* p, const double* w, const double* duals, double* resid) {
  DiagArgs a;
  memset(&a, 0, sizeof(a));
  a.N = p->N; a.ldw = p->ldn; a.A = p->A; a.G = p->G; a.w = w; a.gS = p->pxq; a.duals = duals;
  a.mu = p->d.mu; a.w0 = p->d.w0; a.w_b = p->d.w_b; a.gamma = p->d.gamma; a.lo = p->d.lo; a.hi = p->d.hi; a.hi_full = p->d.hi_full;
  a.tau = p->d.tau; a.kappa = p->d.kappa; a.c_buy = p->d.c_buy; a.lot_slope = p->d.lot_slope; a.lot_width = p->d.lot_width;
  a.band_lo = p->d.band_lo; a.band_hi = p->d.band_hi; a.excl = p->d.excl; a.lot_count = p->d.lot_count; a.group_id = p->d.group_id;
  a.resid = resid; a.delta = 1e-9; a.only_done = nullptr;
  return a;
}

// resid (device, A x NRES) <- diagnostics of w; uses rt and pxq as scratch
static void run_diag(prism_problem* p, Launcher& L, const double* w, const double* duals, double* resid) {
  L.begin(PRISM_K_OTHER);
  L.end(diff_launch(w, p->d.w_b, p->N, p->ldn, p->A, p->rt, L.st));
  L.sigma_apply(p->rt);
  DiagArgs da = make_diag_args(p, w, duals, resid);
  L.begin(PRISM_K_DIAG);
  L.end(diag_launch(da, p->d.lot_count != nullptr, L.st));
}

extern "C" int prism_solve_batch(prism_problem* p, const prism_settings* sp, void* cuda_stream, double* w_out,
                                 int32_t* status_out, int32_t* iters_out, double* resid_out, double* duals_out,
                                 prism_solve_info* info) {
  if (!p) return set_err(PRISM_ERR_NOT_READY, "problem object is NULL%s", "");
  if (!w_out || !status_out || !iters_out) return set_err(PRISM_ERR_INVALID_ARG, "w_out, status_out, iters_out are mandatory%s", "");
  prism_settings s;
  if (sp) s = *sp; else prism_default_settings(&s);
  if (!(s.eps_rel > 0) || !(s.eps_abs >= 0) || s.max_iter < 1 || s.check_every < 1 || !(s.alpha > 0 && s.alpha < 2) || !(s.rho_scale > 0) ||
      (s.gemm_precision < PRISM_GEMM_FP64_TENSOR || s.gemm_precision > PRISM_GEMM_TF32X3))
    return set_err(PRISM_ERR_INVALID_ARG, "invalid settings%s", "");
  if (s.warm_duals && !s.warm_w) return set_err(PRISM_ERR_INVALID_ARG, "warm_duals needs warm_w%s", "");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const auto t0 = std::chrono::steady_clock::now();
  auto elapsed_ms = [&]() { return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count(); };
  cudaEvent_t ev0, ev1;
  CUDA_TRY(cudaEventCreate(&ev0));
  CUDA_TRY(cudaEventCreate(&ev1));
  CUDA_TRY(cudaEventRecord(ev0, st));
  const int A = p->A, G = p->G;
  Launcher L{p, st, p->kp / 8, s.gemm_precision};
  L.prof = s.profile != 0;

  CUDA_TRY(cudaMemsetAsync(p->counters, 0, 4 * sizeof(int32_t), st));
  CUDA_TRY(cudaMemsetAsync(p->resid, 0, (size_t)A * PRISM_NRES * sizeof(double), st));
  InitArgs ia;
  memset(&ia, 0, sizeof(ia));
  ia.N = p->N; ia.ldw = p->ldn; ia.A = A; ia.G = G; ia.w0 = p->d.w0; ia.gamma = p->d.gamma;
  ia.group_id = p->d.group_id; ia.v = p->v; ia.gw0 = p->gw0; ia.lamG = p->lamG; ia.ap = p->ap; ia.rho_scale = s.rho_scale;
  L.begin(PRISM_K_OTHER);
  L.end(init_accounts_launch(ia, st));
  {
    PrecheckArgs pc;
    memset(&pc, 0, sizeof(pc));
    pc.N = p->N; pc.A = A; pc.G = G; pc.max_lots = p->max_lots; pc.w0 = p->d.w0; pc.lo = p->d.lo; pc.hi = p->d.hi; pc.hi_full = p->d.hi_full;
    pc.tau = p->d.tau; pc.band_lo = p->d.band_lo; pc.band_hi = p->d.band_hi; pc.lot_width = p->d.lot_width; pc.excl = p->d.excl;
    pc.lot_count = p->d.lot_count; pc.group_id = p->d.group_id; pc.w_out = w_out; pc.resid = p->resid; pc.duals = p->duals; pc.ap = p->ap;
    pc.counters = p->counters;
    L.begin(PRISM_K_OTHER);
    L.end(precheck_launch(pc, st));
  }
  if (s.warm_w) {
    // warm start from previous weights w and multipliers: at a fixed point of the splitting x = z = w and the dual is
    // y = -(P w + q) = mu - gamma Sigma (w - w_b), so the carried state is v = w + y / rho; thresholds from the duals
    L.begin(PRISM_K_OTHER);
    L.end(diff_launch(s.warm_w, p->d.w_b, p->N, p->ldn, A, p->rt, st));
    L.sigma_apply(p->rt);
    WarmArgs wa;
    memset(&wa, 0, sizeof(wa));
    wa.N = p->N; wa.ldw = p->ldn; wa.A = A; wa.G = G; wa.w = s.warm_w; wa.duals = s.warm_duals; wa.mu = p->d.mu; wa.gS = p->pxq;
    wa.invd = p->invd; wa.gamma = p->d.gamma; wa.tau = p->d.tau; wa.v = p->v; wa.lamG = p->lamG; wa.ap = p->ap;
    L.begin(PRISM_K_OTHER);
    L.end(warm_start_launch(wa, st));
  }
  CUDA_TRY(cudaMemsetAsync(p->rt, 0, (size_t)A * p->ldn * sizeof(double), st));

  ProxArgs pa = make_prox_args(p, s, w_out);
  if (s.warm_w) pa.band_start = -1;      // a warm start carries band multipliers: no band ramp
  SolveArgs sa;
  memset(&sa, 0, sizeof(sa));
  sa.A = A; sa.kp = p->kp; sa.nchunk = p->nchunk; sa.ldv = p->ldv; sa.Tpart = p->Tpart; sa.Sinv = p->Sinv;
  sa.V = p->V; sa.ap = p->ap; sa.act = nullptr; sa.nact = A;
  Gemm2Args g2 = L.g2base();
  g2.relax = s.alpha;
  // H6: the GEMMs and the small solve run over the compacted list of accounts still active (identity until the first
  // account finishes); the list is rebuilt after every check that finished accounts
  const int32_t* act = nullptr;
  int nact = A;

  int it = 1, timed_out = 0, late_iter = -1, ndone = 0;
  for (; it <= s.max_iter; ++it) {
    const bool check = (it > 1) && ((it - 1) % s.check_every == 0) && (it - 1 >= s.first_check);   // residuals of the iterate after it-1 iterations
    launch_prox(L, pa, check ? PROX_CHECK : 0, it - 1);
    if (check || it == 1) {
      L.begin(PRISM_K_FACTOR);
      L.end(factor_launch(p->gram, p->d.f, p->d.gamma, p->ap, A, p->k, p->kp, p->Sinv, st));
    }
    if (check) {
      CUDA_TRY(cudaMemcpyAsync(p->h_counters, p->counters, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
      CUDA_TRY(cudaStreamSynchronize(st));
      if (L.err != cudaSuccess) break;
      const double el = elapsed_ms();
      // accounts that converge at this very check are late if the deadline has already passed
      if (s.deadline_ms > 0 && late_iter < 0 && el > s.deadline_ms) late_iter = it - 2;
      const int ndone_prev = ndone;
      ndone = p->h_counters[0];
      if (ndone >= A) break;
      if (ndone != ndone_prev) {
        L.begin(PRISM_K_OTHER);
        L.end(compact_launch(A, p->ap.done, p->act, st));
        act = p->act; nact = A - ndone;
        sa.act = act; sa.nact = nact; g2.act = act; g2.nact = nact;
      }
      if (s.time_limit_ms > 0 && el > s.time_limit_ms) { timed_out = 1; break; }
    }
    L.gemm1(p->rt, act, nact);
    L.begin(PRISM_K_SOLVE);
    L.end(solve_launch(sa, st));
    const bool next_check = (it % s.check_every == 0) && (it >= s.first_check);
    L.gemm2(next_check ? G2_ADMM_CHECK : G2_ADMM, g2);
    if (it == 1 && L.err != cudaSuccess) break;                 // a launch configuration error shows in the first iteration
  }
  if (L.err != cudaSuccess) {
    cudaStreamSynchronize(st);
    if (L.prof) L.collect(p->prof_ms, p->prof_cnt);
    cudaEventDestroy(ev0); cudaEventDestroy(ev1);
    return set_err(PRISM_ERR_CUDA, "kernel launch failed: %s", cudaGetErrorString(L.err));
  }
  if (ndone < A) {           // iteration cap or time limit: extract z for the accounts still running
    launch_prox(L, pa, PROX_FINAL, it > s.max_iter ? s.max_iter : it - 1);
  }
  // H8 / H9: external diagnostics of the returned weights with the solver's multipliers, then statuses
  // the external diagnostics are always fp64
  if (L.gemm_mode == PRISM_GEMM_FP32_EXPERIMENT) L.gemm_mode = PRISM_GEMM_FP64_FMA;
  if (L.gemm_mode == PRISM_GEMM_TF32X3) L.gemm_mode = PRISM_GEMM_FP64_TENSOR;
  run_diag(p, L, w_out, p->duals, p->resid);
  L.begin(PRISM_K_OTHER);
  L.end(status_launch(A, p->resid, p->ap.conv, p->ap.iters, timed_out, late_iter, 1e-6, p->status, st));
  if (status_out != p->status) CUDA_TRY(cudaMemcpyAsync(status_out, p->status, (size_t)A * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
  CUDA_TRY(cudaMemcpyAsync(iters_out, p->ap.iters, (size_t)A * sizeof(int32_t), cudaMemcpyDeviceToDevice, st));
  if (resid_out) CUDA_TRY(cudaMemcpyAsync(resid_out, p->resid, (size_t)A * PRISM_NRES * sizeof(double), cudaMemcpyDeviceToDevice, st));
  if (duals_out) CUDA_TRY(cudaMemcpyAsync(duals_out, p->duals, (size_t)A * PRISM_NDUAL(G) * sizeof(double), cudaMemcpyDeviceToDevice, st));
  CUDA_TRY(cudaEventRecord(ev1, st));
  std::vector<int32_t> hs((size_t)A), hi((size_t)A);
  CUDA_TRY(cudaMemcpyAsync(hs.data(), p->status, (size_t)A * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaMemcpyAsync(hi.data(), p->ap.iters, (size_t)A * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  CUDA_TRY(cudaGetLastError());
  if (L.err != cudaSuccess) return set_err(PRISM_ERR_CUDA, "kernel launch failed: %s", cudaGetErrorString(L.err));
  if (L.prof) L.collect(p->prof_ms, p->prof_cnt);
  if (info) {
    memset(info, 0, sizeof(*info));
    float ms = 0.f;
    cudaEventElapsedTime(&ms, ev0, ev1);
    info->solve_interval_ms = ms;
    info->device_bytes = p->bytes;
    for (int a = 0; a < A; ++a) {
      info->iters_total += hi[(size_t)a];
      if (hi[(size_t)a] > info->iters_max) info->iters_max = hi[(size_t)a];
      switch (hs[(size_t)a]) {
        case PRISM_STATUS_CERTIFIED: ++info->n_certified; break;
        case PRISM_STATUS_FEASIBLE: ++info->n_feasible; break;
        case PRISM_STATUS_TIMEOUT: ++info->n_timeout; break;
        case PRISM_STATUS_LATE: ++info->n_late; break;
        case PRISM_STATUS_NO_FEASIBLE: ++info->n_no_feasible; break;
        default: ++info->n_failed; break;
      }
    }
    info->kernel_launches = L.launches;
    info->wall_ms = elapsed_ms();
  }
  cudaEventDestroy(ev0);
  cudaEventDestroy(ev1);
  return PRISM_OK;
}

// One exact application of the projection kernel to caller-given points (prism.h): cold account state with
// rho = rho_scale gamma d, v copied into the padded iterate, one PROX_FINAL launch (exact thresholds, z -> z_out).
extern "C" int prism_project(prism_problem* p, const double* v, double rho_scale, void* cuda_stream, double* z_out,
                             double* duals_out) {
  if (!p) return set_err(PRISM_ERR_NOT_READY, "problem object is NULL%s", "");
  if (!v || !z_out || !(rho_scale > 0)) return set_err(PRISM_ERR_INVALID_ARG, "v, z_out and rho_scale > 0 are mandatory%s", "");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int A = p->A, G = p->G;
  Launcher L{p, st, p->kp / 8, 0};
  CUDA_TRY(cudaMemsetAsync(p->counters, 0, 4 * sizeof(int32_t), st));
  InitArgs ia;
  memset(&ia, 0, sizeof(ia));
  ia.N = p->N; ia.ldw = p->ldn; ia.A = A; ia.G = G; ia.w0 = p->d.w0; ia.gamma = p->d.gamma;
  ia.group_id = p->d.group_id; ia.v = p->v; ia.gw0 = p->gw0; ia.lamG = p->lamG; ia.ap = p->ap; ia.rho_scale = rho_scale;
  L.end(init_accounts_launch(ia, st));
  L.end(diff_launch(v, nullptr, p->N, p->ldn, A, p->v, st));
  prism_settings s;
  prism_default_settings(&s);
  ProxArgs pa = make_prox_args(p, s, z_out);
  pa.band_start = -1;                       // no band ramp: the full projection
  launch_prox(L, pa, PROX_FINAL, 0);
  if (duals_out) CUDA_TRY(cudaMemcpyAsync(duals_out, p->duals, (size_t)A * PRISM_NDUAL(G) * sizeof(double), cudaMemcpyDeviceToDevice, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  CUDA_TRY(cudaGetLastError());
  if (L.err != cudaSuccess) return set_err(PRISM_ERR_CUDA, "kernel launch failed: %s", cudaGetErrorString(L.err));
  return PRISM_OK;
}

// T_out[a][j] = sum_i B[i][j] w[a][i]: the problem's own GEMM-1 (H1) on caller-given vectors, split-K partials in the
// workspace allocated at create, reduced in chunk order.  Uses rt as the padded copy of w.
extern "C" int prism_factor_exposures(prism_problem* p, const double* w, void* cuda_stream, double* T_out) {
  if (!p) return set_err(PRISM_ERR_NOT_READY, "problem object is NULL%s", "");
  if (!w || !T_out) return set_err(PRISM_ERR_INVALID_ARG, "w and T_out are mandatory%s", "");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  Launcher L{p, st, p->kp / 8, 0};
  L.end(diff_launch(w, nullptr, p->N, p->ldn, p->A, p->rt, st));
  L.gemm1(p->rt, nullptr, p->A);
  L.end(reduce_partials_launch(p->Tpart, p->nchunk, p->A, p->k, p->ldv, T_out, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if (L.err != cudaSuccess) return set_err(PRISM_ERR_CUDA, "kernel launch failed: %s", cudaGetErrorString(L.err));
  return PRISM_OK;
}

// Measured fp64 rates of this device (register-resident loops, no memory traffic): tflops_out[0] = tensor pipe (DMMA
// mma.sync m8n8k4), tflops_out[1] = FMA pipe.  Uses the problem's counter block as the (never written) sink.
extern "C" int prism_fp64_yardstick(prism_problem* p, void* cuda_stream, double* tflops_out) {
  if (!p || !tflops_out) return set_err(PRISM_ERR_INVALID_ARG, "null argument%s", "");
  const cudaError_t e = fp64_yardstick((cudaStream_t)cuda_stream, p->resid, p->sm_count, tflops_out);
  if (e != cudaSuccess) return set_err(PRISM_ERR_CUDA, "yardstick failed: %s", cudaGetErrorString(e));
  return PRISM_OK;
}

extern "C" int prism_kernel_times(const prism_problem* p, double* ms_out, int64_t* launches_out) {
  if (!p || !ms_out || !launches_out) return set_err(PRISM_ERR_INVALID_ARG, "null argument%s", "");
  for (int i = 0; i < PRISM_NKERN; ++i) { ms_out[i] = p->prof_ms[i]; launches_out[i] = p->prof_cnt[i]; }
  return PRISM_OK;
}

extern "C" int prism_residuals(prism_problem* p, const double* w, const double* duals, void* cuda_stream, double* resid_out) {
  if (!p) return set_err(PRISM_ERR_NOT_READY, "problem object is NULL%s", "");
  if (!w || !resid_out) return set_err(PRISM_ERR_INVALID_ARG, "w and resid_out are mandatory%s", "");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  Launcher L{p, st, p->kp / 8, 0};
  run_diag(p, L, w, duals, resid_out);
  L.end(nan_cols_launch(p->A, resid_out, st));         // the solver-only columns are NaN here
  CUDA_TRY(cudaStreamSynchronize(st));
  CUDA_TRY(cudaGetLastError());
  if (L.err != cudaSuccess) return set_err(PRISM_ERR_CUDA, "kernel launch failed: %s", cudaGetErrorString(L.err));
  return PRISM_OK;
}

extern "C" int prism_solve_batch_host(prism_problem* p, const prism_settings* s, void* cuda_stream, const double* mu_host,
                                      const double* w0_host, double* w_host, int32_t* status_host, int32_t* iters_host,
                                      double* resid_host, prism_solve_info* info) {
  if (!p) return set_err(PRISM_ERR_NOT_READY, "problem object is NULL%s", "");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const auto t0 = std::chrono::steady_clock::now();
  const size_t AN = (size_t)p->A * p->N;
  // the caller lends the device arrays mu and w0 to the problem object for its lifetime (prism.h): this lane refreshes them
  if (mu_host) CUDA_TRY(cudaMemcpyAsync(const_cast<double*>(p->d.mu), mu_host, AN * sizeof(double), cudaMemcpyHostToDevice, st));
  if (w0_host) CUDA_TRY(cudaMemcpyAsync(const_cast<double*>(p->d.w0), w0_host, AN * sizeof(double), cudaMemcpyHostToDevice, st));
  if (mu_host && p->q) {                 // benchmark shift: q = -mu - gamma Sigma w_b depends on mu
    Launcher L{p, st, p->kp / 8, 0};
    L.build_q();
    if (L.err != cudaSuccess) return set_err(PRISM_ERR_CUDA, "kernel launch failed: %s", cudaGetErrorString(L.err));
  }
  int r = prism_solve_batch(p, s, cuda_stream, p->w_stage, p->status, p->i_stage, nullptr, nullptr, info);
  if (r != PRISM_OK) return r;
  if (w_host) CUDA_TRY(cudaMemcpyAsync(w_host, p->w_stage, AN * sizeof(double), cudaMemcpyDeviceToHost, st));
  if (status_host) CUDA_TRY(cudaMemcpyAsync(status_host, p->status, (size_t)p->A * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (iters_host) CUDA_TRY(cudaMemcpyAsync(iters_host, p->i_stage, (size_t)p->A * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (resid_host) CUDA_TRY(cudaMemcpyAsync(resid_host, p->resid, (size_t)p->A * PRISM_NRES * sizeof(double), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if (info) info->wall_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  return PRISM_OK;
}
