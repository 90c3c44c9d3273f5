// prism.cu - C ABI (include/prism.h) and the host driver of the batched ADMM.
// Single translation unit: the kernels live in the .cuh files included here.  No torch types, no CPU fallback.
#include <chrono>
#include <new>
#include <string>
#include <thread>
#include <vector>
#include <cstdlib>

#include "common.cuh"
#include "diag.cuh"
#include "gemm.cuh"
#include "prox.cuh"
#include "prox_fast.cuh"
#include "prox_res.cuh"
#include "small.cuh"

#define PRISM_VERSION_STR "prism-b200 r1 (sm_100a, fp64 DMMA factor GEMMs, streaming two-threshold prox with TMA bulk-copy pipeline)"

static const int kMT[] = {2, 4, 7, 8, 13, 16};
static int pick_mt(int k) {
  for (int m : kMT) if (8 * m >= k) return m;
  return -1;
}
#define MT_SWITCH(mt, ...)                                            \
  switch (mt) {                                                       \
    case 2: { constexpr int MT = 2; __VA_ARGS__; } break;             \
    case 4: { constexpr int MT = 4; __VA_ARGS__; } break;             \
    case 7: { constexpr int MT = 7; __VA_ARGS__; } break;             \
    case 8: { constexpr int MT = 8; __VA_ARGS__; } break;             \
    case 13: { constexpr int MT = 13; __VA_ARGS__; } break;           \
    default: { constexpr int MT = 16; __VA_ARGS__; } break;           \
  }

#define PROX_SMEM_MAX (208 * 1024)   // dynamic shared memory budget of k_prox_smem (plus ~11 KB static)
static size_t g1_smem(int mt) { return (size_t)G1_STAGES * (8 * mt + G1_TA) * G1_LD * sizeof(double); }
static size_t g2_smem(int mt) { return (size_t)(G2_TM + G2_TN) * (8 * mt + 4) * sizeof(double); }

extern "C" void prism_default_settings(prism_settings* s) {
  if (!s) return;
  memset(s, 0, sizeof(*s));
  s->eps_rel = 1e-6; s->max_iter = 4000; s->check_every = 10; s->alpha = 1.6; s->rho_scale = 100.0;
  s->rho_band_scale = 1.0; s->adapt_rho = 1; s->gemm_mode = 0; s->time_limit_ms = 0.0; s->deadline_ms = 0.0;
  s->use_graph = 1; s->prox_window_mult = 32.0; s->first_check = 40; s->reserved0 = 0;
}
extern "C" const char* prism_last_error(void) { return g_err; }
extern "C" const char* prism_version(void) { return PRISM_VERSION_STR; }
extern "C" int64_t prism_problem_device_bytes(const prism_problem* p) { return p ? p->bytes : 0; }

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
  for (int i = 0; i < p->nparts; ++i) {
    prism_problem_destroy(p->parts[i]);
    if (p->part_stream[i]) cudaStreamDestroy(p->part_stream[i]);
    if (p->part_done[i]) cudaEventDestroy(p->part_done[i]);
  }
  void* ptrs[] = {p->Bp, p->Bt, p->invd, p->gram, p->q, p->v, p->rt, p->cc, p->xs, p->pxq, p->Tpart, p->V, p->Sinv,
                  p->gw0, p->lamG, p->resid, p->duals, p->status, p->ap.c, p->ap.alpha, p->ap.beta,
                  p->ap.mode, p->ap.bsum, p->ap.done, p->ap.conv, p->ap.iters, p->ap.refactor,
                  p->ap.nadapt, p->ap.win, p->ap.wins, p->ap.slack, p->counters, p->w_stage, p->i_stage, p->lraw, p->lcomp, p->lcnt, p->cbin, p->chkp, p->lflag, p->stats};
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
  struct Ev { cudaEvent_t a, b; int cls; };
  std::vector<Ev> evs;
  void begin(int cls) {
    if (!prof) return;
    Ev e; e.cls = cls;
    cudaEventCreate(&e.a); cudaEventCreate(&e.b);
    cudaEventRecord(e.a, st);
    evs.push_back(e);
  }
  void end() {
    if (prof) cudaEventRecord(evs.back().b, st);
    ++launches;
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

  Gemm1Args g1args(const double* X, const int32_t* done) const {
    Gemm1Args a;
    a.Bt = p->Bt; a.ldn = p->ldn; a.X = X; a.ldw = p->ldn; a.Tpart = p->Tpart; a.ldv = p->ldv; a.A = p->A;
    a.chunk = p->chunk; a.Npad = p->ldn; a.done = done;
    return a;
  }
  void gemm1(const double* X, const int32_t* done) {
    Gemm1Args a = g1args(X, done);
    begin(PRISM_K_GEMM1);
    if (gemm_mode == 1) {
      const int kp = p->kp;
      dim3 grid(p->nchunk, (unsigned)(((int64_t)p->A * kp + 127) / 128));
      k_gemm1_ref<<<grid, 128, 0, st>>>(a, kp);
    } else {
      dim3 grid(p->nchunk, (p->A + G1_TA - 1) / G1_TA);
      MT_SWITCH(mt, k_gemm1<MT><<<grid, 256, g1_smem(MT), st>>>(a));
    }
    end();
  }
  template <int MODE>
  void gemm2(const Gemm2Args& a) {
    begin(PRISM_K_GEMM2);
    if (gemm_mode == 1) {
      dim3 grid((unsigned)((p->N + 127) / 128), p->A);
      k_gemm2_ref<MODE><<<grid, 128, 0, st>>>(a);
    } else {
      dim3 grid((unsigned)((p->N + G2_TN - 1) / G2_TN), (p->A + G2_TM - 1) / G2_TM);
      MT_SWITCH(mt, k_gemm2<MT, MODE><<<grid, 256, g2_smem(MT), st>>>(a));
    }
    end();
  }
  Gemm2Args g2base() const {
    Gemm2Args a;
    memset(&a, 0, sizeof(a));
    a.Bp = p->Bp; a.kp = p->kp; a.V = p->V; a.ldv = p->ldv; a.N = p->N; a.ldw = p->ldn; a.A = p->A; a.G = 0;     // no consensus rows in the x-update: U = Bp
    a.group_id = nullptr; a.invd = p->invd; a.d = p->d.d; a.gamma = p->d.gamma; a.c = p->ap.c;
    a.v = p->v; a.cc = p->cc; a.rt = p->rt; a.xs = p->xs; a.pxq = p->pxq; a.q = p->q; a.mu = p->d.mu;
    a.relax = 1.0; a.done = nullptr;
    return a;
  }
  // pxq <- gamma Sigma X   (H8: Sigma W = B (F (B'W)) + D o W, fp64)
  void sigma_apply(const double* X) {
    gemm1(X, nullptr);
    begin(PRISM_K_OTHER);
    k_scale_fs<<<p->A, 128, 0, st>>>(p->Tpart, p->nchunk, p->A, p->k, p->kp, p->ldv, p->d.f, p->d.gamma, p->V);
    end();
    Gemm2Args a = g2base();
    a.X = X;
    gemm2<G2_SIGMA>(a);
  }
};

static int set_kernel_attrs(int mt, int Kp) {
  MT_SWITCH(mt, {
    CUDA_TRY(cudaFuncSetAttribute(k_gemm1<MT>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g1_smem(MT)));
    CUDA_TRY(cudaFuncSetAttribute(k_gemm2<MT, G2_ADMM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g2_smem(MT)));
    CUDA_TRY(cudaFuncSetAttribute(k_gemm2<MT, G2_ADMM_CHECK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g2_smem(MT)));
    CUDA_TRY(cudaFuncSetAttribute(k_gemm2<MT, G2_SIGMA>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)g2_smem(MT)));
  });
  CUDA_TRY(cudaFuncSetAttribute(k_prox_smem, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)PROX_SMEM_MAX));
  CUDA_TRY(cudaFuncSetAttribute(k_prox_stream<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stream_smem_bytes(PRISM_MAX_GROUPS)));
  CUDA_TRY(cudaFuncSetAttribute(k_prox_stream<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stream_smem_bytes(PRISM_MAX_GROUPS)));
  CUDA_TRY(cudaFuncSetAttribute(k_factor, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)((size_t)Kp * Kp * sizeof(double))));
  return PRISM_OK;
}

// cluster-resident prox: smallest cluster size for which a slice of the account fits the shared-memory budget
static bool res_geometry(prism_problem* p) {
  static const int kC[] = {1, 2, 4, 8, 16};
  for (int C : kC) {
    int SL = 0;
    if (res_fits(p->N, p->G, C, &SL)) {
      p->res_C = C; p->res_SL = SL; p->res_smem = res_layout(SL, p->G, C).bytes;
      return true;
    }
  }
  return false;
}
template <bool LOTS, bool CHECK>
static int res_attrs_one(const prism_problem* p) {
  CUDA_TRY(cudaFuncSetAttribute(k_prox_res<LOTS, CHECK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->res_smem));
  if (p->res_C > 8) CUDA_TRY(cudaFuncSetAttribute(k_prox_res<LOTS, CHECK>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  return PRISM_OK;
}
static int res_attrs(const prism_problem* p) {
  int r;
  if (p->d.lot_count) { if ((r = res_attrs_one<true, false>(p)) != PRISM_OK) return r; return res_attrs_one<true, true>(p); }
  if ((r = res_attrs_one<false, false>(p)) != PRISM_OK) return r;
  return res_attrs_one<false, true>(p);
}
template <bool LOTS, bool CHECK>
static cudaError_t res_launch(const prism_problem* p, cudaStream_t st, const ProxArgs& a, int mode) {
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3((unsigned)p->res_C, (unsigned)p->A, 1);
  cfg.blockDim = dim3(RES_NT, 1, 1);
  cfg.dynamicSmemBytes = p->res_smem;
  cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = (unsigned)p->res_C; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, k_prox_res<LOTS, CHECK>, a, mode);
}

static bool fast_applicable(const prism_problem* p) {
  return !p->d.lot_count && !p->d.hi_full && p->N < ((int64_t)1 << PROX_META_IDX_BITS) && p->N % 16 == 0 &&
         !getenv("PRISM_PROX_NOFAST");     // N % 16: every row of every streamed array is 16-byte aligned (bulk copies)
}

// ------------------------------------------------------------------------------------------ create (H0)
static int create_one(int64_t N, int32_t k, int32_t accounts, const prism_constraint_set* cs,
                      const prism_data* data, void* cuda_stream, prism_problem** out) {
  if (out) *out = nullptr;
  if (!out || !cs || !data) return set_err(PRISM_ERR_INVALID_ARG, "null argument%s", "");
  const int A = accounts, G = (cs->flags & PRISM_GROUP_BANDS) ? cs->G : 0;
  if (N < 1 || k < 1 || A < 1) return set_err(PRISM_ERR_INVALID_ARG, "N, k, accounts must be >= 1%s", "");
  if (!(cs->flags & PRISM_BUDGET) || !(cs->flags & PRISM_BOX)) return set_err(PRISM_ERR_INVALID_ARG, "PRISM_BUDGET and PRISM_BOX are mandatory%s", "");
  const int mt = pick_mt(k);
  if (mt < 0 || k > PRISM_MAX_FACTORS) return set_err(PRISM_ERR_INVALID_ARG, "k = %s%lld exceeds the supported factor count (128)", "", k);
  if (G < 0 || G > PRISM_MAX_GROUPS || 8 * mt > PRISM_MAX_KPRIME) return set_err(PRISM_ERR_INVALID_ARG, "G = %s%lld out of range", "", G);
  if ((cs->flags & PRISM_GROUP_BANDS) && (G < 1 || !data->group_id || !data->band_lo || !data->band_hi)) return set_err(PRISM_ERR_INVALID_ARG, "group bands need G >= 1, group_id, band_lo, band_hi%s", "");
  if ((cs->flags & PRISM_TAX_LOTS) && (!data->lot_slope || !data->lot_width || !data->lot_count || cs->max_lots < 1 || cs->max_lots > PRISM_MAX_LOTS)) return set_err(PRISM_ERR_INVALID_ARG, "tax lots need lot arrays and 1 <= max_lots <= 4%s", "");
  if (!data->B || !data->f || !data->d || !data->mu || !data->gamma || !data->w0 || !data->lo || !data->hi) return set_err(PRISM_ERR_INVALID_ARG, "missing mandatory data pointer%s", "");
  if (data->d_t) return set_err(PRISM_ERR_INVALID_ARG, "d_t must be NULL: the turnover scaling D_a is the identity in this build%s", "");
  if ((cs->flags & PRISM_BENCHMARK_SHIFT) && !data->w_b) return set_err(PRISM_ERR_INVALID_ARG, "PRISM_BENCHMARK_SHIFT needs w_b%s", "");

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
  // split-K chunking of GEMM-1: about two waves of CTAs
  const int tilesA = (A + G1_TA - 1) / G1_TA;
  int64_t want = (2 * p->sm_count + tilesA - 1) / tilesA;
  const int64_t nst = p->ldn / G1_KS;
  if (want > nst) want = nst;
  if (want < 1) want = 1;
  p->chunk = ((nst + want - 1) / want) * G1_KS;
  p->nchunk = (int)((p->ldn + p->chunk - 1) / p->chunk);
  cudaStream_t st = (cudaStream_t)cuda_stream;

  const size_t AN = (size_t)A * p->ldn;
  ALLOC_TRY(dev_alloc(p, &p->Bp, (size_t)N * p->kp));
  ALLOC_TRY(dev_alloc(p, &p->Bt, (size_t)p->kp * p->ldn));
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
  ALLOC_TRY(dev_alloc(p, &p->counters, (size_t)4));
  p->res = (res_geometry(p) && !getenv("PRISM_PROX_NORES")) ? 1 : 0;
  if (p->res) { int r = res_attrs(p); if (r != PRISM_OK) { prism_problem_destroy(p); return r; } }
  p->fast = (!p->res && fast_applicable(p)) ? 1 : 0;
  if (p->fast) {
    // slices: a few CTAs per resident slot so that the streaming kernel stays bandwidth-bound to the end of the grid
    int64_t target = ((int64_t)4 * 3 * p->sm_count + A - 1) / A;           // CTAs per account wanted
    int64_t sl = (N + target - 1) / target;
    sl = (sl + FAST_CH - 1) / FAST_CH * FAST_CH;
    if (const char* e = getenv("PRISM_PROX_SLICE")) sl = (atoll(e) + FAST_CH - 1) / FAST_CH * FAST_CH;
    if (sl < 2 * FAST_CH) sl = 2 * FAST_CH;
    p->slice_len = sl;
    p->S = (int)((N + sl - 1) / sl);
    p->capw = (int)(sl / FAST_NW);
    p->ldc = (int64_t)p->S * sl;
    const int Gb = G > 0 ? G : 1;
    ALLOC_TRY(dev_alloc(p, &p->lraw, (size_t)A * p->ldc, false));
    ALLOC_TRY(dev_alloc(p, &p->lcomp, (size_t)A * p->ldc, false));
    ALLOC_TRY(dev_alloc(p, &p->lcnt, (size_t)2 * A * p->S * FAST_NW));     // fronts, then backs of the two-level lists
    ALLOC_TRY(dev_alloc(p, &p->cbin, (size_t)2 * A * 2 * Gb));             // bins of the dead assets, then speculative bins
    ALLOC_TRY(dev_alloc(p, &p->chkp, (size_t)A * p->S * 8));
    ALLOC_TRY(dev_alloc(p, &p->lflag, (size_t)A));
  }
  if (getenv("PRISM_PROX_STATS")) ALLOC_TRY(dev_alloc(p, &p->stats, (size_t)4096 * 8));
  if (cudaMallocHost((void**)&p->h_counters, 4 * sizeof(int32_t)) != cudaSuccess) { prism_problem_destroy(p); return set_err(PRISM_ERR_ALLOC, "pinned allocation failed%s", ""); }
  if (p->d.w_b) ALLOC_TRY(dev_alloc(p, &p->q, AN));
  { int r = set_kernel_attrs(mt, p->Kp); if (r != PRISM_OK) { prism_problem_destroy(p); return r; } }

  k_setup_shared<<<(unsigned)((N + 127) / 128), 128, 0, st>>>(data->B, data->B_is_fp32, data->d, N, k, p->kp, p->ldn, p->Bp, p->Bt, p->invd);
  k_gram<<<dim3(p->Kp, p->Kp), 256, 0, st>>>(p->Bt, p->ldn, nullptr, p->invd, N, p->kp, 0, p->gram);
  if (p->d.w_b) {            // q = -mu - gamma Sigma w_b
    Launcher L{p, st, mt, 0};
    k_diff<<<dim3((unsigned)((N + 255) / 256), A), 256, 0, st>>>(p->d.w_b, nullptr, N, p->ldn, p->rt);
    L.sigma_apply(p->rt);
    k_make_q<<<dim3((unsigned)((N + 255) / 256), A), 256, 0, st>>>(p->d.mu, p->pxq, N, p->ldn, p->q);
    cudaMemsetAsync(p->rt, 0, AN * sizeof(double), st);
  }
  {
    std::vector<double> hd((size_t)N);
    cudaMemcpyAsync(hd.data(), data->d, (size_t)N * sizeof(double), cudaMemcpyDeviceToHost, st);
    cudaStreamSynchronize(st);
    double s = 0.0;
    for (int64_t i = 0; i < N; ++i) s += hd[(size_t)i];
    p->dbar = s / (double)N;
  }
  cudaError_t e = cudaStreamSynchronize(st);
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
  a.eps = s.eps_rel;
  a.adapt = s.adapt_rho; a.iter = 0; a.ldw = p->ldn;
  a.lraw = p->lraw; a.lcomp = p->lcomp; a.lcnt = p->lcnt; a.cbin = p->cbin; a.chkp = p->chkp; a.lflag = p->lflag;
  a.S = p->S; a.capw = p->capw; a.slice_len = p->slice_len; a.ldc = p->ldc;
  a.stats = p->stats;
  a.res_C = p->res_C; a.res_SL = p->res_SL;
  a.win_mult = s.prox_window_mult > 0 ? s.prox_window_mult : 32.0;
  if (const char* e = getenv("PRISM_PROX_WIN_MULT")) a.win_mult = atof(e);
  a.band_start = 20;
  if (const char* e = getenv("PRISM_PROX_BAND_START")) a.band_start = atoi(e);
  a.band_wide = 1;
  if (const char* e = getenv("PRISM_PROX_BAND_WIDE")) a.band_wide = atoi(e);
  a.band_ramp = 0;         // measured on configs[2]: a 10 / 20-iteration slack ramp costs 6% / 23% (the thresholds keep moving)
  if (const char* e = getenv("PRISM_PROX_BAND_RAMP")) a.band_ramp = atoi(e);
  a.win_ratio = 16.0;
  if (const char* e = getenv("PRISM_PROX_WIN_RATIO")) a.win_ratio = atof(e);
  return a;
}

// Streaming form (k_prox_stream + k_prox_root, prox_fast.cuh) where it applies; else one of the every-asset kernels.
static void launch_prox(Launcher& L, ProxArgs& a, int mode, int iter) {
  prism_problem* p = L.p;
  cudaStream_t st = L.st;
  a.iter = iter;
  if (p->res) {
    const bool chk = (mode & (PROX_CHECK | PROX_FINAL)) != 0;     // the final extraction also needs w_out
    L.begin(PRISM_K_PROX);
    if (p->d.lot_count) { if (chk) res_launch<true, true>(p, st, a, mode & ~PROX_CHECK); else res_launch<true, false>(p, st, a, mode); }
    else { if (chk) res_launch<false, true>(p, st, a, mode & ~PROX_CHECK); else res_launch<false, false>(p, st, a, mode); }
    L.end();
    return;
  }
  if (p->fast) {
    const bool chk = (mode & (PROX_CHECK | PROX_FINAL)) != 0;     // the final extraction also needs w_out
    const dim3 grid((unsigned)p->S, (unsigned)p->A);
    const size_t sm = stream_smem_bytes(p->G);
    const size_t smr = root_smem_bytes(p->G, 2 * p->S * FAST_NW);
    L.begin(PRISM_K_PROX);
    if (chk) k_prox_stream<true><<<grid, FAST_NW * 32, sm, st>>>(a);
    else k_prox_stream<false><<<grid, FAST_NW * 32, sm, st>>>(a);
    L.end();
    L.begin(PRISM_K_PROX_ROOT);
    if (chk) k_prox_root<true><<<p->A, ROOT_NT, smr, st>>>(a, mode & ~PROX_CHECK);
    else k_prox_root<false><<<p->A, ROOT_NT, smr, st>>>(a, mode);
    L.end();
    return;
  }
  const int grid = p->A < p->sm_count ? p->A : p->sm_count;
  L.begin(PRISM_K_PROX);
  if (p->d.lot_count) k_prox<true><<<grid, 512, 0, st>>>(a, mode);
  else if (p->d.hi_full || (size_t)p->N * 20 + 16 > PROX_SMEM_MAX) k_prox<false><<<grid, 512, 0, st>>>(a, mode);
  else k_prox_smem<<<grid, 512, (size_t)p->N * 20 + 16, st>>>(a, mode);
  L.end();
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
  k_diff<<<dim3((unsigned)((p->N + 255) / 256), p->A), 256, 0, L.st>>>(w, p->d.w_b, p->N, p->ldn, p->rt);
  L.end();
  L.sigma_apply(p->rt);
  DiagArgs da = make_diag_args(p, w, duals, resid);
  L.begin(PRISM_K_DIAG);
  if (p->d.lot_count) k_diag<true><<<p->A, 256, 0, L.st>>>(da);
  else k_diag<false><<<p->A, 256, 0, L.st>>>(da);
  L.end();
}

static int solve_one(prism_problem* p, const prism_settings* sp, void* cuda_stream, double* w_out,
                     int32_t* status_out, int32_t* iters_out, double* resid_out, double* duals_out,
                     prism_solve_info* info) {
  if (!p) return set_err(PRISM_ERR_NOT_READY, "problem object is NULL%s", "");
  if (!w_out || !status_out || !iters_out) return set_err(PRISM_ERR_INVALID_ARG, "w_out, status_out, iters_out are mandatory%s", "");
  prism_settings s;
  if (sp) s = *sp; else prism_default_settings(&s);
  if (!(s.eps_rel > 0) || s.max_iter < 1 || s.check_every < 1 || !(s.alpha > 0 && s.alpha < 2) || !(s.rho_scale > 0) || !(s.rho_band_scale > 0))
    return set_err(PRISM_ERR_INVALID_ARG, "invalid settings%s", "");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const auto t0 = std::chrono::steady_clock::now();
  auto elapsed_ms = [&]() { return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count(); };
  cudaEvent_t ev0, ev1;
  CUDA_TRY(cudaEventCreate(&ev0));
  CUDA_TRY(cudaEventCreate(&ev1));
  CUDA_TRY(cudaEventRecord(ev0, st));
  const int A = p->A, G = p->G;
  Launcher L{p, st, p->kp / 8, s.gemm_mode};

  CUDA_TRY(cudaMemsetAsync(p->counters, 0, 4 * sizeof(int32_t), st));
  CUDA_TRY(cudaMemsetAsync(p->rt, 0, (size_t)A * p->ldn * sizeof(double), st));
  CUDA_TRY(cudaMemsetAsync(p->resid, 0, (size_t)A * PRISM_NRES * sizeof(double), st));
  InitArgs ia;
  memset(&ia, 0, sizeof(ia));
  ia.N = p->N; ia.ldw = p->ldn; ia.A = A; ia.G = G; ia.w0 = p->d.w0; ia.gamma = p->d.gamma;
  ia.group_id = p->d.group_id; ia.v = p->v; ia.gw0 = p->gw0; ia.lamG = p->lamG; ia.ap = p->ap; ia.rho_scale = s.rho_scale;
  L.prof = s.profile != 0;
  L.begin(PRISM_K_OTHER);
  k_init_accounts<<<A, 256, 0, st>>>(ia);
  L.end();

  ProxArgs pa = make_prox_args(p, s, w_out);
  SolveArgs sa;
  memset(&sa, 0, sizeof(sa));
  sa.A = A; sa.kp = p->kp; sa.nchunk = p->nchunk; sa.ldv = p->ldv; sa.Tpart = p->Tpart; sa.Sinv = p->Sinv;
  sa.V = p->V; sa.ap = p->ap;
  Gemm2Args g2 = L.g2base();
  g2.relax = s.alpha; g2.done = p->ap.done;
  const size_t fac_smem = (size_t)p->Kp * p->Kp * sizeof(double);

  int it = 1, timed_out = 0, late_iter = -1, ndone = 0;
  for (; it <= s.max_iter; ++it) {
    const bool check = (it > 1) && ((it - 1) % s.check_every == 0) && (it - 1 >= s.first_check);   // residuals of the iterate after it-1 iterations
    launch_prox(L, pa, check ? PROX_CHECK : 0, it - 1);
    if (check || it == 1) {
      L.begin(PRISM_K_FACTOR);
      k_factor<<<A, 256, fac_smem, st>>>(p->gram, p->d.f, p->d.gamma, p->ap, p->k, p->kp, 0, p->Sinv);
      L.end();
    }
    if (check) {
      CUDA_TRY(cudaMemcpyAsync(p->h_counters, p->counters, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
      CUDA_TRY(cudaStreamSynchronize(st));
      ndone = p->h_counters[0];
      if (ndone >= A) break;
      const double el = elapsed_ms();
      if (s.deadline_ms > 0 && late_iter < 0 && el > s.deadline_ms) late_iter = it - 1;
      if (s.time_limit_ms > 0 && el > s.time_limit_ms) { timed_out = 1; break; }
    }
    L.gemm1(p->rt, p->ap.done);
    L.begin(PRISM_K_SOLVE);
    k_solve<<<A, 256, 0, st>>>(sa);
    L.end();
    const bool next_check = (it % s.check_every == 0) && (it >= s.first_check);
    if (next_check) L.gemm2<G2_ADMM_CHECK>(g2); else L.gemm2<G2_ADMM>(g2);
  }
  if (ndone < A) {           // iteration cap or time limit: extract z for the accounts still running
    launch_prox(L, pa, PROX_FINAL, it > s.max_iter ? s.max_iter : it - 1);
  }
  // H8 / H9: external diagnostics of the returned weights with the solver's multipliers, then statuses
  run_diag(p, L, w_out, p->duals, p->resid);
  L.begin(PRISM_K_OTHER);
  k_status<<<(A + 127) / 128, 128, 0, st>>>(A, p->resid, p->ap.conv, p->ap.iters, timed_out, late_iter, 1e-6, p->status);
  L.end();
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

// debug only (PRISM_PROX_STATS=1 at create): per-iteration counters of the streaming prox; not part of prism.h
extern "C" int prism_debug_prox_stats(prism_problem* p, int32_t* out, int clear) {
  if (p && p->nparts) {                       // sum over the account groups
    std::vector<int32_t> t((size_t)4096 * 8);
    for (size_t j = 0; j < t.size(); ++j) out[j] = 0;
    for (int i = 0; i < p->nparts; ++i) {
      const int r = prism_debug_prox_stats(p->parts[i], t.data(), clear);
      if (r != PRISM_OK) return r;
      for (size_t j = 0; j < t.size(); ++j) out[j] += t[j];
    }
    return PRISM_OK;
  }
  if (!p || !p->stats) return PRISM_ERR_NOT_READY;
  cudaMemcpy(out, p->stats, (size_t)4096 * 8 * sizeof(int32_t), cudaMemcpyDeviceToHost);
  if (clear) cudaMemset(p->stats, 0, (size_t)4096 * 8 * sizeof(int32_t));
  return PRISM_OK;
}

extern "C" int prism_kernel_times(const prism_problem* p, double* ms_out, int64_t* launches_out) {
  if (!p || !ms_out || !launches_out) return set_err(PRISM_ERR_INVALID_ARG, "null argument%s", "");
  for (int i = 0; i < PRISM_NKERN; ++i) { ms_out[i] = p->prof_ms[i]; launches_out[i] = p->prof_cnt[i]; }
  for (int j = 0; j < p->nparts; ++j)
    for (int i = 0; i < PRISM_NKERN; ++i) { ms_out[i] += p->parts[j]->prof_ms[i]; launches_out[i] += p->parts[j]->prof_cnt[i]; }
  return PRISM_OK;
}

static int residuals_one(prism_problem* p, const double* w, const double* duals, void* cuda_stream, double* resid_out) {
  cudaStream_t st = (cudaStream_t)cuda_stream;
  Launcher L{p, st, p->kp / 8, 0};
  run_diag(p, L, w, duals, p->resid);
  const double nanv = NAN;
  std::vector<double> h((size_t)p->A * PRISM_NRES);
  CUDA_TRY(cudaMemcpyAsync(h.data(), p->resid, h.size() * sizeof(double), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  for (int a = 0; a < p->A; ++a) { h[(size_t)a * PRISM_NRES + PRISM_R_PRIMAL] = nanv; h[(size_t)a * PRISM_NRES + PRISM_R_DUAL] = nanv; h[(size_t)a * PRISM_NRES + PRISM_R_RHO] = nanv; h[(size_t)a * PRISM_NRES + PRISM_R_RESERVED] = 0.0; }
  CUDA_TRY(cudaMemcpyAsync(resid_out, h.data(), h.size() * sizeof(double), cudaMemcpyHostToDevice, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  CUDA_TRY(cudaGetLastError());
  return PRISM_OK;
}

// ------------------------------------------------------------------------------------------ account groups
// Accounts are independent programs, and the per-account root kernel is latency-bound with a long tail
// (a launch lasts as long as its slowest account).  A large batch is therefore cut into contiguous account ranges,
// each a complete problem object solved by its own host thread on its own stream: the tail of one group's launch
// overlaps the bandwidth-bound kernels of the others.  Results per account do not depend on the split except through
// the split-K summation order of GEMM-1 (rounding level).
static int pick_parts(int64_t N, int A) {
  // measured on configs[2] (500 x 10,000): 2 / 3 groups solve 5% / 8% faster, but every launch then covers fewer
  // accounts and the streaming kernel runs further from its bandwidth roofline; one group unless asked otherwise.
  int n = 1;
  (void)N;
  if (const char* e = getenv("PRISM_PARTS")) n = atoi(e);
  if (n > PRISM_MAX_PARTS) n = PRISM_MAX_PARTS;
  if (n > A) n = A;
  return n < 1 ? 1 : n;
}
template <typename T>
static const T* off(const T* ptr, int64_t n) { return ptr ? ptr + n : nullptr; }

extern "C" int prism_problem_create(int64_t N, int32_t k, int32_t accounts, const prism_constraint_set* cs,
                                    const prism_data* data, void* cuda_stream, prism_problem** out) {
  if (out) *out = nullptr;
  if (!out || !cs || !data) return set_err(PRISM_ERR_INVALID_ARG, "null argument%s", "");
  const int A = accounts;
  const int np = (N >= 1 && A >= 1) ? pick_parts(N, A) : 1;
  if (np <= 1) return create_one(N, k, accounts, cs, data, cuda_stream, out);
  prism_problem* p = new (std::nothrow) prism_problem();
  if (!p) return set_err(PRISM_ERR_ALLOC, "host allocation failed%s", "");
  memset(p, 0, sizeof(*p));
  const int G = (cs->flags & PRISM_GROUP_BANDS) ? cs->G : 0;
  p->N = N; p->k = k; p->A = A; p->G = G; p->flags = cs->flags; p->d = *data;
  for (int i = 0; i < np; ++i) {
    const int a0 = (int)((int64_t)A * i / np), a1 = (int)((int64_t)A * (i + 1) / np);
    p->part_a0[i] = a0; p->part_a0[i + 1] = a1;
    prism_data d = *data;
    const int64_t aN = (int64_t)a0 * N;
    d.mu = off(d.mu, aN); d.w0 = off(d.w0, aN); d.w_b = off(d.w_b, aN); d.hi_full = off(d.hi_full, aN); d.excl = off(d.excl, aN);
    d.lot_slope = off(d.lot_slope, aN * PRISM_MAX_LOTS); d.lot_width = off(d.lot_width, aN * PRISM_MAX_LOTS); d.lot_count = off(d.lot_count, aN);
    d.gamma = off(d.gamma, a0); d.lo = off(d.lo, a0); d.hi = off(d.hi, a0); d.tau = off(d.tau, a0); d.kappa = off(d.kappa, a0); d.c_buy = off(d.c_buy, a0);
    d.band_lo = off(d.band_lo, (int64_t)a0 * G); d.band_hi = off(d.band_hi, (int64_t)a0 * G);
    int r = create_one(N, k, a1 - a0, cs, &d, cuda_stream, &p->parts[i]);
    if (r == PRISM_OK && cudaStreamCreateWithFlags(&p->part_stream[i], cudaStreamNonBlocking) != cudaSuccess) r = set_err(PRISM_ERR_CUDA, "stream creation failed%s", "");
    if (r == PRISM_OK && cudaEventCreateWithFlags(&p->part_done[i], cudaEventDisableTiming) != cudaSuccess) r = set_err(PRISM_ERR_CUDA, "event creation failed%s", "");
    p->nparts = i + 1;
    if (r != PRISM_OK) { prism_problem_destroy(p); return r; }
    p->bytes += p->parts[i]->bytes;
  }
  ALLOC_TRY(dev_alloc(p, &p->resid, (size_t)A * PRISM_NRES));
  ALLOC_TRY(dev_alloc(p, &p->status, (size_t)A));
  *out = p;
  return PRISM_OK;
}

extern "C" int prism_solve_batch(prism_problem* p, const prism_settings* sp, void* cuda_stream, double* w_out,
                                 int32_t* status_out, int32_t* iters_out, double* resid_out, double* duals_out,
                                 prism_solve_info* info) {
  if (!p) return set_err(PRISM_ERR_NOT_READY, "problem object is NULL%s", "");
  if (!p->nparts) return solve_one(p, sp, cuda_stream, w_out, status_out, iters_out, resid_out, duals_out, info);
  if (!w_out || !status_out || !iters_out) return set_err(PRISM_ERR_INVALID_ARG, "w_out, status_out, iters_out are mandatory%s", "");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const auto t0 = std::chrono::steady_clock::now();
  const int np = p->nparts, G = p->G;
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  cudaEvent_t ev0, ev1;
  CUDA_TRY(cudaEventCreate(&ev0));
  CUDA_TRY(cudaEventCreate(&ev1));
  CUDA_TRY(cudaEventRecord(ev0, st));                      // the groups start after everything queued on the caller's stream
  std::vector<int> rc((size_t)np, PRISM_OK);
  std::vector<prism_solve_info> inf((size_t)np);
  std::vector<std::string> msg((size_t)np);
  auto work = [&](int i) {
    cudaSetDevice(dev);
    prism_problem* q = p->parts[i];
    const int64_t a0 = p->part_a0[i];
    cudaStream_t ps = p->part_stream[i];
    cudaError_t e = cudaStreamWaitEvent(ps, ev0, 0);
    if (e != cudaSuccess) { rc[(size_t)i] = PRISM_ERR_CUDA; msg[(size_t)i] = cudaGetErrorString(e); return; }
    rc[(size_t)i] = solve_one(q, sp, (void*)ps, w_out + a0 * p->N, status_out + a0, iters_out + a0,
                              resid_out ? resid_out + a0 * PRISM_NRES : nullptr,
                              duals_out ? duals_out + a0 * PRISM_NDUAL(G) : nullptr, &inf[(size_t)i]);
    if (rc[(size_t)i] != PRISM_OK) msg[(size_t)i] = g_err;
    cudaEventRecord(p->part_done[i], ps);
  };
  {
    std::vector<std::thread> th;
    const bool serial = sp && sp->profile != 0;          // per-kernel timings: every kernel alone on the device
    if (!serial) for (int i = 1; i < np; ++i) th.emplace_back(work, i);
    work(0);
    if (serial) for (int i = 1; i < np; ++i) work(i);
    for (auto& t : th) t.join();
  }
  for (int i = 0; i < np; ++i) CUDA_TRY(cudaStreamWaitEvent(st, p->part_done[i], 0));
  CUDA_TRY(cudaEventRecord(ev1, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  for (int i = 0; i < np; ++i)
    if (rc[(size_t)i] != PRISM_OK) { cudaEventDestroy(ev0); cudaEventDestroy(ev1); return set_err(rc[(size_t)i], "account group failed: %s", msg[(size_t)i].c_str()); }
  if (info) {
    memset(info, 0, sizeof(*info));
    float ms = 0.f;
    cudaEventElapsedTime(&ms, ev0, ev1);
    info->solve_interval_ms = ms;
    info->device_bytes = p->bytes;
    for (int i = 0; i < np; ++i) {
      const prism_solve_info& x = inf[(size_t)i];
      if (x.iters_max > info->iters_max) info->iters_max = x.iters_max;
      info->iters_total += x.iters_total; info->n_certified += x.n_certified; info->n_feasible += x.n_feasible;
      info->n_timeout += x.n_timeout; info->n_late += x.n_late; info->n_no_feasible += x.n_no_feasible; info->n_failed += x.n_failed;
      info->kernel_launches += x.kernel_launches;
    }
    info->wall_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  }
  cudaEventDestroy(ev0);
  cudaEventDestroy(ev1);
  return PRISM_OK;
}

extern "C" int prism_residuals(prism_problem* p, const double* w, const double* duals, void* cuda_stream, double* resid_out) {
  if (!p) return set_err(PRISM_ERR_NOT_READY, "problem object is NULL%s", "");
  if (!w || !resid_out) return set_err(PRISM_ERR_INVALID_ARG, "w and resid_out are mandatory%s", "");
  if (!p->nparts) return residuals_one(p, w, duals, cuda_stream, resid_out);
  for (int i = 0; i < p->nparts; ++i) {
    const int64_t a0 = p->part_a0[i];
    const int r = residuals_one(p->parts[i], w + a0 * p->N, duals ? duals + a0 * PRISM_NDUAL(p->G) : nullptr, cuda_stream,
                                resid_out + a0 * PRISM_NRES);
    if (r != PRISM_OK) return r;
  }
  return PRISM_OK;
}

extern "C" int prism_solve_batch_host(prism_problem* p, const prism_settings* s, void* cuda_stream, const double* mu_host,
                                      const double* w0_host, double* w_host, int32_t* status_host, int32_t* iters_host,
                                      double* resid_host, prism_solve_info* info) {
  if (!p) return set_err(PRISM_ERR_NOT_READY, "problem object is NULL%s", "");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const auto t0 = std::chrono::steady_clock::now();
  const size_t AN = (size_t)p->A * p->N;
  if (mu_host) CUDA_TRY(cudaMemcpyAsync((void*)p->d.mu, mu_host, AN * sizeof(double), cudaMemcpyHostToDevice, st));
  if (w0_host) CUDA_TRY(cudaMemcpyAsync((void*)p->d.w0, w0_host, AN * sizeof(double), cudaMemcpyHostToDevice, st));
  if (!p->w_stage) {
    if (dev_alloc(p, &p->w_stage, AN) != PRISM_OK || dev_alloc(p, &p->i_stage, (size_t)p->A) != PRISM_OK) return PRISM_ERR_ALLOC;
  }
  int r = prism_solve_batch(p, s, cuda_stream, p->w_stage, p->status, p->i_stage, p->nparts ? p->resid : nullptr, nullptr, info);
  if (r != PRISM_OK) return r;
  if (w_host) CUDA_TRY(cudaMemcpyAsync(w_host, p->w_stage, AN * sizeof(double), cudaMemcpyDeviceToHost, st));
  if (status_host) CUDA_TRY(cudaMemcpyAsync(status_host, p->status, (size_t)p->A * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (iters_host) CUDA_TRY(cudaMemcpyAsync(iters_host, p->i_stage, (size_t)p->A * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  if (resid_host) CUDA_TRY(cudaMemcpyAsync(resid_host, p->resid, (size_t)p->A * PRISM_NRES * sizeof(double), cudaMemcpyDeviceToHost, st));
  CUDA_TRY(cudaStreamSynchronize(st));
  if (info) info->wall_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  return PRISM_OK;
}
