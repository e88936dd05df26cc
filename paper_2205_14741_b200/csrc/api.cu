// C-ABI entry points that dispatch or compose: sm_sign_ns (a3) and sm_density (a5, the whole path
// gather -> sign -> scatter -> D = 1/2 (I - R), PAPER.md:110 steps 1-3 + PAPER.md:91 Eq. 14, S = I).
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <numeric>
#include <utility>
#include <vector>

#include "common.cuh"

using namespace sm;

namespace sm {
// ---- variant selection: one table, filled once from the environment, changed by sm_set_option ---------------
struct OptDef { const char *name, *env; int32_t def; };
static const OptDef kOpt[OPT_COUNT] = {
    {"umma.sym", "SM_UMMA_SYM", 1},           {"umma.dyn", "SM_UMMA_DYN", 1},     {"umma.rev", "SM_UMMA_REV", 1},
    {"umma.stages", "SM_UMMA_STAGES", 0},     {"umma.stream", "SM_UMMA_STREAM", 0}, {"umma.resident", "SM_UMMA_RESIDENT", 1},
    {"umma.lt", "SM_UMMA_LT", 0},             {"f64.simt", "SM_F64_SIMT", 0},     {"gather.tma", "SM_GATHER_TMA", 0},
    {"umma.epi", "SM_UMMA_EPI", 0},           {"f32.sym", "SM_F32_SYM", 1},
    {"f64.tile", "SM_F64_TILE", 0},           {"umma.fold", "SM_UMMA_FOLD", 1},
    {"gather.lean", "SM_GATHER_LEAN", 1},     {"umma.sharea", "SM_UMMA_SHAREA", 1},
    {"umma.ncta", "SM_UMMA_NCTA", 1},         {"umma.mc", "SM_UMMA_MC", 1},       {"umma.tmap", "SM_UMMA_TMAP", 0},
    {"umma.fused", "SM_UMMA_FUSED", 0},       {"umma.slots", "SM_UMMA_SLOTS", 2}, {"umma.dbg", "SM_UMMA_DBG", 0}};
#ifdef SM_MEASURE
static constexpr int kOptUsable = OPT_COUNT;
#else
static constexpr int kOptUsable = OPT_FIRST_MEASURE;      // measurement-only knobs do not exist in this build
#endif
static std::atomic<int32_t> g_opt[OPT_COUNT];
static std::once_flag g_opt_once;
static void opt_init() {
  for (int i = 0; i < OPT_COUNT; ++i) {
    int32_t v = kOpt[i].def;
    if (i < kOptUsable) { const char *e = getenv(kOpt[i].env); if (e && *e) v = atoi(e); }
    g_opt[i].store(v, std::memory_order_relaxed);
  }
}
int32_t opt(int id) {
  std::call_once(g_opt_once, opt_init);
  return g_opt[id].load(std::memory_order_relaxed);
}

// ---- device-side protocol failures: the kernels write a reason code into one pinned, device-mapped host word
// before they trap, so the code survives the sticky context error (sm_last_device_error).
static std::mutex g_err_mu;
static int32_t *g_err_word = nullptr;
int32_t *device_err_word() {
  std::lock_guard<std::mutex> lk(g_err_mu);
  if (!g_err_word) {
    void *p = nullptr;
    if (cudaHostAlloc(&p, 64, cudaHostAllocMapped | cudaHostAllocPortable) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    std::memset(p, 0, 64);
    g_err_word = (int32_t *)p;
  }
  return g_err_word;
}

// Optional per-launch timing of the dominant kernels (bench.py roofline): CUDA events recorded on the
// launching stream around every Newton-Schulz product launch while profiling is enabled.
struct GemmProfile {
  bool on = false;
  std::vector<std::pair<cudaEvent_t, cudaEvent_t>> ev;
  size_t used = 0;
};
static GemmProfile g_prof;

bool prof_enabled() { return g_prof.on; }
int32_t prof_begin(cudaStream_t st, int *slot) {
  *slot = -1;
  if (!g_prof.on) return SM_OK;
  if (g_prof.used == g_prof.ev.size()) {
    std::pair<cudaEvent_t, cudaEvent_t> e;
    SM_CUDA(cudaEventCreate(&e.first));
    SM_CUDA(cudaEventCreate(&e.second));
    g_prof.ev.push_back(e);
  }
  *slot = (int)g_prof.used++;
  SM_CUDA(cudaEventRecord(g_prof.ev[*slot].first, st));
  return SM_OK;
}
int32_t prof_end(cudaStream_t st, int slot) {
  if (slot >= 0) SM_CUDA(cudaEventRecord(g_prof.ev[slot].second, st));
  return SM_OK;
}

static __global__ void k_count_unconverged(int32_t n, const double *__restrict__ residual, double tol,
                                           int32_t *__restrict__ out) {
  int32_t c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c < n && !(residual[c] < tol)) atomicAdd(out, 1);       // also counts NaN
}
}  // namespace sm

extern "C" int32_t sm_set_option(const char *name, int32_t value) {
  if (!name) return SM_ERR_ARG;
  for (int i = 0; i < OPT_COUNT; ++i)
    if (!strcmp(name, kOpt[i].name)) {
      if (i >= kOptUsable) return SM_ERR_UNSUPPORTED;
      (void)opt(i);
      g_opt[i].store(value, std::memory_order_relaxed);
      return SM_OK;
    }
  return SM_ERR_ARG;
}
extern "C" int32_t sm_get_option(const char *name, int32_t *value) {
  if (!name || !value) return SM_ERR_ARG;
  for (int i = 0; i < OPT_COUNT; ++i)
    if (!strcmp(name, kOpt[i].name)) {
      if (i >= kOptUsable) return SM_ERR_UNSUPPORTED;
      *value = opt(i);
      return SM_OK;
    }
  return SM_ERR_ARG;
}
extern "C" int32_t sm_build_info(void) {
#ifdef SM_MEASURE
  return 1;
#else
  return 0;
#endif
}
extern "C" int32_t sm_last_device_error(void) {
  std::lock_guard<std::mutex> lk(g_err_mu);
  return g_err_word ? *(volatile int32_t *)g_err_word : 0;
}

extern "C" int64_t sm_sign_ws_bytes_ex(const sm_pattern_t *P, int32_t n_cols, int64_t packed_elems,
                                       int32_t x_dtype, int32_t flags) {
  if (!P || n_cols <= 0 || packed_elems <= 0) return SM_ERR_ARG;
  if (flags & ~(SM_SIGN_NONSYMMETRIC | SM_SIGN_ORDER3)) return SM_ERR_ARG;
  if (is_16bit(x_dtype))
    return sign_umma_ws_bytes(P, n_cols, packed_elems, x_dtype, flags & SM_SIGN_NONSYMMETRIC, (flags & SM_SIGN_ORDER3) ? 3 : 2);
  if (x_dtype == SM_F32 || x_dtype == SM_F64) return sign_simt_ws_bytes(P, n_cols, packed_elems, x_dtype);
  return SM_ERR_UNSUPPORTED;
}
extern "C" int64_t sm_sign_ws_bytes(const sm_pattern_t *P, int32_t n_cols, int64_t packed_elems,
                                    int32_t x_dtype) {
  return sm_sign_ws_bytes_ex(P, n_cols, packed_elems, x_dtype, 0);
}

extern "C" int32_t sm_sign_ns_ex(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols,
                                 const int64_t *col_off, int64_t packed_elems, int32_t x_dtype, void *X_packed,
                                 void *ws, int64_t ws_bytes, int32_t max_iter, double tol, int32_t flags,
                                 int32_t switch_iter, int32_t *iters, double *residual, void *stream) {
  if (!P || !col_off || !X_packed || !ws || !iters || !residual) return SM_ERR_ARG;
  if (!cols) n_cols = P->n_blk;
  if (n_cols <= 0 || max_iter < 0 || packed_elems <= 0) return SM_ERR_ARG;
  if (flags & ~(SM_SIGN_NONSYMMETRIC | SM_SIGN_ORDER3)) return SM_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  const int32_t nonsym = flags & SM_SIGN_NONSYMMETRIC, order = (flags & SM_SIGN_ORDER3) ? 3 : 2;
  if (order == 3 && nonsym) return SM_ERR_UNSUPPORTED;
  if (is_16bit(x_dtype))
    return sign_umma(P, cols, n_cols, col_off, packed_elems, x_dtype, X_packed, ws, ws_bytes, max_iter, tol,
                     iters, residual, nonsym, switch_iter, order, st);
  if (switch_iter >= 0) return SM_ERR_ARG;
  if (x_dtype == SM_F32 || x_dtype == SM_F64)
    return sign_simt(P, cols, n_cols, col_off, packed_elems, x_dtype, X_packed, ws, ws_bytes, max_iter, tol,
                     iters, residual, nonsym, order, st);
  return SM_ERR_UNSUPPORTED;
}
extern "C" int32_t sm_sign_ns(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols,
                              const int64_t *col_off, int64_t packed_elems, int32_t x_dtype, void *X_packed,
                              void *ws, int64_t ws_bytes, int32_t max_iter, double tol, int32_t *iters,
                              double *residual, void *stream) {
  return sm_sign_ns_ex(P, cols, n_cols, col_off, packed_elems, x_dtype, X_packed, ws, ws_bytes, max_iter, tol, 0, -1,
                       iters, residual, stream);
}

extern "C" int32_t sm_sign_status(const double *residual, int32_t n_cols, double tol, void *scratch,
                                  void *stream) {
  if (!residual || !scratch || n_cols <= 0) return SM_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  // fixed-count mode (tol <= 0): nothing to converge to, but a submatrix whose last residual is not finite or exceeds
  // 1 has DIVERGED (a spectral scale below rho / sqrt(3)); that is reported the same way
  if (!(tol > 0.0)) tol = 1.0;
  int32_t *d = (int32_t *)scratch;
  SM_CUDA(cudaMemsetAsync(d, 0, sizeof(int32_t), st));
  k_count_unconverged<<<(n_cols + 255) / 256, 256, 0, st>>>(n_cols, residual, tol, d);
  SM_LAUNCHED();
  int32_t h = 0;
  SM_CUDA(cudaMemcpyAsync(&h, d, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
  SM_CUDA(cudaStreamSynchronize(st));
  return h > 0 ? SM_WARN_NOT_CONVERGED : SM_OK;
}

namespace {
struct DensityWs { int64_t *col_off; void *X; void *gws; int64_t gws_bytes; void *sws; int64_t sws_bytes; int64_t used; };

DensityWs density_layout(void *ws, int64_t ws_bytes, const sm_bcsr_t *A, const sm_pattern_t *P, int32_t x_dtype,
                         int64_t max_chunk_elems, int32_t sign_flags) {
  WsCursor cur(ws, ws_bytes);
  DensityWs w;
  w.col_off = cur.take<int64_t>(P->n_blk + 1);
  w.X = cur.take<char>(max_chunk_elems * dtype_bytes(x_dtype));
  w.gws_bytes = sm_gather_ws_bytes(A, P, P->n_blk);
  w.gws = cur.take<char>(w.gws_bytes);
  w.sws_bytes = sm_sign_ws_bytes_ex(P, P->n_blk, max_chunk_elems, x_dtype, sign_flags);
  w.sws = cur.take<char>(w.sws_bytes > 0 ? w.sws_bytes : 1);
  w.used = cur.used + 256;
  return w;
}
}  // namespace

extern "C" int64_t sm_density_ws_bytes_ex(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t x_dtype,
                                          int64_t max_chunk_elems, int32_t sign_flags) {
  if (!A || !P || dtype_bytes(x_dtype) == 0) return SM_ERR_ARG;
  if (max_chunk_elems < (int64_t)P->max_dim_pad * P->max_dim_pad) return SM_ERR_ARG;
  if (sign_flags & ~SM_SIGN_ORDER3) return SM_ERR_ARG;
  return density_layout(nullptr, 0, A, P, x_dtype, max_chunk_elems, sign_flags).used;
}
extern "C" int64_t sm_density_ws_bytes(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t x_dtype,
                                       int64_t max_chunk_elems) {
  return sm_density_ws_bytes_ex(A, P, x_dtype, max_chunk_elems, 0);
}

extern "C" int32_t sm_density(const sm_bcsr_t *A, const void *A_vals, int32_t a_dtype, double mu,
                              int32_t x_dtype, int32_t scale_mode, int32_t max_iter, double tol,
                              int32_t symmetrise, const sm_pattern_t *P, const int32_t *h_dim_pad,
                              int64_t max_chunk_elems, void *ws, int64_t ws_bytes, int32_t d_dtype,
                              void *D_vals, double *trace, int32_t *iters, double *residual, double *scale,
                              void *stream) {
  return sm_density_ex(A, A_vals, a_dtype, mu, x_dtype, scale_mode, max_iter, tol, -1, 0, symmetrise, P, h_dim_pad,
                       max_chunk_elems, ws, ws_bytes, d_dtype, D_vals, trace, iters, residual, scale, stream);
}

extern "C" int32_t sm_density_ex(const sm_bcsr_t *A, const void *A_vals, int32_t a_dtype, double mu,
                                 int32_t x_dtype, int32_t scale_mode, int32_t max_iter, double tol, int32_t switch_iter,
                                 int32_t sign_flags, int32_t symmetrise, const sm_pattern_t *P, const int32_t *h_dim_pad,
                                 int64_t max_chunk_elems, void *ws, int64_t ws_bytes, int32_t d_dtype,
                                 void *D_vals, double *trace, int32_t *iters, double *residual, double *scale,
                                 void *stream) {
  if (!A || !A_vals || !P || !h_dim_pad || !ws || !D_vals || !iters || !residual || !scale) return SM_ERR_ARG;
  if (dtype_bytes(x_dtype) == 0) return SM_ERR_UNSUPPORTED;
  if (d_dtype != SM_F64 && d_dtype != SM_F32) return SM_ERR_UNSUPPORTED;
  if (max_chunk_elems < (int64_t)P->max_dim_pad * P->max_dim_pad) return SM_ERR_ARG;
  if (sign_flags & ~SM_SIGN_ORDER3) return SM_ERR_ARG;       // the density path is symmetric
  DensityWs w = density_layout(ws, ws_bytes, A, P, x_dtype, max_chunk_elems, sign_flags);
  if (w.sws_bytes < 0) return (int32_t)w.sws_bytes;
  if (w.used > ws_bytes) return SM_ERR_SPACE;
  const int32_t n = P->n_blk;
  // Same key as P->order: (dim_pad descending, id ascending); chunks are ranges of that order, so
  // the device list of a chunk is P->order + lo.  Output arrays are indexed by order position.
  std::vector<int32_t> ord(n);
  std::iota(ord.begin(), ord.end(), 0);
  std::stable_sort(ord.begin(), ord.end(), [&](int32_t x, int32_t y) { return h_dim_pad[x] > h_dim_pad[y]; });
  int32_t lo = 0;
  while (lo < n) {
    int64_t elems = 0;
    int32_t hi = lo;
    while (hi < n) {
      int64_t e = (int64_t)h_dim_pad[ord[hi]] * h_dim_pad[ord[hi]];
      if (hi > lo && elems + e > max_chunk_elems) break;
      elems += e; ++hi;
    }
    const int32_t nc = hi - lo;
    const int32_t *cols = P->order + lo;
    int32_t rc = sm_plan_columns(P, cols, nc, w.col_off, stream);
    if (rc != SM_OK) return rc;
    rc = sm_gather(A, A_vals, a_dtype, P, cols, nc, w.col_off, mu, scale_mode, x_dtype, w.X, scale + lo, w.gws,
                   w.gws_bytes, stream);
    if (rc != SM_OK) return rc;
    rc = sm_sign_ns_ex(P, cols, nc, w.col_off, elems, x_dtype, w.X, w.sws, w.sws_bytes, max_iter, tol, sign_flags, switch_iter,
                       iters + lo, residual + lo, stream);
    if (rc != SM_OK) return rc;
    // after a bf16 -> fp16 schedule the images hold fp16
    rc = sm_scatter(A, P, cols, nc, w.col_off, switch_iter >= 0 ? SM_F16 : x_dtype, w.X, d_dtype, D_vals, 0, stream);
    if (rc != SM_OK) return rc;
    lo = hi;
  }
  if (symmetrise) return sm::symmetrise_density(A, P, d_dtype, D_vals, trace, (cudaStream_t)stream);
  return sm_density_from_sign(A, P, d_dtype, D_vals, trace, stream);
}

// ---- chemical potential for a fixed electron count (Eq. 14) --------------
extern "C" int32_t sm_mu_search(const sm_bcsr_t *A, const void *A_vals, int32_t a_dtype, double n_target,
                                double mu_lo, double mu_hi, double tol_n, double mu_tol, int32_t max_trials,
                                int32_t x_dtype, int32_t scale_mode, int32_t max_iter, double tol,
                                int32_t symmetrise, const sm_pattern_t *P, const int32_t *h_dim_pad,
                                int64_t max_chunk_elems, void *ws, int64_t ws_bytes, int32_t d_dtype, void *D_vals,
                                double *trace, int32_t *iters, double *residual, double *scale, double *mu_out,
                                double *trace_out, int32_t *trials_out, void *stream) {
  if (!mu_out || !trace_out || !trials_out || !trace) return SM_ERR_ARG;
  if (!(mu_lo < mu_hi) || !(tol_n >= 0.0) || !(mu_tol >= 0.0) || max_trials < 3) return SM_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  int32_t trials = 0;
  auto count = [&](double mu, double *n) -> int32_t {
    int32_t rc = sm_density(A, A_vals, a_dtype, mu, x_dtype, scale_mode, max_iter, tol, symmetrise, P, h_dim_pad,
                            max_chunk_elems, ws, ws_bytes, d_dtype, D_vals, trace, iters, residual, scale, stream);
    if (rc != SM_OK) return rc;
    SM_CUDA(cudaMemcpyAsync(n, trace, sizeof(double), cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));
    ++trials;
    return SM_OK;
  };
  double n_lo = 0.0, n_hi = 0.0, n_mid = 0.0, mu = mu_hi;
  int32_t rc = count(mu_hi, &n_hi);
  if (rc != SM_OK) return rc;
  *mu_out = mu_hi; *trace_out = n_hi; *trials_out = trials;
  if (n_hi < n_target - tol_n) return SM_ERR_ARG;
  rc = count(mu_lo, &n_lo);
  if (rc != SM_OK) return rc;
  *mu_out = mu_lo; *trace_out = n_lo; *trials_out = trials;
  if (n_lo > n_target + tol_n) return SM_ERR_ARG;
  if (fabs(n_lo - n_target) <= tol_n) return SM_OK;          // the lower end already has the right count
  double lo = mu_lo, hi = mu_hi;
  while (trials < max_trials) {
    mu = 0.5 * (lo + hi);
    rc = count(mu, &n_mid);
    if (rc != SM_OK) return rc;
    *mu_out = mu; *trace_out = n_mid; *trials_out = trials;
    if (fabs(n_mid - n_target) <= tol_n) break;
    if (n_mid < n_target) lo = mu; else hi = mu;
    if (hi - lo <= mu_tol) break;
  }
  return SM_OK;
}

// ---- profiling hooks (host; see include/submatrix.h) ------------------------------------------
extern "C" int32_t sm_profile_enable(int32_t on) {
  sm::g_prof.on = on != 0;
  sm::g_prof.used = 0;
  return SM_OK;
}
extern "C" int32_t sm_profile_read(double *gemm_ms, int64_t *gemm_launches) {
  if (!gemm_ms || !gemm_launches) return SM_ERR_ARG;
  double total = 0.0;
  for (size_t i = 0; i < sm::g_prof.used; ++i) {
    SM_CUDA(cudaEventSynchronize(sm::g_prof.ev[i].second));
    float ms = 0.f;
    SM_CUDA(cudaEventElapsedTime(&ms, sm::g_prof.ev[i].first, sm::g_prof.ev[i].second));
    total += ms;
  }
  *gemm_ms = total;
  *gemm_launches = (int64_t)sm::g_prof.used;
  sm::g_prof.used = 0;
  return SM_OK;
}
