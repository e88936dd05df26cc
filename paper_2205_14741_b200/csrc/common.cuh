// Shared host/device helpers of libsubmatrix.so (CUDA path only; the oracle shares nothing).
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdint.h>

#include "../../include/submatrix.h"

namespace sm {

extern thread_local int32_t g_last_cuda_error;
extern thread_local int64_t g_launch_count;

inline int32_t cuda_fail(cudaError_t e) {
  g_last_cuda_error = (int32_t)e;
  return SM_ERR_CUDA;
}

#define SM_CUDA(call)                                   \
  do {                                                  \
    cudaError_t e__ = (call);                           \
    if (e__ != cudaSuccess) return sm::cuda_fail(e__);  \
  } while (0)

// Call after every kernel launch: counts the launch and catches configuration errors.
#define SM_LAUNCHED()                                   \
  do {                                                  \
    ++sm::g_launch_count;                               \
    cudaError_t e__ = cudaGetLastError();               \
    if (e__ != cudaSuccess) return sm::cuda_fail(e__);  \
  } while (0)

inline int64_t align_up(int64_t x, int64_t a) { return (x + a - 1) / a * a; }

inline int32_t dtype_bytes(int32_t dt) {
  switch (dt) {
    case SM_F64: return 8;
    case SM_F32: return 4;
    case SM_BF16: case SM_F16: return 2;
    default: return 0;
  }
}
inline bool is_16bit(int32_t dt) { return dt == SM_BF16 || dt == SM_F16; }

// Bump allocator over a caller-provided workspace.
struct WsCursor {
  char *base; int64_t bytes; int64_t used;
  WsCursor(void *p, int64_t n) : base((char *)p), bytes(n), used(0) {}
  template <typename T> T *take(int64_t count) {
    int64_t off = align_up(used, 256);
    used = off + (int64_t)sizeof(T) * (count > 0 ? count : 1);
    return (T *)(base ? base + off : nullptr);
  }
  bool ok() const { return used <= bytes; }
};

// Element offset of (r, c) inside a Pd x Pd submatrix stored as the K-major 128B-swizzled UMMA
// image (include/submatrix.h, "Packed submatrix buffers").
__host__ __device__ inline int64_t img_off(int32_t Pd, int32_t r, int32_t c) {
  return (int64_t)(c >> 6) * Pd * 64 + (int64_t)r * 64 + ((((c & 63) >> 3) ^ (r & 7)) << 3) + (c & 7);
}

// lower_bound on a sorted int32 range [lo, hi): index of `key` or -1.
__device__ inline int32_t find_sorted(const int32_t *__restrict__ a, int32_t lo, int32_t hi, int32_t key) {
  int32_t l = lo, h = hi - 1;
  while (l <= h) {
    int32_t mid = (l + h) >> 1;
    int32_t v = __ldg(a + mid);
    if (v == key) return mid;
    if (v < key) l = mid + 1; else h = mid - 1;
  }
  return -1;
}

// Largest c in [0, n) with ptr[c] <= t (ptr ascending, ptr[0] = 0, ptr[n] > t).
template <typename T>
__device__ inline int32_t upper_slot(const T *__restrict__ ptr, int32_t n, T t) {
  int32_t lo = 0, hi = n;
  while (hi - lo > 1) {
    int32_t mid = (lo + hi) >> 1;
    if (ptr[mid] <= t) lo = mid; else hi = mid;
  }
  return lo;
}

template <typename T> __device__ inline T from_double(double v);
template <> __device__ inline double from_double<double>(double v) { return v; }
template <> __device__ inline float from_double<float>(double v) { return (float)v; }
template <> __device__ inline __nv_bfloat16 from_double<__nv_bfloat16>(double v) { return __float2bfloat16_rn((float)v); }
template <> __device__ inline __half from_double<__half>(double v) { return __float2half_rn((float)v); }

template <typename T> __device__ inline T from_float(float v) { return from_double<T>((double)v); }
template <> __device__ inline __nv_bfloat16 from_float<__nv_bfloat16>(float v) { return __float2bfloat16_rn(v); }
template <> __device__ inline __half from_float<__half>(float v) { return __float2half_rn(v); }

template <typename T> __device__ inline double to_double(T v);
template <> __device__ inline double to_double<double>(double v) { return v; }
template <> __device__ inline double to_double<float>(float v) { return (double)v; }
template <> __device__ inline double to_double<__nv_bfloat16>(__nv_bfloat16 v) { return (double)__bfloat162float(v); }
template <> __device__ inline double to_double<__half>(__half v) { return (double)__half2float(v); }

// ---- measurement hooks (api.cu): CUDA events around every launch of the Newton-Schulz product kernels
// while sm_profile_enable(1) is in force; slot = -1 when disabled.
bool prof_enabled();                                   // sm_profile_enable(1) is in effect (its events allocate)
int32_t prof_begin(cudaStream_t st, int *slot);
int32_t prof_end(cudaStream_t st, int slot);

// ---- internal entry points implemented across the .cu files
int32_t symmetrise_density(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t d_dtype, void *RD_vals,
                           double *trace, cudaStream_t st);                                  // gather_scatter.cu
int32_t exclusive_scan_i64(int32_t n, const int64_t *in, int64_t *out, cudaStream_t st);   // pattern.cu
int64_t global_scale_ws_bytes(const sm_bcsr_t *A, const sm_pattern_t *P);                    // global_scale.cu
int32_t global_scale(const sm_bcsr_t *A, const void *A_vals, int32_t a_dtype, const sm_pattern_t *P, double mu,
                     int32_t n_cols, double *scale, void *ws, int64_t ws_bytes, cudaStream_t st);
int32_t power_scale(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off,
                    int32_t x_dtype, void *X, double *scale, double *ratio, cudaStream_t st);  // power_scale.cu
// nonsym: the iterates are NOT symmetric (true products X X, X Y on every tile; sm_sign_ns_ex SM_SIGN_NONSYMMETRIC);
// switch_iter >= 0: bf16 -> fp16 precision schedule (16-bit only)
int32_t sign_simt(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off,
                  int64_t packed_elems, int32_t x_dtype, void *X, void *ws, int64_t ws_bytes,
                  int32_t max_iter, double tol, int32_t *iters, double *residual, int32_t nonsym, int32_t order, cudaStream_t st);
int32_t sign_umma(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off,
                  int64_t packed_elems, int32_t x_dtype, void *X, void *ws, int64_t ws_bytes,
                  int32_t max_iter, double tol, int32_t *iters, double *residual, int32_t nonsym, int32_t switch_iter, int32_t order,
                  cudaStream_t st);
int64_t sign_simt_ws_bytes(const sm_pattern_t *P, int32_t n_cols, int64_t packed_elems, int32_t x_dtype);
int32_t dense_product(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off, int32_t x_dtype,
                      const void *A, const void *B, void *O, int32_t *active, int32_t *last_zero, cudaStream_t st);   // sign_simt.cu
int64_t sign_umma_ws_bytes(const sm_pattern_t *P, int32_t n_cols, int64_t packed_elems, int32_t x_dtype, int32_t nonsym,
                           int32_t order);
int32_t umma_product(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off, int64_t packed_elems,
                     int32_t x_dtype, const void *A, const void *B, void *O, void *ws, int64_t ws_bytes, cudaStream_t st);   // sign_umma.cu
int32_t *device_err_word();        // pinned, device-mapped host word the kernels write a protocol-failure code to (api.cu)

// ---- variant selection (api.cu): sm_set_option / environment at first use.  Ids are indices into the table there.
enum OptId {
  OPT_UMMA_SYM = 0, OPT_UMMA_DYN, OPT_UMMA_REV, OPT_UMMA_STAGES, OPT_UMMA_STREAM, OPT_UMMA_RESIDENT, OPT_UMMA_LT,
  OPT_F64_SIMT, OPT_GATHER_TMA, OPT_UMMA_EPI, OPT_F32_SYM, OPT_F64_TILE, OPT_UMMA_FOLD, OPT_GATHER_LEAN, OPT_UMMA_SHAREA,
  OPT_FIRST_MEASURE,                 // the ones below exist only in a -DSM_MEASURE build
  OPT_UMMA_NCTA = OPT_FIRST_MEASURE, OPT_UMMA_MC, OPT_UMMA_TMAP, OPT_UMMA_FUSED, OPT_UMMA_SLOTS, OPT_UMMA_DBG,
  OPT_COUNT
};
int32_t opt(int id);

}  // namespace sm
