// sm_sign_ns_static: the fp64 / fp32 Newton-Schulz sign iteration (a3; PAPER.md:87 Eq. 13, :110 step 2) for callers that
// cannot allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  It is
// sm_sign_ns with the workspace (the Y = X X buffer, the alternate X buffer, the per-submatrix flags and the residual
// partial sums) taken from ONE file-scope device array instead of a caller buffer; inputs and outputs are still the
// caller's.
//
//   * The array is SM_STATIC_WS_BYTES (16 MiB) and every GPU that loads the library holds it until the process exits.
//     Calls whose sm_sign_ws_bytes(...) exceeds it are rejected with SM_ERR_SPACE before anything is launched.
//   * In host code the array's NAME is a host-side stand-in, not a device address.  The device address is taken once
//     per device, with that device current, by cudaGetSymbolAddress (checked), and that pointer is what the kernels get.
//   * No cudaMalloc / cudaFree / allocating library routine on this path: the product kernels of sign_simt.cu, memsets and
//     (convergence mode only) a 4-byte device-to-host copy.  Refused (SM_ERR_UNSUPPORTED) while sm_profile_enable(1)
//     is on, because the profile creates CUDA events per launch, and for the 16-bit types, whose tcgen05 path keeps a
//     pinned host error word that is allocated on first use.
//   * Every call shares the array and finds the previous call's contents in it: everything that must start at zero (both
//     image buffers' padding, the partial sums, the flags) is cleared on the call's stream before the first product.
//     Two calls that overlap on the GPU (different streams, or different host threads) RACE on it: serialise them.
#include <mutex>

#include "common.cuh"

using namespace sm;

namespace {

constexpr int64_t SM_STATIC_WS_BYTES = 16ll << 20;
constexpr int MAX_DEVICES = 64;

static __device__ __align__(256) unsigned char g_static_ws[SM_STATIC_WS_BYTES];

std::mutex g_static_mu;
void *g_static_ptr[MAX_DEVICES] = {};      // device address of g_static_ws on device d (nullptr: not asked yet)

// the array's device address on the CURRENT device
int32_t static_ws(void **out) {
  int dev = -1;
  SM_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) return SM_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lk(g_static_mu);
  if (!g_static_ptr[dev]) {
    void *p = nullptr;
    SM_CUDA(cudaGetSymbolAddress(&p, g_static_ws));
    if (!p || ((uintptr_t)p & 255u) != 0) return SM_ERR_CUDA;
    g_static_ptr[dev] = p;
  }
  *out = g_static_ptr[dev];
  return SM_OK;
}

}  // namespace

extern "C" int64_t sm_sign_ns_static_capacity(void) { return SM_STATIC_WS_BYTES; }

extern "C" int32_t sm_sign_ns_static(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off,
                                     int64_t packed_elems, int32_t x_dtype, void *X_packed, int32_t max_iter, double tol,
                                     int32_t *iters, double *residual, void *stream) {
  if (!P || !col_off || !X_packed || !iters || !residual) return SM_ERR_ARG;
  if (!cols) n_cols = P->n_blk;
  if (n_cols <= 0 || max_iter < 0 || packed_elems <= 0) return SM_ERR_ARG;
  if (x_dtype != SM_F64 && x_dtype != SM_F32) return SM_ERR_UNSUPPORTED;
  if (prof_enabled()) return SM_ERR_UNSUPPORTED;
  const int64_t need = sign_simt_ws_bytes(P, n_cols, packed_elems, x_dtype);
  if (need < 0) return (int32_t)need;
  if (need > SM_STATIC_WS_BYTES) return SM_ERR_SPACE;          // beyond the static array: use sm_sign_ns with a caller buffer
  void *ws = nullptr;
  int32_t rc = static_ws(&ws);
  if (rc != SM_OK) return rc;
  // sign_simt clears the image buffers and the partial sums and initialises the flags on `stream` before its first launch
  return sign_simt(P, cols, n_cols, col_off, packed_elems, x_dtype, X_packed, ws, SM_STATIC_WS_BYTES, max_iter, tol, iters,
                   residual, 0, 2, (cudaStream_t)stream);
}
