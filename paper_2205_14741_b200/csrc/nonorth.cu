// non-orthogonal basis through the same submatrix + sign machinery.
//
//   sign([[0, A], [I, 0]]) = [[0, A^1/2], [A^-1/2, 0]]                          (Eq. 12; reading A20)
//   sign(A) = A (A^2)^-1/2, "various iterative methods"                          (Eq. 13)
//   P = 1/2 (I - sign(S^-1 H - mu I)) S^-1                                       (Eq. 14)
//
// sm_inv_sqrt: for every block column i of the overlap matrix S (same block pattern as H): gather T_i(S) (a2), build
// the 2m x 2m matrix M_i = [[0, T_i], [I, 0]] / s_i with s_i = sqrt(Gershgorin bound of T_i) (its eigenvalues are
// +-sqrt(lambda(T_i)) / s_i, inside (0, 1] in modulus), run the SAME Newton-Schulz kernels on it at doubled dimension
// with the non-symmetric flag (a3, sm_sign_ns_ex), take the lower-left block T_i^-1/2 (and the upper-right T_i^1/2) and
// insert the owned columns into block-sparse results (a4).  sign(M / s) = sign(M): no rescaling of the blocks.
// sm_density_nonorth: Eq. 14 per submatrix of the pair (H, S), all four dtypes: Z = T_S^-1/2 as above, S^-1 = Z Z,
// A = S^-1 T_H - mu I (not symmetric), scaled by its infinity norm (>= spectral radius), sign(A) by the non-symmetric
// Newton-Schulz kernels, P_i = 1/2 (I - sign(A)) S^-1, owned columns inserted; Tr(P S) = electron count.
#include <algorithm>
#include <numeric>
#include <vector>

#include "common.cuh"

using namespace sm;

namespace {

template <typename T, bool IMG> __device__ __forceinline__ int64_t eoff(int32_t Pd, int32_t r, int32_t c) {
  return IMG ? img_off(Pd, r, c) : (int64_t)r * Pd + c;
}

__global__ void k_block2_dims(int32_t n, int32_t pad_to, const int32_t *__restrict__ dim, int32_t *__restrict__ dim2,
                              int32_t *__restrict__ dim_pad2) {
  int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const int32_t m2 = 2 * dim[i];
  dim2[i] = m2;
  dim_pad2[i] = (m2 + pad_to - 1) / pad_to * pad_to;
}

// X2_c = [[0, X_c sqrt(g_c)], [I / sqrt(g_c), 0]] where X_c = T_c / g_c is what sm_gather(GERSHGORIN) wrote; padding 0.
template <typename T, bool IMG>
__global__ void k_block2_build(const int32_t *__restrict__ cols, const int32_t *__restrict__ dim,
                               const int32_t *__restrict__ dim_pad, const int32_t *__restrict__ dim_pad2,
                               const int64_t *__restrict__ col_off, const int64_t *__restrict__ col_off2,
                               const double *__restrict__ g, const T *__restrict__ X, T *__restrict__ X2) {
  const int32_t c = blockIdx.x, i = cols[c];
  const int32_t m = dim[i], Pd = dim_pad[i], Pd2 = dim_pad2[i];
  const double sg = sqrt(g[c]);
  const T *Xs = X + col_off[c];
  T *Xd = X2 + col_off2[c];
  const int64_t n = (int64_t)Pd2 * Pd2;
  for (int64_t e = (int64_t)blockIdx.y * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.y * blockDim.x) {
    const int32_t r = (int32_t)(e / Pd2), cc = (int32_t)(e - (int64_t)r * Pd2);
    double v = 0.0;
    if (r < m && cc >= m && cc < 2 * m) v = to_double<T>(Xs[eoff<T, IMG>(Pd, r, cc - m)]) * sg;
    else if (r >= m && r < 2 * m && cc == r - m) v = 1.0 / sg;
    Xd[eoff<T, IMG>(Pd2, r, cc)] = from_double<T>(v);
  }
}

// Z_c = block (row0.., col0..) of the doubled result, m x m, into an m-dimension packed buffer (padding 0):
// lower-left (m, 0) = T^-1/2, upper-right (0, m) = T^1/2.
template <typename T, bool IMG>
__global__ void k_block2_extract(const int32_t *__restrict__ cols, const int32_t *__restrict__ dim,
                                 const int32_t *__restrict__ dim_pad, const int32_t *__restrict__ dim_pad2,
                                 const int64_t *__restrict__ col_off, const int64_t *__restrict__ col_off2,
                                 int32_t lower_left, const T *__restrict__ X2, T *__restrict__ Z) {
  const int32_t c = blockIdx.x, i = cols[c];
  const int32_t m = dim[i], Pd = dim_pad[i], Pd2 = dim_pad2[i];
  const T *Xs = X2 + col_off2[c];
  T *Zd = Z + col_off[c];
  const int32_t r0 = lower_left ? m : 0, c0 = lower_left ? 0 : m;
  const int64_t n = (int64_t)Pd * Pd;
  for (int64_t e = (int64_t)blockIdx.y * blockDim.x + threadIdx.x; e < n; e += (int64_t)gridDim.y * blockDim.x) {
    const int32_t r = (int32_t)(e / Pd), cc = (int32_t)(e - (int64_t)r * Pd);
    Zd[eoff<T, IMG>(Pd, r, cc)] = (r < m && cc < m) ? Xs[eoff<T, IMG>(Pd2, r0 + r, c0 + cc)] : from_double<T>(0.0);
  }
}

// A_c <- (A_c - mu I) / s_c with s_c = max row sum of |A_c - mu I| (>= spectral radius).
template <typename T, bool IMG>
__global__ void k_shift_scale(const int32_t *__restrict__ cols, const int32_t *__restrict__ dim,
                              const int32_t *__restrict__ dim_pad, const int64_t *__restrict__ col_off, double mu,
                              T *__restrict__ A, double *__restrict__ scale) {
  const int32_t c = blockIdx.x, i = cols[c];
  const int32_t m = dim[i], Pd = dim_pad[i];
  T *Ac = A + col_off[c];
  __shared__ double red[256];
  double best = 0.0;
  for (int32_t r = threadIdx.x; r < m; r += blockDim.x) {
    double sum = 0.0;
    for (int32_t cc = 0; cc < m; ++cc) sum += fabs(to_double<T>(Ac[eoff<T, IMG>(Pd, r, cc)]) - (cc == r ? mu : 0.0));
    best = fmax(best, sum);
  }
  red[threadIdx.x] = best;
  __syncthreads();
  for (int d = blockDim.x / 2; d > 0; d >>= 1) {
    if ((int)threadIdx.x < d) red[threadIdx.x] = fmax(red[threadIdx.x], red[threadIdx.x + d]);
    __syncthreads();
  }
  const double s = red[0] > 0.0 ? red[0] : 1.0;
  if (threadIdx.x == 0) scale[c] = s;
  for (int64_t e = threadIdx.x; e < (int64_t)m * m; e += blockDim.x) {
    const int32_t r = (int32_t)(e / m), cc = (int32_t)(e - (int64_t)r * m);
    const int64_t o = eoff<T, IMG>(Pd, r, cc);
    Ac[o] = from_double<T>((to_double<T>(Ac[o]) - (cc == r ? mu : 0.0)) / s);
  }
}

// Q_c <- 1/2 (I - S_c), true part only (padding stays 0)
template <typename T, bool IMG>
__global__ void k_half_i_minus(const int32_t *__restrict__ cols, const int32_t *__restrict__ dim,
                               const int32_t *__restrict__ dim_pad, const int64_t *__restrict__ col_off,
                               T *__restrict__ S) {
  const int32_t c = blockIdx.x, i = cols[c];
  const int32_t m = dim[i], Pd = dim_pad[i];
  T *Sc = S + col_off[c];
  for (int64_t e = (int64_t)blockIdx.y * blockDim.x + threadIdx.x; e < (int64_t)m * m; e += (int64_t)gridDim.y * blockDim.x) {
    const int32_t r = (int32_t)(e / m), cc = (int32_t)(e - (int64_t)r * m);
    const int64_t o = eoff<T, IMG>(Pd, r, cc);
    Sc[o] = from_double<T>(0.5 * ((cc == r ? 1.0 : 0.0) - to_double<T>(Sc[o])));
  }
}

template <typename T, typename U>
__global__ void k_dot(int64_t n, const T *__restrict__ a, const U *__restrict__ b, double *__restrict__ out) {
  // one CTA, fixed summation order: deterministic
  __shared__ double red[1024];
  double sum = 0.0;
  for (int64_t e = threadIdx.x; e < n; e += blockDim.x) sum += to_double<T>(a[e]) * to_double<U>(b[e]);
  red[threadIdx.x] = sum;
  __syncthreads();
  for (int d = blockDim.x / 2; d > 0; d >>= 1) {
    if ((int)threadIdx.x < d) red[threadIdx.x] += red[threadIdx.x + d];
    __syncthreads();
  }
  if (threadIdx.x == 0) *out = red[0];
}

__global__ void k_fill_i32(int32_t n, int32_t v, int32_t *p) {
  int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) p[i] = v;
}

// the doubled problem as a pattern: only the fields the sign kernels read
sm_pattern_t doubled_pattern(const sm_pattern_t *P, int32_t *dim2, int32_t *dim_pad2) {
  sm_pattern_t Q = *P;
  Q.dim = dim2; Q.dim_pad = dim_pad2;
  Q.max_dim = 2 * P->max_dim;
  Q.max_dim_pad = (2 * P->max_dim + P->pad_to - 1) / P->pad_to * P->pad_to;
  return Q;
}

// element stride between the m-dimension buffers of nonorth_chunk (bulk copies need 16-byte aligned images)
inline int64_t buf_stride(int64_t max2) { return (max2 + 4095) & ~(int64_t)4095; }

struct InvWs {
  int64_t *col_off, *col_off2; int32_t *dim2, *dim_pad2, *ones, *zeros; void *X, *X2, *gws, *sws;
  int64_t gws_bytes, sws_bytes, used;
};
InvWs inv_layout(void *ws, int64_t ws_bytes, const sm_bcsr_t *S, const sm_pattern_t *P, int32_t x_dtype, int64_t max2,
                 int32_t n_extra) {
  WsCursor cur(ws, ws_bytes);
  InvWs w;
  const int32_t n = P->n_blk;
  w.col_off = cur.take<int64_t>(n + 1);
  w.col_off2 = cur.take<int64_t>(n + 1);
  w.dim2 = cur.take<int32_t>(n);
  w.dim_pad2 = cur.take<int32_t>(n);
  w.ones = cur.take<int32_t>(n);
  w.zeros = cur.take<int32_t>(n);
  const int64_t eb = dtype_bytes(x_dtype);
  // m-dimension buffers (each <= the doubled chunk size), at a stride that keeps every one of them 8 KB aligned
  w.X = cur.take<char>(buf_stride(max2) * eb * (1 + n_extra));
  w.X2 = cur.take<char>(max2 * eb);
  w.gws_bytes = sm_gather_ws_bytes(S, P, n);
  w.gws = cur.take<char>(w.gws_bytes);
  sm_pattern_t Q = doubled_pattern(P, nullptr, nullptr);
  const int64_t s2 = sm_sign_ws_bytes_ex(&Q, n, max2, x_dtype, SM_SIGN_NONSYMMETRIC);
  const int64_t s1 = sm_sign_ws_bytes_ex(P, n, max2, x_dtype, SM_SIGN_NONSYMMETRIC);
  w.sws_bytes = s2 > s1 ? s2 : s1;
  w.sws = cur.take<char>(w.sws_bytes > 0 ? w.sws_bytes : 1);
  w.used = cur.used + 256;
  return w;
}

// chunks of P->order whose DOUBLED images fit max2 elements
struct Chunk { int32_t lo, hi; int64_t elems, elems2; };
std::vector<Chunk> plan_chunks(const sm_pattern_t *P, const int32_t *h_dim, int64_t max2, std::vector<int32_t> &ord) {
  const int32_t n = P->n_blk, pad = P->pad_to;
  auto padded = [&](int32_t m) { return (int64_t)((m + pad - 1) / pad * pad); };
  ord.resize(n);
  std::iota(ord.begin(), ord.end(), 0);
  // same key as P->order: (dim_pad descending, id ascending)
  std::stable_sort(ord.begin(), ord.end(), [&](int32_t x, int32_t y) { return padded(h_dim[x]) > padded(h_dim[y]); });
  std::vector<Chunk> out;
  int32_t lo = 0;
  while (lo < n) {
    Chunk ch{lo, lo, 0, 0};
    while (ch.hi < n) {
      const int64_t p1 = padded(h_dim[ord[ch.hi]]), p2 = padded(2 * h_dim[ord[ch.hi]]);
      if (ch.hi > lo && ch.elems2 + p2 * p2 > max2) break;
      ch.elems += p1 * p1; ch.elems2 += p2 * p2; ++ch.hi;
    }
    out.push_back(ch);
    lo = ch.hi;
  }
  return out;
}

template <typename T, bool IMG>
int32_t inv_sqrt_chunk(const sm_bcsr_t *S, const void *S_vals, int32_t s_dtype, int32_t x_dtype, int32_t max_iter, double tol,
                       const sm_pattern_t *P, const sm_pattern_t *Q, const InvWs &w, const Chunk &ch, void *Zbuf,
                       int32_t *iters, double *residual, double *scale, cudaStream_t st) {
  const int32_t nc = ch.hi - ch.lo;
  const int32_t *cols = P->order + ch.lo;
  int32_t rc = sm_plan_columns(P, cols, nc, w.col_off, st);
  if (rc != SM_OK) return rc;
  rc = sm_plan_columns(Q, cols, nc, w.col_off2, st);
  if (rc != SM_OK) return rc;
  rc = sm_gather(S, S_vals, s_dtype, P, cols, nc, w.col_off, 0.0, SM_SCALE_GERSHGORIN, x_dtype, w.X, scale + ch.lo, w.gws,
                 w.gws_bytes, st);
  if (rc != SM_OK) return rc;
  dim3 g2(nc, 16);
  k_block2_build<T, IMG><<<g2, 256, 0, st>>>(cols, P->dim, P->dim_pad, Q->dim_pad, w.col_off, w.col_off2, scale + ch.lo,
                                             (const T *)w.X, (T *)w.X2);
  SM_LAUNCHED();
  rc = sm_sign_ns_ex(Q, cols, nc, w.col_off2, ch.elems2, x_dtype, w.X2, w.sws, w.sws_bytes, max_iter, tol,
                     SM_SIGN_NONSYMMETRIC, -1, iters + ch.lo, residual + ch.lo, st);
  if (rc != SM_OK) return rc;
  k_block2_extract<T, IMG><<<g2, 256, 0, st>>>(cols, P->dim, P->dim_pad, Q->dim_pad, w.col_off, w.col_off2, 1,
                                               (const T *)w.X2, (T *)Zbuf);
  SM_LAUNCHED();
  return SM_OK;
}

}  // namespace

extern "C" int64_t sm_inv_sqrt_ws_bytes(const sm_bcsr_t *S, const sm_pattern_t *P, int32_t x_dtype, int64_t max_chunk_elems2) {
  if (!S || !P || dtype_bytes(x_dtype) == 0) return SM_ERR_ARG;
  const int64_t p2 = (2 * (int64_t)P->max_dim + P->pad_to - 1) / P->pad_to * P->pad_to;
  if (max_chunk_elems2 < p2 * p2) return SM_ERR_ARG;
  return inv_layout(nullptr, 0, S, P, x_dtype, max_chunk_elems2, 0).used;
}

extern "C" int32_t sm_inv_sqrt(const sm_bcsr_t *S, const void *S_vals, int32_t s_dtype, int32_t x_dtype, int32_t max_iter,
                               double tol, const sm_pattern_t *P, const int32_t *h_dim, int64_t max_chunk_elems2, void *ws,
                               int64_t ws_bytes, int32_t z_dtype, void *Z_vals, void *Y_vals, int32_t *iters,
                               double *residual, double *scale, void *stream) {
  if (!S || !S_vals || !P || !h_dim || !ws || !Z_vals || !iters || !residual || !scale) return SM_ERR_ARG;
  if (dtype_bytes(x_dtype) == 0) return SM_ERR_UNSUPPORTED;
  if (z_dtype != SM_F64 && z_dtype != SM_F32) return SM_ERR_UNSUPPORTED;
  const int64_t p2 = (2 * (int64_t)P->max_dim + P->pad_to - 1) / P->pad_to * P->pad_to;
  if (max_chunk_elems2 < p2 * p2) return SM_ERR_ARG;
  InvWs w = inv_layout(ws, ws_bytes, S, P, x_dtype, max_chunk_elems2, 0);
  if (w.sws_bytes < 0) return (int32_t)w.sws_bytes;
  if (w.used > ws_bytes) return SM_ERR_SPACE;
  cudaStream_t st = (cudaStream_t)stream;
  const int32_t n = P->n_blk;
  k_block2_dims<<<(n + 255) / 256, 256, 0, st>>>(n, P->pad_to, P->dim, w.dim2, w.dim_pad2);
  SM_LAUNCHED();
  sm_pattern_t Q = doubled_pattern(P, w.dim2, w.dim_pad2);
  std::vector<int32_t> ord;
  for (const Chunk &ch : plan_chunks(P, h_dim, max_chunk_elems2, ord)) {
    const int32_t nc = ch.hi - ch.lo;
    const int32_t *cols = P->order + ch.lo;
    int32_t rc = SM_ERR_UNSUPPORTED;
    if (x_dtype == SM_F64) rc = inv_sqrt_chunk<double, false>(S, S_vals, s_dtype, x_dtype, max_iter, tol, P, &Q, w, ch, w.X, iters, residual, scale, st);
    else if (x_dtype == SM_F32) rc = inv_sqrt_chunk<float, false>(S, S_vals, s_dtype, x_dtype, max_iter, tol, P, &Q, w, ch, w.X, iters, residual, scale, st);
    else if (x_dtype == SM_BF16) rc = inv_sqrt_chunk<__nv_bfloat16, true>(S, S_vals, s_dtype, x_dtype, max_iter, tol, P, &Q, w, ch, w.X, iters, residual, scale, st);
    else if (x_dtype == SM_F16) rc = inv_sqrt_chunk<__half, true>(S, S_vals, s_dtype, x_dtype, max_iter, tol, P, &Q, w, ch, w.X, iters, residual, scale, st);
    if (rc != SM_OK) return rc;
    // a4: owned columns of T^-1/2 (symmetric: the owned rows are read)
    rc = sm_scatter(S, P, cols, nc, w.col_off, x_dtype, w.X, z_dtype, Z_vals, 0, stream);
    if (rc != SM_OK) return rc;
    if (Y_vals) {
      dim3 g2(nc, 16);
      if (x_dtype == SM_F64) k_block2_extract<double, false><<<g2, 256, 0, st>>>(cols, P->dim, P->dim_pad, Q.dim_pad, w.col_off, w.col_off2, 0, (const double *)w.X2, (double *)w.X);
      else if (x_dtype == SM_F32) k_block2_extract<float, false><<<g2, 256, 0, st>>>(cols, P->dim, P->dim_pad, Q.dim_pad, w.col_off, w.col_off2, 0, (const float *)w.X2, (float *)w.X);
      else if (x_dtype == SM_BF16) k_block2_extract<__nv_bfloat16, true><<<g2, 256, 0, st>>>(cols, P->dim, P->dim_pad, Q.dim_pad, w.col_off, w.col_off2, 0, (const __nv_bfloat16 *)w.X2, (__nv_bfloat16 *)w.X);
      else k_block2_extract<__half, true><<<g2, 256, 0, st>>>(cols, P->dim, P->dim_pad, Q.dim_pad, w.col_off, w.col_off2, 0, (const __half *)w.X2, (__half *)w.X);
      SM_LAUNCHED();
      rc = sm_scatter(S, P, cols, nc, w.col_off, x_dtype, w.X, z_dtype, Y_vals, 0, stream);
      if (rc != SM_OK) return rc;
    }
  }
  return SM_OK;
}

extern "C" int64_t sm_density_nonorth_ws_bytes(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t x_dtype,
                                               int64_t max_chunk_elems2) {
  if (!A || !P) return SM_ERR_ARG;
  if (dtype_bytes(x_dtype) == 0) return SM_ERR_UNSUPPORTED;
  const int64_t p2 = (2 * (int64_t)P->max_dim + P->pad_to - 1) / P->pad_to * P->pad_to;
  if (max_chunk_elems2 < p2 * p2) return SM_ERR_ARG;
  return inv_layout(nullptr, 0, A, P, x_dtype, max_chunk_elems2, 3).used;
}

template <typename T, bool IMG>
static int32_t nonorth_chunk(const sm_bcsr_t *A, const void *H_vals, const void *S_vals, int32_t a_dtype, double mu,
                             int32_t x_dtype, int32_t max_iter, double tol, const sm_pattern_t *P, const sm_pattern_t *Q,
                             const InvWs &w, const Chunk &ch, int64_t max2, int32_t d_dtype, void *P_vals, int32_t *iters,
                             double *residual, double *scale, cudaStream_t st) {
  const int32_t nc = ch.hi - ch.lo;
  const int32_t *cols = P->order + ch.lo;
  const int64_t bs = buf_stride(max2);
  T *B0 = (T *)w.X, *B1 = B0 + bs, *B2 = B1 + bs, *B3 = B2 + bs;
  // the product kernels write the true m x m part only and the DMMA kernel reads whole padded tiles: padding must be 0
  SM_CUDA(cudaMemsetAsync(B2, 0, (size_t)ch.elems * sizeof(T), st));
  SM_CUDA(cudaMemsetAsync(B3, 0, (size_t)ch.elems * sizeof(T), st));
  // fp64 / fp32: the DMMA / FFMA product kernels; 16-bit: the non-symmetric tcgen05 update kernel without its "+ X"
  auto product = [&](const T *Am, const T *Bm, T *Om) -> int32_t {
    if (IMG) return umma_product(P, cols, nc, w.col_off, ch.elems, x_dtype, Am, Bm, Om, w.sws, w.sws_bytes, st);
    return dense_product(P, cols, nc, w.col_off, x_dtype, Am, Bm, Om, w.ones, w.zeros, st);
  };
  // Z = T_S^-1/2 -> B1 (B0 is the gather / extraction scratch of inv_sqrt_chunk)
  int32_t rc = inv_sqrt_chunk<T, IMG>(A, S_vals, a_dtype, x_dtype, max_iter, tol, P, Q, w, ch, B1, iters, residual, scale, st);
  if (rc != SM_OK) return rc;
  // S^-1 = Z Z -> B2
  rc = product(B1, B1, B2);
  if (rc != SM_OK) return rc;
  // T_H (unscaled) -> B0; A = S^-1 T_H -> B3; A <- (A - mu I) / ||A - mu I||_inf
  rc = sm_gather(A, H_vals, a_dtype, P, cols, nc, w.col_off, 0.0, SM_SCALE_NONE, x_dtype, B0, scale + ch.lo, w.gws, w.gws_bytes, st);
  if (rc != SM_OK) return rc;
  rc = product(B2, B0, B3);
  if (rc != SM_OK) return rc;
  k_shift_scale<T, IMG><<<nc, 256, 0, st>>>(cols, P->dim, P->dim_pad, w.col_off, mu, B3, scale + ch.lo);
  SM_LAUNCHED();
  // sign(A), non-symmetric Newton-Schulz at dimension m
  rc = sm_sign_ns_ex(P, cols, nc, w.col_off, ch.elems, x_dtype, B3, w.sws, w.sws_bytes, max_iter, tol, SM_SIGN_NONSYMMETRIC,
                     -1, iters + ch.lo, residual + ch.lo, st);
  if (rc != SM_OK) return rc;
  // P_i = 1/2 (I - sign(A)) S^-1 -> B0, owned columns inserted (P_i is symmetric: the owned rows are read)
  dim3 g2(nc, 16);
  k_half_i_minus<T, IMG><<<g2, 256, 0, st>>>(cols, P->dim, P->dim_pad, w.col_off, B3);
  SM_LAUNCHED();
  rc = product(B3, B2, B0);
  if (rc != SM_OK) return rc;
  return sm_scatter(A, P, cols, nc, w.col_off, x_dtype, B0, d_dtype, P_vals, 0, st);
}

extern "C" int32_t sm_density_nonorth(const sm_bcsr_t *A, const void *H_vals, const void *S_vals, int32_t a_dtype, double mu,
                                      int32_t x_dtype, int32_t max_iter, double tol, int32_t symmetrise,
                                      const sm_pattern_t *P, const int32_t *h_dim, int64_t max_chunk_elems2, void *ws,
                                      int64_t ws_bytes, int32_t d_dtype, void *P_vals, double *trace_ps, int32_t *iters,
                                      double *residual, double *scale, void *stream) {
  if (!A || !H_vals || !S_vals || !P || !h_dim || !ws || !P_vals || !iters || !residual || !scale) return SM_ERR_ARG;
  if (dtype_bytes(x_dtype) == 0) return SM_ERR_UNSUPPORTED;
  const bool img = x_dtype == SM_BF16 || x_dtype == SM_F16;
  if (d_dtype != SM_F64 && d_dtype != SM_F32) return SM_ERR_UNSUPPORTED;
  if (!img && d_dtype != x_dtype) return SM_ERR_UNSUPPORTED;   // fp64 / fp32: P in the arithmetic type
  if (a_dtype != SM_F64 && a_dtype != SM_F32) return SM_ERR_UNSUPPORTED;
  if (!img && a_dtype != x_dtype && a_dtype != SM_F64) return SM_ERR_UNSUPPORTED;
  const int64_t p2 = (2 * (int64_t)P->max_dim + P->pad_to - 1) / P->pad_to * P->pad_to;
  if (max_chunk_elems2 < p2 * p2) return SM_ERR_ARG;
  InvWs w = inv_layout(ws, ws_bytes, A, P, x_dtype, max_chunk_elems2, 3);
  if (w.sws_bytes < 0) return (int32_t)w.sws_bytes;
  if (w.used > ws_bytes) return SM_ERR_SPACE;
  cudaStream_t st = (cudaStream_t)stream;
  const int32_t n = P->n_blk;
  k_block2_dims<<<(n + 255) / 256, 256, 0, st>>>(n, P->pad_to, P->dim, w.dim2, w.dim_pad2);
  SM_LAUNCHED();
  k_fill_i32<<<(n + 255) / 256, 256, 0, st>>>(n, 1, w.ones);
  SM_LAUNCHED();
  k_fill_i32<<<(n + 255) / 256, 256, 0, st>>>(n, 0, w.zeros);
  SM_LAUNCHED();
  sm_pattern_t Q = doubled_pattern(P, w.dim2, w.dim_pad2);
  std::vector<int32_t> ord;
  for (const Chunk &ch : plan_chunks(P, h_dim, max_chunk_elems2, ord)) {
    int32_t rc =
        x_dtype == SM_F64 ? nonorth_chunk<double, false>(A, H_vals, S_vals, a_dtype, mu, x_dtype, max_iter, tol, P, &Q, w, ch, max_chunk_elems2, d_dtype, P_vals, iters, residual, scale, st)
        : x_dtype == SM_F32 ? nonorth_chunk<float, false>(A, H_vals, S_vals, a_dtype, mu, x_dtype, max_iter, tol, P, &Q, w, ch, max_chunk_elems2, d_dtype, P_vals, iters, residual, scale, st)
        : x_dtype == SM_BF16 ? nonorth_chunk<__nv_bfloat16, true>(A, H_vals, S_vals, a_dtype, mu, x_dtype, max_iter, tol, P, &Q, w, ch, max_chunk_elems2, d_dtype, P_vals, iters, residual, scale, st)
                             : nonorth_chunk<__half, true>(A, H_vals, S_vals, a_dtype, mu, x_dtype, max_iter, tol, P, &Q, w, ch, max_chunk_elems2, d_dtype, P_vals, iters, residual, scale, st);
    if (rc != SM_OK) return rc;
  }
  if (symmetrise) {
    int32_t rc = sm_symmetrise(A, P, d_dtype, P_vals, stream);
    if (rc != SM_OK) return rc;
  }
  if (trace_ps) {
    // Tr(P S) = sum_ij P_ij S_ij (S symmetric, same block layout): the electron count of Eq. 14
    int64_t n_vals = 0;
    SM_CUDA(cudaMemcpyAsync(&n_vals, A->val_ptr + A->nnzb, sizeof(int64_t), cudaMemcpyDeviceToHost, st));
    SM_CUDA(cudaStreamSynchronize(st));
    if (d_dtype == SM_F64 && a_dtype == SM_F32) k_dot<double, float><<<1, 1024, 0, st>>>(n_vals, (const double *)P_vals, (const float *)S_vals, trace_ps);
    else if (d_dtype == SM_F64) k_dot<double, double><<<1, 1024, 0, st>>>(n_vals, (const double *)P_vals, (const double *)S_vals, trace_ps);
    else if (a_dtype == SM_F32) k_dot<float, float><<<1, 1024, 0, st>>>(n_vals, (const float *)P_vals, (const float *)S_vals, trace_ps);
    else k_dot<float, double><<<1, 1024, 0, st>>>(n_vals, (const float *)P_vals, (const double *)S_vals, trace_ps);
    SM_LAUNCHED();
  }
  return SM_OK;
}
