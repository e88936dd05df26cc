// Per-submatrix iteration state shared by the two Newton-Schulz back ends (sign_simt.cu: FFMA/DFMA,
// sign_umma.cu: tcgen05).  Stopping rule = DESIGN.md reading A11: at step k compute Y = X_k^2 and
// r_k = ||Y - I||_F / sqrt(m); always apply the update; stop after it if r_k < tol.
#pragma once
#include "common.cuh"

namespace sm {

struct SignState {
  int32_t *active;     // [n_cols] 1 while the submatrix still iterates
  int32_t *last;       // [n_cols] 1 if the update being applied is the final one
  int32_t *n_still;    // [1] submatrices that will continue after the current update
  double *partial;     // [n_cols * parts_per_col] fused ||Y - I||_F^2 partial sums (fixed order)
  int32_t parts_per_col;
};

static __global__ void k_sign_init(int32_t n_cols, int32_t *active, int32_t *last, int32_t *iters,
                                   double *residual) {
  int32_t c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_cols) return;
  active[c] = 1; last[c] = 0; iters[c] = 0; residual[c] = 0.0;
}

// Runs between the Y = X^2 product and the update product of one iteration.  One warp per listed
// column: the n_parts[c] partial sums are added lane-strided and then by a fixed shuffle tree, so the
// result does not depend on scheduling (deterministic), and a column costs ~n_parts/32 loads per lane.
static __global__ void k_sign_post(int32_t n_cols, const int32_t *__restrict__ cols,
                                   const int32_t *__restrict__ dim, SignState s,
                                   const int32_t *__restrict__ n_parts, double tol, int32_t *iters,
                                   double *residual) {
  const int32_t c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (c >= n_cols) return;
  if (s.last[c]) {
    __syncwarp();
    if (lane == 0) { s.active[c] = 0; s.last[c] = 0; }
    return;
  }
  if (!s.active[c]) return;
  const double *p = s.partial + (int64_t)c * s.parts_per_col;
  double sum = 0.0;
  const int32_t np = n_parts[c];
  for (int32_t t = lane; t < np; t += 32) sum += p[t];
  for (int d = 16; d > 0; d >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, d);
  if (lane == 0) {
    const int32_t i = cols ? cols[c] : c;
    const double r = sqrt(sum / (double)dim[i]);
    residual[c] = r;
    iters[c] += 1;
    const bool fin = (tol > 0.0) && (r < tol);
    s.last[c] = fin ? 1 : 0;
    if (!fin) atomicAdd(s.n_still, 1);
  }
}

// After the loop: a submatrix that received an odd number of updates has its result in the
// alternate buffer; copy it back (whole padded image, 16-byte vectors).
static __global__ void k_copy_back(const int32_t *__restrict__ cols, const int64_t *__restrict__ col_off,
                                   const int32_t *__restrict__ iters, int32_t elem_bytes,
                                   const int32_t *__restrict__ dim_pad, int32_t skip_pd,
                                   const char *__restrict__ alt, char *__restrict__ X) {
  int32_t c = blockIdx.x;
  if ((iters[c] & 1) == 0) return;
  if (skip_pd > 0 && dim_pad[cols ? cols[c] : c] <= skip_pd) return;   // iterated in place by another kernel
  int64_t b0 = col_off[c] * elem_bytes, b1 = col_off[c + 1] * elem_bytes;
  int64_t n16 = (b1 - b0) >> 4;
  const uint4 *src = reinterpret_cast<const uint4 *>(alt + b0);
  uint4 *dst = reinterpret_cast<uint4 *>(X + b0);
  for (int64_t e = (int64_t)blockIdx.y * blockDim.x + threadIdx.x; e < n16; e += (int64_t)gridDim.y * blockDim.x)
    dst[e] = src[e];
  if (blockIdx.y == 0) {   // tail bytes (only when Pd*Pd*elem_bytes is not a multiple of 16)
    int64_t done = n16 << 4;
    for (int64_t e = b0 + done + threadIdx.x; e < b1; e += blockDim.x) X[e] = alt[e];
  }
}

}  // namespace sm
