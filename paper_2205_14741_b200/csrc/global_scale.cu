// SM_SCALE_GLOBAL (reading A10, third option): one spectral bound for every submatrix from a short
// power iteration on the WHOLE block-sparse matrix A - mu I.
//
// Every T_i - mu I is a principal submatrix of the symmetric A - mu I ("submatrix T_i(A) for every
// column"; absent pairs inside T_i are absent in A as well), so by Cauchy interlacing its eigenvalues lie between
// the extreme eigenvalues of A - mu I: rho(T_i - mu I) <= rho(A - mu I) for all i.  GLOBAL_STEPS power steps
// v <- (A - mu I) v / ||.|| from a fixed hashed start vector give est = ||(A - mu I) v|| <= rho(A - mu I) (a lower
// bound that is within ~15 % after 10 steps on the water-like workloads); the scale is
//   s_i = min(Gershgorin_i, max(1.05 * est, est + 10 * (est - est of the step before))).
// Newton-Schulz converges for |x| < sqrt(3), so the iteration stays convergent as long as est > 0.55 rho(A - mu I).
// Compared with SM_SCALE_POWER (ten power steps on every gathered submatrix, then a second gather) this reads
// the block-CSR values ten times (0.23 GB each at configs[2]) instead of the packed images (1.3 GB each) and needs
// no second gather; the price is a scale that is ~1.2-1.4x looser than the per-submatrix one (rho(T_i) / rho(A) =
// 0.53-0.83 at configs[2]), i.e. about half a Newton-Schulz step.
#include "common.cuh"

namespace sm {

constexpr int GLOBAL_STEPS = 10;
#ifndef SM_SPMV_WARPS
#define SM_SPMV_WARPS 4
#endif
constexpr int SPMV_WARPS = SM_SPMV_WARPS;
constexpr int GLOBAL_MAX_BLK = 128;

__global__ void k_widen_blk(int32_t n, const int32_t *__restrict__ blk, int64_t *__restrict__ out) {
  int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = blk[i];
}

// v0[r] = 0.25 + hash(r) in [0.25, 1.25): no symmetry of the workload can make it orthogonal to the top eigenvector.
__global__ void k_global_init(int32_t n_blk, const int32_t *__restrict__ blk, const int64_t *__restrict__ voff,
                              double *__restrict__ v, double *__restrict__ scal) {
  int32_t i = blockIdx.x;
  for (int32_t r = threadIdx.x; r < blk[i]; r += blockDim.x) {
    const uint32_t g = (uint32_t)(voff[i] + r);
    const uint32_t h = (g * 2654435761u) >> 8;
    v[voff[i] + r] = 0.25 + (double)(h & 0xFFFFu) * (1.0 / 65536.0);
  }
  if (i == 0 && threadIdx.x == 0) { scal[0] = 1.0; scal[1] = 0.0; scal[2] = 0.0; }   // 1 / ||v||, est, previous est
}

// y = (A - mu I) (inv_norm * v) for block row i; part[i] = sum of y_r^2 over the block row.  One CTA per block
// row; a warp takes every SPMV_WARPS-th stored block and a lane owns one row of it (the 4 KB block is walked
// column by column, so every 128-byte line is fetched once and then served by L1); the per-warp partial rows
// are added in a fixed order (deterministic).
template <typename TA>
__global__ void __launch_bounds__(32 * SPMV_WARPS)
k_global_spmv(const int32_t *__restrict__ blk, const int32_t *__restrict__ rp, const int32_t *__restrict__ ci,
              const int64_t *__restrict__ vp, const TA *__restrict__ vals, double mu,
              const int64_t *__restrict__ voff, const double *__restrict__ v, const double *__restrict__ scal,
              double *__restrict__ y, double *__restrict__ part) {
  extern __shared__ double sm_y[];               // [SPMV_WARPS][slots][rps] <= [SPMV_WARPS][GLOBAL_MAX_BLK]
  const int32_t i = blockIdx.x, bi = blk[i];
  if (bi > GLOBAL_MAX_BLK) {                     // unsupported block size: poison the estimate, the caller keeps Gershgorin
    if (threadIdx.x == 0) part[i] = -1.0;
    return;
  }
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const double inv = scal[0];
  // Small blocks (round 2): with a lane per row a 6 x 6 block keeps 6 of 32 lanes busy (configs[3]: 75 us per step for 45 MB).
  // A warp is cut into `slots` groups of rps = 2^k >= bi lanes; each group takes its own stored block, so a warp walks `slots`
  // blocks at once (6-wide blocks: 4 groups of 8 lanes, 24 of 32 lanes busy).  Every (warp, slot) keeps its own partial rows;
  // they are added in a fixed order at the end: deterministic.  bi > 16: one slot, the walk of round 1.
  int32_t rps = 32;
  while (rps >= 2 * bi && rps > 1) rps >>= 1;
  const int32_t slots = 32 / rps, slot = lane / rps, row = lane - slot * rps;
  double *mine = sm_y + ((size_t)wid * slots + slot) * (bi > 32 ? bi : rps);
  for (int32_t r = row; r < bi; r += rps) mine[r] = 0.0;
  __syncwarp();
  for (int32_t p = rp[i] + wid * slots + slot; p < rp[i + 1]; p += SPMV_WARPS * slots) {
    const int32_t j = ci[p], bj = blk[j];
    const TA *blkp = vals + vp[p];
    const double *vj = v + voff[j];
    for (int32_t r = row; r < bi; r += rps) {              // a lane owns a row: no shuffles, fixed summation order
      const TA *rowp = blkp + (int64_t)r * bj;
      double s = 0.0;
#pragma unroll 8
      for (int32_t c = 0; c < bj; ++c) {
        double a = to_double<TA>(__ldg(rowp + c));
        if (j == i && c == r) a -= mu;
        s = fma(a, vj[c] * inv, s);
      }
      mine[r] += s;
    }
  }
  __syncthreads();
  double sq = 0.0;
  const int32_t stride = bi > 32 ? bi : rps, nparts = SPMV_WARPS * slots;
  for (int32_t r = threadIdx.x; r < bi; r += blockDim.x) {
    double t = 0.0;
    for (int w = 0; w < nparts; ++w) t += sm_y[(size_t)w * stride + r];
    y[voff[i] + r] = t;
    sq += t * t;
  }
  __shared__ double red[SPMV_WARPS];
  for (int d = 16; d > 0; d >>= 1) sq += __shfl_xor_sync(0xffffffffu, sq, d);
  if (lane == 0) red[wid] = sq;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < SPMV_WARPS; ++w) t += red[w];
    part[i] = t;
  }
}

// ||y||_2 from the per-block-row partial sums, one CTA, fixed summation tree: est = ||y||, next 1 / ||v|| = 1 / est.
__global__ void __launch_bounds__(1024) k_global_norm(int32_t n_blk, const double *__restrict__ part,
                                                      double *__restrict__ scal) {
  __shared__ double red[32];
  double s = 0.0;
  bool bad = false;
  for (int32_t i = threadIdx.x; i < n_blk; i += blockDim.x) { s += part[i]; bad |= part[i] < 0.0; }
  bad = __syncthreads_or(bad);
  for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) t += red[w];
    const double nrm = bad ? 0.0 : sqrt(t);      // 0: k_global_apply leaves the Gershgorin scales untouched
    scal[2] = scal[1];                           // the estimate of the step before: its growth guards the margin
    scal[1] = nrm;
    scal[0] = nrm > 0.0 ? 1.0 / nrm : 1.0;
  }
}

__global__ void k_global_apply(int32_t n_cols, const double *__restrict__ scal, double *__restrict__ scale) {
  int32_t c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_cols) return;
  // est is a LOWER bound of rho(A - mu I) that grows monotonically with the power steps.  Margin: 5 %, or ten times
  // the growth of the last step when the iteration has not settled (est still growing by more than 0.5 % per step:
  // a slowly separating spectrum) -- a geometric extrapolation of the remaining distance.  Newton-Schulz needs only
  // rho(T_i) / s_i < sqrt(3), so the scale stays safe unless est is below 0.55 rho while having all but stopped
  // growing; sm_sign_status additionally reports a diverged submatrix (non-finite or > 1 residual) in fixed-count mode.
  const double est = scal[1], grow = fmax(0.0, scal[1] - scal[2]);
  const double g = fmax(1.05 * est, est + 10.0 * grow);
  if (est > 0.0 && g < scale[c]) scale[c] = g;
}

int64_t global_scale_ws_bytes(const sm_bcsr_t *A, const sm_pattern_t *P) {
  WsCursor cur(nullptr, 0);
  cur.take<int64_t>(A->n_blk + 1);
  cur.take<double>((int64_t)A->n_blk * P->max_dim);
  cur.take<double>((int64_t)A->n_blk * P->max_dim);
  cur.take<double>(A->n_blk);
  cur.take<double>(4);
  return cur.used + 256;
}

// scale[c] (already the Gershgorin bound of listed column c) <- min(scale[c], 1.05 * est).
int32_t global_scale(const sm_bcsr_t *A, const void *A_vals, int32_t a_dtype, const sm_pattern_t *P, double mu,
                     int32_t n_cols, double *scale, void *ws, int64_t ws_bytes, cudaStream_t st) {
  const int32_t n = A->n_blk;
  WsCursor cur(ws, ws_bytes);
  int64_t *voff = cur.take<int64_t>(n + 1);
  double *v = cur.take<double>((int64_t)n * P->max_dim);       // n_blk * max block size <= n_blk * max_dim
  double *y = cur.take<double>((int64_t)n * P->max_dim);
  double *part = cur.take<double>(n);
  double *scal = cur.take<double>(4);
  if (!cur.ok()) return SM_ERR_SPACE;
  k_widen_blk<<<(n + 255) / 256, 256, 0, st>>>(n, A->blk_size, voff);
  SM_LAUNCHED();
  { int32_t rc = exclusive_scan_i64(n, voff, voff, st); if (rc != SM_OK) return rc; }
  k_global_init<<<n, 64, 0, st>>>(n, A->blk_size, voff, v, scal);
  SM_LAUNCHED();
  // per-warp partial rows: block sizes up to GLOBAL_MAX_BLK (a larger block makes k_global_spmv flag the call).
  // Kept small on purpose: the strided block walk lives on L1, and a 24 KB request per CTA (max_dim rows) left
  // so little L1 that every column step went back to L2 (measured: 350 us per step at configs[2]).
  const size_t smem = (size_t)SPMV_WARPS * GLOBAL_MAX_BLK * sizeof(double);
  for (int step = 0; step < GLOBAL_STEPS; ++step) {
    if (a_dtype == SM_F64)
      k_global_spmv<double><<<n, 32 * SPMV_WARPS, smem, st>>>(A->blk_size, A->row_ptr, A->col_idx, A->val_ptr,
                                                             (const double *)A_vals, mu, voff, v, scal, y, part);
    else
      k_global_spmv<float><<<n, 32 * SPMV_WARPS, smem, st>>>(A->blk_size, A->row_ptr, A->col_idx, A->val_ptr,
                                                            (const float *)A_vals, mu, voff, v, scal, y, part);
    SM_LAUNCHED();
    k_global_norm<<<1, 1024, 0, st>>>(n, part, scal);
    SM_LAUNCHED();
    double *t = v; v = y; y = t;
  }
  k_global_apply<<<(n_cols + 255) / 256, 256, 0, st>>>(n_cols, scal, scale);
  SM_LAUNCHED();
  return SM_OK;
}

}  // namespace sm
