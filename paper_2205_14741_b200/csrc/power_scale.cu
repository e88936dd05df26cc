// SM_SCALE_POWER (reading A10): tighten the Gershgorin scale by a few power steps.
// X holds X0 = (T - mu I) / s_G.  v0[r] = 0.25 + hash(r); 16 steps v <- X v / ||X v||_2;
// rho_est = ||X v||_2 / ||v||_2 at the last step (a lower bound on rho(X0) for symmetric X0);
// ratio = min(1, 1.05 * rho_est); scale <- scale * ratio (the caller gathers again with the new
// scale, so X0 is rounded to the working type only once).  Newton-Schulz converges
// for |x| < sqrt(3), so an underestimate of up to ~40 % is harmless.
#include "common.cuh"

namespace sm {

constexpr int POWER_STEPS = 16;

template <typename TX, bool IMG>
__device__ inline float px_load(const TX *Xs, int32_t Pd, int32_t r, int32_t c) {
  return (float)to_double<TX>(IMG ? Xs[img_off(Pd, r, c)] : Xs[(int64_t)r * Pd + c]);
}

// One CTA per listed column; dynamic smem: float v[Pd], w[Pd], red[64].
template <typename TX, bool IMG>
__global__ void k_power_scale(const int32_t *__restrict__ cols, const int64_t *__restrict__ col_off,
                              const int32_t *__restrict__ dim, const int32_t *__restrict__ dim_pad,
                              TX *__restrict__ X, double *__restrict__ scale, double *__restrict__ ratio) {
  extern __shared__ float smem_f[];
  const int32_t c = blockIdx.x, i = cols ? cols[c] : c;
  const int32_t m = dim[i], Pd = dim_pad[i];
  float *v = smem_f, *w = smem_f + Pd, *red = smem_f + 2 * Pd;
  for (int32_t r = m + threadIdx.x; r < Pd; r += blockDim.x) { v[r] = 0.f; w[r] = 0.f; }
  TX *Xs = X + col_off[c];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int32_t r = threadIdx.x; r < m; r += blockDim.x) {
    uint32_t h = ((uint32_t)r * 2654435761u) >> 8;
    v[r] = 0.25f + (float)(h & 0xFFFFu) * (1.0f / 65536.0f);
  }
  __syncthreads();
  float rho = 0.f;
  for (int step = 0; step < POWER_STEPS; ++step) {
    // w = X v : one warp per row (X symmetric; rows are contiguous 128-byte runs in either layout)
    for (int32_t r = wid; r < m; r += nw) {
      float acc = 0.f;
      if (IMG) {
        // 16-byte chunks of 8 elements; padding columns of X are zero, v is zero-filled up to Pd
        for (int32_t ch = lane; ch * 8 < m; ch += 32) {
          const uint4 q4 = *reinterpret_cast<const uint4 *>(Xs + img_off(Pd, r, ch * 8));
          const TX *e = reinterpret_cast<const TX *>(&q4);
#pragma unroll
          for (int k = 0; k < 8; ++k) acc += (float)to_double<TX>(e[k]) * v[ch * 8 + k];
        }
      } else {
        for (int32_t cc = lane; cc < m; cc += 32) acc += px_load<TX, IMG>(Xs, Pd, r, cc) * v[cc];
      }
      for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
      if (lane == 0) w[r] = acc;
    }
    __syncthreads();
    float nv = 0.f, nwv = 0.f;
    for (int32_t r = threadIdx.x; r < m; r += blockDim.x) { nv += v[r] * v[r]; nwv += w[r] * w[r]; }
    for (int d = 16; d > 0; d >>= 1) {
      nv += __shfl_xor_sync(0xffffffffu, nv, d);
      nwv += __shfl_xor_sync(0xffffffffu, nwv, d);
    }
    if (lane == 0) { red[wid] = nv; red[32 + wid] = nwv; }
    __syncthreads();
    float sv = 0.f, sw = 0.f;
    for (int k = 0; k < nw; ++k) { sv += red[k]; sw += red[32 + k]; }
    rho = sqrtf(sw / fmaxf(sv, 1e-30f));
    float inv = rsqrtf(fmaxf(sw, 1e-30f));
    __syncthreads();
    for (int32_t r = threadIdx.x; r < m; r += blockDim.x) v[r] = w[r] * inv;
    __syncthreads();
  }
  float rt = fminf(1.0f, 1.05f * rho);
  if (!(rt > 1e-6f)) rt = 1.0f;
  if (threadIdx.x == 0) { ratio[c] = (double)rt; scale[c] *= (double)rt; }
}

template <typename TX, bool IMG>
static int32_t launch_power(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off,
                            void *X, double *scale, double *ratio, cudaStream_t st) {
  size_t smem = (size_t)(2 * P->max_dim_pad + 64) * sizeof(float);
  k_power_scale<TX, IMG><<<n_cols, 512, smem, st>>>(cols, col_off, P->dim, P->dim_pad, (TX *)X, scale, ratio);
  SM_LAUNCHED();
  return SM_OK;
}

int32_t power_scale(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off,
                    int32_t x_dtype, void *X, double *scale, double *ratio, cudaStream_t st) {
  switch (x_dtype) {
    case SM_F64: return launch_power<double, false>(P, cols, n_cols, col_off, X, scale, ratio, st);
    case SM_F32: return launch_power<float, false>(P, cols, n_cols, col_off, X, scale, ratio, st);
    case SM_BF16: return launch_power<__nv_bfloat16, true>(P, cols, n_cols, col_off, X, scale, ratio, st);
    case SM_F16: return launch_power<__half, true>(P, cols, n_cols, col_off, X, scale, ratio, st);
    default: return SM_ERR_UNSUPPORTED;
  }
}

}  // namespace sm
