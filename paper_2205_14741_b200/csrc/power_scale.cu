// SM_SCALE_POWER (reading A10): tighten the Gershgorin scale by a few power steps.
// X holds X0 = (T - mu I) / s_G.  v0[r] = 0.25 + hash(r); 10 steps v <- X v / ||X v||_2;
// rho_est = ||X v||_2 / ||v||_2 at the last step (a lower bound on rho(X0) for symmetric X0);
// ratio = min(1, 1.05 * rho_est); scale <- scale * ratio (the caller gathers again with the new
// scale, so X0 is rounded to the working type only once).  Newton-Schulz converges
// for |x| < sqrt(3), so an underestimate of up to ~40 % is harmless.
#include "common.cuh"

namespace sm {

constexpr int POWER_STEPS = 10;
constexpr int POWER_THREADS = 1024;
constexpr int POWER_UNROLL = 4;
// One CTA per SM (forced through the dynamic shared memory request): the 148 submatrices in flight
// then stay L2-resident across the power steps at the sizes of configs[1]-[3].
constexpr size_t POWER_SMEM_MIN = 120 * 1024;

// 8 consecutive elements (r, 8*ch .. 8*ch+7) as floats.
template <typename TX, bool IMG>
__device__ __forceinline__ void px_load8(const TX *Xs, int32_t Pd, int32_t r, int32_t ch, float (&f)[8]) {
  const TX *src = IMG ? Xs + img_off(Pd, r, ch * 8) : Xs + (int64_t)r * Pd + ch * 8;
  __align__(16) TX e[8];
  if (IMG || ch * 8 + 8 <= Pd) {
#pragma unroll
    for (int q = 0; q < (int)(sizeof(TX) * 8 / 16); ++q)
      reinterpret_cast<uint4 *>(e)[q] = __ldg(reinterpret_cast<const uint4 *>(src) + q);
  } else {                                   // row tail when pad_to % 8 != 0 (row-major only)
#pragma unroll
    for (int k = 0; k < 8; ++k) e[k] = ch * 8 + k < Pd ? src[k] : from_double<TX>(0.0);
  }
#pragma unroll
  for (int k = 0; k < 8; ++k) f[k] = (float)to_double<TX>(e[k]);
}

// One CTA per listed column; dynamic smem: float v[Pd], w[Pd], red[64], part[32 warps][8][32].
// X is symmetric, so w = X v is accumulated as w[c] += X[r][c] v[r]: a lane owns an 8-column chunk,
// a warp walks its rows with coalesced 512-byte row segments and POWER_UNROLL rows in flight, and no
// shuffle sits in the inner loop; the per-warp partial sums are added in a fixed order (deterministic).
template <typename TX, bool IMG>
__global__ void __launch_bounds__(POWER_THREADS, 1)
k_power_scale(const int32_t *__restrict__ cols, const int64_t *__restrict__ col_off,
              const int32_t *__restrict__ dim, const int32_t *__restrict__ dim_pad,
              TX *__restrict__ X, double *__restrict__ scale, double *__restrict__ ratio) {
  extern __shared__ float smem_f[];
  const int32_t c = blockIdx.x, i = cols ? cols[c] : c;
  const int32_t m = dim[i], Pd = dim_pad[i];
  float *v = smem_f, *w = smem_f + Pd, *red = smem_f + 2 * Pd, *part = red + 64;
  const TX *Xs = X + col_off[c];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int32_t r = threadIdx.x; r < Pd; r += blockDim.x) {
    uint32_t h = ((uint32_t)r * 2654435761u) >> 8;
    v[r] = r < m ? 0.25f + (float)(h & 0xFFFFu) * (1.0f / 65536.0f) : 0.f;
    w[r] = 0.f;
  }
  __syncthreads();
  const int32_t n_ch = (m + 7) >> 3;        // padding columns hold zeros
  float rho = 0.f;
  for (int step = 0; step < POWER_STEPS; ++step) {
    for (int32_t g0 = 0; g0 < n_ch; g0 += 32) {
      const int32_t ch = g0 + lane;
      float acc[8];
#pragma unroll
      for (int k = 0; k < 8; ++k) acc[k] = 0.f;
      if (ch < n_ch) {
        int32_t r = wid;
        for (; r + (POWER_UNROLL - 1) * nw < m; r += POWER_UNROLL * nw) {
          float f[POWER_UNROLL][8];
#pragma unroll
          for (int u = 0; u < POWER_UNROLL; ++u) px_load8<TX, IMG>(Xs, Pd, r + u * nw, ch, f[u]);
#pragma unroll
          for (int u = 0; u < POWER_UNROLL; ++u) {
            const float vr = v[r + u * nw];
#pragma unroll
            for (int k = 0; k < 8; ++k) acc[k] = fmaf(f[u][k], vr, acc[k]);
          }
        }
        for (; r < m; r += nw) {
          float f[8];
          px_load8<TX, IMG>(Xs, Pd, r, ch, f);
          const float vr = v[r];
#pragma unroll
          for (int k = 0; k < 8; ++k) acc[k] = fmaf(f[k], vr, acc[k]);
        }
      }
      // fixed-order (deterministic) reduction of the per-warp partial sums of these 256 columns
#pragma unroll
      for (int k = 0; k < 8; ++k) part[(wid * 8 + k) * 32 + lane] = acc[k];
      __syncthreads();
      if (threadIdx.x < 256) {
        const int32_t l = threadIdx.x >> 3, k = threadIdx.x & 7, col = (g0 + l) * 8 + k;
        if (col < Pd) {
          float sum = 0.f;
          for (int q = 0; q < nw; ++q) sum += part[(q * 8 + k) * 32 + l];
          w[col] = sum;
        }
      }
      __syncthreads();
    }
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
    for (int32_t r = threadIdx.x; r < Pd; r += blockDim.x) { v[r] = r < m ? w[r] * inv : 0.f; w[r] = 0.f; }
    __syncthreads();
  }
  float rt = fminf(1.0f, 1.05f * rho);
  if (!(rt > 1e-6f)) rt = 1.0f;
  if (threadIdx.x == 0) { ratio[c] = (double)rt; scale[c] *= (double)rt; }
}

template <typename TX, bool IMG>
static int32_t launch_power(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off,
                            void *X, double *scale, double *ratio, cudaStream_t st) {
  size_t smem = (size_t)(2 * P->max_dim_pad + 64 + POWER_THREADS * 8) * sizeof(float);
  if (smem < POWER_SMEM_MIN) smem = POWER_SMEM_MIN;
  if (smem > 227 * 1024) return SM_ERR_UNSUPPORTED;
  static bool configured = false;
  if (!configured) {
    SM_CUDA(cudaFuncSetAttribute(k_power_scale<TX, IMG>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024));
    configured = true;
  }
  k_power_scale<TX, IMG><<<n_cols, POWER_THREADS, smem, st>>>(cols, col_off, P->dim, P->dim_pad, (TX *)X, scale,
                                                             ratio);
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
