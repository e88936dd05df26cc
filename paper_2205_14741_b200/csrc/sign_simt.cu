// a3, fp32 / fp64 back end: Newton-Schulz X <- 1/2 X (3I - X^2) on row-major packed submatrices
// with FFMA / DFMA register-tiled products (tcgen05 has no fp32/fp64 kind).  PAPER.md:87 (Eq. 13),
// :110 (step 2); iteration and stopping rule: DESIGN.md readings A9, A11.
#include "sign_state.cuh"

namespace sm {

constexpr int ST = 64;    // output tile edge
constexpr int SK = 16;    // k step
constexpr int SPAD = 4;

// PHASE 1: Y = X X, partial ||Y - I||_F^2.   PHASE 2: X' = 1.5 X - 0.5 X Y.   PHASE 3: O = X Y (plain product, f2; the
// third product X' = X Z of the order-3 iteration).   PHASE 4 (order 3, reading A22; Xsrc = Y): Z = (15 I - 10 Y + 3 Y Y) / 8.
template <typename T, int PHASE>
__global__ void __launch_bounds__(256)
k_simt_gemm(const int32_t *__restrict__ cols, const int64_t *__restrict__ col_off,
            const int32_t *__restrict__ dim, const int32_t *__restrict__ dim_pad, int32_t max_tiles_edge,
            const T *__restrict__ Xsrc, const T *__restrict__ Ybuf, T *__restrict__ Out, SignState s) {
  const int32_t tiles_per = max_tiles_edge * max_tiles_edge;
  const int32_t c = blockIdx.x / tiles_per, t = blockIdx.x - c * tiles_per;
  if (!s.active[c]) return;
  if (PHASE == 1 && s.last[c]) return;
  const int32_t i = cols ? cols[c] : c;
  const int32_t m = dim[i], Pd = dim_pad[i];
  const int32_t te = (m + ST - 1) / ST;
  const int32_t tr = t / max_tiles_edge, tc = t - tr * max_tiles_edge;
  if (tr >= te || tc >= te) return;
  const T *A = Xsrc + col_off[c];
  const T *B = ((PHASE == 1 || PHASE == 4) ? Xsrc : Ybuf) + col_off[c];
  T *O = Out + col_off[c];

  __shared__ T As[SK][ST + SPAD];
  __shared__ T Bs[SK][ST + SPAD];
  const int32_t tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int32_t row0 = tr * ST, col0 = tc * ST;
  T acc[4][4];
#pragma unroll
  for (int a = 0; a < 4; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) acc[a][b] = (T)0;

  // Register-staged software pipeline: the global loads of k tile t + 1 are issued before the FMAs of tile t and
  // written to shared memory after them, so their latency overlaps the arithmetic (same summation order as a
  // plain loop: results are bit-identical).
  T ra[4], rb[4];
  auto gload = [&](int32_t k0) {
    // A tile: 64 rows x 16 k (row-major source: k contiguous)
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      int32_t e = threadIdx.x + l * 256;
      int32_t r = e >> 4, k = e & 15;
      int32_t gr = row0 + r, gk = k0 + k;
      ra[l] = (gr < m && gk < m) ? A[(int64_t)gr * Pd + gk] : (T)0;
    }
    // B tile: 16 k x 64 cols (column contiguous)
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      int32_t e = threadIdx.x + l * 256;
      int32_t k = e >> 6, cc = e & 63;
      int32_t gk = k0 + k, gc = col0 + cc;
      rb[l] = (gk < m && gc < m) ? B[(int64_t)gk * Pd + gc] : (T)0;
    }
  };
  auto sstore = [&]() {
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      int32_t e = threadIdx.x + l * 256;
      As[e & 15][e >> 4] = ra[l];
      Bs[e >> 6][e & 63] = rb[l];
    }
  };
  gload(0);
  sstore();
  __syncthreads();
  for (int32_t k0 = 0; k0 < m; k0 += SK) {
    const bool more = k0 + SK < m;
    if (more) gload(k0 + SK);
#pragma unroll
    for (int k = 0; k < SK; ++k) {
      T a[4], b[4];
#pragma unroll
      for (int q = 0; q < 4; ++q) { a[q] = As[k][ty * 4 + q]; b[q] = Bs[k][tx * 4 + q]; }
#pragma unroll
      for (int q = 0; q < 4; ++q)
#pragma unroll
        for (int p = 0; p < 4; ++p) acc[q][p] += a[q] * b[p];
    }
    __syncthreads();
    if (more) sstore();
    __syncthreads();
  }

  double res = 0.0;
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    int32_t gr = row0 + ty * 4 + q;
#pragma unroll
    for (int p = 0; p < 4; ++p) {
      int32_t gc = col0 + tx * 4 + p;
      if (gr < m && gc < m) {
        if (PHASE == 3) {
          O[(int64_t)gr * Pd + gc] = acc[q][p];
        } else if (PHASE == 4) {
          O[(int64_t)gr * Pd + gc] = (T)0.375 * acc[q][p] - (T)1.25 * A[(int64_t)gr * Pd + gc] + (gr == gc ? (T)1.875 : (T)0);
        } else if (PHASE == 1) {
          O[(int64_t)gr * Pd + gc] = acc[q][p];
          double d = (double)acc[q][p] - (gr == gc ? 1.0 : 0.0);
          res += d * d;
        } else {
          T x = A[(int64_t)gr * Pd + gc];
          O[(int64_t)gr * Pd + gc] = (T)1.5 * x - (T)0.5 * acc[q][p];
        }
      }
    }
  }
  if (PHASE == 1) {
    // fixed-order CTA reduction: warp shuffles, then 8 warp sums in order
    __shared__ double red[8];
    for (int d = 16; d > 0; d >>= 1) res += __shfl_xor_sync(0xffffffffu, res, d);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = res;
    __syncthreads();
    if (threadIdx.x == 0) {
      double sum = 0.0;
      for (int w = 0; w < 8; ++w) sum += red[w];
      s.partial[(int64_t)c * s.parts_per_col + tr * te + tc] = sum;
    }
  }
}

// ---- fp64 on the tensor cores: warp-level DMMA (mma.sync.m8n8k4.f64), the only fp64 tensor path sm_100a
// has (tcgen05 has no f64 kind).  128 x 128 output tile per CTA, 8 warps as 4 x 2, warp tile 32 x 64 =
// 4 x 8 m8n8 accumulators; operands staged by 16-byte cp.async into a double-buffered ring:
//   As[128][20]  rows of X, k contiguous (LD = 20: the fragment read row*20 + k is bank-conflict free)
//   Bs[16][132]  rows k of X (PHASE 1) or Y (PHASE 2), n contiguous (true product, no transposition).
// Padding rows/columns of X, Y and the alternate buffer hold zeros (gather / memset), so loads are only
// bounded by the padded dimension.
// TILE = 128 (8 warps as 4 x 2, warp tile 32 x 64) for large submatrices, TILE = 64 (warp tile 16 x 32) where 128-row tiles
// would mostly multiply padding (m ~ 186 pads to 2 x 2 tiles of 128 = 1.9x the work; to 3 x 3 tiles of 64 = 1.07x).
constexpr int DT = 128, DK = 16, DLA = 20;
template <int TILE> struct DCfg {
  static constexpr int LB = TILE + 4;
  static constexpr int STAGE_DOUBLES = TILE * DLA + DK * LB;
  static constexpr int SMEM = 2 * STAGE_DOUBLES * 8;
};
constexpr int DMMA_SMEM = DCfg<128>::SMEM;

__device__ __forceinline__ void dmma_m8n8k4(double (&d)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
               : "+d"(d[0]), "+d"(d[1])
               : "d"(a), "d"(b));
}
__device__ __forceinline__ void cp_async16(void *smem, const void *gmem, bool valid) {
  uint32_t sa = (uint32_t)__cvta_generic_to_shared(smem);
  int32_t n = valid ? 16 : 0;                       // src-size 0: the 16 bytes are zero-filled
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(sa), "l"(gmem), "r"(n) : "memory");
}

template <int PHASE, bool SYM, int TILE = 128>
__global__ void __launch_bounds__(256)
k_dmma_gemm(const int32_t *__restrict__ cols, const int64_t *__restrict__ col_off,
            const int32_t *__restrict__ dim, const int32_t *__restrict__ dim_pad, int32_t max_tiles_edge,
            const double *__restrict__ Xsrc, const double *__restrict__ Ybuf, double *__restrict__ Out,
            SignState s) {
  extern __shared__ double dsm[];
  const int32_t tiles_per = max_tiles_edge * max_tiles_edge;
  const int32_t c = blockIdx.x / tiles_per, t = blockIdx.x - c * tiles_per;
  if (!s.active[c]) return;
  if (PHASE == 1 && s.last[c]) return;
  const int32_t i = cols ? cols[c] : c;
  const int32_t m = dim[i], Pd = dim_pad[i];
  constexpr int DLB = DCfg<TILE>::LB, DMMA_STAGE_DOUBLES = DCfg<TILE>::STAGE_DOUBLES;
  constexpr int NA = TILE / 32, NB = TILE / 16;                 // m8n8 accumulators per warp: NA x NB
  const int32_t te = (m + TILE - 1) / TILE;
  const int32_t tr = t / max_tiles_edge, tc = t - tr * max_tiles_edge;
  if (tr >= te || tc >= te || (SYM && tc > tr)) return;       // SYM: lower-triangle tiles only
  const double *A = Xsrc + col_off[c];
  const double *B = ((PHASE == 1 || PHASE == 4) ? Xsrc : Ybuf) + col_off[c];
  double *O = Out + col_off[c];
  const int32_t row0 = tr * TILE, col0 = tc * TILE;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int wr = (warp >> 1) * (TILE / 4), wc = (warp & 1) * (TILE / 2);      // warp tile origin inside the CTA tile
  const int g = lane >> 2, q = lane & 3;

  double acc[NA][NB][2];
#pragma unroll
  for (int a = 0; a < NA; ++a)
#pragma unroll
    for (int b = 0; b < NB; ++b) acc[a][b][0] = acc[a][b][1] = 0.0;

  auto load_stage = [&](int st, int32_t k0) {
    double *As = dsm + st * DMMA_STAGE_DOUBLES, *Bs = As + TILE * DLA;
    // A: TILE rows x 8 chunks of 2 doubles
#pragma unroll
    for (int l = 0; l < TILE / 32; ++l) {
      int e = threadIdx.x + l * 256;
      int r = e >> 3, ch = e & 7;
      int32_t gr = row0 + r, gk = k0 + ch * 2;
      bool ok = gr < Pd && gk < Pd;
      cp_async16(As + r * DLA + ch * 2, ok ? A + (int64_t)gr * Pd + gk : A, ok);
    }
    // B: 16 k rows x TILE / 2 chunks of 2 doubles
#pragma unroll
    for (int l = 0; l < TILE / 32; ++l) {
      int e = threadIdx.x + l * 256;
      int k = e / (TILE / 2), ch = e % (TILE / 2);
      int32_t gk = k0 + k, gc = col0 + ch * 2;
      bool ok = gk < Pd && gc < Pd;
      cp_async16(Bs + k * DLB + ch * 2, ok ? B + (int64_t)gk * Pd + gc : B, ok);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };

  const int32_t nk = (m + DK - 1) / DK;
  load_stage(0, 0);
  for (int32_t kc = 0; kc < nk; ++kc) {
    if (kc + 1 < nk) {
      load_stage((kc + 1) & 1, (kc + 1) * DK);
      asm volatile("cp.async.wait_group 1;" ::: "memory");
    } else {
      asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
    __syncthreads();
    const double *As = dsm + (kc & 1) * DMMA_STAGE_DOUBLES, *Bs = As + TILE * DLA;
#pragma unroll
    for (int k4 = 0; k4 < DK; k4 += 4) {
      double af[NA], bf[NB];
#pragma unroll
      for (int a = 0; a < NA; ++a) af[a] = As[(wr + a * 8 + g) * DLA + k4 + q];
#pragma unroll
      for (int b = 0; b < NB; ++b) bf[b] = Bs[(k4 + q) * DLB + wc + b * 8 + g];
#pragma unroll
      for (int a = 0; a < NA; ++a)
#pragma unroll
        for (int b = 0; b < NB; ++b) dmma_m8n8k4(acc[a][b], af[a], bf[b]);
    }
    __syncthreads();
  }

  // epilogue: lane holds C[row = g][cols 2q, 2q+1] of every 8 x 8 accumulator.  SYM: X is symmetric and so are
  // Y = X X and X' = p(X): only tiles with tc <= tr are computed, an element (r, c <= r) is stored at
  // (r, c) and mirrored to (c, r), which keeps the iterates exactly symmetric; off-diagonal elements
  // count twice in the residual.
  double res = 0.0;
#pragma unroll
  for (int a = 0; a < NA; ++a) {
    const int32_t gr = row0 + wr + a * 8 + g;
#pragma unroll
    for (int b = 0; b < NB; ++b) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int32_t gc = col0 + wc + b * 8 + 2 * q + e;
        if (gr < m && (SYM ? gc <= gr : gc < m)) {
          double val = acc[a][b][e];
          if (PHASE == 1) {
            const double d = val - (gr == gc ? 1.0 : 0.0);
            res += ((!SYM || gr == gc) ? 1.0 : 2.0) * d * d;
          } else if (PHASE == 2) {
            val = 1.5 * A[(int64_t)gr * Pd + gc] - 0.5 * val;
          } else if (PHASE == 4) {
            val = 0.375 * val - 1.25 * A[(int64_t)gr * Pd + gc] + (gr == gc ? 1.875 : 0.0);
          }
          O[(int64_t)gr * Pd + gc] = val;
          if (SYM && gc < gr) O[(int64_t)gc * Pd + gr] = val;
        }
      }
    }
  }
  if (PHASE == 1) {
    __shared__ double red[8];
    for (int d = 16; d > 0; d >>= 1) res += __shfl_xor_sync(0xffffffffu, res, d);
    if (lane == 0) red[warp] = res;
    __syncthreads();
    if (threadIdx.x == 0) {
      double sum = 0.0;
      for (int w = 0; w < 8; ++w) sum += red[w];
      s.partial[(int64_t)c * s.parts_per_col + tr * te + tc] = sum;
    }
  }
}

// ---- fp32, symmetric iterates: 64 x 64 tiles, 8 x 8 register blocks, cp.async double buffering -------------------
// X and Y are symmetric (exactly: only tiles with tc <= tr are computed and every element (r, c <= r) is stored at (r, c)
// and mirrored to (c, r)), so BOTH operands of a tile can be read as rows k with the tile's rows / columns contiguous:
// A[m][k] = X[k][row0 + m], B[k][n] = B[k][col0 + n] -- 16-byte cp.async without a transposition.  64 threads per
// CTA, thread (ty, tx) of an 8 x 8 grid owns rows ty * 8 .. and columns tx * 8 .. (64 independent FFMA chains per k for
// four 128-bit shared loads), many CTAs per SM.  Against k_simt_gemm (all tiles, 4 x 4 blocks, scalar bounds-checked
// loads, two __syncthreads per 16 k: 0.27 of the FFMA peak at configs[1]) this halves the tiles
// and raises the FFMA share of the issue slots.  Padding rows / columns of X, Y and the alternate buffer are zero
// (gather / memset), so loads are bounded by the padded dimension only.
constexpr int FT = 64, FK = 16;

template <int PHASE>
__global__ void __launch_bounds__(64)
k_ffma_sym(const int32_t *__restrict__ cols, const int64_t *__restrict__ col_off,
           const int32_t *__restrict__ dim, const int32_t *__restrict__ dim_pad, int32_t max_tiles_edge,
           const float *__restrict__ Xsrc, const float *__restrict__ Ybuf, float *__restrict__ Out, SignState s) {
  const int32_t tiles_per = max_tiles_edge * max_tiles_edge;
  const int32_t c = blockIdx.x / tiles_per, t = blockIdx.x - c * tiles_per;
  if (!s.active[c]) return;
  if (PHASE == 1 && s.last[c]) return;
  const int32_t i = cols ? cols[c] : c;
  const int32_t m = dim[i], Pd = dim_pad[i];
  const int32_t te = (m + FT - 1) / FT;
  const int32_t tr = t / max_tiles_edge, tc = t - tr * max_tiles_edge;
  if (tr >= te || tc > tr) return;                              // lower-triangle tiles only
  const float *A = Xsrc + col_off[c];
  const float *B = ((PHASE == 1 || PHASE == 4) ? Xsrc : Ybuf) + col_off[c];
  float *O = Out + col_off[c];
  const int32_t row0 = tr * FT, col0 = tc * FT;
  __shared__ __align__(16) float As[2][FK][FT];
  __shared__ __align__(16) float Bs[2][FK][FT];
  const int tx = threadIdx.x & 7, ty = threadIdx.x >> 3;

  auto load_stage = [&](int st, int32_t k0) {
    // 16 k rows x 16 chunks of 4 floats, for A (columns row0 ..) and B (columns col0 ..): 4 + 4 copies per thread
#pragma unroll
    for (int l = 0; l < 4; ++l) {
      const int e = threadIdx.x + l * 64, k = e >> 4, ch = e & 15;
      const int32_t gk = k0 + k, ga = row0 + ch * 4, gb = col0 + ch * 4;
      const bool oka = gk < Pd && ga < Pd, okb = gk < Pd && gb < Pd;
      cp_async16(&As[st][k][ch * 4], oka ? A + (int64_t)gk * Pd + ga : A, oka);
      cp_async16(&Bs[st][k][ch * 4], okb ? B + (int64_t)gk * Pd + gb : B, okb);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };

  float acc[8][8];
#pragma unroll
  for (int a = 0; a < 8; ++a)
#pragma unroll
    for (int b = 0; b < 8; ++b) acc[a][b] = 0.f;

  const int32_t nk = (m + FK - 1) / FK;
  load_stage(0, 0);
  for (int32_t kc = 0; kc < nk; ++kc) {
    if (kc + 1 < nk) {
      load_stage((kc + 1) & 1, (kc + 1) * FK);
      asm volatile("cp.async.wait_group 1;" ::: "memory");
    } else {
      asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
    __syncthreads();
    const int st = kc & 1;
#pragma unroll
    for (int k = 0; k < FK; ++k) {
      const float4 a0 = *reinterpret_cast<const float4 *>(&As[st][k][ty * 8]);
      const float4 a1 = *reinterpret_cast<const float4 *>(&As[st][k][ty * 8 + 4]);
      const float4 b0 = *reinterpret_cast<const float4 *>(&Bs[st][k][tx * 8]);
      const float4 b1 = *reinterpret_cast<const float4 *>(&Bs[st][k][tx * 8 + 4]);
      const float av[8] = {a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w};
      const float bv[8] = {b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w};
#pragma unroll
      for (int a = 0; a < 8; ++a)
#pragma unroll
        for (int b = 0; b < 8; ++b) acc[a][b] = fmaf(av[a], bv[b], acc[a][b]);
    }
    __syncthreads();
  }

  double res = 0.0;
#pragma unroll
  for (int a = 0; a < 8; ++a) {
    const int32_t gr = row0 + ty * 8 + a;
#pragma unroll
    for (int b = 0; b < 8; ++b) {
      const int32_t gc = col0 + tx * 8 + b;
      if (gr < m && gc <= gr) {
        float val = acc[a][b];
        if (PHASE == 1) {
          const double d = (double)val - (gr == gc ? 1.0 : 0.0);
          res += (gr == gc ? 1.0 : 2.0) * d * d;
        } else if (PHASE == 2) {
          val = 1.5f * A[(int64_t)gr * Pd + gc] - 0.5f * val;
        } else if (PHASE == 4) {
          val = 0.375f * val - 1.25f * A[(int64_t)gr * Pd + gc] + (gr == gc ? 1.875f : 0.f);
        }
        O[(int64_t)gr * Pd + gc] = val;
        if (gc < gr) O[(int64_t)gc * Pd + gr] = val;
      }
    }
  }
  if (PHASE == 1) {
    __shared__ double red[2];
    for (int d = 16; d > 0; d >>= 1) res += __shfl_xor_sync(0xffffffffu, res, d);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = res;
    __syncthreads();
    if (threadIdx.x == 0) s.partial[(int64_t)c * s.parts_per_col + tr * te + tc] = red[0] + red[1];
  }
}

static __global__ void k_tile_nparts(int32_t n_cols, int32_t T, const int32_t *__restrict__ cols,
                                     const int32_t *__restrict__ dim, int32_t *__restrict__ n_parts) {
  int32_t c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_cols) return;
  int32_t te = (dim[cols ? cols[c] : c] + T - 1) / T;
  n_parts[c] = te * te;
}

struct SimtWs {
  void *Y, *X2; int32_t *active, *last, *n_still, *n_parts; double *partial; int32_t parts_per_col;
  int64_t used;
};

static SimtWs simt_layout(void *ws, int64_t ws_bytes, const sm_pattern_t *P, int32_t n_cols,
                          int64_t packed_elems, int32_t eb) {
  WsCursor cur(ws, ws_bytes);
  SimtWs w;
  int32_t edge = (P->max_dim + ST - 1) / ST;
  w.parts_per_col = edge * edge;
  w.Y = cur.take<char>(packed_elems * eb);
  w.X2 = cur.take<char>(packed_elems * eb);
  w.active = cur.take<int32_t>(n_cols);
  w.last = cur.take<int32_t>(n_cols);
  w.n_still = cur.take<int32_t>(1);
  w.n_parts = cur.take<int32_t>(n_cols);
  w.partial = cur.take<double>((int64_t)n_cols * w.parts_per_col);
  w.used = cur.used + 256;
  return w;
}

int64_t sign_simt_ws_bytes(const sm_pattern_t *P, int32_t n_cols, int64_t packed_elems, int32_t x_dtype) {
  return simt_layout(nullptr, 0, P, n_cols, packed_elems, dtype_bytes(x_dtype)).used;
}

// Which product kernel a call uses (one choice per call, every phase).
enum SimtMode { M_GENERIC = 0, M_DMMA_FULL, M_DMMA_SYM64, M_DMMA_SYM128, M_FFMA_SYM };

template <int PHASE>
static int32_t dmma_attrs() {
  // per device attribute: set on every call (a process may use several devices)
  SM_CUDA(cudaFuncSetAttribute(k_dmma_gemm<PHASE, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, DMMA_SMEM));
  SM_CUDA(cudaFuncSetAttribute(k_dmma_gemm<PHASE, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, DMMA_SMEM));
  SM_CUDA(cudaFuncSetAttribute(k_dmma_gemm<PHASE, true, 64>, cudaFuncAttributeMaxDynamicSharedMemorySize, DCfg<64>::SMEM));
  return SM_OK;
}

template <typename T, int PHASE>
static int32_t launch_simt(int mode, int32_t grid, int32_t edge, const sm_pattern_t *P, const int32_t *cols,
                           const int64_t *col_off, const T *A, const T *B, T *O, SignState s, cudaStream_t st) {
  int slot = -1;
  { int32_t rc = prof_begin(st, &slot); if (rc != SM_OK) return rc; }
  bool done = false;
  if constexpr (sizeof(T) == 8) {
    if (mode == M_DMMA_FULL) {
      k_dmma_gemm<PHASE, false><<<grid, 256, DMMA_SMEM, st>>>(cols, col_off, P->dim, P->dim_pad, edge, A, B, O, s);
      done = true;
    } else if (mode == M_DMMA_SYM64) {
      k_dmma_gemm<PHASE, true, 64><<<grid, 256, DCfg<64>::SMEM, st>>>(cols, col_off, P->dim, P->dim_pad, edge, A, B, O, s);
      done = true;
    } else if (mode == M_DMMA_SYM128) {
      k_dmma_gemm<PHASE, true><<<grid, 256, DMMA_SMEM, st>>>(cols, col_off, P->dim, P->dim_pad, edge, A, B, O, s);
      done = true;
    }
  } else {
    if (mode == M_FFMA_SYM) {
      k_ffma_sym<PHASE><<<grid, 64, 0, st>>>(cols, col_off, P->dim, P->dim_pad, edge, A, B, O, s);
      done = true;
    }
  }
  if (!done) k_simt_gemm<T, PHASE><<<grid, 256, 0, st>>>(cols, col_off, P->dim, P->dim_pad, edge, A, B, O, s);
  SM_LAUNCHED();
  return prof_end(st, slot);
}

// order 2: Newton-Schulz, two products per step (Y = X X; X' = 1.5 X - 0.5 X Y), X alternates between X and ws.X2.
// order 3 (f3, reading A22; symmetric iterates only): three products per step on the same three buffers --
//   Y = X X -> the buffer X' will be written to;  Z = (15 I - 10 Y + 3 Y Y) / 8 -> ws.X2;  X' = X Z over the dead Y;
// X alternates between X and ws.Y.
template <typename T>
static int32_t sign_simt_t(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off,
                           int64_t packed_elems, T *X, void *ws, int64_t ws_bytes, int32_t max_iter,
                           double tol, int32_t *iters, double *residual, int32_t nonsym, int32_t order, cudaStream_t st) {
  if ((P->pad_to & 3) != 0) return SM_ERR_ARG;   // 16-byte alignment of every submatrix
  if (order == 3 && nonsym) return SM_ERR_UNSUPPORTED;
  SimtWs w = simt_layout(ws, ws_bytes, P, n_cols, packed_elems, (int32_t)sizeof(T));
  if (w.used > ws_bytes) return SM_ERR_SPACE;
  SignState s{w.active, w.last, w.n_still, w.partial, w.parts_per_col};
  // fp64: DMMA tensor-core tiles of 128 x 128 unless the submatrices are tiny (or option f64.simt = 1)
  const bool dmma = sizeof(T) == 8 && opt(OPT_F64_SIMT) == 0 && P->max_dim > 96;
  // fp32, symmetric iterates: lower-triangle 64 x 64 tiles with 8 x 8 register blocks (option "f32.sym", default on)
  const bool fsym = sizeof(T) == 4 && !nonsym && opt(OPT_F32_SYM) != 0 && (P->pad_to & 3) == 0;
  // fp64 tiles: 64 x 64 where 128-row tiles would mostly multiply padding (option "f64.tile": 0 = by size, 64, 128)
  const int32_t dt = !dmma ? ST : (!nonsym && (opt(OPT_F64_TILE) == 64 || (opt(OPT_F64_TILE) == 0 && P->max_dim <= 384))) ? 64 : DT;
  const int mode = dmma ? (nonsym ? M_DMMA_FULL : dt == 64 ? M_DMMA_SYM64 : M_DMMA_SYM128) : fsym ? M_FFMA_SYM : M_GENERIC;
  const int32_t TS = dt;
  const int32_t edge = (P->max_dim + TS - 1) / TS;
  const int64_t grid64 = (int64_t)n_cols * edge * edge;
  if (grid64 > 0x7fffffffLL) return SM_ERR_UNSUPPORTED;
  const int32_t grid = (int32_t)grid64, nb = (n_cols + 255) / 256;
  k_sign_init<<<nb, 256, 0, st>>>(n_cols, w.active, w.last, iters, residual);
  SM_LAUNCHED();
  k_tile_nparts<<<nb, 256, 0, st>>>(n_cols, TS, cols, P->dim, w.n_parts);
  SM_LAUNCHED();
  if (dmma) {
    int32_t rc = dmma_attrs<1>();
    if (rc == SM_OK) rc = dmma_attrs<2>();
    if (rc == SM_OK && order == 3) rc = dmma_attrs<3>();
    if (rc == SM_OK && order == 3) rc = dmma_attrs<4>();
    if (rc != SM_OK) return rc;
  }
  {
    // padding of the two scratch buffers must read as zeros (the kernels store true elements only; whole padded
    // images are copied back), and so must the partial-sum slots of the skipped upper-triangle tiles, never written
    SM_CUDA(cudaMemsetAsync(w.Y, 0, packed_elems * sizeof(T), st));
    SM_CUDA(cudaMemsetAsync(w.X2, 0, packed_elems * sizeof(T), st));
    SM_CUDA(cudaMemsetAsync(w.partial, 0, (size_t)n_cols * w.parts_per_col * sizeof(double), st));
  }
  T *buf[2] = {X, order == 3 ? (T *)w.Y : (T *)w.X2};
  for (int32_t k = 0; k < max_iter; ++k) {
    T *src = buf[k & 1], *dst = buf[(k + 1) & 1];
    T *Y = order == 3 ? dst : (T *)w.Y;
    int32_t rc = launch_simt<T, 1>(mode, grid, edge, P, cols, col_off, src, Y, Y, s, st);
    if (rc != SM_OK) return rc;
    SM_CUDA(cudaMemsetAsync(w.n_still, 0, sizeof(int32_t), st));
    k_sign_post<<<(n_cols + 7) / 8, 256, 0, st>>>(n_cols, cols, P->dim, s, w.n_parts, tol, iters, residual);
    SM_LAUNCHED();
    if (order == 3) {
      T *Z = (T *)w.X2;
      rc = launch_simt<T, 4>(mode, grid, edge, P, cols, col_off, Y, Y, Z, s, st);
      if (rc == SM_OK) rc = launch_simt<T, 3>(mode, grid, edge, P, cols, col_off, src, Z, dst, s, st);
    } else {
      rc = launch_simt<T, 2>(mode, grid, edge, P, cols, col_off, src, Y, dst, s, st);
    }
    if (rc != SM_OK) return rc;
    if (tol > 0.0 && k >= 5 && (k & 1)) {
      // convergence mode: read back how many submatrices continue (the only host sync of the path)
      int32_t still = 1;
      SM_CUDA(cudaMemcpyAsync(&still, w.n_still, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
      SM_CUDA(cudaStreamSynchronize(st));
      if (still == 0) break;
    }
  }
  dim3 cg(n_cols, 8);
  k_copy_back<<<cg, 256, 0, st>>>(cols, col_off, iters, (int32_t)sizeof(T), P->dim_pad, 0, (const char *)buf[1], (char *)X);
  SM_LAUNCHED();
  return SM_OK;
}

// O_c = A_c B_c for every listed submatrix (row-major packed buffers, zero padding; true products on all tiles).
// `active` is a device array of n_cols ones (the kernels' per-submatrix switch).  Used by sm_density_nonorth (f2).
int32_t dense_product(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off, int32_t x_dtype,
                      const void *A, const void *B, void *O, int32_t *active, int32_t *last_zero, cudaStream_t st) {
  SignState s{active, last_zero, nullptr, nullptr, 0};
  const bool dmma = x_dtype == SM_F64 && opt(OPT_F64_SIMT) == 0 && P->max_dim > 96;
  const int32_t TS = dmma ? DT : ST;
  const int32_t edge = (P->max_dim + TS - 1) / TS;
  const int64_t grid64 = (int64_t)n_cols * edge * edge;
  if (grid64 > 0x7fffffffLL) return SM_ERR_UNSUPPORTED;
  const int32_t grid = (int32_t)grid64;
  if (dmma) {
    SM_CUDA(cudaFuncSetAttribute(k_dmma_gemm<3, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, DMMA_SMEM));
    k_dmma_gemm<3, false><<<grid, 256, DMMA_SMEM, st>>>(cols, col_off, P->dim, P->dim_pad, edge, (const double *)A,
                                                        (const double *)B, (double *)O, s);
  } else if (x_dtype == SM_F64) {
    k_simt_gemm<double, 3><<<grid, 256, 0, st>>>(cols, col_off, P->dim, P->dim_pad, edge, (const double *)A, (const double *)B, (double *)O, s);
  } else if (x_dtype == SM_F32) {
    k_simt_gemm<float, 3><<<grid, 256, 0, st>>>(cols, col_off, P->dim, P->dim_pad, edge, (const float *)A, (const float *)B, (float *)O, s);
  } else {
    return SM_ERR_UNSUPPORTED;
  }
  SM_LAUNCHED();
  return SM_OK;
}

int32_t sign_simt(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off,
                  int64_t packed_elems, int32_t x_dtype, void *X, void *ws, int64_t ws_bytes,
                  int32_t max_iter, double tol, int32_t *iters, double *residual, int32_t nonsym, int32_t order,
                  cudaStream_t st) {
  if (x_dtype == SM_F64)
    return sign_simt_t<double>(P, cols, n_cols, col_off, packed_elems, (double *)X, ws, ws_bytes, max_iter,
                               tol, iters, residual, nonsym, order, st);
  if (x_dtype == SM_F32)
    return sign_simt_t<float>(P, cols, n_cols, col_off, packed_elems, (float *)X, ws, ws_bytes, max_iter,
                              tol, iters, residual, nonsym, order, st);
  return SM_ERR_UNSUPPORTED;
}

}  // namespace sm
