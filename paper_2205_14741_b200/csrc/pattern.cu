// a1: neighbour-pattern build (Fig. 2 step 1 -- "construction of a submatrix
// T_i(A) for every column").  All-integer kernels, bit-exact by construction.
#include "common.cuh"

namespace sm {

thread_local int32_t g_last_cuda_error = 0;
thread_local int64_t g_launch_count = 0;

// ---- validation + sizes -------------------------------------------------------------------
// out[0]=error flag, out[1]=gmap_len, out[2]=packed_elems, out[3]=max_dim, out[4]=max_dim_pad,
// out[5]=max_nbr
__global__ void k_validate_sizes(int32_t n, const int32_t *__restrict__ blk, const int32_t *__restrict__ rp,
                                 const int32_t *__restrict__ ci, int32_t pad_to,
                                 unsigned long long *__restrict__ out) {
  int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  int32_t lo = rp[i], hi = rp[i + 1];
  bool bad = hi < lo, diag = false;
  int64_t dim = 0;
  for (int32_t p = lo; p < hi && !bad; ++p) {
    int32_t j = ci[p];
    if (j < 0 || j >= n) { bad = true; break; }
    if (p > lo && ci[p - 1] >= j) bad = true;
    if (j == i) diag = true;
    // structural symmetry: block (j, i) must be stored
    if (find_sorted(ci, rp[j], rp[j + 1], i) < 0) bad = true;
    dim += blk[j];
  }
  if (!diag) bad = true;
  if (bad) { atomicExch(&out[0], 1ull); return; }
  int64_t cnt = hi - lo;
  int64_t dp = (dim + pad_to - 1) / pad_to * pad_to;
  atomicAdd(&out[1], (unsigned long long)(cnt * cnt));
  atomicAdd(&out[2], (unsigned long long)(dp * dp));
  atomicMax(&out[3], (unsigned long long)dim);
  atomicMax(&out[4], (unsigned long long)dp);
  atomicMax(&out[5], (unsigned long long)cnt);
}

// ---- per-column quantities ----------------------------------------------------------------
// N(i): by the validated structural symmetry the block rows storing column i are the columns
// stored in row i, so nbr_ptr/nbr_idx copy row_ptr/col_idx.
__global__ void k_dims(int32_t n, const int32_t *__restrict__ blk, const int32_t *__restrict__ rp,
                       const int32_t *__restrict__ ci, int32_t pad_to, int32_t *__restrict__ nbr_ptr,
                       int32_t *__restrict__ nbr_idx, int32_t *__restrict__ own_pos,
                       int32_t *__restrict__ dim, int32_t *__restrict__ dim_pad,
                       int32_t *__restrict__ row_off, int64_t *__restrict__ sq_dim_pad,
                       int64_t *__restrict__ sq_cnt) {
  int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i > n) return;
  if (i == n) { nbr_ptr[n] = rp[n]; return; }
  int32_t lo = rp[i], hi = rp[i + 1];
  nbr_ptr[i] = lo;
  int32_t off = 0, own = -1;
  for (int32_t p = lo; p < hi; ++p) {
    int32_t j = ci[p];
    nbr_idx[p] = j;
    row_off[p] = off;
    if (j == i) own = p - lo;
    off += blk[j];
  }
  own_pos[i] = own;
  dim[i] = off;
  int32_t dp = (off + pad_to - 1) / pad_to * pad_to;
  dim_pad[i] = dp;
  sq_dim_pad[i] = (int64_t)dp * dp;
  int64_t cnt = hi - lo;
  sq_cnt[i] = cnt * cnt;
}

// Exclusive scan of in[0..n) into out[0..n], out[n] = total.  One CTA, chunked.
__global__ void k_exclusive_scan_i64(int32_t n, const int64_t *in, int64_t *out) {  // in may alias out
  __shared__ int64_t warp_sums[32];
  __shared__ int64_t carry_s;
  if (threadIdx.x == 0) carry_s = 0;
  __syncthreads();
  const int32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  for (int32_t base = 0; base < n; base += blockDim.x) {
    int32_t i = base + threadIdx.x;
    int64_t v = (i < n) ? in[i] : 0;
    int64_t x = v;
    for (int d = 1; d < 32; d <<= 1) {
      int64_t y = __shfl_up_sync(0xffffffffu, x, d);
      if (lane >= d) x += y;
    }
    if (lane == 31) warp_sums[wid] = x;
    __syncthreads();
    if (wid == 0) {
      int64_t s = (lane < nw) ? warp_sums[lane] : 0;
      for (int d = 1; d < 32; d <<= 1) {
        int64_t y = __shfl_up_sync(0xffffffffu, s, d);
        if (lane >= d) s += y;
      }
      warp_sums[lane] = s;   // inclusive scan of warp totals
    }
    __syncthreads();
    int64_t prefix = carry_s + (wid > 0 ? warp_sums[wid - 1] : 0);
    if (i < n) out[i] = prefix + x - v;
    __syncthreads();
    if (threadIdx.x == 0) carry_s += warp_sums[nw - 1];
    __syncthreads();
  }
  if (threadIdx.x == 0) out[n] = carry_s;
}

// gather map: one CTA per block column i; entry (a, c) = stored-block index of (N(i)[a], N(i)[c]).
__global__ void k_gmap(const int32_t *__restrict__ rp, const int32_t *__restrict__ ci,
                       const int64_t *__restrict__ gmap_ptr, int32_t *__restrict__ gmap) {
  int32_t i = blockIdx.x;
  int32_t lo = rp[i], cnt = rp[i + 1] - lo;
  int64_t base = gmap_ptr[i];
  for (int32_t e = threadIdx.x; e < cnt * cnt; e += blockDim.x) {
    int32_t a = e / cnt, c = e - a * cnt;
    int32_t ja = ci[lo + a], jc = ci[lo + c];
    gmap[base + e] = find_sorted(ci, rp[ja], rp[ja + 1], jc);
  }
}

// transpose map: one CTA per block row i.
__global__ void k_tmap(const int32_t *__restrict__ rp, const int32_t *__restrict__ ci,
                       int32_t *__restrict__ tmap) {
  int32_t i = blockIdx.x;
  for (int32_t p = rp[i] + threadIdx.x; p < rp[i + 1]; p += blockDim.x) {
    int32_t j = ci[p];
    tmap[p] = find_sorted(ci, rp[j], rp[j + 1], i);
  }
}

// order: rank of i under the key (dim_pad descending, id ascending), by counting.  One CTA per
// group of block columns; O(N^2 / threads) integer compares, once per geometry.
__global__ void k_order(int32_t n, const int32_t *__restrict__ dim_pad, int32_t *__restrict__ order) {
  // eight lanes share one i: lane s counts the keys of every eighth vector of four (n threads alone left most of the
  // GPU idle: 169 us at n = 10 000), the partial ranks are added by shuffles
  const int32_t i = (blockIdx.x * blockDim.x + threadIdx.x) >> 3, s = threadIdx.x & 7;
  const bool live = i < n;
  const int32_t key = live ? dim_pad[i] : 0;
  int32_t rank = 0;
  // keys four at a time (cudaMalloc'd arrays are 16-byte aligned); j < i decides ties
  const int32_t n4 = ((reinterpret_cast<uintptr_t>(dim_pad) & 15) == 0) ? (n & ~3) : 0;
  if (live) {
    for (int32_t j = 4 * s; j < n4; j += 32) {
      const int4 k4 = __ldg(reinterpret_cast<const int4 *>(dim_pad + j));
      rank += (k4.x > key) || (k4.x == key && j < i);
      rank += (k4.y > key) || (k4.y == key && j + 1 < i);
      rank += (k4.z > key) || (k4.z == key && j + 2 < i);
      rank += (k4.w > key) || (k4.w == key && j + 3 < i);
    }
    for (int32_t j = n4 + s; j < n; j += 8) {
      const int32_t kj = __ldg(dim_pad + j);
      rank += (kj > key) || (kj == key && j < i);
    }
  }
  rank += __shfl_xor_sync(0xffffffffu, rank, 1);
  rank += __shfl_xor_sync(0xffffffffu, rank, 2);
  rank += __shfl_xor_sync(0xffffffffu, rank, 4);
  if (live && s == 0) order[rank] = i;
}

__global__ void k_plan_columns(const int32_t *__restrict__ cols, int32_t n_cols,
                               const int32_t *__restrict__ dim_pad, int64_t *__restrict__ sq) {
  int32_t c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_cols) return;
  int64_t dp = dim_pad[cols[c]];
  sq[c] = dp * dp;
}

int32_t exclusive_scan_i64(int32_t n, const int64_t *in, int64_t *out, cudaStream_t st) {
  k_exclusive_scan_i64<<<1, 1024, 0, st>>>(n, in, out);
  SM_LAUNCHED();
  return SM_OK;
}

}  // namespace sm

using namespace sm;

extern "C" int32_t sm_last_cuda_error(void) { return g_last_cuda_error; }
extern "C" int64_t sm_launch_count(void) { return g_launch_count; }

extern "C" int32_t sm_pattern_sizes(const sm_bcsr_t *A, int32_t pad_to, sm_sizes_t *out, void *scratch,
                                    void *stream) {
  if (!A || !out || !scratch || pad_to <= 0 || A->n_blk <= 0 || A->nnzb < A->n_blk) return SM_ERR_ARG;
  if (!A->blk_size || !A->row_ptr || !A->col_idx) return SM_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  unsigned long long *d = (unsigned long long *)scratch;
  SM_CUDA(cudaMemsetAsync(d, 0, 8 * sizeof(unsigned long long), st));
  int32_t n = A->n_blk;
  k_validate_sizes<<<(n + 127) / 128, 128, 0, st>>>(n, A->blk_size, A->row_ptr, A->col_idx, pad_to, d);
  SM_LAUNCHED();
  unsigned long long h[8];
  SM_CUDA(cudaMemcpyAsync(h, d, sizeof(h), cudaMemcpyDeviceToHost, st));
  SM_CUDA(cudaStreamSynchronize(st));
  if (h[0]) return SM_ERR_PATTERN;
  out->nbr_len = A->nnzb;
  out->gmap_len = (int64_t)h[1];
  out->packed_elems = (int64_t)h[2];
  out->max_dim = (int32_t)h[3];
  out->max_dim_pad = (int32_t)h[4];
  out->max_nbr = (int32_t)h[5];
  out->reserved = 0;
  out->build_ws_bytes = 2 * align_up((int64_t)(n + 1) * 8, 256) + 512;
  return SM_OK;
}

extern "C" int32_t sm_build_pattern(const sm_bcsr_t *A, int32_t pad_to, sm_pattern_t *P, void *ws,
                                    int64_t ws_bytes, void *stream) {
  if (!A || !P || !ws || pad_to <= 0 || A->n_blk <= 0) return SM_ERR_ARG;
  if (!P->nbr_ptr || !P->nbr_idx || !P->own_pos || !P->dim || !P->dim_pad || !P->row_off ||
      !P->sub_off || !P->gmap_ptr || !P->gmap || !P->tmap || !P->order)
    return SM_ERR_ARG;
  if (P->n_blk != A->n_blk || P->nnzb != A->nnzb || P->pad_to != pad_to) return SM_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  int32_t n = A->n_blk;
  WsCursor cur(ws, ws_bytes);
  int64_t *sq_dp = cur.take<int64_t>(n + 1);
  int64_t *sq_cnt = cur.take<int64_t>(n + 1);
  if (!cur.ok()) return SM_ERR_SPACE;
  k_dims<<<(n + 1 + 127) / 128, 128, 0, st>>>(n, A->blk_size, A->row_ptr, A->col_idx, pad_to, P->nbr_ptr,
                                               P->nbr_idx, P->own_pos, P->dim, P->dim_pad, P->row_off,
                                               sq_dp, sq_cnt);
  SM_LAUNCHED();
  k_exclusive_scan_i64<<<1, 1024, 0, st>>>(n, sq_dp, P->sub_off);
  SM_LAUNCHED();
  k_exclusive_scan_i64<<<1, 1024, 0, st>>>(n, sq_cnt, P->gmap_ptr);
  SM_LAUNCHED();
  k_gmap<<<n, 256, 0, st>>>(A->row_ptr, A->col_idx, P->gmap_ptr, P->gmap);
  SM_LAUNCHED();
  k_tmap<<<n, 64, 0, st>>>(A->row_ptr, A->col_idx, P->tmap);
  SM_LAUNCHED();
  k_order<<<(n + 15) / 16, 128, 0, st>>>(n, P->dim_pad, P->order);      // 8 lanes per block column
  SM_LAUNCHED();
  return SM_OK;
}

extern "C" int32_t sm_plan_columns(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols,
                                   int64_t *col_off, void *stream) {
  if (!P || !cols || !col_off || n_cols <= 0) return SM_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  // col_off doubles as the scan input (in-place exclusive scan is safe: out[i] is written after
  // in[i] has been read by the same thread in the same chunk step).
  k_plan_columns<<<(n_cols + 127) / 128, 128, 0, st>>>(cols, n_cols, P->dim_pad, col_off);
  SM_LAUNCHED();
  k_exclusive_scan_i64<<<1, 1024, 0, st>>>(n_cols, col_off, col_off);
  SM_LAUNCHED();
  return SM_OK;
}
