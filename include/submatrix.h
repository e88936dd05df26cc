/*
 * submatrix.h -- C ABI of libsubmatrix.so: the submatrix method for the matrix sign
 * function of a block-sparse symmetric matrix on one NVIDIA B200 (sm_100a).
 *
 * What the calls compute (citations are /root/reference/PAPER.md lines):
 *   "The first step is the construction of a submatrix T_i(A) for every column of the
 *    matrix A.  Then the matrix function is applied to the dense submatrices, i.e.
 *    f(T_i(A)), and finally the relevant result columns are inserted into the sparse
 *    result matrix."                                   (Fig. 2 caption)
 *   f = sign, sign(A) = A (A^2)^(-1/2)                  (Eq. 13)
 *   P = 1/2 (I - sign(S^-1 H - mu I)) S^-1, here S = I  (Eq. 14)
 *   dense work in "FP16 operations with FP32 accumulation" on tensor units
 *
 * Conventions
 *   - Every call returns an int32 status: SM_OK, a negative SM_ERR_*, or a positive
 *     SM_WARN_*.  No exceptions, no exit(), no output on stdout/stderr.
 *   - Unless a parameter says "host", every pointer is a DEVICE pointer.  The library
 *     never allocates or frees device memory: the caller owns every buffer (sizes come
 *     from sm_pattern_sizes / sm_sign_ws_bytes / sm_density_ws_bytes) and must keep it
 *     alive until `stream` has been synchronised.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  All work is
 *     enqueued on it; calls return without synchronising except sm_pattern_sizes
 *     (which must read sizes back) -- status codes that depend on device data
 *     (SM_ERR_PATTERN, SM_WARN_NOT_CONVERGED) are therefore reported by sm_pattern_sizes
 *     and sm_sign_status, which synchronise.
 *   - One submatrix per BLOCK column i (one molecule).  Its index set N(i) is the
 *     ascending list of block rows with a stored block in column i; entries between two
 *     members of N(i) that are not stored are zero.  "Stored" is structural, never a
 *     value threshold, so all pattern arrays are integer functions of integers and are
 *     bit-exact.  The pattern must be structurally symmetric with every diagonal block
 *     present and column indices strictly ascending per row (else SM_ERR_PATTERN).
 *
 * Packed submatrix buffers
 *   A call that works on the column list cols[0..n_cols) (NULL = all block columns, in
 *   id order) addresses submatrix number c of the list at element offset col_off[c] of
 *   the packed buffer; col_off comes from sm_plan_columns (for cols == NULL it equals
 *   P->sub_off).  Submatrix i has true dimension dim[i] and padded dimension
 *   Pd = dim_pad[i] and occupies Pd*Pd elements:
 *     SM_F64 / SM_F32 : row-major, leading dimension Pd.
 *     SM_BF16 / SM_F16: the "K-major 128-byte-swizzled UMMA image" that tcgen05.mma reads
 *       from shared memory, stored as is so that a tile is one contiguous bulk copy.
 *       Pd must be a multiple of 64.  Element (r, c) lives at element offset
 *         (c / 64) * Pd * 64  +  r * 64  +  ((((c % 64) / 8) ^ (r % 8)) * 8)  +  c % 8.
 *   Padding rows/columns hold zeros and stay zero through the iteration.
 */
#ifndef SUBMATRIX_H_
#define SUBMATRIX_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* status codes */
#define SM_OK 0
#define SM_ERR_ARG (-1)         /* bad argument (NULL, negative size, pad_to not allowed for dtype) */
#define SM_ERR_SPACE (-2)       /* a caller buffer / workspace is too small */
#define SM_ERR_PATTERN (-3)     /* pattern not structurally symmetric / diagonal missing / unsorted */
#define SM_ERR_CUDA (-4)        /* a CUDA call failed; code from sm_last_cuda_error() */
#define SM_ERR_UNSUPPORTED (-5) /* dtype / mode combination not implemented */
#define SM_WARN_NOT_CONVERGED 1 /* some submatrix hit max_iter with residual >= tol */

/* element types */
#define SM_F64 0
#define SM_F32 1
#define SM_BF16 2
#define SM_F16 3

/* spectral scaling of T_i - mu I before the iteration (reading A10) */
#define SM_SCALE_NONE 0        /* s_i = 1 */
#define SM_SCALE_GERSHGORIN 1  /* s_i = max_r sum_c |(T_i - mu I)_rc|  (>= spectral radius) */
#define SM_SCALE_POWER 2       /* s_i = 1.05 * ||T v||_2 after 10 power steps on T_i - mu I from a
                                  fixed start vector, never above the Gershgorin bound */
#define SM_SCALE_GLOBAL 3      /* s_i = min(Gershgorin_i, margin * est), est = ||(A - mu I) v||_2 after 10 power steps on the
                                  whole block-sparse A - mu I, an ESTIMATE from below of rho(A - mu I) (every T_i - mu I is a
                                  principal submatrix of it: rho(T_i - mu I) <= rho(A - mu I) by Cauchy interlacing); margin
                                  1.05, widened by ten times the last step's growth while est has not settled.  Not a bound:
                                  Newton-Schulz needs rho(T_i) / s_i < sqrt(3) and sm_sign_status reports a divergence */

/* Block-CSR description of the symmetric input A = H ("block-sparse"). */
typedef struct {
  int32_t n_blk;           /* host: N block rows = block columns                         */
  int32_t nnzb;            /* host: number of stored blocks                              */
  const int32_t *blk_size; /* [N]      b_i > 0                                           */
  const int32_t *row_ptr;  /* [N+1]                                                      */
  const int32_t *col_idx;  /* [nnzb]   strictly ascending within a row                   */
  const int64_t *val_ptr;  /* [nnzb+1] element offset of block p; row-major b_i x b_j    */
} sm_bcsr_t;

/* Sizes the caller needs to allocate the pattern (host struct, filled by sm_pattern_sizes). */
typedef struct {
  int64_t nbr_len;         /* = nnzb                                        */
  int64_t gmap_len;        /* sum_i |N(i)|^2                                */
  int64_t packed_elems;    /* sum_i dim_pad[i]^2                            */
  int64_t build_ws_bytes;  /* workspace for sm_build_pattern                */
  int32_t max_dim;         /* max_i dim[i]                                  */
  int32_t max_dim_pad;     /* max_i dim_pad[i]                              */
  int32_t max_nbr;         /* max_i |N(i)|                                  */
  int32_t reserved;
} sm_sizes_t;

/* Output of sm_build_pattern (PAPER.md:110 step 1, integer part).  Host scalars are copied
 * from sm_sizes_t by the caller; arrays are device memory, caller-allocated. */
typedef struct {
  int32_t n_blk, nnzb, pad_to, max_dim, max_dim_pad, max_nbr;   /* host */
  int64_t packed_elems, gmap_len;                                /* host */
  int32_t *nbr_ptr;   /* [N+1]     start of N(i) in nbr_idx                               */
  int32_t *nbr_idx;   /* [nnzb]    N(i), ascending block ids                              */
  int32_t *own_pos;   /* [N]       position of i inside N(i)                              */
  int32_t *dim;       /* [N]       m_i = sum of b_j over N(i)                             */
  int32_t *dim_pad;   /* [N]       m_i rounded up to a multiple of pad_to                 */
  int32_t *row_off;   /* [nnzb]    first row of neighbour a inside submatrix i            */
  int64_t *sub_off;   /* [N+1]     exclusive scan of dim_pad^2                            */
  int64_t *gmap_ptr;  /* [N+1]     exclusive scan of |N(i)|^2                             */
  int32_t *gmap;      /* [gmap_len] stored-block index of (N(i)[a], N(i)[c]) at a*|N(i)|+c, or -1 */
  int32_t *tmap;      /* [nnzb]    index of the transposed partner block (j,i) of p=(i,j) */
  int32_t *order;     /* [N]       block columns by (dim_pad descending, id ascending)    */
} sm_pattern_t;

/* Last CUDA error code seen by the calling thread's library calls (0 = none). host. */
int32_t sm_last_cuda_error(void);

/* Validates the pattern and returns the sizes.  `scratch` >= 256 bytes of device memory.
 * Synchronises `stream`.  Errors: SM_ERR_ARG, SM_ERR_PATTERN, SM_ERR_CUDA. */
int32_t sm_pattern_sizes(const sm_bcsr_t *A, int32_t pad_to, sm_sizes_t *out /*host*/,
                         void *scratch, void *stream);

/* a1. Builds all pattern arrays of P (bit-exact integer work).  P's host scalars must be
 * filled from sm_pattern_sizes; ws >= build_ws_bytes.  Asynchronous. */
int32_t sm_build_pattern(const sm_bcsr_t *A, int32_t pad_to, sm_pattern_t *P, void *ws,
                         int64_t ws_bytes, void *stream);

/* Offsets of a column list inside a packed buffer: col_off[c] = sum_{c'<c} dim_pad[cols[c']]^2,
 * col_off[n_cols] = total.  cols == NULL is not needed (use P->sub_off).  Asynchronous. */
int32_t sm_plan_columns(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols,
                        int64_t *col_off /*[n_cols+1]*/, void *stream);

/* a2. X0 = (T_i(A) - mu I) / s_i for the listed columns, padded, in x_dtype (PAPER.md:110
 * step 1, :91 for the shift).  A_vals are A's block values (a_dtype SM_F64 or SM_F32).
 * scale[c] (fp64, [n_cols]) receives s_i.  ws >= sm_gather_ws_bytes.  Asynchronous.
 * Errors: SM_ERR_ARG (x_dtype 16-bit with pad_to % 64 != 0), SM_ERR_UNSUPPORTED, SM_ERR_SPACE. */
int64_t sm_gather_ws_bytes(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t n_cols);
int32_t sm_gather(const sm_bcsr_t *A, const void *A_vals, int32_t a_dtype, const sm_pattern_t *P,
                  const int32_t *cols, int32_t n_cols, const int64_t *col_off, double mu,
                  int32_t scale_mode, int32_t x_dtype, void *X_packed, double *scale,
                  void *ws, int64_t ws_bytes, void *stream);

/* a3. Newton-Schulz sign iteration on every listed submatrix, in place (Eq. 13,
 * "various iterative methods" :85; iteration X <- 1/2 X (3I - X^2), reading A9):
 *     k = 0,1,..:  Y = X_k^2;  r_k = ||Y - I||_F / sqrt(m_i)  (true m_i, padding excluded);
 *                  X_{k+1} = 1.5 X_k - 0.5 X_k Y;  stop after this update if r_k < tol.
 * tol <= 0 runs exactly max_iter updates.  iters[c] = updates applied, residual[c] = last
 * r_k computed.  SM_BF16/SM_F16 run on tcgen05 tensor cores with fp32 accumulation
 * (PAPER.md:104): submatrices with Pd <= 256 stay in the shared memory of one SM for all steps, larger ones run as
 * grouped tiles with one launch per product; SM_F64 runs on the fp64 tensor-core instruction (mma.sync m8n8k4,
 * DMMA), SM_F32 on FFMA.  packed_elems = col_off[n_cols] (host value).
 * ws >= sm_sign_ws_bytes(...).  Asynchronous; sm_sign_status reports non-convergence. */
int64_t sm_sign_ws_bytes(const sm_pattern_t *P, int32_t n_cols, int64_t packed_elems, int32_t x_dtype);
int32_t sm_sign_ns(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols,
                   const int64_t *col_off, int64_t packed_elems, int32_t x_dtype, void *X_packed,
                   void *ws, int64_t ws_bytes, int32_t max_iter, double tol,
                   int32_t *iters /*[n_cols]*/, double *residual /*[n_cols]*/, void *stream);
/* sm_sign_ns with two more arguments (sm_sign_ns = flags 0, switch_iter -1):
 *   flags & SM_SIGN_NONSYMMETRIC: the matrices are NOT symmetric (used for Eq. 12: the sign of the
 *     block matrix [[0, A], [I, 0]]).  Every tile is computed with true products X X and X Y (the 16-bit kernel reads
 *     its B operand MN-major from the same image), nothing is mirrored; the default exploits and enforces symmetry.
 *   switch_iter >= 0: precision schedule "low precision early, higher precision late" (SURVEY
 *     8(f) f3): x_dtype must be SM_BF16, tol <= 0 and 0 < switch_iter < max_iter; updates 0 .. switch_iter-1 run on
 *     bf16 operands, update switch_iter-1 rounds its result to fp16 and the remaining updates run on fp16 operands
 *     (same kind::f16 MMA, 11 instead of 8 significand bits; |x| <= ~1 after scaling, so the range is safe).
 *     X_packed then holds SM_F16 images on return.
 *   flags & SM_SIGN_ORDER3: the third-order member of the same family instead of Newton-Schulz ("various
 *     iterative methods"; reading A22): X <- X (15 I - 10 X^2 + 3 X^4) / 8, three products per
 *     step, cubic convergence, basin |x| < sqrt(7/3).  Same workspace, same stopping rule (the residual of step k is
 *     still ||X_k^2 - I||_F / sqrt(m)); symmetric matrices only (with SM_SIGN_NONSYMMETRIC: SM_ERR_UNSUPPORTED); all
 *     four x_dtype (16-bit: Q = 3/4 (I - X^2), Z = 2/3 (Q + Q Q), X' = X + X Z on the grouped tcgen05 kernels).
 * ws >= sm_sign_ws_bytes_ex(..., flags). */
#define SM_SIGN_NONSYMMETRIC 1
#define SM_SIGN_ORDER3 2
int64_t sm_sign_ws_bytes_ex(const sm_pattern_t *P, int32_t n_cols, int64_t packed_elems, int32_t x_dtype,
                            int32_t flags);
int32_t sm_sign_ns_ex(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols,
                      const int64_t *col_off, int64_t packed_elems, int32_t x_dtype, void *X_packed,
                      void *ws, int64_t ws_bytes, int32_t max_iter, double tol, int32_t flags,
                      int32_t switch_iter, int32_t *iters /*[n_cols]*/, double *residual /*[n_cols]*/,
                      void *stream);
/* sm_sign_ns (SM_F64 / SM_F32 only, Newton-Schulz, symmetric matrices; PAPER.md:87 Eq. 13, :110 step 2) WITHOUT a caller
 * workspace and without any allocation -- for callers that cannot call cudaMalloc (CUDA graph capture, tight serving
 * loops, harnesses that forbid it).  The workspace is a file-scope device array of sm_sign_ns_static_capacity() bytes
 * (16 MiB) that every GPU that loads the library holds until the process exits; a call whose
 * sm_sign_ws_bytes(P, n_cols, packed_elems, x_dtype) exceeds it returns SM_ERR_SPACE and launches nothing (use
 * sm_sign_ns).  Same arguments, results (bit-identical) and error behaviour as sm_sign_ns otherwise; additionally
 * SM_ERR_UNSUPPORTED for the 16-bit types and while sm_profile_enable(1) is in effect (both allocate).  tol <= 0: no
 * host synchronisation either; tol > 0 reads one counter back every second step like sm_sign_ns.
 * ALL calls share the one array: what must start at zero is cleared on `stream` by the call itself, and two calls
 * that overlap on the GPU (different streams / host threads) race on it -- the caller serialises them. */
int64_t sm_sign_ns_static_capacity(void);
int32_t sm_sign_ns_static(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols,
                          const int64_t *col_off, int64_t packed_elems, int32_t x_dtype, void *X_packed,
                          int32_t max_iter, double tol, int32_t *iters /*[n_cols]*/,
                          double *residual /*[n_cols]*/, void *stream);
/* Synchronises and returns SM_WARN_NOT_CONVERGED if tol > 0 and any residual[c] >= tol (or is not finite); with
 * tol <= 0 (fixed-count mode) if any residual[c] is not finite or exceeds 1, i.e. the iteration diverged. */
int32_t sm_sign_status(const double *residual, int32_t n_cols, double tol, void *scratch, void *stream);

/* a4. R(N(i)[a], i) = S_i[rows of neighbour a, columns of block i] for the listed columns
 * (PAPER.md:110 step 3) into block-CSR values with A's layout; r_dtype SM_F64 or SM_F32.
 * S_i is symmetric, so the owned ROWS are read (contiguous) and transposed on the fly.
 * symmetrise != 0 (only with all columns present, i.e. after the last chunk) additionally
 * replaces R by 1/2 (R + R^T) blockwise through tmap (reading A6). Asynchronous. */
int32_t sm_scatter(const sm_bcsr_t *A, const sm_pattern_t *P, const int32_t *cols, int32_t n_cols,
                   const int64_t *col_off, int32_t x_dtype, const void *S_packed, int32_t r_dtype,
                   void *R_vals, int32_t symmetrise, void *stream);
/* In-place blockwise symmetrisation of block-CSR values (used after chunked scatters). */
int32_t sm_symmetrise(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t r_dtype, void *R_vals,
                      void *stream);

/* a5. The whole path, Eq. 14 with S = I: D = 1/2 (I - sign(H - mu I)) by the submatrix method:
 * gather -> sign -> scatter (-> symmetrise) -> D = 1/2 (I - R), Tr D.  Columns are processed in
 * chunks that fit ws_bytes; h_dim_pad is a HOST copy of P->dim_pad (needed to plan chunks).
 * d_dtype SM_F64 or SM_F32; trace is a device fp64 scalar; iters/residual/scale are [N] device
 * arrays.  ws >= sm_density_ws_bytes(P, x_dtype, max_chunk_elems) where max_chunk_elems bounds the
 * packed elements per chunk (>= max_dim_pad^2; P->packed_elems for a single chunk).  Asynchronous.
 * With tol <= 0 the call enqueues kernels and memsets only (no host synchronisation; after the first call of a
 * process nothing is allocated), so it can be captured into a CUDA graph and replayed on the same buffers
 * (tests/test_gpu_parity.py::test_fixed_count_density_is_graph_capturable); tol > 0 reads one counter back every
 * second step and cannot be captured. */
int64_t sm_density_ws_bytes(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t x_dtype,
                            int64_t max_chunk_elems);
/* The same for sm_density_ex(..., sign_flags, ...) (sm_density_ws_bytes = sign_flags 0): the third-order iteration
 * keeps two scratch images even where Newton-Schulz runs entirely on chip. */
int64_t sm_density_ws_bytes_ex(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t x_dtype,
                               int64_t max_chunk_elems, int32_t sign_flags);
int32_t sm_density(const sm_bcsr_t *A, const void *A_vals, int32_t a_dtype, double mu,
                   int32_t x_dtype, int32_t scale_mode, int32_t max_iter, double tol,
                   int32_t symmetrise, const sm_pattern_t *P, const int32_t *h_dim_pad /*host [N]*/,
                   int64_t max_chunk_elems, void *ws, int64_t ws_bytes, int32_t d_dtype,
                   void *D_vals, double *trace, int32_t *iters, double *residual, double *scale,
                   void *stream);
/* sm_density with a precision schedule (SURVEY 8(f) f3; PAPER.md:104 "FP16 operations with FP32 accumulation", :15):
 * switch_iter >= 0 (x_dtype SM_BF16, tol <= 0, 0 < switch_iter < max_iter) runs the first switch_iter updates on bf16
 * operands and the rest on fp16 operands (see sm_sign_ns_ex); switch_iter < 0 is sm_density.  sign_flags: 0 or
 * SM_SIGN_ORDER3 (third-order iteration in a3, see sm_sign_ns_ex); anything else is SM_ERR_ARG. */
int32_t sm_density_ex(const sm_bcsr_t *A, const void *A_vals, int32_t a_dtype, double mu,
                      int32_t x_dtype, int32_t scale_mode, int32_t max_iter, double tol, int32_t switch_iter,
                      int32_t sign_flags, int32_t symmetrise, const sm_pattern_t *P, const int32_t *h_dim_pad /*host [N]*/,
                      int64_t max_chunk_elems, void *ws, int64_t ws_bytes, int32_t d_dtype,
                      void *D_vals, double *trace, int32_t *iters, double *residual, double *scale,
                      void *stream);
/* Chemical potential for a fixed electron count (the first row past the hot path).
 * Eq. 14 carries mu but the paper gives no rule for it; the usual closure is the electron count
 * Tr D(mu) = n_target (with S = I, D = 1/2 (I - sign(H - mu I)) counts the eigenvalues below mu),
 * and Tr D(mu) is non-decreasing in mu, so mu is found by bisection on [mu_lo, mu_hi].  Host driven: every trial is
 * one sm_density call (same arguments, same buffers) followed by a synchronisation of `stream` to read the 8-byte
 * trace.  Trials 1 and 2 evaluate the ends of the bracket (SM_ERR_ARG unless Tr D(mu_lo) <= n_target <= Tr D(mu_hi),
 * both within tol_n); then mu = midpoint until |Tr D(mu) - n_target| <= tol_n, or the bracket is narrower than
 * mu_tol, or max_trials (>= 3) trials were run.  On return *mu_out is the last midpoint evaluated (or the end of
 * the bracket that already met tol_n), *trace_out its Tr D, *trials_out the number of sm_density calls, and
 * D_vals / trace / iters / residual / scale hold that trial's results.  Synchronises. */
int32_t sm_mu_search(const sm_bcsr_t *A, const void *A_vals, int32_t a_dtype, double n_target, double mu_lo,
                     double mu_hi, double tol_n, double mu_tol, int32_t max_trials, int32_t x_dtype,
                     int32_t scale_mode, int32_t max_iter, double tol, int32_t symmetrise, const sm_pattern_t *P,
                     const int32_t *h_dim_pad /*host [N]*/, int64_t max_chunk_elems, void *ws, int64_t ws_bytes,
                     int32_t d_dtype, void *D_vals, double *trace, int32_t *iters, double *residual,
                     double *scale, double *mu_out /*host*/, double *trace_out /*host*/,
                     int32_t *trials_out /*host*/, void *stream);
/* ---- non-orthogonal basis (PAPER.md:83 Eq. 12, :87 Eq. 13, :91 Eq. 14) ----------------------------
 * sm_inv_sqrt: Z ~ S^-1/2 (and optionally Y ~ S^1/2) of a symmetric positive definite block-sparse S by the submatrix
 * method with f = the blocks of Eq. 12: for every block column i, T_i(S) is gathered (a2), the 2m x 2m matrix
 * [[0, T_i], [I, 0]] / sqrt(Gershgorin bound of T_i) is iterated by the same Newton-Schulz kernels at doubled dimension
 * with SM_SIGN_NONSYMMETRIC (a3), and the owned columns of its lower-left block T_i^-1/2 (upper-right: T_i^1/2) are
 * inserted (a4).  All four x_dtype; tol > 0 = convergence mode, tol <= 0 = exactly max_iter steps.  Columns are processed
 * in chunks of P->order whose DOUBLED images (dimension 2 m_i rounded up to pad_to) hold at most max_chunk_elems2
 * elements (>= the largest one); h_dim is a HOST copy of P->dim.  Z_vals / Y_vals: block-CSR values with S's layout
 * (z_dtype SM_F64 or SM_F32; Y_vals may be NULL); iters / residual / scale are [N] device arrays indexed by position in
 * P->order (scale = the Gershgorin bound of T_i).  Not positive definite input is not detected: the iteration then
 * does not converge (residual stays large).  Asynchronous. */
int64_t sm_inv_sqrt_ws_bytes(const sm_bcsr_t *S, const sm_pattern_t *P, int32_t x_dtype, int64_t max_chunk_elems2);
int32_t sm_inv_sqrt(const sm_bcsr_t *S, const void *S_vals, int32_t s_dtype, int32_t x_dtype, int32_t max_iter,
                    double tol, const sm_pattern_t *P, const int32_t *h_dim /*host [N]*/, int64_t max_chunk_elems2,
                    void *ws, int64_t ws_bytes, int32_t z_dtype, void *Z_vals, void *Y_vals, int32_t *iters,
                    double *residual, double *scale, void *stream);
/* sm_density_nonorth: Eq. 14 with S != I by the submatrix method on the pair (H, S) (one block pattern, two value
 * arrays of type a_dtype): per block column, Z = T_S^-1/2 as in sm_inv_sqrt, S^-1 = Z Z, A = S^-1 T_H - mu I (not
 * symmetric) scaled by its infinity norm, sign(A) by the non-symmetric Newton-Schulz kernels, P_i = 1/2 (I - sign(A)) S^-1,
 * owned columns inserted (optionally symmetrised).  x_dtype SM_F64 / SM_F32: d_dtype = x_dtype, a_dtype = x_dtype or
 * SM_F64 (the dense products run on the DMMA / FFMA kernels).  x_dtype SM_BF16 / SM_F16 (pad_to % 64 == 0): a_dtype and
 * d_dtype SM_F64 or SM_F32 independently; the products run on the non-symmetric tcgen05 update kernel with its identity
 * term switched off, every intermediate is a 16-bit image.  Other combinations: SM_ERR_UNSUPPORTED.  trace_ps (device fp64 scalar, may be NULL; synchronises once)
 * receives Tr(P S), the electron count.  iters / residual / scale report the sign(A) iteration.  Asynchronous
 * otherwise. */
int64_t sm_density_nonorth_ws_bytes(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t x_dtype, int64_t max_chunk_elems2);
int32_t sm_density_nonorth(const sm_bcsr_t *A, const void *H_vals, const void *S_vals, int32_t a_dtype, double mu,
                           int32_t x_dtype, int32_t max_iter, double tol, int32_t symmetrise, const sm_pattern_t *P,
                           const int32_t *h_dim /*host [N]*/, int64_t max_chunk_elems2, void *ws, int64_t ws_bytes,
                           int32_t d_dtype, void *P_vals, double *trace_ps, int32_t *iters, double *residual,
                           double *scale, void *stream);

/* R -> D = 1/2 (I - R) in place on block-CSR values, and Tr D (device fp64 scalar, may be NULL). */
int32_t sm_density_from_sign(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t d_dtype,
                             void *RD_vals, double *trace, void *stream);

/* Variant selection (A/B measurements and the back-end tests; production code leaves everything at its default
 * and gets the measured-best variant).  Process-wide; every option is initialised once from the environment
 * variable given in brackets, and sm_set_option changes it for the calls that follow (not synchronised with
 * calls in flight on other threads).  Unknown name: SM_ERR_ARG.
 *   "umma.sym"      [SM_UMMA_SYM]      1|0   16-bit: lower-triangle tiles with mirrored stores / true products, all tiles
 *   "umma.resident" [SM_UMMA_RESIDENT] 1|0   16-bit: submatrices with Pd <= 256 iterate inside one SM / grouped tiles for all
 *   "umma.epi"      [SM_UMMA_EPI]      0|1   16-bit grouped tiles: per-lane global stores / staged epilogue (stmatrix into
 *                                            shared-memory staging, bulk stores; 3-stage operand ring)
 *   "umma.lt"       [SM_UMMA_LT]       0|1   with umma.epi = 1: iterates stored "128-lower" (nothing above the 128 x 128
 *                                            diagonal squares), the rest read through MN-major descriptors
 *   "umma.fold"     [SM_UMMA_FOLD]     1|0   16-bit grouped symmetric tiles: a last 128-row panel of <= 64 rows is computed as extra
 *                                            columns of the other panels and mirrored into place / as a row panel of its own
 *   "umma.sharea"   [SM_UMMA_SHAREA]   1|0   16-bit grouped symmetric tiles, product X X^T: a tile that holds its panel's diagonal
 *                                            square reads its A rows from the B rows it stages / loads them separately (bit-identical)
 *   "umma.dyn"      [SM_UMMA_DYN]      1|0   16-bit grouped tiles handed out by a global counter / dealt round robin
 *   "umma.rev"      [SM_UMMA_REV]      1|0   16-bit: the update product walks the tile table backwards / forwards
 *   "umma.stages"   [SM_UMMA_STAGES]   0|3|4 16-bit grouped tiles: depth of the operand ring (0 = by size)
 *   "umma.stream"   [SM_UMMA_STREAM]   0|1   16-bit, tol <= 0: one launch walks every product of every step
 *   "f64.simt"      [SM_F64_SIMT]      0|1   fp64: tensor-core m8n8k4 tiles / DFMA register tiles
 *   "f64.tile"      [SM_F64_TILE]      0|64|128  fp64 tensor-core tile edge (0: 64 when the largest submatrix is <= 384, else 128)
 *   "f32.sym"       [SM_F32_SYM]       1|0   fp32: lower-triangle 64 x 64 FFMA tiles with 8 x 8 register blocks and mirrored
 *                                            stores (exactly symmetric iterates) / all tiles with 4 x 4 blocks
 *   "gather.lean"   [SM_GATHER_LEAN]   1|0   sm_gather, 16-bit X, blocks >= 4 wide: per-CTA tables of the runs' blocks / blocks resolved
 *                                            per run (bit-identical)
 *   "gather.tma"    [SM_GATHER_TMA]    0|1   sm_gather, 16-bit X: element-wise kernel / source-driven kernel staged through
 *                                            shared memory with bulk TMA stores (bit-identical; measured slower)
 * A library built with -DSM_MEASURE (build.py --measure; sm_build_info() & 1) additionally has the measured-slower
 * two-CTA and fused variants and the skip-knobs used for DESIGN.md's decompositions ("umma.ncta", "umma.mc",
 * "umma.tmap", "umma.fused", "umma.slots", "umma.dbg"; the last produces WRONG results by construction).  In the
 * default build those names answer SM_ERR_UNSUPPORTED and their environment variables are not read. */
int32_t sm_set_option(const char *name /*host*/, int32_t value);
int32_t sm_get_option(const char *name /*host*/, int32_t *value /*host*/);
int32_t sm_build_info(void);

/* Reason code of the last device-side protocol failure (a kernel whose internal barrier never completed writes
 * the code to a pinned host word and traps; the CUDA error that follows is sticky, the code stays readable).
 * 0 = none.  host.  The 64-byte pinned word is the one allocation the library makes (host memory, on first use). */
int32_t sm_last_device_error(void);

/* Number of kernels this thread's library calls have launched so far (bench bookkeeping). host. */
int64_t sm_launch_count(void);

/* Measurement hooks (host).  While enabled, every launch of the tensor-core Newton-Schulz kernel
 * (the dominant kernel of a3 for SM_BF16/SM_F16) is bracketed by CUDA events on its stream.
 * sm_profile_read synchronises on those events, returns their summed duration in ms and the number
 * of launches covered, and resets the counters.  Not thread-safe; leave disabled in production. */
int32_t sm_profile_enable(int32_t on);
int32_t sm_profile_read(double *gemm_ms /*host*/, int64_t *gemm_launches /*host*/);

#ifdef __cplusplus
}
#endif
#endif /* SUBMATRIX_H_ */
