// a3, bf16 / fp16, shared-memory-resident variant for small submatrices (included by sign_umma.cu inside
// namespace sm; uses pack2 / unpack2 and the PTX wrappers).
//
// "dense linear algebra on medium sized local matrices", "evaluation of the matrix function on
// many dense, but much smaller matrices" (PAPER.md:106; :110 step 2; Eq. 13 :87; iteration DESIGN.md A9).
//
// ONE CTA takes ONE submatrix with Pd <= 256 through ALL Newton-Schulz steps: X_0 comes in by one bulk-TMA copy
// (the packed image IS the UMMA shared-memory image), every product reads its operands from shared memory,
// accumulates in TMEM, and the epilogue writes the next operand straight back into shared memory; only the final
// S leaves the SM (one bulk store).  HBM traffic per call: 2 images instead of 5 images per step (the per-phase
// launches at configs[3]: 74 GB for a 1.5 GB problem).
//
// Shared memory: XS = the whole K-major SW128 image of X (Pd x Pd, <= 128 KB); WS = Wh = -1/2 (X X^T - I) stored
// "128-lower": 64-column chunk kc keeps only the rows >= lt0(kc) = (64 kc) & ~127 (everything at or below the
// 128 x 128 diagonal squares: 96 KB at Pd = 256, so that XS + WS fit the 227 KB of an SM).  The part of Wh above
// the diagonal squares is read through its transpose: Wh is symmetric, and the rows 64 kc .. 64 kc + 63 of chunks
// 0, 1 ARE Wh[k][n] for n < 128, i.e. an MN-major SW128 B operand (64 n x 8 k swizzle atoms, the next 64 n at
// LBO = one chunk, the next 8 k at SBO = 1024 B).
//
// Tiles per product (128-row UMMA M, lower triangle at 128 granularity): T0 = rows 0..127 x cols 0..min(128, Pd),
// T1 = rows 128..255 x cols 0..Pd (only if Pd > 128); accumulators: T1 at TMEM columns 128.., T0 at columns 0.. for
// product 1 and at columns 384.. for product 2, so that the early part of a product can be issued while the other
// tile's epilogue of the previous product still converts (schedule: see the MMA issuer).  Symmetry is enforced exactly
// as in k_umma_gemm: only elements (r, c), r >= c, are taken from the accumulators, stored at (r, c) and mirrored to (c, r).
//   product 1: Y = X X^T; epilogue: W = Y - I, fused ||W||_F^2 (warp shuffles + fixed-order sum of the 16 warp
//              partials), Wh = -1/2 W -> WS.
//   product 2: X' = X + X Wh^T; the accumulator holds X Wh^T, the epilogue adds the X tile it reads back from XS
//              (shared memory: cheap here) and writes X' -> XS in place (no MMA is in flight on those rows).
// Roles: warp 0 = loader (pops the next listed column with Pd <= 256 from a global counter, prefetches it into
// L2, waits until XS is free, issues the bulk copy), warp 1 = MMA issuer (one thread; owns TMEM), warps 2..17 =
// epilogue (4 per TMEM lane quadrant).  The stopping rule (A11) is evaluated inside the kernel by every role
// from the same 16 partial sums, so convergence mode needs no host round trip and no second launch.
#pragma once

constexpr int RES_MAX_PD = 256;
constexpr int RES_EPI_WARPS = 16;
constexpr int RES_THREADS = 64 + 32 * RES_EPI_WARPS;
constexpr int RES_XS_BYTES = RES_MAX_PD * RES_MAX_PD * 2;            // 128 KB
constexpr int RES_WS_BYTES = (2 * 256 + 2 * 128) * 128;              // 96 KB: chunks 0, 1 whole, chunks 2, 3 rows 128..255
constexpr int RES_SMEM = RES_XS_BYTES + RES_WS_BYTES + 1024 /*align slack*/ + 512 /*barriers, control*/;

struct RArgs {
  const int32_t *cols; const int64_t *col_off; const int32_t *dim; const int32_t *dim_pad;
  int32_t n_cols, max_iter;
  double tol;                    // <= 0: exactly max_iter updates
  void *X;                       // packed 16-bit images, in / out
  int32_t *iters; double *residual;
  unsigned long long *counter;   // zeroed by the host: next position of the column list to hand out
  int32_t *err_flag;
  int32_t switch_iter;           // mixed precision (f3): updates 0 .. switch_iter-1 run in bf16 and write bf16, the
                                 // update switch_iter-1 writes fp16 and the rest runs in fp16; < 0 = never
};

// first stored row of Wh chunk kc, and the byte offset of that chunk inside WS
__device__ __forceinline__ uint32_t res_lt0(uint32_t kc) { return (kc >> 1) * 128u; }
__device__ __forceinline__ uint32_t res_woff(uint32_t kc, uint32_t Pd) { return 128u * (kc * Pd - (kc == 3u ? 128u : 0u)); }

template <bool BF16_IN>
__global__ void __launch_bounds__(RES_THREADS, 1) k_umma_resident(RArgs a) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = ptx::smem_u32(smem_raw);
  const uint32_t xs = (raw + 1023u) & ~1023u;
  const uint32_t ws = xs + RES_XS_BYTES;
  const uint32_t bars = ws + RES_WS_BYTES;
  // b_w1 / b_w0: the epilogue of product 1 has written T1's / T0's part of Wh (and drained that accumulator);
  // b_x0 / b_x1: the epilogue of product 2 has written T0's / T1's part of X'.  16 warp arrivals each, once per step.
  const uint32_t b_xload = bars, b_tfull0 = bars + 8, b_tfull1 = bars + 16, b_w1 = bars + 24, b_w0 = bars + 32,
                 b_x0 = bars + 40, b_x1 = bars + 48, b_free = bars + 56, tmem_slot = bars + 80;
  volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - raw));
  volatile int64_t *cur_c = reinterpret_cast<volatile int64_t *>(smem_raw + (bars + 64 - raw));
  volatile float *res_s = reinterpret_cast<volatile float *>(smem_raw + (bars + 128 - raw));   // [16]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    ptx::mbar_init(b_xload, 1); ptx::mbar_init(b_tfull0, 1); ptx::mbar_init(b_tfull1, 1);
    ptx::mbar_init(b_w1, RES_EPI_WARPS); ptx::mbar_init(b_w0, RES_EPI_WARPS); ptx::mbar_init(b_x0, RES_EPI_WARPS);
    ptx::mbar_init(b_x1, RES_EPI_WARPS); ptx::mbar_init(b_free, 1);
    ptx::fence_barrier_init();
    ptx::fence_proxy_async();
  }
  if (warp == 1) { ptx::tmem_alloc(tmem_slot, 512); ptx::tmem_relinquish(); }
  ptx::tc_fence_before();
  __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  // per-submatrix facts every role derives from the listed position c
  struct Sub { int32_t m, Pd, kmax, nkc, n0; bool two; };
  auto sub_of = [&](int64_t c) {
    const int32_t i = a.cols ? a.cols[c] : (int32_t)c;
    Sub s; s.m = a.dim[i]; s.Pd = a.dim_pad[i]; s.kmax = (s.m + 15) & ~15; s.nkc = (s.kmax + 63) >> 6;
    s.n0 = s.Pd < 128 ? s.Pd : 128; s.two = s.Pd > 128;
    return s;
  };
  // r_k = sqrt(sum of the 16 warp partials / m), the same fixed-order sum in every role (A11)
  auto residual_now = [&](int32_t m) {
    double sum = 0.0;
#pragma unroll
    for (int w = 0; w < RES_EPI_WARPS; ++w) sum += (double)res_s[w];
    return sqrt(sum / (double)m);
  };

  if (warp == 0) {
    // ===================== loader =====================
    if (lane == 0) {
      uint32_t p_free = 0;
      for (int32_t n = 0;; ++n) {
        int64_t c;
        for (;;) {
          c = (int64_t)atomicAdd(a.counter, 1ULL);
          if (c >= a.n_cols) { c = -1; break; }
          if (a.dim_pad[a.cols ? a.cols[c] : (int32_t)c] <= RES_MAX_PD) break;     // larger ones: grouped path
        }
        uint32_t bytes = 0; const char *src = nullptr; int32_t Pd_l = 64;
        if (c >= 0) {
          Pd_l = a.dim_pad[a.cols ? a.cols[c] : (int32_t)c];
          bytes = (uint32_t)Pd_l * (uint32_t)Pd_l * 2u;
          src = (const char *)a.X + a.col_off[c] * 2;
          ptx::prefetch_l2_bulk(src, bytes);          // the image waits in L2 while the current submatrix iterates
        }
        if (n > 0) { ptx::mbar_wait(b_free, p_free, a.err_flag, 21); p_free ^= 1u; }
        *cur_c = c;
        if (c < 0) { ptx::mbar_arrive(b_xload); break; }
        ptx::mbar_expect_tx(b_xload, bytes);
        const uint32_t cb = bytes / (uint32_t)(Pd_l >> 6);       // one 64-column chunk: Pd rows x 128 B
        for (uint32_t off = 0; off < bytes; off += cb) ptx::tma_bulk_g2s(xs + off, src + off, cb, b_xload);
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer =====================
    // The whole warp runs this loop converged, on warp-uniform values (shuffle broadcasts tell ptxas so); one
    // elected lane issues each MMA / commit (umma_f16_elect).
    //
    // Schedule of one step (two tiles; T0 alternates between the accumulators T0a = TMEM columns 0.. for product 1 and
    // T0b = columns 384.. for product 2, T1 stays at columns 128..).  Chunks kc < 2 are the columns 0..127, chunks
    // kc >= 2 the columns 128.. :
    //   product 1 (Y = X X^T):   T0a[kc < 2]            needs X'[0:128, 0:128]                = T0's epilogue 2   (b_x0)
    //                            T1[all], T0a[kc >= 2]  need all of X'                        + T1's epilogue 2   (b_x1)
    //   product 2 (X Wh^T):      T0b[kc >= 2], T1[kc >= 2] need Wh[128.., :] only             = T1's epilogue 1   (b_w1)
    //                            T0b[kc < 2], T1[kc < 2]   need Wh[0:128, 0:128] as well      + T0's epilogue 1   (b_w0)
    // so the MMAs of the early parts run while the other tile's epilogue is still converting, instead of the whole chain
    // MMA -> epilogue -> MMA being serial (clock64, first version: two hand-overs of ~2 000 cycles per step exposed).
    // Product 1 finishes T1 before T0a and product 2 finishes T0b before T1: T1's mirrored X' stores land in rows
    // 0..127 of XS, which T0b's MMAs read, so T1's epilogue 2 may only start when they are done.
    {
      uint32_t p_xload = 0, p_w1 = 0, p_w0 = 0, p_x0 = 0, p_x1 = 0;
      for (;;) {
        ptx::mbar_wait(b_xload, p_xload, a.err_flag, 22); p_xload ^= 1u;
        const int32_t c = __shfl_sync(0xffffffffu, (int32_t)*cur_c, 0);
        if (c < 0) break;
        Sub s = sub_of(c);
        s.m = __shfl_sync(0xffffffffu, s.m, 0); s.Pd = __shfl_sync(0xffffffffu, s.Pd, 0);
        s.kmax = (s.m + 15) & ~15; s.nkc = (s.kmax + 63) >> 6; s.n0 = s.Pd < 128 ? s.Pd : 128; s.two = s.Pd > 128;
        const uint32_t Pd = (uint32_t)s.Pd;
        const uint32_t dT0a = tmem_base, dT1 = tmem_base + 128u, dT0b = tmem_base + 384u;
        bool bf = BF16_IN;
        // product 1, tile t, chunks [k_lo, k_hi): first = no MMA has written this accumulator yet
        auto p1 = [&](int t, int k_lo, int k_hi, bool first) {
          const uint32_t N = t ? Pd : (uint32_t)s.n0;
          const uint32_t idesc = ptx::make_idesc_f16(bf, 128, N, false);
          const uint32_t d = t ? dT1 : dT0a;
          for (int kc = k_lo; kc < k_hi; ++kc) {
            const uint64_t ad = ptx::make_sw128_kmajor_desc(xs + (uint32_t)kc * Pd * 128u + (t ? 128u * 128u : 0u));
            const uint64_t bd = ptx::make_sw128_kmajor_desc(xs + (uint32_t)kc * Pd * 128u);
            const int ksteps = min(4, (s.kmax - kc * 64) / 16);
            const uint32_t acc0 = (uint32_t)(!first || kc != k_lo);
            if (ksteps == 4) {
              ptx::umma_f16_elect_k4(d, ptx::sw128_kmajor_lo(xs + (uint32_t)kc * Pd * 128u + (t ? 128u * 128u : 0u)),
                                     ptx::sw128_kmajor_lo(xs + (uint32_t)kc * Pd * 128u), idesc, acc0);
            } else {
              for (int ks = 0; ks < ksteps; ++ks) ptx::umma_f16_elect(d, ad + (uint64_t)(2 * ks), bd + (uint64_t)(2 * ks), idesc, acc0 | (uint32_t)(ks != 0));
            }
          }
        };
        // product 2 (A = rows of XS, B = Wh from WS: stored rows K-major, the rest through the transpose)
        auto p2 = [&](int t, int k_lo, int k_hi, bool first) {
          const uint32_t d = t ? dT1 : dT0b;
          for (int kc = k_lo; kc < k_hi; ++kc) {
            const uint64_t ad = ptx::make_sw128_kmajor_desc(xs + (uint32_t)kc * Pd * 128u + (t ? 128u * 128u : 0u));
            const int ksteps = min(4, (s.kmax - kc * 64) / 16);
            const uint32_t acc0 = (uint32_t)(!first || kc != k_lo);
            if (kc < 2) {
              const uint32_t N = t ? Pd : (uint32_t)s.n0;
              const uint32_t idesc = ptx::make_idesc_f16(bf, 128, N, false);
              const uint64_t bd = ptx::make_sw128_kmajor_desc(ws + res_woff((uint32_t)kc, Pd));
              if (ksteps == 4) {
                ptx::umma_f16_elect_k4(d, ptx::sw128_kmajor_lo(xs + (uint32_t)kc * Pd * 128u + (t ? 128u * 128u : 0u)),
                                       ptx::sw128_kmajor_lo(ws + res_woff((uint32_t)kc, Pd)), idesc, acc0);
              } else {
                for (int ks = 0; ks < ksteps; ++ks) ptx::umma_f16_elect(d, ad + (uint64_t)(2 * ks), bd + (uint64_t)(2 * ks), idesc, acc0 | (uint32_t)(ks != 0));
              }
            } else {
              // output columns 0..127: Wh[n][k] = Wh[k][n], rows 64 kc.. of chunks 0 and 1, MN-major;
              // output columns 128..Pd-1 (T1 only): rows 128.. of chunk kc are stored, K-major
              const uint32_t idesc_t = ptx::make_idesc_f16(bf, 128, 128, true);
              const uint64_t bt = ptx::make_sw128_mnmajor_desc(ws + (uint32_t)kc * 64u * 128u, Pd * 128u, 1024u);
              const uint32_t idesc_d = ptx::make_idesc_f16(bf, 128, t ? Pd - 128u : 16u, false);
              const uint64_t bd = ptx::make_sw128_kmajor_desc(ws + res_woff((uint32_t)kc, Pd));
              if (ksteps == 4) {
                const uint32_t a_lo = ptx::sw128_kmajor_lo(xs + (uint32_t)kc * Pd * 128u + (t ? 128u * 128u : 0u));
                ptx::umma_f16_elect_k4_bmn(d, a_lo, ptx::sw128_mnmajor_lo(ws + (uint32_t)kc * 64u * 128u, Pd * 128u), idesc_t, acc0);
                if (t) ptx::umma_f16_elect_k4(d + 128u, a_lo, ptx::sw128_kmajor_lo(ws + res_woff((uint32_t)kc, Pd)), idesc_d, acc0);
              } else {
                for (int ks = 0; ks < ksteps; ++ks) {
                  ptx::umma_f16_elect(d, ad + (uint64_t)(2 * ks), bt + (uint64_t)(128 * ks), idesc_t, acc0 | (uint32_t)(ks != 0));
                  if (t) ptx::umma_f16_elect(d + 128u, ad + (uint64_t)(2 * ks), bd + (uint64_t)(2 * ks), idesc_d, acc0 | (uint32_t)(ks != 0));
                }
              }
            }
          }
        };
        const int klo = s.two ? 2 : s.nkc;            // chunks [0, klo) = columns 0..127; single tile: everything
        for (int32_t k = 0; k < a.max_iter; ++k) {
          if (k == a.switch_iter) bf = false;     // 0 < switch_iter < max_iter (host-checked), tol <= 0
          // ---- product 1
          if (k > 0) { ptx::mbar_wait(b_x0, p_x0, a.err_flag, 24); p_x0 ^= 1u; ptx::tc_fence_after(); }
          p1(0, 0, min(klo, s.nkc), true);
          if (k > 0) { ptx::mbar_wait(b_x1, p_x1, a.err_flag, 24); p_x1 ^= 1u; ptx::tc_fence_after(); }
          if (s.two) {
            p1(1, 0, s.nkc, true);
            ptx::umma_commit_elect(b_tfull1);
            p1(0, klo, s.nkc, false);
          }
          ptx::umma_commit_elect(b_tfull0);
          // ---- product 2
          ptx::mbar_wait(b_w1, p_w1, a.err_flag, 23); p_w1 ^= 1u;
          ptx::tc_fence_after();
          if (s.two) { p2(0, klo, s.nkc, true); p2(1, klo, s.nkc, true); }
          ptx::mbar_wait(b_w0, p_w0, a.err_flag, 23); p_w0 ^= 1u;
          ptx::tc_fence_after();
          bool last = k + 1 == a.max_iter;
          if (a.tol > 0.0 && residual_now(s.m) < a.tol) last = true;
          p2(0, 0, min(klo, s.nkc), !s.two);
          ptx::umma_commit_elect(b_tfull0);
          if (s.two) { p2(1, 0, klo, false); ptx::umma_commit_elect(b_tfull1); }
          if (last) {
            // nothing follows this submatrix: consume the two X' barriers so that the parities stay in step
            ptx::mbar_wait(b_x0, p_x0, a.err_flag, 24); p_x0 ^= 1u;
            ptx::mbar_wait(b_x1, p_x1, a.err_flag, 24); p_x1 ^= 1u;
            ptx::tc_fence_after();
            break;
          }
        }
      }
    }
  } else {
    // ===================== epilogue (warps 2..17) =====================
    const int w = warp - 2;
    const int q = warp & 3;                       // TMEM lane quadrant this warp may access
    const int sub = w >> 2;                       // which column blocks of the quadrant's rows it takes
    uint32_t p_xload = 0, p_t[2] = {0, 0}, p_w0 = 0, p_x0 = 0, p_x1 = 0;
    for (;;) {
      ptx::mbar_wait(b_xload, p_xload, a.err_flag, 25); p_xload ^= 1u;
      const int64_t c = *cur_c;
      if (c < 0) break;
      const Sub s = sub_of(c);
      const uint32_t Pd = (uint32_t)s.Pd;
      int32_t iters_done = 0; double r_last = 0.0;
      bool bf = BF16_IN;
      for (int32_t k = 0; k < a.max_iter; ++k) {
        // one pass over this warp's blocks of both tiles; P2 = false: Wh from Y, P2 = true: X' = acc + X.
        // A 32 x 32 block is read as 4 x 4 tiles of 8 x 8 in the mma fragment layout (tile (ti, tj): this lane holds
        // row 8 ti + g, columns 8 tj + 2 q2, +1), so that after packing pairs every tile is one register and four
        // tiles are one stmatrix: the direct store of a block is four stmatrix.x4 (one 8-row strip each), the mirrored
        // store four stmatrix.x4.trans (one 8-column strip each, transposed in flight) -- instead of 32 two-byte
        // stores with their address arithmetic (ncu, first version of this kernel: 530 instructions per block, the
        // epilogue issue-bound on the sub-partition of the lowest rows).
        // RES: accumulate the residual partial sums (product 1; fixed counts need them only in the last step)
        auto pass = [&](const bool P2, const bool bf_out, const bool RES, float &res) {
          float res2 = 0.f;
          const int g = lane >> 2, q2 = lane & 3, rl = lane & 7, ml = lane >> 3;
          for (int tt = 0; tt < (s.two ? 2 : 1); ++tt) {
            const int t = (s.two && !P2) ? 1 - tt : tt;             // the order the MMAs of this product were issued in
            ptx::mbar_wait(t ? b_tfull1 : b_tfull0, p_t[t], a.err_flag, 26); p_t[t] ^= 1u;
            ptx::tc_fence_after();
            const int32_t R0 = 128 * t + 32 * q;
            if (R0 < s.Pd) {
            const uint32_t taddr = tmem_base + (t ? 128u : (P2 ? 384u : 0u)) + ((uint32_t)(q * 32) << 16);
            const uint32_t rb = ((uint32_t)R0 & 63u) >> 3;            // first 16-byte chunk of columns R0.. in their line
            for (int bi = sub; bi * 32 <= R0; bi += RES_EPI_WARPS / 4) {
              const int32_t C0 = bi * 32;
              uint32_t v[2][16];
              ptx::tmem_ld_16x256b_x4(taddr + (uint32_t)C0, v[0]);                    // rows R0 + {g, g + 8}
              ptx::tmem_ld_16x256b_x4(taddr + (16u << 16) + (uint32_t)C0, v[1]);      // rows R0 + 16 + {g, g + 8}
              const uint32_t kcd = (uint32_t)C0 >> 6, cb = ((uint32_t)C0 & 63u) >> 3;
              // shared address of (row R0 + rl, chunk cb + ml): strip ti adds 8 ti rows
              const uint32_t dbase = (P2 ? xs + kcd * Pd * 128u : ws + res_woff(kcd, Pd) - res_lt0(kcd) * 128u) +
                                     ((uint32_t)(R0 + rl)) * 128u + (((cb + (uint32_t)ml) ^ (uint32_t)rl) << 4);
              uint32_t xf[4][4];
              if (P2) {
#pragma unroll
                for (int ti = 0; ti < 4; ++ti) ptx::ldsm_x4(dbase + ti * 1024u, xf[ti][0], xf[ti][1], xf[ti][2], xf[ti][3]);
              }
              ptx::tmem_ld_wait();
              const bool diag = (C0 == R0);
              uint32_t o[4][4];
              float acc = 0.f;
#pragma unroll
              for (int ti = 0; ti < 4; ++ti) {
#pragma unroll
                for (int tj = 0; tj < 4; ++tj) {
                  float f0 = __uint_as_float(v[ti >> 1][4 * tj + 2 * (ti & 1)]);
                  float f1 = __uint_as_float(v[ti >> 1][4 * tj + 2 * (ti & 1) + 1]);
                  if (!P2) {
                    if (diag) {
                      // row / column inside the block; tiles above the diagonal are not used (overwritten by mirrors)
                      const int rr = 8 * ti + g, c0 = 8 * tj + 2 * q2;
                      if (R0 + rr < s.m) { if (c0 == rr) f0 -= 1.f; if (c0 + 1 == rr) f1 -= 1.f; }   // W = Y - I
                      if (RES && tj <= ti) {
                        if (c0 <= rr) acc = fmaf(c0 == rr ? f0 : 2.f * f0, f0, acc);
                        if (c0 + 1 <= rr) acc = fmaf(c0 + 1 == rr ? f1 : 2.f * f1, f1, acc);
                      }
                    } else if (RES) {
                      acc = fmaf(f0, f0, acc); acc = fmaf(f1, f1, acc);
                    }
                    f0 *= -0.5f; f1 *= -0.5f;
                  } else {
                    const float2 x2 = bf ? unpack2<true>(xf[ti][tj]) : unpack2<false>(xf[ti][tj]);
                    f0 += x2.x; f1 += x2.y;
                  }
                  o[ti][tj] = bf_out ? pack2<true>(f0, f1) : pack2<false>(f0, f1);
                }
              }
              if (!P2) { if (diag) res += acc; else res2 += acc; }
              if (diag) {
                // diagonal tiles: element (r, c > r) := element (c, r), through the transposed fragment
#pragma unroll
                for (int ti = 0; ti < 4; ++ti) {
                  const uint32_t tr = ptx::movmatrix_t(o[ti][ti]);
                  const uint32_t sel = (2 * q2 <= g ? 0x10u : 0x54u) | ((2 * q2 + 1 <= g ? 0x32u : 0x76u) << 8);
                  o[ti][ti] = __byte_perm(o[ti][ti], tr, sel);
                }
              }
              // direct store: four 8-row strips (the upper tiles of a diagonal block hold unused values for now)
#pragma unroll
              for (int ti = 0; ti < 4; ++ti) ptx::stsm_x4(dbase + ti * 1024u, o[ti][0], o[ti][1], o[ti][2], o[ti][3]);
              // mirrored store: tile (ti, tj) transposed -> rows C0 + 8 tj .., columns R0 + 8 ti ...  X' always; Wh only
              // inside the 128 x 128 diagonal squares (the rest of its upper part is not stored).
              if (P2 || C0 >= (R0 & ~127)) {
                const uint32_t kcm = (uint32_t)R0 >> 6;
                const uint32_t mbase = (P2 ? xs + kcm * Pd * 128u : ws + res_woff(kcm, Pd) - res_lt0(kcm) * 128u) +
                                       ((uint32_t)(C0 + rl)) * 128u;
                if (!diag) {
                  const uint32_t ma = mbase + (((rb + (uint32_t)ml) ^ (uint32_t)rl) << 4);
#pragma unroll
                  for (int tj = 0; tj < 4; ++tj) ptx::stsm_x4_t(ma + tj * 1024u, o[0][tj], o[1][tj], o[2][tj], o[3][tj]);
                } else {
                  __syncwarp();       // the direct stores of the upper tiles come first
                  // strictly lower tiles only: column strip 0 -> tiles (1..3, 0), strip 1 -> (2..3, 1), strip 2 -> (3, 2);
                  // the x4 of strip 0 also rewrites the (symmetric) tile (0, 0)
                  ptx::stsm_x4_t(mbase + (((rb + (uint32_t)ml) ^ (uint32_t)rl) << 4), o[0][0], o[1][0], o[2][0], o[3][0]);
                  ptx::stsm_x2_t(mbase + 1024u + (((rb + 2u + (uint32_t)(ml & 1)) ^ (uint32_t)rl) << 4), o[2][1], o[3][1]);
                  ptx::stsm_x1_t(mbase + 2048u + (((rb + 3u) ^ (uint32_t)rl) << 4), o[3][2]);
                }
              }
            }
            }   // R0 < Pd
            // this tile's part of Wh / X' is written and its accumulator drained: tell the MMA issuer.  (The residual
            // partial of the step goes out with the LAST tile of product 1, T0.)
            if (!P2 && t == 0 && RES) {
              float rs = res + 2.f * res2;
              for (int d = 16; d > 0; d >>= 1) rs += __shfl_xor_sync(0xffffffffu, rs, d);
              if (lane == 0) res_s[w] = rs;
            }
            ptx::tc_fence_before();
            ptx::fence_proxy_async_smem();          // generic-proxy stores -> the MMA's async-proxy reads
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(P2 ? (t ? b_x1 : b_x0) : (t ? b_w1 : b_w0));
          }
          if (!s.two && lane == 0) ptx::mbar_arrive(P2 ? b_x1 : b_w1);      // single tile: the T1 barriers complete as well
          res += 2.f * res2;
        };

        // ---- epilogue 1: Wh -> WS, residual
        float res = 0.f;
        bool last = k + 1 == a.max_iter;
        pass(false, bf, a.tol > 0.0 || last, res);
        ptx::mbar_wait(b_w0, p_w0, a.err_flag, 27); p_w0 ^= 1u;        // all 16 partial sums of the step are there
        if (a.tol > 0.0 || last) r_last = residual_now(s.m);          // fixed counts: only the last residual is reported
        if (a.tol > 0.0 && r_last < a.tol) last = true;
        // ---- epilogue 2: X' -> XS (the update that reaches switch_iter writes fp16)
        const bool bf_next = bf && (k + 1 != a.switch_iter);
        float dummy = 0.f;
        pass(true, bf_next, false, dummy);
        bf = bf_next;
        iters_done = k + 1;
        // the partial sums of this step are consumed by every role before any warp can rewrite its slot: a warp
        // rewrites it in the next step's epilogue 1, which follows MMAs that the issuer starts only after b_x0 / b_x1,
        // i.e. after every warp has passed this point
        if (last || k + 1 == a.max_iter) {
          ptx::mbar_wait(b_x0, p_x0, a.err_flag, 28); ptx::mbar_wait(b_x1, p_x1, a.err_flag, 28);
        }
        p_x0 ^= 1u; p_x1 ^= 1u;
        if (last) break;
      }
      if (w == 0 && lane == 0) {
        // the final iterate leaves the SM: one bulk store of the whole image
        char *dst = (char *)a.X + a.col_off[c] * 2;
        for (uint32_t off = 0; off < Pd * Pd * 2u; off += Pd * 128u) ptx::tma_bulk_s2g(dst + off, xs + off, Pd * 128u);
        ptx::bulk_commit();
        a.iters[c] = iters_done;
        a.residual[c] = r_last;
        ptx::bulk_wait_read0();
        ptx::mbar_arrive(b_free);
      }
    }
    if (w == 0 && lane == 0) ptx::bulk_wait0();
  }

  ptx::tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc(tmem_base, 512);
  }
}
