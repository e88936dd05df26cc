// a3, bf16 / fp16, fused variant (included by sign_umma.cu inside namespace sm; uses its tile geometry,
// UCfg<2>, pack2/unpack2, store_row_segment and mirror_store).
//
// Fixed iteration count, CTA pairs (cta_group::2), SYM: a CTA pair takes ONE submatrix through all
// max_iter Newton-Schulz steps (Eq. 13; iteration X <- 1/2 X (3I - X^2), A9) before
// it moves to the next, so that X_k, W and X_{k+1} of the 74 submatrices in flight (~1.2 MB each at
// m ~ 410) stay in the 126 MB L2 instead of streaming through HBM twice per step.  (ncu, round 1,
// configs[2]: the per-phase launches move 2.6 + 4.1 GB of DRAM traffic per step; at 0.4 m FLOP per byte
// the per-phase design is HBM bound below m ~ 600.)  Tiles, operand staging, MMA issue and the epilogue
// are those of k_umma_gemm<.., 2, true>; what is new is the loop nest (submatrix -> step -> phase ->
// tile) and the hand-over between phases: the epilogue warps of both CTAs arrive on `pdone` (release,
// cluster scope, after a gpu-scope fence and a generic->async proxy fence) once their stores of a phase
// are issued, and the two TMA producers wait on it (acquire) before they load the next phase's
// operands.  The last phase of a submatrix has no arrival: the next submatrix does not depend on it.
// Submatrices are dealt to the pairs boustrophedon over the caller's list (sorted by size in
// sm_density), which balances the m^3 work of a size-sorted list to within one submatrix.
#pragma once

struct FArgs {
  const int32_t *cols; const int64_t *col_off; const int32_t *dim; const int32_t *dim_pad;
  int32_t n_cols, max_iter;
  void *X; void *X2; void *W;
  double *partial; int32_t parts_per_col;
  int32_t *err_flag;
  unsigned long long *trace;   // measurement only (SM_UMMA_TRACE): clock64 time line of CTA pair 0, second submatrix
  int32_t dbg;                 // measurement only (SM_UMMA_DBG): 1 = no phase hand-over (wrong results), 2 = no gpu-scope fence, 8 = skip the epilogue's work, 16 / 32 = skip the direct / mirrored stores of off-diagonal blocks
};

// One submatrix of the caller's list as the fused kernel sees it.
struct FSub { int64_t c, base; int32_t m, Pd, valid; };
__device__ __forceinline__ FSub fused_sub(const FArgs &a, int64_t c) {
  FSub s; s.c = c; s.valid = c < a.n_cols ? 1 : 0; s.base = 0; s.m = 0; s.Pd = 0;
  if (s.valid) {
    const int32_t i = a.cols ? a.cols[c] : (int32_t)c;
    s.m = a.dim[i]; s.Pd = a.dim_pad[i]; s.base = a.col_off[c];
  }
  return s;
}

__device__ __forceinline__ int64_t fused_pick(int64_t unit, int64_t n_units, int32_t round) {
  return (int64_t)round * n_units + ((round & 1) ? (n_units - 1 - unit) : unit);
}

// Trace layout: [cta 0..1][role 0..3][TRACE_N] x (clock64, tag); role 0 producer, 1 MMA issuer, 2 first, 3 last
// epilogue warp.  tag = code << 32 | phase << 8 | tile.
constexpr int TRACE_N = 1024;
struct Tracer {
  unsigned long long *p; int n;
  __device__ __forceinline__ void operator()(unsigned code, int32_t ph, int32_t tile) {
    if (p && n < TRACE_N) {
      p[2 * n] = (unsigned long long)clock64();
      p[2 * n + 1] = ((unsigned long long)code << 32) | (unsigned)(ph << 8) | (unsigned)tile;
      ++n;
    }
  }
};

// NSLOT = 2: a pair works on two submatrices at a time, alternating between them phase by phase, so that the
// tail of one (last epilogue, fences, hand-over, first loads: ~13k of ~36k cycles per phase on the clock64 time
// line) is covered by the other's main loop.
template <bool BF16, int NSLOT>
__global__ void __launch_bounds__(UMMA_THREADS, 1) k_umma_fused(FArgs a) {
  using Cfg = UCfg<2>;
  constexpr int USTAGES = Cfg::STAGES;
  constexpr int STAGE_BYTES = Cfg::STAGE_BYTES;
  constexpr int R = Cfg::ROWS;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = ptx::smem_u32(smem_raw);
  const uint32_t tiles = (raw + 1023u) & ~1023u;
  const uint32_t stage_base = tiles + USTAGES * STAGE_BYTES;
  const uint32_t ident = stage_base + EPI_STAGE_BYTES;
  const uint32_t bars = ident + IDENT_BYTES;
  auto full_bar = [&](int s) { return bars + 8u * s; };
  auto empty_bar = [&](int s) { return bars + 8u * (USTAGES + s); };
  auto pfull_bar = [&](int s) { return bars + 8u * (2 * USTAGES + s); };
  auto tfull_bar = [&](int s) { return bars + 8u * (3 * USTAGES + s); };
  auto tempty_bar = [&](int s) { return bars + 8u * (3 * USTAGES + NACC + s); };
  const uint32_t tmem_slot = bars + 8u * (3 * USTAGES + 2 * NACC);
  auto pdone_bar = [&](int sl) { return tmem_slot + 8u + 8u * sl; };   // one per interleaved submatrix slot
  volatile uint32_t *tmem_slot_ptr = reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - raw));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t h = ptx::cluster_ctarank();
  const int64_t unit = blockIdx.x / 2, n_units = gridDim.x / 2;

  ident_fill<BF16>(smem_raw + (ident - raw), true, h, (int)threadIdx.x, UMMA_THREADS);
  ptx::fence_proxy_async();       // generic-proxy writes -> the MMA's async-proxy reads
  if (threadIdx.x == 0) {
    for (int s = 0; s < USTAGES; ++s) {
      ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), 1); ptx::mbar_init(pfull_bar(s), 1);
    }
    for (int s = 0; s < NACC; ++s) { ptx::mbar_init(tfull_bar(s), 1); ptx::mbar_init(tempty_bar(s), EPI_WARPS * 2); }
    ptx::mbar_init(pdone_bar(0), EPI_WARPS * 2); ptx::mbar_init(pdone_bar(1), EPI_WARPS * 2);
    ptx::fence_barrier_init();
    ptx::fence_proxy_async();
  }
  if (warp == 1) { ptx::tmem_alloc2(tmem_slot, TMEM_COLS); ptx::tmem_relinquish2(); }
  ptx::tc_fence_before();
  ptx::cluster_sync_all();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  const int32_t n_rounds = (int32_t)((a.n_cols + n_units - 1) / n_units);
  const int32_t n_ph = 2 * a.max_iter;
  const int32_t trd = max(1, a.dbg >> 8);   // traced round (SM_UMMA_DBG bits 8+; default: the pair's second submatrix)
  unsigned long long *const trace0 = (a.trace && unit == 0) ? a.trace + (size_t)h * 4 * TRACE_N * 2 : nullptr;

  if (warp == 0) {
    // ===================== TMA producer =====================
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0, dphase[2] = {0, 0};
      Tracer tr{trace0, 0};
      for (int32_t rd0 = 0; rd0 < n_rounds; rd0 += NSLOT) {
        FSub S[2] = {fused_sub(a, fused_pick(unit, n_units, rd0)),
                     fused_sub(a, NSLOT > 1 && rd0 + 1 < n_rounds ? fused_pick(unit, n_units, rd0 + 1) : a.n_cols)};
        for (int32_t ph = 0; ph < n_ph; ++ph)
        for (int sl = 0; sl < NSLOT; ++sl) {
          if (!S[sl].valid) continue;
          const int32_t rd = rd0 + sl;
          const int32_t m = S[sl].m, Pd = S[sl].Pd;
          const int64_t boff = S[sl].base * 2;
          const int32_t kmax = u_n16(m), nkc = (kmax + UK - 1) / UK, Tm = u_Tm(m, R);
          const char *src = (const char *)(((ph >> 1) & 1) ? a.X2 : a.X) + boff;
          const char *Bg = (ph & 1) ? (const char *)a.W + boff : src;
          if (ph > 0 && !(a.dbg & 1)) {
            // every store of the previous phase (both CTAs) is visible before this phase's bulk copies read it
            ptx::mbar_wait_cluster(pdone_bar(sl), dphase[sl], a.err_flag, 7);
            dphase[sl] ^= 1u;
            ptx::fence_proxy_async();
            if (rd == trd) tr(1, ph, 0);
          }
          for (int32_t tm = 0; tm < Tm; ++tm) {
            const int32_t cnt = u_row_tiles(m, R, tm), nb = u_row_nb(m, R, tm), nc = u_ncols(m, R, tm);
            const int32_t arow0 = tm * R + (int32_t)h * UM;
            const uint32_t a_bytes = (uint32_t)max(0, min(UM, Pd - arow0)) * 128u;
            for (int32_t tn = 0; tn < cnt; ++tn) {
              const int32_t n0 = tn * nb, nt = min(nb, nc - n0);
              const int32_t b_cnt = nt / 2, brow0 = n0 + (int32_t)h * b_cnt;
              const uint32_t b_bytes = (uint32_t)b_cnt * 128u;
              for (int kc = 0; kc < nkc; ++kc) {
                ptx::mbar_wait(empty_bar(stage), phase ^ 1u, a.err_flag, 1);
                const uint32_t sa = tiles + stage * STAGE_BYTES, sb = sa + A_BYTES;
                if (rd == trd && kc == 0) tr(2, ph, tm * 4 + tn);
                ptx::mbar_expect_tx(full_bar(stage), a_bytes + b_bytes);
                const int64_t chunk = (int64_t)kc * Pd * 128;
                if (a_bytes) ptx::tma_bulk_g2s(sa, src + chunk + (int64_t)arow0 * 128, a_bytes, full_bar(stage));
                ptx::tma_bulk_g2s(sb, Bg + chunk + (int64_t)brow0 * 128, b_bytes, full_bar(stage));
                if (++stage == USTAGES) { stage = 0; phase ^= 1u; }
              }
            }
          }
          if (rd == trd) tr(3, ph, 0);
        }
      }
    }
  } else if (warp == 1 && h != 0) {
    // ===================== relay (peer CTA): tell the leader that this CTA's stage landed ======
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      for (int32_t rd = 0; rd < n_rounds; ++rd) {
        const FSub S = fused_sub(a, fused_pick(unit, n_units, rd));
        if (!S.valid) continue;
        const int32_t m = S.m;
        const int32_t nkc = (u_n16(m) + UK - 1) / UK;
        const int64_t n_chunks = (int64_t)u_tiles(m, R) * nkc * n_ph;     // stage uses, in whatever order
        for (int64_t q = 0; q < n_chunks; ++q) {
          ptx::mbar_wait(full_bar(stage), phase, a.err_flag, 5);
          ptx::mbar_arrive_remote(pfull_bar(stage), 0);
          if (++stage == USTAGES) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA) =====================
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0, it = 0;
      Tracer tr{trace0 ? trace0 + 1 * TRACE_N * 2 : nullptr, 0};
      for (int32_t rd0 = 0; rd0 < n_rounds; rd0 += NSLOT) {
        FSub S[2] = {fused_sub(a, fused_pick(unit, n_units, rd0)),
                     fused_sub(a, NSLOT > 1 && rd0 + 1 < n_rounds ? fused_pick(unit, n_units, rd0 + 1) : a.n_cols)};
        for (int32_t ph = 0; ph < n_ph; ++ph)
        for (int sl = 0; sl < NSLOT; ++sl) {
          if (!S[sl].valid) continue;
          const int32_t rd = rd0 + sl;
          const int32_t m = S[sl].m;
          const int32_t kmax = u_n16(m), nkc = (kmax + UK - 1) / UK, Tm = u_Tm(m, R);
          for (int32_t tm = 0; tm < Tm; ++tm) {
            const int32_t cnt = u_row_tiles(m, R, tm), nb = u_row_nb(m, R, tm), nc = u_ncols(m, R, tm);
            for (int32_t tn = 0; tn < cnt; ++tn) {
              const int32_t n0 = tn * nb, nt = min(nb, nc - n0);
              const uint32_t as = it % NACC, aphase = (it / NACC) & 1u;
              ptx::mbar_wait(tempty_bar(as), aphase ^ 1u, a.err_flag, 2);
              if (rd == trd) tr(4, ph, tm * 4 + tn);
              ptx::tc_fence_after();
              const uint32_t d_tmem = tmem_base + as * UN;
              const uint32_t idesc = ptx::make_idesc_f16(BF16, R, (uint32_t)nt, false);
              for (int kc = 0; kc < nkc; ++kc) {
                ptx::mbar_wait(full_bar(stage), phase, a.err_flag, 3);
                ptx::mbar_wait(pfull_bar(stage), phase, a.err_flag, 6);
                if (rd == trd && (kc == 0 || kc == nkc - 1)) tr(kc == 0 ? 5 : 10, ph, tm * 4 + tn);
                ptx::tc_fence_after();
                const uint32_t sa = tiles + stage * STAGE_BYTES, sb = sa + A_BYTES;
                const uint64_t adesc = ptx::make_sw128_kmajor_desc(sa), bdesc = ptx::make_sw128_kmajor_desc(sb);
                const int ksteps = min(UK / 16, (kmax - kc * UK) / 16);
                for (int ks = 0; ks < ksteps; ++ks)
                  ptx::umma_f16_2cta(d_tmem, adesc + (uint64_t)(2 * ks), bdesc + (uint64_t)(2 * ks), idesc,
                                     (uint32_t)((kc | ks) != 0));
                if (ph & 1) {
                  // "+ X": add the A chunk X[rows, 64 kc ..] to the accumulator columns [lo, hi) it covers
                  const int32_t lo = max(kc * UK, n0), hi = min(kc * UK + UK, n0 + nt);
                  if (lo < hi) {
                    const uint32_t idesc2 = ptx::make_idesc_f16(BF16, R, (uint32_t)(hi - lo), false);
                    const uint64_t idd = ptx::make_sw128_kmajor_desc(ident + ident_row(true, lo - kc * UK, hi - lo) * 128u);
                    for (int ks = 0; ks < UK / 16; ++ks)
                      ptx::umma_f16_2cta(d_tmem + (uint32_t)(lo - n0), adesc + (uint64_t)(2 * ks), idd + (uint64_t)(2 * ks),
                                         idesc2, 1u);
                  }
                }
                ptx::umma_commit_2cta(empty_bar(stage));
                if (++stage == USTAGES) { stage = 0; phase ^= 1u; }
              }
              ptx::umma_commit_2cta(tfull_bar(as));
              if (rd == trd) tr(6, ph, tm * 4 + tn);
              ++it;
            }
          }
        }
      }
    }
  } else {
    // ===================== epilogue (warps 2..17), block handling as in k_umma_gemm =====================
    constexpr int NSUB = EPI_WARPS / 4;
    const int q = warp & 3;
    const int sub = (warp - 2) >> 2;
    uint16_t *const stg0 = reinterpret_cast<uint16_t *>(smem_raw + (stage_base - raw)) + q * NACC * 1024;
    const uint32_t r7 = (uint32_t)lane & 7u;
    const bool swp = (lane & 1) != 0;
    uint32_t it = 0;
    Tracer tr{(trace0 && lane == 0 && (warp == 2 || warp == 17)) ? trace0 + (warp == 2 ? 2 : 3) * TRACE_N * 2 : nullptr, 0};
    for (int32_t rd0 = 0; rd0 < n_rounds; rd0 += NSLOT) {
      FSub S[2] = {fused_sub(a, fused_pick(unit, n_units, rd0)),
                   fused_sub(a, NSLOT > 1 && rd0 + 1 < n_rounds ? fused_pick(unit, n_units, rd0 + 1) : a.n_cols)};
      for (int32_t ph = 0; ph < n_ph; ++ph)
      for (int sl = 0; sl < NSLOT; ++sl) {
        if (!S[sl].valid) continue;
        const int32_t rd = rd0 + sl;
        const int64_t c = S[sl].c, base = S[sl].base;
        const int32_t m = S[sl].m, Pd = S[sl].Pd;
        const int32_t Tm = u_Tm(m, R);
        const bool p2 = (ph & 1) != 0;                  // false: Wh = -1/2 (X X^T - I), true: X' = X + X Wh
        const bool odd = ((ph >> 1) & 1) != 0;
        uint16_t *Og = (p2 ? (uint16_t *)(odd ? a.X : a.X2) : (uint16_t *)a.W) + base;
        int32_t lt = 0;
        for (int32_t tm = 0; tm < Tm; ++tm) {
          const int32_t cnt = u_row_tiles(m, R, tm), nb = u_row_nb(m, R, tm), nc = u_ncols(m, R, tm);
          const int32_t R0 = tm * R + (int32_t)h * UM + q * 32;
          const int32_t r = R0 + lane;
          for (int32_t tn = 0; tn < cnt; ++tn, ++lt) {
            const int32_t n0 = tn * nb, nt = min(nb, nc - n0);
            const uint32_t as = it % NACC, aphase = (it / NACC) & 1u;
            const int nblk = (nt + 31) >> 5;
            uint16_t *const stg = stg0 + as * 1024;      // diagonal-block buffer of (quadrant, accumulator stage)
            ptx::mbar_wait(tfull_bar(as), aphase, a.err_flag, 4);
            if (rd == trd) tr(7, ph, tm * 4 + tn);
            ptx::tc_fence_after();
            const uint32_t taddr = tmem_base + as * UN + ((uint32_t)(q * 32) << 16);
            float res = 0.f, res2 = 0.f;
            if (R0 < Pd && !(a.dbg & 8)) {
              for (int bi = sub; bi < nblk; bi += NSUB) {
                const int32_t C0 = n0 + bi * 32;
                if (C0 > R0) break;
                uint32_t v[32];
                ptx::tmem_ld16(taddr + (uint32_t)(bi * 32), *reinterpret_cast<uint32_t(*)[16]>(&v[0]));
                ptx::tmem_ld16(taddr + (uint32_t)(bi * 32 + 16), *reinterpret_cast<uint32_t(*)[16]>(&v[16]));
                const int64_t rowoff = (int64_t)(C0 >> 6) * Pd * 64 + (int64_t)r * 64;
                const uint32_t c8 = ((uint32_t)C0 >> 3) & 4u;
                const uint32_t sec0 = ((c8 ^ r7) & ~1u) << 3, sec1 = (((c8 + 2u) ^ r7) & ~1u) << 3;
                ptx::tmem_ld_wait();
                const bool diag = (C0 == R0);
                uint32_t o[16];
                float acc = 0.f;
#pragma unroll
                for (int g = 0; g < 4; ++g) {
                  float f[8];
#pragma unroll
                  for (int e = 0; e < 8; ++e) f[e] = __uint_as_float(v[g * 8 + e]);
                  if (!p2) {
                    if (diag && r < m) {
#pragma unroll
                      for (int e = 0; e < 8; ++e)
                        if (g * 8 + e == lane) f[e] -= 1.f;
                    }
                    if (diag) {
#pragma unroll
                      for (int e = 0; e < 8; ++e) {
                        const int j = g * 8 + e;
                        if (j <= lane) acc = fmaf(j == lane ? f[e] : 2.f * f[e], f[e], acc);
                      }
                    } else {
#pragma unroll
                      for (int e = 0; e < 8; ++e) acc = fmaf(f[e], f[e], acc);
                    }
#pragma unroll
                    for (int e = 0; e < 8; ++e) f[e] *= -0.5f;       // Wh = -1/2 W (see ident_fill)
                  }
#pragma unroll
                  for (int e2 = 0; e2 < 4; ++e2) o[g * 4 + e2] = pack2<BF16>(f[2 * e2], f[2 * e2 + 1]);
                }
                if (!p2 && r < m) { if (!diag) res2 += acc; else res += acc; }
                uint16_t *Orow = Og + rowoff;
                if (diag) {
#pragma unroll
                  for (int g = 0; g < 4; ++g)
                    *reinterpret_cast<uint4 *>(stg + lane * 32 + ((g ^ (lane & 3)) << 3)) =
                        make_uint4(o[g * 4], o[g * 4 + 1], o[g * 4 + 2], o[g * 4 + 3]);
                  __syncwarp();
#pragma unroll
                  for (int j = 0; j < 32; ++j) {
                    if (j > lane) {
                      const uint16_t m16 = stg[j * 32 + (((lane >> 3) ^ (j & 3)) << 3) + (lane & 7)];
                      o[j >> 1] = (j & 1) ? ((o[j >> 1] & 0x0000FFFFu) | ((uint32_t)m16 << 16))
                                          : ((o[j >> 1] & 0xFFFF0000u) | (uint32_t)m16);
                    }
                  }
                  __syncwarp();
                  store_row_segment(Orow, sec0, sec1, swp, o);
                } else {
                  if (!(a.dbg & 16)) store_row_segment(Orow, sec0, sec1, swp, o);
                  if (!(a.dbg & 32)) mirror_store(Og, Pd, R0, C0, lane, o);
                }
              }
            }
            res += 2.f * res2;
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive_remote(tempty_bar(as), 0);
            if (rd == trd) tr(8, ph, tm * 4 + tn);
            if (!p2) {
              for (int d = 16; d > 0; d >>= 1) res += __shfl_xor_sync(0xffffffffu, res, d);
              if (lane == 0)
                a.partial[c * a.parts_per_col + (int64_t)lt * (EPI_WARPS * 2) + (int64_t)h * EPI_WARPS + (warp - 2)] =
                    (double)res;
            }
            ++it;
          }
        }
        if (ph + 1 < n_ph && !(a.dbg & 1)) {
          // this warp's stores of the phase: visible gpu-wide and to the async proxy, then tell both producers
          if (!(a.dbg & 2)) __threadfence();
          ptx::fence_proxy_async();
          __syncwarp();
          if (lane == 0) {
            ptx::mbar_arrive_cluster(pdone_bar(sl), 0);
            ptx::mbar_arrive_cluster(pdone_bar(sl), 1);
          }
          if (rd == trd) tr(9, ph, 0);
        }
      }
    }
  }

  ptx::tc_fence_before();
  __syncwarp();
  ptx::cluster_sync_all();
  if (warp == 1) {
    ptx::tc_fence_after();
    ptx::tmem_dealloc2(tmem_base, TMEM_COLS);
  }
}
