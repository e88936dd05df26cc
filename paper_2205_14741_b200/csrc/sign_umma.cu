// a3, bf16 / fp16 back end: Newton-Schulz X <- 1/2 X (3I - X^2) as grouped tcgen05 GEMMs over ragged
// submatrices ("FP16 operations with FP32 accumulation"; "evaluation of the matrix
// function on many dense ... matrices", PAPER.md:106/:110 step 2; Eq. 13).
//
// Data layout: every submatrix is stored in HBM as the K-major 128B-swizzled UMMA shared-memory
// image (include/submatrix.h), so an operand tile (rows x 64 k) is ONE contiguous bulk-TMA copy and
// no tensor map is needed for ragged sizes.  X is symmetric, so the same image serves as the A
// operand (rows of X) and as the B operand (B[n][k] = X[k][n] = X[n][k]): both products are
// "A K-major, B K-major" and read row panels only.
//
// Symmetry is enforced exactly: only elements (r, c) with r >= c are taken from the accumulator and
// each is stored twice, at (r, c) and mirrored at (c, r); tiles that lie entirely above the diagonal
// are never computed.  This is required, not just cheaper: with rounded iterates the X X^T form
// amplifies any antisymmetric perturbation by ~2x per step (measured: NaN after ~18 bf16 steps),
// while exactly symmetric iterates make X X^T == X^2 and keep the iteration on Eq. 13's fixed point.
//
// Kernel: persistent, one CTA per SM, 576 threads = 1 TMA producer warp (warp-convergent: one elected lane issues the
// bulk copies), 1 MMA issuer warp (also owns TMEM; elected-lane issue), 16 epilogue warps (4 per TMEM lane quadrant).
// Tile = 128 x (<=256) fp32 accumulator in TMEM, double buffered (2 x 256 columns) so the epilogue of tile t overlaps
// the main loop of tile t+1; 4-stage smem ring of 48 KB stages; tiles handed out by a global counter.
//   PHASE 1: Y = X X^T; the epilogue stores Wh = -1/2 (Y - I) and the fused ||Y - I||_F^2 partial sums (warp shuffles).
//            A tile that holds its panel's diagonal square reads its A rows from the B rows it stages (share_a_off).
//   PHASE 2: X' = X + X Wh as ONE accumulation (identity MMAs add X); the epilogue only converts and stores.
#include <cuda.h>   // CUtensorMap (type only; the encoder is fetched through cudaGetDriverEntryPoint)
#include <cstdio>
#include <cstdlib>
#include <utility>
#include <vector>

#include "sign_state.cuh"
#include "umma_ptx.cuh"

// Measurement-only skip knobs (wrong results by construction) exist only in a -DSM_MEASURE build
// (build.py --measure); the default library has no such path.
#ifdef SM_MEASURE
#define SM_DBG(a, bit) ((a).dbg & (bit))
#else
#define SM_DBG(a, bit) 0
#endif

namespace sm {

constexpr int UM = 128;          // tile rows per CTA (UMMA M per CTA)
#ifndef SM_UN
#define SM_UN 256
#endif
constexpr int UN = SM_UN;        // max tile cols (UMMA N)
constexpr int NACC = 512 / UN;   // accumulator stages in TMEM (512 columns)
constexpr int UK = 64;           // k chunk = one 128-byte swizzle row of 16-bit elements
constexpr int A_BYTES = UM * UK * 2;           // 16 KB
constexpr int EPI_WARPS = 16;
constexpr int EPI_STAGE_BYTES = 4 * NACC * 2048;    // 32 x 32 x 2 B buffer per (TMEM lane quadrant, accumulator stage): diagonal blocks only
constexpr int IDENT_BYTES = 8192;                   // 64 x 64 identity image(s): B operand that folds "+ X" into the update product
constexpr int UMMA_THREADS = 64 + 32 * EPI_WARPS;
constexpr uint32_t TMEM_COLS = 512;

// NCTA = 1: one CTA per tile of 128 x (<=256).  NCTA = 2: a CTA pair (cta_group::2) per tile of
// 256 x (<=256): each CTA stages its own 128 rows of A and HALF of the B rows, so a pair moves
// (256 + nt) rows per k chunk for 256 x nt outputs instead of 2 x (128 + nt): the L2 -> SM bytes per
// FLOP drop by 1.5x at nt = 256 (ncu, round 1: the single-CTA kernel sits on the L2 throughput cap).
//
// MC (NCTA = 2 only): the same 256-row tile geometry, but each CTA issues its own cta_group::1 MMAs on its
// 128 rows with the WHOLE B tile in its shared memory; each CTA fetches half of the B rows and multicasts
// them to both (cp.async.bulk ... multicast::cluster), so the L2 -> SM bytes equal those of the cta_group::2
// pair while no CTA waits on a relayed "peer's stage landed" signal.
// NST: depth of the operand ring (0 = the default of the variant).  Measured on B200, sm_sign_ns alone: at
// configs[4] (m ~ 1650) single CTAs run 25 steps in 653 ms with 3 stages and 747 ms with 4 (2 stages: 734 ms) --
// a shallower ring keeps the CTAs that share a submatrix's operand panels closer together in L2 --
// while configs[2] (m ~ 410) prefers 4 (27.8 vs 28.7 ms).
// EPI = 1: staged epilogue (two 32 KB output staging buffers, bulk stores; the ring then has 3 stages).
constexpr int EPI_STG_UNIT = 32768;
template <int NCTA, bool MC = false, int NST = 0, int EPI = 0> struct UCfg {
  static constexpr bool G2 = NCTA == 2 && !MC;             // cta_group::2 MMA
  static constexpr int STAGES = NST ? NST : (EPI ? 3 : (G2 ? 6 : 4));
  static constexpr int B_BYTES = (G2 ? UN / 2 : UN) * UK * 2;   // 16 KB / 32 KB
  static constexpr int STAGE_BYTES = A_BYTES + B_BYTES;    // 48 KB / 32 KB
  static constexpr int EPI_BYTES = EPI ? 2 * EPI_STG_UNIT : EPI_STAGE_BYTES;
  static constexpr int SMEM = STAGES * STAGE_BYTES + EPI_BYTES + IDENT_BYTES + 1024 /*align slack*/ + 512 /*barriers, tile queue*/;
  static constexpr int ROWS = UM * NCTA;                   // tile rows
};

struct UTile {
  int32_t c, m, Pd, row0, n0, nt, kmax, lt, valid;
  int32_t fb, fs;   // folded geometry: tile column (virtual index) v >= fb is column v + fs of the matrix (fb = INT_MAX: none)
  int64_t base;   // element offset of the submatrix in the packed buffer
};

// One entry per output tile, built once per sm_sign_ns call (k_umma_build_tiles) so that the
// persistent roles fetch a tile with three 16-byte loads instead of a dependent binary search
// (ncu, round 1: the search's long-scoreboard stalls were the top stall of every role).
struct __align__(16) TileDesc {
  int64_t base;                  // element offset of the submatrix in the packed buffer
  int32_t c, m;                  // listed-column index, true dimension
  int32_t Pd, row0, n0, nt;      // padded dimension, first row, first column, columns of the tile
  int32_t lt, pad0, pad1, pad2;  // tile index inside its submatrix
};

struct UArgs {
  const int32_t *cols; const int64_t *col_off; const int32_t *dim; const int32_t *dim_pad;
  const int64_t *tile_ptr;   // [n_cols+1] exclusive scan of tiles per listed column
  const TileDesc *tiles;     // [tile_ptr[n_cols]]
  int32_t n_cols;
  int32_t check_flags;       // convergence mode: per-submatrix active/last flags are consulted
  const void *Xsrc; const void *Ybuf; void *Out;
  SignState s;
  int32_t *err_flag;
  int32_t rev;               // walk the tile table backwards (alternates per launch)
  unsigned long long *counter;   // DYN: this launch's tile counter (zeroed by the host)
  // PHASE = 0 ("stream": every product of every step in ONE launch; Xsrc / Out are the two X buffers, Ybuf is Wh):
  int32_t n_ph;              // 2 * steps
  int32_t *done;             // [groups][n_ph] epilogue-warp completions of (group, product), zeroed by the host
  int32_t dbg;               // measurement only (SM_UMMA_DBG): 1 = skip output stores, 2 = skip MMA issue, 4 = skip TMA loads, 8 = skip the epilogue's work
  // staged epilogue only (EPI = 1): "128-lower" storage of the iterates.  lt_in: the operands hold valid data only at
  // (r, c) with r >= (c & ~127) -- everything on or below the 128 x 128 diagonal squares -- and the rest is read
  // through the transpose (MN-major descriptors over the rows 64 kc .. of the chunk that holds the wanted columns);
  // lt_out: the output is written that way (no mirrored pieces below the diagonal squares).  The last update of a
  // submatrix writes the full image (lt_out = 0, or s.last in convergence mode): sm_scatter reads whole rows.
  int32_t lt_in, lt_out;
  int32_t out_f16;           // precision schedule (f3): this launch reads bf16 operands and rounds its output to fp16
  // third-order iteration (f3, reading A22): product 1 stores Q = w_scale (Y - I) (-1/2: Newton-Schulz; -3/4: order 3),
  // the update-type product scales its accumulator by out_scale (1; 2/3 for Z = 2/3 (Q + Q Q))
  float w_scale, out_scale;
  int32_t no_ident;          // update product without its "+ X" (identity MMAs skipped): a plain product O = X Wh (f2, Eq. 14)
  int32_t fold;              // the tile table was built with the folded geometry (w_* functions)
  // product 1 (Y = X X^T) only, single-CTA symmetric tiles (option "umma.sharea"): when the tile's A rows are among the B
  // rows it stages (the tile holds its panel's diagonal square), no A copy is issued and the A descriptor points into
  // the B stage -- at m = 414 a quarter of the product's L2 -> SM bytes
  int32_t share_a;
};

// Row offset of a tile's A rows inside its B stage when product 1 can read A from there (share_a), else -1.
__device__ __forceinline__ int32_t share_a_off(const UArgs &a, const UTile &u, bool p2) {
  if (!a.share_a || p2) return -1;
  const int32_t a_rows = min(UM, u.Pd - u.row0);
  const int32_t n1 = min(u.nt, u.fb - u.n0);          // B rows [n0, n0 + n1) are matrix rows of the same index
  return (u.row0 >= u.n0 && u.row0 + a_rows <= u.n0 + n1) ? u.row0 - u.n0 : -1;
}

// Tile geometry.  Only elements (r, c) with c <= r are computed, so tile row tm (rows tm*R ..
// tm*R + R - 1, R = 128 * NCTA) needs the columns [0, min(n16, tm*R + R)); they are split into the
// fewest tiles of <= 256 columns, of equal width rounded up to 32 (the last one takes the rest).
__host__ __device__ inline int32_t u_n16(int32_t m) { return (m + 15) & ~15; }
__host__ __device__ inline int32_t u_Tm(int32_t m, int32_t R) { return (m + R - 1) / R; }
__host__ __device__ inline int32_t u_ncols(int32_t m, int32_t R, int32_t tm) {
  int32_t n32 = (m + 31) & ~31, e = tm * R + R;     // whole 32-column epilogue blocks (n32 <= Pd: zero padding)
  return e < n32 ? e : n32;
}
__host__ __device__ inline int32_t u_row_tiles(int32_t m, int32_t R, int32_t tm) {
  return (u_ncols(m, R, tm) + UN - 1) / UN;
}
__host__ __device__ inline int32_t u_row_nb(int32_t m, int32_t R, int32_t tm) {
  int32_t nc = u_ncols(m, R, tm), Tn = (nc + UN - 1) / UN;
  return (((nc + 31) / 32 + Tn - 1) / Tn) * 32;     // multiple of 32: epilogue blocks never straddle the diagonal
}
__host__ __device__ inline int32_t u_tiles(int32_t m, int32_t R) {
  int32_t t = 0;
  for (int32_t tm = 0; tm < u_Tm(m, R); ++tm) t += u_row_tiles(m, R, tm);
  return t;
}

// "Folded" geometry of the 128-row symmetric tiles (option "umma.fold", single-CTA tiles only).  When the last 128-row
// panel holds at most 64 rows (m rounded up to 32), running it as a row panel costs an M = 128 MMA over ALL columns
// for <= 64 useful rows -- at m = 414 (configs[2]'s median) 35 % of a product's MMA work and 30 % of its B-operand
// loads for 7 % of its rows.  Instead the other panels take those rows as fn extra COLUMNS behind their own (virtual
// column v of panel tm: v < (tm + 1) 128 is column v, else column F0 + v - (tm + 1) 128, F0 = first row of the last
// panel), their mirrored stores fill the last rows, and the last panel keeps only its fn x fn diagonal square.
// MMA work at m = 414: 1184 -> 896 column panels (-24 %), operand rows loaded 1824 -> 1600 (-12 %).
__host__ __device__ inline int32_t w_fold(int32_t m) {
  const int32_t Tm = u_Tm(m, UM);
  if (Tm < 2) return 0;
  const int32_t fn = ((m + 31) & ~31) - (Tm - 1) * UM;
  return fn <= 64 ? fn : 0;
}
__host__ __device__ inline int32_t w_ncols(int32_t m, int32_t tm, int32_t fn) {
  if (!fn) return u_ncols(m, UM, tm);
  return tm + 1 < u_Tm(m, UM) ? (tm + 1) * UM + fn : fn;
}
__host__ __device__ inline int32_t w_row_tiles(int32_t m, int32_t tm, int32_t fn) { return (w_ncols(m, tm, fn) + UN - 1) / UN; }
__host__ __device__ inline int32_t w_row_nb(int32_t m, int32_t tm, int32_t fn) {
  const int32_t nc = w_ncols(m, tm, fn), Tn = (nc + UN - 1) / UN;
  return (((nc + 31) / 32 + Tn - 1) / Tn) * 32;
}
__host__ __device__ inline int32_t w_tiles(int32_t m, int32_t fn) {
  int32_t t = 0;
  for (int32_t tm = 0; tm < u_Tm(m, UM); ++tm) t += w_row_tiles(m, tm, fn);
  return t;
}

// Geometry of the staged epilogue (EPI = 1, 128-row tiles): tile columns are whole 64-column chunks of the image (a
// chunk of a row range is contiguous in memory: one bulk store); the tiles of a row panel start at multiples of 256
// columns, so that every 128-column block -- in particular the panel's 128 x 128 diagonal square -- lies inside one tile.
__host__ __device__ inline int32_t v_ncols(int32_t m, int32_t tm) {
  int32_t n64 = (m + 63) & ~63, e = tm * UM + UM;
  return e < n64 ? e : n64;
}
__host__ __device__ inline int32_t v_row_tiles(int32_t m, int32_t tm) { return (v_ncols(m, tm) + UN - 1) / UN; }
__host__ __device__ inline int32_t v_tiles(int32_t m) {
  int32_t t = 0;
  for (int32_t tm = 0; tm < u_Tm(m, UM); ++tm) t += v_row_tiles(m, tm);
  return t;
}

// FULL mode (true products, no symmetry): every 128*NCTA-row panel of the Pd x Pd image times all Pd
// columns, in tiles of 256 columns (the last one takes the rest, rounded up to whole 64-column
// swizzle atoms per CTA).
__host__ __device__ inline int32_t f_Tm(int32_t Pd, int32_t R) { return (Pd + R - 1) / R; }
__host__ __device__ inline int32_t f_Tn(int32_t Pd) { return (Pd + UN - 1) / UN; }
__host__ __device__ inline int32_t f_tiles(int32_t Pd, int32_t R) { return f_Tm(Pd, R) * f_Tn(Pd); }

__device__ __forceinline__ TileDesc load_desc(const UArgs &a, int64_t t) {
  // a.rev: this launch walks the tile table backwards, so that it starts on the submatrices whose operands the
  // previous launch touched last (still in L2) instead of on the ones evicted longest ago
  if (a.rev) t = a.tile_ptr[a.n_cols] - 1 - t;
  const uint4 *p = reinterpret_cast<const uint4 *>(a.tiles + t);
  uint4 q0 = __ldg(p), q1 = __ldg(p + 1), q2 = __ldg(p + 2);
  TileDesc d;
  d.base = (int64_t)(((uint64_t)q0.y << 32) | q0.x);
  d.c = (int32_t)q0.z; d.m = (int32_t)q0.w;
  d.Pd = (int32_t)q1.x; d.row0 = (int32_t)q1.y; d.n0 = (int32_t)q1.z; d.nt = (int32_t)q1.w;
  d.lt = (int32_t)q2.x; d.pad0 = d.pad1 = d.pad2 = 0;
  return d;
}

template <int PHASE>
__device__ __forceinline__ UTile make_tile(const UArgs &a, const TileDesc &d) {
  UTile u;
  u.c = d.c; u.m = d.m; u.Pd = d.Pd; u.base = d.base;
  u.row0 = d.row0; u.n0 = d.n0; u.nt = d.nt; u.lt = d.lt;
  u.kmax = u_n16(d.m);
  u.fb = 0x7fffffff; u.fs = 0;
  if (a.fold) {
    const int32_t fn = w_fold(d.m), F0 = (u_Tm(d.m, UM) - 1) * UM;
    if (fn && d.row0 < F0) { u.fb = d.row0 + UM; u.fs = F0 - u.fb; }
  }
  int32_t act = 1;
  if (a.check_flags) {
    act = a.s.active[d.c];
    if (PHASE == 1) act = act && !a.s.last[d.c];
  }
  u.valid = act;
  return u;
}

// Column split of a row panel whose tiles start at multiples of nb: with `dl` the tiles before the last one are narrowed
// (whole 32-column blocks) until the last tile starts at or before the panel's first row, so that it holds the whole
// diagonal square and product 1 can take its A rows from the B stage (share_a_off); the tile count does not change.
__host__ __device__ inline int32_t dl_nb(int32_t nb, int32_t cnt, int32_t row0, int32_t nc, int32_t dl) {
  if (!dl || cnt < 2) return nb;
  const int32_t nb2 = min(nb, (row0 / (cnt - 1)) & ~31);
  return (nb2 >= 32 && nc - (cnt - 1) * nb2 <= UN) ? nb2 : nb;
}

static __global__ void k_umma_build_tiles(int32_t n_cols, int32_t R, int32_t sym, int32_t fold, int32_t dl, int32_t skip_pd, const int32_t *__restrict__ cols,
                                          const int32_t *__restrict__ dim, const int32_t *__restrict__ dim_pad,
                                          const int64_t *__restrict__ col_off,
                                          const int64_t *__restrict__ tile_ptr, TileDesc *__restrict__ tiles) {
  int32_t c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_cols) return;
  int32_t i = cols ? cols[c] : c;
  int32_t m = dim[i], Pd = dim_pad[i];
  if (Pd <= skip_pd) return;                      // taken by the resident kernel: no tiles
  TileDesc d;
  d.base = col_off[c]; d.c = c; d.m = m; d.Pd = Pd; d.pad0 = d.pad1 = d.pad2 = 0;
  int64_t t = tile_ptr[c];
  int32_t lt = 0;
  if (sym == 2) {
    for (int32_t tm = 0; tm < u_Tm(m, UM); ++tm) {
      const int32_t cnt = v_row_tiles(m, tm), nc = v_ncols(m, tm);
      for (int32_t tn = 0; tn < cnt; ++tn, ++lt, ++t) {
        d.row0 = tm * UM; d.n0 = tn * UN; d.nt = min(UN, nc - d.n0); d.lt = lt;
        tiles[t] = d;
      }
    }
  } else if (sym && fold && R == UM) {
    const int32_t fn = w_fold(m), Tm = u_Tm(m, UM);
    for (int32_t tm = 0; tm < Tm; ++tm) {
      const int32_t cnt = w_row_tiles(m, tm, fn), nc = w_ncols(m, tm, fn), nb = dl_nb(w_row_nb(m, tm, fn), cnt, tm * UM, nc, dl);
      const int32_t v0 = (fn && tm + 1 == Tm) ? tm * UM : 0;       // the last panel's square starts at its own first column
      for (int32_t tn = 0; tn < cnt; ++tn, ++lt, ++t) {
        d.row0 = tm * UM; d.n0 = v0 + tn * nb; d.nt = tn + 1 < cnt ? nb : v0 + nc - d.n0; d.lt = lt;      // the last tile takes the rest
        tiles[t] = d;
      }
    }
  } else if (sym) {
    for (int32_t tm = 0; tm < u_Tm(m, R); ++tm) {
      int32_t cnt = u_row_tiles(m, R, tm), nc = u_ncols(m, R, tm), nb = dl_nb(u_row_nb(m, R, tm), cnt, tm * R, nc, R == UM ? dl : 0);
      for (int32_t tn = 0; tn < cnt; ++tn, ++lt, ++t) {
        d.row0 = tm * R; d.n0 = tn * nb; d.nt = tn + 1 < cnt ? nb : nc - d.n0; d.lt = lt;
        tiles[t] = d;
      }
    }
  } else {
    const int32_t q = R / 2;                      // 64 columns per CTA of the tile: whole swizzle atoms
    for (int32_t tm = 0; tm < f_Tm(Pd, R); ++tm) {
      for (int32_t tn = 0; tn < f_Tn(Pd); ++tn, ++lt, ++t) {
        d.row0 = tm * R; d.n0 = tn * UN; d.nt = min(UN, (Pd - d.n0 + q - 1) / q * q); d.lt = lt;
        tiles[t] = d;
      }
    }
  }
}

template <bool BF16> __device__ __forceinline__ uint32_t pack2(float lo, float hi);
template <> __device__ __forceinline__ uint32_t pack2<true>(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t *>(&v);
}
template <> __device__ __forceinline__ uint32_t pack2<false>(float lo, float hi) {
  __half2 v = __floats2half2_rn(lo, hi);
  return *reinterpret_cast<uint32_t *>(&v);
}
template <bool BF16> __device__ __forceinline__ float2 unpack2(uint32_t w);
template <> __device__ __forceinline__ float2 unpack2<true>(uint32_t w) {
  return __bfloat1622float2(*reinterpret_cast<__nv_bfloat162 *>(&w));
}
template <> __device__ __forceinline__ float2 unpack2<false>(uint32_t w) {
  return __half22float2(*reinterpret_cast<__half2 *>(&w));
}

// Row segment of 32 packed outputs (o[4g .. 4g+3] = chunk g) as two full 32-byte sectors.
__device__ __forceinline__ void store_row_segment(uint16_t *Orow, uint32_t sec0, uint32_t sec1, bool swp,
                                                  const uint32_t (&o)[16]) {
  ptx::stg256(Orow + sec0, swp ? o[4] : o[0], swp ? o[5] : o[1], swp ? o[6] : o[2], swp ? o[7] : o[3],
              swp ? o[0] : o[4], swp ? o[1] : o[5], swp ? o[2] : o[6], swp ? o[3] : o[7]);
  ptx::stg256(Orow + sec1, swp ? o[12] : o[8], swp ? o[13] : o[9], swp ? o[14] : o[10], swp ? o[15] : o[11],
              swp ? o[8] : o[12], swp ? o[9] : o[13], swp ? o[10] : o[14], swp ? o[11] : o[15]);
}

// Identity operand of the update product.  PHASE 2 computes X' = X - 1/2 X W as ONE accumulation:
// PHASE 1 stores Wh = -1/2 (X X^T - I) (exact scaling), and while the A chunk X[rows, 64 kc ..] that covers
// output columns of the tile sits in shared memory, one more MMA with B = a slice of the identity adds
// X[rows, cols] * 1 to those accumulator columns.  The epilogue then only converts and stores: no global
// read of the X tile (it cost 64 of the ~160 L1 wavefronts of a 32 x 32 block, and 1.3 GB of L2/HBM
// reads per step at configs[2]).  The image is K-major SW128 like every operand: 64 rows x 128 B.
// One CTA: row n has its 1 at k = n; a piece [lo, hi) of the chunk uses rows lo - 64 kc onwards.
// CTA pair (each CTA supplies half of the N rows from the same offset): rows 0-31 serve N = 64 (1 at
// k = 32 h + n), rows 32-47 N = 32 at k-offset 0 (k = 16 h + n'), rows 48-63 N = 32 at k-offset 32.
template <bool BF16>
__device__ __forceinline__ void ident_fill(uint8_t *img, bool pair, uint32_t h, int tid, int nthreads) {
  for (int i = tid; i < IDENT_BYTES / 16; i += nthreads) reinterpret_cast<uint4 *>(img)[i] = make_uint4(0, 0, 0, 0);
  __syncthreads();
  if (tid < 64) {
    const uint32_t n = (uint32_t)tid;
    const uint32_t k = !pair ? n : (n < 32 ? 32 * h + n : (n < 48 ? 16 * h + (n - 32) : 32 + 16 * h + (n - 48)));
    *reinterpret_cast<uint16_t *>(img + n * 128 + (((k >> 3) ^ (n & 7)) << 4) + (k & 7) * 2) = BF16 ? 0x3F80 : 0x3C00;
  }
}
// Row of the identity image at which the B slice of a piece starts (s = lo - 64 kc in {0, 32}, N in {32, 64}).
__device__ __forceinline__ uint32_t ident_row(bool pair, int32_t s, int32_t N) {
  return !pair ? (uint32_t)s : (N == 64 ? 0u : (s ? 48u : 32u));
}

// Mirrored 32 x 32 block straight from the registers of a warp whose lane holds row R0 + lane, columns
// C0 .. C0 + 31 as 16 packed pairs: element (r, C0 + j) goes to row C0 + j, column r of the swizzled image.
__device__ __forceinline__ void mirror_store(uint16_t *Og, int32_t Pd, int32_t R0, int32_t C0, int lane,
                                             const uint32_t (&o)[16]) {
#ifdef SM_MIRROR_U16
  uint16_t *Mb = Og + (int64_t)(R0 >> 6) * Pd * 64 + (int64_t)C0 * 64 + (lane & 7);
  const uint32_t ch = (((uint32_t)R0 & 63u) >> 3) + ((uint32_t)lane >> 3);   // chunk of column r before the swizzle
#pragma unroll
  for (int j = 0; j < 32; ++j)
    Mb[j * 64 + ((ch ^ (uint32_t)(j & 7)) << 3)] = (uint16_t)(o[j >> 1] >> ((j & 1) * 16));
#else
  // Lane pairs (r, r ^ 1) exchange halves first, so that a lane holds the two ADJACENT columns r & ~1, (r & ~1) + 1 of one
  // mirrored row -- the even lane of row C0 + 2e, the odd lane of row C0 + 2e + 1 -- and stores 4 bytes: 16 store
  // instructions per block instead of 32 (each instruction still fills two whole sectors per row, now of two rows).
  const uint32_t odd = (uint32_t)lane & 1u;
  uint16_t *Mb = Og + (int64_t)(R0 >> 6) * Pd * 64 + (int64_t)(C0 + (int32_t)odd) * 64 + (lane & 6);
  const uint32_t chx = ((((uint32_t)R0 & 63u) >> 3) + ((uint32_t)lane >> 3)) ^ odd;   // chunk of column r, swizzle bit 0 of the row folded in
#pragma unroll
  for (int e = 0; e < 16; ++e) {
    const uint32_t x = __shfl_xor_sync(0xffffffffu, o[e], 1);
    const uint32_t w = odd ? __byte_perm(x, o[e], 0x7632) : __byte_perm(o[e], x, 0x5410);
    *reinterpret_cast<uint32_t *>(Mb + (2 * e) * 64 + ((chx ^ (uint32_t)((2 * e) & 7)) << 3)) = w;
  }
#endif
}

// SYM = true : K-major B (X X^T form), lower-triangle tiles, mirrored stores (exactly symmetric iterates).
// SYM = false: MN-major B (true products X X and X Y), all tiles, plain row stores.  The true-product
//              form damps (++ block) or leaves unchanged (+- block) an antisymmetric rounding residue,
//              so exact symmetry is not needed; it trades 1.3-1.7x more MMA work for an epilogue
//              without transposes, which is what bounds the m < ~1000 regime (ncu, round 1).
// TM (cta_group::2 pairs only): operands come through tensor-map TMA (2-D view of the packed buffer: rows of 64
// elements, no swizzle -- the image is stored pre-swizzled) with `.cta_group::2`, which lets BOTH CTAs of a pair
// credit their bytes to the LEADER's "stage full" barrier; no relay warp, no second barrier wait per stage.
// DYN (one CTA per tile only): tiles are handed out by a global counter instead of round robin.  The producer
// thread pops the next index (the atomic's latency overlaps the current tile's loads), reads its descriptor and
// publishes it through a 4-entry shared-memory queue (mbarrier full / empty pairs) to the MMA issuer and the 16
// epilogue warps.  With a static deal the CTAs drift apart by tens of tiles over a launch (tile costs differ), so
// the tiles of one submatrix -- which share their operand panels -- run further apart in time than a line lives
// in L2 (126 MB at ~5 TB/s: ~25 us) and the panels are fetched from DRAM again; a dynamic deal keeps all CTAs
// inside one window of the size-sorted tile table and also evens out the tail of the launch.
constexpr int TQ = 4;
// PHASE = 0, "stream" (fixed iteration counts): ONE launch runs every product of every step.  The dynamic deal walks
// a virtual tile list: the listed columns are cut into super-groups of STREAM_SG submatrices (~77 MB of X, Wh, X' at
// configs[2]: they stay in L2), and a super-group's tiles are walked once per product, all 2 * steps products before
// the next super-group.  A product of a submatrix needs the previous product of the same submatrix complete: the
// dependency is tracked per group of STREAM_G submatrices by a counter that every epilogue warp bumps (after a
// gpu-scope fence and a generic->async proxy fence) when its part of a tile is stored; the producer thread of a
// tile of (group, product ph) waits until the counter of (group, ph - 1) is complete, then fences and issues its bulk
// copies.  The tiles in between (the other groups of the super-group, ~3/4 of it = ~2 tiles per CTA) are what hides
// that wait.  Because tiles are popped in list order and every CTA is resident, a waiting CTA only ever waits for
// tiles that are already running: no deadlock.
#ifndef SM_STREAM_G
#define SM_STREAM_G 16
#endif
#ifndef SM_STREAM_SG
#define SM_STREAM_SG 96
#endif
constexpr int STREAM_G = SM_STREAM_G;
constexpr int STREAM_SG = SM_STREAM_SG;
template <bool BF16, int PHASE, int NCTA, bool SYM, bool MC = false, int NST = 0, bool TM = false, bool DYN = false, int EPI = 0>
__global__ void __launch_bounds__(UMMA_THREADS, 1)
k_umma_gemm(UArgs a, const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB) {
  static_assert(!DYN || NCTA == 1, "dynamic tile scheduling: one CTA per tile");
  static_assert(EPI == 0 || (SYM && NCTA == 1), "staged epilogue: single CTAs, SYM tiles");
  constexpr bool STG = EPI == 1;
  static_assert(PHASE != 0 || (DYN && SYM), "stream mode needs the dynamic deal and symmetric tiles");
  constexpr bool STREAM = PHASE == 0;
  static_assert(!MC || (NCTA == 2 && SYM), "multicast variant: two CTAs, SYM tiles");
  static_assert(!TM || (NCTA == 2 && SYM && !MC), "tensor-map variant: cta_group::2 pairs, SYM tiles");
  using Cfg = UCfg<NCTA, MC, NST, EPI>;
  constexpr int USTAGES = Cfg::STAGES;
  constexpr int STAGE_BYTES = Cfg::STAGE_BYTES;
  constexpr bool PAIR = NCTA == 2 && !MC;                  // cta_group::2 MMAs issued by the leader
  constexpr bool CL2 = NCTA == 2;                          // cluster of two CTAs on one 256-row tile
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = ptx::smem_u32(smem_raw);
  const uint32_t tiles = (raw + 1023u) & ~1023u;           // 1024-byte aligned operand ring
  const uint32_t stage_base = tiles + USTAGES * STAGE_BYTES;   // epilogue transpose / staging buffers (1024-byte aligned)
  const uint32_t ident = stage_base + Cfg::EPI_BYTES;      // identity image (1024-byte aligned)
  const uint32_t bars = ident + IDENT_BYTES;               // barriers behind it
  // barrier slots (8 bytes each): full[S], empty[S], pfull[S] (pair: peer's stage landed, leader only),
  // tmem_full[2], tmem_empty[2]; then the TMEM base address
  auto full_bar = [&](int s) { return bars + 8u * s; };
  auto empty_bar = [&](int s) { return bars + 8u * (USTAGES + s); };
  auto pfull_bar = [&](int s) { return bars + 8u * (2 * USTAGES + s); };
  auto tfull_bar = [&](int s) { return bars + 8u * (3 * USTAGES + s); };
  auto tempty_bar = [&](int s) { return bars + 8u * (3 * USTAGES + NACC + s); };
  const uint32_t tmem_slot = bars + 8u * (3 * USTAGES + 2 * NACC);
  volatile uint32_t *tmem_slot_ptr =
      reinterpret_cast<volatile uint32_t *>(smem_raw + (tmem_slot - raw));
  // DYN: tile queue behind the barriers: full[TQ], empty[TQ], then TQ descriptors (16-byte aligned)
  auto tqf_bar = [&](int s) { return bars + 256u + 8u * s; };
  auto tqe_bar = [&](int s) { return bars + 256u + 8u * (TQ + s); };
  TileDesc *const tq = reinterpret_cast<TileDesc *>(smem_raw + (bars + 256u + 16u * TQ - raw));

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t h = CL2 ? ptx::cluster_ctarank() : 0u;    // rank inside the CTA pair; 0 = leader
  const int64_t unit = blockIdx.x / NCTA, n_units = gridDim.x / NCTA;

  if (PHASE != 1) {
    ident_fill<BF16>(smem_raw + (ident - raw), PAIR, h, (int)threadIdx.x, UMMA_THREADS);
    ptx::fence_proxy_async();       // generic-proxy writes -> the MMA's async-proxy reads
  }
  if (threadIdx.x == 0) {
    for (int s = 0; s < USTAGES; ++s) {
      // MC: a stage is free once the MMAs of BOTH CTAs have read it (each producer writes into both)
      ptx::mbar_init(full_bar(s), 1); ptx::mbar_init(empty_bar(s), MC ? 2 : 1); ptx::mbar_init(pfull_bar(s), 1);
    }
    for (int s = 0; s < NACC; ++s) { ptx::mbar_init(tfull_bar(s), 1); ptx::mbar_init(tempty_bar(s), EPI_WARPS * (PAIR ? 2 : 1)); }
    if (DYN) for (int s = 0; s < TQ; ++s) { ptx::mbar_init(tqf_bar(s), 1); ptx::mbar_init(tqe_bar(s), 1 + EPI_WARPS); }
    ptx::fence_barrier_init();
    ptx::fence_proxy_async();
  }
  if (warp == 1) {
    if (PAIR) { ptx::tmem_alloc2(tmem_slot, TMEM_COLS); ptx::tmem_relinquish2(); }
    else { ptx::tmem_alloc(tmem_slot, TMEM_COLS); ptx::tmem_relinquish(); }
  }
  ptx::tc_fence_before();
  if (CL2) ptx::cluster_sync_all(); else __syncthreads();
  ptx::tc_fence_after();
  const uint32_t tmem_base = *tmem_slot_ptr;

  const int64_t total = a.tile_ptr[a.n_cols];
  constexpr int ESZ = 2;

  if (warp == 0) {
    // ===================== TMA producer (every CTA: its A rows and its share of the B rows) ==========
    // CONV: the whole warp walks the tiles converged and one elected lane issues each copy (tma_bulk_g2s_elect); lane 0
    // alone pops / publishes the tile (fetch) and broadcasts it.  The other variants keep the single producer thread.
    constexpr bool CONV = NCTA == 1 && SYM && !MC && !TM && EPI == 0;
    if (CONV || lane == 0) {
      int stage = 0; uint32_t phase = 0;
      TileDesc nxt = load_desc(a, max((int64_t)0, min(unit, total - 1)));
      int64_t t = DYN ? (lane == 0 ? (int64_t)atomicAdd(a.counter, 1ULL) : 0) : unit;
      uint32_t qs = 0, qp = 0;
      int32_t sg_c0 = 0;                                                     // STREAM: current super-group
      int64_t sg_lo = 0, sg_hi = STREAM ? a.tile_ptr[min(STREAM_SG, a.n_cols)] : 0;
      // next tile of this CTA: static deal (descriptor prefetched one tile ahead) or DYN (pop, publish)
      auto fetch = [&](TileDesc &cur) -> bool {
        if (DYN) {
          const int64_t mine = t;
          ptx::mbar_wait(tqe_bar(qs), qp ^ 1u, a.err_flag, 8);
          if (STREAM) {
            // virtual index -> (super-group S, product ph, tile): super-group S = STREAM_SG consecutive listed
            // columns; its tiles are walked once per product, all products of S before S + 1
            if (mine < total * a.n_ph) {
              while (mine >= (int64_t)a.n_ph * sg_hi) {
                sg_c0 = min(sg_c0 + STREAM_SG, a.n_cols);
                sg_lo = sg_hi; sg_hi = a.tile_ptr[min(sg_c0 + STREAM_SG, a.n_cols)];
              }
              const int64_t off = mine - (int64_t)a.n_ph * sg_lo, ts = sg_hi - sg_lo;
              const int32_t ph = (int32_t)(off / ts);
              cur = load_desc(a, sg_lo + (off - (int64_t)ph * ts));
              const int32_t grp = cur.c / STREAM_G;
              const int32_t g0 = grp * STREAM_G, g1 = min(g0 + STREAM_G, a.n_cols);
              cur.pad0 = ph; cur.pad1 = grp;
              cur.pad2 = (int32_t)(a.tile_ptr[g1] - a.tile_ptr[g0]) * EPI_WARPS;     // completions of one product of the group
            } else cur.c = -1;
          } else if (mine < total) cur = load_desc(a, mine); else cur.c = -1;
          tq[qs] = cur;
          ptx::mbar_arrive(tqf_bar(qs));            // release: the descriptor is visible to the consumers
          if (++qs == TQ) { qs = 0; qp ^= 1u; }
          if (cur.c < 0) return false;
          t = (int64_t)atomicAdd(a.counter, 1ULL);  // its latency overlaps this tile's loads
          if (STREAM && cur.pad0 > 0 && !SM_DBG(a, 64)) {
            // the previous product of this group (written by other CTAs) must be complete and visible to the bulk copies
            const volatile int32_t *flag = a.done + (int64_t)cur.pad1 * a.n_ph + (cur.pad0 - 1);
            for (uint32_t spin = 0; *flag < cur.pad2; ++spin) {
              __nanosleep(64);
              if (spin > 40000000u) { atomicExch(a.err_flag, 11); __threadfence_system(); __trap(); }
            }
            __threadfence();
            ptx::fence_proxy_async();
          }
          return true;
        }
        if (t >= total) return false;
        cur = nxt;
        nxt = load_desc(a, min(t + n_units, total - 1));    // prefetch the next descriptor
        t += n_units;
        return true;
      };
      TileDesc cur;
      if (CONV) {
        constexpr uint32_t FULL = 0xffffffffu;
        for (;;) {
          int32_t ok = 0;
          if (lane == 0) ok = fetch(cur) ? 1 : 0;
          __syncwarp();
          if (!__shfl_sync(FULL, ok, 0)) break;
          {
            uint32_t blo = (uint32_t)(uint64_t)cur.base, bhi = (uint32_t)((uint64_t)cur.base >> 32);
            blo = __shfl_sync(FULL, blo, 0); bhi = __shfl_sync(FULL, bhi, 0);
            cur.base = (int64_t)(((uint64_t)bhi << 32) | blo);
            cur.c = __shfl_sync(FULL, cur.c, 0); cur.m = __shfl_sync(FULL, cur.m, 0);
            cur.Pd = __shfl_sync(FULL, cur.Pd, 0); cur.row0 = __shfl_sync(FULL, cur.row0, 0);
            cur.n0 = __shfl_sync(FULL, cur.n0, 0); cur.nt = __shfl_sync(FULL, cur.nt, 0);
            cur.lt = __shfl_sync(FULL, cur.lt, 0); cur.pad0 = __shfl_sync(FULL, cur.pad0, 0);
          }
          UTile u = make_tile<PHASE>(a, cur);
          u.valid = __shfl_sync(FULL, u.valid, 0);
          if (!u.valid) continue;
          const bool p2 = STREAM ? (cur.pad0 & 1) != 0 : PHASE == 2;
          const void *Xcur = (STREAM && ((cur.pad0 >> 1) & 1)) ? a.Out : a.Xsrc;     // stream: X ping-pongs per step
          const uint32_t a_rows = (uint32_t)max(0, min(UM, u.Pd - u.row0));
          // product 1: the A rows are among the B rows of the stage (share_a_off): no copy of their own
          const uint32_t a_tx = share_a_off(a, u, p2) >= 0 ? 0u : a_rows * 128u;
          // B rows [n0, n0 + nt) of the tile's (virtual) columns: those from u.fb on are the folded rows
          const int32_t n1 = max(0, min(u.nt, u.fb - u.n0));
          const uint32_t b1_tx = (uint32_t)n1 * 128u, b2_tx = (uint32_t)(u.nt - n1) * 128u;
          const char *pA = (const char *)Xcur + u.base * ESZ + (int64_t)u.row0 * 128;
          const char *Bg = (const char *)(p2 ? a.Ybuf : Xcur) + u.base * ESZ;
          const char *pB1 = Bg + (int64_t)u.n0 * 128, *pB2 = Bg + (int64_t)(max(u.n0, u.fb) + u.fs) * 128;
          const int64_t cs = (int64_t)u.Pd * 128;                                  // bytes between k chunks
          const int nkc = (u.kmax + UK - 1) / UK;
          for (int kc = 0; kc < nkc; ++kc) {
            ptx::mbar_wait(empty_bar(stage), phase ^ 1u, a.err_flag, 1);
            const uint32_t sa = tiles + stage * STAGE_BYTES, sb = sa + A_BYTES, fb_ = full_bar(stage);
            if (SM_DBG(a, 4)) {
              if (lane == 0) ptx::mbar_arrive(fb_);
              __syncwarp();
            } else {
              ptx::mbar_expect_tx_elect(fb_, a_tx + b1_tx + b2_tx);
              if (a_tx) ptx::tma_bulk_g2s_elect(sa, pA, a_tx, fb_);
              if (b1_tx) ptx::tma_bulk_g2s_elect(sb, pB1, b1_tx, fb_);
              if (b2_tx) ptx::tma_bulk_g2s_elect(sb + b1_tx, pB2, b2_tx, fb_);
              pA += cs; pB1 += cs; pB2 += cs;
            }
            if (++stage == USTAGES) { stage = 0; phase ^= 1u; }
          }
        }
      } else
      while (fetch(cur)) {
        UTile u = make_tile<PHASE>(a, cur);
        if (!u.valid) continue;
        const bool p2 = STREAM ? (cur.pad0 & 1) != 0 : PHASE == 2;
        const void *Xcur = (STREAM && ((cur.pad0 >> 1) & 1)) ? a.Out : a.Xsrc;     // stream: X ping-pongs per step
        const char *Ag = (const char *)Xcur + u.base * ESZ;
        const char *Bg = (const char *)(p2 ? a.Ybuf : Xcur) + u.base * ESZ;
        const int32_t arow0 = u.row0 + (int32_t)h * UM;
        const uint32_t a_rows = (uint32_t)max(0, min(UM, u.Pd - arow0));
        const int32_t b_cnt = u.nt / NCTA, brow0 = u.n0 + (int32_t)h * b_cnt;   // this CTA's share of B
        // FULL mode: whole 64-column atoms of the image; atoms past the padded dimension are not loaded
        // (their accumulator columns are garbage and never stored).
        const int32_t atom0 = brow0 >> 6, n_atoms = max(0, min(b_cnt >> 6, (u.Pd >> 6) - atom0));
        const uint32_t a_bytes = a_rows * 128u;
        const uint32_t b_bytes = SYM ? (uint32_t)b_cnt * 128u : (uint32_t)n_atoms * 8192u;
        const int nkc = (u.kmax + UK - 1) / UK;
        const bool a_shared = SYM && NCTA == 1 && share_a_off(a, u, p2) >= 0;
        if (TM) {
          // boxes: 128 rows (A: one copy; rows past the padded dimension are harmless) and 64 rows (B: b_cnt rounded
          // up to whole boxes -- few, large copies: ten 2 KB boxes per stage kept the producer thread busy longer
          // than the stage's MMAs take)
          const uint32_t other_rows = (uint32_t)max(0, min(UM, u.Pd - (u.row0 + (int32_t)(1u - h) * UM)));
          const int32_t nb64 = (b_cnt + 63) >> 6;
          const uint32_t tx_all = ((a_rows ? 128u : 0u) + (other_rows ? 128u : 0u)) * 128u + 2u * (uint32_t)nb64 * 8192u;
          const int32_t row_base = (int32_t)(u.base >> 6);            // first image row of the submatrix
          for (int kc = 0; kc < nkc; ++kc) {
            ptx::mbar_wait(empty_bar(stage), phase ^ 1u, a.err_flag, 1);
            const uint32_t sa = tiles + stage * STAGE_BYTES, sb = sa + A_BYTES;
            const uint32_t lead_full = ptx::mapa_u32(full_bar(stage), 0);
            if (h == 0) ptx::mbar_expect_tx(full_bar(stage), tx_all);
            const int32_t y0 = row_base + kc * u.Pd;
            if (a_rows) ptx::tma_tensor2d_g2s_2cta(sa, &mapA, 0, y0 + arow0, lead_full);
            for (int32_t j = 0; j < nb64; ++j)
              ptx::tma_tensor2d_g2s_2cta(sb + (uint32_t)j * 8192u, &mapB, 0, y0 + brow0 + j * 64, lead_full);
            if (++stage == USTAGES) { stage = 0; phase ^= 1u; }
          }
          continue;
        }
        if (STG && a.lt_in) {
          // "128-lower" operands: a 128-row block of a chunk that lies above the diagonal squares is fetched as the
          // transposed pieces (64 k rows x 128 B each, contiguous) of the chunk(s) holding its rows as columns
          const int32_t rb128 = u.row0 >> 7, jb0 = u.n0 >> 7;
          const int32_t np = (u.nt + 127) >> 7;                      // 128-column sub-panels of the B rows
          for (int kc = 0; kc < nkc; ++kc) {
            ptx::mbar_wait(empty_bar(stage), phase ^ 1u, a.err_flag, 1);
            const uint32_t sa = tiles + stage * STAGE_BYTES, sb = sa + A_BYTES;
            const int32_t kb = kc >> 1;
            const int64_t chunk = (int64_t)kc * u.Pd * 128;          // byte offset of k chunk kc
            // bytes first (one expect_tx), then the copies
            uint32_t tx = 0;
            const bool a_dir = rb128 >= kb;
            const int32_t a_pieces = min(2, (u.Pd - u.row0 + 63) >> 6);
            tx += a_dir ? a_bytes : (uint32_t)a_pieces * 8192u;
            for (int pz = 0; pz < np; ++pz) {
              const int32_t rows = min(128, u.nt - 128 * pz);
              tx += (jb0 + pz >= kb) ? (uint32_t)rows * 128u : (uint32_t)((rows + 63) >> 6) * 8192u;
            }
            ptx::mbar_expect_tx(full_bar(stage), tx);
            if (a_dir) ptx::tma_bulk_g2s(sa, Ag + chunk + (int64_t)u.row0 * 128, a_bytes, full_bar(stage));
            else
              for (int32_t j = 0; j < a_pieces; ++j)      // rows 64 kc .. of chunk-column (row0 / 64 + j)
                ptx::tma_bulk_g2s(sa + (uint32_t)j * 8192u, Ag + ((int64_t)((u.row0 >> 6) + j) * u.Pd + (int64_t)kc * UK) * 128, 8192u, full_bar(stage));
            for (int pz = 0; pz < np; ++pz) {
              const int32_t rows = min(128, u.nt - 128 * pz), j0 = u.n0 + 128 * pz;
              if (jb0 + pz >= kb) ptx::tma_bulk_g2s(sb + (uint32_t)pz * 16384u, Bg + chunk + (int64_t)j0 * 128, (uint32_t)rows * 128u, full_bar(stage));
              else
                for (int32_t j = 0; j < ((rows + 63) >> 6); ++j)
                  ptx::tma_bulk_g2s(sb + (uint32_t)pz * 16384u + (uint32_t)j * 8192u, Bg + ((int64_t)((j0 >> 6) + j) * u.Pd + (int64_t)kc * UK) * 128, 8192u, full_bar(stage));
            }
            if (++stage == USTAGES) { stage = 0; phase ^= 1u; }
          }
          continue;
        }
        for (int kc = 0; kc < nkc; ++kc) {
          ptx::mbar_wait(empty_bar(stage), phase ^ 1u, a.err_flag, 1);
          const uint32_t sa = tiles + stage * STAGE_BYTES, sb = sa + A_BYTES;
          if (SM_DBG(a, 4)) {
            ptx::mbar_arrive(full_bar(stage));
            if (++stage == USTAGES) { stage = 0; phase ^= 1u; }
            continue;
          }
          const uint32_t a_tx = a_shared ? 0u : a_bytes;     // product 1: the A rows are among the B rows of this stage
          ptx::mbar_expect_tx(full_bar(stage), a_tx + (MC ? 2u * b_bytes : b_bytes));
          const int64_t chunk = (int64_t)kc * u.Pd * 128;     // byte offset of k chunk kc
          if (a_tx) ptx::tma_bulk_g2s(sa, Ag + chunk + (int64_t)arow0 * 128, a_tx, full_bar(stage));
          if (MC) {
            // this CTA's half of the B rows, delivered into both CTAs at its place in the whole tile
            ptx::tma_bulk_g2s_mc(sb + h * b_bytes, Bg + chunk + (int64_t)brow0 * 128, b_bytes, full_bar(stage), (uint16_t)3);
          } else if (SYM) {
            // rows [brow0, brow0 + b_cnt) of the tile's (virtual) columns: those from u.fb on are the folded rows
            const int32_t n1 = max(0, min(b_cnt, u.fb - brow0));
            if (n1) ptx::tma_bulk_g2s(sb, Bg + chunk + (int64_t)brow0 * 128, (uint32_t)n1 * 128u, full_bar(stage));
            if (n1 < b_cnt)
              ptx::tma_bulk_g2s(sb + (uint32_t)n1 * 128u, Bg + chunk + (int64_t)(max(brow0, u.fb) + u.fs) * 128,
                                (uint32_t)(b_cnt - n1) * 128u, full_bar(stage));
          } else {
            for (int32_t j = 0; j < n_atoms; ++j)    // rows k of chunk-column (atom0 + j): 64 x 128 B
              ptx::tma_bulk_g2s(sb + (uint32_t)j * 8192u,
                                Bg + ((int64_t)(atom0 + j) * u.Pd + (int64_t)kc * UK) * 128, 8192u, full_bar(stage));
          }
          if (++stage == USTAGES) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (PAIR && !TM && warp == 1 && h != 0) {
    // ===================== relay (peer CTA of a pair): tell the leader that this CTA's stage landed ======
    if (lane == 0) {
      int stage = 0; uint32_t phase = 0;
      TileDesc nxt = load_desc(a, max((int64_t)0, min(unit, total - 1)));
      for (int64_t t = unit; t < total; t += n_units) {
        const TileDesc cur = nxt;
        nxt = load_desc(a, min(t + n_units, total - 1));
        UTile u = make_tile<PHASE>(a, cur);
        if (!u.valid) continue;
        const int nkc = (u.kmax + UK - 1) / UK;
        for (int kc = 0; kc < nkc; ++kc) {
          ptx::mbar_wait(full_bar(stage), phase, a.err_flag, 5);
          ptx::mbar_arrive_remote(pfull_bar(stage), 0);
          if (++stage == USTAGES) { stage = 0; phase ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (leader CTA; every CTA when each issues its own MMAs) =====================
    // The whole warp walks the tiles converged, on warp-uniform values (the tile descriptor is broadcast by shuffles,
    // which tells ptxas so), and one elected lane issues each MMA / commit (umma_f16_elect).  Under `if (lane == 0)`
    // every tcgen05.mma was wrapped in an ELECT / R2UR.BROADCAST / BRA.U.ANY loop of ~150 cycles (clock64, round 2),
    // more than the 128 cycles a 128 x 256 x 16 MMA occupies the tensor pipe.
    if (!(PAIR && h != 0)) {
      int stage = 0; uint32_t phase = 0;
      uint32_t it = 0;
      TileDesc nxt = load_desc(a, max((int64_t)0, min(unit, total - 1)));
      int64_t t = unit;
      uint32_t qs = 0, qp = 0;
      auto fetch = [&](TileDesc &cur) -> bool {
        if (DYN) {
          ptx::mbar_wait(tqf_bar(qs), qp, a.err_flag, 9);
          cur = tq[qs];
          __syncwarp();
          if (lane == 0) ptx::mbar_arrive(tqe_bar(qs));
          if (++qs == TQ) { qs = 0; qp ^= 1u; }
          return cur.c >= 0;
        }
        if (t >= total) return false;
        cur = nxt;
        nxt = load_desc(a, min(t + n_units, total - 1));
        t += n_units;
        return true;
      };
      auto mma = [&](uint32_t d, uint64_t ad, uint64_t bd, uint32_t id, uint32_t acc) {
        if (PAIR) ptx::umma_f16_2cta_elect(d, ad, bd, id, acc);
        else ptx::umma_f16_elect(d, ad, bd, id, acc);
      };
      auto commit = [&](uint32_t bar) {
        if (PAIR) ptx::umma_commit_2cta_elect(bar);
        else if (MC) ptx::umma_commit_mc_elect(bar, (uint16_t)3);
        else ptx::umma_commit_elect(bar);
      };
      TileDesc cur;
      while (fetch(cur)) {
        cur.c = __shfl_sync(0xffffffffu, cur.c, 0); cur.m = __shfl_sync(0xffffffffu, cur.m, 0);
        cur.n0 = __shfl_sync(0xffffffffu, cur.n0, 0); cur.nt = __shfl_sync(0xffffffffu, cur.nt, 0);
        cur.pad0 = __shfl_sync(0xffffffffu, cur.pad0, 0);
        const int32_t cur_row0 = __shfl_sync(0xffffffffu, cur.row0, 0);
        UTile u = make_tile<PHASE>(a, cur);
        u.valid = __shfl_sync(0xffffffffu, u.valid, 0);
        if (!u.valid) continue;
        const uint32_t as = it % NACC, aphase = (it / NACC) & 1u;
        ptx::mbar_wait(tempty_bar(as), aphase ^ 1u, a.err_flag, 2);
        ptx::tc_fence_after();
        const uint32_t d_tmem = tmem_base + as * UN;
        const uint32_t idesc = ptx::make_idesc_f16(BF16, PAIR ? 2 * UM : UM, (uint32_t)u.nt, !SYM);
        const int nkc = (u.kmax + UK - 1) / UK;
        const bool p2 = STREAM ? (cur.pad0 & 1) != 0 : PHASE == 2;
        const int32_t a_off = (SYM && NCTA == 1 && !(STG && a.lt_in)) ? __shfl_sync(0xffffffffu, share_a_off(a, u, p2), 0) : -1;
        for (int kc = 0; kc < nkc; ++kc) {
          ptx::mbar_wait(full_bar(stage), phase, a.err_flag, 3);
          if (PAIR && !TM) ptx::mbar_wait(pfull_bar(stage), phase, a.err_flag, 6);
          ptx::tc_fence_after();
          const uint32_t sa = tiles + stage * STAGE_BYTES, sb = sa + A_BYTES;
          const uint64_t adesc = ptx::make_sw128_kmajor_desc(a_off >= 0 ? sb + (uint32_t)a_off * 128u : sa);
          const uint64_t bdesc = SYM ? ptx::make_sw128_kmajor_desc(sb) : ptx::make_sw128_mnmajor_desc(sb, 8192u, 1024u);
          const uint64_t bstep = SYM ? 2u : 128u;   // 16 k: 32 B inside a K-major atom / 16 rows of 128 B
          const int ksteps = SM_DBG(a, 2) ? 0 : min(UK / 16, (u.kmax - kc * UK) / 16);
          if (STG && a.lt_in) {
            // "128-lower" operands (see the producer): per 128-row block of A and of the B rows, K-major as stored or
            // MN-major through the transposed pieces; the two 128-column halves of the tile may differ
            const int32_t kb = kc >> 1, rb128 = cur_row0 >> 7, jb0 = u.n0 >> 7;
            const bool a_t = rb128 < kb;
            const uint64_t ad = a_t ? ptx::make_sw128_mnmajor_desc(sa, 8192u, 1024u) : adesc;
            const uint64_t astep = a_t ? 128u : 2u;
            const bool b0_t = jb0 < kb, b1_t = jb0 + 1 < kb;
            const int32_t n1 = u.nt - 128;                           // columns of the second half (<= 0: none)
            const bool one = n1 <= 0 || b0_t == b1_t;
            const uint32_t id0 = one ? ptx::make_idesc_f16(BF16, UM, (uint32_t)u.nt, b0_t, a_t) : ptx::make_idesc_f16(BF16, UM, 128u, true, a_t);
            const uint32_t id1 = ptx::make_idesc_f16(BF16, UM, (uint32_t)max(n1, 16), false, a_t);
            const uint64_t bd0 = b0_t ? ptx::make_sw128_mnmajor_desc(sb, 8192u, 1024u) : ptx::make_sw128_kmajor_desc(sb);
            const uint64_t bd1 = ptx::make_sw128_kmajor_desc(sb + 16384u);
            const uint64_t b0step = b0_t ? 128u : 2u;
            auto issue = [&](int ks) {
              const uint32_t acc = (uint32_t)((kc | ks) != 0);
              mma(d_tmem, ad + astep * (uint64_t)ks, bd0 + b0step * (uint64_t)ks, id0, acc);
              if (!one) mma(d_tmem + 128u, ad + astep * (uint64_t)ks, bd1 + 2u * (uint64_t)ks, id1, acc);
            };
            if (ksteps == UK / 16) {
#pragma unroll
              for (int ks = 0; ks < UK / 16; ++ks) issue(ks);
            } else {
              for (int ks = 0; ks < ksteps; ++ks) issue(ks);
            }
          } else if (SYM && !PAIR && ksteps == UK / 16) {
            ptx::umma_f16_elect_k4(d_tmem, ptx::sw128_kmajor_lo(a_off >= 0 ? sb + (uint32_t)a_off * 128u : sa), ptx::sw128_kmajor_lo(sb),
                                   idesc, (uint32_t)(kc != 0));
          } else if (ksteps == UK / 16) {
#pragma unroll
            for (int ks = 0; ks < UK / 16; ++ks)
              mma(d_tmem, adesc + (uint64_t)(2 * ks), bdesc + bstep * (uint64_t)ks, idesc, (uint32_t)((kc | ks) != 0));
          } else {
            for (int ks = 0; ks < ksteps; ++ks)
              mma(d_tmem, adesc + (uint64_t)(2 * ks), bdesc + bstep * (uint64_t)ks, idesc, (uint32_t)((kc | ks) != 0));
          }
          if (p2 && !a.no_ident && !SM_DBG(a, 2)) {
            // "+ X": the A chunk in this stage holds X[rows, 64 kc .. 64 kc + 63]; add it to the accumulator
            // columns [lo, hi) of the tile that it covers (B = identity slice, K-major)
            // (tile columns are virtual: [u.n0, min(u.n0 + u.nt, u.fb)) are columns of the same index, the rest -- the
            // folded rows of the last panel -- are columns v + u.fs)
            const int32_t vend = u.n0 + u.nt;
#pragma unroll
            for (int part = 0; part < 2; ++part) {
              const int32_t g0 = part ? max(u.n0, u.fb) + u.fs : u.n0, g1 = part ? vend + u.fs : min(vend, u.fb);
              if (part && vend <= u.fb) break;
              const int32_t lo = max(kc * UK, g0), hi = min(kc * UK + UK, g1);
              if (lo < hi) {
                const uint32_t idesc2 = ptx::make_idesc_f16(BF16, PAIR ? 2 * UM : UM, (uint32_t)(hi - lo), false);
                const uint64_t idd = ptx::make_sw128_kmajor_desc(ident + ident_row(PAIR, lo - kc * UK, hi - lo) * 128u);
                const uint32_t acol = (uint32_t)(lo - (part ? u.fs : 0) - u.n0);
                if (!PAIR) {
                  ptx::umma_f16_elect_k4(d_tmem + acol, ptx::sw128_kmajor_lo(sa),
                                         ptx::sw128_kmajor_lo(ident + ident_row(PAIR, lo - kc * UK, hi - lo) * 128u), idesc2, 1u);
                } else {
#pragma unroll
                  for (int ks = 0; ks < UK / 16; ++ks)
                    mma(d_tmem + acol, adesc + (uint64_t)(2 * ks), idd + (uint64_t)(2 * ks), idesc2, 1u);
                }
              }
            }
          }
          // frees the smem slot (in both CTAs of a pair) when these MMAs finish
          commit(empty_bar(stage));
          if (++stage == USTAGES) { stage = 0; phase ^= 1u; }
        }
        // accumulator ready for the epilogue warps (of both CTAs)
        if (PAIR) ptx::umma_commit_2cta_elect(tfull_bar(as)); else ptx::umma_commit_elect(tfull_bar(as));
        ++it;
      }
    }
  } else if (STG) {
    // ===================== staged epilogue (warps 2..17; EPI = 1) =====================
    // The output of a tile leaves the SM as bulk stores of whole image pieces instead of per-lane global stores
    // (round 1: the epilogue's 2 x 256-bit + 32 x 2-byte global stores per 32 x 32 block and lane made it the
    // bound of configs[2]: 9000 cycles per tile against 3600 of MMA time).  A tile is cut into UNITS that each fill
    // one 32 KB staging buffer: a 64-column chunk left of the panel's diagonal square (direct piece 128 rows x 128 B
    // = rows of the tile in that chunk, plus the mirrored pieces 2 x (64 rows x 128 B) = rows of that chunk in the
    // two chunks of the square's columns), or the diagonal square itself (2 chunks x 128 rows x 128 B, the upper
    // blocks filled by mirroring the lower ones).  Blocks are read from TMEM in the mma fragment layout
    // (tcgen05.ld 16x256b), packed, and written with stmatrix (direct) / stmatrix.trans (mirror) into the staging
    // buffer, which has the swizzled layout of the image; one thread then issues the unit's 1-3 bulk stores.
    // Two teams of 8 warps (2 per TMEM lane quadrant) alternate over the units, each with its own buffer.
    const int q = warp & 3;                        // TMEM lane quadrant this warp may access
    const int sub = (warp - 2) >> 2, team = sub >> 1, tsub = sub & 1;
    const uint32_t stg = stage_base + (uint32_t)team * EPI_STG_UNIT;
    const bool leader = warp == 2 + 8 * team && lane == 0;
    auto team_bar = [&]() { asm volatile("bar.sync %0, %1;" ::"r"(1 + team), "r"(256) : "memory"); };
    const int g = lane >> 2, q2 = lane & 3, rl = lane & 7, ml = lane >> 3;
    int32_t *pend = nullptr;                       // stream: completion counter of the tile whose stores are in flight
    uint32_t it = 0;
    TileDesc nxt = load_desc(a, max((int64_t)0, min(unit, total - 1)));
    int64_t t = unit;
    uint32_t qs = 0, qp = 0;
    auto fetch = [&](TileDesc &cur) -> bool {
      if (DYN) {
        ptx::mbar_wait(tqf_bar(qs), qp, a.err_flag, 10);
        cur = tq[qs];
        __syncwarp();                                   // every lane has its copy before the slot is handed back
        if (lane == 0) ptx::mbar_arrive(tqe_bar(qs));
        if (++qs == TQ) { qs = 0; qp ^= 1u; }
        return cur.c >= 0;
      }
      if (t >= total) return false;
      cur = nxt;
      nxt = load_desc(a, min(t + n_units, total - 1));
      t += n_units;
      return true;
    };
    TileDesc cur;
    while (fetch(cur)) {
      UTile u = make_tile<PHASE>(a, cur);
      if (!u.valid) continue;
      const uint32_t as = it % NACC, aphase = (it / NACC) & 1u;
      const bool p1 = STREAM ? (cur.pad0 & 1) == 0 : PHASE == 1;
      // stream: product ph of step ph / 2 writes Wh (even ph) or the X buffer that step does not read (odd ph)
      uint16_t *Og = (uint16_t *)(!STREAM ? a.Out : p1 ? a.Ybuf : (((cur.pad0 >> 1) & 1) ? (void *)a.Xsrc : a.Out)) + u.base;
      if (SM_DBG(a, 1)) Og = nullptr;
      if (STREAM && leader) {
        // completion of the PREVIOUS tile's bulk stores is signalled one tile late, so that the wait for the stores to
        // land overlaps this tile's MMAs instead of stalling the team (the dependants are whole products away)
        if (pend) { ptx::bulk_wait0(); __threadfence(); atomicAdd(pend, EPI_WARPS / 2); pend = nullptr; }
        if (cur.pad0 + 1 < a.n_ph) pend = a.done + (int64_t)cur.pad1 * a.n_ph + cur.pad0;
      }
      const int32_t R0 = u.row0 + q * 32;                     // this warp's 32 rows of the tile
      const int32_t a_rows = min(UM, u.Pd - u.row0);
      const int32_t n_below = max(0, min(u.nt, u.row0 - u.n0)) >> 6;   // whole chunks left of the diagonal square
      const int32_t n_un = n_below + (u.n0 + u.nt > u.row0 ? 1 : 0);
      const uint32_t rb = ((uint32_t)R0 & 63u) >> 3;
      // mirrored pieces of the units below the diagonal square: always, unless the output is stored "128-lower"
      const bool mirror_out = !a.lt_out || (a.check_flags && a.s.last[u.c]);
      ptx::mbar_wait(tfull_bar(as), aphase, a.err_flag, 4);
      ptx::tc_fence_after();
      const uint32_t taddr = tmem_base + as * UN + ((uint32_t)(q * 32) << 16);
      float res = 0.f, res2 = 0.f;                             // diagonal-block / off-diagonal (counted twice) sums
      for (int ui = team; ui < n_un; ui += 2) {
        if (leader) ptx::bulk_wait_read0();                    // the buffer's previous bulk stores have read it
        team_bar();
        const bool sq = ui == n_below;
        const int32_t cu0 = sq ? u.row0 : u.n0 + 64 * ui;     // first column of the unit
        if (R0 < u.Pd && !SM_DBG(a, 8)) {
          for (int bj = tsub; sq ? (cu0 + 32 * bj <= R0) : (bj < 2); bj += 2) {
            const int32_t C0 = cu0 + 32 * bj;
            uint32_t v[2][16];
            ptx::tmem_ld_16x256b_x4(taddr + (uint32_t)(C0 - u.n0), v[0]);                  // rows R0 + {g, g + 8}
            ptx::tmem_ld_16x256b_x4(taddr + (16u << 16) + (uint32_t)(C0 - u.n0), v[1]);    // rows R0 + 16 + {g, g + 8}
            const uint32_t cb = ((uint32_t)C0 & 63u) >> 3;
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
                if (p1) {
                  if (diag) {
                    const int rr = 8 * ti + g, c0 = 8 * tj + 2 * q2;
                    if (R0 + rr < u.m) { if (c0 == rr) f0 -= 1.f; if (c0 + 1 == rr) f1 -= 1.f; }   // W = Y - I
                    if (tj <= ti) {
                      if (c0 <= rr) acc = fmaf(c0 == rr ? f0 : 2.f * f0, f0, acc);
                      if (c0 + 1 <= rr) acc = fmaf(c0 + 1 == rr ? f1 : 2.f * f1, f1, acc);
                    }
                  } else {
                    acc = fmaf(f0, f0, acc); acc = fmaf(f1, f1, acc);
                  }
                  f0 *= a.w_scale; f1 *= a.w_scale;         // Wh = -1/2 W is what PHASE 2 multiplies by
                } else if (a.out_scale != 1.f) {
                  f0 *= a.out_scale; f1 *= a.out_scale;
                }
                o[ti][tj] = (BF16 && !a.out_f16) ? pack2<true>(f0, f1) : pack2<false>(f0, f1);
              }
            }
            if (p1) { if (diag) res += acc; else res2 += acc; }
            if (diag) {
              // diagonal tiles: element (r, c > r) := element (c, r), through the transposed fragment
#pragma unroll
              for (int ti = 0; ti < 4; ++ti) {
                const uint32_t tr = ptx::movmatrix_t(o[ti][ti]);
                const uint32_t sel = (2 * q2 <= g ? 0x10u : 0x54u) | ((2 * q2 + 1 <= g ? 0x32u : 0x76u) << 8);
                o[ti][ti] = __byte_perm(o[ti][ti], tr, sel);
              }
            }
            // direct: rows R0 .., columns C0 .. of the unit's direct piece
            const uint32_t dbase = stg + (sq ? (uint32_t)((C0 - u.row0) >> 6) * 16384u : 0u) +
                                   (uint32_t)(R0 - u.row0 + rl) * 128u + (((cb + (uint32_t)ml) ^ (uint32_t)rl) << 4);
#pragma unroll
            for (int ti = 0; ti < 4; ++ti) ptx::stsm_x4(dbase + ti * 1024u, o[ti][0], o[ti][1], o[ti][2], o[ti][3]);
            // mirror: tile (ti, tj) transposed -> rows C0 + 8 tj .., columns R0 + 8 ti ..
            const uint32_t mbase = sq ? stg + (uint32_t)((R0 - u.row0) >> 6) * 16384u + (uint32_t)(C0 - u.row0 + rl) * 128u
                                      : stg + 16384u + (uint32_t)((R0 - u.row0) >> 6) * 8192u + (uint32_t)((C0 & 63) + rl) * 128u;
            if (!diag) {
              if (sq || mirror_out) {
                const uint32_t ma = mbase + (((rb + (uint32_t)ml) ^ (uint32_t)rl) << 4);
#pragma unroll
                for (int tj = 0; tj < 4; ++tj) ptx::stsm_x4_t(ma + tj * 1024u, o[0][tj], o[1][tj], o[2][tj], o[3][tj]);
              }
            } else {
              __syncwarp();       // the direct stores of the upper tiles come first
              ptx::stsm_x4_t(mbase + (((rb + (uint32_t)ml) ^ (uint32_t)rl) << 4), o[0][0], o[1][0], o[2][0], o[3][0]);
              ptx::stsm_x2_t(mbase + 1024u + (((rb + 2u + (uint32_t)(ml & 1)) ^ (uint32_t)rl) << 4), o[2][1], o[3][1]);
              ptx::stsm_x1_t(mbase + 2048u + (((rb + 3u) ^ (uint32_t)rl) << 4), o[3][2]);
            }
          }
        }
        ptx::fence_proxy_async_smem();             // generic-proxy stores -> the bulk copies' async-proxy reads
        team_bar();
        if (leader && Og) {
          const int64_t Pd64 = (int64_t)u.Pd * 64;
          if (sq) {
            for (int pz = 0; pz < 2; ++pz)
              if (u.row0 + 64 * pz < u.Pd)
                ptx::tma_bulk_s2g(Og + ((int64_t)((u.row0 >> 6) + pz) * Pd64 + (int64_t)u.row0 * 64), stg + pz * 16384u,
                                  (uint32_t)a_rows * 128u);
          } else {
            ptx::tma_bulk_s2g(Og + ((int64_t)(cu0 >> 6) * Pd64 + (int64_t)u.row0 * 64), stg, (uint32_t)a_rows * 128u);
            for (int pz = 0; pz < 2; ++pz)
              if (mirror_out && u.row0 + 64 * pz < u.Pd)
                ptx::tma_bulk_s2g(Og + ((int64_t)((u.row0 >> 6) + pz) * Pd64 + (int64_t)cu0 * 64), stg + 16384u + pz * 8192u, 8192u);
          }
          ptx::bulk_commit();
        }
      }
      res += 2.f * res2;
      // accumulator drained: hand the TMEM stage back to the MMA warp
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) ptx::mbar_arrive(tempty_bar(as));
      if (p1) {
        for (int d = 16; d > 0; d >>= 1) res += __shfl_xor_sync(0xffffffffu, res, d);
        if (lane == 0)
          a.s.partial[(int64_t)u.c * a.s.parts_per_col + (int64_t)u.lt * EPI_WARPS + (warp - 2)] = (double)res;
      }
      ++it;
    }
    if (leader) {
      ptx::bulk_wait0();
      if (STREAM && pend) { __threadfence(); atomicAdd(pend, EPI_WARPS / 2); }
    }
  } else {
    // ===================== epilogue (warps 2..17) =====================
    // EPI_WARPS / 4 warps per TMEM lane quadrant; a warp owns 32 rows and every (EPI_WARPS/4)-th
    // 32-column block at or below the diagonal.  Tiles start at multiples of 32 columns, so a block is
    // either strictly below the diagonal (stored at (r, c) directly and at (c, r) through a warp-private
    // smem transpose, both as 16-byte stores) or the diagonal block itself (symmetrised in smem: the
    // lower triangle overwrites the upper one, then stored once).  Padding rows/columns of X are zero,
    // so their accumulators are exactly zero and need no special path.
    constexpr int NSUB = EPI_WARPS / 4;
    const int q = warp & 3;                        // TMEM lane quadrant this warp may access
    const int sub = (warp - 2) >> 2;               // which column blocks this warp takes
    uint16_t *const stg0 = reinterpret_cast<uint16_t *>(smem_raw + (stage_base - raw)) + q * NACC * 1024;
    uint32_t it = 0;
    TileDesc nxt = load_desc(a, max((int64_t)0, min(unit, total - 1)));
    int64_t t = unit;
    uint32_t qs = 0, qp = 0;
    auto fetch = [&](TileDesc &cur) -> bool {
      if (DYN) {
        ptx::mbar_wait(tqf_bar(qs), qp, a.err_flag, 10);
        cur = tq[qs];
        __syncwarp();                                   // every lane has its copy before the slot is handed back
        if (lane == 0) ptx::mbar_arrive(tqe_bar(qs));
        if (++qs == TQ) { qs = 0; qp ^= 1u; }
        return cur.c >= 0;
      }
      if (t >= total) return false;
      cur = nxt;
      nxt = load_desc(a, min(t + n_units, total - 1));
      t += n_units;
      return true;
    };
    TileDesc cur;
    while (fetch(cur)) {
      UTile u = make_tile<PHASE>(a, cur);
      if (!u.valid) continue;
      const uint32_t as = it % NACC, aphase = (it / NACC) & 1u;
      // diagonal-block buffer of (quadrant, accumulator stage): a tile has one diagonal block per quadrant, and
      // two tiles on the same stage cannot be in flight at once
      uint16_t *const stg = stg0 + as * 1024;
      const int32_t R0 = u.row0 + (int32_t)h * UM + q * 32;   // this CTA's 128 rows of the tile
      const int32_t r = R0 + lane;
      const bool p1 = STREAM ? (cur.pad0 & 1) == 0 : PHASE == 1;
      // stream: product ph of step ph / 2 writes Wh (even ph) or the X buffer that step does not read (odd ph)
      uint16_t *Og = (uint16_t *)(!STREAM ? a.Out : p1 ? a.Ybuf : (((cur.pad0 >> 1) & 1) ? (void *)a.Xsrc : a.Out)) + u.base;
      if (SM_DBG(a, 1)) Og = nullptr;
      const int nblk = (u.nt + 31) >> 5;
      ptx::mbar_wait(tfull_bar(as), aphase, a.err_flag, 4);
      ptx::tc_fence_after();
      const uint32_t taddr = tmem_base + as * UN + ((uint32_t)(q * 32) << 16);
      float res = 0.f, res2 = 0.f;                             // diagonal-block / off-diagonal (counted twice) sums
      if (R0 < u.Pd && !SM_DBG(a, 8)) {
        const uint32_t r7 = (uint32_t)lane & 7u;                 // r & 7 (R0 is a multiple of 32)
        for (int bi = sub; bi < nblk; bi += NSUB) {
          const int32_t vc = u.n0 + bi * 32;                     // virtual column; from u.fb on: a folded row of the last panel
          const bool fcol = vc >= u.fb;
          const int32_t C0 = fcol ? vc + u.fs : vc;
          if (SYM ? (!fcol && C0 > R0) : (C0 >= u.Pd)) {         // above the diagonal / past the padded dimension
            if (SYM && u.fb != 0x7fffffff) continue;             // folded columns may still follow
            break;
          }
          uint32_t v[32];
          ptx::tmem_ld16(taddr + (uint32_t)(bi * 32), *reinterpret_cast<uint32_t(*)[16]>(&v[0]));
          ptx::tmem_ld16(taddr + (uint32_t)(bi * 32 + 16), *reinterpret_cast<uint32_t(*)[16]>(&v[16]));
          // element offset of (r, C0) in the image and the swizzled positions of its four 16-byte chunks
          const int64_t rowoff = (int64_t)(C0 >> 6) * u.Pd * 64 + (int64_t)r * 64;
          const uint32_t c8 = ((uint32_t)C0 >> 3) & 4u;          // first chunk of the block inside its 128-byte line
          // The four 16-byte chunks of a row segment sit in two 32-byte sectors; chunk 2s and 2s+1 swap places
          // inside sector s when r is odd (128B swizzle).  One 256-bit access per sector keeps every L2
          // request a full sector (ncu, round 1: 16-byte accesses doubled the sector count of these paths).
          const bool swp = (lane & 1) != 0;
          const uint32_t sec0 = ((c8 ^ r7) & ~1u) << 3, sec1 = (((c8 + 2u) ^ r7) & ~1u) << 3;   // element offsets
          ptx::tmem_ld_wait();
          const bool diag = (C0 == R0);
          uint32_t o[16];                                        // 32 output elements, packed pairs
          float acc = 0.f;
#pragma unroll
          for (int g = 0; g < 4; ++g) {
            float f[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) f[e] = __uint_as_float(v[g * 8 + e]);
            if (p1) {
              // W = Y - I is what gets stored: near convergence Y_rr ~ 1 would lose 2^-9 absolute to the 16-bit
              // rounding every step, W_rr ~ 0 loses nothing; PHASE 2 then forms X' = X - 1/2 X W.
              if (diag && r < u.m) {                               // padding rows keep W = 0
#pragma unroll
                for (int e = 0; e < 8; ++e)
                  if (g * 8 + e == lane) f[e] -= 1.f;
              }
              if (SYM && diag) {
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
              for (int e = 0; e < 8; ++e) f[e] *= a.w_scale;       // Wh = -1/2 W is what PHASE 2 multiplies by
            } else if (a.out_scale != 1.f) {
#pragma unroll
              for (int e = 0; e < 8; ++e) f[e] *= a.out_scale;
            }
#pragma unroll
            for (int e2 = 0; e2 < 4; ++e2)
              o[g * 4 + e2] = (BF16 && !a.out_f16) ? pack2<true>(f[2 * e2], f[2 * e2 + 1]) : pack2<false>(f[2 * e2], f[2 * e2 + 1]);
          }
          if (p1 && r < u.m) { if (SYM && !diag) res2 += acc; else res += acc; }
          uint16_t *Orow = Og ? Og + rowoff : nullptr;
          if (!SYM) {
            if (Orow) store_row_segment(Orow, sec0, sec1, swp, o);
          } else if (diag) {
            // S[row][col] in smem; then element (row, j > row) is replaced by element (j, row)
#pragma unroll
            for (int g = 0; g < 4; ++g)
              *reinterpret_cast<uint4 *>(stg + lane * 32 + ((g ^ (lane & 3)) << 3)) =
                  make_uint4(o[g * 4], o[g * 4 + 1], o[g * 4 + 2], o[g * 4 + 3]);
            __syncwarp();
#pragma unroll
            for (int j = 0; j < 32; ++j) {
              if (j > lane) {
                // element (j, lane) sits in row j, chunk (lane >> 3) ^ (j & 3), position lane & 7
                const uint16_t m16 = stg[j * 32 + (((lane >> 3) ^ (j & 3)) << 3) + (lane & 7)];
                o[j >> 1] = (j & 1) ? ((o[j >> 1] & 0x0000FFFFu) | ((uint32_t)m16 << 16))
                                    : ((o[j >> 1] & 0xFFFF0000u) | (uint32_t)m16);
              }
            }
            __syncwarp();
            if (Orow) store_row_segment(Orow, sec0, sec1, swp, o);
          } else {
            if (Orow) store_row_segment(Orow, sec0, sec1, swp, o);
            // Mirrored block straight from the registers: element (r, C0 + j) goes to row C0 + j, column r.  The
            // 32 lanes are 32 consecutive columns of that row = 64 contiguous bytes (four swizzled 16-byte chunks
            // of one 128-byte line), so every 2-byte store instruction fills two whole sectors.  No shared-memory
            // transpose: its 2 KB of sub-word stores per block competed with the MMA and TMA for the shared-memory
            // pipe (clock64 time line, round 1: 600-1000 cycles per block).
            if (Og) mirror_store(Og, u.Pd, R0, C0, lane, o);
          }
        }
      }
      res += 2.f * res2;
      // accumulator drained: hand the TMEM stage back to the MMA warp
      ptx::tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        if (PAIR) ptx::mbar_arrive_remote(tempty_bar(as), 0); else ptx::mbar_arrive(tempty_bar(as));
      }
      if (p1) {
        for (int d = 16; d > 0; d >>= 1) res += __shfl_xor_sync(0xffffffffu, res, d);
        if (lane == 0)
          a.s.partial[(int64_t)u.c * a.s.parts_per_col + (int64_t)u.lt * (EPI_WARPS * NCTA) + (int64_t)h * EPI_WARPS +
                      (warp - 2)] = (double)res;
      }
      if (STREAM && cur.pad0 + 1 < a.n_ph && !SM_DBG(a, 128)) {
        // this warp's stores of the tile: visible gpu-wide and to the async proxy, then counted for the group's product
        __threadfence();
        ptx::fence_proxy_async();
        __syncwarp();
        if (lane == 0) atomicAdd(a.done + (int64_t)cur.pad1 * a.n_ph + cur.pad0, 1);
      }
      ++it;
    }
  }

  ptx::tc_fence_before();
  __syncwarp();
  if (CL2) ptx::cluster_sync_all(); else __syncthreads();
  if (warp == 1) {
    ptx::tc_fence_after();
    if (PAIR) ptx::tmem_dealloc2(tmem_base, TMEM_COLS); else ptx::tmem_dealloc(tmem_base, TMEM_COLS);
  }
}


#ifdef SM_MEASURE
#include "sign_umma_fused.cuh"
#endif
#include "sign_resident.cuh"

// Fixed-iteration bookkeeping of the grouped path: residual of the last step from its partial sums (one warp per
// listed column, fixed order), iters = max_iter.  Columns with Pd <= skip_pd (shared-memory-resident kernel) are
// not touched.
static __global__ void k_fused_post(int32_t n_cols, const int32_t *__restrict__ cols, const int32_t *__restrict__ dim,
                                    const int32_t *__restrict__ dim_pad, int32_t skip_pd,
                                    const double *__restrict__ partial, int32_t parts_per_col,
                                    const int32_t *__restrict__ n_parts, int32_t max_iter, int32_t *iters,
                                    double *residual) {
  const int32_t c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (c >= n_cols) return;
  const int32_t i = cols ? cols[c] : c;
  if (dim_pad[i] <= skip_pd) return;
  const double *p = partial + (int64_t)c * parts_per_col;
  double sum = 0.0;
  const int32_t np = n_parts[c];
  for (int32_t t = lane; t < np; t += 32) sum += p[t];
  for (int d = 16; d > 0; d >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, d);
  if (lane == 0) {
    residual[c] = max_iter > 0 ? sqrt(sum / (double)dim[i]) : 0.0;
    iters[c] = max_iter;
  }
}

static __global__ void k_umma_tilecounts(int32_t n_cols, int32_t R, int32_t sym, int32_t fold, int32_t parts_per_tile, int32_t skip_pd,
                                         const int32_t *__restrict__ cols, const int32_t *__restrict__ dim,
                                         const int32_t *__restrict__ dim_pad, int64_t *__restrict__ tiles,
                                         int32_t *__restrict__ n_parts) {
  int32_t c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_cols) return;
  int32_t i = cols ? cols[c] : c;
  int32_t nt = dim_pad[i] <= skip_pd ? 0
               : sym == 2            ? v_tiles(dim[i])
               : (sym && fold && R == UM) ? w_tiles(dim[i], w_fold(dim[i]))
               : sym                 ? u_tiles(dim[i], R)
                                     : f_tiles(dim_pad[i], R);
  tiles[c] = nt;
  n_parts[c] = nt * parts_per_tile;
}

// What the symmetric single-CTA tiles never write of the two scratch images of a grouped submatrix, zeroed once per call
// instead of clearing both buffers whole (2 x 1.26 GB at configs[2]: 0.5 ms per call; at configs[3] 2 x 0.73 GB for the
// 229 submatrices that are not resident).  The epilogues write every element (r < Pd, c < n32), n32 = m rounded up to 32
// (lower blocks directly, upper ones mirrored) -- except, with the folded geometry, the rows >= n32 left of the last
// panel's square.  Rows [n32, Pd) are read as A-operand rows and columns [n32, Pd) travel with copy-back: both must be 0.
// One CTA per listed column; in the image a row range of a 64-column chunk is contiguous.
static __global__ void __launch_bounds__(256)
k_zero_padding(int32_t n_cols, const int32_t *__restrict__ cols, const int32_t *__restrict__ dim,
               const int32_t *__restrict__ dim_pad, const int64_t *__restrict__ col_off, int32_t skip_pd,
               uint16_t *__restrict__ B0, uint16_t *__restrict__ B1) {
  const int32_t c = blockIdx.x, i = cols ? cols[c] : c;
  const int32_t m = dim[i], Pd = dim_pad[i], n32 = (m + 31) & ~31;
  if (Pd <= skip_pd || n32 >= Pd) return;
  const uint4 z = make_uint4(0u, 0u, 0u, 0u);
  const int32_t pr = Pd - n32;                                   // padding rows = padding columns
#pragma unroll
  for (int b = 0; b < 2; ++b) {
    uint16_t *img = (b ? B1 : B0) + col_off[c];
    // rows [n32, Pd) of every chunk: pr x 128 B contiguous
    const int32_t per = pr * 8;                                  // 16-byte units per chunk
    for (int32_t e = threadIdx.x; e < (Pd >> 6) * per; e += blockDim.x) {
      const int32_t ch = e / per, u = e - ch * per;
      reinterpret_cast<uint4 *>(img + (int64_t)ch * Pd * 64 + (int64_t)n32 * 64)[u] = z;
    }
    // columns [n32, Pd) of rows [0, n32): 16-byte units (n32 & 63) / 8 .. 7 of the last chunk, at their swizzled places
    const int32_t u0 = (n32 & 63) >> 3, nu = 8 - u0;
    uint16_t *last = img + (int64_t)((Pd >> 6) - 1) * Pd * 64;
    for (int32_t e = threadIdx.x; e < n32 * nu; e += blockDim.x) {
      const int32_t r = e / nu, u = u0 + (e - r * nu);
      reinterpret_cast<uint4 *>(last + (int64_t)r * 64)[u ^ (r & 7)] = z;
    }
  }
}

// iters / residual of the columns the resident kernel does not take start at zero; its own are written by it
static __global__ void k_sign_init_grouped(int32_t n_cols, const int32_t *__restrict__ cols,
                                           const int32_t *__restrict__ dim_pad, int32_t skip_pd, int32_t *active,
                                           int32_t *last, int32_t *iters, double *residual) {
  int32_t c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_cols) return;
  const bool mine = dim_pad[cols ? cols[c] : c] > skip_pd;
  active[c] = mine ? 1 : 0; last[c] = 0;
  if (mine) { if (iters) iters[c] = 0; if (residual) residual[c] = 0.0; }
}

constexpr int UMMA_MAX_COUNTERS = 256;      // 2 per step; more steps than that fall back to the static deal
struct UmmaWs {
  void *Y, *X2; int32_t *active, *last, *n_still, *n_parts, *err; int64_t *tile_ptr; double *partial;
  unsigned long long *counters;   // one tile counter per product launch (dynamic scheduling) + 1 for the resident kernel
  int32_t *done;                  // stream mode: [groups][2 * steps] completion counters
  TileDesc *tiles;
  int32_t parts_per_col; int64_t used;
};

// Variant selection (sm_set_option / environment at load; include/submatrix.h lists the names).  Measured on B200
// (sm_sign_ns alone, one box): single CTAs per tile beat every two-CTA variant (configs[4]: 603 vs 653-762 ms;
// configs[2]: 26-28 vs 31-32 ms), SYM beats FULL at every size (configs[2]: 0.77 vs 1.13 ms per launch), the dynamic
// deal beats round robin; the two-CTA and fused variants are therefore only in a -DSM_MEASURE build.
static int32_t umma_ncta() {
#ifdef SM_MEASURE
  return opt(OPT_UMMA_NCTA) == 2 ? 2 : 1;
#else
  return 1;
#endif
}
static bool umma_fused(double tol) {
#ifdef SM_MEASURE
  return !(tol > 0.0) && opt(OPT_UMMA_FUSED) == 1;
#else
  (void)tol; return false;
#endif
}
static int32_t umma_dbg() {
#ifdef SM_MEASURE
  return opt(OPT_UMMA_DBG);
#else
  return 0;
#endif
}
// 0 = true products on all tiles, 1 = symmetric half tiles with per-lane global stores, 2 = symmetric half tiles with
// the staged epilogue (single CTAs, one launch per product)
static int32_t umma_sym_mode(int32_t nonsym, bool fused, int32_t ncta, double tol, int32_t max_iter) {
  if (fused) return 1;
  if (nonsym || opt(OPT_UMMA_SYM) == 0) return 0;
  (void)tol; (void)max_iter;
  return (opt(OPT_UMMA_EPI) != 0 && ncta == 1) ? 2 : 1;
}
// all listed columns with Pd <= this go through k_umma_resident (0: none)
static int32_t umma_resident_pd(int32_t sym) { return (sym && opt(OPT_UMMA_RESIDENT) != 0) ? RES_MAX_PD : 0; }

static UmmaWs umma_layout(void *ws, int64_t ws_bytes, const sm_pattern_t *P, int32_t n_cols,
                          int64_t packed_elems, int32_t sym, bool o3) {
  WsCursor cur(ws, ws_bytes);
  UmmaWs w;
  // sized for whichever variant sign_umma picks (the query does not know tol): per-phase launches with
  // the selected NCTA / SYM, or the fused kernel (CTA pairs, SYM)
  const int32_t ncta = umma_ncta();
  // (the folded geometry can need one tile more than the unfolded one at a smaller dimension: + 1)
  const int32_t t_sel = sym == 2 ? v_tiles(P->max_dim) : sym ? u_tiles(P->max_dim, UM * ncta) + 1 : f_tiles(P->max_dim_pad, UM * ncta);
  const int32_t t_fused = u_tiles(P->max_dim, UM * 2);
  const int32_t max_tiles = t_sel > t_fused ? t_sel : t_fused;
  w.parts_per_col = (t_sel * ncta > t_fused * 2 ? t_sel * ncta : t_fused * 2) * EPI_WARPS;
  // when every listed column can be resident the grouped path's two image buffers are not needed (the third-order
  // iteration has no resident kernel)
  const bool all_res = !o3 && umma_resident_pd(sym) >= P->max_dim_pad;
  w.Y = cur.take<char>(all_res ? 0 : packed_elems * 2);
  w.X2 = cur.take<char>(all_res ? 0 : packed_elems * 2);
  w.active = cur.take<int32_t>(n_cols);
  w.last = cur.take<int32_t>(n_cols);
  w.n_still = cur.take<int32_t>(1);
  w.err = cur.take<int32_t>(1);
  w.counters = cur.take<unsigned long long>(UMMA_MAX_COUNTERS + 1);
  w.done = cur.take<int32_t>((int64_t)(n_cols / STREAM_G + 1) * UMMA_MAX_COUNTERS);
  w.n_parts = cur.take<int32_t>(n_cols);
  w.tile_ptr = cur.take<int64_t>(n_cols + 1);
  w.partial = cur.take<double>((int64_t)n_cols * w.parts_per_col);
  w.tiles = cur.take<TileDesc>((int64_t)n_cols * max_tiles);
  w.used = cur.used + 256;
  return w;
}

int64_t sign_umma_ws_bytes(const sm_pattern_t *P, int32_t n_cols, int64_t packed_elems, int32_t x_dtype,
                           int32_t nonsym, int32_t order) {
  (void)x_dtype;
  // sized for the larger of the tile tables the call may pick (the query does not know tol / max_iter)
  const int64_t a = umma_layout(nullptr, 0, P, n_cols, packed_elems, umma_sym_mode(nonsym, false, umma_ncta(), 0.0, 1), order == 3).used;
  const int64_t b = umma_layout(nullptr, 0, P, n_cols, packed_elems, umma_sym_mode(nonsym, false, umma_ncta(), 1.0, 1), order == 3).used;
  return a > b ? a : b;
}

#ifdef SM_MEASURE
// 2-D tensor maps over a packed 16-bit buffer seen as rows of 64 elements (128 bytes): box = 64 x box_rows, no
// swizzle (the image is stored pre-swizzled).  Used by the TM variant only; the others get zeroed maps.
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static int32_t make_map(CUtensorMap *m, void *buf, int64_t packed_elems, uint32_t box_rows) {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    SM_CUDA(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q));
    if (!p || q != cudaDriverEntryPointSuccess) return SM_ERR_UNSUPPORTED;
    fn = (EncodeTiledFn)p;
  }
  cuuint64_t gdim[2] = {64, (cuuint64_t)(packed_elems / 64)};
  cuuint64_t gstr[1] = {128};
  cuuint32_t box[2] = {64, box_rows};
  cuuint32_t estr[2] = {1, 1};
  CUresult r = fn(m, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, buf, gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                  CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) { g_last_cuda_error = (int32_t)r; return SM_ERR_CUDA; }
  return SM_OK;
}
#endif
struct UMaps { CUtensorMap a, b; };

template <bool BF16, int PHASE, int NCTA, bool SYM, bool MC = false, int NST = 0, bool TM = false, bool DYN = false, int EPI = 0>
static int32_t launch_umma(const UArgs &a, const UMaps &maps, int32_t n_sm, cudaStream_t st) {
  // set on every call: the attribute is per device and a process may use several
  SM_CUDA(cudaFuncSetAttribute(k_umma_gemm<BF16, PHASE, NCTA, SYM, MC, NST, TM, DYN, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                               UCfg<NCTA, MC, NST, EPI>::SMEM));
  int slot = -1;
  { int32_t rc = prof_begin(st, &slot); if (rc != SM_OK) return rc; }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(n_sm / NCTA * NCTA), 1, 1);     // one CTA per SM, whole pairs
  cfg.blockDim = dim3(UMMA_THREADS, 1, 1);
  cfg.dynamicSmemBytes = UCfg<NCTA, MC, NST, EPI>::SMEM;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = NCTA; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  SM_CUDA(cudaLaunchKernelEx(&cfg, k_umma_gemm<BF16, PHASE, NCTA, SYM, MC, NST, TM, DYN, EPI>, a, maps.a, maps.b));
  SM_LAUNCHED();
  return prof_end(st, slot);
}

#ifdef SM_MEASURE
template <bool BF16, int NSLOT>
static int32_t launch_fused(const FArgs &a, int32_t n_sm, cudaStream_t st) {
  SM_CUDA(cudaFuncSetAttribute(k_umma_fused<BF16, NSLOT>, cudaFuncAttributeMaxDynamicSharedMemorySize, UCfg<2>::SMEM));
  int slot = -1;
  { int32_t rc = prof_begin(st, &slot); if (rc != SM_OK) return rc; }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3((unsigned)(n_sm / 2 * 2), 1, 1);
  cfg.blockDim = dim3(UMMA_THREADS, 1, 1);
  cfg.dynamicSmemBytes = UCfg<2>::SMEM;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  SM_CUDA(cudaLaunchKernelEx(&cfg, k_umma_fused<BF16, NSLOT>, a));
  SM_LAUNCHED();
  return prof_end(st, slot);
}
#endif

template <int PHASE, int NCTA, bool SYM, bool MC = false, int NST = 0, bool TM = false, bool DYN = false, int EPI = 0>
static int32_t launch_umma_t(bool bf16, const UArgs &a, const UMaps &m, int32_t n_sm, cudaStream_t st) {
  return bf16 ? launch_umma<true, PHASE, NCTA, SYM, MC, NST, TM, DYN, EPI>(a, m, n_sm, st)
              : launch_umma<false, PHASE, NCTA, SYM, MC, NST, TM, DYN, EPI>(a, m, n_sm, st);
}
// mode: 1 = one CTA per tile; SM_MEASURE builds only: 2 = cta_group::2 pair with relay, 3 = two CTAs with multicast B,
// 4 = pair with tensor maps
template <int PHASE>
static int32_t launch_umma_any(bool bf16, int32_t mode, int32_t sym, int32_t nst, const UArgs &a, const UMaps &m,
                               int32_t n_sm, cudaStream_t st) {
#ifdef SM_MEASURE
  if (mode == 4) return nst == 3 ? launch_umma_t<PHASE, 2, true, false, 3, true>(bf16, a, m, n_sm, st)
                      : nst == 4 ? launch_umma_t<PHASE, 2, true, false, 4, true>(bf16, a, m, n_sm, st)
                                 : launch_umma_t<PHASE, 2, true, false, 6, true>(bf16, a, m, n_sm, st);
  if (mode == 3) return launch_umma_t<PHASE, 2, true, true>(bf16, a, m, n_sm, st);
  if (mode == 2) return sym ? launch_umma_t<PHASE, 2, true>(bf16, a, m, n_sm, st) : launch_umma_t<PHASE, 2, false>(bf16, a, m, n_sm, st);
#else
  (void)mode;
#endif
  if (sym == 2)              // staged epilogue (bulk stores), 3-stage ring
    return a.counter ? launch_umma_t<PHASE, 1, true, false, 0, false, true, 1>(bf16, a, m, n_sm, st)
                     : launch_umma_t<PHASE, 1, true, false, 0, false, false, 1>(bf16, a, m, n_sm, st);
  if (sym && a.counter)      // dynamic tile scheduling
    return nst == 3 ? launch_umma_t<PHASE, 1, true, false, 3, false, true>(bf16, a, m, n_sm, st)
                    : launch_umma_t<PHASE, 1, true, false, 0, false, true>(bf16, a, m, n_sm, st);
  if (sym && nst == 3) return launch_umma_t<PHASE, 1, true, false, 3>(bf16, a, m, n_sm, st);
  return sym ? launch_umma_t<PHASE, 1, true>(bf16, a, m, n_sm, st) : launch_umma_t<PHASE, 1, false>(bf16, a, m, n_sm, st);
}

static int32_t launch_resident(bool bf16, const RArgs &a, int32_t n_sm, cudaStream_t st) {
  auto k = bf16 ? k_umma_resident<true> : k_umma_resident<false>;
  SM_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, RES_SMEM));
  int slot = -1;
  { int32_t rc = prof_begin(st, &slot); if (rc != SM_OK) return rc; }
  const int32_t grid = a.n_cols < n_sm ? a.n_cols : n_sm;
  k<<<grid, RES_THREADS, RES_SMEM, st>>>(a);
  SM_LAUNCHED();
  return prof_end(st, slot);
}

int32_t sign_umma(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off,
                  int64_t packed_elems, int32_t x_dtype, void *X, void *ws, int64_t ws_bytes,
                  int32_t max_iter, double tol, int32_t *iters, double *residual, int32_t nonsym, int32_t switch_iter,
                  int32_t order, cudaStream_t st) {
  if ((P->pad_to % 64) != 0) return SM_ERR_ARG;
  const bool bf16 = x_dtype == SM_BF16;
  // third-order iteration (f3, reading A22): three grouped products per step (no resident / stream / fused variant)
  const bool o3 = order == 3;
  if (o3 && nonsym) return SM_ERR_UNSUPPORTED;
  if (switch_iter >= 0) {
    // mixed schedule (f3): bf16 in, fp16 out; fixed iteration counts, symmetric iterates
    if (!bf16 || nonsym || tol > 0.0 || switch_iter < 1 || switch_iter >= max_iter) return SM_ERR_ARG;
  }
  const bool fused = !nonsym && !o3 && switch_iter < 0 && umma_fused(tol);
  const int32_t ncta = fused ? 2 : umma_ncta(), R = UM * ncta;
  const int32_t sym = umma_sym_mode(nonsym, fused, ncta, tol, max_iter);
  UmmaWs w = umma_layout(ws, ws_bytes, P, n_cols, packed_elems, sym, order == 3);
  if (w.used > ws_bytes) return SM_ERR_SPACE;
  int dev = 0, n_sm = 0;
  SM_CUDA(cudaGetDevice(&dev));
  SM_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  // a kernel protocol failure (a barrier that never completes) writes its reason code here before it traps:
  // pinned host memory, readable after the sticky error (sm_last_device_error)
  w.err = device_err_word();
  const int32_t nb = (n_cols + 255) / 256;

  // ---- small submatrices: all steps inside one CTA (k_umma_resident)
  const int32_t res_pd = (fused || o3) ? 0 : umma_resident_pd(sym);
  if (res_pd > 0) {
    SM_CUDA(cudaMemsetAsync(w.counters + UMMA_MAX_COUNTERS, 0, sizeof(unsigned long long), st));
    RArgs r{cols, col_off, P->dim, P->dim_pad, n_cols, max_iter, tol, X, iters, residual,
            w.counters + UMMA_MAX_COUNTERS, w.err, switch_iter};
    int32_t rc = launch_resident(bf16, r, n_sm, st);
    if (rc != SM_OK) return rc;
    if (res_pd >= P->max_dim_pad) return SM_OK;          // every listed column was resident
  }

  // ---- the rest: grouped tiles, one launch per product (or stream / fused)
  SignState s{w.active, w.last, w.n_still, w.partial, w.parts_per_col};
  k_sign_init_grouped<<<nb, 256, 0, st>>>(n_cols, cols, P->dim_pad, res_pd, w.active, w.last, iters, residual);
  SM_LAUNCHED();
  // folded geometry of the symmetric single-CTA tiles (option "umma.fold"; see w_fold)
  const int32_t fold = (sym == 1 && ncta == 1 && opt(OPT_UMMA_FOLD) != 0) ? 1 : 0;
  k_umma_tilecounts<<<nb, 256, 0, st>>>(n_cols, R, sym, fold, EPI_WARPS * ncta, res_pd, cols, P->dim, P->dim_pad, w.tile_ptr,
                                        w.n_parts);
  SM_LAUNCHED();
  { int32_t rc = exclusive_scan_i64(n_cols, w.tile_ptr, w.tile_ptr, st); if (rc != SM_OK) return rc; }
  // product 1 reads its A rows from the B stage where a tile holds its diagonal square (option "umma.sharea"; see share_a_off)
  const int32_t share_a = (sym == 1 && ncta == 1 && opt(OPT_UMMA_SHAREA) != 0) ? 1 : 0;
  k_umma_build_tiles<<<nb, 256, 0, st>>>(n_cols, R, sym, fold, share_a, res_pd, cols, P->dim, P->dim_pad, col_off, w.tile_ptr, w.tiles);
  SM_LAUNCHED();
  // Y and the alternate X buffer: what the kernels read or copy back without ever writing it must be zero (and never a
  // NaN/Inf bit pattern).  The symmetric single-CTA tiles leave only padding rows / columns unwritten (k_zero_padding);
  // the other variants get both buffers cleared whole.
  if (sym == 1 && ncta == 1) {
    k_zero_padding<<<n_cols, 256, 0, st>>>(n_cols, cols, P->dim, P->dim_pad, col_off, res_pd, (uint16_t *)w.Y, (uint16_t *)w.X2);
    SM_LAUNCHED();
  } else {
    SM_CUDA(cudaMemsetAsync(w.Y, 0, packed_elems * 2, st));
    SM_CUDA(cudaMemsetAsync(w.X2, 0, packed_elems * 2, st));
  }
#ifdef SM_MEASURE
  if (fused) {
    // fixed iteration count: one launch runs every step of every submatrix (k_umma_fused)
    FArgs f{cols, col_off, P->dim, P->dim_pad, n_cols, max_iter, X, w.X2, w.Y, w.partial, w.parts_per_col, w.err, nullptr, umma_dbg()};
    // SM_UMMA_TRACE=<file>: measurement only -- clock64 time line of CTA pair 0 (debug allocation, synchronises)
    const char *trace_path = getenv("SM_UMMA_TRACE");
    const size_t trace_bytes = (size_t)2 * 4 * TRACE_N * 2 * sizeof(unsigned long long);
    if (trace_path) {
      SM_CUDA(cudaMalloc((void **)&f.trace, trace_bytes));
      SM_CUDA(cudaMemsetAsync(f.trace, 0, trace_bytes, st));
    }
    const int32_t nslot = opt(OPT_UMMA_SLOTS) == 1 ? 1 : 2;
    int32_t rc = nslot == 2 ? (bf16 ? launch_fused<true, 2>(f, n_sm, st) : launch_fused<false, 2>(f, n_sm, st))
                            : (bf16 ? launch_fused<true, 1>(f, n_sm, st) : launch_fused<false, 1>(f, n_sm, st));
    if (rc != SM_OK) return rc;
    if (trace_path) {
      std::vector<unsigned long long> hbuf(trace_bytes / sizeof(unsigned long long));
      SM_CUDA(cudaMemcpyAsync(hbuf.data(), f.trace, trace_bytes, cudaMemcpyDeviceToHost, st));
      SM_CUDA(cudaStreamSynchronize(st));
      SM_CUDA(cudaFree(f.trace));
      if (FILE *fp = fopen(trace_path, "wb")) { fwrite(hbuf.data(), 1, trace_bytes, fp); fclose(fp); }
    }
    k_fused_post<<<(n_cols + 7) / 8, 256, 0, st>>>(n_cols, cols, P->dim, P->dim_pad, 0, w.partial, w.parts_per_col, w.n_parts,
                                                   max_iter, iters, residual);
    SM_LAUNCHED();
    dim3 cgf(n_cols, 8);
    k_copy_back<<<cgf, 256, 0, st>>>(cols, col_off, iters, 2, P->dim_pad, 0, (const char *)w.X2, (char *)X);
    SM_LAUNCHED();
    return SM_OK;
  }
  const int32_t mode = (ncta == 2 && sym && opt(OPT_UMMA_MC) != 0) ? 3 : (ncta == 2 && sym && opt(OPT_UMMA_TMAP) == 1) ? 4 : ncta;
#else
  const int32_t mode = 1;
#endif
  UMaps maps[3] = {};              // per buffer: X, alternate X, W (mode 4 only)
#ifdef SM_MEASURE
  if (mode == 4) {
    void *bufs[3] = {X, w.X2, w.Y};
    for (int b = 0; b < 3; ++b) {
      int32_t rc = make_map(&maps[b].a, bufs[b], packed_elems, 128);
      if (rc == SM_OK) rc = make_map(&maps[b].b, bufs[b], packed_elems, 64);
      if (rc != SM_OK) return rc;
    }
  }
#endif
  const int32_t nst_opt = opt(OPT_UMMA_STAGES);
  const int32_t nper = o3 ? 3 : 2;           // products (launches, tile counters) per step
  const bool dyn = opt(OPT_UMMA_DYN) != 0 && mode == 1 && sym && nper * max_iter <= UMMA_MAX_COUNTERS;
  // ring depth: with the static deal large submatrices want the shallow ring (see UCfg); the dynamic deal removes
  // the drift that made the deep ring costly (configs[4], 25 steps: 603 ms with 4 stages, 615 ms with 3)
  const int32_t nst = nst_opt ? nst_opt : (mode == 4 ? 6 : ((!dyn && P->max_dim > 1024) ? 3 : 4));
  if (dyn) SM_CUDA(cudaMemsetAsync(w.counters, 0, sizeof(unsigned long long) * UMMA_MAX_COUNTERS, st));
  if (opt(OPT_UMMA_STREAM) == 1 && dyn && !o3 && !(tol > 0.0) && max_iter > 0 && switch_iter < 0) {
    const int64_t n_done = (int64_t)(n_cols / STREAM_G + 1) * 2 * max_iter;
    SM_CUDA(cudaMemsetAsync(w.done, 0, sizeof(int32_t) * n_done, st));
    UArgs a{cols, col_off, P->dim, P->dim_pad, w.tile_ptr, w.tiles, n_cols, 0, X, w.Y, w.X2, s, w.err, 0, w.counters,
            2 * max_iter, w.done, umma_dbg(), 0, 0, 0, -0.5f, 1.f};
    a.fold = fold; a.share_a = share_a;
    int32_t rc = sym == 2 ? launch_umma_t<0, 1, true, false, 0, false, true, 1>(bf16, a, maps[0], n_sm, st)
                          : launch_umma_t<0, 1, true, false, 0, false, true>(bf16, a, maps[0], n_sm, st);
    if (rc != SM_OK) return rc;
    k_fused_post<<<(n_cols + 7) / 8, 256, 0, st>>>(n_cols, cols, P->dim, P->dim_pad, res_pd, w.partial, w.parts_per_col, w.n_parts,
                                                   max_iter, iters, residual);
    SM_LAUNCHED();
    dim3 cgs(n_cols, 8);
    k_copy_back<<<cgs, 256, 0, st>>>(cols, col_off, iters, 2, P->dim_pad, res_pd, (const char *)w.X2, (char *)X);
    SM_LAUNCHED();
    return SM_OK;
  }
  const int32_t rev_on = opt(OPT_UMMA_REV) != 0 ? 1 : 0;
#ifdef SM_MEASURE
  if (o3 && mode != 1) return SM_ERR_UNSUPPORTED;
#endif
  // Newton-Schulz: X alternates between X and ws.X2, Wh lives in ws.Y.  Order 3: X alternates between X and ws.Y,
  // Q = 3/4 (I - X X) is written where X' will go (it is dead after the second product), Z = 2/3 (Q + Q Q) lives in
  // ws.X2, X' = X + X Z.  The second product IS the update product with X := Q, Wh := Q (the identity MMAs add Q).
  void *buf[2] = {X, o3 ? w.Y : w.X2};
  for (int32_t k = 0; k < max_iter; ++k) {
    void *src = buf[k & 1], *dst = buf[(k + 1) & 1];
    void *Wb = o3 ? dst : w.Y;
    UArgs a{cols, col_off, P->dim, P->dim_pad, w.tile_ptr, w.tiles, n_cols, tol > 0.0 ? 1 : 0, src, Wb, Wb, s, w.err, 0, nullptr, 0, nullptr, umma_dbg(), 0, 0, 0,
            o3 ? -0.75f : -0.5f, 1.f};
    // "128-lower" storage (staged epilogue only): Wh is always written and read that way; X is read that way from the
    // second step on (X0 from sm_gather is a full image, a superset) and written that way except by the last update
    // of a submatrix (fixed counts: the last step; convergence mode: per submatrix, s.last)
    const int32_t lt = (sym == 2 && !o3 && opt(OPT_UMMA_LT) != 0) ? 1 : 0;
    a.lt_in = lt && k > 0; a.lt_out = lt;
    a.fold = fold; a.share_a = share_a;
    int32_t launch = nper * k;                 // launches alternate their walk through the tile table (option umma.rev)
    a.rev = o3 ? (rev_on & launch) & 1 : 0;
    a.counter = dyn ? w.counters + launch : nullptr;
    const UMaps m1{maps[k & 1].a, maps[k & 1].b}, m2{maps[k & 1].a, maps[2].b};
    // precision schedule (f3): updates 0 .. switch_iter-1 run on bf16 operands, update switch_iter-1 rounds X' to fp16
    const bool bf16_k = bf16 && (switch_iter < 0 || k < switch_iter);
    int32_t rc = launch_umma_any<1>(bf16_k, mode, sym, nst, a, m1, n_sm, st);
    if (rc != SM_OK) return rc;
    if (tol > 0.0) {
      SM_CUDA(cudaMemsetAsync(w.n_still, 0, sizeof(int32_t), st));
      k_sign_post<<<(n_cols + 7) / 8, 256, 0, st>>>(n_cols, cols, P->dim, s, w.n_parts, tol, iters, residual);
      SM_LAUNCHED();
    } else if (k == max_iter - 1) {
      // fixed iteration count: nothing depends on the residual, so only the last step's is reduced (and iters set)
      k_fused_post<<<(n_cols + 7) / 8, 256, 0, st>>>(n_cols, cols, P->dim, P->dim_pad, res_pd, w.partial, w.parts_per_col, w.n_parts,
                                                     max_iter, iters, residual);
      SM_LAUNCHED();
    }
    if (o3) {
      ++launch;
      UArgs z = a;
      z.Xsrc = Wb; z.Ybuf = Wb; z.Out = w.X2; z.out_scale = 2.f / 3.f;
      z.rev = (rev_on & launch) & 1;
      z.counter = dyn ? w.counters + launch : nullptr;
      rc = launch_umma_any<2>(bf16_k, mode, sym, nst, z, m2, n_sm, st);
      if (rc != SM_OK) return rc;
      a.Ybuf = w.X2;
    }
    ++launch;
    a.Out = dst;
    a.lt_in = lt;              // PHASE 2 reads X (lower from step 1 on; X0 is full, which is a superset) and Wh (lower)
    a.lt_out = lt && k + 1 < max_iter;     // (convergence mode: an earlier last update is mirrored per submatrix, s.last)
    a.rev = o3 ? (rev_on & launch) & 1 : rev_on;   // PHASE 2 starts where PHASE 1 ended, the next PHASE 1 where this launch ends
    a.counter = dyn ? w.counters + launch : nullptr;
    a.out_f16 = (bf16_k && k + 1 == switch_iter) ? 1 : 0;
    rc = launch_umma_any<2>(bf16_k, mode, sym, nst, a, m2, n_sm, st);
    if (rc != SM_OK) return rc;
    if (tol > 0.0 && k >= 5 && (k & 1)) {
      int32_t still = 1;
      SM_CUDA(cudaMemcpyAsync(&still, w.n_still, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
      SM_CUDA(cudaStreamSynchronize(st));
      if (still == 0) break;
    }
  }
  dim3 cg(n_cols, 8);
  k_copy_back<<<cg, 256, 0, st>>>(cols, col_off, iters, 2, P->dim_pad, res_pd, (const char *)buf[1], (char *)X);
  SM_LAUNCHED();
  return SM_OK;
}

// O_c = A_c B_c for every listed submatrix, 16-bit images, true products on every tile (nothing assumed symmetric):
// the non-symmetric update kernel (A K-major, B MN-major from its image) with the identity MMAs switched off.
// ws: a sign workspace of the same call shape (sm_sign_ws_bytes_ex with SM_SIGN_NONSYMMETRIC); only its tile table and
// flags are used.  Used by sm_density_nonorth (f2, Eq. 14: S^-1 = Z Z, S^-1 T_H, 1/2 (I - sign) S^-1).
int32_t umma_product(const sm_pattern_t *P, const int32_t *cols, int32_t n_cols, const int64_t *col_off,
                     int64_t packed_elems, int32_t x_dtype, const void *A, const void *B, void *O, void *ws,
                     int64_t ws_bytes, cudaStream_t st) {
  if ((P->pad_to % 64) != 0) return SM_ERR_ARG;
  const int32_t sym = 0, ncta = 1, R = UM;
  UmmaWs w = umma_layout(ws, ws_bytes, P, n_cols, packed_elems, sym, true);
  if (w.used > ws_bytes) return SM_ERR_SPACE;
  int dev = 0, n_sm = 0;
  SM_CUDA(cudaGetDevice(&dev));
  SM_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
  w.err = device_err_word();
  const int32_t nb = (n_cols + 255) / 256;
  SignState s{w.active, w.last, w.n_still, w.partial, w.parts_per_col};
  k_sign_init_grouped<<<nb, 256, 0, st>>>(n_cols, cols, P->dim_pad, 0, w.active, w.last, nullptr, nullptr);
  SM_LAUNCHED();
  k_umma_tilecounts<<<nb, 256, 0, st>>>(n_cols, R, sym, 0, EPI_WARPS * ncta, 0, cols, P->dim, P->dim_pad, w.tile_ptr, w.n_parts);
  SM_LAUNCHED();
  { int32_t rc = exclusive_scan_i64(n_cols, w.tile_ptr, w.tile_ptr, st); if (rc != SM_OK) return rc; }
  k_umma_build_tiles<<<nb, 256, 0, st>>>(n_cols, R, sym, 0, 0, 0, cols, P->dim, P->dim_pad, col_off, w.tile_ptr, w.tiles);
  SM_LAUNCHED();
  SM_CUDA(cudaMemsetAsync(O, 0, packed_elems * 2, st));       // padding of the result reads as zeros
  UArgs a{cols, col_off, P->dim, P->dim_pad, w.tile_ptr, w.tiles, n_cols, 0, A, B, O, s, w.err, 0, nullptr, 0, nullptr, 0, 0, 0, 0,
          -0.5f, 1.f, 1};
  UMaps maps{};
  return launch_umma_any<2>(x_dtype == SM_BF16, 1, sym, opt(OPT_UMMA_STAGES) ? opt(OPT_UMMA_STAGES) : 4, a, maps, n_sm, st);
}

}  // namespace sm
