// a2 gather, a4 scatter (+ symmetrise), a5 density/trace: the HBM-bound ends of the path.
// PAPER.md:110 (Fig. 2 steps 1 and 3), PAPER.md:91 (Eq. 14 with S = I).
#include "common.cuh"

namespace sm {

// ---- spectral scale --------------------------------------------------------------------------
// rowbase[i] = sum_{i'<i} |N(i')| * b_i'  (offset of block row i's abs-row-sums).
__global__ void k_rowbase_in(int32_t n, const int32_t *__restrict__ blk, const int32_t *__restrict__ rp,
                             int64_t *__restrict__ out) {
  int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = (int64_t)(rp[i + 1] - rp[i]) * blk[i];
}

// babs[rowbase[i] + (p - rp[i]) * b_i + r] = sum_s |(A - mu I)_p[r, s]| for every stored block p.
template <typename TA>
__global__ void k_block_abs_rowsum(const int32_t *__restrict__ blk, const int32_t *__restrict__ rp,
                                   const int32_t *__restrict__ ci, const int64_t *__restrict__ vp,
                                   const TA *__restrict__ vals, double mu,
                                   const int64_t *__restrict__ rowbase, double *__restrict__ babs) {
  int32_t i = blockIdx.x;
  int32_t bi = blk[i], lo = rp[i], cnt = rp[i + 1] - lo;
  for (int32_t e = threadIdx.x; e < cnt * bi; e += blockDim.x) {
    int32_t q = e / bi, r = e - q * bi;
    int32_t p = lo + q, j = ci[p], bj = blk[j];
    const TA *row = vals + vp[p] + (int64_t)r * bj;
    double s = 0.0;
    for (int32_t c = 0; c < bj; ++c) {
      double v = to_double<TA>(row[c]);
      if (j == i && c == r) v -= mu;
      s += fabs(v);
    }
    babs[rowbase[i] + e] = s;
  }
}

// Gershgorin: scale[c] = max over rows of T_i - mu I of the absolute row sum.  One CTA per column.
__global__ void k_scale_gershgorin(const int32_t *__restrict__ cols, const int32_t *__restrict__ blk,
                                   const int32_t *__restrict__ rp, const int32_t *__restrict__ ci,
                                   const int64_t *__restrict__ gmap_ptr, const int32_t *__restrict__ gmap,
                                   const int64_t *__restrict__ rowbase, const double *__restrict__ babs,
                                   double *__restrict__ scale) {
  int32_t c = blockIdx.x;
  int32_t i = cols ? cols[c] : c;
  int32_t lo = rp[i], cnt = rp[i + 1] - lo;
  const int32_t *g = gmap + gmap_ptr[i];
  double best = 0.0;
  // rows are enumerated as (neighbour a, local row r); neighbour a is block row ja = ci[lo + a].  A warp takes
  // every (blockDim / 32)-th neighbour and a lane one of its rows (the maximum does not depend on the order).
  // Small blocks: a warp is cut into groups of rps = 2^k >= (this column's own block size) lanes that each take a neighbour,
  // so 6-wide blocks keep 24 of 32 lanes busy instead of 6 (configs[3]: 0.24 ms per call).  Same sums, same maximum.
  const int32_t lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
  int32_t rps = 32;
  while (rps >= 2 * blk[i] && rps > 1) rps >>= 1;
  const int32_t slots = 32 / rps, slot = lane / rps, row = lane - slot * rps;
  for (int32_t a = wid * slots + slot; a < cnt; a += nw * slots) {
    int32_t ja = ci[lo + a], ba = blk[ja], rlo = rp[ja];
    for (int32_t r = row; r < ba; r += rps) {
      double s = 0.0;
      for (int32_t cc = 0; cc < cnt; ++cc) {
        int32_t p = g[a * cnt + cc];
        if (p >= 0) s += babs[rowbase[ja] + (int64_t)(p - rlo) * ba + r];
      }
      best = fmax(best, s);
    }
  }
  __shared__ double red[32];
  for (int d = 16; d > 0; d >>= 1) best = fmax(best, __shfl_xor_sync(0xffffffffu, best, d));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x == 0) {
    double m = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) m = fmax(m, red[w]);
    scale[c] = m > 0.0 ? m : 1.0;
  }
}

__global__ void k_fill_double(int32_t n, double v, double *__restrict__ out) {
  int32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = v;
}

// ---- gather ------------------------------------------------------------------------------------
// grid = (listed column, band of GATHER_ROWS rows), 256 threads.  A work item is one 16-byte-aligned
// run of 8 output elements (r, c0..c0+7); items are ordered so that the 8 lanes of a row cover one
// 64-column chunk, i.e. a warp writes four full 128-byte lines of the image (or 4 contiguous row
// segments of the row-major layout).  Dynamic smem: int32 off[cnt+1+GATHER_OFF_PAD]
// (block starts, then m, then the ends of the pseudo blocks behind the last neighbour), uint16 blkof[Pd].
constexpr int GATHER_ROWS = 64;

struct GatherArgs {
  const int32_t *cols; const int64_t *col_off;
  const int32_t *rp; const int64_t *vp; const int32_t *row_off;
  const int64_t *gmap_ptr; const int32_t *gmap;
  const int32_t *dim, *dim_pad;
  const double *scale; double mu;
  int32_t lean;        // 16-bit images, every block of N(i) >= 8 wide: the table-driven walk (k_gather, "lean" branch)
};

// One 8-run through the branch-free walk: the run spans at most NB neighbour blocks (the CTA checked the
// narrowest block of N(i)), so the NB candidate sources are set up once and every element picks its
// source by compares against the block ends -- no divergent block switch, no per-element bounds test
// (columns >= m fall into the pseudo block `cnt`, whose source is null).
template <typename TA, typename TX, int NB>
__device__ __forceinline__ void gather_run(const GatherArgs &g, const TA *__restrict__ vals, const int32_t *off,
                                           const uint16_t *blkof, const int32_t *gm, int32_t cnt, int32_t r,
                                           int32_t c0, float inv_sf, float muf, double inv_s, TX *v) {
  constexpr bool LOWP = sizeof(TX) == 2;
  const int32_t a = blkof[r], ra = r - off[a];
  const int32_t *gm_row = gm + (int64_t)a * cnt;
  const int32_t b = blkof[c0];
  const TA *src[NB];
  int32_t end[NB];
#pragma unroll
  for (int s = 0; s < NB; ++s) {
    const int32_t bb = b + s;
    const bool in = bb < cnt;
    const int32_t bs = off[bb], be = off[bb + 1];        // off[] is padded behind cnt (k_gather)
    const int32_t p = in ? __ldg(gm_row + bb) : -1;
    // element c of the run lives at src[s][c]: row ra of the stored block, shifted by the block's first column
    src[s] = p >= 0 ? vals + __ldg(g.vp + p) + (int64_t)ra * (be - bs) - bs : nullptr;
    end[s] = be;
  }
  bool any = false;
#pragma unroll
  for (int s = 0; s < NB; ++s) any |= src[s] != nullptr;
  if (!any) {                                             // no stored block under the run (about half of all runs)
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = from_double<TX>(0.0);
    return;
  }
  const int32_t kd = r - c0;                              // position of the diagonal inside the run, if 0..7
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const int32_t c = c0 + k;
    const TA *sp = src[0];
#pragma unroll
    for (int s = 1; s < NB; ++s) sp = c >= end[s - 1] ? src[s] : sp;
    if (LOWP) {
      float x = sp ? (float)__ldg(sp + c) : 0.f;
      if (k == kd) x -= muf;
      v[k] = from_float<TX>(x * inv_sf);
    } else {
      double x = sp ? to_double<TA>(__ldg(sp + c)) : 0.0;
      if (k == kd) x -= g.mu;
      v[k] = from_double<TX>(x * inv_s);
    }
  }
}

// The general walk (blocks narrower than 3 columns): one block switch per column at most.
template <typename TA, typename TX>
__device__ __forceinline__ void gather_run_any(const GatherArgs &g, const TA *__restrict__ vals, const int32_t *off,
                                               const uint16_t *blkof, const int32_t *gm, int32_t cnt, int32_t m,
                                               int32_t r, int32_t c0, float inv_sf, float muf, double inv_s, TX *v) {
  constexpr bool LOWP = sizeof(TX) == 2;
  const int32_t a = blkof[r], ra = r - off[a];
  const int32_t *gm_row = gm + (int64_t)a * cnt;
  int32_t b = blkof[c0], bs = off[b], be = off[b + 1];
  int32_t p = __ldg(gm_row + b);
  const TA *src = p >= 0 ? vals + __ldg(g.vp + p) + (int64_t)ra * (be - bs) : nullptr;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const int32_t c = c0 + k;
    if (c < m) {
      while (c >= be) {                                   // next neighbour block (blocks are >= 1 wide)
        ++b; bs = be; be = off[b + 1];
        p = __ldg(gm_row + b);
        src = p >= 0 ? vals + __ldg(g.vp + p) + (int64_t)ra * (be - bs) : nullptr;
      }
      if (LOWP) {
        float x = src ? (float)__ldg(src + (c - bs)) : 0.f;
        if (r == c) x -= muf;
        v[k] = from_float<TX>(x * inv_sf);
      } else {
        double x = src ? to_double<TA>(__ldg(src + (c - bs))) : 0.0;
        if (r == c) x -= g.mu;
        v[k] = from_double<TX>(x * inv_s);
      }
    } else {
      v[k] = from_double<TX>(0.0);
    }
  }
}

// Item loop of the table-driven walk of k_gather (16-bit images).  THREE: blocks narrower than 8 columns -- a run may reach
// into a third neighbour block (CTA-uniform; compiled separately so that the two-block case carries no third pointer).
template <typename TA, typename TX, bool THREE>
__device__ __forceinline__ void gather_lean_items(const TA *__restrict__ vals, TX *__restrict__ Xs, const uint4 *gran,
                                                  const uint32_t *rowinfo, const int64_t *tab, int32_t Pd, int32_t m,
                                                  int32_t r0, int32_t rows, int32_t items, float inv_sf, float muf) {
  for (int32_t e = threadIdx.x; e < items; e += blockDim.x) {
    const int32_t j = e & 7;
    const int32_t rr = rows == GATHER_ROWS ? ((e >> 3) & (GATHER_ROWS - 1)) : (e >> 3) % rows;
    const int32_t cb = rows == GATHER_ROWS ? (e >> 3) / GATHER_ROWS : (e >> 3) / rows;
    const int32_t r = r0 + rr, c0 = (cb << 6) + (j << 3);
    if (c0 >= Pd) continue;
    float x[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) x[k] = 0.f;
    if (r < m && c0 < m) {
      const uint4 q = gran[c0 >> 3];
      const uint32_t ri = rowinfo[rr];
      const int64_t *trow = tab + (ri >> 16) + (q.x & 0xffffu);
      const int64_t e0 = trow[0], e1 = trow[1], e2 = THREE ? trow[2] : (int64_t)-1;
      const int32_t ra = (int32_t)(ri & 0xffffu), s1 = (int32_t)(q.y & 0xffu), s12 = (int32_t)(q.y >> 8);
      if ((e0 & e1 & e2) >= 0) {                             // at least one of the blocks under the run is stored
        const TA *p0 = vals + e0 + ra * (int32_t)(q.w & 0xffffu) + (int32_t)q.z;
        const TA *p1 = vals + e1 + ra * (int32_t)(q.w >> 16) - s1;
        const TA *p2 = vals + e2 + ra * (int32_t)(q.x >> 16) - s12;
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          if constexpr (THREE) {                                 // (measured: a load site per segment is faster here,
            if (k < s1) { if (e0 >= 0) x[k] = (float)__ldg(p0 + k); }        //  one load site behind a pointer select below)
            else if (k < s12) { if (e1 >= 0) x[k] = (float)__ldg(p1 + k); }
            else if (e2 >= 0) x[k] = (float)__ldg(p2 + k);
          } else {
            const bool first = k < s1;
            if (first ? e0 >= 0 : e1 >= 0) x[k] = (float)__ldg((first ? p0 : p1) + k);
          }
        }
        const int32_t kd = r - c0;
        if ((uint32_t)kd < 8u) {
#pragma unroll
          for (int k = 0; k < 8; ++k)
            if (k == kd) x[k] -= muf;
        }
      }
    }
    __align__(16) TX v[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) v[k] = from_float<TX>(x[k] * inv_sf);
    *reinterpret_cast<uint4 *>(Xs + img_off(Pd, r, c0)) = *reinterpret_cast<const uint4 *>(v);
  }
}

constexpr int GATHER_OFF_PAD = 4;   // off[cnt+1 .. cnt+GATHER_OFF_PAD]: ends of the pseudo blocks behind the last one

template <typename TA, typename TX, bool IMG>
__global__ void __launch_bounds__(256) k_gather(GatherArgs g, const TA *__restrict__ vals, TX *__restrict__ X) {
  extern __shared__ int32_t smem_i[];
  __shared__ int32_t s_minb;
  const int32_t c_list = blockIdx.x;
  const int32_t i = g.cols ? g.cols[c_list] : c_list;
  const int32_t Pd = g.dim_pad[i], m = g.dim[i];
  const int32_t r0 = blockIdx.y * GATHER_ROWS;
  if (r0 >= Pd) return;
  const int32_t lo = g.rp[i], cnt = g.rp[i + 1] - lo;
  int32_t *off = smem_i;
  uint16_t *blkof = (uint16_t *)(smem_i + cnt + 1 + GATHER_OFF_PAD);
  if (threadIdx.x == 0) s_minb = 0x7fffffff;
  for (int32_t a = threadIdx.x; a < cnt; a += blockDim.x) off[a] = g.row_off[lo + a];
  if (threadIdx.x <= GATHER_OFF_PAD) off[cnt + threadIdx.x] = threadIdx.x == 0 ? m : 0x3fffffff;
  __syncthreads();
  int32_t minb = 0x7fffffff;
  for (int32_t a = threadIdx.x; a < cnt; a += blockDim.x) {
    minb = min(minb, off[a + 1] - off[a]);
    for (int32_t r = off[a]; r < off[a + 1]; ++r) blkof[r] = (uint16_t)a;
  }
  for (int32_t r = m + threadIdx.x; r < Pd; r += blockDim.x) blkof[r] = (uint16_t)cnt;   // padding: pseudo block
  if (minb != 0x7fffffff) atomicMin(&s_minb, minb);
  __syncthreads();
  // an 8-run that starts on the last column of a block covers 1 + 7 more columns: 2 blocks if every block is
  // >= 7 wide, 3 if >= 4, 4 if >= 3 (CTA-uniform choice)
  const int32_t nb = s_minb >= 7 ? 2 : s_minb >= 4 ? 3 : s_minb >= 3 ? 4 : 0;
  const int32_t *gm = g.gmap + g.gmap_ptr[i];
  const double inv_s = 1.0 / g.scale[c_list];
  TX *Xs = X + g.col_off[c_list];
  const int32_t rows = min(GATHER_ROWS, Pd - r0);
  const int32_t n_cb = (Pd + 63) >> 6;                 // 64-column chunks (last may be partial: Pd % 16 == 0)
  const int32_t items = n_cb * rows * 8;
  const float inv_sf = (float)inv_s, muf = (float)g.mu; // 16-bit outputs: fp32 arithmetic is 2^-15 below their rounding
  if constexpr (IMG && sizeof(TX) == 2) {
    if (g.lean && s_minb >= 4 && r0 < m) {
      // ---- table-driven walk (blocks >= 4 wide: an 8-run touches at most three neighbour blocks, two if they are >= 8
      // wide).  Everything that
      // depends only on the run's column (first block, elements taken from it, offset inside it, the two block
      // widths) or only on the band's block rows (where block (a, b) is stored, or that it is absent) is resolved
      // ONCE per CTA into shared-memory tables; an item then costs two table reads, two address computations and
      // eight predicated loads.  The branch-free walk below re-derives all of it per run: 277 instructions per run
      // (ncu), 0.29 of the HBM peak.  Same arithmetic, same rounding: bit-identical images.
      // (Measured and dropped: a column-per-lane walk -- coalesced 4-byte loads, 2-byte stores of 64 contiguous bytes per
      // warp -- is 1.5x SLOWER than the run-per-lane walks: 16-byte stores per lane are what keeps this kernel moving.)
      uint8_t *dyn = reinterpret_cast<uint8_t *>(blkof + Pd + 2);
      dyn += (16 - ((uintptr_t)dyn & 15)) & 15;
      // [Pd / 8] per run: {b0 | bw2 << 16, s1 | s12 << 8, o0, bw0 | bw1 << 16}: first block, its elements in the run (s1),
      // end of the second block's elements (s12), offset of c0 inside b0, widths of b0, b0 + 1, b0 + 2
      uint4 *gran = reinterpret_cast<uint4 *>(dyn);
      uint32_t *rowinfo = reinterpret_cast<uint32_t *>(gran + (Pd >> 3));  // [GATHER_ROWS]  table row offset << 16 | row inside its block
      int64_t *tab = reinterpret_cast<int64_t *>(rowinfo + GATHER_ROWS);   // [na][cnt + 2]  element offset of block (a, b), -1: absent
      const int32_t r_last = min(r0 + rows, m) - 1;
      const int32_t a_first = blkof[r0], na = blkof[r_last] - a_first + 1, tw = cnt + 2;
      for (int32_t gi = threadIdx.x; gi < (Pd >> 3); gi += blockDim.x) {
        const int32_t c0 = gi << 3;
        uint4 q = make_uint4(0u, 0u, 0u, 0u);
        if (c0 < m) {
          const int32_t b0 = blkof[c0], bs = off[b0], be = off[b0 + 1];
          const int32_t bw1 = b0 + 1 < cnt ? off[b0 + 2] - be : 0, bw2 = b0 + 2 < cnt ? off[b0 + 3] - off[b0 + 2] : 0;
          const int32_t s1 = min(8, be - c0), s12 = min(8, s1 + (b0 + 1 < cnt ? bw1 : 8));
          q = make_uint4((uint32_t)b0 | ((uint32_t)bw2 << 16), (uint32_t)s1 | ((uint32_t)s12 << 8), (uint32_t)(c0 - bs),
                         (uint32_t)(be - bs) | ((uint32_t)bw1 << 16));
        }
        gran[gi] = q;
      }
      for (int32_t rl = threadIdx.x; rl < rows; rl += blockDim.x) {
        const int32_t r = r0 + rl;
        const int32_t a = r < m ? blkof[r] : a_first;
        rowinfo[rl] = ((uint32_t)((a - a_first) * tw) << 16) | (uint32_t)(r < m ? r - off[a] : 0);
      }
      for (int32_t t = threadIdx.x; t < na * tw; t += blockDim.x) {
        const int32_t al = t / tw, b = t - al * tw;
        const int32_t p = b < cnt ? __ldg(gm + (int64_t)(a_first + al) * cnt + b) : -1;
        tab[t] = p >= 0 ? __ldg(g.vp + p) : (int64_t)-1;
      }
      __syncthreads();
      if (s_minb >= 8) gather_lean_items<TA, TX, false>(vals, Xs, gran, rowinfo, tab, Pd, m, r0, rows, items, inv_sf, muf);
      else gather_lean_items<TA, TX, true>(vals, Xs, gran, rowinfo, tab, Pd, m, r0, rows, items, inv_sf, muf);
      return;
    }
  }
  for (int32_t e = threadIdx.x; e < items; e += blockDim.x) {
    const int32_t j = e & 7;
    const int32_t rr = rows == GATHER_ROWS ? ((e >> 3) & (GATHER_ROWS - 1)) : (e >> 3) % rows;
    const int32_t cb = rows == GATHER_ROWS ? (e >> 3) / GATHER_ROWS : (e >> 3) / rows;
    const int32_t r = r0 + rr, c0 = (cb << 6) + (j << 3);
    if (c0 >= Pd) continue;
    __align__(16) TX v[8];
    if (r >= m || c0 >= m) {
#pragma unroll
      for (int k = 0; k < 8; ++k) v[k] = from_double<TX>(0.0);
    } else if (nb == 2) {
      gather_run<TA, TX, 2>(g, vals, off, blkof, gm, cnt, r, c0, inv_sf, muf, inv_s, v);
    } else if (nb == 3) {
      gather_run<TA, TX, 3>(g, vals, off, blkof, gm, cnt, r, c0, inv_sf, muf, inv_s, v);
    } else if (nb == 4) {
      gather_run<TA, TX, 4>(g, vals, off, blkof, gm, cnt, r, c0, inv_sf, muf, inv_s, v);
    } else {
      gather_run_any<TA, TX>(g, vals, off, blkof, gm, cnt, m, r, c0, inv_sf, muf, inv_s, v);
    }
    TX *dst = IMG ? Xs + img_off(Pd, r, c0) : Xs + (int64_t)r * Pd + c0;
    if (IMG || c0 + 8 <= Pd) {
#pragma unroll
      for (int q = 0; q < (int)(sizeof(TX) * 8 / 16); ++q)
        reinterpret_cast<uint4 *>(dst)[q] = reinterpret_cast<const uint4 *>(v)[q];
    } else {                                             // row tail when pad_to % 8 != 0 (row-major only)
      for (int k = 0; c0 + k < Pd; ++k) dst[k] = v[k];
    }
  }
}

// ---- gather, 16-bit images: staged through shared memory, written by bulk TMA stores --------------------------------
// grid = (listed column, band of 64 rows), 256 threads.  The band is produced tile by tile (64 rows x 256 columns =
// four 64-column chunks of the image = 32 KB, two buffers): a tile is zero-filled, then every STORED block pair
// (neighbour a of the band's rows, neighbour cb of the tile's columns) is copied by one warp, source-driven: the lanes
// walk the row-major source block with consecutive addresses (coalesced loads, no per-element search for "which block
// holds this column") and write the shifted / scaled / rounded elements to their swizzled places in the tile, which
// has the layout of the image.  Absent pairs and padding stay zero.  A finished tile leaves as up to four bulk stores
// of 64 rows x 128 B.  Against the element-wise kernel (k_gather: every 8-run resolves its candidate blocks, 33 thread
// instructions per output element, issue-bound at 0.29 of the HBM peak) the work per output
// element is ~1/4.  Arithmetic and rounding are those of k_gather (fp32, one rounding): the images are bit-identical.
constexpr int GS_ROWS = 64, GS_TILE_CHUNKS = 4, GS_TILE_BYTES = GS_TILE_CHUNKS * GS_ROWS * 128;
constexpr int GS_MAX_PAIRS = 512;

template <typename TA, typename TX>
__global__ void __launch_bounds__(256) k_gather_staged(GatherArgs g, const TA *__restrict__ vals, TX *__restrict__ X) {
  extern __shared__ __align__(1024) uint8_t gs_smem[];
  const int32_t c_list = blockIdx.x;
  const int32_t i = g.cols ? g.cols[c_list] : c_list;
  const int32_t Pd = g.dim_pad[i], m = g.dim[i];
  const int32_t r0 = blockIdx.y * GS_ROWS;
  if (r0 >= Pd) return;
  const uint32_t raw = (uint32_t)__cvta_generic_to_shared(gs_smem);
  const uint32_t base = (raw + 1023u) & ~1023u;
  uint8_t *const tile0 = gs_smem + (base - raw);
  int64_t *const pair_src = reinterpret_cast<int64_t *>(tile0 + 2 * GS_TILE_BYTES);          // [GS_MAX_PAIRS]
  uint16_t *const rowblk = reinterpret_cast<uint16_t *>(tile0 + 2 * GS_TILE_BYTES + GS_MAX_PAIRS * 8);    // [GS_ROWS]
  int32_t *const off = reinterpret_cast<int32_t *>(tile0 + 2 * GS_TILE_BYTES + GS_MAX_PAIRS * 8 + GS_ROWS * 2);
  const int32_t lo = g.rp[i], cnt = g.rp[i + 1] - lo;
  for (int32_t a = threadIdx.x; a < cnt; a += blockDim.x) off[a] = g.row_off[lo + a];
  if (threadIdx.x == 0) off[cnt] = m;
  __syncthreads();
  const int32_t rows = min(GS_ROWS, Pd - r0), r1 = min(r0 + rows, m);      // true rows of the band: [r0, r1)
  // neighbours whose rows meet the band: [a_lo, a_hi)
  int32_t a_lo = 0, a_hi = 0;
  if (r1 > r0) {
    int32_t l = 0, h = cnt;                       // last a with off[a] <= r0
    while (h - l > 1) { const int32_t mid = (l + h) >> 1; if (off[mid] <= r0) l = mid; else h = mid; }
    a_lo = l;
    l = a_lo; h = cnt;                            // last a with off[a] < r1
    while (h - l > 1) { const int32_t mid = (l + h) >> 1; if (off[mid] < r1) l = mid; else h = mid; }
    a_hi = l + 1;
  }
  // neighbour block of every true row of the band
  for (int32_t a = a_lo + threadIdx.x; a < a_hi; a += blockDim.x)
    for (int32_t r = max(off[a], r0); r < min(off[a + 1], r1); ++r) rowblk[r - r0] = (uint16_t)a;
  __syncthreads();
  const int32_t *gm = g.gmap + g.gmap_ptr[i];
  const float inv_sf = (float)(1.0 / g.scale[c_list]), muf = (float)g.mu;
  char *Xs = (char *)(X + g.col_off[c_list]);
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int32_t n_chunks = Pd >> 6;
  int32_t cb_lo = 0;                               // first neighbour that may meet the current tile's columns
  for (int32_t t0 = 0, tb = 0; t0 < n_chunks; t0 += GS_TILE_CHUNKS, tb ^= 1) {
    uint8_t *const tile = tile0 + tb * GS_TILE_BYTES;
    const int32_t nch = min(GS_TILE_CHUNKS, n_chunks - t0);
    const int32_t c_beg = t0 * 64, c_end = min((t0 + nch) * 64, m);         // true columns of the tile: [c_beg, c_end)
    // the bulk stores issued from this buffer two tiles ago have read it (one group may stay in flight)
    if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
    __syncthreads();
    for (int32_t e = threadIdx.x; e < nch * GS_ROWS * 8; e += blockDim.x) reinterpret_cast<uint4 *>(tile)[e] = make_uint4(0, 0, 0, 0);
    __syncthreads();
    if (c_end > c_beg && a_hi > a_lo) {
      while (cb_lo + 1 < cnt && off[cb_lo + 1] <= c_beg) ++cb_lo;
      int32_t cb_hi = cb_lo;
      while (cb_hi < cnt && off[cb_hi] < c_end) ++cb_hi;
      const int32_t n_c = cb_hi - cb_lo, n_a = a_hi - a_lo, nrows = r1 - r0;
      // column blocks in chunks whose (row block, column block) pairs fit the table; the pairs are resolved in parallel
      // first (gather-map entry -> value offset: two dependent loads per pair), then every thread takes items
      // (row of the band, column block): it walks the row of the stored block (consecutive source addresses; the
      // lanes of a warp are consecutive rows of the same block, i.e. one contiguous piece of memory) and writes the
      // elements to their swizzled places in the tile
      const int32_t cbc = max(1, GS_MAX_PAIRS / n_a);
      for (int32_t c0 = 0; c0 < n_c; c0 += cbc) {
        const int32_t nc_here = min(cbc, n_c - c0);
        __syncthreads();
        for (int32_t q = threadIdx.x; q < n_a * nc_here; q += blockDim.x) {
          const int32_t a = a_lo + q / nc_here, cb = cb_lo + c0 + q % nc_here;
          const int32_t p = __ldg(gm + (int64_t)a * cnt + cb);
          pair_src[q] = p >= 0 ? __ldg(g.vp + p) : -1;
        }
        __syncthreads();
        for (int32_t it = threadIdx.x; it < nrows * nc_here; it += blockDim.x) {
          const int32_t cbi = it / nrows, rl = it - cbi * nrows;
          const int32_t r = r0 + rl, a = rowblk[rl], cb = cb_lo + c0 + cbi;
          const int64_t so = pair_src[(a - a_lo) * nc_here + cbi];
          if (so < 0) continue;                                            // absent pair: stays zero
          const int32_t rc0 = off[cb], bc = off[cb + 1] - rc0;
          const TA *src = vals + so + (int64_t)(r - off[a]) * bc;
          const int32_t rc_lo = max(0, c_beg - rc0), rc_hi = min(bc, c_end - rc0);
          uint8_t *const trow = tile + (uint32_t)rl * 128u;
          const uint32_t r7 = (uint32_t)r & 7u;
#pragma unroll 4
          for (int32_t rc = rc_lo; rc < rc_hi; ++rc) {
            const int32_t c = rc0 + rc;
            float x = (float)__ldg(src + rc);
            if (r == c) x -= muf;
            const uint32_t o = (uint32_t)((c - c_beg) >> 6) * (GS_ROWS * 128u) + (((((uint32_t)c & 63u) >> 3) ^ r7) << 4) +
                               ((uint32_t)c & 7u) * 2u;
            *reinterpret_cast<TX *>(trow + o) = from_float<TX>(x * inv_sf);
          }
        }
      }
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    __syncthreads();
    if (threadIdx.x == 0) {
      for (int32_t k = 0; k < nch; ++k)
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(Xs + ((int64_t)(t0 + k) * Pd + r0) * 128),
                     "r"(base + (uint32_t)(tb * GS_TILE_BYTES + k * GS_ROWS * 128)), "r"((uint32_t)rows * 128u)
                     : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
  }
  if (threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
}

// ---- scatter -----------------------------------------------------------------------------------
// One CTA per listed column i.  Reads the owned ROWS of S_i (S_i symmetric): element
// S_i[own_off + s, r] goes to block (N(i)[a], i) at [r - off[a], s].  The output dominates the bytes
// (nnzb b^2 e_R against sum m b e_x), so the kernel is organised around its stores: a strip of rows r
// is staged in shared memory as stage[(r - r_lo) * b_i + s] -- which IS the order of the output, the
// blocks (N(i)[a], i) being row-major [r - off[a]][s] -- and streamed out with consecutive threads on
// consecutive output elements (a warp writes 32 contiguous elements of one block, except where it
// crosses into the next neighbour's block).  The loads are 16-byte runs along the owned rows.
// Dynamic smem: int32 off[cnt+1], uint16 blkof[m] (4-byte aligned end), TX stage[SCATTER_STAGE_BYTES / sizeof(TX)].
constexpr int SCATTER_STAGE_BYTES = 48 * 1024;

template <typename TX, typename TR, bool IMG>
__global__ void __launch_bounds__(256) k_scatter(const int32_t *__restrict__ cols, const int64_t *__restrict__ col_off,
                          const int32_t *__restrict__ blk, const int32_t *__restrict__ rp,
                          const int32_t *__restrict__ ci, const int64_t *__restrict__ vp,
                          const int32_t *__restrict__ own_pos, const int32_t *__restrict__ dim,
                          const int32_t *__restrict__ dim_pad, const int32_t *__restrict__ tmap,
                          const int32_t *__restrict__ row_off, int32_t stage_off_bytes,
                          const TX *__restrict__ S, TR *__restrict__ R) {
  extern __shared__ int32_t smem_i[];
  constexpr int VEC = 16 / (int)sizeof(TX);
  constexpr int STAGE = SCATTER_STAGE_BYTES / (int)sizeof(TX);
  const int32_t c_list = blockIdx.x;
  const int32_t i = cols ? cols[c_list] : c_list;
  const int32_t Pd = dim_pad[i], m = dim[i];
  const int32_t lo = rp[i], cnt = rp[i + 1] - lo;
  int32_t *off = smem_i;
  uint16_t *blkof = (uint16_t *)(smem_i + cnt + 1);
  TX *stage = (TX *)((char *)smem_i + stage_off_bytes);
  for (int32_t a = threadIdx.x; a < cnt; a += blockDim.x) off[a] = row_off[lo + a];
  if (threadIdx.x == 0) off[cnt] = m;
  __syncthreads();
  for (int32_t a = threadIdx.x; a < cnt; a += blockDim.x)
    for (int32_t r = off[a]; r < off[a + 1]; ++r) blkof[r] = (uint16_t)a;
  const int32_t own = own_pos[i], own_off = off[own], bi = off[own + 1] - own_off;
  const TX *Ss = S + col_off[c_list];
  // rows per strip: a multiple of VEC so that every 16-byte run of the source lies inside one strip
  const int32_t W = (STAGE / bi) / VEC * VEC;
  if (W <= 0) {                                          // a block wider than the stage: element-wise fallback
    __syncthreads();
    for (int32_t e = threadIdx.x; e < bi * m; e += blockDim.x) {
      int32_t s = e / m, r = e - s * m;
      int32_t row = own_off + s;
      TX v = IMG ? Ss[img_off(Pd, row, r)] : Ss[(int64_t)row * Pd + r];
      int32_t a = blkof[r];
      R[vp[tmap[lo + a]] + (int64_t)(r - off[a]) * bi + s] = (TR)to_double<TX>(v);
    }
    return;
  }
  // 16-byte loads need the rows of this submatrix 16-byte aligned (always true for the image)
  const bool vec_ok = IMG || ((Pd % VEC) == 0 && (col_off[c_list] % VEC) == 0);
  const uint32_t magic = 0xffffffffu / (uint32_t)bi + 1u;  // idx / bi == umulhi(idx, magic) for idx * bi < 2^32
  for (int32_t r_lo = 0; r_lo < m; r_lo += W) {
    const int32_t w = min(W, m - r_lo);
    __syncthreads();                                      // blkof ready / previous strip drained
    if (vec_ok) {
      const int32_t groups = (w + VEC - 1) / VEC;         // a tail group may reach into the zero padding (r < Pd)
      for (int32_t e = threadIdx.x; e < groups * bi; e += blockDim.x) {
        const int32_t s = e / groups, gq = e - s * groups;
        const int32_t r = r_lo + gq * VEC, row = own_off + s;
        const TX *src = IMG ? Ss + img_off(Pd, row, r) : Ss + (int64_t)row * Pd + r;
        __align__(16) TX v[VEC];
        *reinterpret_cast<uint4 *>(v) = __ldg(reinterpret_cast<const uint4 *>(src));
#pragma unroll
        for (int k = 0; k < VEC; ++k)
          if (gq * VEC + k < w) stage[(gq * VEC + k) * bi + s] = v[k];
      }
    } else {
      for (int32_t e = threadIdx.x; e < w * bi; e += blockDim.x) {
        const int32_t s = e / w, q = e - s * w;
        stage[q * bi + s] = Ss[(int64_t)(own_off + s) * Pd + r_lo + q];
      }
    }
    __syncthreads();
    for (int32_t e = threadIdx.x; e < w * bi; e += blockDim.x) {
      const int32_t q = bi == 1 ? e : (int32_t)__umulhi((uint32_t)e, magic);   // (2^32 / 1 does not fit the magic)
      const int32_t r = r_lo + q, a = blkof[r];
      // e - q*bi = s, so the target is block start + (r - off[a]) * bi + s = block start + e + (r_lo - off[a]) * bi
      R[__ldg(vp + __ldg(tmap + lo + a)) + (int64_t)(r_lo - off[a]) * bi + e] = (TR)to_double<TX>(stage[e]);
    }
  }
}

// D = 1/2 (I - 1/2 (R + R^T)) in place: the blockwise symmetrisation R <- 1/2 (R + R^T) (the lower-indexed partner of a
// pair (p, tmap[p]) owns both blocks) followed by k_density, in one pass over the values (same operations in the same
// order, so the bits equal sm_symmetrise followed by sm_density_from_sign).  One CTA per block row,
// one WARP per pair (p, q = tmap[p] >= p): both blocks are read into shared memory with consecutive lanes on
// consecutive elements, and both are written back the same way, the transposition happening in shared memory
// (every value is computed twice, once per target layout, from the same operands in the same order).  Pairs
// whose blocks exceed SYMD_CAP elements take the element-wise path.
constexpr int SYMD_WARPS = 4;
constexpr int SYMD_CAP = 576;   // 24 x 24: 4 warps x 2 blocks x 576 fp64 = 36 KB of static shared memory

// DENS = false: the symmetrisation alone (sm_symmetrise), R <- 1/2 (R + R^T), diagonal elements untouched.
template <typename TR, bool DENS>
__global__ void __launch_bounds__(32 * SYMD_WARPS)
k_symmetrise_density(const int32_t *__restrict__ blk, const int32_t *__restrict__ rp,
                     const int32_t *__restrict__ ci, const int64_t *__restrict__ vp,
                     const int32_t *__restrict__ tmap, TR *R) {
  __shared__ TR sbuf[SYMD_WARPS][2][SYMD_CAP];
  const int32_t i = blockIdx.x, bi = blk[i];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  TR *sa = sbuf[wid][0], *sb = sbuf[wid][1];
  for (int32_t p = rp[i] + wid; p < rp[i + 1]; p += SYMD_WARPS) {
    const int32_t q = tmap[p];
    if (q < p) continue;
    const int32_t bj = blk[ci[p]], ne = bi * bj;
    TR *Rp = R + vp[p], *Rq = R + vp[q];
    if (ne > SYMD_CAP) {
      for (int32_t e = lane; e < ne; e += 32) {
        int32_t r = e / bj, s = e - r * bj;
        if (p == q) {
          if (s < r) continue;
          if (s == r) { if (DENS) Rp[e] = (TR)0.5 * ((TR)1 - Rp[e]); continue; }
        }
        TR a = Rp[(int64_t)r * bj + s], b = Rq[(int64_t)s * bi + r];
        TR v = DENS ? (TR)0.5 * ((TR)0 - (TR)0.5 * (a + b)) : (TR)0.5 * (a + b);
        Rp[(int64_t)r * bj + s] = v;
        Rq[(int64_t)s * bi + r] = v;
      }
      continue;
    }
    __syncwarp();                                         // the previous pair's reads of sa / sb are done
    for (int32_t e = lane; e < ne; e += 32) { sa[e] = Rp[e]; sb[e] = Rq[e]; }
    __syncwarp();
    if (p == q) {                                         // diagonal block: a pair (r, s), (s, r) inside one block
      for (int32_t e = lane; e < ne; e += 32) {
        const int32_t r = e / bj, s = e - r * bj;
        TR v;
        if (s == r) v = DENS ? (TR)0.5 * ((TR)1 - sa[e]) : sa[e];
        else {
          const TR a = s > r ? sa[e] : sa[s * bj + r], b = s > r ? sa[s * bj + r] : sa[e];   // a = upper, b = lower
          v = DENS ? (TR)0.5 * ((TR)0 - (TR)0.5 * (a + b)) : (TR)0.5 * (a + b);
        }
        Rp[e] = v;
      }
    } else {
      for (int32_t e = lane; e < ne; e += 32) {           // block p = (i, j): element (r, s) pairs with q's (s, r)
        const int32_t r = e / bj, s = e - r * bj;
        const TR h = (TR)0.5 * (sa[e] + sb[s * bi + r]);
        Rp[e] = DENS ? (TR)0.5 * ((TR)0 - h) : h;
      }
      for (int32_t e = lane; e < ne; e += 32) {           // block q = (j, i): element (s, r), same operand order
        const int32_t s = e / bi, r = e - s * bi;
        const TR h = (TR)0.5 * (sa[r * bj + s] + sb[e]);
        Rq[e] = DENS ? (TR)0.5 * ((TR)0 - h) : h;
      }
    }
  }
}

// D = 1/2 (I - R) in place (Eq. 14, S = I).  One CTA per block row.
template <typename TR>
__global__ void k_density(const int32_t *__restrict__ blk, const int32_t *__restrict__ rp,
                          const int32_t *__restrict__ ci, const int64_t *__restrict__ vp, TR *RD) {
  int32_t i = blockIdx.x, bi = blk[i];
  for (int32_t p = rp[i]; p < rp[i + 1]; ++p) {
    int32_t j = ci[p], bj = blk[j];
    TR *B = RD + vp[p];
    for (int32_t e = threadIdx.x; e < bi * bj; e += blockDim.x) {
      int32_t r = e / bj, s = e - r * bj;
      TR id = (j == i && r == s) ? (TR)1 : (TR)0;
      B[e] = (TR)0.5 * (id - B[e]);
    }
  }
}

// Tr D: one CTA, fixed summation tree (deterministic).
template <typename TR>
__global__ void k_trace(int32_t n, const int32_t *__restrict__ blk, const int32_t *__restrict__ rp,
                        const int64_t *__restrict__ vp, const int32_t *__restrict__ own_pos,
                        const TR *__restrict__ D, double *__restrict__ trace) {
  __shared__ double red[1024];
  double acc = 0.0;
  for (int32_t i = threadIdx.x; i < n; i += blockDim.x) {
    int32_t b = blk[i];
    const TR *B = D + vp[rp[i] + own_pos[i]];
    double t = 0.0;
    for (int32_t r = 0; r < b; ++r) t += (double)B[(int64_t)r * b + r];
    acc += t;
  }
  red[threadIdx.x] = acc;
  __syncthreads();
  for (int d = blockDim.x >> 1; d > 0; d >>= 1) {
    if ((int)threadIdx.x < d) red[threadIdx.x] += red[threadIdx.x + d];
    __syncthreads();
  }
  if (threadIdx.x == 0) *trace = red[0];
}

}  // namespace sm

using namespace sm;


extern "C" int64_t sm_gather_ws_bytes(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t n_cols) {
  if (!A || !P) return SM_ERR_ARG;
  (void)n_cols;
  WsCursor cur(nullptr, 0);
  cur.take<int64_t>(A->n_blk + 1);
  cur.take<double>((int64_t)A->n_blk * P->max_dim);
  cur.take<double>(A->n_blk);
  return cur.used + 256 + global_scale_ws_bytes(A, P);
}

template <typename TA, typename TX, bool IMG>
static int32_t launch_gather(const GatherArgs &g, const void *vals, void *X, int32_t n_cols, int32_t max_pd,
                             int32_t max_nbr, int32_t max_dim, cudaStream_t st) {
  dim3 grid(n_cols, (max_pd + GATHER_ROWS - 1) / GATHER_ROWS);
  if constexpr (IMG) {
    if (opt(OPT_GATHER_TMA) != 0) {
      const int smem_s = 2 * GS_TILE_BYTES + 1024 + GS_MAX_PAIRS * 8 + GS_ROWS * 2 + (max_nbr + 1) * 4 + 16;
      SM_CUDA(cudaFuncSetAttribute(k_gather_staged<TA, TX>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_s));
      k_gather_staged<TA, TX><<<grid, 256, smem_s, st>>>(g, (const TA *)vals, (TX *)X);
      SM_LAUNCHED();
      return SM_OK;
    }
  }
  size_t smem = (size_t)(max_nbr + 1 + GATHER_OFF_PAD) * 4 + (size_t)(max_pd + 2) * 2;
  if constexpr (IMG)      // tables of the lean branch: run info, row info, block offsets of the band's <= GATHER_ROWS / 4 + 1 block rows
    smem += 16 + (size_t)(max_pd >> 3) * 16 + GATHER_ROWS * 4 + (size_t)(GATHER_ROWS / 4 + 2) * (max_nbr + 2) * 8;
  (void)max_dim;
  if (smem > 48 * 1024) SM_CUDA(cudaFuncSetAttribute(k_gather<TA, TX, IMG>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  k_gather<TA, TX, IMG><<<grid, 256, smem, st>>>(g, (const TA *)vals, (TX *)X);
  SM_LAUNCHED();
  return SM_OK;
}

extern "C" int32_t sm_gather(const sm_bcsr_t *A, const void *A_vals, int32_t a_dtype, const sm_pattern_t *P,
                             const int32_t *cols, int32_t n_cols, const int64_t *col_off, double mu,
                             int32_t scale_mode, int32_t x_dtype, void *X_packed, double *scale, void *ws,
                             int64_t ws_bytes, void *stream) {
  if (!A || !A_vals || !P || !X_packed || !scale || !ws || !col_off) return SM_ERR_ARG;
  if (!cols) n_cols = P->n_blk;
  if (n_cols <= 0) return SM_ERR_ARG;
  if (a_dtype != SM_F64 && a_dtype != SM_F32) return SM_ERR_UNSUPPORTED;
  if (dtype_bytes(x_dtype) == 0) return SM_ERR_UNSUPPORTED;
  if (is_16bit(x_dtype) && (P->pad_to % 64) != 0) return SM_ERR_ARG;
  if (scale_mode < SM_SCALE_NONE || scale_mode > SM_SCALE_GLOBAL) return SM_ERR_UNSUPPORTED;
  if (P->max_dim > 65535) return SM_ERR_UNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  int32_t n = A->n_blk;
  WsCursor cur(ws, ws_bytes);
  int64_t *rowbase = cur.take<int64_t>(n + 1);
  double *babs = cur.take<double>((int64_t)n * P->max_dim);
  double *ratio = cur.take<double>(n);
  if (!cur.ok()) return SM_ERR_SPACE;
  const int64_t g_off = align_up(cur.used, 256);        // SM_SCALE_GLOBAL: its own workspace behind these arrays

  if (scale_mode == SM_SCALE_NONE) {
    k_fill_double<<<(n_cols + 255) / 256, 256, 0, st>>>(n_cols, 1.0, scale);
    SM_LAUNCHED();
  } else {
    k_rowbase_in<<<(n + 127) / 128, 128, 0, st>>>(n, A->blk_size, A->row_ptr, rowbase);
    SM_LAUNCHED();
    { int32_t rc0 = exclusive_scan_i64(n, rowbase, rowbase, st); if (rc0 != SM_OK) return rc0; }
    if (a_dtype == SM_F64)
      k_block_abs_rowsum<double><<<n, 128, 0, st>>>(A->blk_size, A->row_ptr, A->col_idx, A->val_ptr,
                                                    (const double *)A_vals, mu, rowbase, babs);
    else
      k_block_abs_rowsum<float><<<n, 128, 0, st>>>(A->blk_size, A->row_ptr, A->col_idx, A->val_ptr,
                                                   (const float *)A_vals, mu, rowbase, babs);
    SM_LAUNCHED();
    k_scale_gershgorin<<<n_cols, 256, 0, st>>>(cols, A->blk_size, A->row_ptr, A->col_idx, P->gmap_ptr,
                                               P->gmap, rowbase, babs, scale);
    SM_LAUNCHED();
    if (scale_mode == SM_SCALE_GLOBAL) {
      int32_t rcg = global_scale(A, A_vals, a_dtype, P, mu, n_cols, scale, (char *)ws + g_off, ws_bytes - g_off, st);
      if (rcg != SM_OK) return rcg;
    }
  }

  GatherArgs g{cols, col_off, A->row_ptr, A->val_ptr, P->row_off, P->gmap_ptr, P->gmap,
               P->dim, P->dim_pad, scale, mu, opt(OPT_GATHER_LEAN) != 0 ? 1 : 0};
  // SM_SCALE_POWER: gather at the Gershgorin scale, tighten the scale by power steps on that X0
  // (power_scale.cu), then gather again so that X0 is rounded to the working type only once.
  const int passes = (scale_mode == SM_SCALE_POWER) ? 2 : 1;
  for (int pass = 0; pass < passes; ++pass) {
    int32_t rc = SM_ERR_UNSUPPORTED;
#define SM_GATHER_CASE(TA, TX, IMG) \
  rc = launch_gather<TA, TX, IMG>(g, A_vals, X_packed, n_cols, P->max_dim_pad, P->max_nbr, P->max_dim, st)
    if (a_dtype == SM_F64) {
      if (x_dtype == SM_F64) SM_GATHER_CASE(double, double, false);
      else if (x_dtype == SM_F32) SM_GATHER_CASE(double, float, false);
      else if (x_dtype == SM_BF16) SM_GATHER_CASE(double, __nv_bfloat16, true);
      else SM_GATHER_CASE(double, __half, true);
    } else {
      if (x_dtype == SM_F64) SM_GATHER_CASE(float, double, false);
      else if (x_dtype == SM_F32) SM_GATHER_CASE(float, float, false);
      else if (x_dtype == SM_BF16) SM_GATHER_CASE(float, __nv_bfloat16, true);
      else SM_GATHER_CASE(float, __half, true);
    }
#undef SM_GATHER_CASE
    if (rc != SM_OK) return rc;
    if (pass == 0 && passes == 2) {
      rc = power_scale(P, cols, n_cols, col_off, x_dtype, X_packed, scale, ratio, st);
      if (rc != SM_OK) return rc;
    }
  }
  return SM_OK;
}

template <typename TX, typename TR, bool IMG>
static int32_t launch_scatter(const sm_bcsr_t *A, const sm_pattern_t *P, const int32_t *cols, int32_t n_cols,
                              const int64_t *col_off, const void *S, void *R, cudaStream_t st) {
  const int32_t stage_off = (int32_t)align_up((int64_t)(P->max_nbr + 1) * 4 + (int64_t)(P->max_dim + 2) * 2, 16);
  const size_t smem = (size_t)stage_off + SCATTER_STAGE_BYTES;
  static bool attr_set = false;                          // per instantiation: opt in to > 48 KB of dynamic smem
  if (!attr_set) {
    SM_CUDA(cudaFuncSetAttribute(k_scatter<TX, TR, IMG>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024));
    attr_set = true;
  }
  if (smem > 160 * 1024) return SM_ERR_UNSUPPORTED;
  k_scatter<TX, TR, IMG><<<n_cols, 256, smem, st>>>(cols, col_off, A->blk_size, A->row_ptr, A->col_idx,
                                                    A->val_ptr, P->own_pos, P->dim, P->dim_pad, P->tmap,
                                                    P->row_off, stage_off, (const TX *)S, (TR *)R);
  SM_LAUNCHED();
  return SM_OK;
}

extern "C" int32_t sm_symmetrise(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t r_dtype, void *R_vals,
                                 void *stream) {
  if (!A || !P || !R_vals) return SM_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  if (r_dtype == SM_F64)
    k_symmetrise_density<double, false><<<A->n_blk, 32 * SYMD_WARPS, 0, st>>>(A->blk_size, A->row_ptr, A->col_idx,
                                                                             A->val_ptr, P->tmap, (double *)R_vals);
  else if (r_dtype == SM_F32)
    k_symmetrise_density<float, false><<<A->n_blk, 32 * SYMD_WARPS, 0, st>>>(A->blk_size, A->row_ptr, A->col_idx,
                                                                            A->val_ptr, P->tmap, (float *)R_vals);
  else
    return SM_ERR_UNSUPPORTED;
  SM_LAUNCHED();
  return SM_OK;
}

extern "C" int32_t sm_scatter(const sm_bcsr_t *A, const sm_pattern_t *P, const int32_t *cols, int32_t n_cols,
                              const int64_t *col_off, int32_t x_dtype, const void *S_packed, int32_t r_dtype,
                              void *R_vals, int32_t symmetrise, void *stream) {
  if (!A || !P || !S_packed || !R_vals || !col_off) return SM_ERR_ARG;
  if (!cols) n_cols = P->n_blk;
  if (n_cols <= 0) return SM_ERR_ARG;
  if (r_dtype != SM_F64 && r_dtype != SM_F32) return SM_ERR_UNSUPPORTED;
  if (symmetrise && cols && n_cols != P->n_blk) return SM_ERR_ARG;
  if (P->max_dim > 65535) return SM_ERR_UNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  int32_t rc = SM_ERR_UNSUPPORTED;
#define SM_SCATTER_CASE(TX, IMG)                                                                   \
  rc = (r_dtype == SM_F64)                                                                         \
           ? launch_scatter<TX, double, IMG>(A, P, cols, n_cols, col_off, S_packed, R_vals, st)    \
           : launch_scatter<TX, float, IMG>(A, P, cols, n_cols, col_off, S_packed, R_vals, st)
  if (x_dtype == SM_F64) SM_SCATTER_CASE(double, false);
  else if (x_dtype == SM_F32) SM_SCATTER_CASE(float, false);
  else if (x_dtype == SM_BF16) SM_SCATTER_CASE(__nv_bfloat16, true);
  else if (x_dtype == SM_F16) SM_SCATTER_CASE(__half, true);
#undef SM_SCATTER_CASE
  if (rc != SM_OK) return rc;
  if (symmetrise) return sm_symmetrise(A, P, r_dtype, R_vals, stream);
  return SM_OK;
}

// sm_symmetrise followed by sm_density_from_sign in one pass over the values (used by sm_density).
int32_t sm::symmetrise_density(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t d_dtype, void *RD_vals,
                               double *trace, cudaStream_t st) {
  if (d_dtype == SM_F64) {
    k_symmetrise_density<double, true><<<A->n_blk, 32 * SYMD_WARPS, 0, st>>>(A->blk_size, A->row_ptr, A->col_idx, A->val_ptr, P->tmap,
                                                           (double *)RD_vals);
    SM_LAUNCHED();
    if (trace) {
      k_trace<double><<<1, 1024, 0, st>>>(A->n_blk, A->blk_size, A->row_ptr, A->val_ptr, P->own_pos,
                                          (const double *)RD_vals, trace);
      SM_LAUNCHED();
    }
  } else if (d_dtype == SM_F32) {
    k_symmetrise_density<float, true><<<A->n_blk, 32 * SYMD_WARPS, 0, st>>>(A->blk_size, A->row_ptr, A->col_idx, A->val_ptr, P->tmap,
                                                          (float *)RD_vals);
    SM_LAUNCHED();
    if (trace) {
      k_trace<float><<<1, 1024, 0, st>>>(A->n_blk, A->blk_size, A->row_ptr, A->val_ptr, P->own_pos,
                                         (const float *)RD_vals, trace);
      SM_LAUNCHED();
    }
  } else {
    return SM_ERR_UNSUPPORTED;
  }
  return SM_OK;
}

extern "C" int32_t sm_density_from_sign(const sm_bcsr_t *A, const sm_pattern_t *P, int32_t d_dtype,
                                        void *RD_vals, double *trace, void *stream) {
  if (!A || !P || !RD_vals) return SM_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  if (d_dtype == SM_F64) {
    k_density<double><<<A->n_blk, 128, 0, st>>>(A->blk_size, A->row_ptr, A->col_idx, A->val_ptr, (double *)RD_vals);
    SM_LAUNCHED();
    if (trace) {
      k_trace<double><<<1, 1024, 0, st>>>(A->n_blk, A->blk_size, A->row_ptr, A->val_ptr, P->own_pos,
                                          (const double *)RD_vals, trace);
      SM_LAUNCHED();
    }
  } else if (d_dtype == SM_F32) {
    k_density<float><<<A->n_blk, 128, 0, st>>>(A->blk_size, A->row_ptr, A->col_idx, A->val_ptr, (float *)RD_vals);
    SM_LAUNCHED();
    if (trace) {
      k_trace<float><<<1, 1024, 0, st>>>(A->n_blk, A->blk_size, A->row_ptr, A->val_ptr, P->own_pos,
                                         (const float *)RD_vals, trace);
      SM_LAUNCHED();
    }
  } else {
    return SM_ERR_UNSUPPORTED;
  }
  return SM_OK;
}
