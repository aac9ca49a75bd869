// S2 effective charge, default variant (effq_mode 0): Eq. (9) with
// the charge density of Eq. (10) evaluated as the line integral it is
// the closed form of,
//     q(r) = Q' int_0^1 ds prod_{a in x,y,t} N(r_a - p0_a - s d_a; sigma_a),        d = p1 - p0,
// by an m-point Gauss-Legendre rule in s (m chosen per segment from its length in sigmas,
// relative error < 1.5e-7, i.e. below the fp32 rounding of the result).
// Every quadrature point s_k is a product of three 1-D Gaussians, so the sum over the n^3
// Gauss-Legendre nodes of a cuboid with the trilinear coefficients u_{lmn,rst} of Eq. (7)
// factors per axis:
//     Qeff[i,j,k] = K sum_k W_k GX_k[i] GY_k[j] GT_k[k],
//     G_k[i] = sum over the nodes (cuboid c in {i-1,i,i+1} within the bbox, node l) of
//              w_l u_{l,i-c} exp(-(x_{c,l} - p0 - s_k d)^2 / (2 sigma^2)).
// Same nodes, weights, coefficients and bounding box as the closed-form kernel
// (tred_effq.cu); only the order of summation and the evaluation of q differ.
//
// Kernel k_effq_blk: one CTA per (block, sub-tile of TS ticks); the tile [column][tick] lives
// in shared memory and every thread OWNS a column (and a range of its ticks) for the whole
// CTA, so the tile needs no synchronisation between segments, no atomics, and the order of
// the additions is fixed (segments ascending, quadrature points ascending): deterministic.
// The segments of the block are taken 32 records at a time; their quadrature points are cut
// into passes of <= 12 points, and EB_GP passes form a group:
//   phase A (warp per (pass, round of 31 table rows)): the three per-axis tables of the pass,
//            rows along the lanes, the n exponentials of a dual cell shared by the two grid
//            points it touches through a shuffle; everything that depends on the row is a
//            per-lane constant of the loop over the quadrature points;
//   phase B (thread per column): rank-m update of the thread's own tile cells, four ticks
//            per step (LDS.128 of the tile and of the broadcast t-table rows).
// Two __syncthreads per group.
#include <math.h>
#include "tred_common.cuh"

namespace {

constexpr int MMAX = 24;            // quadrature points of the largest rule
constexpr int NGL = MMAX * (MMAX + 1) / 2;

__constant__ float c_gl_s[NGL];     // nodes mapped to [0,1], rule m at offset m(m-1)/2
__constant__ float c_gl_w[NGL];     // weights, sum to 1

// Dual-cell node tables of the n-point rule per axis (same as tred_effq.cu): s = position
// in the dual cell between grid points d and d+1, w = GL weight, side = 0 if the node
// belongs to cuboid d, 1 if to cuboid d+1.  Abramowitz & Stegun 25.4.
template <int N> struct DualGL {
  __host__ __device__ static constexpr float s(int q) {
    return N == 1 ? 0.0f
         : N == 2 ? (q == 0 ? 0.28867513459481287f : 0.71132486540518713f)
         : N == 3 ? (q == 0 ? 0.0f : q == 1 ? 0.38729833462074170f : 0.61270166537925830f)
                  : (q == 0 ? 0.16999052179242816f : q == 1 ? 0.43056815579702630f
                     : q == 2 ? 0.56943184420297370f : 0.83000947820757184f);
  }
  __host__ __device__ static constexpr float w(int q) {
    return N == 1 ? 2.0f
         : N == 2 ? 1.0f
         : N == 3 ? (q == 0 ? 0.88888888888888888f : 0.55555555555555556f)
                  : ((q == 0 || q == 3) ? 0.65214515486254614f : 0.34785484513745386f);
  }
  __host__ __device__ static constexpr int side(int q) {
    return N == 1 ? 0 : N == 2 ? q : N == 3 ? (q == 2 ? 1 : 0) : (q >= 2 ? 1 : 0);
  }
};

__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

// One table entry (used by the truth record below): grid point gi of one axis, quadrature
// centre c (grid units relative to lo), k2 = log2(e) / (2 sigma^2).
template <int N>
__device__ __forceinline__ float axis_entry(int gi, int lo, int hi, float c, float k2) {
  float v = 0.0f;
  const float base = (float)(gi - lo) + 0.5f;
#pragma unroll
  for (int q = 0; q < N; ++q) {
    const float sq = DualGL<N>::s(q), wq = DualGL<N>::w(q);
    {   // dual cell gi (gi is its lower corner): coefficient 1 - s
      const int cub = gi + DualGL<N>::side(q);
      const float z = (base + sq) - c;
      const float e = ex2_approx(-z * z * k2);
      if (cub >= lo && cub <= hi) v = fmaf(wq * (1.0f - sq), e, v);
    }
    if (sq != 0.0f) {   // dual cell gi-1 (gi is its upper corner): coefficient s
      const int cub = gi - 1 + DualGL<N>::side(q);
      const float z = (base - 1.0f + sq) - c;
      const float e = ex2_approx(-z * z * k2);
      if (cub >= lo && cub <= hi) v = fmaf(wq * sq, e, v);
    }
  }
  return v;
}

// Quadrature of a segment record: number of pieces and points per piece from its length W
// in sigmas (same arithmetic wherever it is needed).  The m-point Gauss-Legendre rule of
// int_0^1 N(x - s W) ds has a relative error (of the maximum over x) below 1.5e-7 for
// W <= 1.13, 1.83, 2.58, 3.35, 4.11 (m = 4..8) and then ~0.75 more per extra point up to
// 16.1 at m = 24 (computed against the erf closed form); the thresholds below are 0.95 of that.
struct SegQuad { int npiece, m; };
__device__ __forceinline__ SegQuad seg_quad(int flag, float dx, float dy, float dt, float sx, float sy, float st) {
  SegQuad q;
  q.npiece = 1; q.m = 4;
  if (!flag) {
    const float W = sqrtf((dx / sx) * (dx / sx) + (dy / sy) * (dy / sy) + (dt / st) * (dt / st));
    q.npiece = (int)ceilf(W * (1.0f / 15.3f));
    if (q.npiece < 1) q.npiece = 1;
    const float Wp = W / (float)q.npiece;
    if (Wp <= 3.18f) q.m = Wp <= 1.07f ? 4 : Wp <= 1.74f ? 5 : Wp <= 2.45f ? 6 : 7;
    else {
      q.m = 8 + (int)ceilf((Wp - 3.9f) * (1.0f / 0.7125f));
      q.m = q.m < 8 ? 8 : q.m > MMAX ? MMAX : q.m;
    }
  }
  return q;
}

// ------------------------------------------------------------------ table rows
// Entries of the per-axis tables for the dual cells one lane each (lane = cell gi between
// grid points gi and gi + 1, of the axis with bbox [lo_a, hi_a], segment end p0a, extent da,
// nk2 = -log2(e)/(2 sigma^2)), for the quadrature points [g0, g0 + cnt) of the segment: the n
// exponentials of a cell serve the entry of gi (coefficient 1 - s) and, through a shuffle, the
// entry of gi + 1 (coefficient s) held by the next lane, so lane 0 and the first cell of an axis
// only provide.  Kx = K for the x axis (K W_k is folded into the x table), 1 otherwise.
struct QuadRule { int m, flag, goff; float inv_np; };

template <int N>
__device__ __forceinline__ void effq_cells(int gi, int lo_a, int hi_a, float p0a, float da, float nk2, float Kx,
                                           bool scale_w, bool wr, bool zero, float* __restrict__ dst, int stride,
                                           const QuadRule& qr, int g0, int cnt) {
  const float base = (float)(gi - lo_a) + 0.5f;
  float wo[N], wu[N];
#pragma unroll
  for (int q = 0; q < N; ++q) {
    const int cub = gi + DualGL<N>::side(q);
    const bool ok = cub >= lo_a && cub <= hi_a;
    wo[q] = ok ? DualGL<N>::w(q) * (1.0f - DualGL<N>::s(q)) : 0.0f;
    wu[q] = ok ? DualGL<N>::w(q) * DualGL<N>::s(q) : 0.0f;
  }
  int pc = g0 / qr.m, mi = g0 - pc * qr.m;
  for (int pt = 0; pt < cnt; ++pt, dst += stride) {
    float sk, wk;
    if (qr.flag) { sk = 0.5f; wk = (g0 + pt) == 0 ? 1.0f : 0.0f; }      // point-like: midpoint Gaussian
    else { sk = ((float)pc + c_gl_s[qr.goff + mi]) * qr.inv_np; wk = c_gl_w[qr.goff + mi] * qr.inv_np; }
    const float zb = base - fmaf(sk, da, p0a);
    float own = 0.0f, up = 0.0f;
#pragma unroll
    for (int q = 0; q < N; ++q) {
      const float z = zb + DualGL<N>::s(q);
      const float e = ex2_approx(z * z * nk2);
      own = fmaf(wo[q], e, own);
      if (DualGL<N>::s(q) != 0.0f) up = fmaf(wu[q], e, up);
    }
    const float below = __shfl_up_sync(0xffffffffu, up, 1);
    float val = N > 1 ? own + below : own;
    if (scale_w) val *= Kx * wk;
    if (zero) val = 0.0f;
    if (wr) *dst = val;
    if (++mi == qr.m) { mi = 0; ++pc; }
  }
}

// ------------------------------------------------------------------ tables built once per segment
// A segment meets ~4 blocks x 1.5 tick tiles, and every such CTA needs the same three per-axis
// tables.  With a workspace, tred_effq builds them once per segment (k_effq_tables, one warp per
// segment, whole bounding box) and the tile CTAs fetch the rows they need with bulk copies; without
// one (or for segments whose tables do not fit it) the tile CTAs compute the rows themselves with
// the same code (effq_cells): same values either way.
// Table of segment s at tab + 4 * off[s] floats: chunks of EB_MQ = 12 quadrature points, chunk c
// is [row][cpt] (cpt = points of the chunk rounded up to 4, so every row range is a 16-byte
// aligned contiguous piece); rows = x rows (grid points lox-E .. hix+E), y rows, then t rows
// from the 4-aligned tick tb = align_down(lot - E, 4), ntfp = align_up(hit + E + 1 - tb, 4) of
// them.  Entries of grid points outside the grid are zero (clip and drop, reading G13).
constexpr int EB_MQ = 12;           // quadrature points per pass / table chunk
// Table offsets are int32 prefix sums of table sizes in 16-byte units.  k_effq_sizes also adds
// the sizes up in 64 bits, and the offsets are used only if that total is at most TAB_TOTAL_MAX,
// i.e. if no prefix sum can have wrapped (a wrapped offset could pass every range check and put
// a table in front of the workspace).  Beyond it (tens of millions of marked segments in one
// call, or tens of thousands of long unsplit ones) no segment gets a table: same values,
// computed by the tile CTAs.  One table is at most TAB_SIZE_MAX units (4 MiB).
constexpr int64_t TAB_SIZE_MAX = 1 << 18;
constexpr int64_t TAB_TOTAL_MAX = 0x7fffffff;

struct TabGeom { int nxf, nyf, tb, ntfp, rs; };
__device__ __forceinline__ TabGeom tab_geom(int lox, int loy, int lot, int hix, int hiy, int hit, int E) {
  TabGeom t;
  t.nxf = hix - lox + 1 + 2 * E;
  t.nyf = hiy - loy + 1 + 2 * E;
  t.tb = (lot - E) & ~3;
  t.ntfp = ((hit + E + 1 - t.tb) + 3) & ~3;
  t.rs = t.nxf + t.nyf + t.ntfp;
  return t;
}
// floats of the table of a segment with ptot quadrature points and rs rows
__device__ __forceinline__ int64_t tab_floats(int ptot, int rs) {
  const int nfull = ptot / EB_MQ, rem = ptot - nfull * EB_MQ;
  return (int64_t)rs * (nfull * EB_MQ + ((rem + 3) & ~3));
}

// marks the segments the blocks [0, nb) of this call refer to (idempotent plain stores)
__global__ void __launch_bounds__(256)
k_effq_mark(int64_t nb, const int32_t* __restrict__ blk_off, const int32_t* __restrict__ pair_seg,
            int32_t* __restrict__ mark) {
  const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (warp >= nb) return;
  const int p0 = blk_off[warp], p1 = blk_off[warp + 1];
  for (int p = p0 + lane; p < p1; p += 32) mark[pair_seg[p]] = 1;
}

// mark[s] = size of the table of a marked segment in 16-byte units (0 if not marked);
// *total (zeroed by the caller) += all sizes, in 64 bits (integer atomics: order does not matter)
template <int N>
__global__ void __launch_bounds__(256)
k_effq_sizes(int64_t nseg, const float* __restrict__ augf, const int32_t* __restrict__ augi,
             int32_t* __restrict__ mark, unsigned long long* __restrict__ total) {
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int v = 0;
  if (s < nseg && mark[s]) {
    constexpr int E = N > 1 ? 1 : 0;
    const TabGeom t = tab_geom(augi[0 * nseg + s], augi[1 * nseg + s], augi[2 * nseg + s], augi[3 * nseg + s],
                               augi[4 * nseg + s], augi[5 * nseg + s], E);
    const float p0x = augf[0 * nseg + s], p0y = augf[1 * nseg + s], p0t = augf[2 * nseg + s];
    const SegQuad q = seg_quad(augi[6 * nseg + s], augf[3 * nseg + s] - p0x, augf[4 * nseg + s] - p0y,
                               augf[5 * nseg + s] - p0t, augf[6 * nseg + s], augf[7 * nseg + s], augf[8 * nseg + s]);
    const int64_t sz = tab_floats(q.npiece * q.m, t.rs) >> 2;
    // tables beyond 4 MiB (absurdly large boxes): size 0 = no table, the tile CTAs evaluate the
    // segment themselves
    v = sz <= TAB_SIZE_MAX ? (int)sz : 0;
  }
  if (s <= nseg) mark[s] = v;
  unsigned long long w = (unsigned long long)v;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) w += __shfl_down_sync(0xffffffffu, w, o);
  if ((threadIdx.x & 31) == 0 && w) atomicAdd(total, w);
}

// one warp per 32 consecutive segments; the marked ones among them one after the other
template <int N>
__global__ void __launch_bounds__(128)
k_effq_tables(int64_t nseg, const int32_t* __restrict__ off, const int64_t* __restrict__ total, int64_t cap16,
              const float* __restrict__ augf, const int32_t* __restrict__ augi, float* __restrict__ tab, TredGrid g) {
  const int64_t w = (int64_t)blockIdx.x * 4 + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  const int64_t s_l = w * 32 + lane;
  bool mine = false;
  if (s_l < nseg && *total <= TAB_TOTAL_MAX) {
    const int o0 = off[s_l], o1 = off[s_l + 1];
    mine = o0 >= 0 && o1 > o0 && (int64_t)o1 <= cap16;
  }
  uint32_t todo = __ballot_sync(0xffffffffu, mine);
  constexpr int E = N > 1 ? 1 : 0;
  constexpr float LOG2E_HALF = 0.72134752044448170f;
  while (todo) {
    const int b = __ffs(todo) - 1;
    todo &= todo - 1;
    const int64_t s = w * 32 + b;
    const int lo[3] = {augi[0 * nseg + s], augi[1 * nseg + s], augi[2 * nseg + s]};
    const int hi[3] = {augi[3 * nseg + s], augi[4 * nseg + s], augi[5 * nseg + s]};
    const float p0[3] = {augf[0 * nseg + s], augf[1 * nseg + s], augf[2 * nseg + s]};
    const float d3[3] = {augf[3 * nseg + s] - p0[0], augf[4 * nseg + s] - p0[1], augf[5 * nseg + s] - p0[2]};
    const float sg[3] = {augf[6 * nseg + s], augf[7 * nseg + s], augf[8 * nseg + s]};
    const float K = augf[9 * nseg + s] * 0.063493635934240969f / (sg[0] * sg[1] * sg[2]) * 0.125f;
    const int flag = augi[6 * nseg + s];
    const SegQuad q = seg_quad(flag, d3[0], d3[1], d3[2], sg[0], sg[1], sg[2]);
    const QuadRule qr{q.m, flag, q.m * (q.m - 1) / 2, 1.0f / (float)q.npiece};
    const int ptot = q.npiece * q.m;
    const TabGeom t = tab_geom(lo[0], lo[1], lo[2], hi[0], hi[1], hi[2], E);
    float* T = tab + 4 * (int64_t)off[s];
    // cells: one leading cell per axis, then one per row
    const int ncell = t.rs + 3;
    for (int r0 = 0; r0 < ncell - 1; r0 += 31) {
      const int p = r0 + lane;
      int a, q0, first, rowb, NGa;
      if (p < t.nxf + 1) { a = 0; q0 = p; first = lo[0] - E; rowb = 0; NGa = g.NGx; }
      else if (p < t.nxf + t.nyf + 2) { a = 1; q0 = p - (t.nxf + 1); first = lo[1] - E; rowb = t.nxf; NGa = g.NGy; }
      else { a = 2; q0 = p - (t.nxf + t.nyf + 2); first = t.tb; rowb = t.nxf + t.nyf; NGa = g.NGt; }
      const int gi = first - 1 + q0;
      const bool wr = lane >= 1 && q0 >= 1 && p < ncell;
      const float nk2 = -LOG2E_HALF / (sg[a] * sg[a]);
      for (int g0 = 0; g0 < ptot; g0 += EB_MQ) {
        const int cnt = min(EB_MQ, ptot - g0), cpt = (cnt + 3) & ~3;
        effq_cells<N>(gi, lo[a], hi[a], p0[a], d3[a], nk2, K, a == 0, wr, gi < 0 || gi >= NGa,
                      T + (int64_t)g0 * t.rs + (rowb + q0 - 1) * cpt, 1, qr, g0, cnt);
      }
    }
  }
}

// ------------------------------------------------------------------ the tile kernel
// Warp roles: the LAST warp is the producer, the others are consumers.
//   producer : stages the segment records of the block (32 at a time), finds the ones that meet
//              the tile, cuts their quadrature points into passes of <= 12 points, packs the
//              passes' table rows (x rows, y rows, t rows of the clipped footprint, [row][cpt])
//              into a stage of the table ring -- three bulk copies per pass from the segment's
//              table in global memory, completion on the stage's mbarrier (or, without a table,
//              computed in place) -- and writes one descriptor per pass;
//   consumers: every warp OWNS a rectangle of the tile (wi rows x wj columns x wt ticks) for the
//              whole CTA, so no two warps ever touch the same cell: no atomics, no CTA-wide
//              barrier in the loop, fixed order of additions (passes in order).  Per pass the
//              lanes share out the columns of the footprint inside the rectangle (and its tick
//              quads when those are few) and add the rank-cnt product to the tile.
// The tile is written out with one bulk store (TS floats of a column) per thread.
// The CTAs are persistent (grid = 2 per SM, tiles round-robin): the producer runs ahead of the
// consumers by the depth of the ring, so the dependent loads that start a tile (block key ->
// segment list -> records -> table rows) overlap the arithmetic of the previous one.
constexpr int EB_SB = 32;           // segment records staged per batch
constexpr int EB_NREC = 36;         // int32 words per staged record
constexpr int EB_STAGES = 4;
constexpr int EB_STAGE_FLOATS = 2048;   // 8 KB of table rows per stage
constexpr int EB_LAST = 0x100;      // s_n flag: last stage of the tile
constexpr int EB_MAXP = 32;         // passes per stage at most
constexpr int EB_ND = 12;           // int32 words per pass descriptor
// staged record (producer only, after the batch prologue):
//   0..5 lo, hi (x, y, t)   6 flag   7 m (points per piece)
//   8..10 p0 (x, y, t)      11 K = Q' (2 pi)^-3/2 / (sx sy st) / 8
//   12..14 d = p1 - p0      15 1 / npiece
//   16..18 -log2(e)/(2 sigma^2) (x, y, t)     19 offset of rule m in c_gl_s / c_gl_w
//   20..23 clipped footprint in the tile: x first, nx, y first, ny          (tile-relative)
//   24..27 t first, t last (tile-relative), first / count of the 4-aligned tick range
//   28 quadrature points in total (npiece m)   29 passes
//   30 offset of the segment's table in 16-byte units (-1: none)   31 its rows
//   32 x row, 33 y row, 34 t row of the table that holds the first x / y / aligned t entry of the tile
enum { ER_M = 7, ER_P0 = 8, ER_K = 11, ER_D = 12, ER_INVNP = 15, ER_NK2 = 16, ER_GOFF = 19, ER_FX = 20, ER_FT = 24,
       ER_PTOT = 28, ER_NPASS = 29, ER_TOFF = 30, ER_TRS = 31, ER_TROW = 32 };
// pass descriptor: 0..3 = x first, nx, y first, ny; 4..7 = t first, t last, aligned first, aligned count;
// 8 = points, 9 = points rounded up to 4 (row pitch), 10 = offset of the pass's rows in the stage (floats)
enum { ED_CNT = 8, ED_CPT = 9, ED_SLOT = 10 };

struct BlkParams {
  int TS, nsub;      // ticks per CTA tile, tiles per block
  int ncol;          // Bx * By columns
  int by_shift;      // log2(By)
  int ts_shift;      // log2(TS)
  int CS;            // column stride of the tile in floats (TS + 4: conflict-free LDS.128)
  int RS;            // most rows a pass can have = Bx + By + TS
  // what a consumer warp owns for the whole CTA: wi rows x wj columns-in-a-row x wt ticks
  int wi, wj, wt;
  int nwj, nwi;      // warps along j, along i (warp -> (tick range, i range, j range))
  int ncw;           // consumer warps (the producer is warp ncw)
  int64_t cap16;     // 16-byte units of table workspace (0: no tables)
  const int64_t* tab_total;   // sum of all table sizes (device; read only if there are tables)
};

__device__ __forceinline__ uint32_t eb_smem(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void eb_mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void eb_mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void eb_mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// A wait longer than ~2 s means a broken pipeline: trap instead of hanging the device.
__device__ __forceinline__ void eb_mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok = 0;
  long long t0 = 0;
  for (int it = 0;; ++it) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    if (ok) return;
    if (it == 64) t0 = clock64();
    if (it > 64 && (it & 1023) == 0 && clock64() - t0 > 4000000000ll) {
      printf("k_effq_blk: mbarrier wait timed out (block %d thread %d)\n", blockIdx.x, threadIdx.x);
      __trap();
    }
  }
}
__device__ __forceinline__ void eb_bulk_g2s(float* dst, const float* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(eb_smem(dst)), "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}

// Phase B of one pass for one lane: tile[col][k] += sum_pt X[pt] Y[pt] T[k][pt] for the tick quads
// k = k0, k0 + kstep, ... < k1 of column col.  X, Y, T rows have a pitch of CQ * 4 floats.
template <int CNT>
__device__ __forceinline__ void effq_blk_update(float* __restrict__ tcol, const float* __restrict__ X,
                                                const float* __restrict__ Y, const float* __restrict__ T, int k0,
                                                int k1, int kstep) {
  constexpr int CQ = (CNT + 3) / 4;
  float ab[4 * CQ];
#pragma unroll
  for (int q = 0; q < CQ; ++q) {
    const float4 a = reinterpret_cast<const float4*>(X)[q], b = reinterpret_cast<const float4*>(Y)[q];
    ab[4 * q] = a.x * b.x; ab[4 * q + 1] = a.y * b.y; ab[4 * q + 2] = a.z * b.z; ab[4 * q + 3] = a.w * b.w;
  }
  for (int k = k0; k < k1; k += kstep) {
    float4* tp = reinterpret_cast<float4*>(tcol + k);
    const float4* gt = reinterpret_cast<const float4*>(T + k * (4 * CQ));
    float4 v4 = *tp;
    float v[4] = {v4.x, v4.y, v4.z, v4.w};
#pragma unroll
    for (int kk = 0; kk < 4; ++kk)
#pragma unroll
      for (int q = 0; q < CQ; ++q) {
        const float4 gq = gt[kk * CQ + q];
        if (4 * q < CNT) v[kk] = fmaf(ab[4 * q], gq.x, v[kk]);
        if (4 * q + 1 < CNT) v[kk] = fmaf(ab[4 * q + 1], gq.y, v[kk]);
        if (4 * q + 2 < CNT) v[kk] = fmaf(ab[4 * q + 2], gq.z, v[kk]);
        if (4 * q + 3 < CNT) v[kk] = fmaf(ab[4 * q + 3], gq.w, v[kk]);
      }
    *tp = make_float4(v[0], v[1], v[2], v[3]);
  }
}

template <int N, int MAXT>
__global__ void __launch_bounds__(MAXT, MAXT > 512 ? 1 : 2)
k_effq_blk(int64_t nseg, const int64_t* __restrict__ keys, const int32_t* __restrict__ blk_off,
           const int32_t* __restrict__ pair_seg, const float* __restrict__ augf,
           const int32_t* __restrict__ augi, const int32_t* __restrict__ tabofs, const float* __restrict__ gtab,
           float* __restrict__ payload, int64_t ntiles, TredGrid g, BlkParams P) {
  extern __shared__ __align__(128) float smf[];
  float* tile = smf;                                          // [ncol][CS]
  float* ring = smf + (size_t)P.ncol * P.CS;                  // [EB_STAGES][EB_STAGE_FLOATS]
  int32_t (*s_rec)[EB_NREC] = reinterpret_cast<int32_t (*)[EB_NREC]>(ring + EB_STAGES * EB_STAGE_FLOATS);
  __shared__ __align__(16) int32_t s_desc[EB_STAGES][EB_MAXP][EB_ND];
  __shared__ int s_n[EB_STAGES];
  __shared__ int s_list[EB_SB];
  __shared__ int s_pfx[EB_SB + 1];
  __shared__ __align__(8) uint64_t s_bar[2 * EB_STAGES];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  constexpr int E = N > 1 ? 1 : 0;
  constexpr float LOG2E_HALF = 0.72134752044448170f;          // log2(e) / 2
  const int nct = P.ncw * 32;                                 // consumer threads
  auto full_bar = [&](int s) { return eb_smem(&s_bar[s]); };
  auto empty_bar = [&](int s) { return eb_smem(&s_bar[EB_STAGES + s]); };

  if (threadIdx.x == 0) {
    for (int s = 0; s < EB_STAGES; ++s) { eb_mbar_init(full_bar(s), 1); eb_mbar_init(empty_bar(s), P.ncw); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (threadIdx.x < nct) {
    float4* t4 = reinterpret_cast<float4*>(tile);
    const int n4 = (P.ncol * P.CS) >> 2;
    for (int i = threadIdx.x; i < n4; i += nct) t4[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
  }
  __syncthreads();

  if (warp == P.ncw) {
    // ================================================================ producer
    int stage = 0, sphase = 0;
    // The stage filled last is handed over (arrive) only when the next one is ready or the tile
    // ends, so that the tile's last stage can carry the EB_LAST flag; its copies run meanwhile.
    int pend_stage = -1, pend_n = 0;
    auto hand_over = [&](int flag) {
      if (lane == 0) {
        s_n[pend_stage] = pend_n | flag;
        eb_mbar_arrive(full_bar(pend_stage));
      }
      pend_stage = -1;
    };
    const int W = EB_STAGE_FLOATS - P.RS * EB_MQ;             // passes that START in a window of W floats fit a stage
    const float invW = 1.0f / (float)W;
    // The loads that start a tile are issued one tile (records of its first batch) and two tiles
    // (block key, segment range) ahead and land in registers while the current tile is processed.
    struct Meta { int64_t key; int s_beg, s_end; };
    auto load_meta = [&](int64_t t) {
      Meta m{0, 0, 0};
      if (t < ntiles) { const int b = (int)(t / P.nsub); m.key = keys[b]; m.s_beg = blk_off[b]; m.s_end = blk_off[b + 1]; }
      return m;
    };
    // raw record of one lane: words 0..6 = bbox, flag; 7..16 = p0, p1, sigma, Q'; 17, 18 = table
    // offsets of s, s + 1 (all loads of a record in flight at once)
    const bool tab_ok = tabofs && *P.tab_total <= TAB_TOTAL_MAX;      // offsets cannot have wrapped
    auto load_rec = [&](int b0, int nbatch, int32_t (&v)[19]) {
      if (lane < nbatch) {
        const int64_t s = pair_seg[b0 + lane];
#pragma unroll
        for (int f = 0; f < 7; ++f) v[f] = augi[f * nseg + s];
#pragma unroll
        for (int f = 7; f < 17; ++f) v[f] = __float_as_int(augf[(f - 7) * nseg + s]);
        v[17] = tab_ok ? tabofs[s] : 0;
        v[18] = tab_ok ? tabofs[s + 1] : 0;
      }
    };
    Meta m_cur = load_meta(blockIdx.x), m_nxt = load_meta((int64_t)blockIdx.x + gridDim.x);
    int32_t vpre[19];
    load_rec(m_cur.s_beg, min(EB_SB, m_cur.s_end - m_cur.s_beg), vpre);
    for (int64_t tile_id = blockIdx.x; tile_id < ntiles; tile_id += gridDim.x) {
    const int blk = (int)(tile_id / P.nsub);
    const int sub = (int)(tile_id - (int64_t)blk * P.nsub);
    const int64_t key = m_cur.key;
    const int by = (int)(key % g.NBy);
    const int bx = (int)((key / g.NBy) % g.NBx);
    const int bt = (int)(key / ((int64_t)g.NBy * g.NBx));
    const int I0 = bx * g.Bx, J0 = by * g.By, K0 = bt * g.Bt + sub * P.TS;
    const int s_beg = m_cur.s_beg, s_end = m_cur.s_end;
    __syncwarp();
    if (lane < min(EB_SB, s_end - s_beg)) {
#pragma unroll
      for (int f = 0; f < 19; ++f) s_rec[lane][f] = vpre[f];
    }
    m_cur = m_nxt;
    load_rec(m_cur.s_beg, min(EB_SB, m_cur.s_end - m_cur.s_beg), vpre);      // next tile's first batch
    m_nxt = load_meta(tile_id + 2 * (int64_t)gridDim.x);
    for (int b0 = s_beg; b0 < s_end; b0 += EB_SB) {
      const int nbatch = min(EB_SB, s_end - b0);
      __syncwarp();
      if (b0 > s_beg) {
        int32_t v[19];
        load_rec(b0, nbatch, v);
        if (lane < nbatch) {
#pragma unroll
          for (int f = 0; f < 19; ++f) s_rec[lane][f] = v[f];
        }
      }
      __syncwarp();
      // one lane per record: does the footprint meet this tile?  constants of the segment, once
      int npass_all, nlist;
      {
        const int j = lane;
        bool hit_tile = false;
        int npass = 0;
        if (j < nbatch) {
          int32_t* rec = s_rec[j];
          const int lox = rec[0], loy = rec[1], lot = rec[2], hix = rec[3], hiy = rec[4], hit = rec[5];
          const int ix0 = max(lox - E, I0), ix1 = min(min(hix + E, I0 + g.Bx - 1), g.NGx - 1);
          const int iy0 = max(loy - E, J0), iy1 = min(min(hiy + E, J0 + g.By - 1), g.NGy - 1);
          const int kt0 = max(lot - E, K0), kt1 = min(min(hit + E, K0 + P.TS - 1), g.NGt - 1);
          hit_tile = ix0 <= ix1 && iy0 <= iy1 && kt0 <= kt1;
          if (hit_tile) {
            const int flag = rec[6];
            const float p0x = __int_as_float(rec[7]), p0y = __int_as_float(rec[8]), p0t = __int_as_float(rec[9]);
            const float dx = __int_as_float(rec[10]) - p0x, dy = __int_as_float(rec[11]) - p0y,
                        dt = __int_as_float(rec[12]) - p0t;
            const float sx = __int_as_float(rec[13]), sy = __int_as_float(rec[14]), st = __int_as_float(rec[15]);
            const float Qp = __int_as_float(rec[16]);
            const int o0 = rec[17], o1 = rec[18];
            const SegQuad q = seg_quad(flag, dx, dy, dt, sx, sy, st);
            const int ptot = q.npiece * q.m;
            npass = (ptot + EB_MQ - 1) / EB_MQ;
            rec[ER_M] = q.m;
            rec[ER_P0 + 0] = __float_as_int(p0x); rec[ER_P0 + 1] = __float_as_int(p0y); rec[ER_P0 + 2] = __float_as_int(p0t);
            rec[ER_K] = __float_as_int(Qp * 0.063493635934240969f / (sx * sy * st) * 0.125f);
            rec[ER_D + 0] = __float_as_int(dx); rec[ER_D + 1] = __float_as_int(dy); rec[ER_D + 2] = __float_as_int(dt);
            rec[ER_INVNP] = __float_as_int(1.0f / (float)q.npiece);
            rec[ER_NK2 + 0] = __float_as_int(-LOG2E_HALF / (sx * sx));
            rec[ER_NK2 + 1] = __float_as_int(-LOG2E_HALF / (sy * sy));
            rec[ER_NK2 + 2] = __float_as_int(-LOG2E_HALF / (st * st));
            rec[ER_GOFF] = q.m * (q.m - 1) / 2;
            rec[ER_FX + 0] = ix0 - I0; rec[ER_FX + 1] = ix1 - ix0 + 1;
            rec[ER_FX + 2] = iy0 - J0; rec[ER_FX + 3] = iy1 - iy0 + 1;
            const int a0 = (kt0 - K0) & ~3, a1 = ((kt1 - K0) | 3) + 1;
            rec[ER_FT + 0] = kt0 - K0; rec[ER_FT + 1] = kt1 - K0; rec[ER_FT + 2] = a0; rec[ER_FT + 3] = a1 - a0;
            rec[ER_PTOT] = ptot; rec[ER_NPASS] = npass;
            const TabGeom t = tab_geom(lox, loy, lot, hix, hiy, hit, E);
            const bool has = o0 >= 0 && o1 > o0 && (int64_t)o1 <= P.cap16;
            rec[ER_TOFF] = has ? o0 : -1;
            rec[ER_TRS] = t.rs;
            rec[ER_TROW + 0] = ix0 - (lox - E);
            rec[ER_TROW + 1] = t.nxf + iy0 - (loy - E);
            rec[ER_TROW + 2] = t.nxf + t.nyf + (K0 + a0 - t.tb);
          }
        }
        const uint32_t bal = __ballot_sync(0xffffffffu, hit_tile);
        const int pos = __popc(bal & ((1u << j) - 1u));
        if (hit_tile) s_list[pos] = j;
        int incl = npass;                               // 0 for records that do not hit
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int v = __shfl_up_sync(0xffffffffu, incl, o);
          if (lane >= o) incl += v;
        }
        if (hit_tile) s_pfx[pos] = incl - npass;
        nlist = __popc(bal);
        npass_all = __shfl_sync(0xffffffffu, incl, 31);
        if (lane == 31) s_pfx[nlist] = incl;
      }
      __syncwarp();
      // lanes = passes, 32 at a time
      for (int p0 = 0; p0 < npass_all; p0 += 32) {
        const int pi = p0 + lane;
        const bool valid = pi < npass_all;
        int l = 0;
        if (valid) {                                    // largest l with s_pfx[l] <= pi
          int lo_ = 0, hi_ = nlist - 1;
          while (lo_ < hi_) { const int mid = (lo_ + hi_ + 1) >> 1; if (s_pfx[mid] <= pi) lo_ = mid; else hi_ = mid - 1; }
          l = lo_;
        }
        const int32_t* rec = s_rec[valid ? s_list[l] : 0];
        const int lp = valid ? pi - s_pfx[l] : 0;
        int4 fx = make_int4(0, 0, 0, 0), ft = make_int4(0, 0, 0, 0);
        int cnt = 0, cpt = 0, size = 0;
        if (valid) {
          fx = *reinterpret_cast<const int4*>(rec + ER_FX);
          ft = *reinterpret_cast<const int4*>(rec + ER_FT);
          cnt = min(EB_MQ, rec[ER_PTOT] - lp * EB_MQ);
          cpt = (cnt + 3) & ~3;
          size = (fx.y + fx.w + ft.w) * cpt;
        }
        int incl = size;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
          const int v = __shfl_up_sync(0xffffffffu, incl, o);
          if (lane >= o) incl += v;
        }
        const int excl = incl - size;
        const int wid = valid ? (int)(((float)excl + 0.5f) * invW) : -1;
        const int wid_max = __reduce_max_sync(0xffffffffu, wid);
        for (int gw = 0; gw <= wid_max; ++gw) {
          const bool in = valid && wid == gw;
          const uint32_t m = __ballot_sync(0xffffffffu, in);
          if (!m) continue;
          const int head = __ffs(m) - 1;
          const int slot = excl - __shfl_sync(0xffffffffu, excl, head);
          const int idx = __popc(m & ((1u << lane) - 1u));
          const int toff = in ? rec[ER_TOFF] : -1;
          const uint32_t bytes = (in && toff >= 0) ? (uint32_t)size * 4u : 0u;
          const uint32_t tot = __reduce_add_sync(0xffffffffu, bytes);
          if (pend_stage >= 0) hand_over(0);
          if (lane == 0) eb_mbar_wait(empty_bar(stage), sphase ^ 1);
          __syncwarp();
          float* sbase = ring + stage * EB_STAGE_FLOATS;
          if (in) {
            int32_t* d = s_desc[stage][idx];
            *reinterpret_cast<int4*>(d) = fx;
            *reinterpret_cast<int4*>(d + 4) = ft;
            d[ED_CNT] = cnt; d[ED_CPT] = cpt; d[ED_SLOT] = slot;
          }
          pend_stage = stage; pend_n = __popc(m);
          // passes of segments without a table: the warp computes their rows in place
          uint32_t mc = __ballot_sync(0xffffffffu, in && toff < 0);
          while (mc) {
            const int b = __ffs(mc) - 1;
            mc &= mc - 1;
            const int lb = __shfl_sync(0xffffffffu, l, b), lpb = __shfl_sync(0xffffffffu, lp, b);
            const int slotb = __shfl_sync(0xffffffffu, slot, b);
            const int32_t* rb = s_rec[s_list[lb]];
            const int4 fxb = *reinterpret_cast<const int4*>(rb + ER_FX);
            const int4 ftb = *reinterpret_cast<const int4*>(rb + ER_FT);
            const int nx = fxb.y, ny = fxb.w, nta = ftb.w;
            const int g0 = lpb * EB_MQ;
            const int cntb = min(EB_MQ, rb[ER_PTOT] - g0), cptb = (cntb + 3) & ~3;
            const QuadRule qr{rb[ER_M], rb[6], rb[ER_GOFF], __int_as_float(rb[ER_INVNP])};
            const int ncell = nx + ny + nta + 3;
            for (int r0 = 0; r0 < ncell - 1; r0 += 31) {
              const int p = r0 + lane;
              int a, q0, first, rowb;
              if (p < nx + 1) { a = 0; q0 = p; first = I0 + fxb.x; rowb = 0; }
              else if (p < nx + ny + 2) { a = 1; q0 = p - (nx + 1); first = J0 + fxb.z; rowb = nx; }
              else { a = 2; q0 = p - (nx + ny + 2); first = K0 + ftb.z; rowb = nx + ny; }
              const int gi = first - 1 + q0;           // dual cell between grid points gi and gi + 1
              const bool wr = lane >= 1 && q0 >= 1 && p < ncell;
              // the 4-aligned tick range may reach beyond the clipped footprint: zeros there
              const bool zero = a == 2 && (gi < K0 + ftb.x || gi > K0 + ftb.y);
              effq_cells<N>(gi, rb[a], rb[3 + a], __int_as_float(rb[ER_P0 + a]), __int_as_float(rb[ER_D + a]),
                            __int_as_float(rb[ER_NK2 + a]), __int_as_float(rb[ER_K]), a == 0, wr, zero,
                            sbase + slotb + (rowb + q0 - 1) * cptb, 1, qr, g0, cntb);
            }
          }
          __syncwarp();
          if (lane == 0 && tot) eb_mbar_expect_tx(full_bar(stage), tot);
          __syncwarp();
          if (in && toff >= 0) {
            const int trs = rec[ER_TRS];
            const float* G = gtab + 4 * (int64_t)toff + (int64_t)lp * EB_MQ * trs;
            float* D = sbase + slot;
            eb_bulk_g2s(D, G + rec[ER_TROW + 0] * cpt, (uint32_t)(fx.y * cpt * 4), full_bar(stage));
            eb_bulk_g2s(D + fx.y * cpt, G + rec[ER_TROW + 1] * cpt, (uint32_t)(fx.w * cpt * 4), full_bar(stage));
            eb_bulk_g2s(D + (fx.y + fx.w) * cpt, G + rec[ER_TROW + 2] * cpt, (uint32_t)(ft.w * cpt * 4), full_bar(stage));
          }
          if (++stage == EB_STAGES) { stage = 0; sphase ^= 1; }
        }
      }
    }
    // end of the tile: its last stage carries the flag (an empty one if the tile had no pass)
    __syncwarp();
    if (pend_stage < 0) {
      if (lane == 0) eb_mbar_wait(empty_bar(stage), sphase ^ 1);
      pend_stage = stage; pend_n = 0;
      if (++stage == EB_STAGES) { stage = 0; sphase ^= 1; }
    }
    hand_over(EB_LAST);
    }
  } else {
    // ================================================================ consumers
    // what this warp owns: rows [wi0, wi0 + wi) x columns-in-a-row [wj0, wj0 + wj) x ticks [wt0, wt0 + wt)
    const int wjj = warp % P.nwj, wrest = warp / P.nwj;
    const int wii = wrest % P.nwi, wtt = wrest / P.nwi;
    const int wi0 = wii * P.wi, wj0 = wjj * P.wj, wt0 = wtt * P.wt;
    int stage = 0, sphase = 0;
    for (int64_t tile_id = blockIdx.x; tile_id < ntiles; tile_id += gridDim.x) {
    for (;;) {
      eb_mbar_wait(full_bar(stage), sphase);
      const int nflag = s_n[stage];
      const int n = nflag & (EB_LAST - 1);
      const float* sbase = ring + stage * EB_STAGE_FLOATS;
      for (int pl = 0; pl < n; ++pl) {
        const int32_t* d = s_desc[stage][pl];
        const int4 fx = *reinterpret_cast<const int4*>(d);
        const int4 ft = *reinterpret_cast<const int4*>(d + 4);
        const int ia = max(fx.x, wi0), ib = min(fx.x + fx.y, wi0 + P.wi);
        const int ja = max(fx.z, wj0), jb = min(fx.z + fx.w, wj0 + P.wj);
        const int ka = max(ft.z, wt0), kb = min(ft.z + ft.w, wt0 + P.wt);
        if (ia < ib && ja < jb && ka < kb) {
          const int4 dd = *reinterpret_cast<const int4*>(d + 8);        // cnt, cpt, slot
          const int cnt = dd.x, cpt = dd.y;
          const float* S = sbase + dd.z;
          const int nj = jb - ja;
          const int rows_it = nj >= 32 ? 1 : 32 / nj;                   // rows of the rectangle dealt at once
          const float rnj = __frcp_rn((float)nj);
          for (int i0 = ia; i0 < ib; i0 += rows_it) {
            const int ni = min(rows_it, ib - i0), nc = ni * nj;
            const int G = 32 / nc;                                       // lane groups: tick quads round-robin
            const int grp = (int)(((float)lane + 0.5f) * __frcp_rn((float)nc));
            const int c = lane - grp * nc;
            const int ii = (int)(((float)c + 0.5f) * rnj);
            const int jj = c - ii * nj;
            if (grp < G) {
              const int ci = i0 + ii, cj = ja + jj;
              float* tcol = tile + (size_t)((ci << P.by_shift) + cj) * P.CS;
              const float* X = S + (ci - fx.x) * cpt;
              const float* Y = S + (fx.y + cj - fx.z) * cpt;
              const float* T = S + (fx.y + fx.w - ft.z) * cpt;           // row of tile-relative tick 0
              const int k0 = ka + 4 * grp, ks = 4 * G;
              switch (cnt) {
                case 1: effq_blk_update<1>(tcol, X, Y, T, k0, kb, ks); break;
                case 2: effq_blk_update<2>(tcol, X, Y, T, k0, kb, ks); break;
                case 3: effq_blk_update<3>(tcol, X, Y, T, k0, kb, ks); break;
                case 4: effq_blk_update<4>(tcol, X, Y, T, k0, kb, ks); break;
                case 5: effq_blk_update<5>(tcol, X, Y, T, k0, kb, ks); break;
                case 6: effq_blk_update<6>(tcol, X, Y, T, k0, kb, ks); break;
                case 7: effq_blk_update<7>(tcol, X, Y, T, k0, kb, ks); break;
                case 8: effq_blk_update<8>(tcol, X, Y, T, k0, kb, ks); break;
                case 9: effq_blk_update<9>(tcol, X, Y, T, k0, kb, ks); break;
                case 10: effq_blk_update<10>(tcol, X, Y, T, k0, kb, ks); break;
                case 11: effq_blk_update<11>(tcol, X, Y, T, k0, kb, ks); break;
                default: effq_blk_update<12>(tcol, X, Y, T, k0, kb, ks); break;
              }
            }
          }
          __syncwarp();                                // the next pass deals the cells to other lanes
        }
      }
      __syncwarp();
      if (lane == 0) eb_mbar_arrive(empty_bar(stage));
      if (++stage == EB_STAGES) { stage = 0; sphase ^= 1; }
      if (nflag & EB_LAST) break;
    }
    // tile -> payload[blk][col][sub * TS + k] (float4 copies, TS floats contiguous per column),
    // clearing the tile for the next one on the way
    asm volatile("bar.sync 1, %0;" ::"r"(nct) : "memory");
    {
      const int64_t blk = tile_id / P.nsub;
      const int sub = (int)(tile_id - blk * P.nsub);
      float* out = payload + blk * P.ncol * g.Bt + sub * P.TS;
      const int qs = P.ts_shift - 2;                              // float4 per column = 1 << qs
      const int kq = threadIdx.x & ((1 << qs) - 1), c0 = threadIdx.x >> qs, cstep = nct >> qs;
      float4* tp = reinterpret_cast<float4*>(tile + (size_t)c0 * P.CS) + kq;
      float4* op = reinterpret_cast<float4*>(out + (int64_t)c0 * g.Bt) + kq;
      const int tstep = (cstep * P.CS) >> 2;
      const int64_t ostep = ((int64_t)cstep * g.Bt) >> 2;
#pragma unroll 4
      for (int c = c0; c < P.ncol; c += cstep, tp += tstep, op += ostep) {
        *op = *tp;
        *tp = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
      }
    }
    asm volatile("bar.sync 1, %0;" ::"r"(nct) : "memory");
    }
  }
}

// Gauss-Legendre nodes / weights of the m-point rule on [-1,1] by Newton iteration on
// P_m (fp64, host); textbook algorithm (e.g. Numerical Recipes "gauleg").
void gauleg(int m, double* x, double* w) {
  for (int i = 0; i < (m + 1) / 2; ++i) {
    double z = cos(3.14159265358979323846 * (i + 0.75) / (m + 0.5)), pp = 1.0;
    for (int itn = 0; itn < 100; ++itn) {
      double p1 = 1.0, p2 = 0.0;
      for (int j = 1; j <= m; ++j) { const double p3 = p2; p2 = p1; p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j; }
      pp = m * (z * p1 - p2) / (z * z - 1.0);
      const double z1 = z;
      z = z1 - p1 / pp;
      if (fabs(z - z1) < 1e-15) break;
    }
    x[i] = -z; x[m - 1 - i] = z;
    w[i] = w[m - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
  }
}

}  // namespace

int tred_effq_init_tables(void) {
  float hs[NGL], hw[NGL];
  double x[MMAX], w[MMAX];
  for (int m = 1; m <= MMAX; ++m) {
    gauleg(m, x, w);
    for (int i = 0; i < m; ++i) {
      hs[m * (m - 1) / 2 + i] = (float)(0.5 * (x[i] + 1.0));
      hw[m * (m - 1) / 2 + i] = (float)(0.5 * w[i]);
    }
  }
  TRED_CUDA(cudaMemcpyToSymbol(c_gl_s, hs, sizeof(hs)));
  TRED_CUDA(cudaMemcpyToSymbol(c_gl_w, hw, sizeof(hw)));
  return TRED_OK;
}

// ------------------------------------------------------------------ N4: truth record
// "segment-id -> charge per (channel, short time slice)".  Reading G24:
// the effective charge of segment s summed over the grid points of every pixel and time tile
// (Bt ticks) its clipped footprint [lo - e, hi + e] reaches.  With the factored form of the
// charge the sum over a pixel x tile box factors too:
//   Q[s][px][py][tb] = sum_m (K W_m sum_{i in px} GX_m[i]) (sum_{j in py} GY_m[j]) (sum_{k in tb} GT_m[k]).
constexpr int TR_MAXG = 32;          // pixel / tile groups per axis a segment may reach (more: reported, see tred_truth)

struct TruthBox { int lo[3], hi[3], g0[3], ng[3]; };

__device__ __forceinline__ bool truth_box(const int32_t* __restrict__ augi, int64_t nseg, int64_t s, const TredGrid& g,
                                          int E, TruthBox& b, bool* over = nullptr) {
  const int NG[3] = {g.NGx, g.NGy, g.NGt}, div[3] = {g.S, g.S, g.Bt};
  bool ok = true;
  for (int a = 0; a < 3; ++a) {
    b.lo[a] = max(augi[a * nseg + s] - E, 0);
    b.hi[a] = min(augi[(3 + a) * nseg + s] + E, NG[a] - 1);
    ok = ok && b.lo[a] <= b.hi[a];
    b.g0[a] = b.lo[a] / div[a];
    b.ng[a] = ok ? min(b.hi[a] / div[a] - b.g0[a] + 1, TR_MAXG) : 0;
    if (over && ok && b.hi[a] / div[a] - b.g0[a] + 1 > TR_MAXG) *over = true;
  }
  return ok;
}

template <int N>
__global__ void __launch_bounds__(256)
k_truth_count(int64_t nseg, const int32_t* __restrict__ augi, TredGrid g, int32_t* __restrict__ cnt,
              int32_t* __restrict__ over_flag) {
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s > nseg) return;
  int c = 0;
  if (s < nseg) {
    TruthBox b;
    bool over = false;
    if (truth_box(augi, nseg, s, g, N > 1 ? 1 : 0, b, &over)) c = b.ng[0] * b.ng[1] * b.ng[2];
    if (over) atomicOr(over_flag, 1);            // a segment reaches more groups than a record holds
  }
  cnt[s] = c;
}

// one warp per segment
template <int N>
__global__ void __launch_bounds__(128)
k_truth_fill(int64_t nseg, const float* __restrict__ augf, const int32_t* __restrict__ augi,
             const int32_t* __restrict__ first, TredGrid g, int64_t cap, int32_t* __restrict__ rec_seg,
             int64_t* __restrict__ rec_key, float* __restrict__ rec_q, int64_t* __restrict__ d_nrec,
             const int32_t* __restrict__ over_flag) {
  __shared__ float sums[4][3 * TR_MAXG][MMAX];
  const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t s = (int64_t)blockIdx.x * 4 + wid;
  if (blockIdx.x == 0 && threadIdx.x == 0) *d_nrec = *over_flag ? -1 : (int64_t)first[nseg];
  if (s >= nseg) return;
  constexpr int E = N > 1 ? 1 : 0;
  constexpr float LOG2E_HALF = 0.72134752044448170f;
  TruthBox b;
  if (!truth_box(augi, nseg, s, g, E, b)) return;
  const int nrec = b.ng[0] * b.ng[1] * b.ng[2];
  const int64_t f0 = first[s];
  const int lo3[3] = {augi[0 * nseg + s], augi[1 * nseg + s], augi[2 * nseg + s]};
  const int hi3[3] = {augi[3 * nseg + s], augi[4 * nseg + s], augi[5 * nseg + s]};
  const int flag = augi[6 * nseg + s];
  const float p0[3] = {augf[0 * nseg + s], augf[1 * nseg + s], augf[2 * nseg + s]};
  const float d3[3] = {augf[3 * nseg + s] - p0[0], augf[4 * nseg + s] - p0[1], augf[5 * nseg + s] - p0[2]};
  const float sg[3] = {augf[6 * nseg + s], augf[7 * nseg + s], augf[8 * nseg + s]};
  const float Qp = augf[9 * nseg + s];
  const float k2[3] = {LOG2E_HALF / (sg[0] * sg[0]), LOG2E_HALF / (sg[1] * sg[1]), LOG2E_HALF / (sg[2] * sg[2])};
  const float K = Qp * 0.063493635934240969f / (sg[0] * sg[1] * sg[2]) * 0.125f;
  const SegQuad q = seg_quad(flag, d3[0], d3[1], d3[2], sg[0], sg[1], sg[2]);
  const int m = q.m, goff = m * (m - 1) / 2;
  const float inv_np = 1.0f / (float)q.npiece;
  const int div[3] = {g.S, g.S, g.Bt};
  float (*S)[MMAX] = sums[wid];
  float acc = 0.0f;                                       // record `lane` (+ 32, ... handled below)
  const int ngt = b.ng[0] + b.ng[1] + b.ng[2];
  for (int r0 = 0; r0 < nrec; r0 += 32) {                 // 32 records at a time (usually one round)
    acc = 0.0f;
    for (int pc = 0; pc < q.npiece; ++pc) {
      __syncwarp();
      // group sums: lane -> (group, mi), grid points of the group summed in ascending order
      for (int e = lane; e < ngt * m; e += 32) {
        const int gi = e / m, mi = e - gi * m;
        const int a = gi < b.ng[0] ? 0 : gi < b.ng[0] + b.ng[1] ? 1 : 2;
        const int gl = gi - (a == 0 ? 0 : a == 1 ? b.ng[0] : b.ng[0] + b.ng[1]);
        float sk, wk;
        if (flag) { sk = 0.5f; wk = mi == 0 ? 1.0f : 0.0f; }
        else { sk = ((float)pc + c_gl_s[goff + mi]) * inv_np; wk = c_gl_w[goff + mi] * inv_np; }
        const float c = fmaf(sk, d3[a], p0[a]);
        const int i0 = max((b.g0[a] + gl) * div[a], b.lo[a]), i1 = min((b.g0[a] + gl + 1) * div[a] - 1, b.hi[a]);
        float v = 0.0f;
        for (int i = i0; i <= i1; ++i) v += axis_entry<N>(i, lo3[a], hi3[a], c, k2[a]);
        S[gi][mi] = a == 0 ? v * (K * wk) : v;
      }
      __syncwarp();
      const int rr = r0 + lane;
      if (rr < nrec) {
        const int gy = rr % b.ng[1], gx = (rr / b.ng[1]) % b.ng[0], gt = rr / (b.ng[1] * b.ng[0]);
        const float* sx = S[gx];
        const float* sy = S[b.ng[0] + gy];
        const float* stt = S[b.ng[0] + b.ng[1] + gt];
        float v = 0.0f;
        for (int mi = 0; mi < m; ++mi) v = fmaf(sx[mi] * sy[mi], stt[mi], v);
        acc += v;
      }
    }
    const int rr = r0 + lane;
    if (rr < nrec && f0 + rr < cap) {
      const int gy = rr % b.ng[1], gx = (rr / b.ng[1]) % b.ng[0], gt = rr / (b.ng[1] * b.ng[0]);
      rec_seg[f0 + rr] = (int32_t)s;
      rec_key[f0 + rr] = ((int64_t)(b.g0[2] + gt) * g.npx + (b.g0[0] + gx)) * g.npy + (b.g0[1] + gy);
      rec_q[f0 + rr] = acc;
    }
  }
}



struct EffqWork { int32_t* off; void* scan; int64_t* total; float* tab; int64_t cap16; size_t fixed; };

static EffqWork carve_effq(void* base, int64_t nseg, size_t work_bytes) {
  EffqWork w;
  size_t o = 0; char* b = (char*)base;
  auto take = [&](size_t bytes) { void* p = b ? b + o : nullptr; o += align_up(bytes, 256); return p; };
  w.off = (int32_t*)take((size_t)(nseg + 1) * 4);
  w.scan = take(tred_scan_work_bytes(nseg + 1));
  w.total = (int64_t*)take(sizeof(int64_t));
  w.fixed = o;
  w.tab = (float*)(b ? b + o : nullptr);
  w.cap16 = work_bytes > o ? (int64_t)((work_bytes - o) / 16) : 0;
  if (w.cap16 > 0x7fffffff) w.cap16 = 0x7fffffff;              // offsets are int32, in 16-byte units
  return w;
}

// Workspace for the per-segment tables: the fixed part plus ~2 KB per segment (a segment of the
// paper's workloads needs 1-1.5 KB), at most 4 GiB.  Less is allowed: segments whose tables do not
// fit are evaluated by the tile CTAs themselves.
extern "C" size_t tred_effq_work_bytes(const tred_ctx* ctx, int64_t nseg) {
  if (!ctx || nseg < 0) return 0;
  size_t t = (size_t)nseg * 2048;
  if (t > ((size_t)4 << 30)) t = (size_t)4 << 30;
  return carve_effq(nullptr, nseg, 0).fixed + t;
}

// shape of the tile kernel for this configuration; false if the block shape is outside what it
// supports (then the closed-form kernel runs)
static bool effq_blk_shape(const tred_ctx* ctx, const TredGrid& g, BlkParams& P, int& threads, size_t& smem) {
  const int ncol = g.Bx * g.By;
  if (ncol < 16 || ncol > 1024 || g.Bt < 4 || ((g.Bx + g.By) & 3)) return false;
  P.ncol = ncol;
  P.by_shift = 0;
  while ((1 << P.by_shift) < g.By) ++P.by_shift;
  // 1024-column blocks run one CTA per SM and may use most of its shared memory
  const size_t budget = ncol >= 1024 ? 150 * 1024 : 72 * 1024;
  int TS = g.Bt;
  while (TS > 4 && (size_t)ncol * (TS + 4) * sizeof(float) > budget) TS /= 2;
  P.TS = TS; P.nsub = g.Bt / TS;
  P.ts_shift = 0;
  while ((1 << P.ts_shift) < TS) ++P.ts_shift;
  P.CS = TS + 4;
  P.RS = g.Bx + g.By + TS;
  if (P.RS * EB_MQ + 256 > EB_STAGE_FLOATS) return false;      // a stage holds any one pass and then some
  // consumer warps: 32 (16 for a 4x4 block, 64 for 1024 columns) columns each, as wi rows x wj
  // columns of a row
  const int wcols = ncol >= 1024 ? 64 : ncol >= 32 ? 32 : ncol;
  P.wj = g.By < wcols ? g.By : wcols;
  P.wi = wcols / P.wj;
  P.nwj = g.By / P.wj;
  P.nwi = g.Bx / P.wi;
  int nwarps = P.nwj * P.nwi;                       // one tick range
  int nparts = 1;
  while (nwarps * nparts * 2 <= 8 && TS / (nparts * 2) >= 4) nparts *= 2;
  P.wt = TS / nparts;
  P.ncw = nwarps * nparts;
  threads = (P.ncw + 1) * 32;
  if (threads > 1024) return false;
  smem = ((size_t)ncol * P.CS + (size_t)EB_STAGES * EB_STAGE_FLOATS) * sizeof(float) + (size_t)EB_SB * EB_NREC * 4;
  return smem <= (size_t)ctx->smem_optin;
}

template <int N>
static int effq_launch(tred_ctx* ctx, const TredGrid& g, BlkParams P, int threads, size_t smem, int64_t nseg,
                       int64_t nblocks, const int64_t* d_keys, const int32_t* d_blk_off, const int32_t* d_pair_seg,
                       const float* d_augf, const int32_t* d_augi, float* d_payload, void* d_work, size_t work_bytes,
                       cudaStream_t st) {
  EffqWork w = carve_effq(d_work, nseg, work_bytes);
  // few blocks: the four extra launches cost more than the tables save
  const bool tables = d_work && w.cap16 >= 4096 && nseg > 0 && nblocks >= 1024;
  P.cap16 = tables ? w.cap16 : 0;
  P.tab_total = w.total;
  if (tables) {
    TRED_CUDA(cudaMemsetAsync(w.off, 0, (size_t)(nseg + 1) * 4, st));
    k_effq_mark<<<cdiv(nblocks * 32, 256), 256, 0, st>>>(nblocks, d_blk_off, d_pair_seg, w.off);
    TRED_CUDA(cudaMemsetAsync(w.total, 0, sizeof(int64_t), st));
    k_effq_sizes<N><<<cdiv(nseg + 1, 256), 256, 0, st>>>(nseg, d_augf, d_augi, w.off, (unsigned long long*)w.total);
    int rc = tred_exclusive_scan_i32(w.off, w.off, nseg + 1, nullptr, w.scan, st);
    if (rc != TRED_OK) return rc;
    k_effq_tables<N><<<cdiv(nseg, 128), 128, 0, st>>>(nseg, w.off, w.total, w.cap16, d_augf, d_augi, w.tab, g);
    TRED_COUNT_LAUNCH(5);
  }
  const int32_t* tabofs = tables ? w.off : nullptr;
  // persistent CTAs: as many as are resident at once
  const int64_t ntiles = nblocks * P.nsub;
  const int per_sm = threads > 512 ? 1 : (int)((size_t)ctx->smem_sm / (smem + 4096) < 1 ? 1 : (size_t)ctx->smem_sm / (smem + 4096));
  int64_t grid64 = (int64_t)ctx->num_sms * (per_sm > 4 ? 4 : per_sm);
  if (grid64 > ntiles) grid64 = ntiles;
  const unsigned grid = (unsigned)grid64;
  if (threads > 288) {
    TRED_CUDA(cudaFuncSetAttribute(k_effq_blk<N, 1024>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_effq_blk<N, 1024><<<grid, threads, smem, st>>>(
        nseg, d_keys, d_blk_off, d_pair_seg, d_augf, d_augi, tabofs, w.tab, d_payload, ntiles, g, P);
  } else {
    TRED_CUDA(cudaFuncSetAttribute(k_effq_blk<N, 288>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k_effq_blk<N, 288><<<grid, threads, smem, st>>>(
        nseg, d_keys, d_blk_off, d_pair_seg, d_augf, d_augi, tabofs, w.tab, d_payload, ntiles, g, P);
  }
  TRED_COUNT_LAUNCH(1);
  TRED_LAUNCH_CHECK("k_effq_blk");
  return TRED_OK;
}

extern "C" int tred_effq(tred_ctx* ctx, int64_t nseg, int64_t nblocks,
                         const int64_t* d_keys, const int32_t* d_blk_off, const int32_t* d_pair_seg,
                         const float* d_augf, const int32_t* d_augi,
                         float* d_payload, void* d_work, size_t work_bytes, void* stream) {
  if (!ctx || nseg < 0 || nblocks < 0) return TRED_EINVAL;
  TRED_CHECK_DEVICE(ctx);
  if (nblocks == 0) return TRED_OK;
  if (!d_keys || !d_blk_off || !d_pair_seg || !d_augf || !d_augi || !d_payload) return TRED_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  if (ctx->cfg.effq_mode != 0 && ctx->cfg.effq_mode != 1) return TRED_EINVAL;
  const TredGrid g = make_grid(ctx);
  BlkParams P;
  int threads = 0;
  size_t smem = 0;
  if (ctx->cfg.effq_mode == 1 || !effq_blk_shape(ctx, g, P, threads, smem))
    return tred_effq_closed_form(ctx, nseg, nblocks, d_keys, d_blk_off, d_pair_seg, d_augf, d_augi,
                                 d_payload, st);
  if (nblocks * P.nsub >= (1ll << 31)) return TRED_EUNSUPPORTED;
  TredProfScope ps(ctx, ST_EFFQ, st);
  switch (g.gl_n) {
    case 1: return effq_launch<1>(ctx, g, P, threads, smem, nseg, nblocks, d_keys, d_blk_off, d_pair_seg, d_augf,
                                  d_augi, d_payload, d_work, work_bytes, st);
    case 2: return effq_launch<2>(ctx, g, P, threads, smem, nseg, nblocks, d_keys, d_blk_off, d_pair_seg, d_augf,
                                  d_augi, d_payload, d_work, work_bytes, st);
    case 3: return effq_launch<3>(ctx, g, P, threads, smem, nseg, nblocks, d_keys, d_blk_off, d_pair_seg, d_augf,
                                  d_augi, d_payload, d_work, work_bytes, st);
    case 4: return effq_launch<4>(ctx, g, P, threads, smem, nseg, nblocks, d_keys, d_blk_off, d_pair_seg, d_augf,
                                  d_augi, d_payload, d_work, work_bytes, st);
    default: return TRED_EINVAL;
  }
}

extern "C" size_t tred_truth_work_bytes(const tred_ctx* ctx, int64_t nseg) {
  if (!ctx || nseg < 0) return 0;
  return align_up((size_t)(nseg + 1) * 4, 256) + tred_scan_work_bytes(nseg + 1) + 256;
}

extern "C" int tred_truth(tred_ctx* ctx, int64_t nseg, const float* d_augf, const int32_t* d_augi, int64_t cap_rec,
                          int32_t* d_rec_seg, int64_t* d_rec_key, float* d_rec_q, int64_t* d_nrec, void* d_work,
                          size_t work_bytes, void* stream) {
  if (!ctx || nseg < 0 || cap_rec < 0 || !d_nrec) return TRED_EINVAL;
  TRED_CHECK_DEVICE(ctx);
  cudaStream_t st = (cudaStream_t)stream;
  if (nseg == 0) { TRED_CUDA(cudaMemsetAsync(d_nrec, 0, sizeof(int64_t), st)); return TRED_OK; }
  if (!d_augf || !d_augi || !d_work) return TRED_EINVAL;
  if (work_bytes < tred_truth_work_bytes(ctx, nseg)) return TRED_ECAP;
  if (cap_rec > 0 && (!d_rec_seg || !d_rec_key || !d_rec_q)) return TRED_EINVAL;
  const TredGrid g = make_grid(ctx);
  int32_t* first = (int32_t*)d_work;
  void* scan = (char*)d_work + align_up((size_t)(nseg + 1) * 4, 256);
  int32_t* over = (int32_t*)((char*)scan + tred_scan_work_bytes(nseg + 1));
  TRED_CUDA(cudaMemsetAsync(over, 0, 4, st));
#define TRUTH(NN)                                                                                          \
  do {                                                                                                     \
    k_truth_count<NN><<<cdiv(nseg + 1, 256), 256, 0, st>>>(nseg, d_augi, g, first, over);                  \
    int rc = tred_exclusive_scan_i32(first, first, nseg + 1, nullptr, scan, st);                           \
    if (rc != TRED_OK) return rc;                                                                          \
    k_truth_fill<NN><<<cdiv(nseg, 4), 128, 0, st>>>(nseg, d_augf, d_augi, first, g, cap_rec, d_rec_seg,     \
                                                    d_rec_key, d_rec_q, d_nrec, over);                     \
  } while (0)
  switch (g.gl_n) {
    case 1: TRUTH(1); break;
    case 2: TRUTH(2); break;
    case 3: TRUTH(3); break;
    case 4: TRUTH(4); break;
    default: return TRED_EINVAL;
  }
#undef TRUTH
  TRED_COUNT_LAUNCH(2);
  TRED_LAUNCH_CHECK("tred_truth");
  return TRED_OK;
}
