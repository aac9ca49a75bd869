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
// One CTA per block tile (all of Bx x By, TS ticks) staged in shared memory.  Per segment
// of the block: phase A builds the three tables (double-buffered), one __syncthreads,
// phase B adds the rank-m product into the tile, one thread per (column, tick chunk).
// No atomics; the summation order is fixed (segments ascending), so results are
// deterministic.
#include <math.h>
#include "tred_common.cuh"

namespace {

constexpr int MMAX = 24;            // quadrature points per pass
constexpr int MP = MMAX + 4;        // table row pitch (floats): conflict-free LDS.128
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

struct FactParams {
  int TS;        // ticks per CTA tile
  int nsub;      // Bt / TS
  int plane;     // Bx*By + 1
};

// One table entry: grid point gi of one axis, quadrature centre c (grid units relative to
// lo), k2 = log2(e) / (2 sigma^2).
// Contributions of the n nodes of dual cell gi (between grid points gi and gi + 1) to the
// table entries of gi (coefficient 1 - s) and of gi + 1 (coefficient s): the same n
// exponentials serve both, so a row of entries costs n, not 2n, exponentials per entry
// (entry(gi) = own(gi) + up(gi - 1)); same arithmetic per term as axis_entry.
template <int N>
__device__ __forceinline__ void axis_cell(int gi, int lo, int hi, float c, float k2, float& own, float& up) {
  own = 0.0f; up = 0.0f;
  const float base = (float)(gi - lo) + 0.5f;
#pragma unroll
  for (int q = 0; q < N; ++q) {
    const float sq = DualGL<N>::s(q), wq = DualGL<N>::w(q);
    const int cub = gi + DualGL<N>::side(q);
    const float z = (base + sq) - c;
    const float e = ex2_approx(-z * z * k2);
    if (cub >= lo && cub <= hi) {
      own = fmaf(wq * (1.0f - sq), e, own);
      if (sq != 0.0f) up = fmaf(wq * sq, e, up);
    }
  }
}

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

// ------------------------------------------------------------------ tables built once
// A segment meets ~4 blocks x 2 tick sub-tiles, and every such CTA would rebuild the same
// three per-axis tables (8 ex2 per entry for n = 4): ncu showed the tile kernel issue-bound
// on exactly that.  So the tables of the segments a range of blocks refers to are built once
// (k_effq_tables) into a slot of TAB_ROWS x TAB_M floats and the tile kernel copies the rows
// it needs.  Segments that do not fit a slot (more than TAB_M quadrature points, several
// pieces, a bounding box of more than TAB_ROWS grid rows in total, or no free slot) are
// evaluated in the tile kernel as before.
constexpr int TAB_M = 12;
constexpr int TAB_ROWS = 96;
constexpr int TAB_FLOATS = TAB_ROWS * TAB_M;
constexpr int64_t EFFQ_MAX_SLOTS = 1 << 18;          // 262144 slots = 1.2 GB of tables at most
constexpr int EFFQ_RANGE_BLOCKS = 8192;              // blocks per pass of (mark, tables, tiles)

// Quadrature of a segment record: number of pieces and points per piece from its length
// in sigmas (same arithmetic wherever it is needed).
struct SegQuad { int npiece, m; };
__device__ __forceinline__ SegQuad seg_quad(int flag, float dx, float dy, float dt, float sx, float sy, float st) {
  SegQuad q;
  q.npiece = 1; q.m = 4;
  if (!flag) {
    const float W = sqrtf((dx / sx) * (dx / sx) + (dy / sy) * (dy / sy) + (dt / st) * (dt / st));
    q.npiece = (int)ceilf(W * (1.0f / 15.5f));
    if (q.npiece < 1) q.npiece = 1;
    const float Wp = W / (float)q.npiece;
    q.m = Wp <= 1.0f ? 4 : Wp <= 3.9f ? 8 : Wp <= 6.9f ? 12 : Wp <= 9.9f ? 16 : Wp <= 12.8f ? 20 : 24;
  }
  return q;
}

// marks the segments the blocks [k0, k0 + nb) refer to (idempotent plain stores)
__global__ void __launch_bounds__(256)
k_effq_mark(int nb, int k0, const int32_t* __restrict__ blk_off, const int32_t* __restrict__ pair_seg,
            int32_t* __restrict__ mark) {
  const int warp = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
  if (warp >= nb) return;
  const int p0 = blk_off[k0 + warp], p1 = blk_off[k0 + warp + 1];
  for (int p = p0 + lane; p < p1; p += 32) mark[pair_seg[p]] = 1;
}

// slot[] = exclusive scan of the marks; lists the marked segments and resets tabslot
__global__ void __launch_bounds__(256)
k_effq_list(int64_t nseg, const int32_t* __restrict__ slot, int32_t* __restrict__ seglist, int cap,
            int32_t* __restrict__ tabslot) {
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= nseg) return;
  const int sl = slot[s];
  const bool marked = slot[s + 1] != sl;
  if (marked && sl < cap) seglist[sl] = (int32_t)s;
  tabslot[s] = -1;
}

// One warp per listed segment: the three tables of its bounding box (grid points
// lo - E .. hi + E per axis), rows of TAB_M floats, X rows first (with K W_k folded in),
// then Y, then T.
template <int N>
__global__ void __launch_bounds__(128)
k_effq_tables(int64_t nseg, const int32_t* __restrict__ slot, const int32_t* __restrict__ seglist, int cap,
              const float* __restrict__ augf, const int32_t* __restrict__ augi, float* __restrict__ tab,
              int32_t* __restrict__ tabslot) {
  const int sl = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  const int total = min(slot[nseg], cap);
  if (sl >= total) return;
  const int64_t s = seglist[sl];
  constexpr int E = N > 1 ? 1 : 0;
  constexpr float LOG2E_HALF = 0.72134752044448170f;
  const int lox = augi[0 * nseg + s], loy = augi[1 * nseg + s], lot = augi[2 * nseg + s];
  const int hix = augi[3 * nseg + s], hiy = augi[4 * nseg + s], hit = augi[5 * nseg + s];
  const int flag = augi[6 * nseg + s];
  const float p0x = augf[0 * nseg + s], p0y = augf[1 * nseg + s], p0t = augf[2 * nseg + s];
  const float p1x = augf[3 * nseg + s], p1y = augf[4 * nseg + s], p1t = augf[5 * nseg + s];
  const float sx = augf[6 * nseg + s], sy = augf[7 * nseg + s], st = augf[8 * nseg + s];
  const float Qp = augf[9 * nseg + s];
  const float dx = p1x - p0x, dy = p1y - p0y, dt = p1t - p0t;
  const SegQuad q = seg_quad(flag, dx, dy, dt, sx, sy, st);
  const int nxf = hix - lox + 1 + 2 * E, nyf = hiy - loy + 1 + 2 * E, ntf = hit - lot + 1 + 2 * E;
  if (q.npiece != 1 || q.m > TAB_M || nxf + nyf + ntf > TAB_ROWS) return;      // tile kernel evaluates it
  const float k2x = LOG2E_HALF / (sx * sx), k2y = LOG2E_HALF / (sy * sy), k2t = LOG2E_HALF / (st * st);
  const float K = Qp * 0.063493635934240969f / (sx * sy * st) * 0.125f;
  const int m = q.m, goff = m * (m - 1) / 2;
  float* T = tab + (int64_t)sl * TAB_FLOATS;
  const int nent = (nxf + nyf + ntf) * TAB_M;
  for (int e = lane; e < nent; e += 32) {
    const int r = e / TAB_M, mi = e - r * TAB_M;
    float v = 0.0f;
    if (mi < m) {
      float sk, wk;
      if (flag) { sk = 0.5f; wk = mi == 0 ? 1.0f : 0.0f; }
      else { sk = c_gl_s[goff + mi]; wk = c_gl_w[goff + mi]; }
      if (r < nxf) v = axis_entry<N>(lox - E + r, lox, hix, fmaf(sk, dx, p0x), k2x) * (K * wk);
      else if (r < nxf + nyf) v = axis_entry<N>(loy - E + (r - nxf), loy, hiy, fmaf(sk, dy, p0y), k2y);
      else v = axis_entry<N>(lot - E + (r - nxf - nyf), lot, hit, fmaf(sk, dt, p0t), k2t);
    }
    T[e] = v;
  }
  if (lane == 0) tabslot[s] = sl;
}

// Phase B of one (segment, piece): tile[k][i][j] += sum_mi GX[i][mi] GY[j][mi] GT[k][mi] over
// the clipped footprint.  A thread owns one column (and one tick chunk of it); the products
// GX GY of its column stay in registers (MQ = m / 4 float4), every tile value is read and
// written once per piece.
template <int MQ>
__device__ __forceinline__ void effq_phase_b(float* __restrict__ tp, int plane, const float* __restrict__ GXr,
                                             const float* __restrict__ GYr, const float* __restrict__ GT,
                                             int ka, int kb) {
  float4 ab[MQ];
#pragma unroll
  for (int q = 0; q < MQ; ++q) {
    const float4 a = *reinterpret_cast<const float4*>(GXr + 4 * q);
    const float4 b = *reinterpret_cast<const float4*>(GYr + 4 * q);
    ab[q] = make_float4(a.x * b.x, a.y * b.y, a.z * b.z, a.w * b.w);
  }
#pragma unroll 2
  for (int k = ka; k < kb; ++k) {
    float v = tp[k * plane];
#pragma unroll
    for (int q = 0; q < MQ; ++q) {
      const float4 c = *reinterpret_cast<const float4*>(GT + k * MP + 4 * q);
      v = fmaf(ab[q].x, c.x, v); v = fmaf(ab[q].y, c.y, v);
      v = fmaf(ab[q].z, c.z, v); v = fmaf(ab[q].w, c.w, v);
    }
    tp[k * plane] = v;
  }
}

#ifndef TRED_EFFQ_MINB
#define TRED_EFFQ_MINB 4            // resident CTAs per SM the register allocation aims at
#endif
#ifndef TRED_EFFQ_TILE_KB
#define TRED_EFFQ_TILE_KB 64        // largest tile (floats x 4) a CTA stages
#endif

#ifndef TRED_EFFQ_THREADS
#define TRED_EFFQ_THREADS 256       // largest CTA
#endif

template <int N>
__global__ void __launch_bounds__(TRED_EFFQ_THREADS, TRED_EFFQ_MINB)
k_effq_fact(int64_t nseg, const int64_t* __restrict__ keys, const int32_t* __restrict__ blk_off,
            const int32_t* __restrict__ pair_seg, const float* __restrict__ augf,
            const int32_t* __restrict__ augi, const int32_t* __restrict__ tabslot,
            const float* __restrict__ tab, float* __restrict__ payload, TredGrid g, FactParams P) {
  extern __shared__ float smf[];
  float* tile = smf;                                   // [TS][plane]
  const int tabn = (g.Bx + g.By + P.TS) * MP;          // floats of one table set
  float* tabs = smf + (((size_t)P.TS * P.plane + 3) & ~(size_t)3);   // 2 sets, 16-byte aligned
  const int NT = blockDim.x;
  const int blk = blockIdx.x / P.nsub;
  const int sub = blockIdx.x - blk * P.nsub;
  const int64_t key = keys[blk];
  const int by = (int)(key % g.NBy);
  const int bx = (int)((key / g.NBy) % g.NBx);
  const int bt = (int)(key / ((int64_t)g.NBy * g.NBx));
  const int I0 = bx * g.Bx, J0 = by * g.By, K0 = bt * g.Bt + sub * P.TS;
  constexpr int E = N > 1 ? 1 : 0;
  constexpr float LOG2E_HALF = 0.72134752044448170f;   // log2(e) / 2

  for (int i = threadIdx.x; i < P.TS * P.plane; i += NT) tile[i] = 0.0f;
  // the first __syncthreads of the segment loop (or the one after it) orders this

  // Segment records of the block are staged in shared memory SB at a time (one pass of
  // coalesced loads instead of two dependent global loads per segment and thread).
  constexpr int SB = 32, NF = 18;                      // 7 int fields (bbox, flag), 10 floats, table slot
  constexpr int NX = 21;    // derived once per segment: k2x, k2y, k2t, K, npiece, m, clipped box, work split
  __shared__ int32_t s_rec[SB][NF + NX + 1];
  __shared__ int s_list[SB];
  __shared__ int s_cnt;
  const int s_beg = blk_off[blk], s_end = blk_off[blk + 1];
  int it = 0;
  for (int b0 = s_beg; b0 < s_end; b0 += SB) {
  const int nbatch = min(SB, s_end - b0);
  __syncthreads();                                     // the previous batch's records are no longer read
  for (int e = threadIdx.x; e < nbatch * NF; e += NT) {
    const int j = e / NF, f = e - j * NF;
    const int64_t s = pair_seg[b0 + j];
    s_rec[j][f] = f < 7 ? augi[f * nseg + s]
                : f < 17 ? __float_as_int(augf[(f - 7) * nseg + s]) : (tabslot ? tabslot[s] : -1);
  }
  __syncthreads();
  // one lane per record: does the footprint meet this tile? per-segment constants once
  if (threadIdx.x < 32) {
    const int j = threadIdx.x;
    bool hit_tile = false;
    if (j < nbatch) {
      int32_t* rec = s_rec[j];
      hit_tile = max(rec[0] - E, I0) <= min(min(rec[3] + E, I0 + g.Bx - 1), g.NGx - 1) &&
                 max(rec[1] - E, J0) <= min(min(rec[4] + E, J0 + g.By - 1), g.NGy - 1) &&
                 max(rec[2] - E, K0) <= min(min(rec[5] + E, K0 + P.TS - 1), g.NGt - 1);
      if (hit_tile) {
        const float sx = __int_as_float(rec[13]), sy = __int_as_float(rec[14]), st = __int_as_float(rec[15]);
        const float dx = __int_as_float(rec[10]) - __int_as_float(rec[7]);
        const float dy = __int_as_float(rec[11]) - __int_as_float(rec[8]);
        const float dt = __int_as_float(rec[12]) - __int_as_float(rec[9]);
        const SegQuad q = seg_quad(rec[6], dx, dy, dt, sx, sy, st);
        rec[NF + 0] = __float_as_int(LOG2E_HALF / (sx * sx));
        rec[NF + 1] = __float_as_int(LOG2E_HALF / (sy * sy));
        rec[NF + 2] = __float_as_int(LOG2E_HALF / (st * st));
        rec[NF + 3] = __float_as_int(__int_as_float(rec[16]) * 0.063493635934240969f / (sx * sy * st) * 0.125f);
        rec[NF + 4] = q.npiece;
        rec[NF + 5] = q.m;
        // clipped footprint and the phase-B work split (ncol columns x nsplit tick chunks); item / ncolp,
        // col / ny and entry / m by multiplication: exact for arguments < 2048 and divisors <= 1024
        const int ix0 = max(rec[0] - E, I0), ix1 = min(min(rec[3] + E, I0 + g.Bx - 1), g.NGx - 1);
        const int iy0 = max(rec[1] - E, J0), iy1 = min(min(rec[4] + E, J0 + g.By - 1), g.NGy - 1);
        const int kt0 = max(rec[2] - E, K0), kt1 = min(min(rec[5] + E, K0 + P.TS - 1), g.NGt - 1);
        const int nx = ix1 - ix0 + 1, ny = iy1 - iy0 + 1, nt = kt1 - kt0 + 1;
        const int ncol = nx * ny, ncolp = (ncol + 31) & ~31;
        const int nsplit = ncolp < NT ? NT / ncolp : 1;
        rec[NF + 6] = ix0; rec[NF + 7] = nx; rec[NF + 8] = iy0; rec[NF + 9] = ny;
        rec[NF + 10] = kt0; rec[NF + 11] = nt;
        rec[NF + 12] = ncolp; rec[NF + 13] = nsplit; rec[NF + 14] = (nt + nsplit - 1) / nsplit;
        rec[NF + 15] = (65536 + ncolp - 1) / ncolp; rec[NF + 16] = (65536 + ny - 1) / ny;
        rec[NF + 17] = (65536 + q.m - 1) / q.m;
        rec[NF + 18] = q.m * (q.m - 1) / 2;
        rec[NF + 19] = __float_as_int(1.0f / (float)q.npiece);
        rec[NF + 20] = (65536 + (nx + ny + nt) - 1) / (nx + ny + nt);
      }
    }
    const uint32_t bal = __ballot_sync(0xffffffffu, hit_tile);
    if (hit_tile) s_list[__popc(bal & ((1u << j) - 1u))] = j;
    if (j == 0) s_cnt = __popc(bal);
  }
  __syncthreads();
  const int nlist = s_cnt;
  for (int sl = 0; sl < nlist; ++sl) {
    const int32_t* rec = s_rec[s_list[sl]];
    const int lox = rec[0], loy = rec[1], lot = rec[2];
    const int hix = rec[3], hiy = rec[4], hit = rec[5];
    const int flag = rec[6];
    const float p0x = __int_as_float(rec[7]), p0y = __int_as_float(rec[8]), p0t = __int_as_float(rec[9]);
    const float dx = __int_as_float(rec[10]) - p0x, dy = __int_as_float(rec[11]) - p0y,
                dt = __int_as_float(rec[12]) - p0t;
    const float k2x = __int_as_float(rec[NF + 0]), k2y = __int_as_float(rec[NF + 1]),
                k2t = __int_as_float(rec[NF + 2]), K = __int_as_float(rec[NF + 3]);
    const int npiece = rec[NF + 4], m = rec[NF + 5];
    const int slot = rec[17];
    // clipped footprint and work split, computed once per segment by the batch prologue
    const int ix0 = rec[NF + 6], nx = rec[NF + 7], iy0 = rec[NF + 8], ny = rec[NF + 9];
    const int kt0 = rec[NF + 10], nt = rec[NF + 11];
    const int ncol = nx * ny, ncolp = rec[NF + 12], nsplit = rec[NF + 13], chunk = rec[NF + 14];
    const int inv_ncolp = rec[NF + 15], inv_ny = rec[NF + 16], goff = rec[NF + 18];
    const float inv_np = __int_as_float(rec[NF + 19]);
    const int nr = nx + ny + nt, inv_nr = rec[NF + 20];

    for (int pc = 0; pc < npiece; ++pc, ++it) {
      float* GX = tabs + (it & 1) * tabn;             // [Bx][MP]
      float* GY = GX + g.Bx * MP;                     // [By][MP]
      float* GT = GY + g.By * MP;                     // [TS][MP]
      // ---- phase A: tables (copied from the segment's slot if it has one)
      const int nent = (nx + ny + nt) * m;
      if (slot >= 0) {
        const float* T = tab + (int64_t)slot * TAB_FLOATS;
        const int nxf = hix - lox + 1 + 2 * E, nyf = hiy - loy + 1 + 2 * E;
        const int rx = ix0 - (lox - E), ry = nxf + iy0 - (loy - E), rt = nxf + nyf + kt0 - (lot - E);
        constexpr int Q = TAB_M / 4;                   // float4 per table row
        for (int e = threadIdx.x; e < (nx + ny + nt) * Q; e += NT) {
          const int r = e / Q, c4 = e - r * Q;
          int src, dst;
          if (r < nx) { src = rx + r; dst = r * MP; }
          else if (r < nx + ny) { src = ry + (r - nx); dst = (g.Bx + (r - nx)) * MP; }
          else { src = rt + (r - nx - ny); dst = (g.Bx + g.By + (r - nx - ny)) * MP; }
          *reinterpret_cast<float4*>(GX + dst + 4 * c4) =
              __ldg(reinterpret_cast<const float4*>(T + src * TAB_M) + c4);
        }
      } else
      // entry e = (quadrature point mi, row r of the concatenated x | y | t rows), rows along the
      // lanes: a lane evaluates the n exponentials of dual cell gi once, for its own entry and
      // for the entry of gi + 1, which the next lane picks up by a shuffle (the first row of an
      // axis and lane 0 evaluate the cell below themselves)
      for (int e = threadIdx.x; e - (int)(threadIdx.x & 31) < nent; e += NT) {
        const bool act = e < nent;
        const int ee = act ? e : nent - 1;
        const int mi = (ee * inv_nr) >> 16, r = ee - mi * nr;     // ee / nr
        float sk, wk;
        if (flag) { sk = 0.5f; wk = mi == 0 ? 1.0f : 0.0f; }      // point-like: midpoint Gaussian
        else { sk = ((float)pc + c_gl_s[goff + mi]) * inv_np; wk = c_gl_w[goff + mi] * inv_np; }
        int gi, lo_a, hi_a, rr; float c, k2a, scale; float* dstp;
        if (r < nx) {
          rr = r; gi = ix0 + rr; lo_a = lox; hi_a = hix; c = fmaf(sk, dx, p0x); k2a = k2x; scale = K * wk;
          dstp = GX + rr * MP + mi;
        } else if (r < nx + ny) {
          rr = r - nx; gi = iy0 + rr; lo_a = loy; hi_a = hiy; c = fmaf(sk, dy, p0y); k2a = k2y; scale = 1.0f;
          dstp = GY + rr * MP + mi;
        } else {
          rr = r - nx - ny; gi = kt0 + rr; lo_a = lot; hi_a = hit; c = fmaf(sk, dt, p0t); k2a = k2t; scale = 1.0f;
          dstp = GT + rr * MP + mi;
        }
        float own, up;
        axis_cell<N>(gi, lo_a, hi_a, c, k2a, own, up);
        float below = __shfl_up_sync(0xffffffffu, up, 1);
        if (N > 1 && (rr == 0 || (threadIdx.x & 31) == 0)) {       // no lane holds cell gi - 1 of this axis
          float o2;
          axis_cell<N>(gi - 1, lo_a, hi_a, c, k2a, o2, below);
        }
        if (act) *dstp = (N > 1 ? own + below : own) * scale;
      }
      __syncthreads();
      // ---- phase B: tile[k][i][j] += sum_mi GX[i][mi] GY[j][mi] GT[k][mi]
      for (int item = threadIdx.x; item < ncolp * nsplit; item += NT) {
        const int sp = (item * inv_ncolp) >> 16, col = item - sp * ncolp;      // item / ncolp, exact here
        if (col >= ncol) continue;
        const int cx = (col * inv_ny) >> 16, cy = col - cx * ny;               // col / ny
        const int ka = sp * chunk, kb = min(ka + chunk, nt);
        float* tp = tile + (size_t)(kt0 - K0) * P.plane + (ix0 - I0 + cx) * g.By + (iy0 - J0 + cy);
        const float* GXr = GX + cx * MP;
        const float* GYr = GY + cy * MP;
        switch (m >> 2) {
          case 1: effq_phase_b<1>(tp, P.plane, GXr, GYr, GT, ka, kb); break;
          case 2: effq_phase_b<2>(tp, P.plane, GXr, GYr, GT, ka, kb); break;
          case 3: effq_phase_b<3>(tp, P.plane, GXr, GYr, GT, ka, kb); break;
          case 4: effq_phase_b<4>(tp, P.plane, GXr, GYr, GT, ka, kb); break;
          case 5: effq_phase_b<5>(tp, P.plane, GXr, GYr, GT, ka, kb); break;
          default: effq_phase_b<6>(tp, P.plane, GXr, GYr, GT, ka, kb); break;
        }
      }
      // no barrier here: the next phase A writes the other table set, and its barrier
      // orders this phase B before the next one
    }
  }
  }
  __syncthreads();
  // tile -> payload[blk][i][j][k], k contiguous: a thread writes 4 consecutive ticks
  float* out = payload + (int64_t)blk * g.Bx * g.By * g.Bt + sub * P.TS;
  const int nij = g.Bx * g.By;
  if ((P.TS & 3) == 0) {
    const int q4 = P.TS >> 2;                           // float4 per column
    for (int idx = threadIdx.x; idx < nij * q4; idx += NT) {
      const int ij = idx / q4, k = (idx - ij * q4) << 2;
      const float* t = tile + k * P.plane + ij;
      *reinterpret_cast<float4*>(out + (int64_t)ij * g.Bt + k) =
          make_float4(t[0], t[P.plane], t[2 * P.plane], t[3 * P.plane]);
    }
  } else {
    for (int idx = threadIdx.x; idx < nij * P.TS; idx += NT) {
      const int k = idx % P.TS, ij = idx / P.TS;
      out[(int64_t)ij * g.Bt + k] = tile[k * P.plane + ij];
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
constexpr int TR_MAXG = 16;          // pixel / tile groups per axis a segment may reach

struct TruthBox { int lo[3], hi[3], g0[3], ng[3]; };

__device__ __forceinline__ bool truth_box(const int32_t* __restrict__ augi, int64_t nseg, int64_t s, const TredGrid& g,
                                          int E, TruthBox& b) {
  const int NG[3] = {g.NGx, g.NGy, g.NGt}, div[3] = {g.S, g.S, g.Bt};
  bool ok = true;
  for (int a = 0; a < 3; ++a) {
    b.lo[a] = max(augi[a * nseg + s] - E, 0);
    b.hi[a] = min(augi[(3 + a) * nseg + s] + E, NG[a] - 1);
    ok = ok && b.lo[a] <= b.hi[a];
    b.g0[a] = b.lo[a] / div[a];
    b.ng[a] = ok ? min(b.hi[a] / div[a] - b.g0[a] + 1, TR_MAXG) : 0;
  }
  return ok;
}

template <int N>
__global__ void __launch_bounds__(256)
k_truth_count(int64_t nseg, const int32_t* __restrict__ augi, TredGrid g, int32_t* __restrict__ cnt) {
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s > nseg) return;
  int c = 0;
  if (s < nseg) {
    TruthBox b;
    if (truth_box(augi, nseg, s, g, N > 1 ? 1 : 0, b)) c = b.ng[0] * b.ng[1] * b.ng[2];
  }
  cnt[s] = c;
}

// one warp per segment
template <int N>
__global__ void __launch_bounds__(128)
k_truth_fill(int64_t nseg, const float* __restrict__ augf, const int32_t* __restrict__ augi,
             const int32_t* __restrict__ first, TredGrid g, int64_t cap, int32_t* __restrict__ rec_seg,
             int64_t* __restrict__ rec_key, float* __restrict__ rec_q, int64_t* __restrict__ d_nrec) {
  __shared__ float sums[4][3 * TR_MAXG][MMAX];
  const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int64_t s = (int64_t)blockIdx.x * 4 + wid;
  if (blockIdx.x == 0 && threadIdx.x == 0) *d_nrec = first[nseg];
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

struct EffqWork { int32_t* slot; int32_t* tabslot; int32_t* seglist; void* scan; float* tab; int cap; size_t total; };

static EffqWork carve_effq(void* base, int64_t nseg, size_t work_bytes) {
  EffqWork w;
  size_t o = 0; char* b = (char*)base;
  auto take = [&](size_t bytes) { void* p = b ? b + o : nullptr; o += align_up(bytes, 256); return p; };
  w.slot = (int32_t*)take((size_t)(nseg + 1) * 4);
  w.tabslot = (int32_t*)take((size_t)(nseg > 0 ? nseg : 1) * 4);
  w.scan = take(tred_scan_work_bytes(nseg + 1));
  const size_t fixed = o;
  int64_t cap = nseg < EFFQ_MAX_SLOTS ? nseg : EFFQ_MAX_SLOTS;
  if (work_bytes) {                                  // what the given workspace holds
    const size_t per = (size_t)TAB_FLOATS * 4 + 4;
    cap = work_bytes > fixed + 4096 ? (int64_t)((work_bytes - fixed - 4096) / per) : 0;
    if (cap > nseg) cap = nseg;
    if (cap > EFFQ_MAX_SLOTS) cap = EFFQ_MAX_SLOTS;
  }
  if (cap < 0) cap = 0;
  w.cap = (int)cap;
  w.seglist = (int32_t*)take((size_t)(cap > 0 ? cap : 1) * 4);
  w.tab = (float*)take((size_t)(cap > 0 ? cap : 1) * TAB_FLOATS * 4);
  w.total = o;
  return w;
}

extern "C" size_t tred_effq_work_bytes(const tred_ctx* ctx, int64_t nseg) {
  if (!ctx || nseg < 0) return 0;
  return carve_effq(nullptr, nseg, 0).total;
}

extern "C" int tred_effq(tred_ctx* ctx, int64_t nseg, int64_t nblocks,
                         const int64_t* d_keys, const int32_t* d_blk_off, const int32_t* d_pair_seg,
                         const float* d_augf, const int32_t* d_augi,
                         float* d_payload, void* d_work, size_t work_bytes, void* stream) {
  if (!ctx || nseg < 0 || nblocks < 0) return TRED_EINVAL;
  if (nblocks == 0) return TRED_OK;
  if (!d_keys || !d_blk_off || !d_pair_seg || !d_augf || !d_augi || !d_payload) return TRED_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  if (ctx->cfg.effq_mode == 1)
    return tred_effq_closed_form(ctx, nseg, nblocks, d_keys, d_blk_off, d_pair_seg, d_augf, d_augi,
                                 d_payload, st);
  if (ctx->cfg.effq_mode != 0) return TRED_EINVAL;
  const TredGrid g = make_grid(ctx);
  FactParams P;
  P.plane = g.Bx * g.By + 1;
  // largest TS (power of two, <= Bt) whose tile fits ~64 KB
  int TS = g.Bt;
  while (TS > 4 && (size_t)TS * P.plane * sizeof(float) > TRED_EFFQ_TILE_KB * 1024) TS /= 2;
  P.TS = TS; P.nsub = g.Bt / TS;
  const size_t tile_floats = ((size_t)TS * P.plane + 3) & ~(size_t)3;
  const size_t smem = (tile_floats + 2 * (size_t)(g.Bx + g.By + TS) * MP) * sizeof(float);
  if (smem > (size_t)ctx->smem_optin) return TRED_EUNSUPPORTED;
  int threads = g.Bx * g.By * 4;
  threads = threads < 64 ? 64 : threads > TRED_EFFQ_THREADS ? TRED_EFFQ_THREADS : threads;
  if (nblocks * P.nsub >= (1ll << 31)) return TRED_EUNSUPPORTED;
  EffqWork w = carve_effq(d_work, nseg, work_bytes);
  const bool tables = d_work && w.total <= work_bytes && w.cap >= 1024;
  TredProfScope ps(ctx, ST_EFFQ, st);
  for (int64_t k0 = 0; k0 < nblocks; k0 += tables ? EFFQ_RANGE_BLOCKS : nblocks) {
    const int nb = (int)(tables ? (nblocks - k0 < EFFQ_RANGE_BLOCKS ? nblocks - k0 : EFFQ_RANGE_BLOCKS) : nblocks);
    if (tables) {
      TRED_CUDA(cudaMemsetAsync(w.slot, 0, (size_t)(nseg + 1) * 4, st));
      k_effq_mark<<<cdiv((int64_t)nb * 32, 256), 256, 0, st>>>(nb, (int)k0, d_blk_off, d_pair_seg, w.slot);
      int rc = tred_exclusive_scan_i32(w.slot, w.slot, nseg + 1, nullptr, w.scan, st);
      if (rc != TRED_OK) return rc;
      k_effq_list<<<cdiv(nseg, 256), 256, 0, st>>>(nseg, w.slot, w.seglist, w.cap, w.tabslot);
      TRED_COUNT_LAUNCH(4);
    }
#define LAUNCH(NN)                                                                                     \
  do {                                                                                                 \
    if (tables)                                                                                        \
      k_effq_tables<NN><<<cdiv(w.cap, 4), 128, 0, st>>>(nseg, w.slot, w.seglist, w.cap, d_augf, d_augi, \
                                                        w.tab, w.tabslot);                             \
    TRED_CUDA(cudaFuncSetAttribute(k_effq_fact<NN>, cudaFuncAttributeMaxDynamicSharedMemorySize,       \
                                   (int)smem));                                                        \
    k_effq_fact<NN><<<(unsigned)((int64_t)nb * P.nsub), threads, smem, st>>>(                          \
        nseg, d_keys + k0, d_blk_off + k0, d_pair_seg, d_augf, d_augi, tables ? w.tabslot : nullptr,   \
        w.tab, d_payload + k0 * g.Bx * g.By * g.Bt, g, P);                                             \
  } while (0)
    TRED_COUNT_LAUNCH(tables ? 2 : 1);
    switch (g.gl_n) {
      case 1: LAUNCH(1); break;
      case 2: LAUNCH(2); break;
      case 3: LAUNCH(3); break;
      case 4: LAUNCH(4); break;
      default: return TRED_EINVAL;
    }
#undef LAUNCH
  }
  TRED_LAUNCH_CHECK("k_effq_fact");
  return TRED_OK;
}


extern "C" size_t tred_truth_work_bytes(const tred_ctx* ctx, int64_t nseg) {
  if (!ctx || nseg < 0) return 0;
  return align_up((size_t)(nseg + 1) * 4, 256) + tred_scan_work_bytes(nseg + 1);
}

extern "C" int tred_truth(tred_ctx* ctx, int64_t nseg, const float* d_augf, const int32_t* d_augi, int64_t cap_rec,
                          int32_t* d_rec_seg, int64_t* d_rec_key, float* d_rec_q, int64_t* d_nrec, void* d_work,
                          size_t work_bytes, void* stream) {
  if (!ctx || nseg < 0 || cap_rec < 0 || !d_nrec) return TRED_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  if (nseg == 0) { TRED_CUDA(cudaMemsetAsync(d_nrec, 0, sizeof(int64_t), st)); return TRED_OK; }
  if (!d_augf || !d_augi || !d_work) return TRED_EINVAL;
  if (work_bytes < tred_truth_work_bytes(ctx, nseg)) return TRED_ECAP;
  if (cap_rec > 0 && (!d_rec_seg || !d_rec_key || !d_rec_q)) return TRED_EINVAL;
  const TredGrid g = make_grid(ctx);
  int32_t* first = (int32_t*)d_work;
  void* scan = (char*)d_work + align_up((size_t)(nseg + 1) * 4, 256);
#define TRUTH(NN)                                                                                          \
  do {                                                                                                     \
    k_truth_count<NN><<<cdiv(nseg + 1, 256), 256, 0, st>>>(nseg, d_augi, g, first);                        \
    int rc = tred_exclusive_scan_i32(first, first, nseg + 1, nullptr, scan, st);                           \
    if (rc != TRED_OK) return rc;                                                                          \
    k_truth_fill<NN><<<cdiv(nseg, 4), 128, 0, st>>>(nseg, d_augf, d_augi, first, g, cap_rec, d_rec_seg,     \
                                                    d_rec_key, d_rec_q, d_nrec);                           \
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
