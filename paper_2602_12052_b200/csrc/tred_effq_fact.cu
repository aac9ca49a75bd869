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

#ifndef TRED_EFFQ_MINB
#define TRED_EFFQ_MINB 4            // resident CTAs per SM the register allocation aims at
#endif
#ifndef TRED_EFFQ_TILE_KB
#define TRED_EFFQ_TILE_KB 64        // largest tile (floats x 4) a CTA stages
#endif

template <int N>
__global__ void __launch_bounds__(256, TRED_EFFQ_MINB)
k_effq_fact(int64_t nseg, const int64_t* __restrict__ keys, const int32_t* __restrict__ blk_off,
            const int32_t* __restrict__ pair_seg, const float* __restrict__ augf,
            const int32_t* __restrict__ augi, float* __restrict__ payload, TredGrid g, FactParams P) {
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
  constexpr int SB = 32, NF = 17;                      // 7 int fields (bbox, flag) + 10 floats
  __shared__ int32_t s_rec[SB][NF + 1];
  const int s_beg = blk_off[blk], s_end = blk_off[blk + 1];
  int it = 0;
  for (int b0 = s_beg; b0 < s_end; b0 += SB) {
  const int nbatch = min(SB, s_end - b0);
  __syncthreads();                                     // the previous batch's records are no longer read
  for (int e = threadIdx.x; e < nbatch * NF; e += NT) {
    const int j = e / NF, f = e - j * NF;
    const int64_t s = pair_seg[b0 + j];
    s_rec[j][f] = f < 7 ? augi[f * nseg + s] : __float_as_int(augf[(f - 7) * nseg + s]);
  }
  __syncthreads();
  for (int sj = 0; sj < nbatch; ++sj) {
    const int32_t* rec = s_rec[sj];
    const int lox = rec[0], loy = rec[1], lot = rec[2];
    const int hix = rec[3], hiy = rec[4], hit = rec[5];
    // grid points of the segment's footprint inside this tile (and the grid)
    const int ix0 = max(lox - E, I0), ix1 = min(min(hix + E, I0 + g.Bx - 1), g.NGx - 1);
    const int iy0 = max(loy - E, J0), iy1 = min(min(hiy + E, J0 + g.By - 1), g.NGy - 1);
    const int kt0 = max(lot - E, K0), kt1 = min(min(hit + E, K0 + P.TS - 1), g.NGt - 1);
    if (ix0 > ix1 || iy0 > iy1 || kt0 > kt1) continue;            // CTA-uniform
    const int nx = ix1 - ix0 + 1, ny = iy1 - iy0 + 1, nt = kt1 - kt0 + 1;
    const int flag = rec[6];
    const float p0x = __int_as_float(rec[7]), p0y = __int_as_float(rec[8]), p0t = __int_as_float(rec[9]);
    const float p1x = __int_as_float(rec[10]), p1y = __int_as_float(rec[11]), p1t = __int_as_float(rec[12]);
    const float sx = __int_as_float(rec[13]), sy = __int_as_float(rec[14]), st = __int_as_float(rec[15]);
    const float Qp = __int_as_float(rec[16]);
    const float dx = p1x - p0x, dy = p1y - p0y, dt = p1t - p0t;
    const float k2x = LOG2E_HALF / (sx * sx), k2y = LOG2E_HALF / (sy * sy), k2t = LOG2E_HALF / (st * st);
    const float K = Qp * 0.063493635934240969f / (sx * sy * st) * 0.125f;   // (2 pi)^-3/2 / 8
    // number of quadrature points from the segment length in sigmas, W = sqrt(a)
    int npiece = 1, m = 4;
    if (!flag) {
      const float W = sqrtf((dx / sx) * (dx / sx) + (dy / sy) * (dy / sy) + (dt / st) * (dt / st));
      npiece = (int)ceilf(W * (1.0f / 15.5f));
      if (npiece < 1) npiece = 1;
      const float Wp = W / (float)npiece;
      m = Wp <= 1.0f ? 4 : Wp <= 3.9f ? 8 : Wp <= 6.9f ? 12 : Wp <= 9.9f ? 16 : Wp <= 12.8f ? 20 : 24;
    }
    const int goff = m * (m - 1) / 2;
    const float inv_np = 1.0f / (float)npiece;
    // phase-B work split: ncol columns x nsplit tick chunks
    const int ncol = nx * ny;
    const int ncolp = (ncol + 31) & ~31;
    const int nsplit = ncolp < NT ? NT / ncolp : 1;
    const int chunk = (nt + nsplit - 1) / nsplit;

    for (int pc = 0; pc < npiece; ++pc, ++it) {
      float* GX = tabs + (it & 1) * tabn;             // [Bx][MP]
      float* GY = GX + g.Bx * MP;                     // [By][MP]
      float* GT = GY + g.By * MP;                     // [TS][MP]
      // ---- phase A: tables
      const int nent = (nx + ny + nt) * m;
      for (int e = threadIdx.x; e < nent; e += NT) {
        const int r = e / m, mi = e - r * m;
        float sk, wk;
        if (flag) { sk = 0.5f; wk = mi == 0 ? 1.0f : 0.0f; }      // point-like: midpoint Gaussian
        else { sk = ((float)pc + c_gl_s[goff + mi]) * inv_np; wk = c_gl_w[goff + mi] * inv_np; }
        if (r < nx) {
          const float v = axis_entry<N>(ix0 + r, lox, hix, fmaf(sk, dx, p0x), k2x);
          GX[r * MP + mi] = v * (K * wk);
        } else if (r < nx + ny) {
          const int rr = r - nx;
          GY[rr * MP + mi] = axis_entry<N>(iy0 + rr, loy, hiy, fmaf(sk, dy, p0y), k2y);
        } else {
          const int rr = r - nx - ny;
          GT[rr * MP + mi] = axis_entry<N>(kt0 + rr, lot, hit, fmaf(sk, dt, p0t), k2t);
        }
      }
      __syncthreads();
      // ---- phase B: tile[k][i][j] += sum_mi GX[i][mi] GY[j][mi] GT[k][mi]
      for (int item = threadIdx.x; item < ncolp * nsplit; item += NT) {
        const int sp = item / ncolp, col = item - sp * ncolp;
        if (col >= ncol) continue;
        const int cx = col / ny, cy = col - cx * ny;
        const int ka = sp * chunk, kb = min(ka + chunk, nt);
        float* tp = tile + (size_t)(kt0 - K0) * P.plane + (ix0 - I0 + cx) * g.By + (iy0 - J0 + cy);
        for (int mg = 0; mg < m; mg += 4) {
          const float4 a = *reinterpret_cast<const float4*>(GX + cx * MP + mg);
          const float4 b = *reinterpret_cast<const float4*>(GY + cy * MP + mg);
          const float4 ab = make_float4(a.x * b.x, a.y * b.y, a.z * b.z, a.w * b.w);
#pragma unroll 4
          for (int k = ka; k < kb; ++k) {
            const float4 c = *reinterpret_cast<const float4*>(GT + k * MP + mg);
            float v = tp[k * P.plane];
            v = fmaf(ab.x, c.x, v); v = fmaf(ab.y, c.y, v);
            v = fmaf(ab.z, c.z, v); v = fmaf(ab.w, c.w, v);
            tp[k * P.plane] = v;
          }
        }
      }
      // no barrier here: the next phase A writes the other table set, and its barrier
      // orders this phase B before the next one
    }
  }
  }
  __syncthreads();
  // tile -> payload[blk][i][j][k], k contiguous
  float* out = payload + (int64_t)blk * g.Bx * g.By * g.Bt + sub * P.TS;
  const int nij = g.Bx * g.By;
  for (int idx = threadIdx.x; idx < nij * P.TS; idx += NT) {
    const int k = idx % P.TS, ij = idx / P.TS;
    out[(int64_t)ij * g.Bt + k] = tile[k * P.plane + ij];
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

extern "C" int tred_effq(tred_ctx* ctx, int64_t nseg, int64_t nblocks,
                         const int64_t* d_keys, const int32_t* d_blk_off, const int32_t* d_pair_seg,
                         const float* d_augf, const int32_t* d_augi,
                         float* d_payload, void* stream) {
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
  threads = threads < 64 ? 64 : threads > 256 ? 256 : threads;
  const int64_t grid = nblocks * P.nsub;
  if (grid >= (1ll << 31)) return TRED_EUNSUPPORTED;
#define LAUNCH(NN)                                                                                 \
  do {                                                                                             \
    TRED_CUDA(cudaFuncSetAttribute(k_effq_fact<NN>, cudaFuncAttributeMaxDynamicSharedMemorySize,   \
                                   (int)smem));                                                    \
    k_effq_fact<NN><<<(unsigned)grid, threads, smem, st>>>(nseg, d_keys, d_blk_off, d_pair_seg,    \
                                                           d_augf, d_augi, d_payload, g, P);       \
  } while (0)
  TredProfScope ps(ctx, ST_EFFQ, st);
  TRED_COUNT_LAUNCH(1);
  switch (g.gl_n) {
    case 1: LAUNCH(1); break;
    case 2: LAUNCH(2); break;
    case 3: LAUNCH(3); break;
    case 4: LAUNCH(4); break;
    default: return TRED_EINVAL;
  }
#undef LAUNCH
  TRED_LAUNCH_CHECK("k_effq_fact");
  return TRED_OK;
}
