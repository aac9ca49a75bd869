// S2 effective charge, closed-form variant (effq_mode 1): Eq. (9) with Eq. (10) / the
// point-like branch evaluated with exp and erf at every Gauss-Legendre node
// (PAPER.md:L85-148, L197).  The default variant is tred_effq_fact.cu; this one is kept as
// the literal per-node evaluation and as a cross-check of the factored form.
//
// Re-bracketing used here (same nodes, weights and coefficients as Eq. (9), only the
// order of summation differs): the Gauss-Legendre nodes are grouped by DUAL CELL, the
// cell between grid points d and d+1 per axis.  A node of cuboid c with xi >= 0 lies in
// dual cell c at s = xi/2; one with xi < 0 lies in dual cell c-1 at s = 1 + xi/2.  Every
// dual cell holds n nodes per axis, and a node's trilinear coefficients u (Eq. 7) are
// (1-s, s) towards grid points (d, d+1): exactly the 8 corners of the dual cell.
//
// One CTA owns a tile of one block (all of Bx x By, TS ticks) in shared memory; warp w
// owns ticks [w*KW, (w+1)*KW) of it for ALL segments, so no two warps ever touch the
// same word.  Inside a warp the dual cells are processed in 8 colours (parity of the cell
// index per axis): cells of one colour share no corner, so the read-modify-write of the
// 8 corners needs no atomics and the summation order is fixed (deterministic).
#include "tred_common.cuh"

namespace {

// Dual-cell node tables.  s: position in the dual cell, w: GL weight, side: 0 = node of
// cuboid d, 1 = node of cuboid d+1.  Closed forms: Abramowitz & Stegun 25.4:
//   n=1: xi = 0, w = 2;  n=2: xi = +-1/sqrt(3), w = 1;  n=3: xi = 0, +-sqrt(3/5), w = 8/9, 5/9;
//   n=4: xi = +-0.33998104, +-0.86113631, w = (18 +- sqrt(30))/36.
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

struct EffqParams {
  int TS;        // ticks per CTA tile
  int KW;        // ticks owned by one warp
  int nsub;      // Bt / TS
  int plane;     // Bx*By + 1 (padded plane stride of the shared tile)
};

template <int N>
__global__ void __launch_bounds__(256)
k_effq(int64_t nseg, const int64_t* __restrict__ keys, const int32_t* __restrict__ blk_off,
       const int32_t* __restrict__ pair_seg, const float* __restrict__ augf,
       const int32_t* __restrict__ augi, float* __restrict__ payload, TredGrid g, EffqParams P) {
  extern __shared__ float tile[];                 // [TS][plane]
  const int blk = blockIdx.x / P.nsub;
  const int sub = blockIdx.x - blk * P.nsub;
  const int64_t key = keys[blk];
  const int by = (int)(key % g.NBy);
  const int bx = (int)((key / g.NBy) % g.NBx);
  const int bt = (int)(key / ((int64_t)g.NBy * g.NBx));
  const int I0 = bx * g.Bx, J0 = by * g.By, K0 = bt * g.Bt + sub * P.TS;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

  for (int i = threadIdx.x; i < P.TS * P.plane; i += blockDim.x) tile[i] = 0.0f;
  __syncthreads();

  const int kw0 = K0 + warp * P.KW, kw1 = kw0 + P.KW - 1;     // ticks owned by this warp
  const int s_beg = blk_off[blk], s_end = blk_off[blk + 1];
  constexpr float INV_SQRT2 = 0.70710678118654752f;

  for (int si = s_beg; si < s_end; ++si) {
    const int s = pair_seg[si];
    const int lox = augi[0 * nseg + s], loy = augi[1 * nseg + s], lot = augi[2 * nseg + s];
    const int hix = augi[3 * nseg + s], hiy = augi[4 * nseg + s], hit = augi[5 * nseg + s];
    // dual cells that hold a node of this segment AND touch this warp's part of the tile
    const int dx0 = max(lox - 1, I0 - 1), dx1 = min(hix, I0 + g.Bx - 1);
    const int dy0 = max(loy - 1, J0 - 1), dy1 = min(hiy, J0 + g.By - 1);
    const int dt0 = max(lot - 1, kw0 - 1), dt1 = min(hit, kw1);
    if (dx0 > dx1 || dy0 > dy1 || dt0 > dt1) continue;        // warp-uniform
    const int flag = augi[6 * nseg + s];
    const float p0x = augf[0 * nseg + s], p0y = augf[1 * nseg + s], p0t = augf[2 * nseg + s];
    const float p1x = augf[3 * nseg + s], p1y = augf[4 * nseg + s], p1t = augf[5 * nseg + s];
    const float sx = augf[6 * nseg + s], sy = augf[7 * nseg + s], st = augf[8 * nseg + s];
    const float Qp = augf[9 * nseg + s];
    // per-segment constants (grid units).  Line form: q = K exp(beta^2 - c/2) *
    // [erf(beta) - erf(beta - alpha)], beta = b/sqrt(2a), alpha = sqrt(a/2)  (Eq. 10 with
    // the exponent -B/(2 Delta^2), reading G1).  Point form: Gaussian at the midpoint.
    const float isx = INV_SQRT2 / sx, isy = INV_SQRT2 / sy, ist = INV_SQRT2 / st;
    float ox, oy, ot, wax, way, wat, alpha, K;
    if (flag) {
      ox = 0.5f * (p0x + p1x); oy = 0.5f * (p0y + p1y); ot = 0.5f * (p0t + p1t);
      wax = way = wat = 0.0f; alpha = 0.0f;
      K = Qp * 0.063493635934240969f / (sx * sy * st) * 0.125f;        // (2 pi)^-3/2 / 8
    } else {
      ox = p0x; oy = p0y; ot = p0t;
      const float dx = p1x - p0x, dy = p1y - p0y, dt = p1t - p0t;
      const float a = (dx / sx) * (dx / sx) + (dy / sy) * (dy / sy) + (dt / st) * (dt / st);
      const float rs2a = rsqrtf(2.0f * a);
      wax = dx / (sx * sx) * rs2a; way = dy / (sy * sy) * rs2a; wat = dt / (st * st) * rs2a;
      alpha = sqrtf(0.5f * a);
      K = Qp * 0.079577471545947668f / (sx * sy * st * sqrtf(a)) * 0.125f;   // 1/(4 pi) / 8
    }

    for (int col = 0; col < 8; ++col) {
      const int px = col & 1, py = (col >> 1) & 1, pt = col >> 2;
      const int fx = dx0 + ((dx0 ^ px) & 1), fy = dy0 + ((dy0 ^ py) & 1), ft = dt0 + ((dt0 ^ pt) & 1);
      const int cx = fx <= dx1 ? (dx1 - fx) / 2 + 1 : 0;
      const int cy = fy <= dy1 ? (dy1 - fy) / 2 + 1 : 0;
      const int ct = ft <= dt1 ? (dt1 - ft) / 2 + 1 : 0;
      const int ncell = cx * cy * ct;
      for (int idx = lane; idx < ncell; idx += 32) {
        const int iy = idx % cy, r = idx / cy;
        const int ix = r % cx, it = r / cx;
        const int dx = fx + 2 * ix, dy = fy + 2 * iy, dt = ft + 2 * it;
        // per-axis node terms
        float bxn[N], cxn[N], ux0[N], ux1[N];
        float byn[N], cyn[N], uy0[N], uy1[N];
        float btn[N], ctn[N], ut0[N], ut1[N];
#pragma unroll
        for (int q = 0; q < N; ++q) {
          const float sq = DualGL<N>::s(q), wq = DualGL<N>::w(q);
          {
            const int c = dx + DualGL<N>::side(q);
            const float w = (c >= lox && c <= hix) ? wq : 0.0f;
            const float rr = ((float)(dx - lox) + 0.5f + sq) - ox;
            bxn[q] = wax * rr; const float z = rr * isx; cxn[q] = z * z;
            ux1[q] = w * sq; ux0[q] = w - ux1[q];
          }
          {
            const int c = dy + DualGL<N>::side(q);
            const float w = (c >= loy && c <= hiy) ? wq : 0.0f;
            const float rr = ((float)(dy - loy) + 0.5f + sq) - oy;
            byn[q] = way * rr; const float z = rr * isy; cyn[q] = z * z;
            uy1[q] = w * sq; uy0[q] = w - uy1[q];
          }
          {
            const int c = dt + DualGL<N>::side(q);
            const float w = (c >= lot && c <= hit) ? wq : 0.0f;
            const float rr = ((float)(dt - lot) + 0.5f + sq) - ot;
            btn[q] = wat * rr; const float z = rr * ist; ctn[q] = z * z;
            ut1[q] = w * sq; ut0[q] = w - ut1[q];
          }
        }
        float X[2][2][2] = {};
#pragma unroll
        for (int l = 0; l < N; ++l) {
          float Y[2][2] = {};
#pragma unroll
          for (int m = 0; m < N; ++m) {
            float T0 = 0.0f, T1 = 0.0f;
            const float bxy = bxn[l] + byn[m], cxy = cxn[l] + cyn[m];
#pragma unroll
            for (int n = 0; n < N; ++n) {
              const float c2 = cxy + ctn[n];
              float v;
              if (flag) {
                v = __expf(-c2);
              } else {
                const float beta = bxy + btn[n];
                v = __expf(fmaf(beta, beta, -c2)) * (erff(beta) - erff(beta - alpha));
              }
              T0 = fmaf(v, ut0[n], T0);
              T1 = fmaf(v, ut1[n], T1);
            }
            Y[0][0] = fmaf(uy0[m], T0, Y[0][0]); Y[0][1] = fmaf(uy0[m], T1, Y[0][1]);
            Y[1][0] = fmaf(uy1[m], T0, Y[1][0]); Y[1][1] = fmaf(uy1[m], T1, Y[1][1]);
          }
#pragma unroll
          for (int b = 0; b < 2; ++b)
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              X[0][b][c] = fmaf(ux0[l], Y[b][c], X[0][b][c]);
              X[1][b][c] = fmaf(ux1[l], Y[b][c], X[1][b][c]);
            }
        }
        // scatter to the 8 corners that lie in this warp's part of the tile (and the grid)
#pragma unroll
        for (int a = 0; a < 2; ++a) {
          const int gi = dx + a;
          if (gi < I0 || gi >= I0 + g.Bx || gi >= g.NGx) continue;
#pragma unroll
          for (int b = 0; b < 2; ++b) {
            const int gj = dy + b;
            if (gj < J0 || gj >= J0 + g.By || gj >= g.NGy) continue;
#pragma unroll
            for (int c = 0; c < 2; ++c) {
              const int gk = dt + c;
              if (gk < kw0 || gk > kw1 || gk >= g.NGt) continue;
              float* p = &tile[(gk - K0) * P.plane + (gi - I0) * g.By + (gj - J0)];
              *p += K * X[a][b][c];
            }
          }
        }
      }
      __syncwarp();
    }
  }
  __syncthreads();
  // tile -> payload[blk][i][j][k], k contiguous
  float* out = payload + (int64_t)blk * g.Bx * g.By * g.Bt + sub * P.TS;
  const int nij = g.Bx * g.By;
  for (int idx = threadIdx.x; idx < nij * P.TS; idx += blockDim.x) {
    const int k = idx % P.TS, ij = idx / P.TS;
    out[(int64_t)ij * g.Bt + k] = tile[k * P.plane + ij];
  }
}

}  // namespace

int tred_effq_closed_form(tred_ctx* ctx, int64_t nseg, int64_t nblocks,
                          const int64_t* d_keys, const int32_t* d_blk_off, const int32_t* d_pair_seg,
                          const float* d_augf, const int32_t* d_augi,
                          float* d_payload, cudaStream_t st) {
  const TredGrid g = make_grid(ctx);
  EffqParams P;
  P.plane = g.Bx * g.By + 1;
  // largest TS (power of two, <= Bt) whose tile fits ~64 KB; warps own KW ticks each
  int TS = g.Bt;
  while (TS > 4 && (size_t)TS * P.plane * sizeof(float) > 64 * 1024) TS /= 2;
  if ((size_t)TS * P.plane * sizeof(float) > (size_t)ctx->smem_optin) return TRED_EUNSUPPORTED;
  int KW = 16;
  const char* env = getenv("TRED_EFFQ_KW");
  if (env && atoi(env) > 0) KW = atoi(env);
  if (KW > TS) KW = TS;
  while (TS / KW > 8) KW *= 2;
  if (TS % KW) return TRED_EUNSUPPORTED;
  P.TS = TS; P.KW = KW; P.nsub = g.Bt / TS;
  const int threads = 32 * (TS / KW);
  const size_t smem = (size_t)TS * P.plane * sizeof(float);
  const int64_t grid = nblocks * P.nsub;
  if (grid >= (1ll << 31)) return TRED_EUNSUPPORTED;
#define LAUNCH(NN)                                                                            \
  do {                                                                                        \
    TRED_CUDA(cudaFuncSetAttribute(k_effq<NN>, cudaFuncAttributeMaxDynamicSharedMemorySize,   \
                                   (int)smem));                                               \
    k_effq<NN><<<(unsigned)grid, threads, smem, st>>>(nseg, d_keys, d_blk_off, d_pair_seg,    \
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
  TRED_LAUNCH_CHECK("k_effq");
  return TRED_OK;
}
