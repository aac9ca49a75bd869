// S4 interlaced FFT convolution (Eq. (12), L223-232 Eq. (14)) and
// S5 overlap-add on unique pixels.
//
// The paper-literal form (S*S zero-padded 3-D FFTs per block) is pruned to
// the time axis; the pixel-plane part of Eq. (12) is done directly, per frequency, as one
// batched complex matrix product:
//   (a) charge pixels: the (time slab, pixel) pairs met by an occupied block.  Real FFT
//       along time (length L >= Bt+Tr-1) of the S*S fine columns of every charge pixel
//       -> qhat[f][row][phase]                                          (k_fft_fwd)
//   (b) T[f][off][row] = sum_phase qhat[f][row][phase] * Rhat[f][phase][off]: the product
//       of the [rows x S*S] spectra with the [S*S x (2H+1)^2] response spectrum of the
//       frequency                                      (k_mac_fma / tred_mac_tc.cu)
//   (c) out_hat[sp][f] = sum_off T[f][off][row(pixel(sp) - off)]: sum before the inverse
//       FFT (Eq. (14) second line), sources in ascending row order        (k_accum)
//   (d) one inverse real FFT per slab pixel                               (k_ifft)
//   (e) overlap-add of the slab outputs into tiles (pixel, Bt ticks)      (k_gather_*)
// Spectra hold L/2 complex numbers: slot 0 packs (DC, Nyquist), both real.
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include "tred_common.cuh"
#include "tred_fft.cuh"

namespace {

// ------------------------------------------------------------------ response spectrum
// Computed ONCE per response, in fp64 by a direct DFT and rounded to
// fp32 at the end.  Induction-only pixels have a bipolar response whose DC bin is a
// cancellation to ~0; an fp32 FFT would leave ~1e-7 * sum|R| there, which the
// convolution multiplies by the whole collected charge.
// One CTA per response row (row = ((jx*S+jy)*K+kx)*K+ky = phase * noff + off).
//   W   [f][phase][kp] float2               (fp32 FMA path)
//   Bhi [f][2 kp][2 nph] float, Blo same    (tensor path: real-ified, K-major, tf32 split)
//     n = 2 off + c' (output re / im), kk = 2 phase + c (input re / im):
//     B[n][kk] = c == 0 ? (c' == 0 ? Wre : Wim) : (c' == 0 ? -Wim : Wre)
//     slot f = 0 packs DC (real part lane) and Nyquist (imaginary part lane):
//     B[2 off][2 phase] = W_DC, B[2 off + 1][2 phase + 1] = W_Nyq, others 0.
__device__ __forceinline__ float tf32_trunc(float x) {
  return __uint_as_float(__float_as_uint(x) & 0xffffe000u);
}

__global__ void __launch_bounds__(256)
k_resp_dft64(const float* __restrict__ resp, float2* __restrict__ W, float* __restrict__ Bhi,
             float* __restrict__ Blo, __nv_bfloat16* __restrict__ Bhb, __nv_bfloat16* __restrict__ Blb,
             int Tr, int L, int noff, int kp, int nph) {
  extern __shared__ double smd[];
  double2* tw = reinterpret_cast<double2*>(smd);       // [L]  exp(-2 pi i k / L)
  double* r = smd + 2 * L;                              // [Tr]
  const int row = blockIdx.x;
  const int phase = row / noff, off = row - phase * noff;
  for (int k = threadIdx.x; k < L; k += blockDim.x) {
    double sn, cs;
    sincospi(-2.0 * (double)k / (double)L, &sn, &cs);
    tw[k] = make_double2(cs, sn);
  }
  for (int i = threadIdx.x; i < Tr; i += blockDim.x) r[i] = (double)resp[(int64_t)row * Tr + i];
  __syncthreads();
  const int nf = L >> 1;
  const int64_t bplane = (int64_t)(2 * kp) * (2 * nph);
  for (int f = threadIdx.x; f <= nf; f += blockDim.x) {
    double re = 0.0, im = 0.0;
    for (int t = 0; t < Tr; ++t) {
      const double2 w = tw[(int)(((int64_t)f * t) % L)];
      re += r[t] * w.x; im += r[t] * w.y;
    }
    const float fre = (float)re, fim = (float)im;
    float* bh = Bhi + (int64_t)(f == nf ? 0 : f) * bplane;
    float* bl = Blo + (int64_t)(f == nf ? 0 : f) * bplane;
    __nv_bfloat16* bhb = Bhb + (int64_t)(f == nf ? 0 : f) * bplane;
    __nv_bfloat16* blb = Blb + (int64_t)(f == nf ? 0 : f) * bplane;
    auto put = [&](int n, int kk, float v) {
      const float h = tf32_trunc(v);
      bh[(int64_t)n * (2 * nph) + kk] = h;
      bl[(int64_t)n * (2 * nph) + kk] = tf32_trunc(v - h);
      bhb[(int64_t)n * (2 * nph) + kk] = __float2bfloat16_rn(h);        // operands of the bf16 corrections
      blb[(int64_t)n * (2 * nph) + kk] = __float2bfloat16_rn(v - h);
    };
    if (f == 0) {                       // DC: real lane of slot 0
      W[(int64_t)phase * kp + off].x = fre;
      put(2 * off, 2 * phase, fre);
    } else if (f == nf) {               // Nyquist: imaginary lane of slot 0
      W[(int64_t)phase * kp + off].y = fre;
      put(2 * off + 1, 2 * phase + 1, fre);
    } else {
      W[((int64_t)f * nph + phase) * kp + off] = make_float2(fre, fim);
      put(2 * off, 2 * phase, fre);
      put(2 * off + 1, 2 * phase, fim);
      put(2 * off, 2 * phase + 1, -fim);
      put(2 * off + 1, 2 * phase + 1, fre);
    }
  }
}

// fp16 hi / lo operands of the three-product tensor-core path (tred_mac_h3.cu): per frequency
// slot a power-of-two scale s_f with max |W[f]| / s_f in [2^14, 2^15), then
// B16[f][n][block(kk)] = fp16 parts of B[n][kk] / s_f, B as above, kk in blocks of (16 hi | 16 lo).
__device__ __forceinline__ float h16_scale(float m) {       // power of two s, m / s in [2^14, 2^15); 1 for m = 0
  const int ex = (int)((__float_as_uint(m) >> 23) & 0xffu);
  if (ex == 0 || ex == 255) return 1.0f;
  const int se = max(1, ex - 14);
  return __uint_as_float((uint32_t)se << 23);
}
__device__ __forceinline__ float pow2_inverse(float s) {    // 1 / s for s = 2^k, exponent field in [1, 253]
  return __uint_as_float((254u - (__float_as_uint(s) >> 23)) << 23);
}

__global__ void __launch_bounds__(256)
k_resp_h16_scale(const float2* __restrict__ W, float* __restrict__ bscale, int nph, int kp, int noff) {
  __shared__ float red[8];
  const int f = blockIdx.x;
  float m = 0.0f;
  for (int i = threadIdx.x; i < nph * kp; i += 256)
    if (i % kp < noff) {
      const float2 w = W[(int64_t)f * nph * kp + i];
      m = fmaxf(m, fmaxf(fabsf(w.x), fabsf(w.y)));
    }
  for (int o = 16; o; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = m;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) m = fmaxf(m, red[w]);
    bscale[f] = h16_scale(m);
  }
}

__global__ void __launch_bounds__(256)
k_resp_h16(const float2* __restrict__ W, const float* __restrict__ bscale, __half* __restrict__ B16,
           int nf, int nph, int noff, int kp, int kp16) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (int64_t)nf * nph * noff) return;
  const int off = (int)(i % noff);
  const int ph = (int)((i / noff) % nph);
  const int f = (int)(i / ((int64_t)noff * nph));
  const float2 w = W[((int64_t)f * nph + ph) * kp + off];
  const float inv = pow2_inverse(bscale[f]);
  __half* plane = B16 + (int64_t)f * (2 * kp) * kp16;
  auto put = [&](int n, int kk, float v) {
    v *= inv;
    const __half h = __float2half_rn(v);
    __half* e = plane + (int64_t)n * kp16 + (kk >> 4) * 32 + (kk & 15);
    e[0] = h;
    e[16] = __float2half_rn(v - __half2float(h));
  };
  if (f == 0) {                         // slot 0: DC in the real lane, Nyquist in the imaginary lane
    put(2 * off, 2 * ph, w.x);
    put(2 * off + 1, 2 * ph + 1, w.y);
  } else {
    put(2 * off, 2 * ph, w.x);
    put(2 * off + 1, 2 * ph, w.y);
    put(2 * off, 2 * ph + 1, -w.y);
    put(2 * off + 1, 2 * ph + 1, w.x);
  }
}

// ------------------------------------------------------------------ mirror symmetry (MPCP)
// PAPER.md:L199-221 (Mirror-Pair Complex Packing): a pixel response with the reflection
// symmetry R_{-i}^{-j} = R_i^j lets the paper pack the mirror phases Q^j + i Q^{-j} into one
// transform and halve the FFT count.  Here the time FFT is already real-to-half-complex, so
// the same symmetry is spent on the spectrum product instead: with phase p' = nph-1-p the
// mirror of p and offset o' = noff-1-o the mirror of o,
//   T[o] + T[o'] = sum_{p < nph/2} (q[p] + q[p']) (W[p][o] + W[p'][o]),
//   T[o] - T[o'] = sum_{p < nph/2} (q[p] - q[p']) (W[p][o] - W[p'][o]),
// two products of half the inner length and half the offsets: half the tensor-core work.
// k_resp_symcheck tests the response (exact equality); k_resp_sym builds the two matrices
// Bs, Bd [f][SYM_N][nph] (real-ified like B, tf32 hi / lo parts).
__global__ void __launch_bounds__(256)
k_resp_symcheck(const float* __restrict__ resp, int nph, int noff, int Tr, int* __restrict__ flag) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t n = (int64_t)(nph / 2) * noff * Tr;
  if (i >= n) return;
  const int tau = (int)(i % Tr);
  const int64_t r = i / Tr;
  const int off = (int)(r % noff), ph = (int)(r / noff);
  const float a = resp[((int64_t)ph * noff + off) * Tr + tau];
  const float b = resp[((int64_t)(nph - 1 - ph) * noff + (noff - 1 - off)) * Tr + tau];
  if (a != b) atomicOr(flag, 1);
}

__global__ void __launch_bounds__(256)
k_resp_sym(const float2* __restrict__ W, float* __restrict__ Bs_hi, float* __restrict__ Bs_lo,
           float* __restrict__ Bd_hi, float* __restrict__ Bd_lo, int nf, int nph, int noff, int kp) {
  const int nh = nph / 2, no = (noff + 1) / 2;
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (int64_t)nf * no * nh) return;
  const int p = (int)(i % nh);
  const int o = (int)((i / nh) % no);
  const int f = (int)(i / ((int64_t)nh * no));
  const float2 w1 = W[((int64_t)f * nph + p) * kp + o], w2 = W[((int64_t)f * nph + (nph - 1 - p)) * kp + o];
  const float2 ws = make_float2(w1.x + w2.x, w1.y + w2.y), wd = make_float2(w1.x - w2.x, w1.y - w2.y);
  const int64_t plane = (int64_t)f * SYM_N * nph;
  auto put = [&](float* hi, float* lo, int n, int kk, float v) {
    const float h = tf32_trunc(v);
    hi[plane + (int64_t)n * nph + kk] = h;
    lo[plane + (int64_t)n * nph + kk] = tf32_trunc(v - h);
  };
  auto fill = [&](float* hi, float* lo, float2 w) {
    if (f == 0) {                       // slot 0: DC in the real lane, Nyquist in the imaginary lane
      put(hi, lo, 2 * o, 2 * p, w.x);
      put(hi, lo, 2 * o + 1, 2 * p + 1, w.y);
    } else {
      put(hi, lo, 2 * o, 2 * p, w.x);
      put(hi, lo, 2 * o + 1, 2 * p, w.y);
      put(hi, lo, 2 * o, 2 * p + 1, -w.y);
      put(hi, lo, 2 * o + 1, 2 * p + 1, w.x);
    }
  };
  fill(Bs_hi, Bs_lo, ws);
  fill(Bd_hi, Bd_lo, wd);
}

// ------------------------------------------------------------------ plan (O6)
// flags over the map m = bt * npix + px * npy + py
// d_nb: device-side block count (NULL: nblocks is exact); nblocks is then the capacity of keys
__global__ void __launch_bounds__(256)
k_mark_blocks(int64_t nblocks, const int64_t* __restrict__ d_nb, const int64_t* __restrict__ keys,
              int32_t* __restrict__ cp_flag, int32_t* __restrict__ sp_flag, TredGrid g) {
  const int warp = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
  if (d_nb && *d_nb < nblocks) nblocks = *d_nb;
  if (warp >= nblocks) return;
  const int64_t key = keys[warp];
  const int by = (int)(key % g.NBy), bx = (int)((key / g.NBy) % g.NBx);
  const int bt = (int)(key / ((int64_t)g.NBy * g.NBx));
  const int64_t base = (int64_t)bt * g.npx * g.npy;
  const int cx0 = (g.Bx * bx) / g.S, cx1 = min((g.Bx * bx + g.Bx - 1) / g.S, g.npx - 1);
  const int cy0 = (g.By * by) / g.S, cy1 = min((g.By * by + g.By - 1) / g.S, g.npy - 1);
  {
    const int ny = cy1 - cy0 + 1, n = (cx1 - cx0 + 1) * ny;
    for (int i = lane; i < n; i += 32) cp_flag[base + (cx0 + i / ny) * g.npy + (cy0 + i % ny)] = 1;
  }
  const int x0 = max(cx0 - g.H, 0), x1 = min(cx1 + g.H, g.npx - 1);
  const int y0 = max(cy0 - g.H, 0), y1 = min(cy1 + g.H, g.npy - 1);
  const int ny = y1 - y0 + 1, n = (x1 - x0 + 1) * ny;
  for (int i = lane; i < n; i += 32) sp_flag[base + (x0 + i / ny) * g.npy + (y0 + i % ny)] = 1;
}

__global__ void __launch_bounds__(256)
k_compact_keys(int64_t n, const int32_t* __restrict__ idx, int64_t cap, int64_t* __restrict__ out_keys,
               int64_t* __restrict__ d_count, int32_t* __restrict__ slab_off, int nslab, int64_t npix) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0 && d_count) *d_count = idx[n];
  if (slab_off && i <= nslab) slab_off[i] = idx[i * npix];
  if (i >= n) return;
  const int p = idx[i];
  if (idx[i + 1] != p && p < cap) out_keys[p] = i;
}

__global__ void __launch_bounds__(256)
k_mark_tiles(int64_t nsp_map, const int32_t* __restrict__ sp_idx, int32_t* __restrict__ tile_flag, TredGrid g) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nsp_map) return;
  if (sp_idx[i + 1] == sp_idx[i]) return;
  const int64_t npix = (int64_t)g.npx * g.npy;
  const int bt = (int)(i / npix);
  const int64_t p = i - bt * npix;
  const int t1 = min(g.Bt * bt + g.Bt + g.Tr - 2, g.nticks - 1);
  for (int tb = bt; tb <= t1 / g.Bt; ++tb) tile_flag[tb * npix + p] = 1;
}

__global__ void __launch_bounds__(256)
k_fill_blockmap(int64_t nblocks, const int64_t* __restrict__ keys, int32_t* __restrict__ blockmap) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < nblocks) blockmap[keys[i]] = (int32_t)i;
}

// ------------------------------------------------------------------ row tiles
// The tensor-core path orders the charge pixels of a slab by (strip = px / 8, py, px % 8)
// and cuts every (slab, strip) sequence into row tiles of at most RT_ROWS consecutive rows,
// at most RT_PY - 2H lines tall (a py-line may be split between two tiles).  The outputs of a row tile then fall in
// the patch [8 strip - H, 8 strip + 7 + H] x [py0 - H, py0 + ny - 1 + H], small enough to
// be summed over the offsets in shared memory by the GEMM epilogue.
struct RtGeom { int nstrip, ngrp, capy; int64_t nmap2, cap_rt; };

static inline RtGeom rt_geom(const tred_ctx* c) {
  RtGeom r;
  r.nstrip = (c->cfg.npix_x + RT_SW - 1) / RT_SW;
  r.ngrp = (int)c->dims.NB[2] * r.nstrip;
  r.capy = RT_PY - 2 * c->cfg.resp_half;
  if (r.capy < 1) r.capy = 1;
  r.nmap2 = (int64_t)r.ngrp * c->cfg.npix_y * RT_SW;
  const int npy = c->cfg.npix_y;
  r.cap_rt = (int64_t)r.ngrp * ((npy * RT_SW + RT_ROWS - RT_SW) / (RT_ROWS - RT_SW + 1) + (npy + r.capy - 1) / r.capy + 1);
  return r;
}

// occupancy flags in strip order: m2 = ((bt * nstrip + strip) * npy + py) * 8 + px % 8
__global__ void __launch_bounds__(256)
k_rt_flags(int64_t nmap2, const int32_t* __restrict__ cp_idx, int32_t* __restrict__ ridx, int nstrip, TredGrid g) {
  const int64_t m2 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (m2 > nmap2) return;
  int v = 0;
  if (m2 < nmap2) {
    const int xl = (int)(m2 & (RT_SW - 1));
    const int64_t rest = m2 >> 3;
    const int py = (int)(rest % g.npy);
    const int64_t grp = rest / g.npy;
    const int strip = (int)(grp % nstrip), bt = (int)(grp / nstrip);
    const int px = strip * RT_SW + xl;
    if (px < g.npx) {
      const int64_t m = ((int64_t)bt * g.npx + px) * g.npy + py;
      v = cp_idx[m + 1] != cp_idx[m];
    }
  }
  ridx[m2] = v;
}

__global__ void __launch_bounds__(256)
k_rt_rows(int64_t nmap2, const int32_t* __restrict__ ridx, int32_t* __restrict__ row_m2) {
  const int64_t m2 = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (m2 >= nmap2) return;
  const int r = ridx[m2];
  if (ridx[m2 + 1] != r) row_m2[r] = (int32_t)m2;
}

// One thread per (slab, strip): greedy cut into row tiles.  WRITE = false counts them.
template <bool WRITE>
__global__ void __launch_bounds__(128)
k_rt_tiles(int ngrp, int npy, int capy, const int32_t* __restrict__ ridx, int32_t* __restrict__ cnt,
           const int32_t* __restrict__ off, int4* __restrict__ desc, int64_t cap_rt) {
  const int grp = blockIdx.x * blockDim.x + threadIdx.x;
  if (grp >= ngrp) return;
  const int32_t* line = ridx + (int64_t)grp * npy * RT_SW;      // line[py * 8] = first row of the line
  int t = WRITE ? off[grp] : 0;
  int py = 0, used = 0;                 // used: rows of line py already given to a tile
  while (py < npy) {
    if (line[(py + 1) * RT_SW] - line[py * RT_SW] - used == 0) { ++py; used = 0; continue; }
    // a tile takes rows in order until it holds RT_ROWS (a line may be split between two tiles:
    // every row carries its own pixel, the patch only has to cover the lines of its rows)
    const int py0 = py, row0 = line[py * RT_SW] + used;
    int rows = 0, last = py;
    while (py < npy && py - py0 < capy) {
      const int c = line[(py + 1) * RT_SW] - line[py * RT_SW] - used;
      const int take = min(c, RT_ROWS - rows);
      if (take > 0) last = py;
      rows += take;
      if (take < c) { used += take; break; }             // full inside this line
      ++py; used = 0;
      if (rows == RT_ROWS) break;
    }
    if (WRITE && t < cap_rt) desc[t] = make_int4(row0, rows, py0, last - py0 + 1);
    ++t;
  }
  if (!WRITE) cnt[grp] = t;
}

// first row tile of every slab (and the total in slot NBt)
__global__ void k_rt_slab_off(int NBt, int nstrip, const int32_t* __restrict__ off, int32_t* __restrict__ rt_off) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i <= NBt) rt_off[i] = off[i * nstrip];
}

// Where the forward FFT finds the charge pixel of the row a CTA works on: the sorted
// charge-pixel list (row = index from r0), or the row tiles (row = padded row of the
// chunk, 128 per tile; rows beyond the tile's count do not exist).
struct RowSrc {
  const int64_t* cp_keys; int r0;
  const int4* rt_desc; const int32_t* row_m2; int t0, nstrip, tiled;
};

__device__ __forceinline__ bool row_pixel(const RowSrc& rs, int row, const TredGrid& g, int& px, int& py, int& bt) {
  if (!rs.tiled) {
    const int64_t key = rs.cp_keys[rs.r0 + row];
    py = (int)(key % g.npy); px = (int)((key / g.npy) % g.npx);
    bt = (int)(key / ((int64_t)g.npy * g.npx));
    return true;
  }
  const int4 d = rs.rt_desc[rs.t0 + (row >> 7)];
  const int r = row & (RT_ROWS - 1);
  if (r >= d.y) return false;
  const int m2 = rs.row_m2[d.x + r];
  const int rest = m2 >> 3;
  py = rest % g.npy;
  const int grp = rest / g.npy;
  bt = grp / rs.nstrip;
  px = (grp - bt * rs.nstrip) * RT_SW + (m2 & (RT_SW - 1));
  return true;
}

// ------------------------------------------------------------------ twiddles
__global__ void __launch_bounds__(256) k_fill_twiddles(float2* __restrict__ tw, int N) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k < N) tw[k] = twiddle_N(k, N);
}

// ------------------------------------------------------------------ (a) forward FFT
// One CTA per (charge pixel of the chunk, group of CG = JG*S fine columns).
// Shared buffers are [sample][column] (tred_fft.cuh).  qhat[f][row][phase], plane stride
// rp rows.
__global__ void __launch_bounds__(256)
k_fft_fwd(const float* __restrict__ payload, const int32_t* __restrict__ blockmap,
          RowSrc rs, int rp, int JG,
          float2* __restrict__ qhat, const float2* __restrict__ gtw, TredGrid g, FftPlan pl) {
  extern __shared__ float2 sm[];
  const int N = g.L, M = N >> 1;
  const int CG = JG * g.S;
  float2* A = sm;                   // [M][CG]
  float2* B = sm + CG * M;          // [M][CG]
  float2* tw = sm + 2 * CG * M;     // [N]
  __shared__ long long colbase[64];
  const int ngrp = (g.S + JG - 1) / JG;
  const int row = blockIdx.x / ngrp, grp = blockIdx.x - row * ngrp;
  int px, py, bt;
  if (!row_pixel(rs, row, g, px, py, bt)) return;
  load_twiddles_N(tw, gtw, N);
  if (threadIdx.x < CG) {
    const int jx = grp * JG + threadIdx.x / g.S, jy = threadIdx.x % g.S;
    long long base = -1;
    if (jx < g.S) {
      const int i = px * g.S + jx, j = py * g.S + jy;
      const int bx = i / g.Bx, by = j / g.By;
      const int slot = blockmap[((int64_t)bt * g.NBx + bx) * g.NBy + by];
      if (slot >= 0) base = (((long long)slot * g.Bx + (i - bx * g.Bx)) * g.By + (j - by * g.By)) * g.Bt;
    }
    colbase[threadIdx.x] = base;
  }
  __syncthreads();
  // 4 consecutive lanes read one 32-byte sector of a column; samples >= Bt/2 are the zero
  // padding, which the first pass does not read
  const int hb = g.Bt >> 1, hq = (hb + 3) >> 2;
  for (int i = threadIdx.x; i < CG * hq * 4; i += blockDim.x) {
    const int m4 = i & 3, rest = i >> 2;
    const int c = rest % CG, m = (rest / CG) * 4 + m4;
    if (m >= hb) continue;
    float2 v = make_float2(0.0f, 0.0f);
    const long long base = colbase[c];
    if (base >= 0) v = *reinterpret_cast<const float2*>(payload + base + 2 * m);
    A[m * CG + c] = v;
  }
  __syncthreads();
  const float2* Z = fft_stockham<false>(A, B, tw, pl, CG, hb);
  const int jbase = grp * CG;
  const int ncol = min(CG, g.nph - jbase);
  for (int i = threadIdx.x; i < M * CG; i += blockDim.x) {
    const int f = i / CG, c = i - f * CG;
    if (c < ncol) qhat[((int64_t)f * rp + row) * g.nph + jbase + c] = rfft_post(Z, CG, c, tw, M, f);
  }
}

// Same kernel with the length M = L/2 and the CG = 20 columns per CTA (S = 10, JG = 2) as
// compile-time constants (tred_fft.cuh, fft_stockham_ct): no runtime divisions.
template <int M>
__global__ void __launch_bounds__(256)
k_fft_fwd_ct(const float* __restrict__ payload, const int32_t* __restrict__ blockmap,
             RowSrc rs, int rp,
             float2* __restrict__ qhat, const float2* __restrict__ gtw, TredGrid g) {
  extern __shared__ float2 sm[];
  constexpr int N = 2 * M, CG = 20, S = 10, JG = 2, NGRP = 5, NPH = 100;
  float2* A = sm;                   // [M][CG]
  float2* B = sm + CG * M;          // [M][CG]
  float2* tw = sm + 2 * CG * M;     // [N]
  __shared__ long long colbase[CG];
  const int row = blockIdx.x / NGRP, grp = blockIdx.x - row * NGRP;
  int px, py, bt;
  if (!row_pixel(rs, row, g, px, py, bt)) return;
  load_twiddles_N(tw, gtw, N);
  if (threadIdx.x < CG) {
    const int jx = grp * JG + threadIdx.x / S, jy = threadIdx.x % S;
    const int i = px * S + jx, j = py * S + jy;
    const int bx = i / g.Bx, by = j / g.By;
    const int slot = blockmap[((int64_t)bt * g.NBx + bx) * g.NBy + by];
    long long base = -1;
    if (slot >= 0) base = (((long long)slot * g.Bx + (i - bx * g.Bx)) * g.By + (j - by * g.By)) * g.Bt;
    colbase[threadIdx.x] = base;
  }
  __syncthreads();
  const int hb = g.Bt >> 1, hq = (hb + 3) >> 2;
  for (int i = threadIdx.x; i < CG * hq * 4; i += 256) {
    const int m4 = i & 3, rest = i >> 2;
    const int c = rest % CG, m = (rest / CG) * 4 + m4;
    if (m >= hb) continue;
    float2 v = make_float2(0.0f, 0.0f);
    const long long base = colbase[c];
    if (base >= 0) v = *reinterpret_cast<const float2*>(payload + base + 2 * m);
    A[m * CG + c] = v;
  }
  __syncthreads();
  const float2* Z = fft_stockham_ct<M, 1, false, CG, 256>(A, B, tw, hb);
  float2* out = qhat + (int64_t)row * NPH + grp * CG;
  const int64_t fstride = (int64_t)rp * NPH;
  for (int i = threadIdx.x; i < M * CG; i += 256) {
    const int f = i / CG, c = i - f * CG;
    out[f * fstride + c] = rfft_post(Z, CG, c, tw, M, f);
  }
}

// Forward FFT, two-step form for the zero-padded columns (only the first Bt/2 of the
// M complex samples are non-zero).  M = A B with B a power of two, sample n = B a + b,
// frequency k = ka + A kb:
//   step 1 (thread per column and b):  Y_b[ka] = sum_{a < nza} z[B a + b] W_M^{(B a + b) ka}
//           -- a pruned DFT, nza = ceil(Bt / 2 / B) <= 4 terms, twiddles by recurrence;
//   step 2 (thread per column and ka): X[ka + A kb] = sum_b Y_b[ka] W_B^{b kb}
//           -- a B-point FFT held in registers (fft_reg_dif);
//   then the half-length real-FFT post-processing on pairs (k, M - k).
// One shared-memory round trip between the steps and one before the post-processing,
// instead of one per radix pass.  CG = 20 columns (S = 10, two phase rows) per CTA.
// SYM: the 20 columns of the CTA are the sums (first 10) and differences (last 10) of the
// mirror phase pairs p = 10 grp + pl and nph-1-p (the FFT is linear, so they are formed
// on the samples), written to qhat[f][row][s: 50 | d: 50] for the mirror-symmetric product.
// MODE 2 (H16): the spectra leave as fp16 hi / lo parts in the block layout of tred_mac_h3.cu,
// qhat = [tile][f][128 rows][KP16] halves, scaled per row by the power of two rscale[row] chosen from
// sum |q| over the row's columns (no spectrum value can exceed it, so nothing overflows).
template <int M, int B, int NZA, int MODE>
__global__ void __launch_bounds__((20 * (M / B) + 31) / 32 * 32, MODE == 2 ? 65536 / 80 / ((20 * (M / B) + 31) / 32 * 32) : 1)
k_fft_fwd_2s(const float* __restrict__ payload, const int32_t* __restrict__ blockmap,
             RowSrc rs, int rp, float2* __restrict__ qhat, float* __restrict__ rscale,
             const float2* __restrict__ gtw, TredGrid g) {
  constexpr bool SYM = MODE == 1, H16 = MODE == 2;
  constexpr int A = M / B, CG = 20, S = 10, JG = 2, NGRP = 5, NPH = 100;
  constexpr int KP16 = (2 * NPH + 15) / 16 * 32;
  constexpr int NT = (CG * A + 31) / 32 * 32;
  constexpr int BP = B + 1, ZP = M + 1;
  constexpr int LOGB = tred_log2(B);
  static_assert(NT % B == 0, "step 1 keeps one b per thread");
  extern __shared__ float2 buf[];           // step 1 -> 2: [col][ka][b (+1)]; then Z: [col][k (+1)]
  __shared__ long long colbase_all[NGRP * CG];
  __shared__ long long colbase2_all[SYM ? NGRP * CG : 1];   // SYM: the mirror column
  const int row = blockIdx.x;                               // one CTA per row, its 5 column groups in turn
  int px, py, bt;
  if (!row_pixel(rs, row, g, px, py, bt)) return;
  auto column_base = [&](int jx, int jy) {
    const int i = px * S + jx, j = py * S + jy;
    const int bx = i / g.Bx, by = j / g.By;
    const int slot = blockmap[((int64_t)bt * g.NBx + bx) * g.NBy + by];
    long long base = -1;
    if (slot >= 0) base = (((long long)slot * g.Bx + (i - bx * g.Bx)) * g.By + (j - by * g.By)) * g.Bt;
    return base;
  };
  for (int t = threadIdx.x; t < NGRP * CG; t += NT) {
    const int gq = t / CG, cq = t - gq * CG;
    if (SYM) {
      const int pl = cq % S;                               // pair p = (jx = gq, jy = pl), mirror (S-1-gq, S-1-pl)
      colbase_all[t] = column_base(gq, pl);
      colbase2_all[t] = column_base(S - 1 - gq, S - 1 - pl);
    } else {
      colbase_all[t] = column_base(gq * JG + cq / S, cq % S);
    }
  }
  __syncthreads();
  const int hb = g.Bt >> 1;
  const int64_t fstride = (int64_t)rp * NPH;
  float sdown = 1.0f;                                        // H16: 1 / rscale[row]
  if constexpr (H16) {
    __shared__ float red[NT / 32];
    float sum = 0.0f;
    const int nq = g.Bt >> 2;
    for (int i = threadIdx.x; i < NGRP * CG * nq; i += NT) {
      const int c = i / nq, q4 = i - c * nq;
      const long long base = colbase_all[c];
      if (base >= 0) {
        const float4 v = __ldg(reinterpret_cast<const float4*>(payload + base) + q4);
        sum += (fabsf(v.x) + fabsf(v.y)) + (fabsf(v.z) + fabsf(v.w));
      }
    }
    for (int o = 16; o; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = sum;
    __syncthreads();
    float tot = red[0];
#pragma unroll
    for (int w = 1; w < NT / 32; ++w) tot += red[w];
    const float sc = h16_scale(tot);
    sdown = pow2_inverse(sc);
    if (threadIdx.x == 0) rscale[row] = sc;
  }
#pragma unroll 1
  for (int grp = 0; grp < NGRP; ++grp) {
  const long long* colbase = colbase_all + grp * CG;
  const long long* colbase2 = SYM ? colbase2_all + grp * CG : colbase2_all;
  // ---- step 1 (NT is a multiple of B: a thread keeps the same b for all its columns; all
  // global loads are issued before the arithmetic)
  {
    constexpr int NIT = (CG * B + NT - 1) / NT;
    const int b = threadIdx.x % B;
    float2 w[NZA], p[NIT][NZA];
#pragma unroll
    for (int a = 0; a < NZA; ++a) {
      const int n = B * a + b;
      w[a] = n < hb ? __ldg(gtw + 2 * n) : make_float2(1.0f, 0.0f);       // W_M^n = exp(-2 pi i 2n / N)
    }
#pragma unroll
    for (int i = 0; i < NIT; ++i) {
      const int it = threadIdx.x + i * NT;
      const long long base = it < CG * B ? colbase[it / B] : -1;
      const long long base2 = (SYM && it < CG * B) ? colbase2[it / B] : -1;
      const float sgn = (SYM && it / B >= S) ? -1.0f : 1.0f;
#pragma unroll
      for (int a = 0; a < NZA; ++a) {
        const int n = B * a + b;
        p[i][a] = (n < hb && base >= 0) ? __ldg(reinterpret_cast<const float2*>(payload + base + 2 * n))
                                        : make_float2(0.0f, 0.0f);
        if (SYM && n < hb && base2 >= 0) {
          const float2 x2 = __ldg(reinterpret_cast<const float2*>(payload + base2 + 2 * n));
          p[i][a].x = fmaf(sgn, x2.x, p[i][a].x);
          p[i][a].y = fmaf(sgn, x2.y, p[i][a].y);
        }
      }
    }
#pragma unroll
    for (int i = 0; i < NIT; ++i) {
      const int it = threadIdx.x + i * NT;
      if (it >= CG * B) break;
      const int c = it / B;
      float2* dst = buf + (c * A) * BP + b;
      if (SYM ? (colbase[c] < 0 && colbase2[c] < 0) : (colbase[c] < 0)) {   // column outside the occupied blocks
#pragma unroll
        for (int ka = 0; ka < A; ++ka) dst[ka * BP] = make_float2(0.0f, 0.0f);
        continue;
      }
#pragma unroll
      for (int ka = 0; ka < A; ++ka) {
        float2 acc = p[i][0];
#pragma unroll
        for (int a = 1; a < NZA; ++a) { acc.x += p[i][a].x; acc.y += p[i][a].y; }
        dst[ka * BP] = acc;
#pragma unroll
        for (int a = 0; a < NZA; ++a) p[i][a] = cmulf(p[i][a], w[a]);
      }
    }
  }
  __syncthreads();
  // ---- step 2
  {
    const int it = threadIdx.x;                            // NT >= CG * A: one item per thread
    float2 y[B];
    const bool on = it < CG * A;
    const int c = it / A, ka = it - c * A;
    const bool live = on && (colbase[c] >= 0 || (SYM && colbase2[c] >= 0));
    if (live) {
      const float2* src = buf + it * BP;
#pragma unroll
      for (int b = 0; b < B; ++b) y[b] = src[b];
      fft_reg_dif<B>(y);
    } else {
#pragma unroll
      for (int b = 0; b < B; ++b) y[b] = make_float2(0.0f, 0.0f);
    }
    __syncthreads();                                       // every Y read before Z overwrites the buffer
    if (on) {
      float2* z = buf + c * ZP + ka;
#pragma unroll
      for (int q = 0; q < B; ++q) z[A * tred_bitrev(q, LOGB)] = y[q];
    }
  }
  __syncthreads();
  // ---- real-FFT post-processing on pairs (k, M - k); slot 0 packs (DC, Nyquist).
  // Thread (kr, c): column c, pairs k = 1 + kr, 1 + kr + KR, ...; the two output pointers
  // advance by a constant, no index arithmetic in the loop.
  if constexpr (H16) {
    // thread (kr, cp): the two adjacent columns 2 cp, 2 cp + 1 (phases p0, p0 + 1 share a block
    // of 8 phases, so their hi parts are 8 contiguous bytes and their lo parts the 8 bytes 32
    // bytes further on)
    constexpr int CP = CG / 2, KR = NT / CP;
    const int cp = threadIdx.x % CP, kr = threadIdx.x / CP;
    const int p0 = grp * CG + 2 * cp;
    // [tile][f][128 rows][KP16]: the box of one (row tile, frequency) is contiguous
    __half* out = reinterpret_cast<__half*>(qhat) +
                  ((int64_t)(row >> 7) * M * RT_ROWS + (row & (RT_ROWS - 1))) * KP16 + (p0 >> 3) * 32 + (p0 & 7) * 2;
    const int64_t fstride_h = (int64_t)RT_ROWS * KP16;
    const float2* Z0 = buf + (2 * cp) * ZP;
    const float2* Z1 = Z0 + ZP;
    auto h2u = [](__half2 h) { return *reinterpret_cast<uint32_t*>(&h); };
    // (the operands arrive already scaled by sdown.)  Phases 98, 99 end the last block of 16 reals:
    // that thread also zeroes the block's 8 padding reals (hi and lo), which the tensor core reads
    const bool pad = (2 * NPH) % 16 != 0 && p0 == NPH - 2;
    auto put = [&](__half* o, float2 a, float2 b) {
      const __half2 ha = __floats2half2_rn(a.x, a.y), hb2 = __floats2half2_rn(b.x, b.y);
      const float2 fa = __half22float2(ha), fb = __half22float2(hb2);
      const __half2 la = __floats2half2_rn(a.x - fa.x, a.y - fa.y), lb = __floats2half2_rn(b.x - fb.x, b.y - fb.y);
      *reinterpret_cast<uint2*>(o) = make_uint2(h2u(ha), h2u(hb2));
      *reinterpret_cast<uint2*>(o + 16) = make_uint2(h2u(la), h2u(lb));
      if (pad) {
        *reinterpret_cast<uint4*>(o + 4) = make_uint4(0u, 0u, 0u, 0u);
        *reinterpret_cast<uint4*>(o + 20) = make_uint4(0u, 0u, 0u, 0u);
      }
    };
    const float hs = 0.5f * sdown;
    if (kr < KR) {
      if (kr == 0) {
        const float2 a = Z0[0], b = Z1[0];
        put(out, make_float2(sdown * (a.x + a.y), sdown * (a.x - a.y)),
            make_float2(sdown * (b.x + b.y), sdown * (b.x - b.y)));
      } else if (kr == 1) {
        const float2 a = Z0[M / 2], b = Z1[M / 2];                  // X[M/2] = conj(Z[M/2])
        put(out + (M / 2) * fstride_h, make_float2(sdown * a.x, -sdown * a.y), make_float2(sdown * b.x, -sdown * b.y));
      }
      __half* o1 = out + (int64_t)(1 + kr) * fstride_h;
      __half* o2 = out + (int64_t)(M - 1 - kr) * fstride_h;
      const int64_t step = (int64_t)KR * fstride_h;
#pragma unroll 2
      for (int k = 1 + kr; k < M / 2; k += KR, o1 += step, o2 -= step) {
        const float2 w = __ldg(gtw + k);
        float2 x1[2], x2[2];
#pragma unroll
        for (int j = 0; j < 2; ++j) {
          const float2* Z = j ? Z1 : Z0;
          const float2 pz = Z[k], qz = Z[M - k];
          const float2 e = make_float2(hs * (pz.x + qz.x), hs * (pz.y - qz.y));
          const float2 o = make_float2(hs * (pz.x - qz.x), hs * (pz.y + qz.y));
          const float2 wo = cmulf(w, o);
          x1[j] = make_float2(e.x + wo.y, e.y - wo.x);              // X[k]
          x2[j] = make_float2(e.x - wo.y, -e.y - wo.x);             // X[M-k]
        }
        put(o1, x1[0], x1[1]);
        put(o2, x2[0], x2[1]);
      }
    }
  } else {
    constexpr int KR = NT / CG;                                    // pair rows per sweep
    const int c = threadIdx.x % CG, kr = threadIdx.x / CG;
    const int cm = SYM ? (c < S ? c : c - S + NPH / 2) : c;
    float2* out = qhat + (int64_t)row * NPH + (SYM ? grp * S : grp * CG) + cm;
    const float2* Z = buf + c * ZP;
    if (kr < KR) {
      if (kr == 0) {
        const float2 z0 = Z[0];
        out[0] = make_float2(z0.x + z0.y, z0.x - z0.y);
      } else if (kr == 1) {
        const float2 z = Z[M / 2];                                  // X[M/2] = conj(Z[M/2])
        out[(M / 2) * fstride] = make_float2(z.x, -z.y);
      }
      float2* o1 = out + (int64_t)(1 + kr) * fstride;
      float2* o2 = out + (int64_t)(M - 1 - kr) * fstride;
      const int64_t step = (int64_t)KR * fstride;
#pragma unroll 4
      for (int k = 1 + kr; k < M / 2; k += KR, o1 += step, o2 -= step) {
        const float2 pz = Z[k], qz = Z[M - k];
        const float2 e = make_float2(0.5f * (pz.x + qz.x), 0.5f * (pz.y - qz.y));
        const float2 o = make_float2(0.5f * (pz.x - qz.x), 0.5f * (pz.y + qz.y));
        const float2 wo = cmulf(__ldg(gtw + k), o);
        *o1 = make_float2(e.x + wo.y, e.y - wo.x);                 // X[k]
        *o2 = make_float2(e.x - wo.y, -e.y - wo.x);                // X[M-k]
      }
    }
  }
  __syncthreads();                                                 // buf is rewritten by the next group
  }
}

// ------------------------------------------------------------------ (b) spectrum product, fp32 FMA
// T[f][off][row] = sum_phase qhat[f][row][phase] * W[f][phase][off]  (complex).
// grid (nf, Y).  CTA: W[f] in shared memory; tiles of MT rows x all offsets; thread tile
// 8 rows (2 tx + 32 q + {0,1}) x 8 offsets (8 conflict-free LDS.128 per 256 FFMA).  Slot f = 0 holds (DC, Nyquist): two real
// products.
constexpr int MAC_MT = 128;
constexpr int MAC_AS = MAC_MT + 2;      // padded row stride of the transposed A tile (float2)

__global__ void __launch_bounds__(256)
k_mac_fma(const float2* __restrict__ qhat, const float2* __restrict__ W, float2* __restrict__ T,
          int nrows, int rp, TredGrid g) {
  extern __shared__ float2 sm[];
  float2* Ws = sm;                          // [nph][kp]
  float2* As = sm + g.nph * g.kp;           // [nph][MAC_AS]
  const int f = blockIdx.x;
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int kgroups = g.kp >> 3;
  for (int i = threadIdx.x; i < g.nph * g.kp; i += blockDim.x) Ws[i] = W[(int64_t)f * g.nph * g.kp + i];
  const int ntiles = (nrows + MAC_MT - 1) / MAC_MT;
  for (int tile = blockIdx.y; tile < ntiles; tile += gridDim.y) {
    const int t0 = tile * MAC_MT;
    __syncthreads();
    for (int i = threadIdx.x; i < MAC_MT * g.nph; i += blockDim.x) {
      const int r = i / g.nph, j = i - r * g.nph;
      float2 v = make_float2(0.0f, 0.0f);
      if (t0 + r < nrows) v = qhat[((int64_t)f * rp + t0 + r) * g.nph + j];
      As[j * MAC_AS + r] = v;
    }
    __syncthreads();
    if (ty >= kgroups) continue;
    float2 acc[8][8];
#pragma unroll
    for (int i = 0; i < 8; ++i)
#pragma unroll
      for (int k = 0; k < 8; ++k) acc[i][k] = make_float2(0.0f, 0.0f);
    const float4* ap = reinterpret_cast<const float4*>(As + 2 * tx);   // rows 2 tx + 32 q + {0,1}
    const float4* wp = reinterpret_cast<const float4*>(Ws + 8 * ty);
    if (f != 0) {
      for (int j = 0; j < g.nph; ++j) {
        float2 a[8], w[8];
#pragma unroll
        for (int q = 0; q < 4; ++q) *reinterpret_cast<float4*>(&a[2 * q]) = ap[j * (MAC_AS / 2) + 16 * q];
#pragma unroll
        for (int q = 0; q < 4; ++q) *reinterpret_cast<float4*>(&w[2 * q]) = wp[j * (g.kp >> 1) + q];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            acc[i][k].x = fmaf(a[i].x, w[k].x, acc[i][k].x);
            acc[i][k].x = fmaf(-a[i].y, w[k].y, acc[i][k].x);
            acc[i][k].y = fmaf(a[i].x, w[k].y, acc[i][k].y);
            acc[i][k].y = fmaf(a[i].y, w[k].x, acc[i][k].y);
          }
      }
    } else {
      for (int j = 0; j < g.nph; ++j) {
        float2 a[8], w[8];
#pragma unroll
        for (int q = 0; q < 4; ++q) *reinterpret_cast<float4*>(&a[2 * q]) = ap[j * (MAC_AS / 2) + 16 * q];
#pragma unroll
        for (int q = 0; q < 4; ++q) *reinterpret_cast<float4*>(&w[2 * q]) = wp[j * (g.kp >> 1) + q];
#pragma unroll
        for (int i = 0; i < 8; ++i)
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            acc[i][k].x = fmaf(a[i].x, w[k].x, acc[i][k].x);
            acc[i][k].y = fmaf(a[i].y, w[k].y, acc[i][k].y);
          }
      }
    }
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      const int off = 8 * ty + k;
      if (off >= g.noff) continue;
      float2* dst = T + ((int64_t)f * g.kp + off) * rp + t0 + 2 * tx;     // rp % 128 == 0: 16-byte aligned
#pragma unroll
      for (int q = 0; q < 4; ++q)
        *reinterpret_cast<float4*>(dst + 32 * q) =
            make_float4(acc[2 * q][k].x, acc[2 * q][k].y, acc[2 * q + 1][k].x, acc[2 * q + 1][k].y);
    }
  }
}

// ------------------------------------------------------------------ (c) sum over the offsets
// One CTA per 32 consecutive slab pixels; lane = slab pixel, warps stride over f.
// Sources in ascending charge-pixel order, so the running sum kept in ohat across chunks
// adds the same numbers in the same order whatever the chunking.
__global__ void __launch_bounds__(256)
k_accum(const float2* __restrict__ T, const int64_t* __restrict__ sp_keys, int s0, int ns,
        const int32_t* __restrict__ cp_idx, int r0, int nrows, int rp,
        float2* __restrict__ ohat, int sbase, TredGrid g) {
  extern __shared__ int32_t src[];          // [noff][32] local row of the source or -1
  const int K = 2 * g.H + 1;
  const int64_t npix = (int64_t)g.npx * g.npy;
  int any = 0;
  for (int i = threadIdx.x; i < g.noff * 32; i += blockDim.x) {
    const int o = i >> 5, l = i & 31;
    int v = -1;
    const int spl = blockIdx.x * 32 + l;
    if (spl < ns) {
      const int64_t key = sp_keys[s0 + spl];
      const int py = (int)(key % g.npy), px = (int)((key / g.npy) % g.npx);
      const int64_t bt = key / npix;
      const int qx = px - g.H + o / K, qy = py - g.H + o % K;
      if (qx >= 0 && qx < g.npx && qy >= 0 && qy < g.npy) {
        const int64_t m = bt * npix + (int64_t)qx * g.npy + qy;
        const int c = cp_idx[m];
        if (cp_idx[m + 1] != c && c >= r0 && c < r0 + nrows) v = c - r0;
      }
    }
    src[i] = v;
    any |= (v >= 0);
  }
  if (!__syncthreads_or(any)) return;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  const int spl = blockIdx.x * 32 + lane;
  int mine = 0;
  for (int o = 0; o < g.noff; ++o) mine |= (src[o * 32 + lane] >= 0);
  if (spl >= ns || !mine) return;
  float2* op = ohat + (int64_t)(s0 + spl - sbase) * g.nf;
  for (int f = w; f < g.nf; f += nw) {
    float2 a = op[f];
    const float2* Tf = T + (int64_t)f * g.kp * rp;
    for (int o = 0; o < g.noff; ++o) {
      const int r = src[o * 32 + lane];
      if (r >= 0) {
        const float2 v = Tf[(int64_t)(g.noff - 1 - o) * rp + r];
        a.x += v.x; a.y += v.y;
      }
    }
    op[f] = a;
  }
}

// ------------------------------------------------------------------ (c') sum of the row-tile patches
// Tensor-core path: the GEMM epilogue (tred_mac_tc.cu) has already summed the products
// over the offsets inside every row tile's patch, opart[tile][f][X][Y].  A slab pixel is
// covered by at most two tiles of each of at most three strips; they are added in ascending
// tile order onto the running value of ohat, so the sequence of additions is the same for
// any chunking.  One CTA per 32 consecutive slab pixels; reads are coalesced over the
// pixels, the ohat update over the frequencies (transposed through shared memory).
constexpr int ACC_MAXE = 12;

__global__ void __launch_bounds__(256)
k_accum_tiles(const float2* __restrict__ opart, const int64_t* __restrict__ sp_keys, int s0, int ns,
              const int32_t* __restrict__ grp_off, const int4* __restrict__ rt_desc, int t0, int t1, int nstrip,
              float2* __restrict__ ohat, int sbase, TredGrid g) {
  __shared__ int32_t ent[32][ACC_MAXE];
  __shared__ int cnt[32];
  __shared__ float2 tile[32][33];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const int PX = RT_SW + 2 * g.H;
  const int64_t npos = (int64_t)PX * RT_PY;
  int n = 0;
  if (threadIdx.x < 32) {
    const int spl = blockIdx.x * 32 + threadIdx.x;
    if (spl < ns) {
      const int64_t key = sp_keys[s0 + spl];
      const int py = (int)(key % g.npy), px = (int)((key / g.npy) % g.npx);
      const int bt = (int)(key / ((int64_t)g.npy * g.npx));
      const int s_lo = px >= g.H ? (px - g.H) >> 3 : 0;
      const int s_hi = min(nstrip - 1, (px + g.H) >> 3);
      for (int sx = s_lo; sx <= s_hi; ++sx) {
        const int grp = bt * nstrip + sx;
        const int ta = max(grp_off[grp], t0), tb = min(grp_off[grp + 1], t1);
        for (int t = ta; t < tb; ++t) {
          const int4 d = rt_desc[t];
          if (py >= d.z - g.H && py <= d.z + d.w - 1 + g.H && n < ACC_MAXE)
            ent[threadIdx.x][n++] = ((t - t0) << 11) | ((px - (sx * RT_SW - g.H)) * RT_PY + (py - (d.z - g.H)));
        }
      }
    }
    cnt[threadIdx.x] = n;
  }
  if (!__syncthreads_or(n > 0)) return;
  const int my_n = cnt[lane];
  for (int f0 = 0; f0 < g.nf; f0 += 32) {
    // running values, coalesced over f
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int sl = w * 4 + i, f = f0 + lane;
      float2 v = make_float2(0.0f, 0.0f);
      if (cnt[sl] > 0 && f < g.nf) v = ohat[(int64_t)(s0 + blockIdx.x * 32 + sl - sbase) * g.nf + f];
      tile[lane][sl] = v;
    }
    __syncthreads();
    if (my_n > 0) {
      // this warp's four frequencies of the block together: per covering tile the four patch
      // values are loaded before any is added (four loads in flight instead of one); for every
      // (slab pixel, frequency) the additions are still in ascending tile order
      float2 a[4];
      const int fb = f0 + w * 4;
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = tile[w * 4 + i][lane];
      for (int e = 0; e < my_n; ++e) {
        const int en = ent[lane][e];
        const float2* src = opart + ((int64_t)(en >> 11) * g.nf + fb) * npos + (en & 2047);
        float2 v[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) v[i] = fb + i < g.nf ? src[(int64_t)i * npos] : make_float2(0.0f, 0.0f);
#pragma unroll
        for (int i = 0; i < 4; ++i) { a[i].x += v[i].x; a[i].y += v[i].y; }
      }
#pragma unroll
      for (int i = 0; i < 4; ++i) if (fb + i < g.nf) tile[w * 4 + i][lane] = a[i];
    }
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const int sl = w * 4 + i, f = f0 + lane;
      if (cnt[sl] > 0 && f < g.nf) ohat[(int64_t)(s0 + blockIdx.x * 32 + sl - sbase) * g.nf + f] = tile[lane][sl];
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------ (d) inverse FFT
// One CTA per IP slab pixels ([sample][pixel] in shared memory); sp_data[sp][n_over*Bt].
// Lanes: pixel fastest, 4 consecutive samples per pixel -> full 32-byte sectors in HBM,
// contiguous shared-memory rows.
__global__ void __launch_bounds__(256)
k_ifft(const float2* __restrict__ ohat, int s0, int ns, int sbase, float* __restrict__ sp_data,
       const float2* __restrict__ gtw, TredGrid g, FftPlan pl, int IP, int out_len) {
  extern __shared__ float2 sm[];
  const int N = g.L, M = N >> 1;
  float2* A = sm;                   // [M][IP]
  float2* B = sm + IP * M;          // [M][IP]
  float2* tw = sm + 2 * IP * M;     // [N]
  const int a0 = blockIdx.x * IP;
  load_twiddles_N(tw, gtw, N);
  __syncthreads();
  const int mq = (M + 3) >> 2;
  for (int i = threadIdx.x; i < IP * mq * 4; i += blockDim.x) {
    const int k4 = i & 3, rest = i >> 2;
    const int c = rest % IP, k = (rest / IP) * 4 + k4;
    if (k >= M) continue;
    float2 z = make_float2(0.0f, 0.0f);
    if (a0 + c < ns) {
      const float2* X = ohat + (int64_t)(s0 + a0 + c - sbase) * M;
      const float2 p = X[k], q = X[k ? M - k : 0];
      z = rfft_pre_inverse(p, q, tw, k);
    }
    A[k * IP + c] = z;
  }
  __syncthreads();
  const float2* Z = fft_stockham<true>(A, B, tw, pl, IP, M);
  const int row = g.nover * g.Bt, hrow = row >> 1, hq = (hrow + 3) >> 2;
  const float sc = 1.0f / (float)N;
  for (int i = threadIdx.x; i < IP * hq * 4; i += blockDim.x) {
    const int m4 = i & 3, rest = i >> 2;
    const int c = rest % IP, m = (rest / IP) * 4 + m4;
    if (m >= hrow || a0 + c >= ns) continue;
    float2 v = make_float2(0.0f, 0.0f);
    if (m < M) {
      const float2 z = Z[m * IP + c];
      v.x = (2 * m < out_len) ? z.x * sc : 0.0f;
      v.y = (2 * m + 1 < out_len) ? z.y * sc : 0.0f;
    }
    reinterpret_cast<float2*>(sp_data + (int64_t)(s0 + a0 + c) * row)[m] = v;
  }
}

template <int M, int IP>
__global__ void __launch_bounds__(256)
k_ifft_ct(const float2* __restrict__ ohat, int s0, int ns, int sbase, float* __restrict__ sp_data,
          const float2* __restrict__ gtw, TredGrid g, int out_len) {
  extern __shared__ float2 sm[];
  constexpr int N = 2 * M;
  float2* A = sm;                   // [M][IP]
  float2* B = sm + IP * M;          // [M][IP]
  float2* tw = sm + 2 * IP * M;     // [N]
  const int a0 = blockIdx.x * IP;
  load_twiddles_N(tw, gtw, N);
  __syncthreads();
  constexpr int MQ = (M + 3) >> 2;
  for (int i = threadIdx.x; i < IP * MQ * 4; i += 256) {
    const int k4 = i & 3, rest = i >> 2;
    const int c = rest % IP, k = (rest / IP) * 4 + k4;
    if (k >= M) continue;
    float2 z = make_float2(0.0f, 0.0f);
    if (a0 + c < ns) {
      const float2* X = ohat + (int64_t)(s0 + a0 + c - sbase) * M;
      const float2 p = X[k], q = X[k ? M - k : 0];
      z = rfft_pre_inverse(p, q, tw, k);
    }
    A[k * IP + c] = z;
  }
  __syncthreads();
  const float2* Z = fft_stockham_ct<M, 1, true, IP, 256>(A, B, tw, M);
  const int row = g.nover * g.Bt, hrow = row >> 1, hq = (hrow + 3) >> 2;
  const float sc = 1.0f / (float)N;
  for (int i = threadIdx.x; i < IP * hq * 4; i += 256) {
    const int m4 = i & 3, rest = i >> 2;
    const int c = rest % IP, m = (rest / IP) * 4 + m4;
    if (m >= hrow || a0 + c >= ns) continue;
    float2 v = make_float2(0.0f, 0.0f);
    if (m < M) {
      const float2 z = Z[m * IP + c];
      v.x = (2 * m < out_len) ? z.x * sc : 0.0f;
      v.y = (2 * m + 1 < out_len) ? z.y * sc : 0.0f;
    }
    reinterpret_cast<float2*>(sp_data + (int64_t)(s0 + a0 + c) * row)[m] = v;
  }
}

// lengths with a compile-time instance (others use the run-time plan kernels)
#define TRED_FFT_CT_LENGTHS(X) X(128) X(144) X(216) X(256) X(288) X(384) X(512)

// ------------------------------------------------------------------ (e) S5 overlap-add
// One thread per 4 ticks of a tile (float4), Bt / 4 threads per tile, 256 / (Bt / 4) tiles per CTA.
// VEC = false: one thread per tick (Bt not a multiple of 4, or more than 1024 ticks per tile).
template <bool VEC>
__global__ void __launch_bounds__(256)
k_gather_tiles(int64_t tile_begin, int64_t ntiles, const int64_t* __restrict__ tile_keys,
               const int32_t* __restrict__ sp_idx, const float* __restrict__ sp_data, float* __restrict__ tile_data,
               int accumulate, TredGrid g) {
  const int64_t npix = (int64_t)g.npx * g.npy;
  const int row = g.nover * g.Bt;
  if (VEC) {
    const int q = g.Bt >> 2;                                       // float4 per tile
    const int per = 256 / q;                                       // tiles per CTA
    const int tl = threadIdx.x / q, k4 = threadIdx.x - tl * q;
    const int64_t tile = tile_begin + (int64_t)blockIdx.x * per + tl;
    if (tl >= per || tile >= tile_begin + ntiles) return;
    const int64_t key = tile_keys[tile];
    const int tb = (int)(key / npix);
    const int64_t p = key - tb * npix;
    float4* out = reinterpret_cast<float4*>(tile_data + tile * g.Bt) + k4;
    // accumulate: continue the running sum left by the earlier chunks (slab ranges in
    // ascending order), so the additions are the same sequence as in one pass
    float4 acc = accumulate ? *out : make_float4(0.0f, 0.0f, 0.0f, 0.0f);
    for (int bt = max(tb - g.nover + 1, 0); bt <= tb; ++bt) {        // ascending slab order
      const int64_t m = bt * npix + p;
      const int i0 = sp_idx[m];
      if (sp_idx[m + 1] != i0) {
        const float4 v = *(reinterpret_cast<const float4*>(sp_data + (int64_t)i0 * row + (tb - bt) * g.Bt) + k4);
        acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
      }
    }
    const int t = tb * g.Bt + 4 * k4;
    if (t >= g.nticks) acc.x = 0.0f;
    if (t + 1 >= g.nticks) acc.y = 0.0f;
    if (t + 2 >= g.nticks) acc.z = 0.0f;
    if (t + 3 >= g.nticks) acc.w = 0.0f;
    *out = acc;
  } else {
    const int64_t tile = tile_begin + blockIdx.x;
    const int64_t key = tile_keys[tile];
    const int tb = (int)(key / npix);
    const int64_t p = key - tb * npix;
    for (int t = threadIdx.x; t < g.Bt; t += blockDim.x) {
      float acc = accumulate ? tile_data[tile * g.Bt + t] : 0.0f;
      for (int bt = max(tb - g.nover + 1, 0); bt <= tb; ++bt) {
        const int64_t m = bt * npix + p;
        const int i0 = sp_idx[m];
        if (sp_idx[m + 1] != i0) acc += sp_data[(int64_t)i0 * row + (tb - bt) * g.Bt + t];
      }
      if (tb * g.Bt + t >= g.nticks) acc = 0.0f;
      tile_data[tile * g.Bt + t] = acc;
    }
  }
}

__global__ void __launch_bounds__(256)
k_gather_dense(int64_t npix_req, const int32_t* __restrict__ pix_ids, const int32_t* __restrict__ tile_idx,
               const float* __restrict__ tile_data, float* __restrict__ dense, TredGrid g) {
  const int64_t r = blockIdx.x;
  const int64_t npix = (int64_t)g.npx * g.npy;
  const int p = pix_ids[r];
  for (int t = threadIdx.x; t < g.nticks; t += blockDim.x) {
    const int tb = t / g.Bt;
    float v = 0.0f;
    if (p >= 0 && p < npix) {
      const int64_t m = tb * npix + p;
      const int i0 = tile_idx[m];
      if (tile_idx[m + 1] != i0) v = tile_data[(int64_t)i0 * g.Bt + (t - tb * g.Bt)];
    }
    dense[r * g.nticks + t] = v;
  }
}

// Launch helpers: 1 if a compile-time instance ran, 0 if there is none for this shape,
// < 0 on a CUDA error.
static int launch_fft_fwd_ct(const tred_ctx* ctx, const TredGrid& g, const float* payload, const int32_t* blockmap,
                             const RowSrc& rs, int nr, int rp, float2* qhat, const float2* tw, cudaStream_t st) {
  if (g.S != 10 || nr < 1) return 0;
  const int M = g.L / 2;
  const size_t smem = (size_t)(2 * 20 * M + g.L) * sizeof(float2);
  if (smem > (size_t)ctx->smem_optin) return 0;
  switch (M) {
#define X(MM)                                                                                             \
  case MM: {                                                                                              \
    static bool set_dev[64] = {false};                                                                              \
    if (!set_dev[ctx->device & 63]) {                                                                                           \
      TRED_CUDA(cudaFuncSetAttribute(k_fft_fwd_ct<MM>, cudaFuncAttributeMaxDynamicSharedMemorySize,       \
                                     (int)smem));                                                         \
      set_dev[ctx->device & 63] = true;                                                                                         \
    }                                                                                                     \
    k_fft_fwd_ct<MM><<<(unsigned)(nr * 5), 256, smem, st>>>(payload, blockmap, rs, rp, qhat, tw, g);      \
    return 1;                                                                                             \
  }
    TRED_FFT_CT_LENGTHS(X)
#undef X
    default: return 0;
  }
}

#define TRED_FFT_2S_SHAPES(X) X(128, 32) X(144, 16) X(256, 32) X(288, 32) X(384, 32) X(512, 32)

template <int MM, int BB, int NZA, int MODE>
static int launch_fft_fwd_2s_t(const tred_ctx* ctx, const TredGrid& g, const float* payload, const int32_t* blockmap,
                               const RowSrc& rs, int nr, int rp, float2* qhat, float* rscale, const float2* tw,
                               cudaStream_t st) {
  constexpr int A = MM / BB;
  constexpr int NT = (20 * A + 31) / 32 * 32;
  constexpr size_t smem =
      sizeof(float2) * (size_t)((20 * A * (BB + 1) > 20 * (MM + 1)) ? 20 * A * (BB + 1) : 20 * (MM + 1));
  if (smem > (size_t)ctx->smem_optin) return 0;
  static bool set_dev[64] = {false};
  if (!set_dev[ctx->device & 63]) {
    TRED_CUDA(cudaFuncSetAttribute(k_fft_fwd_2s<MM, BB, NZA, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    set_dev[ctx->device & 63] = true;
  }
  k_fft_fwd_2s<MM, BB, NZA, MODE><<<(unsigned)nr, NT, smem, st>>>(payload, blockmap, rs, rp, qhat, rscale, tw, g);
  return 1;
}

// MODE 0: fp32 spectra, 1: mirror-pair sums / differences (fp32), 2: fp16 hi / lo parts + row scales
template <int MODE>
static int launch_fft_fwd_2s(const tred_ctx* ctx, const TredGrid& g, const float* payload, const int32_t* blockmap,
                             const RowSrc& rs, int nr, int rp, float2* qhat, float* rscale, const float2* tw,
                             cudaStream_t st) {
  if (g.S != 10 || nr < 1) return 0;
  if (MODE == 2 && (g.Bt & 3)) return 0;
  const int M = g.L / 2, hb = g.Bt / 2;
  switch (M) {
#define X(MM, BB)                                                                                          \
  case MM: {                                                                                               \
    const int nza = (hb + BB - 1) / BB;                                                                    \
    if (nza <= 1) return launch_fft_fwd_2s_t<MM, BB, 1, MODE>(ctx, g, payload, blockmap, rs, nr, rp, qhat, rscale, tw, st); \
    if (nza == 2) return launch_fft_fwd_2s_t<MM, BB, 2, MODE>(ctx, g, payload, blockmap, rs, nr, rp, qhat, rscale, tw, st); \
    if (nza <= 4) return launch_fft_fwd_2s_t<MM, BB, 4, MODE>(ctx, g, payload, blockmap, rs, nr, rp, qhat, rscale, tw, st); \
    return 0;                                                                                              \
  }
    TRED_FFT_2S_SHAPES(X)
#undef X
    default: return 0;
  }
}

// is there a two-step forward FFT instance for this shape?
static bool fft_fwd_2s_available(const TredGrid& g) {
  if (g.S != 10) return false;
  const int M = g.L / 2, hb = g.Bt / 2;
  switch (M) {
#define X(MM, BB) case MM: return (hb + BB - 1) / BB <= 4;
    TRED_FFT_2S_SHAPES(X)
#undef X
    default: return false;
  }
}

static int launch_ifft_ct(const tred_ctx* ctx, const TredGrid& g, const float2* ohat, int s0, int ns, int sbase,
                          float* sp_data, const float2* tw, int out_len, cudaStream_t st) {
  constexpr int IP = 8;
  const int M = g.L / 2;
  const size_t smem = (size_t)(2 * IP * M + g.L) * sizeof(float2);
  if (smem > (size_t)ctx->smem_optin || ns < 1) return 0;
  switch (M) {
#define X(MM)                                                                                             \
  case MM: {                                                                                              \
    static bool set_dev[64] = {false};                                                                              \
    if (!set_dev[ctx->device & 63]) {                                                                                           \
      TRED_CUDA(cudaFuncSetAttribute(k_ifft_ct<MM, IP>, cudaFuncAttributeMaxDynamicSharedMemorySize,      \
                                     (int)smem));                                                         \
      set_dev[ctx->device & 63] = true;                                                                                         \
    }                                                                                                     \
    k_ifft_ct<MM, IP><<<cdiv(ns, IP), 256, smem, st>>>(ohat, s0, ns, sbase, sp_data, tw, g, out_len);     \
    return 1;                                                                                             \
  }
    TRED_FFT_CT_LENGTHS(X)
#undef X
    default: return 0;
  }
}

struct PlanWork {
  int32_t* cp_idx; int32_t* sp_idx; int32_t* tile_idx; void* scan;
  int32_t* ridx; int32_t* row_m2; int32_t* grp_off; int4* rt_desc;      // row tiles
  size_t total; int64_t nmap;
};

static PlanWork carve_plan(const tred_ctx* c, void* base) {
  PlanWork w;
  size_t o = 0; char* b = (char*)base;
  auto take = [&](size_t bytes) { void* p = b ? b + o : nullptr; o += align_up(bytes, 256); return p; };
  w.nmap = (int64_t)c->dims.NB[2] * c->cfg.npix_x * c->cfg.npix_y;
  w.cp_idx = (int32_t*)take((w.nmap + 1) * 4);
  w.sp_idx = (int32_t*)take((w.nmap + 1) * 4);
  w.tile_idx = (int32_t*)take((w.nmap + 1) * 4);
  const RtGeom rg = rt_geom(c);
  w.scan = take(tred_scan_work_bytes((rg.nmap2 > w.nmap ? rg.nmap2 : w.nmap) + 1));
  w.ridx = (int32_t*)take((rg.nmap2 + 1) * 4);
  w.row_m2 = (int32_t*)take(rg.nmap2 * 4);
  w.grp_off = (int32_t*)take((size_t)(rg.ngrp + 1) * 4);
  w.rt_desc = (int4*)take((size_t)rg.cap_rt * sizeof(int4));
  w.total = o;
  return w;
}

struct ConvWork {
  int32_t* blockmap; float2* tw; float2* ohat; float2* qhat; float2* T;
  size_t total;
};

static int64_t pad_rows(int64_t rows) { return (rows + 127) / 128 * 128; }

static ConvWork carve_conv(const tred_ctx* c, void* base, int64_t rows, int64_t nsp) {
  ConvWork w;
  size_t o = 0; char* b = (char*)base;
  auto take = [&](size_t bytes) { void* p = b ? b + o : nullptr; o += align_up(bytes, 1024); return p; };
  const tred_dims& d = c->dims;
  if (rows < 1) rows = 1;
  if (nsp < 1) nsp = 1;
  const int64_t rp = pad_rows(rows);
  w.blockmap = (int32_t*)take((size_t)(d.NB[0] * d.NB[1] * d.NB[2]) * 4);
  w.tw = (float2*)take((size_t)d.fft_len * 8);
  w.ohat = (float2*)take((size_t)nsp * d.n_freq * 8);
  w.qhat = (float2*)take((size_t)d.n_freq * rp * d.n_phase * 8);
  w.T = (float2*)take((size_t)d.n_freq * d.n_off_pad * rp * 8);
  w.total = o;
  return w;
}

struct TiledWork {
  int32_t* blockmap; float2* tw; float2* ohat; float2* qhat; float2* opart; float* rscale;
  size_t total, per_tile;
};

static TiledWork carve_tiled(const tred_ctx* c, void* base, int64_t ntile, int64_t nsp) {
  TiledWork w;
  size_t o = 0; char* b = (char*)base;
  auto take = [&](size_t bytes) { void* p = b ? b + o : nullptr; o += align_up(bytes, 1024); return p; };
  const tred_dims& d = c->dims;
  if (ntile < 1) ntile = 1;
  if (nsp < 1) nsp = 1;
  const size_t npos = (size_t)(RT_SW + 2 * c->cfg.resp_half) * RT_PY;
  w.blockmap = (int32_t*)take((size_t)(d.NB[0] * d.NB[1] * d.NB[2]) * 4);
  w.tw = (float2*)take((size_t)d.fft_len * 8);
  w.ohat = (float2*)take((size_t)nsp * d.n_freq * 8);
  // a row of spectra: fp32 complex [phase], or fp16 hi / lo blocks (h16_kp halves)
  const size_t row_bytes = (size_t)d.n_phase * 8 > (size_t)h16_kp(d) * 2 ? (size_t)d.n_phase * 8 : (size_t)h16_kp(d) * 2;
  w.qhat = (float2*)take((size_t)d.n_freq * ntile * RT_ROWS * row_bytes);
  w.opart = (float2*)take((size_t)ntile * d.n_freq * npos * 8);
  w.rscale = (float*)take((size_t)ntile * RT_ROWS * 4);
  w.per_tile = (size_t)d.n_freq * (RT_ROWS * row_bytes + npos * 8) + RT_ROWS * 4;
  w.total = o;
  return w;
}

}  // namespace

// tensor-core variant of step (b) (tred_mac_tc.cu); returns TRED_EUNSUPPORTED if it
// cannot run this configuration
int tred_mac_tc(tred_ctx* ctx, const float* qhat, const float* Bhi, const float* Blo, float* T,
                int nrows, int rp, cudaStream_t st);
// fused variant over row tiles: the epilogue sums the products over the offsets
bool tred_mac_tc_fused_supported(const tred_ctx* ctx);
int tred_mac_tc_fused(tred_ctx* ctx, const float* qhat, const float* Bhi, const float* Blo, float* opart,
                      int ntile, int t0, const void* rt_desc, const int32_t* row_m2, cudaStream_t st);

// the same on CTA pairs (tred_mac_tc2.cu)
bool tred_mac_tc2_supported(const tred_ctx* ctx);
int tred_mac_tc2(tred_ctx* ctx, const float* qhat, const float* Bhi, const float* Blo, const void* Bhb,
                 const void* Blb, float* opart, int ntile, int t0, const void* rt_desc, const int32_t* row_m2,
                 cudaStream_t st);

// three fp16 products on CTA pairs, operands pre-split by the forward FFT (tred_mac_h3.cu)
bool tred_mac_h3_supported(const tred_ctx* ctx);
int tred_mac_h3(tred_ctx* ctx, const void* qh, const float* rscale, const void* Bh16, const float* bscale,
                float* opart, int ntile, int t0, const void* rt_desc, const int32_t* row_m2, cudaStream_t st);

// forward transform as a DFT-matrix contraction on the tensor cores (tred_dft_h16.cu)
bool tred_dft_h16_supported(const tred_ctx* ctx);
int tred_dft_matrix(tred_ctx* ctx, void* d_Wd, cudaStream_t st);
int tred_dft_h16(tred_ctx* ctx, const float* payload, const int32_t* blockmap, const void* rt_desc,
                 const int32_t* row_m2, int t0, int ntile, int nstrip, const void* d_Wd,
                 void* qh, float* rscale, cudaStream_t st);

// mirror-symmetric response (tred_mac_tc2s.cu)
bool tred_mac_tc2s_supported(const tred_ctx* ctx);
int tred_mac_tc2s(tred_ctx* ctx, const float* qhat, const float* Bs_hi, const float* Bs_lo, const float* Bd_hi,
                  const float* Bd_lo, float* opart, int ntile, int t0, const void* rt_desc, const int32_t* row_m2,
                  cudaStream_t st);

static bool use_tiled(const tred_ctx* ctx) {
  return (ctx->cfg.mac_mode == 0 || ctx->cfg.mac_mode >= 3) && tred_mac_tc_fused_supported(ctx);
}

// Tensor-core path of tred_convolve: row tiles (tred_convolve_plan), forward FFT into
// qhat[f][tile * 128 + r][phase], fused spectrum product + sum over offsets per tile,
// sum of the tile patches onto the slab pixels, inverse FFT.
static int convolve_tiled(tred_ctx* ctx, int64_t nblocks, const int64_t* d_keys, const float* d_payload,
                          const float* d_rhat, const int64_t* d_sp_keys, const int32_t* h_sp_off,
                          const int32_t* h_rt_off, const PlanWork& pw, float* d_sp_data,
                          void* d_work, size_t work_bytes, cudaStream_t st) {
  const TredGrid g = make_grid(ctx);
  const tred_dims& d = ctx->dims;
  const RtGeom rg = rt_geom(ctx);
  FftPlan pl;
  if (!tred_make_fft_plan(g.L / 2, &pl)) return TRED_EUNSUPPORTED;
  const int M = g.L / 2;
  int JG = g.S;
  auto fwd_smem = [&](int jg) { return (size_t)(2 * jg * g.S * M + g.L) * sizeof(float2); };
  while (JG > 1 && (fwd_smem(JG) > 100 * 1024 || JG * g.S > 64)) --JG;
  if (fwd_smem(JG) > (size_t)ctx->smem_optin || JG * g.S > 64) return TRED_EUNSUPPORTED;
  const int ngrp = (g.S + JG - 1) / JG;
  TRED_CUDA(cudaFuncSetAttribute(k_fft_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fwd_smem(JG)));
  int IP = 8;
  auto inv_smem = [&](int ip) { return (size_t)(2 * ip * M + g.L) * sizeof(float2); };
  while (IP > 1 && inv_smem(IP) > 64 * 1024) IP /= 2;
  if (inv_smem(IP) > (size_t)ctx->smem_optin) return TRED_EUNSUPPORTED;
  TRED_CUDA(cudaFuncSetAttribute(k_ifft, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)inv_smem(IP)));

  const TiledWork w0 = carve_tiled(ctx, d_work, 1, 1);
  if (work_bytes < w0.total) return TRED_ECAP;
  {
    TredProfScope ps(ctx, ST_MISC, st);
    TRED_CUDA(cudaMemsetAsync(w0.blockmap, 0xff, (size_t)g.NBx * g.NBy * g.NBt * 4, st));
    k_fill_blockmap<<<cdiv(nblocks, 256), 256, 0, st>>>(nblocks, d_keys, w0.blockmap);
    k_fill_twiddles<<<cdiv(g.L, 256), 256, 0, st>>>(w0.tw, g.L);
    TRED_COUNT_LAUNCH(3);
  }
  const RhatLayout rl = rhat_layout(d);
  const int64_t wfl = rl.bhi, bfl = rl.blo - rl.bhi;
  // mirror-symmetric response: sums / differences of the mirror phase pairs, half-size product
  // (mac_mode 4 only: measured slower than the general product at config 3)
  const bool sym = ctx->cfg.mac_mode == 4 && ctx->sym_rhat == (const void*)d_rhat && g.nph == 100 &&
                   tred_mac_tc2s_supported(ctx) && fft_fwd_2s_available(g);
  // default: three fp16 products, the forward FFT writes the operands already split
  const bool h16 = (ctx->cfg.mac_mode == 0 || ctx->cfg.mac_mode == 7) && g.nph == 100 && (g.Bt & 3) == 0 &&
                   tred_mac_h3_supported(ctx) && fft_fwd_2s_available(g);
  if (ctx->cfg.mac_mode == 7 && !h16) return TRED_EUNSUPPORTED;
  const bool dft = h16 && ctx->cfg.fft_mode == 0 && tred_dft_h16_supported(ctx);
  ctx->last_mac_mode = 0;
  int b0 = 0;
  while (b0 < g.NBt) {
    if (h_rt_off[b0 + 1] == h_rt_off[b0]) { ++b0; continue; }
    int b1 = b0 + 1;
    while (b1 < g.NBt && carve_tiled(ctx, nullptr, 1, h_sp_off[b1 + 1] - h_sp_off[b0]).total <= work_bytes / 4) ++b1;
    const int sbase = h_sp_off[b0], nsb = h_sp_off[b1] - sbase;
    const int T0 = h_rt_off[b0], T1 = h_rt_off[b1];
    const TiledWork w1 = carve_tiled(ctx, nullptr, 1, nsb);
    if (w1.total > work_bytes) return TRED_ECAP;
    int64_t cap = 1 + (int64_t)((work_bytes - w1.total) / w1.per_tile);
    while (cap > 1 && carve_tiled(ctx, nullptr, cap, nsb).total > work_bytes) --cap;
    if (cap > T1 - T0) cap = T1 - T0;
    if (cap * RT_ROWS * (int64_t)ngrp >= (1ll << 31)) cap = ((1ll << 31) - 1) / (RT_ROWS * ngrp);

    const TiledWork w = carve_tiled(ctx, d_work, cap, nsb);
    {
      TredProfScope ps(ctx, ST_ACCUM, st);
      TRED_CUDA(cudaMemsetAsync(w.ohat, 0, (size_t)nsb * g.nf * 8, st));
      TRED_COUNT_LAUNCH(1);
    }
    for (int t0 = T0; t0 < T1; t0 += (int)cap) {
      const int nt = (int)((T1 - t0 < cap) ? (T1 - t0) : cap);
      const int rp = nt * RT_ROWS;
      {
        TredProfScope ps(ctx, ST_FFT_FWD, st);
        const RowSrc rs{nullptr, 0, pw.rt_desc, pw.row_m2, t0, rg.nstrip, 1};
        int ct = 0;
        if (dft) {
          const int rc = tred_dft_h16(ctx, d_payload, w.blockmap, pw.rt_desc, pw.row_m2, t0, nt, rg.nstrip,
                                      d_rhat + rl.wdft, w.qhat, w.rscale, st);
          if (rc != TRED_OK) return rc;
          ct = 1;
        } else
        ct = sym ? launch_fft_fwd_2s<1>(ctx, g, d_payload, w.blockmap, rs, rp, rp, w.qhat, nullptr, w.tw, st)
               : h16 ? launch_fft_fwd_2s<2>(ctx, g, d_payload, w.blockmap, rs, rp, rp, w.qhat, w.rscale, w.tw, st)
                     : launch_fft_fwd_2s<0>(ctx, g, d_payload, w.blockmap, rs, rp, rp, w.qhat, nullptr, w.tw, st);
        if ((sym || h16) && ct == 0) return TRED_EUNSUPPORTED;
        if (ct == 0) ct = launch_fft_fwd_ct(ctx, g, d_payload, w.blockmap, rs, rp, rp, w.qhat, w.tw, st);
        if (ct < 0) return ct;
        if (ct == 0)
          k_fft_fwd<<<(unsigned)(rp * ngrp), 256, fwd_smem(JG), st>>>(d_payload, w.blockmap, rs, rp, JG, w.qhat,
                                                                    w.tw, g, pl);
        TRED_COUNT_LAUNCH(1);
      }
      {
        TredProfScope ps(ctx, ST_MAC, st);
        int rc = TRED_EUNSUPPORTED;
        if (sym) {
          rc = tred_mac_tc2s(ctx, (const float*)w.qhat, d_rhat + rl.bs_hi, d_rhat + rl.bs_lo, d_rhat + rl.bd_hi,
                             d_rhat + rl.bd_lo, (float*)w.opart, nt, t0, pw.rt_desc, pw.row_m2, st);
          if (rc != TRED_OK) return rc;
          ctx->last_mac_mode = 4;
        } else if (h16) {
          rc = tred_mac_h3(ctx, w.qhat, w.rscale, d_rhat + rl.b16, d_rhat + rl.bsc, (float*)w.opart, nt, t0,
                           pw.rt_desc, pw.row_m2, st);
          if (rc != TRED_OK) return rc;
          ctx->last_mac_mode = 7;
        } else if (ctx->cfg.mac_mode != 3 && tred_mac_tc2_supported(ctx)) {
          ctx->last_mac_mode = ctx->cfg.mac_mode == 5 ? 5 : 6;
          rc = tred_mac_tc2(ctx, (const float*)w.qhat, d_rhat + wfl, d_rhat + wfl + bfl,
                            ctx->cfg.mac_mode != 5 ? (const void*)(d_rhat + rl.bhb) : nullptr,
                            ctx->cfg.mac_mode != 5 ? (const void*)(d_rhat + rl.blb) : nullptr, (float*)w.opart, nt,
                            t0, pw.rt_desc, pw.row_m2, st);
        }
        if (rc == TRED_EUNSUPPORTED) {
          ctx->last_mac_mode = 3;
          rc = tred_mac_tc_fused(ctx, (const float*)w.qhat, d_rhat + wfl, d_rhat + wfl + bfl, (float*)w.opart, nt,
                                 t0, pw.rt_desc, pw.row_m2, st);
        }
        if (rc != TRED_OK) return rc;
        TRED_COUNT_LAUNCH(1);
      }
      {
        int sa = b0;
        while (h_rt_off[sa + 1] <= t0) ++sa;
        int sb = sa;
        while (sb + 1 < b1 && h_rt_off[sb + 1] < t0 + nt) ++sb;
        const int s0 = h_sp_off[sa], ns = h_sp_off[sb + 1] - s0;
        TredProfScope ps(ctx, ST_ACCUM, st);
        if (ns > 0)
          k_accum_tiles<<<cdiv(ns, 32), 256, 0, st>>>(w.opart, d_sp_keys, s0, ns, pw.grp_off, pw.rt_desc, t0,
                                                     t0 + nt, rg.nstrip, w.ohat, sbase, g);
        TRED_COUNT_LAUNCH(1);
      }
      TRED_LAUNCH_CHECK("convolve tile chunk");
    }
    {
      TredProfScope ps(ctx, ST_IFFT, st);
      const int ct = launch_ifft_ct(ctx, g, w.ohat, sbase, nsb, sbase, d_sp_data, w.tw, d.out_len, st);
      if (ct < 0) return ct;
      if (ct == 0)
        k_ifft<<<cdiv(nsb, IP), 256, inv_smem(IP), st>>>(w.ohat, sbase, nsb, sbase, d_sp_data, w.tw, g, pl, IP,
                                                         d.out_len);
      TRED_COUNT_LAUNCH(1);
    }
    TRED_LAUNCH_CHECK("convolve ifft");
    b0 = b1;
  }
  return TRED_OK;
}

// ==================================================================== exported calls
extern "C" int tred_prepare_response(tred_ctx* ctx, const float* d_resp, float* d_rhat, void* stream) {
  if (!ctx || !d_resp || !d_rhat) return TRED_EINVAL;
  TRED_CHECK_DEVICE(ctx);
  cudaStream_t st = (cudaStream_t)stream;
  const TredGrid g = make_grid(ctx);
  const int nrows = g.nph * g.noff;
  const size_t smem = (size_t)(2 * g.L + g.Tr) * sizeof(double);
  if (smem > (size_t)ctx->smem_optin) return TRED_EUNSUPPORTED;
  TRED_CUDA(cudaFuncSetAttribute(k_resp_dft64, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const RhatLayout rl = rhat_layout(ctx->dims);
  const int64_t wfl = rl.bhi, bfl = rl.blo - rl.bhi;
  {
    TredProfScope ps(ctx, ST_RESP, st);
    TRED_CUDA(cudaMemsetAsync(d_rhat, 0, (size_t)ctx->dims.rhat_floats * 4, st));
    k_resp_dft64<<<nrows, 256, smem, st>>>(d_resp, (float2*)d_rhat, d_rhat + wfl, d_rhat + wfl + bfl,
                                           reinterpret_cast<__nv_bfloat16*>(d_rhat + rl.bhb),
                                           reinterpret_cast<__nv_bfloat16*>(d_rhat + rl.blb),
                                           g.Tr, g.L, g.noff, g.kp, g.nph);
    TRED_COUNT_LAUNCH(1);
  }
  {
    TredProfScope ps(ctx, ST_RESP, st);
    float* bsc = d_rhat + rl.bsc;
    k_resp_h16_scale<<<g.nf, 256, 0, st>>>((const float2*)d_rhat, bsc, g.nph, g.kp, g.noff);
    const int64_t n = (int64_t)g.nf * g.nph * g.noff;
    k_resp_h16<<<cdiv(n, 256), 256, 0, st>>>((const float2*)d_rhat, bsc, reinterpret_cast<__half*>(d_rhat + rl.b16),
                                            g.nf, g.nph, g.noff, g.kp, h16_kp(ctx->dims));
    TRED_COUNT_LAUNCH(2);
    if (tred_dft_h16_supported(ctx)) {
      const int rc = tred_dft_matrix(ctx, d_rhat + rl.wdft, st);
      if (rc != TRED_OK) return rc;
    }
  }
  TRED_LAUNCH_CHECK("k_resp_dft64");
  // mirror-symmetric responses get the half-size matrices as well.  This
  // is the one call that waits for the device: it runs once per response, and the host has to
  // know which path tred_convolve will take.
  if (ctx->sym_rhat == d_rhat) ctx->sym_rhat = nullptr;
  if ((g.nph & 1) == 0 && (g.noff & 1) == 1 && g.noff + 1 <= SYM_N) {
    int* flag = reinterpret_cast<int*>(d_rhat + rl.flag);
    const int64_t n = (int64_t)(g.nph / 2) * g.noff * g.Tr;
    k_resp_symcheck<<<cdiv(n, 256), 256, 0, st>>>(d_resp, g.nph, g.noff, g.Tr, flag);
    const int64_t ns = (int64_t)g.nf * ((g.noff + 1) / 2) * (g.nph / 2);
    k_resp_sym<<<cdiv(ns, 256), 256, 0, st>>>((const float2*)d_rhat, d_rhat + rl.bs_hi, d_rhat + rl.bs_lo,
                                             d_rhat + rl.bd_hi, d_rhat + rl.bd_lo, g.nf, g.nph, g.noff, g.kp);
    TRED_COUNT_LAUNCH(2);
    TRED_LAUNCH_CHECK("k_resp_sym");
    int h_flag = 1;
    TRED_CUDA(cudaMemcpyAsync(&h_flag, flag, sizeof(int), cudaMemcpyDeviceToHost, st));
    TRED_CUDA(cudaStreamSynchronize(st));
    if (h_flag == 0) ctx->sym_rhat = d_rhat;
  }
  return TRED_OK;
}

extern "C" size_t tred_plan_work_bytes(const tred_ctx* ctx) {
  return ctx ? carve_plan(ctx, nullptr).total : 0;
}

// first tile of every time tile index tb (slot NBt: the number of tiles), from the plan's scan
__global__ void k_tile_offsets(int NBt, int64_t npix, const int32_t* __restrict__ tile_idx, int32_t* __restrict__ out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i <= NBt) out[i] = tile_idx[(int64_t)i * npix];
}

int tred_plan_tile_offsets(tred_ctx* ctx, const void* d_plan_work, int32_t* d_tile_off, cudaStream_t st) {
  const PlanWork w = carve_plan(ctx, (void*)d_plan_work);
  const TredGrid g = make_grid(ctx);
  k_tile_offsets<<<cdiv(g.NBt + 1, 128), 128, 0, st>>>(g.NBt, (int64_t)g.npx * g.npy, w.tile_idx, d_tile_off);
  TRED_COUNT_LAUNCH(1);
  TRED_LAUNCH_CHECK("k_tile_offsets");
  return TRED_OK;
}

extern "C" int tred_convolve_plan(tred_ctx* ctx, int64_t nblocks, const int64_t* d_keys,
                                  int64_t cap_cp, int64_t* d_cp_keys, int32_t* d_cp_off, int64_t* d_ncp,
                                  int64_t cap_sp, int64_t* d_sp_keys, int32_t* d_sp_off, int64_t* d_nsp,
                                  int64_t cap_tiles, int64_t* d_tile_keys, int64_t* d_ntiles,
                                  int32_t* d_rt_off,
                                  void* d_plan_work, size_t plan_work_bytes, void* stream) {
  return tred_convolve_plan_dev(ctx, nblocks, nullptr, d_keys, cap_cp, d_cp_keys, d_cp_off, d_ncp, cap_sp, d_sp_keys,
                                d_sp_off, d_nsp, cap_tiles, d_tile_keys, d_ntiles, d_rt_off, d_plan_work,
                                plan_work_bytes, stream);
}

// As tred_convolve_plan with the block count read on the device: nblocks is the capacity of
// d_keys, *d_nblocks (if not NULL) the number of valid keys.
int tred_convolve_plan_dev(tred_ctx* ctx, int64_t nblocks, const int64_t* d_nblocks, const int64_t* d_keys,
                           int64_t cap_cp, int64_t* d_cp_keys, int32_t* d_cp_off, int64_t* d_ncp,
                           int64_t cap_sp, int64_t* d_sp_keys, int32_t* d_sp_off, int64_t* d_nsp,
                           int64_t cap_tiles, int64_t* d_tile_keys, int64_t* d_ntiles,
                           int32_t* d_rt_off,
                           void* d_plan_work, size_t plan_work_bytes, void* stream) {
  if (!ctx || nblocks < 0 || !d_ncp || !d_cp_off || !d_nsp || !d_ntiles || !d_sp_off || !d_rt_off)
    return TRED_EINVAL;
  TRED_CHECK_DEVICE(ctx);
  PlanWork w = carve_plan(ctx, d_plan_work);
  if (!d_plan_work || plan_work_bytes < w.total) return TRED_ECAP;
  if (nblocks > 0 && !d_keys) return TRED_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const TredGrid g = make_grid(ctx);
  const int64_t npix = (int64_t)g.npx * g.npy;
  TredProfScope ps(ctx, ST_PLAN, st);
  TRED_CUDA(cudaMemsetAsync(w.cp_idx, 0, (w.nmap + 1) * 4, st));
  TRED_CUDA(cudaMemsetAsync(w.sp_idx, 0, (w.nmap + 1) * 4, st));
  TRED_CUDA(cudaMemsetAsync(w.tile_idx, 0, (w.nmap + 1) * 4, st));
  TRED_COUNT_LAUNCH(4 + (nblocks > 0 ? 1 : 0));
  if (nblocks > 0)
    k_mark_blocks<<<cdiv(nblocks * 32, 256), 256, 0, st>>>(nblocks, d_nblocks, d_keys, w.cp_idx, w.sp_idx, g);
  int rc = tred_exclusive_scan_i32(w.cp_idx, w.cp_idx, w.nmap + 1, nullptr, w.scan, st);
  if (rc != TRED_OK) return rc;
  k_compact_keys<<<cdiv(w.nmap + 1, 256), 256, 0, st>>>(w.nmap, w.cp_idx, cap_cp, d_cp_keys, d_ncp,
                                                       d_cp_off, g.NBt, npix);
  rc = tred_exclusive_scan_i32(w.sp_idx, w.sp_idx, w.nmap + 1, nullptr, w.scan, st);
  if (rc != TRED_OK) return rc;
  k_compact_keys<<<cdiv(w.nmap + 1, 256), 256, 0, st>>>(w.nmap, w.sp_idx, cap_sp, d_sp_keys, d_nsp,
                                                       d_sp_off, g.NBt, npix);
  k_mark_tiles<<<cdiv(w.nmap, 256), 256, 0, st>>>(w.nmap, w.sp_idx, w.tile_idx, g);
  rc = tred_exclusive_scan_i32(w.tile_idx, w.tile_idx, w.nmap + 1, nullptr, w.scan, st);
  if (rc != TRED_OK) return rc;
  k_compact_keys<<<cdiv(w.nmap + 1, 256), 256, 0, st>>>(w.nmap, w.tile_idx, cap_tiles, d_tile_keys, d_ntiles,
                                                       nullptr, 0, npix);
  {
    // row tiles of the tensor-core path (strip order of the charge pixels)
    const RtGeom rg = rt_geom(ctx);
    k_rt_flags<<<cdiv(rg.nmap2 + 1, 256), 256, 0, st>>>(rg.nmap2, w.cp_idx, w.ridx, rg.nstrip, g);
    rc = tred_exclusive_scan_i32(w.ridx, w.ridx, rg.nmap2 + 1, nullptr, w.scan, st);
    if (rc != TRED_OK) return rc;
    k_rt_rows<<<cdiv(rg.nmap2, 256), 256, 0, st>>>(rg.nmap2, w.ridx, w.row_m2);
    TRED_CUDA(cudaMemsetAsync(w.grp_off, 0, (size_t)(rg.ngrp + 1) * 4, st));
    k_rt_tiles<false><<<cdiv(rg.ngrp, 128), 128, 0, st>>>(rg.ngrp, g.npy, rg.capy, w.ridx, w.grp_off, nullptr,
                                                         nullptr, 0);
    rc = tred_exclusive_scan_i32(w.grp_off, w.grp_off, rg.ngrp + 1, nullptr, w.scan, st);
    if (rc != TRED_OK) return rc;
    k_rt_tiles<true><<<cdiv(rg.ngrp, 128), 128, 0, st>>>(rg.ngrp, g.npy, rg.capy, w.ridx, nullptr, w.grp_off,
                                                        w.rt_desc, rg.cap_rt);
    k_rt_slab_off<<<cdiv(g.NBt + 1, 128), 128, 0, st>>>(g.NBt, rg.nstrip, w.grp_off, d_rt_off);
    TRED_COUNT_LAUNCH(8);
  }
  TRED_LAUNCH_CHECK("convolve_plan");
  return TRED_OK;
}

extern "C" size_t tred_convolve_work_bytes(const tred_ctx* ctx, int64_t rows_chunk, int64_t nsp_batch) {
  if (!ctx) return 0;
  if (use_tiled(ctx))      // row tiles are >= 121 rows full unless cut by a strip end or the patch height
    return carve_tiled(ctx, nullptr, rows_chunk / 100 + 2, nsp_batch).total;
  return carve_conv(ctx, nullptr, rows_chunk, nsp_batch).total;
}

extern "C" int tred_convolve(tred_ctx* ctx, int64_t nblocks, const int64_t* d_keys, const float* d_payload,
                             const float* d_rhat,
                             int64_t ncp, const int64_t* d_cp_keys, const int32_t* h_cp_off,
                             int64_t nsp, const int64_t* d_sp_keys, const int32_t* h_sp_off,
                             const int32_t* h_rt_off,
                             const void* d_plan_work, float* d_sp_data,
                             void* d_work, size_t work_bytes, void* stream) {
  if (!ctx || nblocks < 0 || nsp < 0 || ncp < 0) return TRED_EINVAL;
  TRED_CHECK_DEVICE(ctx);
  if (nblocks == 0 || nsp == 0 || ncp == 0) return TRED_OK;
  if (!d_keys || !d_payload || !d_rhat || !d_cp_keys || !h_cp_off || !d_sp_keys || !h_sp_off ||
      !d_plan_work || !d_sp_data || !d_work)
    return TRED_EINVAL;
  if (ncp >= (1ll << 31) || nsp >= (1ll << 31)) return TRED_EUNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  const TredGrid g = make_grid(ctx);
  const tred_dims& d = ctx->dims;
  if (h_cp_off[g.NBt] != ncp || h_sp_off[g.NBt] != nsp) return TRED_EINVAL;
  if (g.Bt < 2 || (g.Bt & 1)) return TRED_EUNSUPPORTED;
  const PlanWork pw = carve_plan(ctx, (void*)d_plan_work);
  if (use_tiled(ctx)) {
    if (!h_rt_off) return TRED_EINVAL;
    return convolve_tiled(ctx, nblocks, d_keys, d_payload, d_rhat, d_sp_keys, h_sp_off, h_rt_off, pw, d_sp_data,
                          d_work, work_bytes, st);
  }
  FftPlan pl;
  if (!tred_make_fft_plan(g.L / 2, &pl)) return TRED_EUNSUPPORTED;
  const int M = g.L / 2;

  // forward FFT: CG = JG*S columns per CTA, two ping-pong buffers + twiddles
  int JG = g.S;
  auto fwd_smem = [&](int jg) { return (size_t)(2 * jg * g.S * M + g.L) * sizeof(float2); };
  while (JG > 1 && (fwd_smem(JG) > 100 * 1024 || JG * g.S > 64)) --JG;
  if (fwd_smem(JG) > (size_t)ctx->smem_optin || JG * g.S > 64) return TRED_EUNSUPPORTED;
  const int ngrp = (g.S + JG - 1) / JG;
  TRED_CUDA(cudaFuncSetAttribute(k_fft_fwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fwd_smem(JG)));
  int IP = 8;
  auto inv_smem = [&](int ip) { return (size_t)(2 * ip * M + g.L) * sizeof(float2); };
  while (IP > 1 && inv_smem(IP) > 64 * 1024) IP /= 2;
  if (inv_smem(IP) > (size_t)ctx->smem_optin) return TRED_EUNSUPPORTED;
  TRED_CUDA(cudaFuncSetAttribute(k_ifft, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)inv_smem(IP)));
  const size_t mac_smem = (size_t)(g.nph * g.kp + g.nph * MAC_AS) * sizeof(float2);
  if (mac_smem > (size_t)ctx->smem_optin) return TRED_EUNSUPPORTED;
  TRED_CUDA(cudaFuncSetAttribute(k_mac_fma, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mac_smem));
  const size_t acc_smem = (size_t)g.noff * 32 * sizeof(int32_t);

  const ConvWork w0 = carve_conv(ctx, d_work, 1, 1);
  if (work_bytes < w0.total) return TRED_ECAP;
  const int64_t nbtot = (int64_t)g.NBx * g.NBy * g.NBt;
  {
    TredProfScope ps(ctx, ST_MISC, st);
    TRED_CUDA(cudaMemsetAsync(w0.blockmap, 0xff, nbtot * 4, st));
    k_fill_blockmap<<<cdiv(nblocks, 256), 256, 0, st>>>(nblocks, d_keys, w0.blockmap);
    k_fill_twiddles<<<cdiv(g.L, 256), 256, 0, st>>>(w0.tw, g.L);
    TRED_COUNT_LAUNCH(3);
  }
  const float* Wf = d_rhat;
  const RhatLayout rl = rhat_layout(d);
  const int64_t wfl = rl.bhi, bfl = rl.blo - rl.bhi;

  // slab batches (ohat of all their slab pixels resident) x row chunks (qhat, T resident)
  int b0 = 0;
  while (b0 < g.NBt) {
    if (h_cp_off[b0 + 1] == h_cp_off[b0]) { ++b0; continue; }
    int b1 = b0 + 1;
    while (b1 < g.NBt && carve_conv(ctx, nullptr, 128, h_sp_off[b1 + 1] - h_sp_off[b0]).total <= work_bytes / 4)
      ++b1;
    const int sbase = h_sp_off[b0], nsb = h_sp_off[b1] - sbase;
    const int R0 = h_cp_off[b0], R1 = h_cp_off[b1];
    // rows per chunk from the remaining workspace
    const size_t fixed = carve_conv(ctx, nullptr, 128, nsb).total - 128 * (size_t)d.conv_row_bytes;
    if (fixed + 128 * (size_t)d.conv_row_bytes > work_bytes) return TRED_ECAP;
    int64_t cap = (int64_t)((work_bytes - fixed) / (size_t)d.conv_row_bytes) / 128 * 128;
    // alignment slack of the carve
    while (cap > 128 && carve_conv(ctx, nullptr, cap, nsb).total > work_bytes) cap -= 128;
    if (cap > R1 - R0) cap = pad_rows(R1 - R0);
    const ConvWork w = carve_conv(ctx, d_work, cap, nsb);
    if (w.total > work_bytes) return TRED_ECAP;
    const int rp = (int)pad_rows(cap);
    {
      TredProfScope ps(ctx, ST_ACCUM, st);
      TRED_CUDA(cudaMemsetAsync(w.ohat, 0, (size_t)nsb * g.nf * 8, st));
      TRED_COUNT_LAUNCH(1);
    }
    for (int r0 = R0; r0 < R1; r0 += (int)cap) {
      const int nr = (int)((R1 - r0 < cap) ? (R1 - r0) : cap);
      {
        TredProfScope ps(ctx, ST_FFT_FWD, st);
        const RowSrc rs{d_cp_keys, r0, nullptr, nullptr, 0, 0, 0};
        int ct = launch_fft_fwd_2s<0>(ctx, g, d_payload, w.blockmap, rs, nr, rp, w.qhat, nullptr, w.tw, st);
        if (ct == 0) ct = launch_fft_fwd_ct(ctx, g, d_payload, w.blockmap, rs, nr, rp, w.qhat, w.tw, st);
        if (ct < 0) return ct;
        if (ct == 0)
          k_fft_fwd<<<(unsigned)(nr * ngrp), 256, fwd_smem(JG), st>>>(d_payload, w.blockmap, rs, rp, JG, w.qhat,
                                                                    w.tw, g, pl);
        TRED_COUNT_LAUNCH(1);
      }
      {
        TredProfScope ps(ctx, ST_MAC, st);
        int rc = TRED_EUNSUPPORTED;
        ctx->last_mac_mode = 2;
        if (ctx->cfg.mac_mode != 1)
          rc = tred_mac_tc(ctx, (const float*)w.qhat, d_rhat + wfl, d_rhat + wfl + bfl, (float*)w.T, nr, rp, st);
        if (rc == TRED_EUNSUPPORTED && ctx->cfg.mac_mode != 2) {
          const int ntile = (nr + MAC_MT - 1) / MAC_MT;
          int gy = (2 * ctx->num_sms + g.nf - 1) / g.nf;
          if (gy < 1) gy = 1;
          if (gy > ntile) gy = ntile;
          k_mac_fma<<<dim3(g.nf, gy), 256, mac_smem, st>>>(w.qhat, (const float2*)Wf, w.T, nr, rp, g);
          ctx->last_mac_mode = 1;
          rc = TRED_OK;
        }
        if (rc != TRED_OK) return rc;
        TRED_COUNT_LAUNCH(1);
      }
      {
        // slab pixels of the slabs this chunk's rows belong to
        int sa = b0, sb = b0;
        while (h_cp_off[sa + 1] <= r0) ++sa;
        sb = sa;
        while (sb + 1 < b1 && h_cp_off[sb + 1] < r0 + nr) ++sb;
        const int s0 = h_sp_off[sa], ns = h_sp_off[sb + 1] - s0;
        TredProfScope ps(ctx, ST_ACCUM, st);
        if (ns > 0)
          k_accum<<<cdiv(ns, 32), 256, acc_smem, st>>>(w.T, d_sp_keys, s0, ns, pw.cp_idx, r0, nr, rp, w.ohat,
                                                      sbase, g);
        TRED_COUNT_LAUNCH(1);
      }
      TRED_LAUNCH_CHECK("convolve chunk");
    }
    {
      TredProfScope ps(ctx, ST_IFFT, st);
      const int ct = launch_ifft_ct(ctx, g, w.ohat, sbase, nsb, sbase, d_sp_data, w.tw, d.out_len, st);
      if (ct < 0) return ct;
      if (ct == 0)
        k_ifft<<<cdiv(nsb, IP), 256, inv_smem(IP), st>>>(w.ohat, sbase, nsb, sbase, d_sp_data, w.tw, g, pl, IP,
                                                         d.out_len);
      TRED_COUNT_LAUNCH(1);
    }
    TRED_LAUNCH_CHECK("convolve ifft");
    b0 = b1;
  }
  return TRED_OK;
}

extern "C" int tred_gather_waveforms(tred_ctx* ctx, int64_t nsp, const float* d_sp_data,
                                     const void* d_plan_work, const void* d_tile_plan_work,
                                     int64_t tile_begin, int64_t ntiles, const int64_t* d_tile_keys,
                                     float* d_tile_data, int accumulate,
                                     int64_t npix_req, const int32_t* d_pix_ids, float* d_dense,
                                     void* stream) {
  if (!ctx || nsp < 0 || ntiles < 0 || tile_begin < 0 || npix_req < 0 || !d_plan_work) return TRED_EINVAL;
  TRED_CHECK_DEVICE(ctx);
  cudaStream_t st = (cudaStream_t)stream;
  const TredGrid g = make_grid(ctx);
  PlanWork w = carve_plan(ctx, (void*)d_plan_work);
  const PlanWork wt = carve_plan(ctx, (void*)(d_tile_plan_work ? d_tile_plan_work : d_plan_work));
  TredProfScope ps(ctx, ST_GATHER, st);
  TRED_COUNT_LAUNCH((ntiles > 0 ? 1 : 0) + (npix_req > 0 ? 1 : 0));
  if (ntiles > 0) {
    if (!d_tile_keys || !d_tile_data || (nsp > 0 && !d_sp_data)) return TRED_EINVAL;
    if (ntiles >= (1ll << 31)) return TRED_EUNSUPPORTED;
    const bool vec = (g.Bt & 3) == 0 && g.Bt <= 1024 && ((uintptr_t)d_sp_data & 15) == 0 &&
                     ((uintptr_t)d_tile_data & 15) == 0;
    if (vec) {
      const int per = 256 / (g.Bt >> 2);
      k_gather_tiles<true><<<(unsigned)((ntiles + per - 1) / per), 256, 0, st>>>(
          tile_begin, ntiles, d_tile_keys, w.sp_idx, d_sp_data, d_tile_data, accumulate, g);
    } else {
      k_gather_tiles<false><<<(unsigned)ntiles, g.Bt < 256 ? (g.Bt < 32 ? 32 : g.Bt) : 256, 0, st>>>(
          tile_begin, ntiles, d_tile_keys, w.sp_idx, d_sp_data, d_tile_data, accumulate, g);
    }
  }
  if (npix_req > 0) {
    if (!d_pix_ids || !d_dense) return TRED_EINVAL;
    if (!d_tile_data) return TRED_EINVAL;
    k_gather_dense<<<(unsigned)npix_req, 256, 0, st>>>(npix_req, d_pix_ids, wt.tile_idx, d_tile_data, d_dense, g);
  }
  TRED_LAUNCH_CHECK("gather_waveforms");
  return TRED_OK;
}
