// S4 interlaced FFT convolution (Eq. (12), L223-232 Eq. (14)) and
// S5 overlap-add on unique pixels.
//
// Per block the paper-literal form (100 zero-padded 3-D FFTs) is pruned to:
//   (a) real FFT along time of every fine column (length L >= Bt+Tr-1),
//   (b) per frequency, multiply-accumulate of the column spectra with the response
//       spectrum of the column's sub-pixel phase onto the (2H+1)^2 neighbouring pixels
//       (the pixel-plane part of Eq. (12) done directly, the time part by Eq. (14)),
//   (c) sum over all blocks of a time slab in the frequency domain (sum before the
//       inverse FFT, Eq. (14) second line), one inverse FFT per (slab, pixel),
//   (d) overlap-add of the slab outputs into tiles (pixel, Bt ticks) in fixed order.
// Spectra hold L/2 complex numbers: slot 0 packs (DC, Nyquist), both real.
#include "tred_common.cuh"

namespace {

// ------------------------------------------------------------------ shared-memory FFT
// In-place radix-2 decimation-in-time FFT of `nb` transforms of length L stored in
// x[b*L + i]; input must be in bit-reversed order, output is in natural order.
// tw[k] = exp(-2 pi i k / L), k < L/2.  inverse: conjugate twiddles, no scaling.
__device__ __forceinline__ void fft_dit_smem(float2* x, const float2* tw, int L, int logL,
                                             int nb, bool inverse, int twmul = 1) {
  const int half_total = nb * (L >> 1);
  for (int s = 1; s <= logL; ++s) {
    const int half = 1 << (s - 1);
    const int tstep = L >> s;
    for (int t = threadIdx.x; t < half_total; t += blockDim.x) {
      const int b = t / (L >> 1), r = t - b * (L >> 1);
      const int j = r & (half - 1);
      const int i0 = ((r >> (s - 1)) << s) + j + b * L;
      const int i1 = i0 + half;
      float2 w = tw[j * tstep * twmul];
      if (inverse) w.y = -w.y;
      const float2 a = x[i0], c = x[i1];
      const float2 m = make_float2(w.x * c.x - w.y * c.y, w.x * c.y + w.y * c.x);
      x[i0] = make_float2(a.x + m.x, a.y + m.y);
      x[i1] = make_float2(a.x - m.x, a.y - m.y);
    }
    __syncthreads();
  }
}

__device__ __forceinline__ void fill_twiddles(float2* tw, int L) {
  for (int k = threadIdx.x; k < (L >> 1); k += blockDim.x) {
    float sn, cs;
    sincospif(-2.0f * (float)k / (float)L, &sn, &cs);
    tw[k] = make_float2(cs, sn);
  }
}

__device__ __forceinline__ int bitrev(int i, int logL) { return (int)(__brev((unsigned)i) >> (32 - logL)); }

// Real FFT of length N = 2M through one complex FFT of length M (no pairing of two
// signals, so no rounding cross-talk between columns / pixels):
//   forward:  z[m] = x[2m] + i x[2m+1],  Z = FFT_M(z),
//             X[k] = (Z[k] + conj Z[M-k])/2 - (i/2) e^{-2 pi i k/N} (Z[k] - conj Z[M-k]),
//             X[0] = Re Z[0] + Im Z[0] (DC), X[M] = Re Z[0] - Im Z[0] (Nyquist).
//   inverse:  Z[k] = (X[k] + conj X[M-k]) + i e^{+2 pi i k/N} (X[k] - conj X[M-k]),
//             z = IFFT_M(Z) (unnormalised), x[2m] = Re z[m]/N, x[2m+1] = Im z[m]/N.
// twN[k] = exp(-2 pi i k / N), k < M; the M-point twiddles are twN[2k].
__device__ __forceinline__ float2 rfft_post(const float2* Z, const float2* twN, int M, int k) {
  if (k == 0) { const float2 z0 = Z[0]; return make_float2(z0.x + z0.y, z0.x - z0.y); }  // (DC, Nyquist)
  const float2 p = Z[k], q = Z[M - k];
  const float2 e = make_float2(0.5f * (p.x + q.x), 0.5f * (p.y - q.y));     // (Z[k] + conj Z[M-k])/2
  const float2 o = make_float2(0.5f * (p.x - q.x), 0.5f * (p.y + q.y));     // (Z[k] - conj Z[M-k])/2
  const float2 w = twN[k];
  // -i * w * o
  const float2 wo = make_float2(w.x * o.x - w.y * o.y, w.x * o.y + w.y * o.x);
  return make_float2(e.x + wo.y, e.y - wo.x);
}

// X: packed half spectrum (slot 0 = (DC, Nyquist)); returns Z[k] of the inverse.
__device__ __forceinline__ float2 rfft_pre_inverse(const float2* X, const float2* twN, int M, int k) {
  if (k == 0) { const float2 x0 = X[0]; return make_float2(x0.x + x0.y, x0.x - x0.y); }
  const float2 p = X[k], q = X[M - k];
  const float2 e = make_float2(p.x + q.x, p.y - q.y);                       // X[k] + conj X[M-k]
  const float2 o = make_float2(p.x - q.x, p.y + q.y);                       // X[k] - conj X[M-k]
  const float2 w = make_float2(twN[k].x, -twN[k].y);                        // e^{+2 pi i k/N}
  // i * w * o
  const float2 wo = make_float2(w.x * o.x - w.y * o.y, w.x * o.y + w.y * o.x);
  return make_float2(e.x - wo.y, e.y + wo.x);
}

// ------------------------------------------------------------------ response spectrum
// Computed ONCE per response, in fp64 by a direct DFT and rounded to
// fp32 at the end.  Induction-only pixels have a bipolar response whose DC bin is a
// cancellation to ~0; an fp32 FFT would leave ~1e-7 * sum|R| there, which the
// convolution multiplies by the whole collected charge.
// One CTA per response row (row = ((jx*S+jy)*K+kx)*K+ky); rhat[f][row].
__global__ void __launch_bounds__(256)
k_resp_dft64(const float* __restrict__ resp, float2* __restrict__ rhat, int nrows, int Tr, int L) {
  extern __shared__ double smd[];
  double2* tw = reinterpret_cast<double2*>(smd);       // [L]  exp(-2 pi i k / L)
  double* r = smd + 2 * L;                              // [Tr]
  const int row = blockIdx.x;
  for (int k = threadIdx.x; k < L; k += blockDim.x) {
    double sn, cs;
    sincospi(-2.0 * (double)k / (double)L, &sn, &cs);
    tw[k] = make_double2(cs, sn);
  }
  for (int i = threadIdx.x; i < Tr; i += blockDim.x) r[i] = (double)resp[(int64_t)row * Tr + i];
  __syncthreads();
  const int nf = L >> 1;
  for (int f = threadIdx.x; f <= nf; f += blockDim.x) {
    double re = 0.0, im = 0.0;
    for (int t = 0; t < Tr; ++t) {
      const double2 w = tw[(f * t) & (L - 1)];
      re += r[t] * w.x; im += r[t] * w.y;
    }
    if (f == 0) rhat[row].x = (float)re;                          // DC
    else if (f == nf) rhat[row].y = (float)re;                    // Nyquist, packed in slot 0
    else rhat[(int64_t)f * nrows + row] = make_float2((float)re, (float)im);
  }
}

// ------------------------------------------------------------------ plan (O6)
__global__ void __launch_bounds__(256)
k_mark_sp(int64_t nblocks, const int64_t* __restrict__ keys, int32_t* __restrict__ sp_flag, TredGrid g) {
  const int warp = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
  if (warp >= nblocks) return;
  const int64_t key = keys[warp];
  const int by = (int)(key % g.NBy), bx = (int)((key / g.NBy) % g.NBx);
  const int bt = (int)(key / ((int64_t)g.NBy * g.NBx));
  const int x0 = max((g.Bx * bx) / g.S - g.H, 0), x1 = min((g.Bx * bx + g.Bx - 1) / g.S + g.H, g.npx - 1);
  const int y0 = max((g.By * by) / g.S - g.H, 0), y1 = min((g.By * by + g.By - 1) / g.S + g.H, g.npy - 1);
  const int ny = y1 - y0 + 1, n = (x1 - x0 + 1) * ny;
  const int64_t base = (int64_t)bt * g.npx * g.npy;
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

// ------------------------------------------------------------------ forward FFT of blocks
// One CTA per (block of the chunk, group of CP columns).  qhat[f][slot][col].
template <int CP>
__global__ void __launch_bounds__(256)
k_fft_fwd(const float* __restrict__ payload, int blk0, int nchunk, float2* __restrict__ qhat, TredGrid g, int logM) {
  extern __shared__ float2 sm[];
  const int N = g.L, M = N >> 1;
  float2* Z = sm;                 // [CP][M]
  float2* tw = sm + CP * M;       // [M]  exp(-2 pi i k / N)
  const int ncols = g.Bx * g.By;
  const int groups = ncols / CP;
  const int slot = blockIdx.x / groups, grp = blockIdx.x - slot * groups;
  const int col0 = grp * CP;
  fill_twiddles(tw, N);
  const float2* src = reinterpret_cast<const float2*>(payload + ((int64_t)(blk0 + slot) * ncols + col0) * g.Bt);
  const int hb = g.Bt >> 1;       // float2 samples per column
  for (int i = threadIdx.x; i < CP * M; i += blockDim.x) {
    const int c = i / M, m = i - c * M;
    float2 v = make_float2(0.0f, 0.0f);
    if (m < hb) v = src[c * hb + m];
    Z[c * M + bitrev(m, logM)] = v;
  }
  __syncthreads();
  fft_dit_smem(Z, tw, M, logM, CP, false, 2);
  for (int i = threadIdx.x; i < M * CP; i += blockDim.x) {
    const int f = i / CP, c = i - f * CP;
    qhat[((int64_t)f * nchunk + slot) * ncols + col0 + c] = rfft_post(Z + c * M, tw, M, f);
  }
}

// ------------------------------------------------------------------ class bundles
// Blocks whose origin has the same sub-pixel alignment (class) share the map
// column -> (phase, pixel offset); the MAC kernel tiles NB such blocks per thread.
constexpr int MAC_NB = 8;

struct ClassInfo { int pcx, pcy, ncls; };

__device__ __forceinline__ int block_class(int64_t key, const TredGrid& g, const ClassInfo& ci) {
  const int by = (int)(key % g.NBy), bx = (int)((key / g.NBy) % g.NBx);
  return (bx % ci.pcx) * ci.pcy + (by % ci.pcy);
}

__global__ void __launch_bounds__(256)
k_class_count(const int64_t* __restrict__ keys, int blk0, int nchunk, int32_t* __restrict__ cls_cnt,
              TredGrid g, ClassInfo ci) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nchunk) return;
  atomicAdd(&cls_cnt[block_class(keys[blk0 + i], g, ci)], 1);
}

// single warp: class offsets, bundle table {class, start, count}; resets the cursors
__global__ void k_class_scan(int32_t* __restrict__ cls_cnt, int32_t* __restrict__ cls_off,
                             int32_t* __restrict__ cls_cur, int32_t* __restrict__ bundles,
                             int32_t* __restrict__ nbundles, int ncls) {
  if (threadIdx.x != 0) return;
  int off = 0, nb = 0;
  for (int c = 0; c < ncls; ++c) {
    const int n = cls_cnt[c];
    cls_off[c] = off; cls_cur[c] = 0;
    for (int s = 0; s < n; s += MAC_NB) {
      bundles[3 * nb + 0] = c; bundles[3 * nb + 1] = off + s; bundles[3 * nb + 2] = min(MAC_NB, n - s);
      ++nb;
    }
    off += n;
  }
  *nbundles = nb;
}

__global__ void __launch_bounds__(256)
k_class_place(const int64_t* __restrict__ keys, int blk0, int nchunk, const int32_t* __restrict__ cls_off,
              int32_t* __restrict__ cls_cur, int32_t* __restrict__ order, TredGrid g, ClassInfo ci) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nchunk) return;
  const int c = block_class(keys[blk0 + i], g, ci);
  order[cls_off[c] + atomicAdd(&cls_cur[c], 1)] = i;   // order inside a class does not change results
}

// ------------------------------------------------------------------ spectrum MAC
// grid (L/2, Y).  CTA: response spectrum of one frequency in shared memory
// W[jx][jy][kx][ky]; G thread groups of OUTP threads, one output pixel of the block
// footprint per thread, MAC_NB blocks of one class per thread (register tile).
// chat[slot][f][rel].
struct MacParams {
  int outp;      // outx*outy
  int gthreads;  // threads per group (outp rounded up to a warp multiple)
  int G;         // groups per CTA
  int nrows;     // S*S*K*K
};

__global__ void __launch_bounds__(1024)
k_mac(const float2* __restrict__ qhat, const float2* __restrict__ rhat, float2* __restrict__ chat,
      const int32_t* __restrict__ order, const int32_t* __restrict__ bundles,
      const int32_t* __restrict__ nbundles_p, int nchunk, TredGrid g, ClassInfo ci, MacParams mp) {
  extern __shared__ float2 sm[];
  float2* W = sm;                                   // [nrows]
  const int ncols = g.Bx * g.By;
  float2* Qs_all = sm + mp.nrows;                   // [G][ncols][MAC_NB]
  const int f = blockIdx.x;
  const int nf = g.L >> 1;
  const int grp = threadIdx.x / mp.gthreads, tg = threadIdx.x - grp * mp.gthreads;
  float2* Qs = Qs_all + (size_t)grp * ncols * MAC_NB;
  const int K = 2 * g.H + 1;

  for (int i = threadIdx.x; i < mp.nrows; i += blockDim.x) W[i] = rhat[(int64_t)f * mp.nrows + i];
  const int nbundles = *nbundles_p;
  const bool packed = (f == 0);          // slot 0 holds (DC, Nyquist): two real products
  const int u = tg / g.outy, v = tg - u * g.outy;   // output pixel relative to footprint corner
  const bool active = tg < mp.outp;
  __syncthreads();

  const int stride = gridDim.y * mp.G;
  const int iters = (nbundles + stride - 1) / stride;
  for (int it = 0; it < iters; ++it) {
    const int j = it * stride + blockIdx.y * mp.G + grp;
    const bool have = j < nbundles;
    int cls = 0, start = 0, cnt = 0;
    if (have) { cls = bundles[3 * j]; start = bundles[3 * j + 1]; cnt = bundles[3 * j + 2]; }
    // stage the column spectra of the bundle's blocks: Qs[col][b]
    for (int i = tg; i < ncols * MAC_NB; i += mp.gthreads) {
      const int b = i / ncols, c = i - b * ncols;
      float2 q = make_float2(0.0f, 0.0f);
      if (b < cnt) q = qhat[((int64_t)f * nchunk + order[start + b]) * ncols + c];
      Qs[c * MAC_NB + b] = q;
    }
    __syncthreads();
    if (have && active) {
      const int ox = (g.Bx * (cls / ci.pcy)) % g.S, oy = (g.By * (cls % ci.pcy)) % g.S;
      float2 acc[MAC_NB];
#pragma unroll
      for (int b = 0; b < MAC_NB; ++b) acc[b] = make_float2(0.0f, 0.0f);
      for (int cx = 0; cx < g.Bx; ++cx) {
        const int fx = ox + cx, Px = fx / g.S, jx = fx - Px * g.S;
        const int kx = u - Px;                       // = displacement + H
        if (kx < 0 || kx >= K) continue;
        for (int cy = 0; cy < g.By; ++cy) {
          const int fy = oy + cy, Py = fy / g.S, jy = fy - Py * g.S;
          const int ky = v - Py;
          if (ky < 0 || ky >= K) continue;
          const float2 w = W[((jx * g.S + jy) * K + kx) * K + ky];
          const float w_im_self = packed ? w.y : w.x;    // multiplies q.im into acc.im
          const float w_cross = packed ? 0.0f : w.y;
          const float4* q4 = reinterpret_cast<const float4*>(Qs + (cx * g.By + cy) * MAC_NB);
#pragma unroll
          for (int b2 = 0; b2 < MAC_NB / 2; ++b2) {
            const float4 q = q4[b2];
            acc[2 * b2].x = fmaf(w.x, q.x, acc[2 * b2].x);
            acc[2 * b2].x = fmaf(-w_cross, q.y, acc[2 * b2].x);
            acc[2 * b2].y = fmaf(w_im_self, q.y, acc[2 * b2].y);
            acc[2 * b2].y = fmaf(w_cross, q.x, acc[2 * b2].y);
            acc[2 * b2 + 1].x = fmaf(w.x, q.z, acc[2 * b2 + 1].x);
            acc[2 * b2 + 1].x = fmaf(-w_cross, q.w, acc[2 * b2 + 1].x);
            acc[2 * b2 + 1].y = fmaf(w_im_self, q.w, acc[2 * b2 + 1].y);
            acc[2 * b2 + 1].y = fmaf(w_cross, q.z, acc[2 * b2 + 1].y);
          }
        }
      }
#pragma unroll
      for (int b = 0; b < MAC_NB; ++b)
        if (b < cnt) chat[((int64_t)order[start + b] * nf + f) * mp.outp + tg] = acc[b];
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------ sum over blocks of a slab
// One CTA per slab-pixel of the chunk: collects, in ascending (bx, by) order, the blocks
// of its slab whose footprint holds the pixel, then sums their spectra per frequency.
constexpr int ACC_MAXHIT = 1024;

__global__ void __launch_bounds__(256)
k_accum(const float2* __restrict__ chat, const int64_t* __restrict__ sp_keys, int sp0, int nsp_chunk,
        const int32_t* __restrict__ blockmap, int blk0, float2* __restrict__ ohat, TredGrid g, int outp) {
  __shared__ int hit_slot[ACC_MAXHIT];
  __shared__ int hit_rel[ACC_MAXHIT];
  __shared__ int nhit_s;
  const int spl = blockIdx.x;
  const int64_t key = sp_keys[sp0 + spl];
  const int py = (int)(key % g.npy), px = (int)((key / g.npy) % g.npx);
  const int bt = (int)(key / ((int64_t)g.npy * g.npx));
  const int bx_lo = max(0, ((px - g.H) * g.S - (g.Bx - 1) + 1024 * g.Bx) / g.Bx - 1024);
  const int bx_hi = min(g.NBx - 1, ((px + g.H) * g.S + g.S - 1) / g.Bx);
  const int by_lo = max(0, ((py - g.H) * g.S - (g.By - 1) + 1024 * g.By) / g.By - 1024);
  const int by_hi = min(g.NBy - 1, ((py + g.H) * g.S + g.S - 1) / g.By);
  const int ncy = by_hi - by_lo + 1, ncand = (bx_hi - bx_lo + 1) * ncy;
  if (threadIdx.x < 32) {
    int nhit = 0;
    for (int base = 0; base < ncand; base += 32) {
      const int i = base + threadIdx.x;
      int slot = -1, rel = 0;
      if (i < ncand) {
        const int bx = bx_lo + i / ncy, by = by_lo + i % ncy;
        const int P0x = (g.Bx * bx) / g.S, P1x = (g.Bx * bx + g.Bx - 1) / g.S;
        const int P0y = (g.By * by) / g.S, P1y = (g.By * by + g.By - 1) / g.S;
        if (px >= P0x - g.H && px <= P1x + g.H && py >= P0y - g.H && py <= P1y + g.H) {
          const int m = blockmap[((int64_t)bt * g.NBx + bx) * g.NBy + by];
          if (m >= 0) { slot = m - blk0; rel = (px - (P0x - g.H)) * g.outy + (py - (P0y - g.H)); }
        }
      }
      const unsigned bal = __ballot_sync(0xffffffffu, slot >= 0);
      if (slot >= 0) {
        const int pos = nhit + __popc(bal & ((1u << threadIdx.x) - 1u));
        if (pos < ACC_MAXHIT) { hit_slot[pos] = slot; hit_rel[pos] = rel; }
      }
      nhit += __popc(bal);
    }
    if (threadIdx.x == 0) nhit_s = min(nhit, ACC_MAXHIT);
  }
  __syncthreads();
  const int nhit = nhit_s, nf = g.L >> 1;
  for (int f = threadIdx.x; f < nf; f += blockDim.x) {
    float2 a = make_float2(0.0f, 0.0f);
    for (int h = 0; h < nhit; ++h) {
      const float2 c = chat[((int64_t)hit_slot[h] * nf + f) * outp + hit_rel[h]];
      a.x += c.x; a.y += c.y;
    }
    ohat[(int64_t)spl * nf + f] = a;
  }
}

__global__ void __launch_bounds__(256)
k_fill_blockmap(int64_t nblocks, const int64_t* __restrict__ keys, int32_t* __restrict__ blockmap) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < nblocks) blockmap[keys[i]] = (int32_t)i;
}

// ------------------------------------------------------------------ inverse FFT
// One CTA per IP slab-pixels; sp_data[sp][n_over*Bt].
template <int IP>
__global__ void __launch_bounds__(256)
k_ifft(const float2* __restrict__ ohat, int sp0, int nsp_chunk, float* __restrict__ sp_data, TredGrid g,
       int logM, int out_len) {
  extern __shared__ float2 sm[];
  const int N = g.L, M = N >> 1;
  float2* Z = sm;                 // [IP][M]
  float2* X = sm + IP * M;        // [IP][M] staged spectra
  float2* tw = sm + 2 * IP * M;   // [M]
  const int a0 = blockIdx.x * IP;
  fill_twiddles(tw, N);
  for (int i = threadIdx.x; i < IP * M; i += blockDim.x) {
    const int c = i / M, k = i - c * M;
    X[i] = (a0 + c < nsp_chunk) ? ohat[(int64_t)(a0 + c) * M + k] : make_float2(0.0f, 0.0f);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < IP * M; i += blockDim.x) {
    const int c = i / M, k = i - c * M;
    Z[c * M + bitrev(k, logM)] = rfft_pre_inverse(X + c * M, tw, M, k);
  }
  __syncthreads();
  fft_dit_smem(Z, tw, M, logM, IP, true, 2);
  const int row = g.nover * g.Bt, hrow = row >> 1;
  const float sc = 1.0f / (float)N;
  for (int i = threadIdx.x; i < IP * hrow; i += blockDim.x) {
    const int c = i / hrow, m = i - c * hrow;
    if (a0 + c >= nsp_chunk) continue;
    const float2 z = Z[c * M + m];
    float2 v;
    v.x = (2 * m < out_len) ? z.x * sc : 0.0f;
    v.y = (2 * m + 1 < out_len) ? z.y * sc : 0.0f;
    reinterpret_cast<float2*>(sp_data + (int64_t)(sp0 + a0 + c) * row)[m] = v;
  }
}

// ------------------------------------------------------------------ S5 overlap-add
__global__ void __launch_bounds__(256)
k_gather_tiles(int64_t ntiles, const int64_t* __restrict__ tile_keys, const int32_t* __restrict__ sp_idx,
               const float* __restrict__ sp_data, float* __restrict__ tile_data, TredGrid g) {
  const int64_t tile = blockIdx.x;
  const int64_t key = tile_keys[tile];
  const int64_t npix = (int64_t)g.npx * g.npy;
  const int tb = (int)(key / npix);
  const int64_t p = key - tb * npix;
  const int row = g.nover * g.Bt;
  for (int t = threadIdx.x; t < g.Bt; t += blockDim.x) {
    float acc = 0.0f;
    for (int bt = max(tb - g.nover + 1, 0); bt <= tb; ++bt) {        // ascending slab order
      const int64_t m = bt * npix + p;
      const int i0 = sp_idx[m];
      if (sp_idx[m + 1] != i0) acc += sp_data[(int64_t)i0 * row + (tb - bt) * g.Bt + t];
    }
    if (tb * g.Bt + t >= g.nticks) acc = 0.0f;
    tile_data[tile * g.Bt + t] = acc;
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

static int ilog2(int x) { int l = 0; while ((1 << l) < x) ++l; return l; }
static int gcd_i(int a, int b) { while (b) { int t = a % b; a = b; b = t; } return a; }

static ClassInfo make_class(const TredGrid& g) {
  ClassInfo ci;
  ci.pcx = g.S / gcd_i(g.S, g.Bx);
  ci.pcy = g.S / gcd_i(g.S, g.By);
  ci.ncls = ci.pcx * ci.pcy;
  return ci;
}

struct PlanWork { int32_t* sp_idx; int32_t* tile_idx; void* scan; size_t total; int64_t nmap; };

static PlanWork carve_plan(const tred_ctx* c, void* base) {
  PlanWork w;
  size_t o = 0; char* b = (char*)base;
  auto take = [&](size_t bytes) { void* p = b ? b + o : nullptr; o += align_up(bytes, 256); return p; };
  w.nmap = (int64_t)c->dims.NB[2] * c->cfg.npix_x * c->cfg.npix_y;
  w.sp_idx = (int32_t*)take((w.nmap + 1) * 4);
  w.tile_idx = (int32_t*)take((w.nmap + 1) * 4);
  w.scan = take(tred_scan_work_bytes(w.nmap + 1));
  w.total = o;
  return w;
}

struct ConvWork {
  int32_t* blockmap; float2* qhat; float2* chat; float2* ohat;
  int32_t *order, *cls_cnt, *cls_off, *cls_cur, *bundles, *nbundles;
  size_t total;
};

static ConvWork carve_conv(const tred_ctx* c, void* base, int64_t nb, int64_t ns) {
  ConvWork w;
  size_t o = 0; char* b = (char*)base;
  auto take = [&](size_t bytes) { void* p = b ? b + o : nullptr; o += align_up(bytes, 256); return p; };
  const tred_dims& d = c->dims;
  const int64_t L = d.fft_len, ncols = (int64_t)c->cfg.block[0] * c->cfg.block[1];
  const int64_t outp = (int64_t)d.out_px * d.out_py;
  if (nb < 1) nb = 1;
  if (ns < 1) ns = 1;
  w.blockmap = (int32_t*)take((size_t)(d.NB[0] * d.NB[1] * d.NB[2]) * 4);
  w.qhat = (float2*)take((size_t)nb * ncols * L * 4);
  w.chat = (float2*)take((size_t)nb * outp * L * 4);
  w.ohat = (float2*)take((size_t)(ns + 1) * L * 4);
  w.order = (int32_t*)take((size_t)nb * 4);
  w.cls_cnt = (int32_t*)take((size_t)d.n_class * 4);
  w.cls_off = (int32_t*)take((size_t)d.n_class * 4);
  w.cls_cur = (int32_t*)take((size_t)d.n_class * 4);
  w.bundles = (int32_t*)take((size_t)(nb / MAC_NB + d.n_class + 1) * 3 * 4);
  w.nbundles = (int32_t*)take(4);
  w.total = o;
  return w;
}

}  // namespace

// ==================================================================== exported calls
extern "C" int tred_prepare_response(tred_ctx* ctx, const float* d_resp, float* d_rhat, void* stream) {
  if (!ctx || !d_resp || !d_rhat) return TRED_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const TredGrid g = make_grid(ctx);
  const int K = 2 * g.H + 1, nrows = g.S * g.S * K * K;
  const size_t smem = (size_t)(2 * g.L + g.Tr) * sizeof(double);
  if (smem > (size_t)ctx->smem_optin) return TRED_EUNSUPPORTED;
  TRED_CUDA(cudaFuncSetAttribute(k_resp_dft64, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  {
    TredProfScope ps(ctx, ST_RESP, st);
    k_resp_dft64<<<nrows, 256, smem, st>>>(d_resp, (float2*)d_rhat, nrows, g.Tr, g.L);
    TRED_COUNT_LAUNCH(1);
  }
  TRED_LAUNCH_CHECK("k_resp_dft64");
  return TRED_OK;
}

extern "C" size_t tred_plan_work_bytes(const tred_ctx* ctx) {
  return ctx ? carve_plan(ctx, nullptr).total : 0;
}

extern "C" int tred_convolve_plan(tred_ctx* ctx, int64_t nblocks, const int64_t* d_keys,
                                  int64_t cap_sp, int64_t* d_sp_keys, int32_t* d_sp_off, int64_t* d_nsp,
                                  int64_t cap_tiles, int64_t* d_tile_keys, int64_t* d_ntiles,
                                  void* d_plan_work, size_t plan_work_bytes, void* stream) {
  if (!ctx || nblocks < 0 || !d_nsp || !d_ntiles || !d_sp_off) return TRED_EINVAL;
  PlanWork w = carve_plan(ctx, d_plan_work);
  if (!d_plan_work || plan_work_bytes < w.total) return TRED_ECAP;
  if (nblocks > 0 && !d_keys) return TRED_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const TredGrid g = make_grid(ctx);
  const int64_t npix = (int64_t)g.npx * g.npy;
  TredProfScope ps(ctx, ST_PLAN, st);
  TRED_CUDA(cudaMemsetAsync(w.sp_idx, 0, (w.nmap + 1) * 4, st));
  TRED_CUDA(cudaMemsetAsync(w.tile_idx, 0, (w.nmap + 1) * 4, st));
  TRED_COUNT_LAUNCH(3 + (nblocks > 0 ? 1 : 0));
  if (nblocks > 0) k_mark_sp<<<cdiv(nblocks * 32, 256), 256, 0, st>>>(nblocks, d_keys, w.sp_idx, g);
  int rc = tred_exclusive_scan_i32(w.sp_idx, w.sp_idx, w.nmap + 1, nullptr, w.scan, st);
  if (rc != TRED_OK) return rc;
  k_compact_keys<<<cdiv(w.nmap + 1, 256), 256, 0, st>>>(w.nmap, w.sp_idx, cap_sp, d_sp_keys, d_nsp,
                                                       d_sp_off, g.NBt, npix);
  k_mark_tiles<<<cdiv(w.nmap, 256), 256, 0, st>>>(w.nmap, w.sp_idx, w.tile_idx, g);
  rc = tred_exclusive_scan_i32(w.tile_idx, w.tile_idx, w.nmap + 1, nullptr, w.scan, st);
  if (rc != TRED_OK) return rc;
  k_compact_keys<<<cdiv(w.nmap + 1, 256), 256, 0, st>>>(w.nmap, w.tile_idx, cap_tiles, d_tile_keys, d_ntiles,
                                                       nullptr, 0, npix);
  TRED_LAUNCH_CHECK("convolve_plan");
  return TRED_OK;
}

extern "C" size_t tred_convolve_work_bytes(const tred_ctx* ctx, int64_t nblocks_chunk, int64_t nsp_chunk) {
  return ctx ? carve_conv(ctx, nullptr, nblocks_chunk, nsp_chunk).total : 0;
}

extern "C" int tred_convolve(tred_ctx* ctx, int64_t nblocks, const int64_t* d_keys,
                             const int32_t* h_slab_off, const float* d_payload, const float* d_rhat,
                             int64_t nsp, const int64_t* d_sp_keys, const int32_t* h_sp_off,
                             const void* d_plan_work, float* d_sp_data,
                             void* d_work, size_t work_bytes, void* stream) {
  if (!ctx || nblocks < 0 || nsp < 0) return TRED_EINVAL;
  if (nblocks == 0 || nsp == 0) return TRED_OK;
  if (!d_keys || !h_slab_off || !d_payload || !d_rhat || !d_sp_keys || !h_sp_off || !d_sp_data || !d_work)
    return TRED_EINVAL;
  (void)d_plan_work;
  cudaStream_t st = (cudaStream_t)stream;
  const TredGrid g = make_grid(ctx);
  const ClassInfo ci = make_class(g);
  const int logL = ilog2(g.L), nf = g.L / 2;
  const int ncols = g.Bx * g.By, outp = g.outx * g.outy;
  const int K = 2 * g.H + 1;
  if (h_slab_off[g.NBt] != nblocks || h_sp_off[g.NBt] != nsp) return TRED_EINVAL;
  if (ncols < 8) return TRED_EUNSUPPORTED;

  MacParams mp;
  mp.outp = outp; mp.gthreads = (outp + 31) / 32 * 32; mp.nrows = g.S * g.S * K * K;
  mp.G = 2;
  while (mp.G > 1 && mp.G * mp.gthreads > 1024) --mp.G;
  if (mp.gthreads > 1024) return TRED_EUNSUPPORTED;
  const size_t mac_smem = ((size_t)mp.nrows + (size_t)mp.G * ncols * MAC_NB) * sizeof(float2);
  if (mac_smem > (size_t)ctx->smem_optin) return TRED_EUNSUPPORTED;
  TRED_CUDA(cudaFuncSetAttribute(k_mac, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)mac_smem));
  constexpr int CP = 8, IP = 4;
  const int M = g.L / 2, logM = logL - 1;
  if (g.Bt < 2) return TRED_EUNSUPPORTED;
  const size_t fft_smem = (size_t)(CP * M + M) * sizeof(float2);
  TRED_CUDA(cudaFuncSetAttribute(k_fft_fwd<CP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fft_smem));
  const size_t ifft_smem = (size_t)(2 * IP * M + M) * sizeof(float2);
  TRED_CUDA(cudaFuncSetAttribute(k_ifft<IP>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ifft_smem));

  // block map of the whole event (lives at the start of the workspace)
  ConvWork w0 = carve_conv(ctx, d_work, 1, 1);
  if (work_bytes < w0.total) return TRED_ECAP;
  const int64_t nbtot = (int64_t)g.NBx * g.NBy * g.NBt;
  {
    TredProfScope ps(ctx, ST_CLASS, st);
    TRED_CUDA(cudaMemsetAsync(w0.blockmap, 0xff, nbtot * 4, st));
    k_fill_blockmap<<<cdiv(nblocks, 256), 256, 0, st>>>(nblocks, d_keys, w0.blockmap);
    TRED_COUNT_LAUNCH(1);
  }

  // process the slabs in groups that fit the workspace
  int s0 = 0;
  while (s0 < g.NBt) {
    int s1 = s0 + 1;
    while (s1 < g.NBt &&
           carve_conv(ctx, nullptr, h_slab_off[s1 + 1] - h_slab_off[s0], h_sp_off[s1 + 1] - h_sp_off[s0]).total
               <= work_bytes)
      ++s1;
    const int blk0 = h_slab_off[s0], nb = h_slab_off[s1] - blk0;
    const int sp0 = h_sp_off[s0], ns = h_sp_off[s1] - sp0;
    s0 = s1;
    if (nb == 0 || ns == 0) continue;
    ConvWork w = carve_conv(ctx, d_work, nb, ns);
    if (w.total > work_bytes) return TRED_ECAP;
    {
      TredProfScope ps(ctx, ST_FFT_FWD, st);
      k_fft_fwd<CP><<<nb * (ncols / CP), 256, fft_smem, st>>>(d_payload, blk0, nb, w.qhat, g, logM);
      TRED_COUNT_LAUNCH(1);
    }
    {
      TredProfScope ps(ctx, ST_CLASS, st);
      TRED_CUDA(cudaMemsetAsync(w.cls_cnt, 0, ci.ncls * 4, st));
      k_class_count<<<cdiv(nb, 256), 256, 0, st>>>(d_keys, blk0, nb, w.cls_cnt, g, ci);
      k_class_scan<<<1, 32, 0, st>>>(w.cls_cnt, w.cls_off, w.cls_cur, w.bundles, w.nbundles, ci.ncls);
      k_class_place<<<cdiv(nb, 256), 256, 0, st>>>(d_keys, blk0, nb, w.cls_off, w.cls_cur, w.order, g, ci);
      TRED_COUNT_LAUNCH(3);
    }
    const int nb_ub = nb / MAC_NB + ci.ncls;
    int gy = (nb_ub + mp.G * 16 - 1) / (mp.G * 16);
    if (gy < 1) gy = 1;
    if (gy > 65535) gy = 65535;
    {
      TredProfScope ps(ctx, ST_MAC, st);
      k_mac<<<dim3(nf, gy), mp.G * mp.gthreads, mac_smem, st>>>(w.qhat, (const float2*)d_rhat, w.chat, w.order,
                                                                w.bundles, w.nbundles, nb, g, ci, mp);
      TRED_COUNT_LAUNCH(1);
    }
    {
      TredProfScope ps(ctx, ST_ACCUM, st);
      k_accum<<<ns, 256, 0, st>>>(w.chat, d_sp_keys, sp0, ns, w0.blockmap, blk0, w.ohat, g, outp);
      TRED_COUNT_LAUNCH(1);
    }
    {
      TredProfScope ps(ctx, ST_IFFT, st);
      k_ifft<IP><<<(ns + IP - 1) / IP, 256, ifft_smem, st>>>(w.ohat, sp0, ns, d_sp_data, g, logM, ctx->dims.out_len);
      TRED_COUNT_LAUNCH(1);
    }
    TRED_LAUNCH_CHECK("convolve chunk");
  }
  return TRED_OK;
}

extern "C" int tred_gather_waveforms(tred_ctx* ctx, int64_t nsp, const float* d_sp_data,
                                     const void* d_plan_work,
                                     int64_t ntiles, const int64_t* d_tile_keys, float* d_tile_data,
                                     int64_t npix_req, const int32_t* d_pix_ids, float* d_dense,
                                     void* stream) {
  if (!ctx || nsp < 0 || ntiles < 0 || npix_req < 0 || !d_plan_work) return TRED_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  const TredGrid g = make_grid(ctx);
  PlanWork w = carve_plan(ctx, (void*)d_plan_work);
  TredProfScope ps(ctx, ST_GATHER, st);
  TRED_COUNT_LAUNCH((ntiles > 0 ? 1 : 0) + (npix_req > 0 ? 1 : 0));
  if (ntiles > 0) {
    if (!d_tile_keys || !d_tile_data || (nsp > 0 && !d_sp_data)) return TRED_EINVAL;
    if (ntiles >= (1ll << 31)) return TRED_EUNSUPPORTED;
    k_gather_tiles<<<(unsigned)ntiles, g.Bt < 256 ? (g.Bt < 32 ? 32 : g.Bt) : 256, 0, st>>>(
        ntiles, d_tile_keys, w.sp_idx, d_sp_data, d_tile_data, g);
  }
  if (npix_req > 0) {
    if (!d_pix_ids || !d_dense) return TRED_EINVAL;
    k_gather_dense<<<(unsigned)npix_req, 256, 0, st>>>(npix_req, d_pix_ids, w.tile_idx, d_tile_data, d_dense, g);
  }
  TRED_LAUNCH_CHECK("gather_waveforms");
  return TRED_OK;
}
