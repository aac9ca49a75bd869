// Forward transform of Eq. (14) as a dense DFT-matrix contraction on the
// tensor cores, writing the spectra straight in the operand format of the spectrum product
// (tred_mac_h3.cu: fp16 hi / lo parts in blocks of 16 reals, one power-of-two scale per row).
//
// Why a contraction: a block column holds only Bt (<= 128) non-zero ticks of the L-point
// transform, so the pruned DFT  X[n] = sum_t q[t] W[t][n],  n = 2 f + (re | im),  is a
// [columns x Bt] x [Bt x L] product -- 2 Bt L flops per column against ~2.5 L log2 L for an
// FFT, but on the tensor cores, with no shared-memory butterflies, and the kernel is bound by
// writing the spectra to HBM (the shared-memory FFT kernel k_fft_fwd_2s is bound by its
// L1 / shared-memory traffic at less than half of that rate).
//
// One work item = one charge pixel (row): its S*S = 100 fine columns are the M rows of the
// product (lanes 100..127 idle), K = Bt ticks, N = L reals in chunks of NC <= 256 columns.
// CTA pairs (cta_group::2, M = 256): each CTA converts its own row and holds ITS HALF of the
// whole DFT matrix resident in shared memory (loaded once per kernel), so the only traffic of
// the main loop is the payload in and the spectra out.  Three fp16 products per K step,
//     D += A_hi W_hi,  D += A_lo W_hi,  D += A_hi W_lo,
// with A = q / s_row and W = exp(-2 pi i f t / L), both split hi + lo (22 bits; the lo part
// of W is <= 2^-12 and partly subnormal in fp16, absolute error <= 2^-25: fp32 level).
//
// Per CTA: warp 1 MMA issuer (leader CTA only), warps 2-9 epilogue (TMEM -> registers ->
// fp16 hi / lo -> global, one lane per fine column, two warps per TMEM lane quadrant taking
// alternate groups of 16 frequencies, 32-byte sectors written whole), warps 10-17 converters (payload -> registers, sum |q| -> row scale, fp16 hi / lo -> the swizzled A
// tile).  The A tile is single-buffered (the DFT matrix takes the rest of shared memory): the
// converters fetch the next row into registers while the tensor core works and only store it
// once the last MMA of the current row has retired.
#include <cuda_fp16.h>
#include "tred_tc2_common.cuh"

namespace {

constexpr int DF_THREADS = 576;          // 18 warps: W loader, MMA issuer, 8 epilogue, 8 converters
constexpr int DF_EPI0 = 2 * 32;          // first epilogue thread
constexpr int DF_CONV0 = 10 * 32;        // first converter thread
constexpr int DF_NCONV = 256;            // converter threads
constexpr int DF_MAXF4 = 13;             // float4 per converter thread: ceil(100 * 32 / 256)
constexpr int DF_NPH = 100;              // fine columns per charge pixel (S = 10)
constexpr int DF_KP16 = (2 * DF_NPH + 15) / 16 * 32;          // halves per row of spectra
constexpr int DF_FSTRIDE = RT_ROWS * DF_KP16;                 // halves between the planes of f and f + 1

struct DftParams {
  int nrows, row0;              // compact rows of the chunk: row_m2[row0 .. row0 + nrows); read from rt_desc
  int t0, ntile, rp;            // row tiles of the chunk, padded rows = ntile * 128
  int nf, Bt, nkc, nnc, NC;     // K chunks of 32 ticks, N chunks of NC reals
  int kp16;                     // halves per output row
  const int4* rt_desc;
  const int32_t* row_m2;
  const int32_t* blockmap;
  const float* payload;
  __half* qh;                   // [tile][nf][128][kp16]: the (row tile, frequency) box the spectrum product loads
                                // is one contiguous 104 KB run
  float* rscale;                // [rp]
  TredGrid g;
  int nstrip;
};

__device__ __forceinline__ void tc_mma_f16_pair2(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                                 uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ uint64_t desc_sw128(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3ffff) >> 4);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)(1024 >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;
  return d;
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(bar)
      : "memory");
}
// Wait of a whole warp group on an mbarrier: one warp polls (try_wait with a suspend-time hint),
// the others sleep at the named barrier `bar` (nthreads wide) instead of spending issue slots.
__device__ __forceinline__ void group_wait(uint32_t mbar, uint32_t parity, bool poller, uint32_t bar, uint32_t nthreads) {
  if (poller) {
    uint32_t ok = 0;
    long long t0 = 0;
    for (int it = 0; !ok; ++it) {
      asm volatile(
          "{\n\t.reg .pred p;\n\t"
          "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
          "selp.u32 %0, 1, 0, p;\n\t}"
          : "=r"(ok)
          : "r"(mbar), "r"(parity)
          : "memory");
      if (it == 64) t0 = clock64();
      if (it > 64 && (it & 255) == 0 && clock64() - t0 > 4000000000ll) {
        printf("tred_dft_h16: mbarrier wait timed out (block %d thread %d)\n", blockIdx.x, threadIdx.x);
        __trap();
      }
    }
  }
  asm volatile("bar.sync %0, %1;" ::"r"(bar), "r"(nthreads) : "memory");
}

__device__ __forceinline__ float dft_h16_scale(float m) {     // as h16_scale in tred_conv.cu
  const int ex = (int)((__float_as_uint(m) >> 23) & 0xffu);
  if (ex == 0 || ex == 255) return 1.0f;
  const int se = max(1, ex - 14);
  return __uint_as_float((uint32_t)se << 23);
}

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(DF_THREADS, 1)
k_dft_h16(const __grid_constant__ CUtensorMap tmW, DftParams p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  uint8_t* base_ptr = smem_raw + (base - raw);
  const int NCh = p.NC >> 1;                                 // DFT-matrix rows per CTA and N chunk
  const uint32_t bstage = (uint32_t)NCh * 128u;              // one (N chunk, K chunk) box of W
  const uint32_t wbytes = bstage * (uint32_t)(p.nnc * p.nkc);
  const uint32_t sW = base;
  const uint32_t sAt = base + ((wbytes + 1023u) & ~1023u);  // A tile: nkc chunks of 128 rows x 128 bytes
  uint8_t* a_ptr = base_ptr + (sAt - base);
  const uint32_t abytes = (uint32_t)p.nkc * 16384u;
  const uint32_t bars = sAt + abytes;
  const uint32_t wbar = bars, alocal = bars + 8, rcons = bars + 16;   // rcons: the epilogue has read rowinfo
  auto tfull_bar = [&](int a) { return bars + 24u + 8u * a; };
  auto tempty_bar = [&](int a) { return bars + 40u + 8u * a; };
  auto afull_bar = [&](int kc) { return bars + 56u + 8u * kc; };      // leader: K chunk kc of both A tiles stored
  auto aempty_bar = [&](int kc) { return bars + 88u + 8u * kc; };     // the tensor core is done with K chunk kc
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(a_ptr + abytes + 120);
  int* rowinfo = reinterpret_cast<int*>(a_ptr + abytes + 124);         // padded row of the A tile or -1
  float* red = reinterpret_cast<float*>(a_ptr + abytes + 128);         // [8] converter warp sums
  long long* colbase = reinterpret_cast<long long*>(a_ptr + abytes + 160);   // [100]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int cid = blockIdx.x >> 1, ncl = gridDim.x >> 1;
  {   // the compact rows of the chunk's row tiles (tile t holds rows rt_desc[t].x .. + rt_desc[t].y)
    const int4 dl = p.rt_desc[p.t0 + p.ntile - 1];
    p.row0 = p.rt_desc[p.t0].x;
    p.nrows = dl.x + dl.y - p.row0;
  }
  const int npairs = (p.nrows + 1) >> 1;

  if (threadIdx.x == 0) {
    mbar_init(wbar, 1);
    for (int kc = 0; kc < 4; ++kc) { mbar_init(afull_bar(kc), 2); mbar_init(aempty_bar(kc), 1); }
    mbar_init(alocal, 1);
    mbar_init(rcons, 1);
    for (int a = 0; a < 2; ++a) { mbar_init(tfull_bar(a), 1); mbar_init(tempty_bar(a), 2); }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                 "r"(512)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ------------------------------------------------------------ this CTA's half of the DFT matrix, once
    if (lane == 0) {
      mbar_expect_tx(wbar, wbytes);
      for (int nc = 0; nc < p.nnc; ++nc)
        for (int kc = 0; kc < p.nkc; ++kc)
          tma_load_2d(sW + (uint32_t)(nc * p.nkc + kc) * bstage, &tmW, kc * 64, nc * p.NC + (int)rank * NCh, wbar);
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------ MMA issuer (leader CTA)
    if (lane == 0 && rank == 0) {
      const uint32_t idesc = (1u << 4) | ((uint32_t)(p.NC >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
      int aphase = 0, acc = 0, tphase = 0;
      for (int pr = cid; pr < npairs; pr += ncl) {
        for (int nc = 0; nc < p.nnc; ++nc) {
          mbar_wait(tempty_bar(acc), tphase ^ 1);
          tc_fence_after();
          const uint32_t d_tmem = tmem_base + (uint32_t)(acc * 256);
          for (int kc = 0; kc < p.nkc; ++kc) {
            if (nc == 0) {                                       // both CTAs: K chunk stored (and W resident)
              mbar_wait(afull_bar(kc), aphase);
              tc_fence_after();
            }
            const uint64_t da = desc_sw128(sAt + (uint32_t)kc * 16384u);
            const uint64_t db = desc_sw128(sW + (uint32_t)(nc * p.nkc + kc) * bstage);
#pragma unroll
            for (int j = 0; j < 2; ++j) {
              const uint64_t hi = (uint64_t)(4 * j), lo = (uint64_t)(4 * j + 2);
              tc_mma_f16_pair2(d_tmem, da + hi, db + hi, idesc, (kc | j) != 0);
              tc_mma_f16_pair2(d_tmem, da + lo, db + hi, idesc, 1);
              tc_mma_f16_pair2(d_tmem, da + hi, db + lo, idesc, 1);
            }
            if (nc == p.nnc - 1) tc_commit_pair(aempty_bar(kc)); // this K chunk of both A tiles may be overwritten
          }
          tc_commit_pair(tfull_bar(acc));
          if (++acc == 2) { acc = 0; tphase ^= 1; }
        }
        aphase ^= 1;
      }
    }
  } else if (warp < 10) {
    // ------------------------------------------------------------ epilogue: spectra -> fp16 hi / lo -> HBM
    const int q = warp & 3;
    const int eh = (warp - 2) >> 2;                             // which half of the 16-frequency groups
    const int et = threadIdx.x - DF_EPI0;
    const bool poller = warp == 2;
    const int col = q * 32 + lane;                              // fine column = phase of this lane
    const int NPH = p.g.nph;
    const bool live = col < NPH;
    const bool padlane = col == NPH && (2 * NPH) % 16 != 0;     // zeroes the padding reals of the last block
    const int pos = (col >> 3) * 32 + (col & 7) * 2;            // hi part of (re, im); lo 16 halves further
    const int padpos = ((2 * NPH) >> 4) * 32 + ((2 * NPH) & 15);
    constexpr int fstride = DF_FSTRIDE;                         // qh is [tile][f][128 rows][kp16]: compile-time
                                                                // stride, the 16 stores of a group use immediates
    int lphase = 0, acc = 0, tphase = 0;
    for (int pr = cid; pr < npairs; pr += ncl) {
      group_wait(alocal, lphase, poller, 1, 256);
      lphase ^= 1;
      const int prow = *reinterpret_cast<volatile int*>(rowinfo);
      asm volatile("bar.sync 1, 256;" ::: "memory");
      if (et == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(rcons) : "memory");
      const int prow0 = prow < 0 ? 0 : prow;
      __half* orow = p.qh + ((int64_t)(prow0 >> 7) * p.nf * RT_ROWS + (prow0 & (RT_ROWS - 1))) * p.kp16 +
                     (live ? pos : padpos);
      for (int nc = 0; nc < p.nnc; ++nc) {
        group_wait(tfull_bar(acc), tphase, poller, 1, 256);
        tc_fence_after();
        const uint32_t taddr = tmem_base + (uint32_t)(acc * 256) + ((uint32_t)(q * 32) << 16);
        for (int g = eh; g * 32 < p.NC; g += 2) {
          uint32_t v[32];
          tmem_ld32(v, taddr + (uint32_t)(g * 32));
          asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
          if (prow >= 0 && (live || padlane)) {
            __half* o = orow + (int64_t)(nc * (p.NC >> 1) + g * 16) * fstride;
            if (live) {
#pragma unroll
              for (int i = 0; i < 16; ++i) {
                const float re = __uint_as_float(v[2 * i]), im = __uint_as_float(v[2 * i + 1]);
                const __half2 h = __floats2half2_rn(re, im);
                const float2 hf = __half22float2(h);
                const __half2 l = __floats2half2_rn(re - hf.x, im - hf.y);
                *reinterpret_cast<__half2*>(o + i * fstride) = h;
                *reinterpret_cast<__half2*>(o + i * fstride + 16) = l;
              }
            } else {
#pragma unroll
              for (int i = 0; i < 16; ++i) {
                *reinterpret_cast<uint4*>(o + i * fstride) = make_uint4(0u, 0u, 0u, 0u);
                *reinterpret_cast<uint4*>(o + i * fstride + 16) = make_uint4(0u, 0u, 0u, 0u);
              }
            }
          }
        }
        tc_fence_before();
        asm volatile("bar.sync 1, 256;" ::: "memory");
        if (et == 0) mbar_arrive_cluster(mapa(tempty_bar(acc), 0));
        if (++acc == 2) { acc = 0; tphase ^= 1; }
      }
    }
  } else {
    // ------------------------------------------------------------ converters: payload -> A tile
    const int tc = threadIdx.x - DF_CONV0;                     // 0 .. 255
    const int cw = tc >> 5;
    const int NPH = p.g.nph, S = p.g.S;
    // K chunk kc (32 ticks = 8 float4 per column) belongs to a group of 8 / nkc warps: it waits
    // for, fills and hands over its quarter of the A tile on its own
    const int TG = DF_NCONV / p.nkc;                           // threads per group
    const int kc = tc / TG, l = tc - kc * TG;
    const bool poller = l < 32;
    const uint32_t gbar = 3 + kc;
    const int nf4 = NPH * 8;
    int ephase = 0;
    int tile = p.t0;
    bool first = true;
    for (int pr = cid; pr < npairs; pr += ncl) {
      const int c = 2 * pr + (int)rank;
      const bool exists = c < p.nrows;
      int prow = -1;
      if (exists && tc < NPH) {
        const int m2 = p.row_m2[p.row0 + c];
        const int rest = m2 >> 3;
        const int py = rest % p.g.npy, grp = rest / p.g.npy;
        const int bt = grp / p.nstrip;
        const int px = (grp - bt * p.nstrip) * RT_SW + (m2 & (RT_SW - 1));
        const int i = px * S + tc / S, j = py * S + tc % S;
        const int bx = i / p.g.Bx, by = j / p.g.By;
        const int slot = p.blockmap[((int64_t)bt * p.g.NBx + bx) * p.g.NBy + by];
        colbase[tc] = slot >= 0 ? (((long long)slot * p.g.Bx + (i - bx * p.g.Bx)) * p.g.By + (j - by * p.g.By)) * p.Bt
                                : -1;
      }
      asm volatile("bar.sync 2, 256;" ::: "memory");
      float4 v[DF_MAXF4];
      float sum = 0.0f;
#pragma unroll
      for (int i = 0; i < DF_MAXF4; ++i) {
        const int idx = l + TG * i;
        v[i] = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
        if (exists && idx < nf4) {
          const long long b = colbase[idx >> 3];
          if (b >= 0) v[i] = __ldg(reinterpret_cast<const float4*>(p.payload + b) + 8 * kc + (idx & 7));
        }
        sum += (fabsf(v[i].x) + fabsf(v[i].y)) + (fabsf(v[i].z) + fabsf(v[i].w));
      }
      if (exists && tc == 0) {
        // row tile of compact row gr (this thread alone needs it, and only when it publishes the
        // row): rows advance by 2 ncl per iteration, so a forward scan from the previous tile
        // takes a load or two, in the shadow of the payload loads above
        const int gr = p.row0 + c;
        while (tile + 1 < p.t0 + p.ntile && p.rt_desc[tile + 1].x <= gr) ++tile;
        prow = (tile - p.t0) * RT_ROWS + (gr - p.rt_desc[tile].x);
      }
      for (int o = 16; o; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
      if (lane == 0) red[cw] = sum;
      asm volatile("bar.sync 2, 256;" ::: "memory");
      float tot = red[0];
#pragma unroll
      for (int w = 1; w < 8; ++w) tot += red[w];
      const float sc = dft_h16_scale(tot);
      const float sdown = __uint_as_float((254u - (__float_as_uint(sc) >> 23)) << 23);
      // split into fp16 hi / lo in registers NOW (the packed parts take the place of the fp32 values):
      // only the shared-memory stores are left for after the wait, which is on the row's critical path
      uint4 hl[DF_MAXF4];                                     // (hi01, hi23, lo01, lo23)
#pragma unroll
      for (int i = 0; i < DF_MAXF4; ++i) {
        const float x0 = v[i].x * sdown, x1 = v[i].y * sdown, x2 = v[i].z * sdown, x3 = v[i].w * sdown;
        const __half2 h01 = __floats2half2_rn(x0, x1), h23 = __floats2half2_rn(x2, x3);
        const float2 f01 = __half22float2(h01), f23 = __half22float2(h23);
        const __half2 l01 = __floats2half2_rn(x0 - f01.x, x1 - f01.y), l23 = __floats2half2_rn(x2 - f23.x, x3 - f23.y);
        hl[i] = make_uint4(*reinterpret_cast<const uint32_t*>(&h01), *reinterpret_cast<const uint32_t*>(&h23),
                           *reinterpret_cast<const uint32_t*>(&l01), *reinterpret_cast<const uint32_t*>(&l23));
      }
      // the tensor core must be done with this K chunk of the previous row before it is overwritten
      if (!first) { group_wait(aempty_bar(kc), ephase, poller, gbar, TG); ephase ^= 1; }
#pragma unroll
      for (int i = 0; i < DF_MAXF4; ++i) {
        const int idx = l + TG * i;
        if (idx < nf4) {
          const int cc = idx >> 3;
          const int t0 = 4 * (idx & 7);                          // tick within the K chunk
          // K chunk of 32 ticks = one 128-byte row: [hi 16 | lo 16 | hi 16 | lo 16]; 16-byte units swizzled by row
          const int off = (t0 >> 4) * 64 + (t0 & 15) * 2;
          uint8_t* rowp = a_ptr + kc * 16384 + cc * 128;
          const int u_hi = (off >> 4) ^ (cc & 7), u_lo = ((off + 32) >> 4) ^ (cc & 7);
          *reinterpret_cast<uint2*>(rowp + u_hi * 16 + (off & 15)) = make_uint2(hl[i].x, hl[i].y);
          *reinterpret_cast<uint2*>(rowp + u_lo * 16 + (off & 15)) = make_uint2(hl[i].z, hl[i].w);
        }
      }
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");      // generic writes -> tensor core reads
      if (tc == 0) {
        if (!first) mbar_wait(rcons, ephase ^ 1);               // the epilogue has taken the previous row's record
        *reinterpret_cast<volatile int*>(rowinfo) = prow;
        if (prow >= 0) p.rscale[prow] = sc;
      }
      asm volatile("bar.sync %0, %1;" ::"r"(gbar), "r"(TG) : "memory");
      if (l == 0) {
        if (first) mbar_wait(wbar, 0);                          // this CTA's half of W has landed
        if (tc == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(alocal) : "memory");
        mbar_arrive_cluster(mapa(afull_bar(kc), 0));
      }
      first = false;
    }
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync_all();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
  }
}

// DFT matrix in the operand layout: Wd[n][block(t)] fp16 hi / lo parts of w(t, n),
// n = 2 f + c: f = 0 packs DC (c = 0: w = 1) and Nyquist (c = 1: w = (-1)^t); else
// w = cos(2 pi f t / L) for c = 0 and -sin(2 pi f t / L) for c = 1.
__global__ void __launch_bounds__(256) k_dft_matrix(__half* __restrict__ Wd, int L, int Bt) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= L * Bt) return;
  const int n = i / Bt, t = i - n * Bt;
  const int f = n >> 1, c = n & 1;
  double w;
  if (f == 0) w = c == 0 ? 1.0 : ((t & 1) ? -1.0 : 1.0);
  else {
    double sn, cs;
    sincospi(2.0 * (double)(((int64_t)f * t) % L) / (double)L, &sn, &cs);
    w = c == 0 ? cs : -sn;
  }
  const float x = (float)w;
  const __half h = __float2half_rn(x);
  __half* e = Wd + (int64_t)n * (2 * Bt) + (t >> 4) * 32 + (t & 15);
  e[0] = h;
  e[16] = __float2half_rn(x - __half2float(h));
}

}  // namespace

typedef CUresult (*PFN_encodeTiledDF)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                      const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                      CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static PFN_encodeTiledDF get_encode_fn_df() {
  static PFN_encodeTiledDF fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (PFN_encodeTiledDF)p;
  }
  return fn;
}

// N chunk: the largest divisor of L that is a multiple of 32 and at most 256 (0: none)
static int dft_nchunk(int L) {
  for (int nc = 256; nc >= 32; nc -= 32)
    if (L % nc == 0 && L / nc >= 2) return nc;
  return 0;
}

static size_t dft_smem(const tred_ctx* ctx) {
  const int L = ctx->dims.fft_len, Bt = ctx->cfg.block[2];
  const size_t wbytes = (size_t)(L / 2) * Bt * 4;               // half of the matrix, hi + lo
  return 1024 + ((wbytes + 1023) & ~(size_t)1023) + (size_t)(Bt / 32) * 16384 + 160 + 100 * 8 + 64;
}

bool tred_dft_h16_supported(const tred_ctx* ctx) {
  const int Bt = ctx->cfg.block[2];
  return ctx->dims.n_phase == DF_NPH && h16_kp(ctx->dims) == DF_KP16 && ctx->cfg.sub == 10 && Bt >= 32 && Bt <= 128 && (Bt % 32) == 0 &&
         dft_nchunk(ctx->dims.fft_len) > 0 && dft_smem(ctx) <= (size_t)ctx->smem_optin && ctx->num_sms >= 2 &&
         get_encode_fn_df() != nullptr;
}

// floats the DFT matrix takes in the response-spectrum buffer
int64_t tred_dft_matrix_floats(const tred_dims& d, int Bt) { return (int64_t)d.fft_len * Bt; }

int tred_dft_matrix(tred_ctx* ctx, void* d_Wd, cudaStream_t st) {
  const int L = ctx->dims.fft_len, Bt = ctx->cfg.block[2];
  k_dft_matrix<<<cdiv((int64_t)L * Bt, 256), 256, 0, st>>>(reinterpret_cast<__half*>(d_Wd), L, Bt);
  TRED_COUNT_LAUNCH(1);
  TRED_LAUNCH_CHECK("k_dft_matrix");
  return TRED_OK;
}

// Spectra of the compact rows [row0, row0 + nrows) of the chunk's row tiles [t0, t0 + ntile):
// qh [ntile][nf][128][kp16] fp16 hi / lo blocks, rscale [ntile * 128].
int tred_dft_h16(tred_ctx* ctx, const float* payload, const int32_t* blockmap, const void* rt_desc,
                 const int32_t* row_m2, int t0, int ntile, int nstrip, const void* d_Wd,
                 void* qh, float* rscale, cudaStream_t st) {
  if (!tred_dft_h16_supported(ctx)) return TRED_EUNSUPPORTED;
  if (ntile < 1) return TRED_OK;
  const tred_dims& d = ctx->dims;
  const int L = d.fft_len, Bt = ctx->cfg.block[2];
  DftParams p;
  p.nrows = 0; p.row0 = 0; p.t0 = t0; p.ntile = ntile; p.rp = ntile * RT_ROWS;
  p.nf = d.n_freq; p.Bt = Bt; p.nkc = Bt / 32; p.NC = dft_nchunk(L); p.nnc = L / p.NC;
  p.kp16 = h16_kp(d);
  p.rt_desc = (const int4*)rt_desc; p.row_m2 = row_m2; p.blockmap = blockmap; p.payload = payload;
  p.qh = reinterpret_cast<__half*>(qh); p.rscale = rscale; p.g = make_grid(ctx); p.nstrip = nstrip;
  CUtensorMap tm;
  {
    const cuuint64_t dims[2] = {(cuuint64_t)(2 * Bt), (cuuint64_t)L};
    const cuuint64_t strides[1] = {(cuuint64_t)(2 * Bt) * 2};
    const cuuint32_t box[2] = {64, (cuuint32_t)(p.NC / 2)};
    const cuuint32_t estr[2] = {1, 1};
    if (get_encode_fn_df()(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void*>(d_Wd), dims, strides, box, estr,
                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                           CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return TRED_EUNSUPPORTED;
  }
  const size_t smem = dft_smem(ctx);
  TRED_CUDA(cudaFuncSetAttribute(k_dft_h16, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const int npairs_max = ntile * (RT_ROWS / 2);
  int ncl = ctx->num_sms / 2;
  if (ncl > npairs_max) ncl = npairs_max;
  k_dft_h16<<<2 * ncl, DF_THREADS, smem, st>>>(tm, p);
  TRED_LAUNCH_CHECK("k_dft_h16");
  return TRED_OK;
}
