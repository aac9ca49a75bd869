// Spectrum product for a MIRROR-SYMMETRIC response, on CTA pairs (tcgen05 cta_group::2).
//
// PAPER.md:L199-221 (Mirror-Pair Complex Packing) uses the reflection symmetry
// R_{-i}^{-j} = R_i^j to halve the number of FFTs.  Here the symmetry is
// spent on the spectrum product (tred_conv.cu, "mirror symmetry"): the rows of qhat hold the
// sums and differences of the mirror phase pairs, [s: nph floats | d: nph floats], and
//   S = A_s Bs^T  (TMEM columns [0, 128)),   D = A_d Bd^T  (columns [128, 256)),
// each of inner length nph and SYM_N = 128 columns -- half the tensor-core work of k_mac_tc2
// -- give the products of offset o and of its mirror o' = noff - 1 - o as
//   T[o] = (S_o + D_o) / 2,   T[o'] = (S_o - D_o) / 2      (o < noff / 2; centre: S / 2).
// Same pipeline, barriers and fused epilogue as k_mac_tc2 (tred_mac_tc2.cu); 3xTF32.
#include "tred_tc2_common.cuh"

namespace {

constexpr int S2_STAGES = 3;
constexpr int S2_BQ_BYTES = (SYM_N / 2) * T2_KC * 4;               // 4 KB: this CTA's half of one matrix chunk
constexpr int S2_STAGE_BYTES = 4 * T2_A_BYTES + 4 * S2_BQ_BYTES;    // As, As_lo, Ad, Ad_lo, Bs_h, Bs_l, Bd_h, Bd_l
constexpr size_t S2_SMEM = (size_t)S2_STAGES * S2_STAGE_BYTES + 1024 + 256 + 4 * T2_PATCH_FLOAT2 * 8;

__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2, int c3,
                                            uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar)
      : "memory");
}

struct S2Maps { CUtensorMap a, bsh, bsl, bdh, bdl; };

__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(T2_THREADS, 1)
k_mac_tc2_sym(const __grid_constant__ S2Maps tm, T2Params p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;
  uint8_t* base_ptr = smem_raw + (base - raw);
  const uint32_t bars = base + S2_STAGES * S2_STAGE_BYTES;
  auto full_bar = [&](int s) { return bars + 8u * s; };
  auto conv_bar = [&](int s) { return bars + 8u * (S2_STAGES + s); };            // used in the leader
  auto empty_bar = [&](int s) { return bars + 8u * (2 * S2_STAGES + s); };
  auto tfull_bar = [&](int a) { return bars + 8u * (3 * S2_STAGES + a); };
  auto tempty_bar = [&](int a) { return bars + 8u * (3 * S2_STAGES + 2 + a); };   // used in the leader
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(base_ptr + S2_STAGES * S2_STAGE_BYTES + 8 * (3 * S2_STAGES + 4));
  // stage: [As][As_lo][Ad][Ad_lo][Bs_h][Bs_l][Bd_h][Bd_l]
  auto sA = [&](int s, int i) { return base + s * S2_STAGE_BYTES + i * T2_A_BYTES; };
  auto sB = [&](int s, int i) { return base + s * S2_STAGE_BYTES + 4 * T2_A_BYTES + i * S2_BQ_BYTES; };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int KH = p.K2 >> 1;                                     // floats per half row (= nph)
  const int nkc = (KH + T2_KC - 1) / T2_KC;
  const int nitems = p.nf * p.npair;
  const int cid = blockIdx.x >> 1, ncl = gridDim.x >> 1;

  if (threadIdx.x == 0) {
    for (int s = 0; s < S2_STAGES; ++s) {
      mbar_init(full_bar(s), 1);
      mbar_init(conv_bar(s), 2);
      mbar_init(empty_bar(s), 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(tfull_bar(a), 1);
      mbar_init(tempty_bar(a), 2);
    }
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
    // ------------------------------------------------------------ TMA producer (each CTA)
    if (lane == 0) {
      const uint32_t tx = (uint32_t)(2 * T2_A_BYTES + 4 * S2_BQ_BYTES);
      const int nh = SYM_N / 2;
      int stage = 0, phase = 0;
      for (int item = cid; item < nitems; item += ncl) {
        const int f = item / p.npair, pr = item - f * p.npair;
        const int mt = min(2 * pr + (int)rank, p.ntile - 1);
        for (int kc = 0; kc < nkc; ++kc) {
          mbar_wait(empty_bar(stage), phase ^ 1);
          mbar_expect_tx(full_bar(stage), tx);
          // columns beyond nph of the last chunk are out of bounds of the map: filled with zeros
          tma_load_4d(sA(stage, 0), &tm.a, kc * T2_KC, 0, mt * T2_M, f, full_bar(stage));
          tma_load_4d(sA(stage, 2), &tm.a, kc * T2_KC, 1, mt * T2_M, f, full_bar(stage));
          tma_load_3d(sB(stage, 0), &tm.bsh, kc * T2_KC, (int)rank * nh, f, full_bar(stage));
          tma_load_3d(sB(stage, 1), &tm.bsl, kc * T2_KC, (int)rank * nh, f, full_bar(stage));
          tma_load_3d(sB(stage, 2), &tm.bdh, kc * T2_KC, (int)rank * nh, f, full_bar(stage));
          tma_load_3d(sB(stage, 3), &tm.bdl, kc * T2_KC, (int)rank * nh, f, full_bar(stage));
          if (++stage == S2_STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------ MMA issuer (leader CTA)
    if (lane == 0 && rank == 0) {
      // D fp32, A/B tf32, both K-major, N = SYM_N, M = 256 over the pair
      const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(SYM_N >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
      int stage = 0, phase = 0, as = 0, aphase = 0;
      for (int item = cid; item < nitems; item += ncl) {
        mbar_wait(tempty_bar(as), aphase ^ 1);
        tc_fence_after();
        const uint32_t dS = tmem_base + (uint32_t)(as * T2_NMAX), dD = dS + (uint32_t)SYM_N;
        for (int kc = 0; kc < nkc; ++kc) {
          mbar_wait(conv_bar(stage), phase);
          tc_fence_after();
          const int nks = (min(T2_KC, KH - kc * T2_KC) + 7) >> 3;
          const uint64_t as_h = make_desc_sw64(sA(stage, 0)), as_l = make_desc_sw64(sA(stage, 1));
          const uint64_t ad_h = make_desc_sw64(sA(stage, 2)), ad_l = make_desc_sw64(sA(stage, 3));
          const uint64_t bs_h = make_desc_sw64(sB(stage, 0)), bs_l = make_desc_sw64(sB(stage, 1));
          const uint64_t bd_h = make_desc_sw64(sB(stage, 2)), bd_l = make_desc_sw64(sB(stage, 3));
          for (int ks = 0; ks < nks; ++ks) {
            const uint64_t adv = (uint64_t)(ks * 2);
            const uint32_t acc = (kc | ks) != 0;
            tc_mma_tf32_pair(dS, as_h + adv, bs_h + adv, idesc, acc);
            tc_mma_tf32_pair(dS, as_l + adv, bs_h + adv, idesc, 1);
            tc_mma_tf32_pair(dS, as_h + adv, bs_l + adv, idesc, 1);
            tc_mma_tf32_pair(dD, ad_h + adv, bd_h + adv, idesc, acc);
            tc_mma_tf32_pair(dD, ad_l + adv, bd_h + adv, idesc, 1);
            tc_mma_tf32_pair(dD, ad_h + adv, bd_l + adv, idesc, 1);
          }
          tc_commit_pair(empty_bar(stage));
          if (++stage == S2_STAGES) { stage = 0; phase ^= 1; }
        }
        tc_commit_pair(tfull_bar(as));
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
  } else if (warp < 6) {
    // ------------------------------------------------------------ converters: A -> A_hi, A_lo (s and d)
    const int tc = threadIdx.x - 64;
    int stage = 0, phase = 0;
    for (int item = cid; item < nitems; item += ncl) {
      for (int kc = 0; kc < nkc; ++kc) {
        mbar_wait(full_bar(stage), phase);
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          float4* a = reinterpret_cast<float4*>(base_ptr + stage * S2_STAGE_BYTES + (2 * h) * T2_A_BYTES);
          float4* lo = reinterpret_cast<float4*>(base_ptr + stage * S2_STAGE_BYTES + (2 * h + 1) * T2_A_BYTES);
#pragma unroll
          for (int i = 0; i < T2_A_BYTES / 16 / 128; ++i) {
            const float4 v = a[tc + 128 * i];
            float4 hh, l;
            hh.x = tf32_hi(v.x); hh.y = tf32_hi(v.y); hh.z = tf32_hi(v.z); hh.w = tf32_hi(v.w);
            l.x = tf32_hi(v.x - hh.x); l.y = tf32_hi(v.y - hh.y); l.z = tf32_hi(v.z - hh.z); l.w = tf32_hi(v.w - hh.w);
            a[tc + 128 * i] = hh;
            lo[tc + 128 * i] = l;
          }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
        asm volatile("bar.sync 2, 128;" ::: "memory");
        if (tc == 0) mbar_arrive_cluster(mapa(conv_bar(stage), 0));
        if (++stage == S2_STAGES) { stage = 0; phase ^= 1; }
      }
    }
  } else {
    // ------------------------------------------------------------ epilogue (K = 2H + 1 = 11)
    constexpr int KK = 11, NOFF = KK * KK, CEN = NOFF / 2;          // centre offset 60 = (5, 5)
    const int q = warp & 3;
    const int et = threadIdx.x - 192;
    float2* patch = reinterpret_cast<float2*>(base_ptr + S2_STAGES * S2_STAGE_BYTES + 256);
    float2* P = patch + q * T2_PATCH_FLOAT2;
    for (int i = et; i < 4 * T2_PATCH_FLOAT2; i += 128) patch[i] = make_float2(0.0f, 0.0f);
    asm volatile("bar.sync 1, 128;" ::: "memory");
    const int PX = RT_SW + 2 * p.H;
    int as = 0, aphase = 0;
    auto item_tile = [&](int it) { return it < nitems ? 2 * (it % p.npair) + (int)rank : p.ntile; };
    auto load_desc = [&](int it) {
      const int t = item_tile(it);
      return t < p.ntile ? p.rt_desc[p.t0 + t] : make_int4(0, 0, 0, 0);
    };
    const int r = q * 32 + lane;
    int4 d_cur = load_desc(cid), d_nxt = load_desc(cid + ncl);
    int m2_cur = r < d_cur.y ? p.row_m2[d_cur.x + r] : 0;
    for (int item = cid; item < nitems; item += ncl) {
      const int f = item / p.npair, pr = item - f * p.npair;
      const int mt = 2 * pr + (int)rank;
      const bool has_tile = mt < p.ntile;
      const int4 d = d_cur;
      const int m2 = m2_cur;
      const int m2_nxt = r < d_nxt.y ? p.row_m2[d_nxt.x + r] : 0;
      const int4 d_nn = load_desc(item + 2 * ncl);
      const bool valid = r < d.y;
      const uint32_t vmask = __ballot_sync(0xffffffffu, valid);
      const int yl = (m2 >> 3) % p.npy - d.z;
      const int cell0 = valid ? (m2 & (RT_SW - 1)) * RT_PYS + yl : 0;
      mbar_wait(tfull_bar(as), aphase);
      tc_fence_after();
      const uint32_t taddr = tmem_base + (uint32_t)(as * T2_NMAX) + ((uint32_t)(q * 32) << 16);
      if (vmask) {
        const int ylo = __reduce_min_sync(vmask, valid ? yl : 0x7fffffff);
        const int yhi = __reduce_max_sync(vmask, valid ? yl : -0x7fffffff);
        const bool narrow = (yhi - ylo) <= 4;       // then offsets 5 lines apart never meet in a cell
        float2* Pc = P + cell0;
        auto rmw = [&](int kx, int ky, float re, float im) {
          float2* e = Pc + kx * RT_PYS + ky;
          float2 a = *e;
          a.x += re;
          a.y += im;
          *e = a;
        };
#pragma unroll
        for (int kx = 0; kx <= KK / 2; ++kx) {
          uint32_t vs[32], vd[32];
          tmem_ld32(vs, taddr + (uint32_t)(2 * KK * kx));
          // the 32-column load of D must stay inside this accumulator's 256 columns
          const int dcol = min(SYM_N + 2 * KK * kx, T2_NMAX - 32), dsh = SYM_N + 2 * KK * kx - dcol;
          tmem_ld32(vd, taddr + (uint32_t)dcol);
          asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
          if (valid) {
            // T[o] for o = (kx, ky), then T[o'] for the mirror o' = (10 - kx, 10 - ky)
#pragma unroll
            for (int pass = 0; pass < 2; ++pass) {
              const float sg = pass ? -0.5f : 0.5f;
#pragma unroll
              for (int j = 0; j < KK; ++j) {
                // order 0,5, 1,6, 2,7, 3,8, 4,9, 10: in a narrow warp the two offsets of a
                // pair (5 lines apart) never meet in a cell and share one barrier
                const int ky = j == KK - 1 ? KK - 1 : ((j & 1) ? 5 + (j >> 1) : (j >> 1));
                const int o = kx * KK + ky;
                if (o <= CEN && !(pass && o == CEN)) {                  // centre: once, T = S / 2
                  const float re = fmaf(sg, __uint_as_float(vd[(dsh + 2 * ky) & 31]), 0.5f * __uint_as_float(vs[2 * ky]));
                  const float im = fmaf(sg, __uint_as_float(vd[(dsh + 2 * ky + 1) & 31]), 0.5f * __uint_as_float(vs[2 * ky + 1]));
                  if (pass) rmw(KK - 1 - kx, KK - 1 - ky, re, im);
                  else rmw(kx, ky, re, im);
                }
                if (!narrow || (j & 1) || j == KK - 1) __syncwarp(vmask);
              }
            }
          }
        }
      }
      d_cur = d_nxt; d_nxt = d_nn; m2_cur = m2_nxt;
      tc_fence_before();
      asm volatile("bar.sync 1, 128;" ::: "memory");
      if (et == 0) mbar_arrive_cluster(mapa(tempty_bar(as), 0));
      if (++as == 2) { as = 0; aphase ^= 1; }
      if (has_tile) {
        const int nyp = d.w + 2 * p.H, ncell = PX * nyp;
        float2* dst = p.opart + ((int64_t)mt * p.nf + f) * (PX * RT_PY);
        for (int i = et; i < ncell; i += 128) {
          const int X = i / nyp, Y = i - X * nyp;
          const int c = X * RT_PYS + Y;
          float2 a = patch[c];
#pragma unroll
          for (int w = 1; w < 4; ++w) {
            const float2 b = patch[w * T2_PATCH_FLOAT2 + c];
            a.x += b.x; a.y += b.y;
          }
#pragma unroll
          for (int w = 0; w < 4; ++w) patch[w * T2_PATCH_FLOAT2 + c] = make_float2(0.0f, 0.0f);
          dst[X * RT_PY + Y] = a;
        }
      }
      asm volatile("bar.sync 1, 128;" ::: "memory");
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

}  // namespace

// ---------------------------------------------------------------------------- host side
typedef CUresult (*PFN_encodeTiledS)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                     const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                     CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static PFN_encodeTiledS get_encode_fns() {
  static PFN_encodeTiledS fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (PFN_encodeTiledS)p;
  }
  return fn;
}

bool tred_mac_tc2s_supported(const tred_ctx* ctx) {
  const tred_dims& d = ctx->dims;
  return ctx->cfg.resp_half == 5 && (d.n_phase & 3) == 0 && (d.n_off & 1) == 1 && d.n_off + 1 <= SYM_N &&
         (size_t)ctx->smem_optin >= S2_SMEM && ctx->num_sms >= 2 && get_encode_fns() != nullptr;
}

// Same contract as tred_mac_tc2; qhat rows are [s: nph floats | d: nph floats] and the
// matrices are the mirror-symmetric halves Bs, Bd [f][SYM_N][nph] (hi / lo parts).
int tred_mac_tc2s(tred_ctx* ctx, const float* qhat, const float* Bs_hi, const float* Bs_lo, const float* Bd_hi,
                  const float* Bd_lo, float* opart, int ntile, int t0, const void* rt_desc, const int32_t* row_m2,
                  cudaStream_t st) {
  const tred_dims& d = ctx->dims;
  if (ntile < 1 || !tred_mac_tc2s_supported(ctx)) return TRED_EUNSUPPORTED;
  if ((((uintptr_t)qhat) | ((uintptr_t)Bs_hi) | ((uintptr_t)Bs_lo) | ((uintptr_t)Bd_hi) | ((uintptr_t)Bd_lo)) & 15)
    return TRED_EUNSUPPORTED;
  PFN_encodeTiledS enc = get_encode_fns();
  const int nph = d.n_phase;
  const int64_t rp = (int64_t)ntile * T2_M;
  S2Maps tm;
  {
    const cuuint64_t dims[4] = {(cuuint64_t)nph, 2, (cuuint64_t)rp, (cuuint64_t)d.n_freq};
    const cuuint64_t strides[3] = {(cuuint64_t)nph * 4, (cuuint64_t)nph * 8, (cuuint64_t)nph * 8 * (cuuint64_t)rp};
    const cuuint32_t box[4] = {(cuuint32_t)T2_KC, 1, (cuuint32_t)T2_M, 1};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    if (enc(&tm.a, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, (void*)qhat, dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return TRED_EUNSUPPORTED;
  }
  auto bmap = [&](CUtensorMap* m, const float* base) {
    const cuuint64_t dims[3] = {(cuuint64_t)nph, (cuuint64_t)SYM_N, (cuuint64_t)d.n_freq};
    const cuuint64_t strides[2] = {(cuuint64_t)nph * 4, (cuuint64_t)nph * 4 * SYM_N};
    const cuuint32_t box[3] = {(cuuint32_t)T2_KC, (cuuint32_t)(SYM_N / 2), 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    return enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)base, dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
  };
  if (!bmap(&tm.bsh, Bs_hi) || !bmap(&tm.bsl, Bs_lo) || !bmap(&tm.bdh, Bd_hi) || !bmap(&tm.bdl, Bd_lo))
    return TRED_EUNSUPPORTED;
  static bool attr_set[64] = {false};
  if (!attr_set[ctx->device & 63]) {
    TRED_CUDA(cudaFuncSetAttribute(k_mac_tc2_sym, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)S2_SMEM));
    attr_set[ctx->device & 63] = true;
  }
  T2Params p;
  p.nf = d.n_freq; p.ntile = ntile; p.npair = (ntile + 1) / 2;
  p.N = SYM_N; p.K2 = 2 * nph; p.noff = d.n_off;
  p.K = 2 * ctx->cfg.resp_half + 1; p.H = ctx->cfg.resp_half; p.npy = ctx->cfg.npix_y; p.t0 = t0;
  p.rt_desc = (const int4*)rt_desc; p.row_m2 = row_m2; p.opart = reinterpret_cast<float2*>(opart);
  const int64_t items = (int64_t)p.nf * p.npair;
  int64_t ncl = ctx->num_sms / 2;
  if (ncl > items) ncl = items;
  k_mac_tc2_sym<<<(int)(2 * ncl), T2_THREADS, S2_SMEM, st>>>(tm, p);
  TRED_LAUNCH_CHECK("k_mac_tc2_sym");
  return TRED_OK;
}
