// Spectrum product of Eq. (14) on CTA PAIRS: tcgen05.mma.cta_group::2,
// M = 256 (two row tiles of 128 charge pixels, one per CTA), N = 2 kp, 3xTF32, with the sum
// over the response offsets fused into the epilogue (same arithmetic and layouts as
// k_mac_tc<true> in tred_mac_tc.cu; see there and tred_conv.cu for the row tiles).
//
// Why pairs: with one CTA per tile every MMA reads 4 KB of A and 8 KB of B from shared
// memory in 128 cycles (96 B/clk of the SM's 128 B/clk) and every K chunk refills 40 KB
// through TMA; ncu showed the tensor pipe 63 % active with the shared-memory pipe as the
// co-bottleneck.  In a pair each CTA stages only half of B (its N/2 rows), so the operand
// reads drop to 64 B/clk per SM, the TMA fill to 24 KB per chunk, and a stage to 32 KB
// (5 stages instead of 3).
//
// Per CTA: warp 0 TMA producer (own A tile, own half of B_hi / B_lo), warp 1 MMA issuer
// (leader CTA only), warps 2-5 converters (A -> A_hi in place, A_lo), warps 6-9 epilogue.
// Barriers: full / empty / tfull are local to each CTA (empty and tfull arrive through
// tcgen05.commit multicast); conv and tempty live in the leader and count one arrival per CTA.
#include "tred_tc2_common.cuh"

namespace {

// BF: the two correction products A_lo B_hi and A_hi B_lo (2^-11 of the main product) run as
// bf16 MMAs (kind::f16, K = 16 per instruction, twice the tf32 rate): the stage then holds
// A fp32 | A_hi bf16 | A_lo bf16 | B_hi tf32 | B_hi bf16 | B_lo bf16 (the bf16 tiles in 32-byte
// swizzled rows), and tmBl / tmBl2 are the maps of the bf16 copies of B_hi / B_lo.
struct T2Maps { CUtensorMap a, bh, bl, bl2; };

__device__ __forceinline__ void tc_mma_bf16_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                                 uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// K-major operand tile of 32-byte swizzled rows (8 rows = one 256-byte swizzle atom)
__device__ __forceinline__ uint64_t make_desc_sw32(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3ffff) >> 4);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)(256 >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)6 << 61;                           // SWIZZLE_32B
  return d;
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {      // round to nearest even
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));
  return r;
}

template <int KC, bool BF>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(T2_THREADS, 1)
k_mac_tc2(const __grid_constant__ T2Maps tm, T2Params p) {
  const CUtensorMap& tmA = tm.a;
  const CUtensorMap& tmBh = tm.bh;
  const CUtensorMap& tmBl = tm.bl;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;                  // identical in both CTAs of the pair
  uint8_t* base_ptr = smem_raw + (base - raw);
  const uint32_t bars = base + T2_STAGES * T2_STAGE_BYTES;
  auto full_bar = [&](int s) { return bars + 8u * s; };
  auto conv_bar = [&](int s) { return bars + 8u * (T2_STAGES + s); };          // used in the leader
  auto empty_bar = [&](int s) { return bars + 8u * (2 * T2_STAGES + s); };
  auto tfull_bar = [&](int a) { return bars + 8u * (3 * T2_STAGES + a); };
  auto tempty_bar = [&](int a) { return bars + 8u * (3 * T2_STAGES + 2 + a); }; // used in the leader
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(base_ptr + T2_STAGES * T2_STAGE_BYTES + 8 * (3 * T2_STAGES + 4));
  auto sA = [&](int s) { return base + s * T2_STAGE_BYTES; };
  auto sAlo = [&](int s) { return base + s * T2_STAGE_BYTES + T2_A_BYTES; };
  auto sBh = [&](int s) { return base + s * T2_STAGE_BYTES + 2 * T2_A_BYTES; };
  auto sBl = [&](int s) { return base + s * T2_STAGE_BYTES + 2 * T2_A_BYTES + T2_BH_BYTES; };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int nkc = (p.K2 + T2_KC - 1) / T2_KC;
  const int nitems = p.nf * p.npair;
  const int cid = blockIdx.x >> 1, ncl = gridDim.x >> 1;

  if (threadIdx.x == 0) {
    for (int s = 0; s < T2_STAGES; ++s) {
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
  cluster_sync_all();                                             // both CTAs' barriers exist
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ------------------------------------------------------------ TMA producer (each CTA)
    if (lane == 0) {
      const int nh = p.N >> 1;
      // tf32: B_hi + B_lo rows of 64 bytes; bf16: B_hi 64-byte rows + two bf16 copies of 32-byte rows
      const uint32_t tx = (uint32_t)(T2_A_BYTES + 2 * nh * T2_KC * 4);
      int stage = 0, phase = 0;
      for (int item = cid; item < nitems; item += ncl) {
        const int f = item / p.npair, pr = item - f * p.npair;
        const int mt = min(2 * pr + (int)rank, p.ntile - 1);
        // qhat streams from HBM once: have L2 fetch the next item's A tile now, so that the
        // loads below (issued when a stage frees up) see an L2 hit instead of a DRAM round trip
        if (item + ncl < nitems) {
          const int fn = (item + ncl) / p.npair, prn = (item + ncl) - fn * p.npair;
          const int mtn = min(2 * prn + (int)rank, p.ntile - 1);
          for (int kc = 0; kc < nkc; ++kc) tma_prefetch_3d(&tmA, kc * T2_KC, mtn * T2_M, fn);
        }
        for (int kc = 0; kc < nkc; ++kc) {
          mbar_wait(empty_bar(stage), phase ^ 1);
          mbar_expect_tx(full_bar(stage), tx);
          tma_load_3d(sA(stage), &tmA, kc * T2_KC, mt * T2_M, f, full_bar(stage));
          tma_load_3d(sBh(stage), &tmBh, kc * T2_KC, (int)rank * nh, f, full_bar(stage));
          tma_load_3d(sBl(stage), &tmBl, kc * T2_KC, (int)rank * nh, f, full_bar(stage));
          if (BF) tma_load_3d(sBl(stage) + T2_BH_BYTES / 2, &tm.bl2, kc * T2_KC, (int)rank * nh, f, full_bar(stage));
          if (++stage == T2_STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------ MMA issuer (leader CTA)
    if (lane == 0 && rank == 0) {
      // instruction descriptor: D fp32, A/B tf32, both K-major, N, M = 256 over the pair
      const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(p.N >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
      int stage = 0, phase = 0, as = 0, aphase = 0;
      for (int item = cid; item < nitems; item += ncl) {
        mbar_wait(tempty_bar(as), aphase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(as * T2_NMAX);
        for (int kc = 0; kc < nkc; ++kc) {
          mbar_wait(conv_bar(stage), phase);                       // both CTAs: loaded and split
          tc_fence_after();
          const int nks = min(T2_KC, p.K2 - kc * T2_KC) >> 3;
          const uint64_t da = make_desc_sw64(sA(stage)), dbh = make_desc_sw64(sBh(stage));
          if (BF) {
            // bf16 tiles: A_hi | A_lo at sAlo, B_hi | B_lo copies at sBl (32-byte swizzled rows, K = 16)
            const uint32_t idesc_b = (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(p.N >> 3) << 17) |
                                     ((uint32_t)(256 >> 4) << 24);
            for (int ks = 0; ks < nks; ++ks)
              tc_mma_tf32_pair(d_tmem, da + (uint64_t)(ks * 2), dbh + (uint64_t)(ks * 2), idesc, (kc | ks) != 0);
            tc_mma_bf16_pair(d_tmem, make_desc_sw32(sAlo(stage) + T2_A_BYTES / 2), make_desc_sw32(sBl(stage)), idesc_b, 1);
            tc_mma_bf16_pair(d_tmem, make_desc_sw32(sAlo(stage)), make_desc_sw32(sBl(stage) + T2_BH_BYTES / 2), idesc_b, 1);
          } else {
            const uint64_t dl = make_desc_sw64(sAlo(stage)), dbl = make_desc_sw64(sBl(stage));
            for (int ks = 0; ks < nks; ++ks) {
              const uint64_t adv = (uint64_t)(ks * 2);
              tc_mma_tf32_pair(d_tmem, da + adv, dbh + adv, idesc, (kc | ks) != 0);
              tc_mma_tf32_pair(d_tmem, dl + adv, dbh + adv, idesc, 1);
              tc_mma_tf32_pair(d_tmem, da + adv, dbl + adv, idesc, 1);
            }
          }
          tc_commit_pair(empty_bar(stage));                        // frees the stage in both CTAs
          if (++stage == T2_STAGES) { stage = 0; phase ^= 1; }
        }
        tc_commit_pair(tfull_bar(as));                             // accumulators complete in both CTAs
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
  } else if (warp < 6) {
    // ------------------------------------------------------------ converters: A -> A_hi, A_lo
    const int tc = threadIdx.x - 64;
    int stage = 0, phase = 0;
    for (int item = cid; item < nitems; item += ncl) {
      for (int kc = 0; kc < nkc; ++kc) {
        mbar_wait(full_bar(stage), phase);
        float4* a = reinterpret_cast<float4*>(base_ptr + stage * T2_STAGE_BYTES);
        float4* lo = reinterpret_cast<float4*>(base_ptr + stage * T2_STAGE_BYTES + T2_A_BYTES);
#pragma unroll
        for (int i = 0; i < T2_A_BYTES / 16 / 128; ++i) {
          const int j = tc + 128 * i;
          const float4 v = a[j];
          float4 h, l;
          h.x = tf32_hi(v.x); h.y = tf32_hi(v.y); h.z = tf32_hi(v.z); h.w = tf32_hi(v.w);
          // A_hi stays as loaded: kind::tf32 reads only the upper 19 bits of an operand (h is what it sees)
          if (BF) {
            // float4 j of the 64-byte swizzled fp32 tile is row j / 4, logical 16-byte chunk
            // (j % 4) ^ ((row >> 1) & 3), i.e. floats k0 .. k0 + 3; in a 32-byte swizzled bf16 tile
            // they are 8 bytes of row `row`, 16-byte chunk (k0 / 8) ^ ((row >> 2) & 1)
            const int row = j >> 2, k0 = 4 * ((j & 3) ^ ((row >> 1) & 3));
            const int ob = row * 32 + (((k0 >> 3) ^ ((row >> 2) & 1)) << 4) + ((k0 & 7) << 1);
            uint8_t* tb = base_ptr + stage * T2_STAGE_BYTES + T2_A_BYTES;
            *reinterpret_cast<uint2*>(tb + ob) = make_uint2(pack_bf16(h.x, h.y), pack_bf16(h.z, h.w));
            *reinterpret_cast<uint2*>(tb + T2_A_BYTES / 2 + ob) =
                make_uint2(pack_bf16(v.x - h.x, v.y - h.y), pack_bf16(v.z - h.z, v.w - h.w));
          } else {
            l.x = tf32_hi(v.x - h.x); l.y = tf32_hi(v.y - h.y); l.z = tf32_hi(v.z - h.z); l.w = tf32_hi(v.w - h.w);
            lo[j] = l;
          }
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes -> tensor core reads
        asm volatile("bar.sync 2, 128;" ::: "memory");
        if (tc == 0) mbar_arrive_cluster(mapa(conv_bar(stage), 0));
        if (++stage == T2_STAGES) { stage = 0; phase ^= 1; }
      }
    }
  } else {
    // ------------------------------------------------------------ epilogue: sum over offsets
    const int q = warp & 3;
    const int et = threadIdx.x - 192;
    float2* patch = reinterpret_cast<float2*>(base_ptr + T2_STAGES * T2_STAGE_BYTES + 256);
    float2* P = patch + q * T2_PATCH_FLOAT2;
    for (int i = et; i < 4 * T2_PATCH_FLOAT2; i += 128) patch[i] = make_float2(0.0f, 0.0f);
    asm volatile("bar.sync 1, 128;" ::: "memory");
    const int PX = RT_SW + 2 * p.H;
    int as = 0, aphase = 0;
    // Row tile descriptor and this thread's row record are fetched one / two items ahead
    // (two dependent global loads otherwise sit on the epilogue's critical path).
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
      // prefetch: record of the next item (its descriptor arrived an iteration ago), descriptor of the one after
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
        if constexpr (KC == 11) {
          // Offsets (kx, ky) and (kx + 8, ky) never meet in one cell (rows of a tile lie in an
          // 8-pixel-wide strip), nor do (kx, ky) and (kx, ky + 5) when the rows of this warp span
          // at most 5 lines: such offsets are added in one step (independent shared-memory
          // read-modify-writes), the others one after the other.
          const int ylo = __reduce_min_sync(vmask, valid ? yl : 0x7fffffff);
          const int yhi = __reduce_max_sync(vmask, valid ? yl : -0x7fffffff);
          const bool narrow = (yhi - ylo) <= 4;
          float2* Pc = P + cell0;
          auto rmw = [&](int kx, int ky, uint32_t re, uint32_t im) {
            float2* e = Pc + kx * RT_PYS + ky;
            float2 a = *e;
            a.x += __uint_as_float(re);
            a.y += __uint_as_float(im);
            *e = a;
          };
#pragma unroll
          for (int g = 0; g < 8; ++g) {
            const bool paired = g < 3;
            uint32_t va[32], vb[32];
            tmem_ld32(va, taddr + (uint32_t)(22 * g));
            if (paired) tmem_ld32(vb, taddr + (uint32_t)(22 * (g + 8)));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (valid) {
              if (narrow) {
#pragma unroll
                for (int ky = 0; ky < 5; ++ky) {
                  rmw(g, ky, va[2 * ky], va[2 * ky + 1]);
                  rmw(g, ky + 5, va[2 * ky + 10], va[2 * ky + 11]);
                  if (paired) {
                    rmw(g + 8, ky, vb[2 * ky], vb[2 * ky + 1]);
                    rmw(g + 8, ky + 5, vb[2 * ky + 10], vb[2 * ky + 11]);
                  }
                  __syncwarp(vmask);
                }
                rmw(g, 10, va[20], va[21]);
                if (paired) rmw(g + 8, 10, vb[20], vb[21]);
                __syncwarp(vmask);
              } else {
#pragma unroll
                for (int ky = 0; ky < 11; ++ky) {
                  rmw(g, ky, va[2 * ky], va[2 * ky + 1]);
                  if (paired) rmw(g + 8, ky, vb[2 * ky], vb[2 * ky + 1]);
                  __syncwarp(vmask);
                }
              }
            }
          }
        } else {
          const int KK = p.K, noff = p.noff;
          for (int c0 = 0; c0 * 16 < noff; ++c0) {
            uint32_t v[32];
            tmem_ld32(v, taddr + (uint32_t)(c0 * 32));
            asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
            if (valid) {
              float2* Pc = P + cell0;
#pragma unroll
              for (int j = 0; j < 16; ++j) {
                const int off = c0 * 16 + j;
                if (off < noff) {
                  const int kx = off / KK, ky = off - kx * KK;
                  float2* e = Pc + kx * RT_PYS + ky;
                  float2 a = *e;
                  a.x += __uint_as_float(v[2 * j]);
                  a.y += __uint_as_float(v[2 * j + 1]);
                  *e = a;
                }
                __syncwarp(vmask);   // another row's next offset may land on this cell
              }
            }
          }
        }
      }
      d_cur = d_nxt; d_nxt = d_nn; m2_cur = m2_nxt;
      tc_fence_before();
      asm volatile("bar.sync 1, 128;" ::: "memory");
      if (et == 0) mbar_arrive_cluster(mapa(tempty_bar(as), 0));   // this CTA's accumulator is free
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
  cluster_sync_all();                 // the peer's shared memory and barriers are no longer in use
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
  }
}

}  // namespace

// ---------------------------------------------------------------------------- host side
typedef CUresult (*PFN_encodeTiled2)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                     const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                     CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static PFN_encodeTiled2 get_encode_fn2() {
  static PFN_encodeTiled2 fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (PFN_encodeTiled2)p;
  }
  return fn;
}

// [nslot][rows][k2] fp32, K contiguous; box = 16 floats x box_rows rows of one slot, 64-byte swizzle
static bool make_map2(PFN_encodeTiled2 enc, CUtensorMap* tm, const float* base, int k2, int64_t rows, int nslot,
                      int box_rows) {
  const cuuint64_t dims[3] = {(cuuint64_t)k2, (cuuint64_t)rows, (cuuint64_t)nslot};
  const cuuint64_t strides[2] = {(cuuint64_t)k2 * 4, (cuuint64_t)k2 * 4 * (cuuint64_t)rows};
  const cuuint32_t box[3] = {(cuuint32_t)T2_KC, (cuuint32_t)box_rows, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)base, dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool tred_mac_tc2_supported(const tred_ctx* ctx) {
  const tred_dims& d = ctx->dims;
  const int N = 2 * d.n_off_pad, K2 = 2 * d.n_phase;
  return N <= T2_NMAX && (N % 32) == 0 && (K2 & 7) == 0 && (size_t)ctx->smem_optin >= T2_SMEM &&
         ctx->cfg.resp_half <= RT_MAXH && ctx->num_sms >= 2 && get_encode_fn2() != nullptr;
}

// [nslot][rows][k2] bf16, K contiguous; box = 16 elements (32 bytes) x box_rows rows, 32-byte swizzle
static bool make_map2_bf16(PFN_encodeTiled2 enc, CUtensorMap* tm, const void* base, int k2, int64_t rows, int nslot,
                           int box_rows) {
  const cuuint64_t dims[3] = {(cuuint64_t)k2, (cuuint64_t)rows, (cuuint64_t)nslot};
  const cuuint64_t strides[2] = {(cuuint64_t)k2 * 2, (cuuint64_t)k2 * 2 * (cuuint64_t)rows};
  const cuuint32_t box[3] = {(cuuint32_t)T2_KC, (cuuint32_t)box_rows, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, (void*)base, dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_32B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// Same contract as tred_mac_tc_fused (tred_mac_tc.cu), on CTA pairs.  Bhb / Blb: the bf16
// copies of B_hi / B_lo; non-NULL selects the variant whose two correction products are bf16.
int tred_mac_tc2(tred_ctx* ctx, const float* qhat, const float* Bhi, const float* Blo, const void* Bhb,
                 const void* Blb, float* opart, int ntile, int t0, const void* rt_desc, const int32_t* row_m2,
                 cudaStream_t st) {
  const tred_dims& d = ctx->dims;
  const int N = 2 * d.n_off_pad, K2 = 2 * d.n_phase;
  const bool bf = Bhb && Blb;
  if (ntile < 1 || !tred_mac_tc2_supported(ctx)) return TRED_EUNSUPPORTED;
  if ((((uintptr_t)qhat) | ((uintptr_t)Bhi) | ((uintptr_t)Blo) | ((uintptr_t)Bhb) | ((uintptr_t)Blb)) & 15)
    return TRED_EUNSUPPORTED;
  PFN_encodeTiled2 enc = get_encode_fn2();
  const int rp = ntile * T2_M;
  T2Maps tm;
  if (!make_map2(enc, &tm.a, qhat, K2, rp, d.n_freq, T2_M) || !make_map2(enc, &tm.bh, Bhi, K2, N, d.n_freq, N / 2))
    return TRED_EUNSUPPORTED;
  if (bf) {
    if (!make_map2_bf16(enc, &tm.bl, Bhb, K2, N, d.n_freq, N / 2) ||
        !make_map2_bf16(enc, &tm.bl2, Blb, K2, N, d.n_freq, N / 2))
      return TRED_EUNSUPPORTED;
  } else {
    if (!make_map2(enc, &tm.bl, Blo, K2, N, d.n_freq, N / 2)) return TRED_EUNSUPPORTED;
    tm.bl2 = tm.bl;
  }
  static bool attr_set[64] = {false};
  if (!attr_set[ctx->device & 63]) {
    TRED_CUDA(cudaFuncSetAttribute(k_mac_tc2<0, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T2_SMEM));
    TRED_CUDA(cudaFuncSetAttribute(k_mac_tc2<11, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T2_SMEM));
    TRED_CUDA(cudaFuncSetAttribute(k_mac_tc2<0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T2_SMEM));
    TRED_CUDA(cudaFuncSetAttribute(k_mac_tc2<11, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T2_SMEM));
    attr_set[ctx->device & 63] = true;
  }
  T2Params p;
  p.nf = d.n_freq; p.ntile = ntile; p.npair = (ntile + 1) / 2;
  p.N = N; p.K2 = K2; p.noff = d.n_off;
  p.K = 2 * ctx->cfg.resp_half + 1; p.H = ctx->cfg.resp_half; p.npy = ctx->cfg.npix_y; p.t0 = t0;
  p.rt_desc = (const int4*)rt_desc; p.row_m2 = row_m2; p.opart = reinterpret_cast<float2*>(opart);
  const int64_t items = (int64_t)p.nf * p.npair;
  int64_t ncl = ctx->num_sms / 2;
  if (ncl > items) ncl = items;
  const int grid = (int)(2 * ncl);
  if (p.K == 11) {
    if (bf) k_mac_tc2<11, true><<<grid, T2_THREADS, T2_SMEM, st>>>(tm, p);
    else k_mac_tc2<11, false><<<grid, T2_THREADS, T2_SMEM, st>>>(tm, p);
  } else {
    if (bf) k_mac_tc2<0, true><<<grid, T2_THREADS, T2_SMEM, st>>>(tm, p);
    else k_mac_tc2<0, false><<<grid, T2_THREADS, T2_SMEM, st>>>(tm, p);
  }
  TRED_LAUNCH_CHECK("k_mac_tc2");
  return TRED_OK;
}
