// Spectrum product of Eq. (14) as THREE fp16 tensor-core products on
// CTA pairs (tcgen05.mma.cta_group::2 kind::f16, fp32 accumulation in TMEM), with the sum
// over the response offsets fused into the epilogue (row tiles: see tred_conv.cu).
//
// Split: every operand is x = s (hi + lo) with s a power of two (per row of A: from the
// column sums of the charge, which bound every spectrum value; per frequency for B),
// hi = fp16(x / s), lo = fp16(x / s - hi).  fp16 carries 11 significant bits, so hi + lo
// carries 22; the product is  A B = s_A s_B (A_hi B_hi + A_lo B_hi + A_hi B_lo)  up to the
// dropped 2^-22 term, the same error class as 3xTF32 at three quarters of its tensor time
// (kind::f16 runs at twice the tf32 rate) and with half the operand bytes.
//
// Operand layout in HBM (written by the forward FFT / tred_prepare_response), K-major, the
// reals kk = 2 phase + (re | im) in blocks of 16:
//     row = [ hi(kk 0..15) | lo(kk 0..15) | hi(kk 16..31) | lo(kk 16..31) | ... ]  fp16
// A K chunk is one 128-byte swizzled row (SWIZZLE_128B, the widest operand rows the tensor
// core reads) = two blocks; TMA fills a stage, the MMAs of a block are
//     D += A_hi B_hi,  D += A_lo B_hi,  D += A_hi B_lo        (K = 16 each)
// picked by 32-byte steps of the shared-memory descriptors.  There are no converter warps:
// the stage goes from TMA straight to the tensor core.
//
// Per CTA: warp 0 TMA producer (own A tile, own half of B), warp 1 MMA issuer (leader CTA
// only), warps 2-5 and 6-9 two epilogue sets: set s owns TMEM accumulator s (the items of
// the cluster alternate between the two) and its own four patch copies, so the epilogue of
// an item has two MMA periods to finish (its chain of shared-memory read-modify-writes takes
// longer than one).  Barriers: `full` lives in the leader: both CTAs' producers
// arrive on it with their byte counts and both CTAs' TMA loads (cta_group::2) complete on it,
// so the MMA issuer waits on one barrier per stage; empty / tfull are local to each CTA and
// arrive through tcgen05.commit multicast; tempty lives in the leader, one arrival per CTA.
#include <cuda_fp16.h>
#include "tred_tc2_common.cuh"

namespace {

constexpr int H3_STAGES = 4;
constexpr int H3_A_BYTES = T2_M * 128;                   // 128 rows x 128 bytes
constexpr int H3_B_BYTES = (T2_NMAX / 2) * 128;          // this CTA's half of B
constexpr int H3_STAGE_BYTES = H3_A_BYTES + H3_B_BYTES;  // 32 KB
constexpr int H3_THREADS = 320;
constexpr size_t H3_SMEM = (size_t)H3_STAGES * H3_STAGE_BYTES + 1024 + 256 + 8 * T2_PATCH_FLOAT2 * 8;

struct H3Maps { CUtensorMap a, b; };

struct H3Params {
  int nf, ntile, npair;
  int N, nb16, noff;            // nb16: blocks of 16 reals per row = ceil(2 nph / 16)
  int K, H, npy, t0;
  const int4* rt_desc;
  const int32_t* row_m2;
  const float* rscale;          // [ntile * 128] power-of-two scale of every row of A
  const float* bscale;          // [nf] power-of-two scale of B per frequency
  float2* opart;                // [tile][f][8 + 2H][RT_PY]
};

__device__ __forceinline__ void tc_mma_f16_pair(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                                uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void mbar_expect_tx_cluster(uint32_t bar_cluster_addr, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cluster.b64 _, [%0], %1;" ::"r"(bar_cluster_addr), "r"(bytes)
               : "memory");
}
// TMA load into this CTA's shared memory whose completion is signalled on a barrier of the
// pair's leader CTA
__device__ __forceinline__ void tma_load_3d_pair(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2,
                                                 uint32_t bar_cluster_addr) {
  asm volatile(
      "cp.async.bulk.tensor.3d.cta_group::2.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(c2), "r"(bar_cluster_addr)
      : "memory");
}
// K-major operand tile of 128-byte swizzled rows (8 rows = one 1024-byte swizzle atom)
__device__ __forceinline__ uint64_t make_desc_sw128(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3ffff) >> 4);
  d |= (uint64_t)1 << 16;
  d |= (uint64_t)(1024 >> 4) << 32;
  d |= (uint64_t)1 << 46;
  d |= (uint64_t)2 << 61;                           // SWIZZLE_128B
  return d;
}

template <int KC>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(H3_THREADS, 1)
k_mac_h3(const __grid_constant__ H3Maps tm, H3Params p) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;                  // identical in both CTAs of the pair
  uint8_t* base_ptr = smem_raw + (base - raw);
  const uint32_t bars = base + H3_STAGES * H3_STAGE_BYTES;
  auto full_bar = [&](int s) { return bars + 8u * s; };
  auto empty_bar = [&](int s) { return bars + 8u * (H3_STAGES + s); };
  auto tfull_bar = [&](int a) { return bars + 8u * (2 * H3_STAGES + a); };
  auto tempty_bar = [&](int a) { return bars + 8u * (2 * H3_STAGES + 2 + a); }; // used in the leader
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(base_ptr + H3_STAGES * H3_STAGE_BYTES + 8 * (2 * H3_STAGES + 4));
  auto sA = [&](int s) { return base + s * H3_STAGE_BYTES; };
  auto sB = [&](int s) { return base + s * H3_STAGE_BYTES + H3_A_BYTES; };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const uint32_t rank = cluster_ctarank();
  const int nkc = (p.nb16 + 1) >> 1;
  const int nitems = p.nf * p.npair;
  const int cid = blockIdx.x >> 1, ncl = gridDim.x >> 1;

  if (threadIdx.x == 0) {
    for (int s = 0; s < H3_STAGES; ++s) {
      mbar_init(full_bar(s), 2);
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
      const uint32_t tx = (uint32_t)(H3_A_BYTES + nh * 128);
      int stage = 0, phase = 0;
      for (int item = cid; item < nitems; item += ncl) {
        const int f = item / p.npair, pr = item - f * p.npair;
        const int mt = min(2 * pr + (int)rank, p.ntile - 1);
        // qhat streams from HBM once: have L2 fetch the next item's A tile now
        if (item + ncl < nitems) {
          const int fn = (item + ncl) / p.npair, prn = (item + ncl) - fn * p.npair;
          const int mtn = min(2 * prn + (int)rank, p.ntile - 1);
          for (int kc = 0; kc < nkc; ++kc) tma_prefetch_3d(&tm.a, kc * 64, 0, mtn * p.nf + fn);
        }
        for (int kc = 0; kc < nkc; ++kc) {
          mbar_wait(empty_bar(stage), phase ^ 1);
          const uint32_t fb = mapa(full_bar(stage), 0);            // the leader's barrier
          mbar_expect_tx_cluster(fb, tx);
          tma_load_3d_pair(sA(stage), &tm.a, kc * 64, 0, mt * p.nf + f, fb);
          tma_load_3d_pair(sB(stage), &tm.b, kc * 64, (int)rank * nh, f, fb);
          if (++stage == H3_STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------ MMA issuer (leader CTA)
    if (lane == 0 && rank == 0) {
      // instruction descriptor: D fp32, A / B fp16, both K-major, N, M = 256 over the pair
      const uint32_t idesc = (1u << 4) | ((uint32_t)(p.N >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
      int stage = 0, phase = 0, as = 0, aphase = 0;
      for (int item = cid; item < nitems; item += ncl) {
        mbar_wait(tempty_bar(as), aphase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(as * T2_NMAX);
        for (int kc = 0; kc < nkc; ++kc) {
          mbar_wait(full_bar(stage), phase);                       // both CTAs' loads have landed
          tc_fence_after();
          const int nb = min(2, p.nb16 - 2 * kc);
          const uint64_t da = make_desc_sw128(sA(stage)), db = make_desc_sw128(sB(stage));
          for (int j = 0; j < nb; ++j) {
            const uint64_t hi = (uint64_t)(4 * j), lo = (uint64_t)(4 * j + 2);     // 16-byte units
            tc_mma_f16_pair(d_tmem, da + hi, db + hi, idesc, (kc | j) != 0);
            tc_mma_f16_pair(d_tmem, da + lo, db + hi, idesc, 1);
            tc_mma_f16_pair(d_tmem, da + hi, db + lo, idesc, 1);
          }
          tc_commit_pair(empty_bar(stage));                        // frees the stage in both CTAs
          if (++stage == H3_STAGES) { stage = 0; phase ^= 1; }
        }
        tc_commit_pair(tfull_bar(as));                             // accumulators complete in both CTAs
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
  } else {
    // ------------------------------------------------------------ epilogue: sum over offsets
    const int q = warp & 3;
    const int es = (warp - 2) >> 2;                               // epilogue set = accumulator
    const int et = (threadIdx.x - 64) & 127;
    const uint32_t ebar = 1 + es;                                  // named barrier of the set
    float2* patch = reinterpret_cast<float2*>(base_ptr + H3_STAGES * H3_STAGE_BYTES + 256) + es * 4 * T2_PATCH_FLOAT2;
    float2* P = patch + q * T2_PATCH_FLOAT2;
    for (int i = et; i < 4 * T2_PATCH_FLOAT2; i += 128) patch[i] = make_float2(0.0f, 0.0f);
    asm volatile("bar.sync %0, 128;" ::"r"(ebar) : "memory");
    const int PX = RT_SW + 2 * p.H;
    const int as = es;
    int aphase = 0;
    const int first = cid + es * ncl, stride = 2 * ncl;            // this set's items
    // Row tile descriptor and this thread's row record are fetched one / two items ahead
    // (two dependent global loads otherwise sit on the epilogue's critical path).
    auto item_tile = [&](int it) { return it < nitems ? 2 * (it % p.npair) + (int)rank : p.ntile; };
    auto load_desc = [&](int it) {
      const int t = item_tile(it);
      return t < p.ntile ? p.rt_desc[p.t0 + t] : make_int4(0, 0, 0, 0);
    };
    const int r = q * 32 + lane;
    int4 d_cur = load_desc(first), d_nxt = load_desc(first + stride);
    int m2_cur = r < d_cur.y ? p.row_m2[d_cur.x + r] : 0;
    float rs_cur = r < d_cur.y ? p.rscale[item_tile(first) * T2_M + r] : 0.0f;
    for (int item = first; item < nitems; item += stride) {
      const int f = item / p.npair, pr = item - f * p.npair;
      const int mt = 2 * pr + (int)rank;
      const bool has_tile = mt < p.ntile;
      const int4 d = d_cur;
      const int m2 = m2_cur;
      const float sc = rs_cur * __ldg(p.bscale + f);
      // prefetch: record of the next item (its descriptor arrived an iteration ago), descriptor of the one after
      const int m2_nxt = r < d_nxt.y ? p.row_m2[d_nxt.x + r] : 0;
      const float rs_nxt = r < d_nxt.y ? p.rscale[item_tile(item + stride) * T2_M + r] : 0.0f;
      const int4 d_nn = load_desc(item + 2 * stride);
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
            a.x = fmaf(__uint_as_float(re), sc, a.x);
            a.y = fmaf(__uint_as_float(im), sc, a.y);
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
                  a.x = fmaf(__uint_as_float(v[2 * j]), sc, a.x);
                  a.y = fmaf(__uint_as_float(v[2 * j + 1]), sc, a.y);
                  *e = a;
                }
                __syncwarp(vmask);   // another row's next offset may land on this cell
              }
            }
          }
        }
      }
      d_cur = d_nxt; d_nxt = d_nn; m2_cur = m2_nxt; rs_cur = rs_nxt;
      tc_fence_before();
      asm volatile("bar.sync %0, 128;" ::"r"(ebar) : "memory");
      if (et == 0) mbar_arrive_cluster(mapa(tempty_bar(as), 0));   // this CTA's accumulator is free
      aphase ^= 1;
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
      asm volatile("bar.sync %0, 128;" ::"r"(ebar) : "memory");
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
typedef CUresult (*PFN_encodeTiledH3)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                      const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                      CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static PFN_encodeTiledH3 get_encode_fn_h3() {
  static PFN_encodeTiledH3 fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (PFN_encodeTiledH3)p;
  }
  return fn;
}

// [nslot][rows][kp] fp16, K contiguous; box = 64 halves (128 bytes) x box_rows rows of one slot
static bool make_map_h3(PFN_encodeTiledH3 enc, CUtensorMap* tm, const void* base, int kp, int64_t rows, int nslot,
                        int box_rows) {
  const cuuint64_t dims[3] = {(cuuint64_t)kp, (cuuint64_t)rows, (cuuint64_t)nslot};
  const cuuint64_t strides[2] = {(cuuint64_t)kp * 2, (cuuint64_t)kp * 2 * (cuuint64_t)rows};
  const cuuint32_t box[3] = {64, (cuuint32_t)box_rows, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 3, (void*)base, dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool tred_mac_h3_supported(const tred_ctx* ctx) {
  const tred_dims& d = ctx->dims;
  const int N = 2 * d.n_off_pad;
  return N <= T2_NMAX && (N % 32) == 0 && (size_t)ctx->smem_optin >= H3_SMEM &&
         ctx->cfg.resp_half <= RT_MAXH && ctx->num_sms >= 2 && get_encode_fn_h3() != nullptr;
}

// qh: [ntile][nf][128][kp16] fp16 in the hi / lo block layout (kp16 = h16_kp(dims)), rscale
// [ntile * 128]; Bh16: [nf][N][kp16] fp16, bscale [nf].  Same outputs as tred_mac_tc2.
int tred_mac_h3(tred_ctx* ctx, const void* qh, const float* rscale, const void* Bh16, const float* bscale,
                float* opart, int ntile, int t0, const void* rt_desc, const int32_t* row_m2, cudaStream_t st) {
  const tred_dims& d = ctx->dims;
  const int N = 2 * d.n_off_pad;
  const int kp16 = h16_kp(d);
  if (ntile < 1 || !tred_mac_h3_supported(ctx)) return TRED_EUNSUPPORTED;
  if ((((uintptr_t)qh) | ((uintptr_t)Bh16)) & 15) return TRED_EUNSUPPORTED;
  PFN_encodeTiledH3 enc = get_encode_fn_h3();
  H3Maps tm;
  if ((int64_t)ntile * d.n_freq >= (1ll << 31)) return TRED_EUNSUPPORTED;
  if (!make_map_h3(enc, &tm.a, qh, kp16, T2_M, ntile * d.n_freq, T2_M) ||
      !make_map_h3(enc, &tm.b, Bh16, kp16, N, d.n_freq, N / 2))
    return TRED_EUNSUPPORTED;
  TRED_CUDA(cudaFuncSetAttribute(k_mac_h3<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)H3_SMEM));
  TRED_CUDA(cudaFuncSetAttribute(k_mac_h3<11>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)H3_SMEM));
  H3Params p;
  p.nf = d.n_freq; p.ntile = ntile; p.npair = (ntile + 1) / 2;
  p.N = N; p.nb16 = kp16 / 32; p.noff = d.n_off;
  p.K = 2 * ctx->cfg.resp_half + 1; p.H = ctx->cfg.resp_half; p.npy = ctx->cfg.npix_y; p.t0 = t0;
  p.rt_desc = (const int4*)rt_desc; p.row_m2 = row_m2; p.rscale = rscale; p.bscale = bscale;
  p.opart = reinterpret_cast<float2*>(opart);
  const int64_t items = (int64_t)p.nf * p.npair;
  int64_t ncl = ctx->num_sms / 2;
  if (ncl > items) ncl = items;
  const int grid = (int)(2 * ncl);
  if (p.K == 11) k_mac_h3<11><<<grid, H3_THREADS, H3_SMEM, st>>>(tm, p);
  else k_mac_h3<0><<<grid, H3_THREADS, H3_SMEM, st>>>(tm, p);
  TRED_LAUNCH_CHECK("k_mac_h3");
  return TRED_OK;
}
