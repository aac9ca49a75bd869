// Tensor-core variant of the spectrum product (step (b) of tred_conv.cu), tcgen05 / TMEM.
//
// Per frequency slot f the complex product of Eq. (14)
//   T[f][off][row] = sum_phase qhat[f][row][phase] * Rhat[f][phase][off]
// is the real matrix product D[row][n] = sum_kk A[row][kk] * B[n][kk] with
//   A = qhat[f] read as [rows][2 nph] floats (re, im interleaved),
//   B[n = 2 off + c'][kk = 2 phase + c] the real-ified response spectrum (tred_conv.cu).
// fp32 accuracy comes from the 3xTF32 split: every operand x = hi + lo with hi = x
// truncated to tf32 and lo = (x - hi) truncated to tf32, and D = A_hi B_hi + A_lo B_hi +
// A_hi B_lo accumulated in fp32 in tensor memory (the dropped term is ~2^-22 relative).
// B_hi / B_lo are precomputed once per response (tred_prepare_response); A is split in
// shared memory by converter warps, so qhat is read from HBM once, as fp32.
//
// Persistent kernel, one CTA per SM, warp roles:
//   warp 0      TMA producer: K chunks of 16 floats (64-byte swizzled rows) of A, B_hi, B_lo
//   warp 1      MMA issuer (one thread): tcgen05.mma kind::tf32, M = 128, N = 2 kp, K = 8
//   warps 2-5   converters: A -> A_hi (in place), A_lo
//   warps 6-9   epilogue: tcgen05.ld of the accumulator, stores T[f][off][row]
// Two accumulators (2 x 256 TMEM columns) overlap the epilogue of a tile with the MMAs of
// the next.
#include <cuda.h>
#include "tred_common.cuh"

namespace {

constexpr int TC_M = 128;                 // rows per tile (TMEM lanes)
constexpr int TC_KC = 16;                 // floats per K chunk = one 64-byte swizzle row
constexpr int TC_STAGES_PLAIN = 4;        // K-chunk pipeline depth, T written to memory
constexpr int TC_STAGES_FUSED = 3;        // with the patch buffers of the fused epilogue
constexpr int TC_NMAX = 256;              // max N = 2 kp
constexpr int TC_A_BYTES = TC_M * TC_KC * 4;          // 8 KB
constexpr int TC_B_BYTES = TC_NMAX * TC_KC * 4;       // 16 KB
constexpr int TC_STAGE_BYTES = 2 * TC_A_BYTES + 2 * TC_B_BYTES;   // A, A_lo, B_hi, B_lo
constexpr int TC_THREADS = 320;
constexpr int TC_PATCH_FLOAT2 = RT_PXMAX * RT_PYS;                  // one warp's patch accumulator
constexpr size_t TC_SMEM_PLAIN = (size_t)TC_STAGES_PLAIN * TC_STAGE_BYTES + 1024 + 256;
constexpr size_t TC_SMEM_FUSED = (size_t)TC_STAGES_FUSED * TC_STAGE_BYTES + 1024 + 256 + 4 * TC_PATCH_FLOAT2 * 8;

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// Waits for the phase of the given parity to complete.  A wait that lasts longer than
// ~2 s means a broken pipeline: trap instead of hanging the device.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
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
      printf("tred_mac_tc: mbarrier wait timed out (block %d thread %d bar %u parity %u)\n", blockIdx.x,
             threadIdx.x, bar, parity);
      __trap();
    }
  }
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, int c2,
                                            uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(dst), "l"(reinterpret_cast<uint64_t>(tm)), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]^T, kind::tf32, issued by one thread
__device__ __forceinline__ void tc_mma_tf32(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc,
                                            uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t}"
      ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// K-major operand tile of 64-byte swizzled rows (8 rows = one 512-byte swizzle atom)
__device__ __forceinline__ uint64_t make_desc_sw64(uint32_t saddr) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr & 0x3ffff) >> 4);          // start address, 16-byte units
  d |= (uint64_t)1 << 16;                           // leading byte offset (unused for swizzled K-major)
  d |= (uint64_t)(512 >> 4) << 32;                  // stride byte offset: 8 rows x 64 bytes
  d |= (uint64_t)1 << 46;                           // descriptor version (sm_100)
  d |= (uint64_t)4 << 61;                           // layout type SWIZZLE_64B
  return d;
}
__device__ __forceinline__ float tf32_hi(float x) { return __uint_as_float(__float_as_uint(x) & 0xffffe000u); }

struct TcParams {
  int nf, ntile, nrows, rp;     // frequency slots, row tiles, valid rows, padded rows per slot
  int N;                        // 2 kp (multiple of 16, <= 256)
  int K2;                       // 2 nph floats per row (multiple of 8)
  int noff, kp;
  // fused epilogue (row tiles, tred_conv.cu): sum over the offsets into the tile's patch
  int K, H, npy, t0;            // 2H+1, H, pixels along y, first row tile of the chunk
  const int4* rt_desc;          // {first row, rows, py0, ny} per row tile
  const int32_t* row_m2;        // strip-order map index of every row
  float2* opart;                // [tile][f][8 + 2H][RT_PY]
};

// KC: compile-time 2H+1 of the fused epilogue (offset -> patch cell becomes an immediate
// address offset), 0 = read it from the parameters.
template <bool FUSED, int KC>
__global__ void __launch_bounds__(TC_THREADS, 1)
k_mac_tc(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmBh,
         const __grid_constant__ CUtensorMap tmBl, float2* __restrict__ T, TcParams p) {
  constexpr int TC_STAGES = FUSED ? TC_STAGES_FUSED : TC_STAGES_PLAIN;
  extern __shared__ uint8_t smem_raw[];
  const uint32_t raw = smem_u32(smem_raw);
  const uint32_t base = (raw + 1023u) & ~1023u;                  // swizzle atoms need aligned tiles
  uint8_t* base_ptr = smem_raw + (base - raw);
  const uint32_t bars = base + TC_STAGES * TC_STAGE_BYTES;       // 8-byte mbarriers
  auto full_bar = [&](int s) { return bars + 8u * s; };
  auto conv_bar = [&](int s) { return bars + 8u * (TC_STAGES + s); };
  auto empty_bar = [&](int s) { return bars + 8u * (2 * TC_STAGES + s); };
  auto tfull_bar = [&](int a) { return bars + 8u * (3 * TC_STAGES + a); };
  auto tempty_bar = [&](int a) { return bars + 8u * (3 * TC_STAGES + 2 + a); };
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(base_ptr + TC_STAGES * TC_STAGE_BYTES + 8 * (3 * TC_STAGES + 4));
  auto sA = [&](int s) { return base + s * TC_STAGE_BYTES; };
  auto sAlo = [&](int s) { return base + s * TC_STAGE_BYTES + TC_A_BYTES; };
  auto sBh = [&](int s) { return base + s * TC_STAGE_BYTES + 2 * TC_A_BYTES; };
  auto sBl = [&](int s) { return base + s * TC_STAGE_BYTES + 2 * TC_A_BYTES + TC_B_BYTES; };

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int nkc = (p.K2 + TC_KC - 1) / TC_KC;
  const int nitems = p.nf * p.ntile;

  if (threadIdx.x == 0) {
    for (int s = 0; s < TC_STAGES; ++s) {
      mbar_init(full_bar(s), 1);
      mbar_init(conv_bar(s), 128);
      mbar_init(empty_bar(s), 1);
    }
    for (int a = 0; a < 2; ++a) {
      mbar_init(tfull_bar(a), 1);
      mbar_init(tempty_bar(a), 128);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)),
                 "r"(512)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_base = *tmem_slot;

  if (warp == 0) {
    // ------------------------------------------------------------ TMA producer
    if (lane == 0) {
      const uint32_t tx = (uint32_t)(TC_A_BYTES + 2 * p.N * TC_KC * 4);
      int stage = 0, phase = 0;
      for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
        const int f = item / p.ntile, mt = item - f * p.ntile;
        for (int kc = 0; kc < nkc; ++kc) {
          mbar_wait(empty_bar(stage), phase ^ 1);
          mbar_expect_tx(full_bar(stage), tx);
          tma_load_3d(sA(stage), &tmA, kc * TC_KC, mt * TC_M, f, full_bar(stage));
          tma_load_3d(sBh(stage), &tmBh, kc * TC_KC, 0, f, full_bar(stage));
          tma_load_3d(sBl(stage), &tmBl, kc * TC_KC, 0, f, full_bar(stage));
          if (++stage == TC_STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == 1) {
    // ------------------------------------------------------------ MMA issuer
    if (lane == 0) {
      // instruction descriptor: D fp32, A/B tf32, both K-major, N, M = 128
      const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(p.N >> 3) << 17) | ((uint32_t)(TC_M >> 4) << 24);
      int stage = 0, phase = 0, as = 0, aphase = 0;
      for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
        mbar_wait(tempty_bar(as), aphase ^ 1);
        tc_fence_after();
        const uint32_t d_tmem = tmem_base + (uint32_t)(as * TC_NMAX);
        for (int kc = 0; kc < nkc; ++kc) {
          mbar_wait(full_bar(stage), phase);
          mbar_wait(conv_bar(stage), phase);
          tc_fence_after();
          const int nks = min(TC_KC, p.K2 - kc * TC_KC) >> 3;      // K = 8 floats per MMA
          const uint64_t da = make_desc_sw64(sA(stage)), dl = make_desc_sw64(sAlo(stage));
          const uint64_t dbh = make_desc_sw64(sBh(stage)), dbl = make_desc_sw64(sBl(stage));
          for (int ks = 0; ks < nks; ++ks) {
            const uint64_t adv = (uint64_t)(ks * 2);               // 32 bytes along K, 16-byte units
            tc_mma_tf32(d_tmem, da + adv, dbh + adv, idesc, (kc | ks) != 0);
            tc_mma_tf32(d_tmem, dl + adv, dbh + adv, idesc, 1);
            tc_mma_tf32(d_tmem, da + adv, dbl + adv, idesc, 1);
          }
          tc_commit(empty_bar(stage));                             // frees the stage when the MMAs retire
          if (++stage == TC_STAGES) { stage = 0; phase ^= 1; }
        }
        tc_commit(tfull_bar(as));                                  // accumulator complete
        if (++as == 2) { as = 0; aphase ^= 1; }
      }
    }
  } else if (warp < 6) {
    // ------------------------------------------------------------ converters: A -> A_hi, A_lo
    const int tc = threadIdx.x - 64;
    int stage = 0, phase = 0;
    for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
      for (int kc = 0; kc < nkc; ++kc) {
        mbar_wait(full_bar(stage), phase);
        float4* a = reinterpret_cast<float4*>(base_ptr + stage * TC_STAGE_BYTES);
        float4* lo = reinterpret_cast<float4*>(base_ptr + stage * TC_STAGE_BYTES + TC_A_BYTES);
#pragma unroll
        for (int i = 0; i < TC_A_BYTES / 16 / 128; ++i) {
          const float4 v = a[tc + 128 * i];
          float4 h, l;
          h.x = tf32_hi(v.x); h.y = tf32_hi(v.y); h.z = tf32_hi(v.z); h.w = tf32_hi(v.w);
          l.x = tf32_hi(v.x - h.x); l.y = tf32_hi(v.y - h.y); l.z = tf32_hi(v.z - h.z); l.w = tf32_hi(v.w - h.w);
          a[tc + 128 * i] = h;
          lo[tc + 128 * i] = l;
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic writes -> tensor core reads
        mbar_arrive(conv_bar(stage));
        if (++stage == TC_STAGES) { stage = 0; phase ^= 1; }
      }
    }
  } else if (!FUSED) {
    // ------------------------------------------------------------ epilogue: store T
    const int q = warp & 3;                                        // TMEM lane quadrant of this warp
    int as = 0, aphase = 0;
    for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
      const int f = item / p.ntile, mt = item - f * p.ntile;
      mbar_wait(tfull_bar(as), aphase);
      tc_fence_after();
      const int row = mt * TC_M + q * 32 + lane;
      const uint32_t taddr = tmem_base + (uint32_t)(as * TC_NMAX) + ((uint32_t)(q * 32) << 16);
      float2* dst = T + (int64_t)f * p.kp * p.rp + row;
      for (int c0 = 0; c0 * 16 < p.noff; ++c0) {
        uint32_t r[32];
        asm volatile(
            "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
            "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
            "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
            : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
              "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
              "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
              "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
            : "r"(taddr + (uint32_t)(c0 * 32))
            : "memory");
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        if (row < p.nrows) {
#pragma unroll
          for (int j = 0; j < 16; ++j) {
            const int off = c0 * 16 + j;
            if (off < p.noff)
              dst[(int64_t)off * p.rp] = make_float2(__uint_as_float(r[2 * j]), __uint_as_float(r[2 * j + 1]));
          }
        }
      }
      tc_fence_before();
      mbar_arrive(tempty_bar(as));
      if (++as == 2) { as = 0; aphase ^= 1; }
    }
  } else {
    // ------------------------------------------------------------ epilogue: sum over offsets
    // Row r of the tile is the charge pixel (8 strip + xl, py0 + yl); its product with
    // offset (kx, ky) belongs to patch cell (xl + kx + H, yl + ky + H).  For a fixed offset
    // the rows of a warp hit distinct cells, so each warp adds into its own patch copy
    // without atomics; the four copies are then summed in a fixed order.
    const int q = warp & 3;                                        // TMEM lane quadrant of this warp
    const int et = threadIdx.x - 192;                              // 0..127
    float2* patch = reinterpret_cast<float2*>(base_ptr + TC_STAGES * TC_STAGE_BYTES + 256);
    float2* P = patch + q * TC_PATCH_FLOAT2;
    for (int i = et; i < 4 * TC_PATCH_FLOAT2; i += 128) patch[i] = make_float2(0.0f, 0.0f);
    asm volatile("bar.sync 1, 128;" ::: "memory");
    const int PX = RT_SW + 2 * p.H;
    int as = 0, aphase = 0;
    for (int item = blockIdx.x; item < nitems; item += gridDim.x) {
      const int f = item / p.ntile, mt = item - f * p.ntile;
      const int4 d = p.rt_desc[p.t0 + mt];
      const int r = q * 32 + lane;
      const bool valid = r < d.y;
      const uint32_t vmask = __ballot_sync(0xffffffffu, valid);
      int cell0 = 0;
      if (valid) {
        const int m2 = p.row_m2[d.x + r];
        cell0 = (m2 & (RT_SW - 1)) * RT_PYS + ((m2 >> 3) % p.npy - d.z);
      }
      mbar_wait(tfull_bar(as), aphase);
      tc_fence_after();
      const uint32_t taddr = tmem_base + (uint32_t)(as * TC_NMAX) + ((uint32_t)(q * 32) << 16);
      const int KK = KC ? KC : p.K;
      const int noff = KC ? KC * KC : p.noff;
#pragma unroll
      for (int c0 = 0; c0 < (KC ? (KC * KC + 15) / 16 : 8); ++c0) {
        if (!KC && c0 * 16 >= noff) break;
        uint32_t v[32];
        asm volatile(
            "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
            "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
            "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
            : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]),
              "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]),
              "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]),
              "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
            : "r"(taddr + (uint32_t)(c0 * 32))
            : "memory");
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
            __syncwarp(vmask);       // another row's next offset may land on this cell
          }
        }
      }
      tc_fence_before();
      mbar_arrive(tempty_bar(as));                                 // accumulator free for the next tile
      if (++as == 2) { as = 0; aphase ^= 1; }
      asm volatile("bar.sync 1, 128;" ::: "memory");
      const int nyp = d.w + 2 * p.H, ncell = PX * nyp;
      float2* dst = p.opart + ((int64_t)mt * p.nf + f) * (PX * RT_PY);
      for (int i = et; i < ncell; i += 128) {
        const int X = i / nyp, Y = i - X * nyp;
        const int c = X * RT_PYS + Y;
        float2 a = patch[c];
#pragma unroll
        for (int w = 1; w < 4; ++w) {
          const float2 b = patch[w * TC_PATCH_FLOAT2 + c];
          a.x += b.x; a.y += b.y;
        }
#pragma unroll
        for (int w = 0; w < 4; ++w) patch[w * TC_PATCH_FLOAT2 + c] = make_float2(0.0f, 0.0f);
        dst[X * RT_PY + Y] = a;
      }
      asm volatile("bar.sync 1, 128;" ::: "memory");
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem_base), "r"(512) : "memory");
  }
}

}  // namespace

// ---------------------------------------------------------------------------- host side
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static PFN_encodeTiled get_encode_fn() {
  static PFN_encodeTiled fn = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = (PFN_encodeTiled)p;
  }
  return fn;
}

// [nslot][rows][k2] fp32, K contiguous; box = 16 floats x box_rows rows of one slot, 64-byte swizzle
static bool make_map(PFN_encodeTiled enc, CUtensorMap* tm, const float* base, int k2, int64_t rows, int nslot,
                     int box_rows) {
  const cuuint64_t dims[3] = {(cuuint64_t)k2, (cuuint64_t)rows, (cuuint64_t)nslot};
  const cuuint64_t strides[2] = {(cuuint64_t)k2 * 4, (cuuint64_t)k2 * 4 * (cuuint64_t)rows};
  const cuuint32_t box[3] = {(cuuint32_t)TC_KC, (cuuint32_t)box_rows, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)base, dims, strides, box, estr,
             CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
             CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

static int tc_check(const tred_ctx* ctx, const float* qhat, const float* Bhi, const float* Blo, int rp, size_t smem,
                    PFN_encodeTiled* enc) {
  const tred_dims& d = ctx->dims;
  const int N = 2 * d.n_off_pad, K2 = 2 * d.n_phase;
  if (N > TC_NMAX || (N & 15) || (K2 & 7) || (rp % TC_M) || rp < TC_M) return TRED_EUNSUPPORTED;
  if ((size_t)ctx->smem_optin < smem) return TRED_EUNSUPPORTED;
  if ((((uintptr_t)qhat) | ((uintptr_t)Bhi) | ((uintptr_t)Blo)) & 15) return TRED_EUNSUPPORTED;
  *enc = get_encode_fn();
  return *enc ? TRED_OK : TRED_EUNSUPPORTED;
}

// Can the fused (row tile) path run this configuration at all?  (tred_conv.cu asks before
// it lays the workspace out.)
bool tred_mac_tc_fused_supported(const tred_ctx* ctx) {
  const tred_dims& d = ctx->dims;
  const int N = 2 * d.n_off_pad, K2 = 2 * d.n_phase;
  return !(N > TC_NMAX || (N & 15) || (K2 & 7)) && (size_t)ctx->smem_optin >= TC_SMEM_FUSED &&
         ctx->cfg.resp_half <= RT_MAXH && get_encode_fn() != nullptr;
}

// Fused variant: ntile row tiles of 128 padded rows each (rp = 128 ntile), the products
// summed over the offsets into opart[tile][f][8 + 2H][RT_PY].
int tred_mac_tc_fused(tred_ctx* ctx, const float* qhat, const float* Bhi, const float* Blo, float* opart,
                      int ntile, int t0, const void* rt_desc, const int32_t* row_m2, cudaStream_t st) {
  const tred_dims& d = ctx->dims;
  const int N = 2 * d.n_off_pad, K2 = 2 * d.n_phase;
  const int rp = ntile * TC_M;
  PFN_encodeTiled enc = nullptr;
  if (ntile < 1 || ctx->cfg.resp_half > RT_MAXH) return TRED_EUNSUPPORTED;
  int rc = tc_check(ctx, qhat, Bhi, Blo, rp, TC_SMEM_FUSED, &enc);
  if (rc != TRED_OK) return rc;
  CUtensorMap tmA, tmBh, tmBl;
  if (!make_map(enc, &tmA, qhat, K2, rp, d.n_freq, TC_M) || !make_map(enc, &tmBh, Bhi, K2, N, d.n_freq, N) ||
      !make_map(enc, &tmBl, Blo, K2, N, d.n_freq, N))
    return TRED_EUNSUPPORTED;
  static bool attr_set[64] = {false};
  if (!attr_set[ctx->device & 63]) {
    TRED_CUDA(cudaFuncSetAttribute(k_mac_tc<true, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM_FUSED));
    TRED_CUDA(cudaFuncSetAttribute(k_mac_tc<true, 11>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM_FUSED));
    attr_set[ctx->device & 63] = true;
  }
  TcParams p;
  p.nf = d.n_freq; p.ntile = ntile; p.nrows = rp; p.rp = rp;
  p.N = N; p.K2 = K2; p.noff = d.n_off; p.kp = d.n_off_pad;
  p.K = 2 * ctx->cfg.resp_half + 1; p.H = ctx->cfg.resp_half; p.npy = ctx->cfg.npix_y; p.t0 = t0;
  p.rt_desc = (const int4*)rt_desc; p.row_m2 = row_m2; p.opart = reinterpret_cast<float2*>(opart);
  const int64_t items = (int64_t)p.nf * p.ntile;
  const int grid = (int)(items < ctx->num_sms ? items : ctx->num_sms);
  if (p.K == 11)
    k_mac_tc<true, 11><<<grid, TC_THREADS, TC_SMEM_FUSED, st>>>(tmA, tmBh, tmBl, nullptr, p);
  else
    k_mac_tc<true, 0><<<grid, TC_THREADS, TC_SMEM_FUSED, st>>>(tmA, tmBh, tmBl, nullptr, p);
  TRED_LAUNCH_CHECK("k_mac_tc<fused>");
  return TRED_OK;
}

// Returns TRED_EUNSUPPORTED when this configuration cannot run on the tensor-core kernel
// (tred_convolve then uses the fp32 FMA kernel unless mac_mode forces this one).
int tred_mac_tc(tred_ctx* ctx, const float* qhat, const float* Bhi, const float* Blo, float* T, int nrows, int rp,
                cudaStream_t st) {
  const tred_dims& d = ctx->dims;
  const int N = 2 * d.n_off_pad, K2 = 2 * d.n_phase;
  if (N > TC_NMAX || (N & 15) || (K2 & 7) || (rp % TC_M) || nrows < 1) return TRED_EUNSUPPORTED;
  if ((size_t)ctx->smem_optin < TC_SMEM_PLAIN) return TRED_EUNSUPPORTED;
  if ((((uintptr_t)qhat) | ((uintptr_t)Bhi) | ((uintptr_t)Blo)) & 15) return TRED_EUNSUPPORTED;
  PFN_encodeTiled enc = get_encode_fn();
  if (!enc) return TRED_EUNSUPPORTED;
  CUtensorMap tmA, tmBh, tmBl;
  if (!make_map(enc, &tmA, qhat, K2, rp, d.n_freq, TC_M) || !make_map(enc, &tmBh, Bhi, K2, N, d.n_freq, N) ||
      !make_map(enc, &tmBl, Blo, K2, N, d.n_freq, N))
    return TRED_EUNSUPPORTED;
  static bool attr_set[64] = {false};
  if (!attr_set[ctx->device & 63]) {
    TRED_CUDA(cudaFuncSetAttribute(k_mac_tc<false, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TC_SMEM_PLAIN));
    attr_set[ctx->device & 63] = true;
  }
  TcParams p;
  p.nf = d.n_freq; p.ntile = (nrows + TC_M - 1) / TC_M; p.nrows = nrows; p.rp = rp;
  p.N = N; p.K2 = K2; p.noff = d.n_off; p.kp = d.n_off_pad;
  p.K = 0; p.H = 0; p.npy = 0; p.t0 = 0; p.rt_desc = nullptr; p.row_m2 = nullptr; p.opart = nullptr;
  const int64_t items = (int64_t)p.nf * p.ntile;
  const int grid = (int)(items < ctx->num_sms ? items : ctx->num_sms);
  k_mac_tc<false, 0><<<grid, TC_THREADS, TC_SMEM_PLAIN, st>>>(tmA, tmBh, tmBl, reinterpret_cast<float2*>(T), p);
  TRED_LAUNCH_CHECK("k_mac_tc");
  return TRED_OK;
}
