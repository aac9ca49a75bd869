// Context, derived sizes, S1 drift and S3 block binning
// (PAPER.md:L57,L236-240).
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include "tred_common.cuh"

// ------------------------------------------------------------------ errors
static thread_local char g_cuda_err[512] = "";

void tred_set_cuda_error(cudaError_t e, const char* where) {
  snprintf(g_cuda_err, sizeof(g_cuda_err), "%s: %s (%s)", where, cudaGetErrorName(e),
           cudaGetErrorString(e));
}

extern "C" const char* tred_last_cuda_error(void) { return g_cuda_err; }

// ------------------------------------------------------------------ stage profiling
thread_local int64_t g_tred_launches = 0;

TredProfScope::TredProfScope(tred_ctx* ctx, int stage_, cudaStream_t st_)
    : c(ctx), stage(stage_), st(st_), l0(g_tred_launches), rec(-1) {
  if (!c || !c->prof_on) return;
  if (c->nrecs == c->cap_recs) {
    int nc = c->cap_recs ? 2 * c->cap_recs : 256;
    TredProfRec* nr = (TredProfRec*)realloc(c->recs, sizeof(TredProfRec) * nc);
    if (!nr) return;
    c->recs = nr; c->cap_recs = nc;
  }
  TredProfRec& r = c->recs[c->nrecs];
  r.stage = stage;
  if (cudaEventCreate(&r.a) != cudaSuccess) return;
  if (cudaEventCreate(&r.b) != cudaSuccess) { cudaEventDestroy(r.a); return; }
  cudaEventRecord(r.a, st);
  rec = c->nrecs++;
}

TredProfScope::~TredProfScope() {
  if (c) c->launches[stage] += g_tred_launches - l0;
  if (rec >= 0) cudaEventRecord(c->recs[rec].b, st);
}

static void prof_clear(tred_ctx* c) {
  for (int i = 0; i < c->nrecs; ++i) { cudaEventDestroy(c->recs[i].a); cudaEventDestroy(c->recs[i].b); }
  c->nrecs = 0;
  for (int s = 0; s < ST_COUNT; ++s) c->launches[s] = 0;
}

extern "C" int tred_profile_begin(tred_ctx* c, int record_events) {
  if (!c) return TRED_EINVAL;
  TRED_CHECK_DEVICE(c);
  prof_clear(c);
  c->prof_on = record_events ? 1 : 0;
  return TRED_OK;
}

extern "C" int tred_profile_end(tred_ctx* c, int nstage, float* h_ms, int64_t* h_launches) {
  if (!c || nstage < 0) return TRED_EINVAL;
  TRED_CHECK_DEVICE(c);
  for (int s = 0; s < nstage; ++s) { if (h_ms) h_ms[s] = 0.0f; if (h_launches) h_launches[s] = 0; }
  for (int i = 0; i < c->nrecs; ++i) {
    TredProfRec& r = c->recs[i];
    TRED_CUDA(cudaEventSynchronize(r.b));
    float ms = 0.0f;
    TRED_CUDA(cudaEventElapsedTime(&ms, r.a, r.b));
    if (h_ms && r.stage < nstage) h_ms[r.stage] += ms;
  }
  for (int s = 0; s < nstage && s < ST_COUNT; ++s) if (h_launches) h_launches[s] = c->launches[s];
  prof_clear(c);
  c->prof_on = 0;
  return TRED_OK;
}

// ------------------------------------------------------------------ fp32 FMA peak (measurement aid)
// 8 independent FMA chains per thread, nothing else in the loop: what the fp32 pipes of
// this device sustain, the denominator bench.py uses for the "alu" rooflines.
__global__ void __launch_bounds__(256) k_bench_fma(int iters, float seed, float* __restrict__ out) {
  float a[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) a[j] = seed + (float)(threadIdx.x + j);
  const float m = 1.0f - 1e-7f * seed, c = 1e-3f;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u)
#pragma unroll
      for (int j = 0; j < 8; ++j) a[j] = fmaf(a[j], m, c);
  }
  float s = 0.0f;
#pragma unroll
  for (int j = 0; j < 8; ++j) s += a[j];
  if (s == 12345.678f) out[0] = s;                   // keeps the chains alive
}

extern "C" int tred_bench_fma(tred_ctx* ctx, int32_t iters, float* d_out, double* h_flops, void* stream) {
  if (!ctx || iters < 1 || !d_out) return TRED_EINVAL;
  TRED_CHECK_DEVICE(ctx);
  const int blocks = ctx->num_sms * 8;
  k_bench_fma<<<blocks, 256, 0, (cudaStream_t)stream>>>(iters, 1.0f, d_out);
  TRED_COUNT_LAUNCH(1);
  TRED_LAUNCH_CHECK("k_bench_fma");
  if (h_flops) *h_flops = 2.0 * 64.0 * (double)iters * 256.0 * (double)blocks;
  return TRED_OK;
}

extern "C" int tred_stage_count(void) { return ST_COUNT; }

extern "C" const char* tred_stage_name(int s) {
  static const char* names[ST_COUNT] = {"drift", "pairs", "sort", "rle", "effq", "plan", "resp_dft",
                                        "fft_fwd", "conv_misc", "mac", "accum", "ifft", "gather"};
  return (s >= 0 && s < ST_COUNT) ? names[s] : "?";
}
extern "C" int tred_abi_version(void) { return 2; }
extern "C" int tred_last_mac_mode(const tred_ctx* c) { return c ? c->last_mac_mode : TRED_EINVAL; }

extern "C" const char* tred_strerror(int s) {
  switch (s) {
    case TRED_OK: return "ok";
    case TRED_EINVAL: return "invalid argument or configuration";
    case TRED_ECAP: return "capacity or workspace too small";
    case TRED_ECUDA: return "CUDA error (see tred_last_cuda_error)";
    case TRED_EUNSUPPORTED: return "configuration not supported by the kernels";
    default: return "unknown status";
  }
}

// ------------------------------------------------------------------ dims / context
static bool is_pow2(int x) { return x > 0 && (x & (x - 1)) == 0; }

extern "C" int tred_get_dims(const tred_config* c, tred_dims* d) {
  if (!c || !d) return TRED_EINVAL;
  if (c->npix_x <= 0 || c->npix_y <= 0 || c->sub <= 0 || c->nticks <= 0) return TRED_EINVAL;
  if (c->gl_n < 1 || c->gl_n > 4) return TRED_EINVAL;
  if (c->resp_half < 0 || c->resp_nticks <= 0) return TRED_EINVAL;
  if (c->effq_mode < 0 || c->effq_mode > 1 || c->mac_mode < 0 || c->mac_mode > 7) return TRED_EINVAL;
  if (c->fft_mode < 0 || c->fft_mode > 1) return TRED_EINVAL;
  if (!(c->pitch_mm > 0) || !(c->tick_us > 0) || !(c->v_mm_us > 0) || !(c->lifetime_us > 0))
    return TRED_EINVAL;
  if (!(c->nsigma > 0) || !(c->sigma_min_xy_mm > 0) || !(c->sigma_min_t_us > 0)) return TRED_EINVAL;
  for (int a = 0; a < 3; ++a)
    if (!is_pow2(c->block[a])) return TRED_EUNSUPPORTED;
  d->NG[0] = (int64_t)c->sub * c->npix_x;
  d->NG[1] = (int64_t)c->sub * c->npix_y;
  d->NG[2] = c->nticks;
  for (int a = 0; a < 3; ++a) d->NB[a] = (d->NG[a] + c->block[a] - 1) / c->block[a];
  if (d->NB[0] * d->NB[1] * d->NB[2] >= (1ll << 31)) return TRED_EUNSUPPORTED;
  if ((int64_t)c->npix_x * c->npix_y * d->NB[2] >= (1ll << 31)) return TRED_EUNSUPPORTED;
  d->out_len = c->block[2] + c->resp_nticks - 1;
  // Padding: any L >= Bt + Tr - 1 gives the linear convolution (PAPER.md:L264 pads to a
  // power of two; reading G20).  L = smallest 2^a 3^b >= out_len with a >= 3: fewer
  // frequencies for the spectrum multiply-accumulate, still short radix-{8,4,2,3} FFTs.
  int L = 0;
  for (int p3 = 1; p3 <= 8192; p3 *= 3)
    for (int p2 = 8; p2 * p3 <= 8192; p2 *= 2) {
      const int cand = p2 * p3;
      if (cand >= d->out_len && cand >= 64 && (L == 0 || cand < L)) L = cand;
    }
  if (L == 0 || L > 4096) return TRED_EUNSUPPORTED;
  d->fft_len = L;
  d->n_over = (d->out_len + c->block[2] - 1) / c->block[2];
  d->n_freq = L / 2;
  d->n_phase = c->sub * c->sub;
  const int K = 2 * c->resp_half + 1;
  d->n_off = K * K;
  d->n_off_pad = (d->n_off + 7) / 8 * 8;
  if (d->n_off_pad > 128) return TRED_EUNSUPPORTED;      // MAC tiles hold all offsets
  // pixels spanned by B consecutive fine points starting anywhere in a pixel
  d->pix_per_block = ((c->sub - 1 + c->block[0] - 1) / c->sub + 1) *
                     ((c->sub - 1 + c->block[1] - 1) / c->sub + 1);
  // response spectrum: fp32 [f][phase][off_pad] complex (2 floats) + tf32 hi and lo
  // [f][2 off_pad][2 phase] (4 floats each)
  d->dft_ticks = c->block[2];
  d->rhat_floats = rhat_layout(*d).total;
  d->block_floats = (int64_t)c->block[0] * c->block[1] * c->block[2];
  // per charge pixel in flight: spectra [f][phase] + products [f][off_pad], complex fp32
  d->conv_row_bytes = (int64_t)d->n_freq * (d->n_phase + d->n_off_pad) * 8;
  return TRED_OK;
}

extern "C" int tred_create(const tred_config* cfg, tred_ctx** out) {
  if (!cfg || !out) return TRED_EINVAL;
  tred_dims d;
  int rc = tred_get_dims(cfg, &d);
  if (rc != TRED_OK) return rc;
  int ndev = 0;
  cudaError_t e = cudaGetDeviceCount(&ndev);
  if (e != cudaSuccess || ndev == 0) {     // no CPU fallback: fail loudly
    tred_set_cuda_error(e != cudaSuccess ? e : cudaErrorNoDevice, "tred_create");
    return TRED_ECUDA;
  }
  int dev = 0;
  TRED_CUDA(cudaGetDevice(&dev));
  tred_ctx* c = (tred_ctx*)calloc(1, sizeof(tred_ctx));
  if (!c) return TRED_EINVAL;
  c->cfg = *cfg;
  c->dims = d;
  TRED_CUDA(cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev));
  TRED_CUDA(cudaDeviceGetAttribute(&c->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
  TRED_CUDA(cudaDeviceGetAttribute(&c->smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev));
  c->device = dev;
  rc = tred_effq_init_tables();
  if (rc != TRED_OK) { free(c); return rc; }
  *out = c;
  return TRED_OK;
}

extern "C" void tred_destroy(tred_ctx* c) {
  if (!c) return;
  prof_clear(c);
  free(c->recs);
  if (c->h_counts) cudaFreeHost(c->h_counts);
  free(c);
}

// ------------------------------------------------------------------ S1 drift
struct DriftParams {
  double v, two_v, two_DT, two_DL, tau, smin_xy, smin_t, nsig, pthr;
  double org[3], h[3];
  int NG[3], B[3];
  int e;   // grid-point halo of the footprint: 1 if gl_n > 1
};

__device__ __forceinline__ int clamp_floor_i32(double x) {
  x = floor(x);
  x = fmin(fmax(x, -1073741824.0), 1073741824.0);
  return (int)x;
}

// One thread per segment.  Index path (everything that decides an integer) in fp64 with
// explicit round-to-nearest intrinsics so that nvcc cannot contract a*b+c into an FMA:
// same operations, same order as DESIGN.md "index path" (reading G14).
__global__ void __launch_bounds__(256)
k_drift(int64_t nseg, const float* __restrict__ seg, float* __restrict__ augf,
        int32_t* __restrict__ augi, unsigned long long* __restrict__ npairs, DriftParams P) {
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  unsigned long long mypairs = 0;
  if (s < nseg) {
    const double x0 = seg[0 * nseg + s], y0 = seg[1 * nseg + s], z0 = seg[2 * nseg + s];
    const double x1 = seg[3 * nseg + s], y1 = seg[4 * nseg + s], z1 = seg[5 * nseg + s];
    const double q = seg[6 * nseg + s], t0 = seg[7 * nseg + s];
    const double ta0 = __dadd_rn(t0, __ddiv_rn(z0, P.v));
    const double ta1 = __dadd_rn(t0, __ddiv_rn(z1, P.v));
    const double tm = __ddiv_rn(__dadd_rn(z0, z1), P.two_v);
    const double tmc = fmax(tm, 0.0);
    const double sxy = fmax(__dsqrt_rn(__dmul_rn(P.two_DT, tmc)), P.smin_xy);
    const double st = fmax(__ddiv_rn(__dsqrt_rn(__dmul_rn(P.two_DL, tmc)), P.v), P.smin_t);
    const double Qp = q * exp(-tm / P.tau);
    const int flag = (fabs(__dsub_rn(x1, x0)) < __dmul_rn(P.pthr, sxy)) &&
                     (fabs(__dsub_rn(y1, y0)) < __dmul_rn(P.pthr, sxy)) &&
                     (fabs(__dsub_rn(ta1, ta0)) < __dmul_rn(P.pthr, st));
    const double a0[3] = {x0, y0, ta0}, a1[3] = {x1, y1, ta1};
    const double sg[3] = {sxy, sxy, st};
    int lo[3], hi[3];
    long long np = 1;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const double m = __dmul_rn(P.nsig, sg[a]);
      lo[a] = clamp_floor_i32(__ddiv_rn(__dsub_rn(__dsub_rn(fmin(a0[a], a1[a]), m), P.org[a]), P.h[a]));
      hi[a] = clamp_floor_i32(__ddiv_rn(__dsub_rn(__dadd_rn(fmax(a0[a], a1[a]), m), P.org[a]), P.h[a]));
      const int flo = max(lo[a] - P.e, 0), fhi = min(hi[a] + P.e, P.NG[a] - 1);
      np = (flo <= fhi && np > 0) ? np * (fhi / P.B[a] - flo / P.B[a] + 1) : 0;
      // segment ends and sigma in grid units, relative to the bbox corner (fp64 -> fp32)
      augf[(0 + a) * nseg + s] = (float)((a0[a] - P.org[a]) / P.h[a] - (double)lo[a]);
      augf[(3 + a) * nseg + s] = (float)((a1[a] - P.org[a]) / P.h[a] - (double)lo[a]);
      augf[(6 + a) * nseg + s] = (float)(sg[a] / P.h[a]);
      augi[(0 + a) * nseg + s] = lo[a];
      augi[(3 + a) * nseg + s] = hi[a];
    }
    augf[9 * nseg + s] = (float)Qp;
    augi[6 * nseg + s] = flag;
    augi[7 * nseg + s] = (int)np;
    mypairs = (unsigned long long)np;
  }
  // CTA reduction of the pair count (integer: order-independent)
  __shared__ unsigned long long wsum[8];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mypairs += __shfl_down_sync(0xffffffffu, mypairs, o);
  if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = mypairs;
  __syncthreads();
  if (threadIdx.x == 0) {
    unsigned long long t = 0;
    for (int w = 0; w < 8; ++w) t += wsum[w];
    if (t) atomicAdd(npairs, t);
  }
}

static DriftParams make_drift_params(const tred_ctx* c) {
  DriftParams P;
  const tred_config& f = c->cfg;
  P.v = f.v_mm_us; P.two_v = 2.0 * f.v_mm_us;
  P.two_DT = 2.0 * f.DT_mm2_us; P.two_DL = 2.0 * f.DL_mm2_us;
  P.tau = f.lifetime_us; P.smin_xy = f.sigma_min_xy_mm; P.smin_t = f.sigma_min_t_us;
  P.nsig = f.nsigma; P.pthr = f.point_thresh;
  P.org[0] = f.origin_x_mm; P.org[1] = f.origin_y_mm; P.org[2] = f.t_origin_us;
  P.h[0] = P.h[1] = f.pitch_mm / (double)f.sub; P.h[2] = f.tick_us;
  for (int a = 0; a < 3; ++a) { P.NG[a] = (int)c->dims.NG[a]; P.B[a] = f.block[a]; }
  P.e = f.gl_n > 1 ? 1 : 0;
  return P;
}

extern "C" int tred_drift(tred_ctx* ctx, int64_t nseg, const float* d_seg, float* d_augf,
                          int32_t* d_augi, int64_t* d_npairs, void* stream) {
  if (!ctx || nseg < 0 || !d_npairs) return TRED_EINVAL;
  TRED_CHECK_DEVICE(ctx);
  cudaStream_t st = (cudaStream_t)stream;
  TRED_CUDA(cudaMemsetAsync(d_npairs, 0, sizeof(int64_t), st));
  if (nseg == 0) return TRED_OK;
  if (!d_seg || !d_augf || !d_augi) return TRED_EINVAL;
  {
    TredProfScope ps(ctx, ST_DRIFT, st);
    k_drift<<<cdiv(nseg, 256), 256, 0, st>>>(nseg, d_seg, d_augf, d_augi,
                                            (unsigned long long*)d_npairs, make_drift_params(ctx));
    TRED_COUNT_LAUNCH(1);
  }
  TRED_LAUNCH_CHECK("k_drift");
  return TRED_OK;
}

// ------------------------------------------------------------------ S3 block binning
__global__ void __launch_bounds__(256)
k_pair_expand(int64_t nseg, const int32_t* __restrict__ augi, const int32_t* __restrict__ pair_off,
              int64_t cap_pairs, uint32_t* __restrict__ keys, int32_t* __restrict__ vals, TredGrid g) {
  const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (s >= nseg) return;
  const int np = augi[7 * nseg + s];
  if (np == 0) return;
  const int e = g.gl_n > 1 ? 1 : 0;
  const int NG[3] = {g.NGx, g.NGy, g.NGt}, B[3] = {g.Bx, g.By, g.Bt};
  int blo[3], bhi[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    blo[a] = max(augi[a * nseg + s] - e, 0) / B[a];
    bhi[a] = min(augi[(3 + a) * nseg + s] + e, NG[a] - 1) / B[a];
  }
  int64_t o = pair_off[s];
  for (int bt = blo[2]; bt <= bhi[2]; ++bt)
    for (int bx = blo[0]; bx <= bhi[0]; ++bx)
      for (int by = blo[1]; by <= bhi[1]; ++by, ++o)
        if (o >= 0 && o < cap_pairs) {
          keys[o] = (uint32_t)((bt * g.NBx + bx) * g.NBy + by);
          vals[o] = (int32_t)s;
        }
}

__global__ void __launch_bounds__(256)
k_rle_flags(const uint32_t* __restrict__ keys, int64_t cap, const int64_t* __restrict__ d_n,
            int32_t* __restrict__ flags) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= cap) return;
  const int64_t n = min((int64_t)*d_n, cap);
  flags[i] = (i < n && (i == 0 || keys[i] != keys[i - 1])) ? 1 : 0;
}

__global__ void __launch_bounds__(256)
k_rle_write(const uint32_t* __restrict__ keys, const int32_t* __restrict__ pos, int64_t cap,
            const int64_t* __restrict__ d_n, const int64_t* __restrict__ d_nblk, int64_t cap_blocks,
            int64_t* __restrict__ out_keys, int32_t* __restrict__ blk_off,
            int32_t* __restrict__ slab_off, TredGrid g) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  const int64_t n = min((int64_t)*d_n, cap);
  const int64_t nblk = *d_nblk;
  if (i == 0) {
    if (nblk <= cap_blocks) blk_off[nblk] = (int32_t)n;
    if (n == 0) for (int b = 0; b <= g.NBt; ++b) slab_off[b] = 0;
  }
  if (i >= n) return;
  const uint32_t k = keys[i];
  const bool first = (i == 0) || (keys[i - 1] != k);
  if (!first) return;
  const int p = pos[i];
  if (p < cap_blocks) { out_keys[p] = (int64_t)k; blk_off[p] = (int32_t)i; }
  const int plane = g.NBx * g.NBy;
  const int bt = (int)(k / (uint32_t)plane);
  const int bt_prev = (i == 0) ? -1 : (int)(keys[i - 1] / (uint32_t)plane);
  for (int b = bt_prev + 1; b <= bt; ++b) slab_off[b] = p;
  if (p == nblk - 1) for (int b = bt + 1; b <= g.NBt; ++b) slab_off[b] = (int32_t)nblk;
}

struct BinWork {
  int64_t* cnt;   // [0] pair count, [1] block count
  int32_t* pair_off; uint32_t *ka, *kb; int32_t* vb; int32_t* flags; void* scan; void* sort;
  size_t total;
};

static BinWork carve_bin_work(void* base, int64_t nseg, int64_t cap_pairs) {
  BinWork w;
  size_t o = 0;
  char* b = (char*)base;
  auto take = [&](size_t bytes) { void* p = b ? b + o : nullptr; o += align_up(bytes, 256); return p; };
  int64_t cp = cap_pairs > 0 ? cap_pairs : 1, ns = nseg > 0 ? nseg : 1;
  w.cnt = (int64_t*)take(2 * sizeof(int64_t));
  w.pair_off = (int32_t*)take(ns * 4);
  w.ka = (uint32_t*)take(cp * 4);
  w.kb = (uint32_t*)take(cp * 4);
  w.vb = (int32_t*)take(cp * 4);
  w.flags = (int32_t*)take(cp * 4);
  w.scan = take(tred_scan_work_bytes(ns > cp ? ns : cp));
  w.sort = take(tred_sort_work_bytes(cp));
  w.total = o;
  return w;
}

extern "C" size_t tred_blockbin_work_bytes(const tred_ctx* ctx, int64_t nseg, int64_t cap_pairs) {
  (void)ctx;
  return carve_bin_work(nullptr, nseg, cap_pairs).total;
}

extern "C" int tred_blockbin(tred_ctx* ctx, int64_t nseg, const int32_t* d_augi,
                             int64_t cap_pairs, int64_t cap_blocks,
                             int64_t* d_keys, int32_t* d_blk_off, int32_t* d_pair_seg,
                             int32_t* d_slab_off, int64_t* d_nblocks,
                             void* d_work, size_t work_bytes, void* stream) {
  if (!ctx || nseg < 0 || cap_pairs < 0 || cap_blocks < 0 || !d_nblocks || !d_slab_off) return TRED_EINVAL;
  TRED_CHECK_DEVICE(ctx);
  if (cap_pairs >= (1ll << 31) || nseg >= (1ll << 31)) return TRED_EUNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  const TredGrid g = make_grid(ctx);
  BinWork w = carve_bin_work(d_work, nseg, cap_pairs);
  if (!d_work || work_bytes < w.total) return TRED_ECAP;
  if (nseg == 0 || cap_pairs == 0) {
    TRED_CUDA(cudaMemsetAsync(d_nblocks, 0, sizeof(int64_t), st));
    TRED_CUDA(cudaMemsetAsync(d_slab_off, 0, sizeof(int32_t) * (g.NBt + 1), st));
    if (d_blk_off) TRED_CUDA(cudaMemsetAsync(d_blk_off, 0, sizeof(int32_t), st));
    return TRED_OK;
  }
  if (!d_augi || !d_keys || !d_blk_off || !d_pair_seg) return TRED_EINVAL;
  int64_t* d_np = w.cnt;         // device-side pair count
  int64_t* d_nb = w.cnt + 1;     // device-side block count
  // pair offsets = exclusive scan of the per-segment pair counts
  int rc;
  {
    TredProfScope ps(ctx, ST_PAIRS, st);
    rc = tred_exclusive_scan_i32(d_augi + 7 * nseg, w.pair_off, nseg, d_np, w.scan, st);
  }
  if (rc != TRED_OK) return rc;
  int total_bits = 1;
  while ((1ll << total_bits) < (int64_t)g.NBx * g.NBy * g.NBt) ++total_bits;
  const int passes = (total_bits + 7) / 8;
  // choose the value buffers so that the last pass lands in d_pair_seg
  uint32_t* ka = w.ka; uint32_t* kb = w.kb;
  int32_t* va = (passes % 2 == 0) ? d_pair_seg : w.vb;
  int32_t* vb = (passes % 2 == 0) ? w.vb : d_pair_seg;
  {
    TredProfScope ps(ctx, ST_PAIRS, st);
    k_pair_expand<<<cdiv(nseg, 256), 256, 0, st>>>(nseg, d_augi, w.pair_off, cap_pairs, ka, va, g);
    TRED_COUNT_LAUNCH(1);
  }
  TRED_LAUNCH_CHECK("k_pair_expand");
  uint32_t* ks; int32_t* vs;
  {
    TredProfScope ps(ctx, ST_SORT, st);
    rc = tred_radix_sort_pairs(ka, va, kb, vb, cap_pairs, d_np, passes * 8, w.sort, st, &ks, &vs);
  }
  if (rc != TRED_OK) return rc;
  if (vs != d_pair_seg) return TRED_EINVAL;   // cannot happen
  // run-length compaction of the sorted keys
  {
    TredProfScope ps(ctx, ST_RLE, st);
    k_rle_flags<<<cdiv(cap_pairs, 256), 256, 0, st>>>(ks, cap_pairs, d_np, w.flags);
    TRED_COUNT_LAUNCH(1);
    rc = tred_exclusive_scan_i32(w.flags, w.flags, cap_pairs, d_nb, w.scan, st);
    if (rc != TRED_OK) return rc;
    k_rle_write<<<cdiv(cap_pairs, 256), 256, 0, st>>>(ks, w.flags, cap_pairs, d_np, d_nb,
                                                     cap_blocks, d_keys, d_blk_off, d_slab_off, g);
    TRED_COUNT_LAUNCH(1);
  }
  TRED_LAUNCH_CHECK("k_rle_write");
  TRED_CUDA(cudaMemcpyAsync(d_nblocks, d_nb, sizeof(int64_t), cudaMemcpyDeviceToDevice, st));
  return TRED_OK;
}
