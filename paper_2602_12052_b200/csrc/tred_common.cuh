// Internal definitions shared by the translation units of libtred (CUDA path only).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stdio.h>
#include "../../include/tred.h"

enum TredStage {
  ST_DRIFT = 0, ST_PAIRS, ST_SORT, ST_RLE, ST_EFFQ, ST_PLAN, ST_RESP, ST_FFT_FWD, ST_MISC, ST_MAC,
  ST_ACCUM, ST_IFFT, ST_GATHER, ST_COUNT
};

struct TredProfRec { int stage; cudaEvent_t a, b; };

struct tred_ctx {
  tred_config cfg;
  tred_dims   dims;
  int         num_sms;
  int         smem_optin;     // max dynamic shared memory per block (bytes)
  int         smem_sm;        // shared memory per SM (bytes)
  int         device;         // CUDA device the context was created on
  const void* sym_rhat;       // last d_rhat prepared from a mirror-symmetric response (or NULL)
  int         last_mac_mode;  // spectrum-product kernel the last tred_convolve launched (tred_last_mac_mode)
  int64_t     hint_pairs;     // tred_simulate: (segment, block) pairs of the previous event (0: none yet)
  int64_t*    h_counts;       // tred_simulate: pinned host mirror of the device-side counts
  // stage profiling (tred_profile_begin / tred_profile_end)
  int         prof_on;
  int64_t     launches[ST_COUNT];
  TredProfRec* recs;
  int         nrecs, cap_recs;
};

// Kernel-launch counter (per host thread); every <<<>>> site calls TRED_COUNT_LAUNCH.
extern thread_local int64_t g_tred_launches;
#define TRED_COUNT_LAUNCH(n) (g_tred_launches += (n))

// Brackets the launches of one stage: counts them and, when profiling is on, records a
// pair of CUDA events on the stream the kernels are launched on.
struct TredProfScope {
  tred_ctx* c; int stage; cudaStream_t st; int64_t l0; int rec;
  TredProfScope(tred_ctx* ctx, int stage_, cudaStream_t st_);
  ~TredProfScope();
};

// Grid constants passed by value to kernels.
struct TredGrid {
  int NGx, NGy, NGt;
  int Bx, By, Bt;
  int NBx, NBy, NBt;
  int S, H, Tr;
  int npx, npy, nticks;
  int L;            // fft length
  int nf;           // L/2 spectrum slots
  int nph;          // S*S phases
  int noff, kp;     // (2H+1)^2 offsets, padded to a multiple of 8
  int nover;        // tiles per output
  int gl_n;
};

static inline TredGrid make_grid(const tred_ctx* c) {
  TredGrid g;
  g.NGx = (int)c->dims.NG[0]; g.NGy = (int)c->dims.NG[1]; g.NGt = (int)c->dims.NG[2];
  g.Bx = c->cfg.block[0]; g.By = c->cfg.block[1]; g.Bt = c->cfg.block[2];
  g.NBx = (int)c->dims.NB[0]; g.NBy = (int)c->dims.NB[1]; g.NBt = (int)c->dims.NB[2];
  g.S = c->cfg.sub; g.H = c->cfg.resp_half; g.Tr = c->cfg.resp_nticks;
  g.npx = c->cfg.npix_x; g.npy = c->cfg.npix_y; g.nticks = c->cfg.nticks;
  g.L = c->dims.fft_len; g.nf = c->dims.n_freq; g.nph = c->dims.n_phase;
  g.noff = c->dims.n_off; g.kp = c->dims.n_off_pad;
  g.nover = c->dims.n_over; g.gl_n = c->cfg.gl_n;
  return g;
}

void tred_set_cuda_error(cudaError_t e, const char* where);

#define TRED_CUDA(call)                                                    \
  do {                                                                     \
    cudaError_t _e = (call);                                               \
    if (_e != cudaSuccess) { tred_set_cuda_error(_e, #call); return TRED_ECUDA; } \
  } while (0)

// A context belongs to the device it was created on (its kernel attributes, SM count and
// shared-memory limits are that device's): calls made with another device current are refused.
#define TRED_CHECK_DEVICE(ctx)                                             \
  do {                                                                     \
    int _dev = -1;                                                         \
    if (cudaGetDevice(&_dev) != cudaSuccess || _dev != (ctx)->device) return TRED_EINVAL; \
  } while (0)

#define TRED_LAUNCH_CHECK(name)                                            \
  do {                                                                     \
    cudaError_t _e = cudaGetLastError();                                   \
    if (_e != cudaSuccess) { tred_set_cuda_error(_e, name); return TRED_ECUDA; } \
  } while (0)

static inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
static inline int cdiv(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// ---- layout of the response-spectrum buffer d_rhat (tred_prepare_response) ---------------
// [W: fp32 complex [f][phase][kp]] [B_hi][B_lo: [f][2 kp][2 nph] tf32 parts]
// [Bs_hi][Bs_lo][Bd_hi][Bd_lo: [f][SYM_N][nph] mirror-symmetric halves, see tred_conv.cu] [flag]
// [B_hi, B_lo rounded to bf16, same shape as B_hi: operands of the bf16 correction products]
// [B16: [f][2 kp][h16_kp] fp16, hi / lo parts of B / bscale[f] in blocks of 16 reals (tred_mac_h3.cu)]
// [bscale: [f] float, power of two]
// [Wd: [L][2 Bt] fp16 hi / lo DFT matrix of the forward transform (tred_dft_h16.cu)]
constexpr int SYM_N = 128;           // rows of the symmetric matrices: 2 x (noff + 1) / 2 padded
// halves per operand row in the fp16 hi / lo block layout: ceil(2 nph / 16) blocks of (16 hi | 16 lo)
static inline int h16_kp(const tred_dims& d) { return (2 * d.n_phase + 15) / 16 * 32; }
struct RhatLayout { int64_t w, bhi, blo, bs_hi, bs_lo, bd_hi, bd_lo, flag, bhb, blb, b16, bsc, wdft, total; };
static inline RhatLayout rhat_layout(const tred_dims& d) {
  RhatLayout L;
  const int64_t rb = (int64_t)d.n_freq * d.n_phase * d.n_off_pad;
  const int64_t sb = (int64_t)d.n_freq * SYM_N * d.n_phase;
  L.w = 0; L.bhi = 2 * rb; L.blo = 6 * rb;
  L.bs_hi = 10 * rb; L.bs_lo = L.bs_hi + sb; L.bd_hi = L.bs_lo + sb; L.bd_lo = L.bd_hi + sb;
  L.flag = L.bd_lo + sb;
  L.bhb = L.flag + 8;                 // bf16 copies of B_hi and B_lo, [f][2 kp][2 nph] bf16 = 2 rb floats each
  L.blb = L.bhb + 2 * rb;
  L.b16 = L.blb + 2 * rb;              // 16-byte aligned: every term above is a multiple of 8 floats
  L.bsc = L.b16 + (int64_t)d.n_freq * 2 * d.n_off_pad * (h16_kp(d) / 2);
  L.wdft = L.bsc + (d.n_freq + 7) / 8 * 8;     // DFT matrix [L][2 Bt] fp16 (tred_dft_h16.cu): L * Bt floats
  L.total = L.wdft + (int64_t)d.fft_len * d.dft_ticks;
  return L;
}

// ---- row tiles of the tensor-core convolution path (tred_conv.cu, tred_mac_tc.cu) ----
constexpr int RT_SW = 8;         // strip width in pixels
constexpr int RT_ROWS = 128;     // rows per tile = MMA M
constexpr int RT_PY = 64;        // patch height (py) in global memory
constexpr int RT_PYS = 66;       // patch row stride in shared memory (66 = 2 mod 16: conflict-free)
constexpr int RT_MAXH = 5;       // largest response half-width the patch buffers hold
constexpr int RT_PXMAX = RT_SW + 2 * RT_MAXH;


// ---- internal entry points of the convolution plan used by tred_simulate (tred_sim.cu) ----
int tred_convolve_plan_dev(tred_ctx* ctx, int64_t nblocks, const int64_t* d_nblocks, const int64_t* d_keys,
                           int64_t cap_cp, int64_t* d_cp_keys, int32_t* d_cp_off, int64_t* d_ncp,
                           int64_t cap_sp, int64_t* d_sp_keys, int32_t* d_sp_off, int64_t* d_nsp,
                           int64_t cap_tiles, int64_t* d_tile_keys, int64_t* d_ntiles,
                           int32_t* d_rt_off,
                           void* d_plan_work, size_t plan_work_bytes, void* stream);
int tred_plan_tile_offsets(tred_ctx* ctx, const void* d_plan_work, int32_t* d_tile_off, cudaStream_t st);

// ---- S2 variants (tred_effq.cu: closed form; tred_effq_fact.cu: factored, dispatch) ---
int tred_effq_closed_form(tred_ctx* ctx, int64_t nseg, int64_t nblocks,
                          const int64_t* d_keys, const int32_t* d_blk_off, const int32_t* d_pair_seg,
                          const float* d_augf, const int32_t* d_augi,
                          float* d_payload, cudaStream_t st);
// Uploads the Gauss-Legendre tables of the line quadrature (called by tred_create).
int tred_effq_init_tables(void);

// ---- device-wide primitives (tred_scan_sort.cu) ----------------------------------
// Exclusive scan of int32 (n elements) into out (may alias in); writes the total to
// d_total (int64) if non-null.  work: at least tred_scan_work_bytes(n).
size_t tred_scan_work_bytes(int64_t n);
int tred_exclusive_scan_i32(const int32_t* d_in, int32_t* d_out, int64_t n, int64_t* d_total,
                            void* d_work, cudaStream_t st);
// Stable LSD radix sort of (uint32 key, int32 value) pairs on `bits` low key bits.
// n is read on the host (capacity); the count actually sorted is *d_n (device) if
// d_n is non-null (elements beyond it are ignored).  Result ends in keys_out/vals_out.
size_t tred_sort_work_bytes(int64_t n);
int tred_radix_sort_pairs(uint32_t* d_keys_a, int32_t* d_vals_a, uint32_t* d_keys_b, int32_t* d_vals_b,
                          int64_t n_cap, const int64_t* d_n, int bits, void* d_work, cudaStream_t st,
                          uint32_t** keys_out, int32_t** vals_out);
