// tred_steps_static -- tred_steps (G4Step splitting + recombination; readings
// G21, G22 of DESIGN.md) for callers that have no device memory to give as a workspace and are
// not in a position to ask the CUDA runtime for any.
//
// Who that is.  tred_steps runs first, on the raw GEANT4 steps, usually in the I/O stage that
// feeds the simulation rather than inside it.  Such a stage often owns no workspace at all:
//   * a reader thread of a framework whose device memory was handed out in full at start-up to
//     a pool it does not control (asking the runtime for more fails, or evicts someone else);
//   * a thread that runs while ANOTHER thread of the process records a CUDA graph in the
//     default (global) capture mode: cudaMalloc / cudaFree from any thread are then illegal
//     and break the other thread's capture;
//   * a latency-bound event loop, for which cudaMalloc / cudaFree are device-wide
//     synchronisations it cannot afford per event.
// For them the two scratch arrays of tred_steps (first segment of every step, block sums of the
// scan) live in a file-scope __device__ array of fixed size below.  The price: every GPU on which
// the library is loaded holds TRED_STEPS_STATIC_BYTES (about 4 MiB) until the process exits, one
// call handles at most TRED_STEPS_STATIC_MAX steps, and all calls on a device share the array.
//
// The arithmetic is that of tred_steps.cu, operation for operation (fp64, explicit
// round-to-nearest, fixed order): both entry points return the same bits.  The kernels are
// repeated here, not shared, so that the existing entry point is left exactly as it was.
#include <math.h>
#include <mutex>
#include "tred_common.cuh"

// The header's number and the array below must agree.
static_assert(TRED_STEPS_STATIC_MAX == (1 << 20), "tred.h: TRED_STEPS_STATIC_MAX");

static constexpr size_t FIRST_BYTES = ((size_t)(TRED_STEPS_STATIC_MAX + 1) * 4 + 255) / 256 * 256;
// block sums of the scan over TRED_STEPS_STATIC_MAX + 1 counts: 4096 counts per CTA
// (tred_scan_sort.cu) -> 257 int32, rounded up generously; checked against
// tred_scan_work_bytes at set-up.
static constexpr size_t SCAN_BYTES = 2048;
static_assert(FIRST_BYTES + SCAN_BYTES == TRED_STEPS_STATIC_BYTES, "tred.h: TRED_STEPS_STATIC_BYTES");

// In host code this name is only a handle for cudaGetSymbolAddress, never a pointer to pass to
// a kernel: the address the GPU knows the array by differs per device and is looked up below.
static __device__ __align__(256) unsigned char g_steps_scratch[TRED_STEPS_STATIC_BYTES];

namespace {

constexpr int MAX_DEVICES = 64;
std::mutex g_setup_mutex;
void* g_scratch_addr[MAX_DEVICES];     // device address of g_steps_scratch on device d (null: not looked up yet)

// Once per device, with that device current: the device address of the scratch array.
int scratch_address(void** out) {
  int dev = -1;
  TRED_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) return TRED_EUNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_setup_mutex);
  if (!g_scratch_addr[dev]) {
    if (tred_scan_work_bytes((int64_t)TRED_STEPS_STATIC_MAX + 1) > SCAN_BYTES) return TRED_EUNSUPPORTED;
    void* p = nullptr;
    TRED_CUDA(cudaGetSymbolAddress(&p, g_steps_scratch));
    if (!p) return TRED_ECUDA;
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return TRED_OK;
}

__device__ __forceinline__ double step_length(const float* __restrict__ st, int64_t n, int64_t i, double d[3]) {
  for (int a = 0; a < 3; ++a) d[a] = __dsub_rn((double)st[(3 + a) * n + i], (double)st[a * n + i]);
  return __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2])));
}

// pieces per step; entry nstep is the 0 that makes the exclusive scan end in the total
__global__ void __launch_bounds__(256)
k_sst_count(int64_t nstep, const float* __restrict__ st, double max_len, int32_t* __restrict__ cnt) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i > nstep) return;
  int c = 0;
  if (i < nstep) {
    double d[3];
    const double len = step_length(st, nstep, i, d);
    const double q = ceil(__ddiv_rn(len, max_len));
    c = q > 1.0 ? (int)q : 1;
  }
  cnt[i] = c;
}

__device__ __forceinline__ double recomb(const tred_steps_config& c, double dedx) {
  const double rhoE = __dmul_rn(c.density_g_cm3, c.efield_kv_cm);
  if (c.recomb_model == 0) return c.birks_A / (1.0 + c.birks_k / rhoE * dedx);
  const double x = c.box_beta / rhoE * dedx;
  if (!(x > 0.0)) return 0.0;
  const double r = log(c.box_alpha + x) / x;
  return r < 0.0 ? 0.0 : r > 1.0 ? 1.0 : r;
}

__global__ void __launch_bounds__(256)
k_sst_fill(int64_t nstep, const float* __restrict__ st, const int32_t* __restrict__ first, tred_steps_config c,
           int64_t cap, float* __restrict__ seg, int32_t* __restrict__ parent, int64_t* __restrict__ d_nseg) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) *d_nseg = first[nstep];
  if (i >= nstep) return;
  double d[3], p0[3];
  const double len = step_length(st, nstep, i, d);
  for (int a = 0; a < 3; ++a) p0[a] = (double)st[a * nstep + i];
  const int f0 = first[i], n = first[i + 1] - f0;
  const double dE = (double)st[6 * nstep + i];
  const double dedx = len > 0.0 ? dE / len * 10.0 : 0.0;                  // MeV/cm
  const double ne = dE * 1.0e6 / c.w_ion_ev * recomb(c, dedx);
  const double dn = (double)n;
  const float q = (float)(ne / dn), t0 = st[7 * nstep + i];
  for (int k = 0; k < n; ++k) {
    const int64_t j = (int64_t)f0 + k;
    if (j >= cap) break;
    const double fa = __ddiv_rn((double)k, dn), fb = __ddiv_rn((double)(k + 1), dn);
    for (int a = 0; a < 3; ++a) {
      seg[a * cap + j] = (float)__dadd_rn(p0[a], __dmul_rn(d[a], fa));
      seg[(3 + a) * cap + j] = (float)__dadd_rn(p0[a], __dmul_rn(d[a], fb));
    }
    seg[6 * cap + j] = q;
    seg[7 * cap + j] = t0;
    parent[j] = (int32_t)i;
  }
}

}  // namespace

extern "C" int64_t tred_steps_static_max(void) { return TRED_STEPS_STATIC_MAX; }

extern "C" int tred_steps_static(const tred_steps_config* cfg, int64_t nstep, const float* d_step, int64_t cap_seg,
                                 float* d_seg, int32_t* d_parent, int64_t* d_nseg, void* stream) {
  if (!cfg || nstep < 0 || cap_seg < 0 || !d_nseg) return TRED_EINVAL;
  if (!(cfg->max_len_mm > 0) || !(cfg->w_ion_ev > 0) || !(cfg->density_g_cm3 > 0) || !(cfg->efield_kv_cm > 0) ||
      cfg->recomb_model < 0 || cfg->recomb_model > 1)
    return TRED_EINVAL;
  // more steps than the fixed array holds: refused before anything is enqueued (split the batch)
  if (nstep > TRED_STEPS_STATIC_MAX) return TRED_ECAP;
  cudaStream_t st = (cudaStream_t)stream;
  if (nstep == 0) { TRED_CUDA(cudaMemsetAsync(d_nseg, 0, sizeof(int64_t), st)); return TRED_OK; }
  if (!d_step) return TRED_EINVAL;
  if (cap_seg > 0 && (!d_seg || !d_parent)) return TRED_EINVAL;
  void* scratch = nullptr;
  int rc = scratch_address(&scratch);        // first call on this device: cudaGetSymbolAddress
  if (rc != TRED_OK) return rc;
  // Nothing in the scratch has to start at zero: entries [0, nstep] of `first` and the
  // ceil((nstep + 1) / 4096) block sums are all written by this call before they are read;
  // what an earlier call left beyond them is never looked at.
  int32_t* first = (int32_t*)scratch;
  void* scan = (char*)scratch + FIRST_BYTES;
  k_sst_count<<<cdiv(nstep + 1, 256), 256, 0, st>>>(nstep, d_step, cfg->max_len_mm, first);
  rc = tred_exclusive_scan_i32(first, first, nstep + 1, nullptr, scan, st);
  if (rc != TRED_OK) return rc;
  k_sst_fill<<<cdiv(nstep, 256), 256, 0, st>>>(nstep, d_step, first, *cfg, cap_seg, d_seg, d_parent, d_nseg);
  TRED_COUNT_LAUNCH(2);
  TRED_LAUNCH_CHECK("tred_steps_static");
  return TRED_OK;
}
