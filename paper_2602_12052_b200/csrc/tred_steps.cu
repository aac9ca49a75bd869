// N2: G4Step preprocessing -- PAPER.md:L57 (steps longer than a
// threshold are divided into step-segments that keep dE/dx) and PAPER.md:L41,L57 (ionisation
// electrons that survive recombination).  Readings G21, G22 of DESIGN.md.
//   pass 1  pieces per step n = max(1, ceil(len / max_len)), len in fp64 with explicit
//           round-to-nearest operations in a fixed order (bit-exact counts)
//   scan    first segment of every step
//   pass 2  one thread per step writes its n equal pieces: ends p0 + d k/n, charge N_e / n
#include <math.h>
#include "tred_common.cuh"

namespace {

__device__ __forceinline__ double step_length(const float* __restrict__ st, int64_t n, int64_t i, double d[3]) {
  for (int a = 0; a < 3; ++a) d[a] = __dsub_rn((double)st[(3 + a) * n + i], (double)st[a * n + i]);
  return __dsqrt_rn(__dadd_rn(__dadd_rn(__dmul_rn(d[0], d[0]), __dmul_rn(d[1], d[1])), __dmul_rn(d[2], d[2])));
}

__global__ void __launch_bounds__(256)
k_steps_count(int64_t nstep, const float* __restrict__ st, double max_len, int32_t* __restrict__ cnt) {
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
k_steps_fill(int64_t nstep, const float* __restrict__ st, const int32_t* __restrict__ first, tred_steps_config c,
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

extern "C" size_t tred_steps_work_bytes(int64_t nstep) {
  if (nstep < 0) return 0;
  return align_up((size_t)(nstep + 1) * 4, 256) + tred_scan_work_bytes(nstep + 1);
}

extern "C" int tred_steps(const tred_steps_config* cfg, int64_t nstep, const float* d_step, int64_t cap_seg,
                          float* d_seg, int32_t* d_parent, int64_t* d_nseg, void* d_work, size_t work_bytes,
                          void* stream) {
  if (!cfg || nstep < 0 || cap_seg < 0 || !d_nseg) return TRED_EINVAL;
  if (!(cfg->max_len_mm > 0) || !(cfg->w_ion_ev > 0) || !(cfg->density_g_cm3 > 0) || !(cfg->efield_kv_cm > 0) ||
      cfg->recomb_model < 0 || cfg->recomb_model > 1)
    return TRED_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  if (nstep == 0) { TRED_CUDA(cudaMemsetAsync(d_nseg, 0, sizeof(int64_t), st)); return TRED_OK; }
  if (nstep >= (1ll << 31) - 1) return TRED_EUNSUPPORTED;
  if (!d_step || !d_work || work_bytes < tred_steps_work_bytes(nstep)) return d_work ? TRED_ECAP : TRED_EINVAL;
  if (cap_seg > 0 && (!d_seg || !d_parent)) return TRED_EINVAL;
  int32_t* first = (int32_t*)d_work;
  void* scan = (char*)d_work + align_up((size_t)(nstep + 1) * 4, 256);
  k_steps_count<<<cdiv(nstep + 1, 256), 256, 0, st>>>(nstep, d_step, cfg->max_len_mm, first);
  int rc = tred_exclusive_scan_i32(first, first, nstep + 1, nullptr, scan, st);
  if (rc != TRED_OK) return rc;
  k_steps_fill<<<cdiv(nstep, 256), 256, 0, st>>>(nstep, d_step, first, *cfg, cap_seg, d_seg, d_parent, d_nseg);
  TRED_COUNT_LAUNCH(2);
  TRED_LAUNCH_CHECK("tred_steps");
  return TRED_OK;
}
