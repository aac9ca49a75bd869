// N3: trigger-reset pixel readout, PAPER.md:L185, L189 (Fig. 4), noise
// terms PAPER.md:L262; reading G23 of DESIGN.md.  Per channel, tick by tick:
//   WAIT  q += I[t]; the discriminator fires when q >= threshold + d_thr[h];
//   INTEG q += I[t] for n_integ more ticks, then the record (tick, q + d_adc[h]) is written;
//   RESET q = d_base[h], the next n_reset ticks are dead.
// The crossing tick is an integer decided by a floating-point comparison, so the running sum
// is a plain fp32 sum in tick order (one thread per channel; the oracle does the same).
// One warp per 32 channels, four warps per CTA: the rows are staged chunk by chunk in shared
// memory with coalesced loads, then every lane walks its own row.
#include "tred_common.cuh"

namespace {

constexpr int RO_CH = 64;             // ticks per staged chunk
constexpr int RO_WARPS = 4;           // warps (groups of 32 channels) per CTA

__global__ void __launch_bounds__(32 * RO_WARPS)
k_readout(int64_t npix, int nticks, const float* __restrict__ wave, const float* __restrict__ noise,
          tred_readout_config c, int32_t* __restrict__ nhit, int32_t* __restrict__ hit_tick,
          float* __restrict__ hit_adc) {
  __shared__ float tiles[RO_WARPS][32][RO_CH + 1];
  const int lane = threadIdx.x & 31;
  float (*tile)[RO_CH + 1] = tiles[threadIdx.x >> 5];
  const int64_t p0 = ((int64_t)blockIdx.x * RO_WARPS + (threadIdx.x >> 5)) * 32, p = p0 + lane;
  const bool on = p < npix;
  const int mh = c.max_hits;
  const float thr0 = (float)c.threshold_e, lsb = (float)c.adc_lsb_e;
  const float* nz = (noise && on) ? noise + (size_t)p * mh * 3 : nullptr;
  float q = 0.0f;
  int h = 0, state = 0, left = 0;     // 0 WAIT, 1 INTEG, 2 DEAD
  float thr = thr0 + ((nz && mh > 0) ? nz[0] : 0.0f);
  if (on) for (int i = 0; i < mh; ++i) hit_tick[(size_t)p * mh + i] = -1, hit_adc[(size_t)p * mh + i] = 0.0f;
  for (int t0 = 0; t0 < nticks; t0 += RO_CH) {
    const int nt = min(RO_CH, nticks - t0);
    __syncwarp();
    for (int r = 0; r < 32; ++r) {                       // row r of the group, lanes along the ticks
      if (p0 + r >= npix) break;
      const float* src = wave + (size_t)(p0 + r) * nticks + t0;
      for (int k = lane; k < nt; k += 32) tile[r][k] = src[k];
    }
    __syncwarp();
    if (!on) continue;
    for (int k = 0; k < nt && h < mh; ++k) {
      if (state == 2) {
        if (--left == 0) state = 0;
        continue;
      }
      q += tile[lane][k];
      bool fire = false;
      if (state == 0) {
        if (q >= thr) {
          if (c.n_integ == 0) fire = true;
          else { state = 1; left = c.n_integ; }
        }
      } else {
        fire = (--left == 0);
      }
      if (fire) {
        float v = q + (nz ? nz[3 * h + 1] : 0.0f);
        if (lsb > 0.0f) v = floorf(__fdiv_rn(v, lsb) + 0.5f) * lsb;
        hit_tick[(size_t)p * mh + h] = t0 + k;
        hit_adc[(size_t)p * mh + h] = v;
        q = nz ? nz[3 * h + 2] : 0.0f;
        ++h;
        if (h < mh) thr = thr0 + (nz ? nz[3 * h] : 0.0f);
        if (c.n_reset > 0) { state = 2; left = c.n_reset; } else { state = 0; left = 0; }
      }
    }
  }
  if (on) nhit[p] = h;
}

}  // namespace

extern "C" int tred_readout(const tred_readout_config* cfg, int64_t npix, int32_t nticks, const float* d_wave,
                            const float* d_noise, int32_t* d_nhit, int32_t* d_hit_tick, float* d_hit_adc,
                            void* stream) {
  if (!cfg || npix < 0 || nticks < 0 || cfg->max_hits < 0 || cfg->n_integ < 0 || cfg->n_reset < 0)
    return TRED_EINVAL;
  if (npix == 0) return TRED_OK;
  if (!d_nhit || (nticks > 0 && !d_wave) || (cfg->max_hits > 0 && (!d_hit_tick || !d_hit_adc))) return TRED_EINVAL;
  const int64_t per_cta = 32 * RO_WARPS;
  if ((npix + per_cta - 1) / per_cta >= (1ll << 31)) return TRED_EUNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  k_readout<<<(unsigned)((npix + per_cta - 1) / per_cta), 32 * RO_WARPS, 0, st>>>(npix, nticks, d_wave, d_noise, *cfg, d_nhit, d_hit_tick,
                                                          d_hit_adc);
  TRED_COUNT_LAUNCH(1);
  TRED_LAUNCH_CHECK("k_readout");
  return TRED_OK;
}
