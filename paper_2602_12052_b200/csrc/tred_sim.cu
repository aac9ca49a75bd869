// tred_simulate: the whole path in one call -- segments in, per-pixel current waveforms out
// (Fig. 1) -- on buffers carved from ONE caller-provided workspace.
//
//   drift -> block binning -> convolution plan          (capacities from the previous event)
//   one read of the device-side counts                   (the only host wait of a steady stream)
//   effective charge -> convolution -> overlap-add, either in one pass or, when the block
//   payload exceeds `payload_budget_bytes`, over ranges of time slabs whose payload fits
//   (chunks bounded by device memory; one more read per chunk).
//
// The stepwise calls of include/tred.h do the work; this file only sizes, carves and loops.
#include <string.h>
#include "tred_common.cuh"

namespace {

struct Carver {
  char* base; size_t off, cap;
  void* take(size_t bytes) {
    const size_t o = align_up(off, 1024);
    off = o + bytes;
    return (base && off <= cap) ? base + o : nullptr;
  }
};

// device-side counts, mirrored to pinned host memory in one copy
enum { C_NPAIRS = 0, C_NBLOCKS, C_NCP, C_NSP, C_NTILES, C_HDR = 8 };   // then int32 arrays, see count_layout

struct CountLayout { int slab, cp, sp, rt, tl, total; };     // offsets in int64 units
static CountLayout count_layout(int NBt) {
  CountLayout L;
  const int n = (NBt + 1 + 1) / 2;                   // int64 slots holding NBt + 1 int32
  L.slab = C_HDR; L.cp = L.slab + n; L.sp = L.cp + n; L.rt = L.sp + n; L.tl = L.rt + n; L.total = L.tl + n;
  return L;
}

struct PlanBufs {
  int64_t *cp_keys, *sp_keys, *tile_keys;
  void* work;
};

static PlanBufs carve_planbufs(Carver& c, const tred_ctx* ctx, int64_t cap_cp, int64_t cap_sp, int64_t cap_tiles) {
  PlanBufs p;
  p.cp_keys = (int64_t*)c.take((size_t)(cap_cp > 0 ? cap_cp : 1) * 8);
  p.sp_keys = (int64_t*)c.take((size_t)(cap_sp > 0 ? cap_sp : 1) * 8);
  p.tile_keys = (int64_t*)c.take((size_t)(cap_tiles > 0 ? cap_tiles : 1) * 8);
  p.work = c.take(tred_plan_work_bytes(ctx));
  return p;
}

static size_t conv_want(const tred_ctx* ctx, int64_t ncp, int64_t nsp, size_t conv_min) {   // what tred_convolve can use
  size_t w = tred_convolve_work_bytes(ctx, ncp, nsp);
  if (w > ((size_t)16 << 30)) w = (size_t)16 << 30;
  return w > conv_min ? w : conv_min;
}

static int read_counts(tred_ctx* ctx, const int64_t* d_counts, int n64, cudaStream_t st, int* reads) {
  TRED_CUDA(cudaMemcpyAsync(ctx->h_counts, d_counts, (size_t)n64 * 8, cudaMemcpyDeviceToHost, st));
  TRED_CUDA(cudaStreamSynchronize(st));
  ++*reads;
  return TRED_OK;
}

}  // namespace

extern "C" int tred_simulate(tred_ctx* ctx, int64_t nseg, const float* seg, int seg_on_host, const float* d_rhat,
                             int64_t payload_budget_bytes, void* d_work, size_t work_bytes,
                             int64_t cap_tiles, int64_t* tile_keys, float* tile_data, int out_on_host,
                             int64_t npix_req, const int32_t* d_pix_ids, float* d_dense,
                             tred_sim_result* res, void* stream) {
  if (res) memset(res, 0, sizeof(*res));                 // defined on every return, errors included
  if (!ctx || nseg < 0 || !res || cap_tiles < 0 || npix_req < 0) return TRED_EINVAL;
  res->nseg = nseg;
  TRED_CHECK_DEVICE(ctx);
  if (nseg > 0 && !seg) return TRED_EINVAL;
  if (nseg >= (1ll << 31)) return TRED_EUNSUPPORTED;
  cudaStream_t st = (cudaStream_t)stream;
  const tred_dims& d = ctx->dims;
  const int NBt = (int)d.NB[2];
  const int Bt = ctx->cfg.block[2];
  const int64_t npix = (int64_t)ctx->cfg.npix_x * ctx->cfg.npix_y;
  const int64_t nmap = (int64_t)NBt * npix;
  const CountLayout cl = count_layout(NBt);
  if (cl.total * 8 > 65536) return TRED_EUNSUPPORTED;
  if (!ctx->h_counts) TRED_CUDA(cudaHostAlloc((void**)&ctx->h_counts, 65536, cudaHostAllocDefault));
  int64_t* hc = ctx->h_counts;
  int reads = 0;
  auto ecap = [&](size_t need, size_t conv_share = 0, size_t conv_min = 0) {
    res->work_bytes_needed = (int64_t)need; res->conv_bytes_needed = (int64_t)conv_share;
    res->conv_bytes_min = (int64_t)conv_min; res->host_reads = reads;
    return TRED_ECAP;
  };
  auto empty_event = [&]() -> int {                             // no charge inside the grid: empty outputs
    if (npix_req > 0 && d_dense)
      TRED_CUDA(cudaMemsetAsync(d_dense, 0, (size_t)npix_req * ctx->cfg.nticks * 4, st));
    res->host_reads = reads;
    return (int)TRED_OK;
  };
  if (nseg == 0) return empty_event();

  Carver c{(char*)d_work, 0, work_bytes};
  int64_t* d_counts = (int64_t*)c.take((size_t)cl.total * 8);
  float* seg_d = seg_on_host ? (float*)c.take((size_t)8 * nseg * 4) : const_cast<float*>(seg);
  float* augf = (float*)c.take((size_t)TRED_AUG_NF * nseg * 4);
  int32_t* augi = (int32_t*)c.take((size_t)TRED_AUG_NI * nseg * 4);
  if (!augi) return ecap(c.off + ((size_t)64 << 20));
  if (seg_on_host) TRED_CUDA(cudaMemcpyAsync(seg_d, seg, (size_t)8 * nseg * 4, cudaMemcpyHostToDevice, st));
  TRED_CUDA(cudaMemsetAsync(d_counts, 0, (size_t)cl.total * 8, st));
  int rc = tred_drift(ctx, nseg, seg_d, augf, augi, d_counts + C_NPAIRS, st);
  if (rc != TRED_OK) return rc;

  // ---- binning + plan with capacities from the previous event; exact capacities if they overflow
  int64_t cap_pairs = ctx->hint_pairs > 0 ? ctx->hint_pairs + ctx->hint_pairs / 8 + 1024 : 0;
  const size_t off_after_drift = c.off;
  int64_t *keys = nullptr; int32_t *blk_off = nullptr, *pair_seg = nullptr;
  PlanBufs pb{};
  int64_t npairs = 0, nblocks = 0;
  for (int attempt = 0;; ++attempt) {
    if (cap_pairs == 0) {                                  // no usable hint: read the pair count first
      rc = read_counts(ctx, d_counts, C_HDR, st, &reads);
      if (rc != TRED_OK) return rc;
      cap_pairs = hc[C_NPAIRS];
      if (cap_pairs == 0) return empty_event();            // nothing inside the grid
    }
    if (cap_pairs >= (1ll << 31)) return TRED_EUNSUPPORTED;
    c.off = off_after_drift;
    keys = (int64_t*)c.take((size_t)cap_pairs * 8);       // nblocks <= npairs
    blk_off = (int32_t*)c.take((size_t)(cap_pairs + 1) * 4);
    pair_seg = (int32_t*)c.take((size_t)cap_pairs * 4);
    const size_t bin_bytes = tred_blockbin_work_bytes(ctx, nseg, cap_pairs);
    void* bin_work = c.take(bin_bytes);
    pb = carve_planbufs(c, ctx, nmap, nmap, nmap);
    if (!pb.work) return ecap(c.off + ((size_t)64 << 20));
    int32_t* cnt32 = reinterpret_cast<int32_t*>(d_counts);
    rc = tred_blockbin(ctx, nseg, augi, cap_pairs, cap_pairs, keys, blk_off, pair_seg, cnt32 + 2 * cl.slab,
                       d_counts + C_NBLOCKS, bin_work, bin_bytes, st);
    if (rc != TRED_OK) return rc;
    rc = tred_convolve_plan_dev(ctx, cap_pairs, d_counts + C_NBLOCKS, keys, nmap, pb.cp_keys, cnt32 + 2 * cl.cp,
                                d_counts + C_NCP, nmap, pb.sp_keys, cnt32 + 2 * cl.sp, d_counts + C_NSP, nmap,
                                pb.tile_keys, d_counts + C_NTILES, cnt32 + 2 * cl.rt, pb.work,
                                tred_plan_work_bytes(ctx), st);
    if (rc != TRED_OK) return rc;
    rc = tred_plan_tile_offsets(ctx, pb.work, cnt32 + 2 * cl.tl, st);
    if (rc != TRED_OK) return rc;
    rc = read_counts(ctx, d_counts, cl.total, st, &reads);
    if (rc != TRED_OK) return rc;
    npairs = hc[C_NPAIRS]; nblocks = hc[C_NBLOCKS];
    if (npairs <= cap_pairs) break;
    if (attempt > 0) return TRED_ECUDA;                    // cannot happen: the second pass is exact
    cap_pairs = npairs;
  }
  ctx->hint_pairs = npairs;
  const int64_t ncp = hc[C_NCP], nsp = hc[C_NSP], ntiles = hc[C_NTILES];
  const int32_t* h32 = reinterpret_cast<const int32_t*>(hc);
  const int32_t* h_slab = h32 + 2 * cl.slab;
  const int32_t* h_tile_off = h32 + 2 * cl.tl;
  res->npairs = npairs; res->nblocks = nblocks; res->ncp = ncp; res->nsp = nsp; res->ntiles = ntiles;
  res->nrt = (h32 + 2 * cl.rt)[NBt];
  res->host_reads = reads;
  if (nblocks == 0 || ntiles == 0) return empty_event();
  if (ntiles > cap_tiles) return TRED_ECAP;                // res->ntiles tells the caller what to provide
  if (!tile_keys || !tile_data) return TRED_EINVAL;

  // ---- outputs on the device (staged in the workspace if the caller's buffers are host memory)
  int64_t* d_tile_keys = pb.tile_keys;
  float* d_tile_data = out_on_host ? (float*)c.take((size_t)ntiles * Bt * 4) : tile_data;
  const int64_t blk_bytes = d.block_floats * 4;
  const bool chunked = payload_budget_bytes > 0 && nblocks * blk_bytes > payload_budget_bytes;
  const int64_t row = (int64_t)d.n_over * Bt;
  const size_t effq_bytes = tred_effq_work_bytes(ctx, nseg) < ((size_t)1 << 30) || !chunked
                                ? tred_effq_work_bytes(ctx, nseg) : ((size_t)1 << 30);
  void* effq_work = c.take(effq_bytes);

  if (!chunked) {
    float* payload = (float*)c.take((size_t)nblocks * blk_bytes);
    float* sp_data = (float*)c.take((size_t)nsp * row * 4);
    const size_t o = align_up(c.off, 1024);
    int32_t ns_max = 0;
    for (int b = 0; b < NBt; ++b) ns_max = max(ns_max, (h32 + 2 * cl.sp)[b + 1] - (h32 + 2 * cl.sp)[b]);
    const size_t conv_min = tred_convolve_work_bytes(ctx, 128, ns_max);
    if (!sp_data || o + conv_min > work_bytes)
      return ecap(o + conv_want(ctx, ncp, nsp, conv_min), conv_want(ctx, ncp, nsp, conv_min), conv_min);
    size_t conv_bytes = work_bytes - o;
    if (conv_bytes > ((size_t)16 << 30)) conv_bytes = (size_t)16 << 30;
    rc = tred_effq(ctx, nseg, nblocks, keys, blk_off, pair_seg, augf, augi, payload, effq_work, effq_bytes, st);
    if (rc != TRED_OK) return rc;
    rc = tred_convolve(ctx, nblocks, keys, payload, d_rhat, ncp, pb.cp_keys, h32 + 2 * cl.cp, nsp, pb.sp_keys,
                       h32 + 2 * cl.sp, h32 + 2 * cl.rt, pb.work, sp_data, (char*)d_work + o, conv_bytes, st);
    if (rc != TRED_OK) return rc;
    rc = tred_gather_waveforms(ctx, nsp, sp_data, pb.work, nullptr, 0, ntiles, d_tile_keys, d_tile_data, 0, npix_req,
                               d_pix_ids, d_dense, st);
    if (rc != TRED_OK) return rc;
    res->nchunks = 1;
  } else {
    // ---- ranges of time slabs whose payload fits the budget (blocks are sorted slab-major)
    const int64_t max_blk = payload_budget_bytes / blk_bytes > 0 ? payload_budget_bytes / blk_bytes : 1;
    int64_t big = 0;
    for (int b0 = 0; b0 < NBt;) {                           // largest chunk, for the payload buffer
      if (h_slab[b0 + 1] == h_slab[b0]) { ++b0; continue; }
      int b1 = b0 + 1;
      while (b1 < NBt && h_slab[b1 + 1] - h_slab[b0] <= max_blk) ++b1;
      big = max(big, (int64_t)(h_slab[b1] - h_slab[b0]));
      b0 = b1;
    }
    float* payload = (float*)c.take((size_t)big * blk_bytes);
    int64_t* d_cc = (int64_t*)c.take((size_t)cl.total * 8);          // the chunk plan's counts
    PlanBufs cb = carve_planbufs(c, ctx, nmap, nmap, 1);
    if (!cb.work) return ecap(c.off + ((size_t)6 << 30));
    const size_t off_chunk = c.off;
    TRED_CUDA(cudaMemsetAsync(d_tile_data, 0, (size_t)ntiles * Bt * 4, st));
    // the host copies of the global plan's offsets are overwritten by the chunk reads: keep them
    int32_t slab_h[4096], tile_off_h[4096];
    if (NBt + 1 > 4096) return TRED_EUNSUPPORTED;
    memcpy(slab_h, h_slab, (size_t)(NBt + 1) * 4);
    memcpy(tile_off_h, h_tile_off, (size_t)(NBt + 1) * 4);
    int64_t s_ncp = 0, s_nsp = 0, s_nrt = 0;
    for (int b0 = 0; b0 < NBt;) {
      if (slab_h[b0 + 1] == slab_h[b0]) { ++b0; continue; }
      int b1 = b0 + 1;
      while (b1 < NBt && slab_h[b1 + 1] - slab_h[b0] <= max_blk) ++b1;
      const int64_t k0 = slab_h[b0], nb = slab_h[b1] - k0;
      rc = tred_effq(ctx, nseg, nb, keys + k0, blk_off + k0, pair_seg, augf, augi, payload, effq_work, effq_bytes, st);
      if (rc != TRED_OK) return rc;
      int32_t* cc32 = reinterpret_cast<int32_t*>(d_cc);
      int64_t dummy_cap = 1;
      rc = tred_convolve_plan_dev(ctx, nb, nullptr, keys + k0, nmap, cb.cp_keys, cc32 + 2 * cl.cp, d_cc + C_NCP, nmap,
                                  cb.sp_keys, cc32 + 2 * cl.sp, d_cc + C_NSP, dummy_cap, cb.tile_keys, d_cc + C_NTILES,
                                  cc32 + 2 * cl.rt, cb.work, tred_plan_work_bytes(ctx), st);
      if (rc != TRED_OK) return rc;
      rc = read_counts(ctx, d_cc, cl.total, st, &reads);
      if (rc != TRED_OK) return rc;
      const int64_t c_ncp = hc[C_NCP], c_nsp = hc[C_NSP];
      c.off = off_chunk;
      float* sp_data = (float*)c.take((size_t)c_nsp * row * 4);
      const size_t o = align_up(c.off, 1024);
      int32_t ns_max = 0;
      for (int b = 0; b < NBt; ++b) ns_max = max(ns_max, (h32 + 2 * cl.sp)[b + 1] - (h32 + 2 * cl.sp)[b]);
      const size_t conv_min = tred_convolve_work_bytes(ctx, 128, ns_max);
      if (!sp_data || o + conv_min > work_bytes)
        return ecap(o + conv_want(ctx, c_ncp, c_nsp, conv_min), conv_want(ctx, c_ncp, c_nsp, conv_min), conv_min);
      size_t conv_bytes = work_bytes - o;
      if (conv_bytes > ((size_t)16 << 30)) conv_bytes = (size_t)16 << 30;
      rc = tred_convolve(ctx, nb, keys + k0, payload, d_rhat, c_ncp, cb.cp_keys, h32 + 2 * cl.cp, c_nsp, cb.sp_keys,
                         h32 + 2 * cl.sp, h32 + 2 * cl.rt, cb.work, sp_data, (char*)d_work + o, conv_bytes, st);
      if (rc != TRED_OK) return rc;
      // tiles this slab range reaches: time tiles b0 .. b1 - 1 + n_over - 1, clipped to the window
      const int tb_hi = min(b1 - 1 + d.n_over, NBt);
      const int64_t t_lo = tile_off_h[b0], t_hi = tile_off_h[tb_hi];
      if (t_hi > t_lo) {
        rc = tred_gather_waveforms(ctx, c_nsp, sp_data, cb.work, pb.work, t_lo, t_hi - t_lo, d_tile_keys, d_tile_data, 1,
                                   0, nullptr, nullptr, st);
        if (rc != TRED_OK) return rc;
      }
      s_ncp += c_ncp; s_nsp += c_nsp; s_nrt += (h32 + 2 * cl.rt)[NBt];
      ++res->nchunks;
      b0 = b1;
    }
    res->ncp = s_ncp; res->nsp = s_nsp; res->nrt = s_nrt;
    if (npix_req > 0) {
      rc = tred_gather_waveforms(ctx, 0, nullptr, pb.work, pb.work, 0, 0, d_tile_keys, d_tile_data, 0, npix_req,
                                 d_pix_ids, d_dense, st);
      if (rc != TRED_OK) return rc;
    }
  }
  res->host_reads = reads;
  res->mac_mode = ctx->last_mac_mode;
  res->work_bytes_used = (int64_t)c.off;
  // ---- hand the tiles to the caller
  const cudaMemcpyKind kind = out_on_host ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
  TRED_CUDA(cudaMemcpyAsync(tile_keys, d_tile_keys, (size_t)ntiles * 8, kind, st));
  if (out_on_host) TRED_CUDA(cudaMemcpyAsync(tile_data, d_tile_data, (size_t)ntiles * Bt * 4, kind, st));
  return TRED_OK;
}
