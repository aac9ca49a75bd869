// Device-wide exclusive scan and stable LSD radix sort used by the block binning (S3)
// and the output-tile planning (S5).  Hand-written for sm_100a; no CUB/Thrust.
#include "tred_common.cuh"

namespace {

constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 16;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;   // 4096 elements per CTA

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += t;
  }
  return v;
}

// Exclusive scan of one value per thread across the CTA; returns the exclusive prefix and
// the CTA total through *total.  `smem` holds blockDim.x/32 + 1 ints.
__device__ __forceinline__ int block_excl_scan(int v, int* smem, int* total) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  int inc = warp_incl_scan(v, lane);
  if (lane == 31) smem[w] = inc;
  __syncthreads();
  if (w == 0) {
    int s = lane < nw ? smem[lane] : 0;
    int si = warp_incl_scan(s, lane);
    if (lane < nw) smem[lane] = si - s;
    if (lane == nw - 1) smem[nw] = si;
  }
  __syncthreads();
  int res = inc - v + smem[w];
  *total = smem[nw];
  __syncthreads();
  return res;
}

__global__ void __launch_bounds__(SCAN_THREADS)
k_scan_reduce(const int32_t* __restrict__ in, int64_t n, int32_t* __restrict__ sums) {
  __shared__ int sm[SCAN_THREADS / 32 + 1];
  const int64_t base = (int64_t)blockIdx.x * SCAN_TILE;
  int acc = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    int64_t i = base + (int64_t)k * SCAN_THREADS + threadIdx.x;
    if (i < n) acc += in[i];
  }
  int tot;
  block_excl_scan(acc, sm, &tot);
  if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}

// Single CTA: exclusive scan of `m` block sums in place, total to d_total.
__global__ void __launch_bounds__(1024)
k_scan_sums(int32_t* __restrict__ sums, int m, int64_t* __restrict__ d_total) {
  __shared__ int sm[1024 / 32 + 1];
  long long carry = 0;
  for (int base = 0; base < m; base += 1024) {
    int i = base + threadIdx.x;
    int v = i < m ? sums[i] : 0;
    int tot;
    int ex = block_excl_scan(v, sm, &tot);
    if (i < m) sums[i] = (int)(carry + ex);
    carry += tot;
  }
  if (threadIdx.x == 0 && d_total) *d_total = carry;
}

__global__ void __launch_bounds__(SCAN_THREADS)
k_scan_apply(const int32_t* __restrict__ in, int32_t* __restrict__ out, int64_t n,
             const int32_t* __restrict__ sums) {
  __shared__ int sm[SCAN_THREADS / 32 + 1];
  // thread-contiguous items: thread t owns elements [t*ITEMS, (t+1)*ITEMS) of the tile
  const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
  int v[SCAN_ITEMS];
  int acc = 0;
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    int64_t i = base + k;
    v[k] = i < n ? in[i] : 0;
    acc += v[k];
  }
  int tot;
  int ex = block_excl_scan(acc, sm, &tot) + sums[blockIdx.x];
#pragma unroll
  for (int k = 0; k < SCAN_ITEMS; ++k) {
    int64_t i = base + k;
    if (i < n) out[i] = ex;
    ex += v[k];
  }
}

// ------------------------------------------------------------------ radix sort
constexpr int SORT_THREADS = 256;
constexpr int SORT_WARPS = SORT_THREADS / 32;
constexpr int SORT_STEPS = 16;                               // 32 keys per warp per step
constexpr int SORT_TILE = SORT_THREADS * SORT_STEPS;         // 4096 keys per CTA

__device__ __forceinline__ void warp_digit_counts(const uint32_t* __restrict__ keys, int64_t n,
                                                  int64_t wbase, int shift, int lane, int* cnt) {
  for (int s = 0; s < SORT_STEPS; ++s) {
    int64_t i = wbase + (int64_t)s * 32 + lane;
    int d = i < n ? (int)((keys[i] >> shift) & 255u) : 256;
    unsigned m = __match_any_sync(0xffffffffu, d);
    if (d < 256 && lane == (__ffs(m) - 1)) cnt[d] += __popc(m);
    __syncwarp();
  }
}

__global__ void __launch_bounds__(SORT_THREADS)
k_sort_hist(const uint32_t* __restrict__ keys, int64_t n_cap, const int64_t* __restrict__ d_n,
            int shift, int32_t* __restrict__ counts, int ncta) {
  __shared__ int cnt[SORT_WARPS][256];
  const int64_t n = d_n ? min((int64_t)*d_n, n_cap) : n_cap;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < SORT_WARPS * 256; i += SORT_THREADS) (&cnt[0][0])[i] = 0;
  __syncthreads();
  const int64_t wbase = (int64_t)blockIdx.x * SORT_TILE + (int64_t)w * (SORT_STEPS * 32);
  warp_digit_counts(keys, n, wbase, shift, lane, cnt[w]);
  __syncthreads();
  for (int d = threadIdx.x; d < 256; d += SORT_THREADS) {
    int s = 0;
#pragma unroll
    for (int ww = 0; ww < SORT_WARPS; ++ww) s += cnt[ww][d];
    counts[(int64_t)d * ncta + blockIdx.x] = s;
  }
}

__global__ void __launch_bounds__(SORT_THREADS)
k_sort_scatter(const uint32_t* __restrict__ keys, const int32_t* __restrict__ vals,
               uint32_t* __restrict__ keys_out, int32_t* __restrict__ vals_out,
               int64_t n_cap, const int64_t* __restrict__ d_n, int shift,
               const int32_t* __restrict__ offsets, int ncta) {
  __shared__ int cnt[SORT_WARPS][256];
  const int64_t n = d_n ? min((int64_t)*d_n, n_cap) : n_cap;
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int i = threadIdx.x; i < SORT_WARPS * 256; i += SORT_THREADS) (&cnt[0][0])[i] = 0;
  __syncthreads();
  const int64_t wbase = (int64_t)blockIdx.x * SORT_TILE + (int64_t)w * (SORT_STEPS * 32);
  warp_digit_counts(keys, n, wbase, shift, lane, cnt[w]);
  __syncthreads();
  // per-warp starting offsets: global base of (digit, cta) + counts of the warps before
  for (int d = threadIdx.x; d < 256; d += SORT_THREADS) {
    int run = offsets[(int64_t)d * ncta + blockIdx.x];
#pragma unroll
    for (int ww = 0; ww < SORT_WARPS; ++ww) {
      int c = cnt[ww][d];
      cnt[ww][d] = run;
      run += c;
    }
  }
  __syncthreads();
  int* off = cnt[w];
  for (int s = 0; s < SORT_STEPS; ++s) {
    int64_t i = wbase + (int64_t)s * 32 + lane;
    bool ok = i < n;
    uint32_t k = ok ? keys[i] : 0u;
    int v = ok ? vals[i] : 0;
    int d = ok ? (int)((k >> shift) & 255u) : 256;
    unsigned m = __match_any_sync(0xffffffffu, d);
    int rank = __popc(m & ((1u << lane) - 1u));
    int pos = 0;
    if (ok) pos = off[d] + rank;
    __syncwarp();
    if (ok && lane == (__ffs(m) - 1)) off[d] += __popc(m);
    __syncwarp();
    if (ok) { keys_out[pos] = k; vals_out[pos] = v; }
  }
}

}  // namespace

size_t tred_scan_work_bytes(int64_t n) {
  int64_t nb = (n + SCAN_TILE - 1) / SCAN_TILE;
  if (nb < 1) nb = 1;
  return align_up((size_t)nb * sizeof(int32_t), 256);
}

int tred_exclusive_scan_i32(const int32_t* d_in, int32_t* d_out, int64_t n, int64_t* d_total,
                            void* d_work, cudaStream_t st) {
  if (n <= 0) {
    if (d_total) TRED_CUDA(cudaMemsetAsync(d_total, 0, sizeof(int64_t), st));
    return TRED_OK;
  }
  int nb = cdiv(n, SCAN_TILE);
  int32_t* sums = (int32_t*)d_work;
  k_scan_reduce<<<nb, SCAN_THREADS, 0, st>>>(d_in, n, sums);
  k_scan_sums<<<1, 1024, 0, st>>>(sums, nb, d_total);
  k_scan_apply<<<nb, SCAN_THREADS, 0, st>>>(d_in, d_out, n, sums);
  TRED_COUNT_LAUNCH(3);
  TRED_LAUNCH_CHECK("exclusive_scan");
  return TRED_OK;
}

size_t tred_sort_work_bytes(int64_t n) {
  int64_t ncta = (n + SORT_TILE - 1) / SORT_TILE;
  if (ncta < 1) ncta = 1;
  size_t counts = align_up((size_t)ncta * 256 * sizeof(int32_t), 256);
  return counts + tred_scan_work_bytes(ncta * 256);
}

int tred_radix_sort_pairs(uint32_t* ka, int32_t* va, uint32_t* kb, int32_t* vb,
                          int64_t n_cap, const int64_t* d_n, int bits, void* d_work, cudaStream_t st,
                          uint32_t** keys_out, int32_t** vals_out) {
  *keys_out = ka; *vals_out = va;
  if (n_cap <= 0) return TRED_OK;
  int ncta = cdiv(n_cap, SORT_TILE);
  int32_t* counts = (int32_t*)d_work;
  void* scan_work = (char*)d_work + align_up((size_t)ncta * 256 * sizeof(int32_t), 256);
  for (int shift = 0; shift < bits; shift += 8) {
    k_sort_hist<<<ncta, SORT_THREADS, 0, st>>>(ka, n_cap, d_n, shift, counts, ncta);
    int rc = tred_exclusive_scan_i32(counts, counts, (int64_t)ncta * 256, nullptr, scan_work, st);
    if (rc != TRED_OK) return rc;
    k_sort_scatter<<<ncta, SORT_THREADS, 0, st>>>(ka, va, kb, vb, n_cap, d_n, shift, counts, ncta);
    TRED_COUNT_LAUNCH(2);
    TRED_LAUNCH_CHECK("radix_sort");
    uint32_t* tk = ka; ka = kb; kb = tk;
    int32_t* tv = va; va = vb; vb = tv;
  }
  *keys_out = ka; *vals_out = va;
  return TRED_OK;
}
