// Shared-memory mixed-radix FFT used by the block convolution (S4, PAPER.md:L223-232
// Eq. (14); padding rule PAPER.md:L264, reading G20).
//
// Batched complex Stockham autosort FFT of length M = 2^a 3^b, radices {8, 4, 2, 3},
// ping-pong between two shared buffers laid out [element][transform]; every thread does
// whole radix-R butterflies in registers.  Real transforms of length N = 2M go through one complex FFT of length M
// (no pairing of two signals, so no rounding cross-talk between columns / pixels):
//   forward:  z[m] = x[2m] + i x[2m+1],  Z = FFT_M(z),
//             X[k] = (Z[k] + conj Z[M-k])/2 - (i/2) e^{-2 pi i k/N} (Z[k] - conj Z[M-k]),
//             X[0] = Re Z[0] + Im Z[0] (DC), X[M] = Re Z[0] - Im Z[0] (Nyquist).
//   inverse:  Z[k] = (X[k] + conj X[M-k]) + i e^{+2 pi i k/N} (X[k] - conj X[M-k]),
//             z = IFFT_M(Z) (unnormalised), x[2m] = Re z[m]/N, x[2m+1] = Im z[m]/N.
// Spectra hold M complex numbers: slot 0 packs (DC, Nyquist), both real.
#pragma once
#include <cuda_runtime.h>

struct FftPlan {
  int M;            // complex length
  int npass;
  int radix[12];
};

static inline bool tred_make_fft_plan(int M, FftPlan* p) {
  p->M = M; p->npass = 0;
  int m = M;
  while (m % 8 == 0) { p->radix[p->npass++] = 8; m /= 8; }
  while (m % 4 == 0) { p->radix[p->npass++] = 4; m /= 4; }
  while (m % 2 == 0) { p->radix[p->npass++] = 2; m /= 2; }
  while (m % 3 == 0) { p->radix[p->npass++] = 3; m /= 3; }
  return m == 1 && p->npass <= 12;
}

__device__ __forceinline__ float2 cmulf(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
// multiply by -i (forward) or +i (inverse)
template <bool INV> __device__ __forceinline__ float2 mul_mi(float2 a) {
  return INV ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}

template <bool INV> __device__ __forceinline__ void dft2(float2& a, float2& b) {
  const float2 t = a;
  a = make_float2(t.x + b.x, t.y + b.y);
  b = make_float2(t.x - b.x, t.y - b.y);
}

template <bool INV> __device__ __forceinline__ void dft4(float2* v) {
  dft2<INV>(v[0], v[2]);
  dft2<INV>(v[1], v[3]);
  v[3] = mul_mi<INV>(v[3]);
  dft2<INV>(v[0], v[1]);
  dft2<INV>(v[2], v[3]);
  const float2 t = v[1]; v[1] = v[2]; v[2] = t;       // bit reversal of 2 bits
}

template <bool INV> __device__ __forceinline__ void dft8(float2* v) {
  constexpr float H = 0.70710678118654752f;
  dft2<INV>(v[0], v[4]); dft2<INV>(v[1], v[5]); dft2<INV>(v[2], v[6]); dft2<INV>(v[3], v[7]);
  // twiddles w8^1, w8^2, w8^3 on the odd half
  { const float2 t = v[5]; v[5] = INV ? make_float2(H * (t.x - t.y), H * (t.x + t.y))
                                      : make_float2(H * (t.x + t.y), H * (t.y - t.x)); }
  v[6] = mul_mi<INV>(v[6]);
  { const float2 t = v[7]; v[7] = INV ? make_float2(-H * (t.x + t.y), H * (t.x - t.y))
                                      : make_float2(H * (t.y - t.x), -H * (t.x + t.y)); }
  dft2<INV>(v[0], v[2]); dft2<INV>(v[1], v[3]); dft2<INV>(v[4], v[6]); dft2<INV>(v[5], v[7]);
  v[3] = mul_mi<INV>(v[3]); v[7] = mul_mi<INV>(v[7]);
  dft2<INV>(v[0], v[1]); dft2<INV>(v[2], v[3]); dft2<INV>(v[4], v[5]); dft2<INV>(v[6], v[7]);
  // bit reversal of 3 bits: (1,4) (3,6)
  float2 t = v[1]; v[1] = v[4]; v[4] = t;
  t = v[3]; v[3] = v[6]; v[6] = t;
}

template <bool INV> __device__ __forceinline__ void dft3(float2* v) {
  constexpr float S60 = 0.86602540378443865f;
  const float2 t = make_float2(v[1].x + v[2].x, v[1].y + v[2].y);
  const float2 u = make_float2(v[1].x - v[2].x, v[1].y - v[2].y);
  const float2 m = make_float2(v[0].x - 0.5f * t.x, v[0].y - 0.5f * t.y);
  // forward: -i sin60 u ; inverse: +i sin60 u
  const float2 n = INV ? make_float2(-S60 * u.y, S60 * u.x) : make_float2(S60 * u.y, -S60 * u.x);
  v[0] = make_float2(v[0].x + t.x, v[0].y + t.y);
  v[1] = make_float2(m.x + n.x, m.y + n.y);
  v[2] = make_float2(m.x - n.x, m.y - n.y);
}

// twN[k] = exp(-2 pi i k / N), k < N = 2M.  w_M^e = twN[2e].  Filled once per call into
// global memory (k_fill_twiddles in tred_conv.cu), copied to shared memory by each CTA.
__device__ __forceinline__ float2 twiddle_N(int k, int N) {
  float sn, cs;
  sincospif(-2.0f * (float)k / (float)N, &sn, &cs);
  return make_float2(cs, sn);
}
__device__ __forceinline__ void load_twiddles_N(float2* twN, const float2* __restrict__ gtw, int N) {
  for (int k = threadIdx.x; k < N; k += blockDim.x) twN[k] = gtw[k];
}

// One Stockham pass of radix R over nb transforms of length M.
// src/dst: [M][nb] shared buffers, the batch index fastest: the threads of a warp work on
// neighbouring transforms at the same butterfly, so every shared-memory access of a warp
// is a contiguous run (no bank conflicts) and the twiddle loads are broadcasts.
// Ns = product of the radices of earlier passes.  Elements >= nz of src are taken as zero
// without being read (zero padding of the first pass).
template <int R, bool INV>
__device__ __forceinline__ void stockham_pass(const float2* __restrict__ src, float2* __restrict__ dst,
                                              const float2* __restrict__ twN, int M, int Ns, int nb, int nz) {
  const int per = M / R;
  const int tws = (M / (Ns * R)) * 2;       // exponent step in units of twN
  const int jstep = blockDim.x / nb;
  const int b = threadIdx.x % nb;
  if ((int)threadIdx.x >= jstep * nb) return;
  for (int j = threadIdx.x / nb; j < per; j += jstep) {
    const int k = j % Ns;
    float2 v[R];
#pragma unroll
    for (int t = 0; t < R; ++t) {
      const int e = j + t * per;
      v[t] = (e < nz) ? src[e * nb + b] : make_float2(0.0f, 0.0f);
    }
    if (Ns > 1) {
#pragma unroll
      for (int t = 1; t < R; ++t) {
        float2 w = twN[k * t * tws];
        if (INV) w.y = -w.y;
        v[t] = cmulf(v[t], w);
      }
    }
    if (R == 2) dft2<INV>(v[0], v[1]);
    else if (R == 3) dft3<INV>(v);
    else if (R == 4) dft4<INV>(v);
    else dft8<INV>(v);
    const int o = (j - k) * R + k;
#pragma unroll
    for (int t = 0; t < R; ++t) dst[(o + t * Ns) * nb + b] = v[t];
  }
}

// Runs all passes; data starts in `a` ([M][nb], elements >= nz are zero and need not be
// stored), returns the buffer that holds the result (natural order).  Contains the
// __syncthreads between passes and one after the last.  Needs blockDim.x >= nb.
template <bool INV>
__device__ __forceinline__ float2* fft_stockham(float2* a, float2* b, const float2* twN,
                                                const FftPlan& pl, int nb, int nz) {
  int Ns = 1;
  for (int p = 0; p < pl.npass; ++p) {
    const int R = pl.radix[p];
    if (R == 8) stockham_pass<8, INV>(a, b, twN, pl.M, Ns, nb, nz);
    else if (R == 4) stockham_pass<4, INV>(a, b, twN, pl.M, Ns, nb, nz);
    else if (R == 2) stockham_pass<2, INV>(a, b, twN, pl.M, Ns, nb, nz);
    else stockham_pass<3, INV>(a, b, twN, pl.M, Ns, nb, nz);
    __syncthreads();
    Ns *= R;
    nz = pl.M;
    float2* t = a; a = b; b = t;
  }
  return a;
}

// Z: complex spectrum of the packed signals ([M][nb], natural order); returns X[k], k < M,
// of transform b (slot 0 = (DC, Nyquist)).
__device__ __forceinline__ float2 rfft_post(const float2* Z, int nb, int b, const float2* twN, int M, int k) {
  if (k == 0) { const float2 z0 = Z[b]; return make_float2(z0.x + z0.y, z0.x - z0.y); }
  const float2 p = Z[k * nb + b], q = Z[(M - k) * nb + b];
  const float2 e = make_float2(0.5f * (p.x + q.x), 0.5f * (p.y - q.y));     // (Z[k] + conj Z[M-k])/2
  const float2 o = make_float2(0.5f * (p.x - q.x), 0.5f * (p.y + q.y));     // (Z[k] - conj Z[M-k])/2
  const float2 w = twN[k];
  const float2 wo = cmulf(w, o);
  return make_float2(e.x + wo.y, e.y - wo.x);                                // e - i w o
}

// p = X[k], q = X[M-k] of a packed half spectrum (k > 0); returns Z[k] of the inverse.
// For k = 0 pass p = q = X[0] = (DC, Nyquist).
__device__ __forceinline__ float2 rfft_pre_inverse(float2 p, float2 q, const float2* twN, int k) {
  if (k == 0) return make_float2(p.x + p.y, p.x - p.y);
  const float2 e = make_float2(p.x + q.x, p.y - q.y);                       // X[k] + conj X[M-k]
  const float2 o = make_float2(p.x - q.x, p.y + q.y);                       // X[k] - conj X[M-k]
  const float2 w = make_float2(twN[k].x, -twN[k].y);                        // e^{+2 pi i k/N}
  const float2 wo = cmulf(w, o);
  return make_float2(e.x - wo.y, e.y + wo.x);                                // e + i w o
}

// ---------------------------------------------------------------------------------
// Compile-time variant of the same Stockham passes: length M, transforms per CTA NB and
// threads NT are template parameters, so every index (division by NB, modulo by the
// pass stride, twiddle step) is a constant expression and the passes unroll.  Same
// radix order as tred_make_fft_plan (8s, 4s, 2s, then 3s), same arithmetic.
template <int REM> struct NextRadix {
  static constexpr int R = (REM % 8 == 0) ? 8 : (REM % 4 == 0) ? 4 : (REM % 2 == 0) ? 2 : 3;
};

template <int R, int M, int NS, bool INV, int NB, int NT>
__device__ __forceinline__ void stockham_pass_ct(const float2* __restrict__ src, float2* __restrict__ dst,
                                                 const float2* __restrict__ twN, int nz) {
  constexpr int PER = M / R;
  constexpr int TWS = (M / (NS * R)) * 2;
  constexpr int JSTEP = NT / NB;
  const int b = threadIdx.x % NB;
  const int jt = threadIdx.x / NB;
  if (jt >= JSTEP) return;
#pragma unroll 1
  for (int j = jt; j < PER; j += JSTEP) {
    const int k = j % NS;
    float2 v[R];
#pragma unroll
    for (int t = 0; t < R; ++t) {
      const int e = j + t * PER;
      v[t] = (e < nz) ? src[e * NB + b] : make_float2(0.0f, 0.0f);
    }
    if (NS > 1) {
#pragma unroll
      for (int t = 1; t < R; ++t) {
        float2 w = twN[k * (t * TWS)];
        if (INV) w.y = -w.y;
        v[t] = cmulf(v[t], w);
      }
    }
    if (R == 2) dft2<INV>(v[0], v[1]);
    else if (R == 3) dft3<INV>(v);
    else if (R == 4) dft4<INV>(v);
    else dft8<INV>(v);
    const int o = (j - k) * R + k;
#pragma unroll
    for (int t = 0; t < R; ++t) dst[(o + t * NS) * NB + b] = v[t];
  }
}

template <int M, int NS, bool INV, int NB, int NT>
__device__ __forceinline__ float2* fft_stockham_ct(float2* a, float2* b, const float2* twN, int nz) {
  if constexpr (NS >= M) {
    return a;
  } else {
    constexpr int R = NextRadix<M / NS>::R;
    stockham_pass_ct<R, M, NS, INV, NB, NT>(a, b, twN, nz);
    __syncthreads();
    return fft_stockham_ct<M, NS * R, INV, NB, NT>(b, a, twN, M);
  }
}

// ---------------------------------------------------------------------------------
// In-register radix-2 decimation-in-frequency FFT of B = 8, 16 or 32 points (forward).
// Fully unrolled: every index and twiddle is a compile-time constant.  Element p of the
// result holds X[bitrev_B(p)].
__device__ constexpr float TRED_C32[17] = {
    1.0f, 0.98078528040323043f, 0.92387953251128674f, 0.83146961230254524f, 0.70710678118654752f,
    0.55557023301960218f, 0.38268343236508978f, 0.19509032201612825f, 0.0f, -0.19509032201612825f,
    -0.38268343236508978f, -0.55557023301960218f, -0.70710678118654752f, -0.83146961230254524f,
    -0.92387953251128674f, -0.98078528040323043f, -1.0f};
__device__ constexpr float TRED_S32[17] = {
    0.0f, 0.19509032201612825f, 0.38268343236508978f, 0.55557023301960218f, 0.70710678118654752f,
    0.83146961230254524f, 0.92387953251128674f, 0.98078528040323043f, 1.0f, 0.98078528040323043f,
    0.92387953251128674f, 0.83146961230254524f, 0.70710678118654752f, 0.55557023301960218f,
    0.38268343236508978f, 0.19509032201612825f, 0.0f};

__host__ __device__ constexpr int tred_bitrev(int x, int bits) {
  int r = 0;
  for (int i = 0; i < bits; ++i) r |= ((x >> i) & 1) << (bits - 1 - i);
  return r;
}
__host__ __device__ constexpr int tred_log2(int x) { int l = 0; while ((1 << l) < x) ++l; return l; }

template <int B, int H> struct FftRegStage {
  static __device__ __forceinline__ void run(float2 (&y)[B]) {
    constexpr float HS = 0.70710678118654752f;
#pragma unroll
    for (int i0 = 0; i0 < B; i0 += 2 * H) {
#pragma unroll
      for (int j = 0; j < H; ++j) {
        const float2 a = y[i0 + j], b = y[i0 + j + H];
        y[i0 + j] = make_float2(a.x + b.x, a.y + b.y);
        const float2 d = make_float2(a.x - b.x, a.y - b.y);
        const int t = j * (16 / H);                        // twiddle exp(-2 pi i t / 32)
        float2 r;
        if (t == 0) r = d;
        else if (t == 8) r = make_float2(d.y, -d.x);
        else if (t == 4) r = make_float2(HS * (d.x + d.y), HS * (d.y - d.x));
        else if (t == 12) r = make_float2(HS * (d.y - d.x), -HS * (d.x + d.y));
        else r = make_float2(d.x * TRED_C32[t] + d.y * TRED_S32[t], d.y * TRED_C32[t] - d.x * TRED_S32[t]);
        y[i0 + j + H] = r;
      }
    }
    FftRegStage<B, H / 2>::run(y);
  }
};
template <int B> struct FftRegStage<B, 0> {
  static __device__ __forceinline__ void run(float2 (&)[B]) {}
};
template <int B> __device__ __forceinline__ void fft_reg_dif(float2 (&y)[B]) {
  static_assert(B == 8 || B == 16 || B == 32, "register FFT sizes");
  FftRegStage<B, B / 2>::run(y);
}
