// fft_smem.cuh — batched power-of-two complex FFT inside one thread block, in shared memory.
//
// Used by every FFT pass of the path: F_2D of Eq. 7 on the projections and the inverse FFT of the
// USFFT ("second step is replaced to inverse 3D FFT") along x1, x2 and x3.
//
// Algorithm: in-place decimation-in-frequency, ceil(log2 N / 4) passes of radix 4..16.  In a pass every work item
// holds R = 2^rb elements (stride S) in registers, runs a radix-R butterfly there, applies the inter-pass twiddles
// and writes back to the same addresses.  The result is left in (mixed-radix) digit-reversed order; consumers read
// X[k] at fft_pos<LOGN>(k), so the permutation costs nothing.  Shared-memory index i is stored at i + i/16
// (fft_phys) which keeps both the stride-S reads of early passes and the stride-1 groups of the last pass free of
// bank conflicts for 8-byte elements.  Twiddles: one table lookup e^{-2 pi i j/L} per work item (table computed in
// double on the host), its powers by at most log-depth complex products.
#pragma once
#include <cuda_runtime.h>

namespace lam {

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }

__host__ __device__ constexpr int fft_phys(int i) { return i + (i >> 4); }
__host__ __device__ constexpr int fft_pitch(int n) { return n + (n >> 4); }

template <int LOGN>
struct FftShape {
  static constexpr int NP = (LOGN + 3) / 4;  // passes
  __host__ __device__ static constexpr int rb(int i) { return LOGN / NP + (i < LOGN % NP ? 1 : 0); }  // radix bits
  __host__ __device__ static constexpr int sb(int i) {  // stride bits of pass i (bits left after it)
    int s = LOGN;
    for (int k = 0; k <= i; ++k) s -= rb(k);
    return s;
  }
};

// position (logical, before fft_phys) of output bin k after all passes
template <int LOGN>
__device__ __forceinline__ int fft_pos(int k) {
  using F = FftShape<LOGN>;
  int p = 0, sh = 0;
#pragma unroll
  for (int i = 0; i < F::NP; ++i) {
    p |= ((k >> sh) & ((1 << F::rb(i)) - 1)) << F::sb(i);
    sh += F::rb(i);
  }
  return p;
}

// d * e^{DIR * 2 pi i k16 / 16}, k16 a compile-time constant after unrolling
template <int DIR>
__device__ __forceinline__ float2 rot16(float2 d, int k16) {
  const float C[8] = {1.f, 0.92387953251128674f, 0.70710678118654752f, 0.38268343236508977f,
                      0.f, -0.38268343236508977f, -0.70710678118654752f, -0.92387953251128674f};
  const float S[8] = {0.f, 0.38268343236508977f, 0.70710678118654752f, 0.92387953251128674f,
                      1.f, 0.92387953251128674f, 0.70710678118654752f, 0.38268343236508977f};
  if (k16 == 0) return d;
  if (k16 == 4) return DIR > 0 ? make_float2(-d.y, d.x) : make_float2(d.y, -d.x);
  float c = C[k16], s = DIR > 0 ? S[k16] : -S[k16];
  return make_float2(fmaf(d.x, c, -d.y * s), fmaf(d.x, s, d.y * c));
}

__host__ __device__ constexpr int brev_bits(int v, int bits) {
  int r = 0;
  for (int i = 0; i < bits; ++i) r |= ((v >> i) & 1) << (bits - 1 - i);
  return r;
}

// radix-R DIF FFT of a[0..R) in registers; output bin q ends up in a[brev(q)]
template <int R, int DIR>
__device__ __forceinline__ void fft_reg(float2 (&a)[R]) {
#pragma unroll
  for (int half = R / 2; half >= 1; half >>= 1) {
#pragma unroll
    for (int g = 0; g < R; g += 2 * half) {
#pragma unroll
      for (int i = 0; i < half; ++i) {
        float2 u = a[g + i], v = a[g + i + half];
        a[g + i] = cadd(u, v);
        a[g + i + half] = rot16<DIR>(csub(u, v), i * (8 / half));
      }
    }
  }
}

// one work item of pass I on one transform s[] (logical indexing through fft_phys)
template <int LOGN, int DIR, int I>
__device__ __forceinline__ void fft_pass_item(float2* s, int u, const float2* __restrict__ tw) {
  using F = FftShape<LOGN>;
  constexpr int RB = F::rb(I), R = 1 << RB, SB = F::sb(I), S = 1 << SB;
  const int j = u & (S - 1);
  const int base = ((u >> SB) << (SB + RB)) | j;
  float2 a[R];
#pragma unroll
  for (int k = 0; k < R; ++k) a[k] = s[fft_phys(base + k * S)];
  fft_reg<R, DIR>(a);
  if (SB > 0) {
    float2 w[R];
    w[1] = __ldg(&tw[j << (LOGN - SB - RB)]);  // e^{-2 pi i j / L}, L = R*S
    if (DIR > 0) w[1].y = -w[1].y;
#pragma unroll
    for (int q = 2; q < R; ++q) w[q] = (q & 1) ? cmul(w[q - 1], w[1]) : cmul(w[q / 2], w[q / 2]);
#pragma unroll
    for (int q = 1; q < R; ++q) a[brev_bits(q, RB)] = cmul(a[brev_bits(q, RB)], w[q]);
  }
#pragma unroll
  for (int q = 0; q < R; ++q) s[fft_phys(base + q * S)] = a[brev_bits(q, RB)];
}

template <int LOGN, int DIR, int I>
__device__ __forceinline__ void fft_passes(float2* s, int nb, int pitch, const float2* __restrict__ tw) {
  using F = FftShape<LOGN>;
  if constexpr (I < F::NP) {
    constexpr int IB = LOGN - F::rb(I);  // log2(items per transform)
    const int total = nb << IB;
    for (int it = threadIdx.x; it < total; it += blockDim.x)
      fft_pass_item<LOGN, DIR, I>(s + (it >> IB) * pitch, it & ((1 << IB) - 1), tw);
    __syncthreads();
    fft_passes<LOGN, DIR, I + 1>(s, nb, pitch, tw);
  }
}

// nb transforms of length 2^LOGN, transform t at s + t*pitch (pitch >= fft_pitch(N)), element i at fft_phys(i).
// DIR = -1: X[k] = sum x[i] e^{-2 pi i ik/N};  DIR = +1: e^{+...} (unnormalised).  tw: N entries e^{-2 pi i k/N}.
// Must be called by all threads of the block; ends with a __syncthreads().  Caller syncs after filling s.
template <int LOGN, int DIR>
__device__ __forceinline__ void block_fft(float2* s, int nb, int pitch, const float2* __restrict__ tw) {
  fft_passes<LOGN, DIR, 0>(s, nb, pitch, tw);
}

}  // namespace lam
