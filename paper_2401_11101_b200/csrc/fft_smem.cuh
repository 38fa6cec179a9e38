// fft_smem.cuh — batched power-of-two complex FFT inside one thread block: radix stages in registers, the
// exchanges between stages through shared memory.
//
// Used by every FFT pass of the path: F_2D of Eq. 7 on the projections and the inverse FFT of the
// USFFT ("second step is replaced to inverse 3D FFT") along x1, x2 and x3.
//
// Algorithm: decimation in frequency in ceil(log2 N / 4) passes of radix 4..16.  Pass 0 takes its inputs straight
// from a caller-supplied loader (global memory, coalesced: work item u reads elements u + k*S0), every pass runs a
// radix-R butterfly in registers and applies the inter-pass twiddles, passes exchange through shared memory
// in place, and the last pass hands its outputs to a caller-supplied sink (global memory, coalesced: work item v
// holds the bins v + q*N/R_last) or leaves them in shared memory for an epilogue that needs other bins.
// The data in shared memory is in mixed-radix digit-reversed order; bin k lives at fft_at<LOGN>(k).
// Shared-memory position p is stored at fft_swz<LOGN>(p): an XOR of the low four position bits with the
// bit-reversed leading digit (and one bit of the second digit for four-pass sizes), which makes every access
// pattern of every pass (16 lanes of a half-warp, 8-byte elements) hit 16 distinct banks; two-pass sizes
// (N <= 256) use the additive padding p + p/16 instead.  Twiddles: one table lookup e^{-2 pi i j/L} per work item
// (table computed in double on the host), its powers by at most log-depth complex products.
#pragma once
#include <cuda_runtime.h>

namespace lam {

// Complex arithmetic on the packed fp32x2 pipe of sm_100a (FFMA2 / FMUL2 / FADD2: one issue slot per complex add, two
// per complex product; ptxas folds the swap and the sign of (-a.y, a.x) into operand modifiers).  The FFT passes are
// bound by instruction issue, not by the FMA pipe, so halving their floating-point instruction count is what counts.
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  const float2 t = __fmul2_rn(make_float2(-a.y, a.x), make_float2(b.y, b.y));  // (-a.y b.y, a.x b.y)
  return __ffma2_rn(a, make_float2(b.x, b.x), t);                              // (a.x b.x - a.y b.y, a.y b.x + a.x b.y)
}
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }

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

// elements of shared memory one transform of length n occupies (before the caller's own row padding)
__host__ __device__ constexpr int fft_span(int n) { return n <= 256 ? n + (n >> 4) : n; }

// shared-memory pitch of a TFAST block_fft: a multiple of 16 plus 16/nb (nb <= 16 transforms) or 1
__host__ __device__ constexpr int fft_tfast_pitch(int n, int nb) { return ((fft_span(n) + 15) & ~15) + (nb >= 16 ? 1 : 16 / nb); }

// swizzle constant of logical position p (three- and four-pass sizes): depends on the leading digit of p and, for
// four-pass sizes, on the lowest bit of the second digit only, so one evaluation serves a whole work item
template <int LOGN>
__device__ __forceinline__ int fft_xor(int p) {
  using F = FftShape<LOGN>;
  const int d0 = p >> F::sb(0);
  int x = (int)(__brev((unsigned)d0) >> 28);
  if constexpr (F::rb(0) == 3) x ^= d0 & 1;
  if constexpr (F::NP == 4) x ^= ((p >> F::sb(1)) & 1) << 3;
  return x;
}

// physical index of logical position p of a transform
template <int LOGN>
__device__ __forceinline__ int fft_swz(int p) {
  using F = FftShape<LOGN>;
  if constexpr (F::NP <= 2) {
    return p + (p >> 4);
  } else {
    return p ^ fft_xor<LOGN>(p);
  }
}

// physical index of position base + off of a work item whose swizzle constant xb was taken at `base`; `flip8` toggles
// swizzle bit 3 (pass 1 of four-pass sizes, where the element index k walks the second digit: flip8 = k & 1)
template <int LOGN>
__device__ __forceinline__ int fft_swz_item(int base, int off, int xb, bool flip8 = false) {
  using F = FftShape<LOGN>;
  if constexpr (F::NP <= 2) {
    return (base + off) + ((base + off) >> 4);
  } else {
    return (base + off) ^ (flip8 ? xb ^ 8 : xb);
  }
}

// logical position of output bin k after all passes (mixed-radix digit reversal)
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
template <int LOGN>
__device__ __forceinline__ int fft_at(int k) {
  return fft_swz<LOGN>(fft_pos<LOGN>(k));
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
  return cmul(d, make_float2(c, s));
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

// butterfly of pass I on registers a[k] = x[base + k*S] (j = index inside the stride) followed by the inter-pass
// twiddles; on return a[brev(q)] is output digit q
template <int LOGN, int DIR, int I>
__device__ __forceinline__ void fft_bfly(float2 (&a)[1 << FftShape<LOGN>::rb(I)], int j, const float2* __restrict__ tw) {
  using F = FftShape<LOGN>;
  constexpr int RB = F::rb(I), R = 1 << RB, SB = F::sb(I);
  fft_reg<R, DIR>(a);
  if constexpr (SB > 0) {
    float2 w[R];
    w[1] = __ldg(&tw[j << (LOGN - SB - RB)]);  // e^{-2 pi i j / L}, L = R*S
    if (DIR > 0) w[1].y = -w[1].y;
#pragma unroll
    for (int q = 2; q < R; ++q) w[q] = (q & 1) ? cmul(w[q - 1], w[1]) : cmul(w[q / 2], w[q / 2]);
#pragma unroll
    for (int q = 1; q < R; ++q) a[brev_bits(q, RB)] = cmul(a[brev_bits(q, RB)], w[q]);
  }
}

// work item -> (transform t, item u).  TFAST: consecutive threads take consecutive transforms (column FFTs whose
// transforms are adjacent in global memory; nb = 1 << lognb); otherwise consecutive threads take consecutive items.
template <bool TFAST>
__device__ __forceinline__ void fft_split(int it, int itembits, int lognb, int& t, int& u) {
  if (TFAST) {
    t = it & ((1 << lognb) - 1);
    u = it >> lognb;
  } else {
    t = it >> itembits;
    u = it & ((1 << itembits) - 1);
  }
}

template <int LOGN, int DIR, bool TFAST, int I>
__device__ __forceinline__ void fft_mid_passes(float2* s, int nb, int lognb, int pitch, const float2* __restrict__ tw) {
  using F = FftShape<LOGN>;
  if constexpr (I < F::NP - 1) {
    constexpr int RB = F::rb(I), R = 1 << RB, SB = F::sb(I), S = 1 << SB, IB = LOGN - RB;
    for (int it = threadIdx.x; it < nb << IB; it += blockDim.x) {
      int t, u;
      fft_split<TFAST>(it, IB, lognb, t, u);
      const int j = u & (S - 1), base = ((u >> SB) << (SB + RB)) | j;
      float2* st = s + t * pitch;
      const int xb = F::NP > 2 ? fft_xor<LOGN>(base) : 0;
      constexpr bool WALK2 = F::NP == 4 && I == 1;  // the element index walks the second digit
      float2 a[R];
#pragma unroll
      for (int k = 0; k < R; ++k) a[k] = st[fft_swz_item<LOGN>(base, k * S, xb, WALK2 && (k & 1))];
      fft_bfly<LOGN, DIR, I>(a, j, tw);
#pragma unroll
      for (int q = 0; q < R; ++q) st[fft_swz_item<LOGN>(base, q * S, xb, WALK2 && (q & 1))] = a[brev_bits(q, RB)];
    }
    __syncthreads();
    fft_mid_passes<LOGN, DIR, TFAST, I + 1>(s, nb, lognb, pitch, tw);
  }
}

// nb transforms of length N = 2^LOGN (transform t at s + t*pitch, pitch >= fft_span(N)).
//   ld(t, i)     -> float2 input element i of transform t           (called once per element, pass 0)
//   st(t, k, v)  :  output bin k of transform t                     (SINK = true; called once per bin, last pass)
//   SINK = false :  the outputs stay in shared memory, bin k at s[t*pitch + fft_at<LOGN>(k)]; ends with a barrier.
// DIR = -1: X[k] = sum x[i] e^{-2 pi i ik/N};  DIR = +1: e^{+...} (unnormalised).  tw: N entries e^{-2 pi i k/N}.
// Must be called by all threads of the block.  In TFAST mode nb = 1 << lognb and pitch = fft_tfast_pitch(N, nb)
// (a multiple of 16 plus 16/nb) makes every access conflict-free; otherwise lognb is ignored.
template <int LOGN, int DIR, bool TFAST, bool SINK, class LD, class ST>
__device__ __forceinline__ void block_fft(float2* s, int nb, int lognb, int pitch, const float2* __restrict__ tw, LD ld, ST st) {
  using F = FftShape<LOGN>;
  {  // pass 0: global -> registers -> shared
    constexpr int RB = F::rb(0), R = 1 << RB, SB = F::sb(0), S = 1 << SB, IB = LOGN - RB;
    for (int it = threadIdx.x; it < nb << IB; it += blockDim.x) {
      int t, u;
      fft_split<TFAST>(it, IB, lognb, t, u);
      float2 a[R];
#pragma unroll
      for (int k = 0; k < R; ++k) a[k] = ld(t, u + k * S);
      fft_bfly<LOGN, DIR, 0>(a, u, tw);
      float2* sp = s + t * pitch;
      // leading digit = q: the swizzle constant is a compile-time value (plus one bit of u for four-pass sizes)
#pragma unroll
      for (int q = 0; q < R; ++q) {
        if constexpr (F::NP <= 2) {
          sp[fft_swz<LOGN>(u + q * S)] = a[brev_bits(q, RB)];
        } else {
          const int x = fft_xor<LOGN>((q << SB) | (F::NP == 4 ? (u & (1 << F::sb(1))) : 0));
          sp[(u ^ x) + q * S] = a[brev_bits(q, RB)];
        }
      }
    }
    __syncthreads();
  }
  fft_mid_passes<LOGN, DIR, TFAST, 1>(s, nb, lognb, pitch, tw);
  {  // last pass: shared -> registers -> sink (or back in place)
    constexpr int I = F::NP - 1, RB = F::rb(I), R = 1 << RB, IB = LOGN - RB;
    for (int it = threadIdx.x; it < nb << IB; it += blockDim.x) {
      int t, e;
      fft_split<TFAST>(it, IB, lognb, t, e);
      // item v holds the bins v + q*2^IB.  In TFAST mode with nb < 16 transforms a half-warp holds 16/nb items:
      // enumerate them with the low four bits reversed, so that consecutive items differ in the high bits of the
      // leading digit = the low bits of the swizzled bank.
      int v = e;
      if (TFAST && F::rb(0) == 4 && IB >= 4) v = (e & ~15) | (int)(__brev((unsigned)e) >> 28);
      int base = 0, sh = 0;
#pragma unroll
      for (int i = 0; i < I; ++i) {
        base |= ((v >> sh) & ((1 << F::rb(i)) - 1)) << F::sb(i);
        sh += F::rb(i);
      }
      float2* sp = s + t * pitch;
      const int xb = F::NP > 2 ? fft_xor<LOGN>(base) : 0;
      float2 a[R];
#pragma unroll
      for (int k = 0; k < R; ++k) a[k] = sp[fft_swz_item<LOGN>(base, k, xb)];
      fft_reg<R, DIR>(a);
      if constexpr (SINK) {
#pragma unroll
        for (int q = 0; q < R; ++q) st(t, v + (q << IB), a[brev_bits(q, RB)]);
      } else {
#pragma unroll
        for (int q = 0; q < R; ++q) sp[fft_swz_item<LOGN>(base, q, xb)] = a[brev_bits(q, RB)];
      }
    }
    if constexpr (!SINK) __syncthreads();
  }
}

}  // namespace lam
