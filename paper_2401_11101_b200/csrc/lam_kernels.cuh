// lam_kernels.cuh — sm_100a kernels of the laminographic back-projection (see include/lam.h for the operator).
//
// Stage map (S-numbers are SURVEY.md §8(a) rows):
//   k_rows     S0+S1  -log prep, row FFT along u of two real rows per complex transform, filter H[k_u] (Eq. 3)
//   k_cols     S1     column FFT along v, Hermitian fold onto the k_v >= 0 planes, centring phases
//   k_jobs, k_spread  S2  gridding in (xi1, xi2): lam_spread.cuh
//   k_ifft_x1  S3     inverse FFT along xi1 -> x1, cropped to the n central outputs
//   k_ifft_x2  S3     inverse FFT along xi2 -> x2, cropped
//   k_zstage   S2+S3+S4  gridding in xi3 (depends on k_v only, Eq. 6), inverse FFT to x3, crop, real part,
//                     division by the kernel transform on all three axes
#pragma once
#include <cstdint>
#include <cuda.h>
#include <cuda_runtime.h>

#include "fft_smem.cuh"
#include "lam_math.h"

namespace lam {

// (dark, flat) -> (dark, 1 / max(flat - dark, 1)): the per-pixel constants of the -log prep (reading Q12)
__global__ void k_darkflat(const float* dark, const float* flat, float2* df, size_t cnt) {
  size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < cnt) df[i] = make_float2(dark[i], 1.0f / fmaxf(flat[i] - dark[i], 1.0f));
}

// ---------------------------------------------------------------------------------------------------------------
// S0 + S1a: rows
// ---------------------------------------------------------------------------------------------------------------
struct RowsArgs {
  const void* proj;     // chunk base: [nth][h][w] float or uint16
  const float2* df;     // [h][w] (dark, 1 / max(flat - dark, 1))
  float tmin;
  float2* R;            // [nth][h][WR]  filtered half spectra of the rows
  const float2* Pu;     // [w/2+1]  H[k] e^{2 pi i k c_u / w} / (w h)
  const float2* tw;     // twiddles of length w
  int h, WR, nb;        // nb: row pairs per block
};

template <int LOGW, bool RAW>
__global__ void __launch_bounds__(256, 4) k_rows(RowsArgs a) {
  constexpr int w = 1 << LOGW, P = fft_span(w);
  extern __shared__ float2 sm[];
  const int th = blockIdx.y, pair0 = blockIdx.x * a.nb;
  const size_t pbase = (size_t)th * a.h * w;
  auto ld = [&](int t, int ju) -> float2 {
    const int jv = 2 * (pair0 + t);
    if (RAW) {
      const uint16_t* p = (const uint16_t*)a.proj + pbase + (size_t)jv * w + ju;
      float r0 = (float)p[0], r1 = (float)p[w];
      const float2 g0 = __ldg(&a.df[jv * w + ju]), g1 = __ldg(&a.df[(jv + 1) * w + ju]);
      float t0 = (r0 - g0.x) * g0.y, t1 = (r1 - g1.x) * g1.y;
      return make_float2(-logf(fmaxf(t0, a.tmin)), -logf(fmaxf(t1, a.tmin)));
    } else {
      const float* p = (const float*)a.proj + pbase + (size_t)jv * w + ju;
      return make_float2(p[0], p[w]);
    }
  };
  block_fft<LOGW, -1, false, false>(sm, a.nb, 0, P, a.tw, ld, [](int, int, float2) {});
  constexpr int NK = w / 2 + 1;
  for (int idx = threadIdx.x; idx < a.nb * NK; idx += blockDim.x) {
    int t = idx / NK, k = idx - t * NK, jv = 2 * (pair0 + t);
    float2 zk = sm[t * P + fft_at<LOGW>(k)];
    float2 zn = sm[t * P + fft_at<LOGW>((w - k) & (w - 1))];
    float2 ra = make_float2(0.5f * (zk.x + zn.x), 0.5f * (zk.y - zn.y));   // spectrum of the even row
    float2 rb = make_float2(0.5f * (zk.y + zn.y), -0.5f * (zk.x - zn.x));  // spectrum of the odd row
    float2 pu = a.Pu[k];
    size_t o = ((size_t)th * a.h + jv) * a.WR + k;
    a.R[o] = cmul(ra, pu);
    a.R[o + a.WR] = cmul(rb, pu);
  }
}

// S0 + S1a with u-padding (lam.h pad_u, reading Q11b): the two packed rows are extended to 2w samples by replicating
// their edge values, transformed at length 2w, multiplied by the filter response of that length (Hp, real and even,
// 1/(2w) included), transformed back, cropped to the w detector samples and only then transformed at length w as in
// k_rows (Pu carries the centring phase and 1/(wh) but no filter).  Three transforms in shared memory, two buffers.
struct RowsPadArgs {
  RowsArgs r;          // r.Pu: phase and normalisation only; r.tw: twiddles of length w
  const float* Hp;     // [w + 1]  filter response of the 2w-sample row for k = 0..w, times 1/(2w)
  const float2* tw2;   // twiddles of length 2w
};

template <int LOGW, bool RAW>
__global__ void __launch_bounds__(256) k_rows_pad(RowsPadArgs pa) {
  constexpr int w = 1 << LOGW, LP = LOGW + 1, wp = 2 * w, off = w / 2, PP = fft_span(wp), P = fft_span(w);
  const RowsArgs& a = pa.r;
  extern __shared__ float2 sm[];
  float2* bufA = sm;
  float2* bufB = sm + a.nb * PP;
  const int th = blockIdx.y, pair0 = blockIdx.x * a.nb;
  const size_t pbase = (size_t)th * a.h * w;
  auto ld0 = [&](int t, int j) -> float2 {
    const int jv = 2 * (pair0 + t), ju = min(max(j - off, 0), w - 1);
    if (RAW) {
      const uint16_t* p = (const uint16_t*)a.proj + pbase + (size_t)jv * w + ju;
      float r0 = (float)p[0], r1 = (float)p[w];
      const float2 g0 = __ldg(&a.df[jv * w + ju]), g1 = __ldg(&a.df[(jv + 1) * w + ju]);
      float t0 = (r0 - g0.x) * g0.y, t1 = (r1 - g1.x) * g1.y;
      return make_float2(-logf(fmaxf(t0, a.tmin)), -logf(fmaxf(t1, a.tmin)));
    } else {
      const float* p = (const float*)a.proj + pbase + (size_t)jv * w + ju;
      return make_float2(p[0], p[w]);
    }
  };
  block_fft<LP, -1, false, false>(bufA, a.nb, 0, PP, pa.tw2, ld0, [](int, int, float2) {});
  auto ld1 = [&](int t, int i) -> float2 {
    const float hv = pa.Hp[i <= w ? i : wp - i];
    const float2 z = bufA[t * PP + fft_at<LP>(i)];
    return make_float2(z.x * hv, z.y * hv);
  };
  block_fft<LP, +1, false, false>(bufB, a.nb, 0, PP, pa.tw2, ld1, [](int, int, float2) {});
  auto ld2 = [&](int t, int ju) -> float2 { return bufB[t * PP + fft_at<LP>(ju + off)]; };
  block_fft<LOGW, -1, false, false>(bufA, a.nb, 0, P, a.tw, ld2, [](int, int, float2) {});
  constexpr int NK = w / 2 + 1;
  for (int idx = threadIdx.x; idx < a.nb * NK; idx += blockDim.x) {
    int t = idx / NK, k = idx - t * NK, jv = 2 * (pair0 + t);
    float2 zk = bufA[t * P + fft_at<LOGW>(k)];
    float2 zn = bufA[t * P + fft_at<LOGW>((w - k) & (w - 1))];
    float2 ra = make_float2(0.5f * (zk.x + zn.x), 0.5f * (zk.y - zn.y));
    float2 rb = make_float2(0.5f * (zk.y + zn.y), -0.5f * (zk.x - zn.x));
    float2 pu = a.Pu[k];
    size_t o = ((size_t)th * a.h + jv) * a.WR + k;
    a.R[o] = cmul(ra, pu);
    a.R[o + a.WR] = cmul(rb, pu);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// S1b: columns.  Output planes S[p][theta][q], p = 0..h/2 (k_v = p, p = h/2 stands for k_v = -h/2),
// q = 0..w (k_u = q - w/2; q = w is the +w/2 copy of the Nyquist column, reading Q8).
// ---------------------------------------------------------------------------------------------------------------
struct ColsArgs {
  const float2* R;   // [nth][h][WR]
  float2* S;         // [h/2+1][ntheta][WQ]
  const float2* Pv;  // [h/2+1]  e^{2 pi i k_v c_v / h}
  const float2* tw;  // length h
  int w, WR, WQ, ntheta, th0, lcb;  // 1 << lcb columns per block
  int p_lo, p_hi;  // only the planes p_lo <= p < p_hi are written (S points at plane 0 even when it is not stored: banded spill mode)
  float alpha;  // 2-D low-pass 1/(1 + alpha ((k_u/w)^2 + (k_v/h)^2)) on the projection spectrum (lam.h spectral_alpha)
};


template <int LOGH>
__global__ void __launch_bounds__(512) k_cols(ColsArgs a) {
  constexpr int h = 1 << LOGH;
  extern __shared__ float2 sm[];
  const int kColsLog = a.lcb, kColsCb = 1 << a.lcb, P = fft_tfast_pitch(h, kColsCb);
  const int thl = blockIdx.y, k0 = blockIdx.x * kColsCb;
  const int nc = min(kColsCb, a.w / 2 + 1 - k0);
  const float2* Rb = a.R + (size_t)thl * h * a.WR + k0;
  auto ld = [&](int t, int jv) -> float2 { return t < nc ? Rb[(size_t)jv * a.WR + t] : make_float2(0.f, 0.f); };
  block_fft<LOGH, -1, true, false>(sm, kColsCb, kColsLog, P, a.tw, ld, [](int, int, float2) {});
  const int hw = a.w / 2, th = a.th0 + thl;
  auto emit = [&](int p, int c) {
    if (c >= nc || p < a.p_lo || p >= a.p_hi) return;
    int k = k0 + c;
    float2 cp = sm[c * P + fft_at<LOGH>(p)];
    float2 cm = sm[c * P + fft_at<LOGH>((h - p) & (h - 1))];
    cm.y = -cm.y;
    float2 pv = a.Pv[p];
    bool mid = p > 0 && p < h / 2;
    float wplus = mid ? (k < hw ? 2.f : 1.f) : (k < hw ? 1.f : 0.f);
    float wminus = mid ? (k < hw ? 2.f : 1.f) : 1.f;
    float2* Srow = a.S + ((size_t)p * a.ntheta + th) * a.WQ;
    if (a.alpha != 0.f) {  // same value at (+-k_u, +-k_v)
      const float fu = (float)k / (float)a.w, fv = (float)p / (float)h, m = 1.0f / (1.0f + a.alpha * (fu * fu + fv * fv));
      wplus *= m;
      wminus *= m;
    }
    float2 vp = cmul(cp, pv), vm = cmul(cm, pv);
    Srow[hw + k] = make_float2(vp.x * wplus, vp.y * wplus);
    if (k > 0) Srow[hw - k] = make_float2(vm.x * wminus, vm.y * wminus);
  };
  for (int idx = threadIdx.x; idx < (h / 2) * kColsCb; idx += blockDim.x) {
    int e = idx >> kColsLog, c = idx & (kColsCb - 1);
    int p = e;  // radix-16 leading digit: low four bits reversed, as in the last FFT pass (distinct banks)
    if (FftShape<LOGH>::rb(0) == 4 && h / 2 >= 16) p = (e & ~15) | (int)(__brev((unsigned)e) >> 28);
    emit(p, c);
  }
  if (threadIdx.x < kColsCb) emit(h / 2, threadIdx.x);
}

// ---------------------------------------------------------------------------------------------------------------
// S3: inverse FFT along xi1 (rows of a plane, contiguous), cropped to the n central x1.
//   T[pl][i2][ix] = (-1)^x sum_i G[pl][i2][i] e^{+2 pi i x i / M},  x = ix - n/2  (grid index i = m + M/2)
// ---------------------------------------------------------------------------------------------------------------
struct IfftArgs {
  const float2* in;
  float2* out;
  const float2* tw;
  int n, nb, lnb;  // nb = 1 << lnb: rows (x1 pass) or columns (x2 pass) per block
};

template <int LOGM>
__global__ void __launch_bounds__(256, 4) k_ifft_x1(IfftArgs a) {
  constexpr int M = 1 << LOGM, P = fft_span(M);
  extern __shared__ float2 sm[];
  const int pl = blockIdx.y, r0 = blockIdx.x * a.nb;
  const float2* in = a.in + ((size_t)pl * M + r0) * M;
  float2* out = a.out + ((size_t)pl * M + r0) * a.n;
  const int n = a.n, hn = a.n / 2;
  auto ld = [&](int t, int i) -> float2 { return __ldcs(&in[(size_t)t * M + i]); };  // G is read once: evict-first
  auto st = [&](int t, int k, float2 v) {
    int ix = k < hn ? k + hn : k - (M - hn);  // x = k (k < n/2) or k - M (k >= M - n/2)
    if (k >= hn && k < M - hn) return;
    if (k & 1) { v.x = -v.x; v.y = -v.y; }
    out[(size_t)t * n + ix] = v;
  };
  block_fft<LOGM, +1, false, true>(sm, a.nb, 0, P, a.tw, ld, st);
}

// S3: inverse FFT along xi2 (columns), cropped:  A[p][ix2][ix1] = (-1)^x2 sum_i2 T[pl][i2][ix1] e^{+2 pi i x2 i2/M}
template <int LOGM>
__global__ void __launch_bounds__(512) k_ifft_x2(IfftArgs a) {
  constexpr int M = 1 << LOGM;
  extern __shared__ float2 sm[];
  const int P = fft_tfast_pitch(M, a.nb);
  const int pl = blockIdx.y, c0 = blockIdx.x * a.nb;
  const int n = a.n, hn = a.n / 2;
  const float2* in = a.in + (size_t)pl * M * n + c0;
  float2* out = a.out + (size_t)pl * n * n + c0;
  auto ld = [&](int t, int i) -> float2 { return in[(size_t)i * n + t]; };
  auto st = [&](int t, int k, float2 v) {
    int ix = k < hn ? k + hn : k - (M - hn);
    if (k >= hn && k < M - hn) return;
    if (k & 1) { v.x = -v.x; v.y = -v.y; }
    out[(size_t)ix * n + t] = v;
  };
  block_fft<LOGM, +1, true, true>(sm, a.nb, a.lnb, P, a.tw, ld, st);
}

// ---------------------------------------------------------------------------------------------------------------
// Single-slice mode (lam_backproject_slice; the `try` / `try-lamino` searches of PAPER.md:254-270).  For one slice x3
// the x3 transform of Eq. 9 is the exact phase e^{2 pi i x3 k_v cos(phi)/h} per plane, so all planes
// add up on ONE fine grid before a single 2-D inverse FFT:  Gs += sum_p zph[p] G[p].
// ---------------------------------------------------------------------------------------------------------------
__global__ void k_slice_reduce(const float2* __restrict__ G, float2* __restrict__ Gs, const float2* __restrict__ zph, int np,
                               size_t cells) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < cells; i += (size_t)gridDim.x * blockDim.x) {
    float2 acc = Gs[i];
    for (int pl = 0; pl < np; ++pl) {
      const float2 g = __ldcs(&G[(size_t)pl * cells + i]), z = zph[pl];
      acc.x += g.x * z.x - g.y * z.y;
      acc.y += g.x * z.y + g.y * z.x;
    }
    Gs[i] = acc;
  }
}

// rotation-axis search: S[p][theta][q] *= ph[q], ph[q] = e^{2 pi i (q - w/2) delta / w} moves the axis by delta pixels
// (reading Q13: the axis position is a phase on the k_u spectrum)
__global__ void k_center_shift(float2* __restrict__ S, const float2* __restrict__ ph, int WQ, int nq, size_t rows) {
  const int q = blockIdx.x * blockDim.x + threadIdx.x;
  if (q >= nq) return;
  const float2 f = ph[q];
  for (size_t r = blockIdx.y; r < rows; r += gridDim.y) {
    float2* e = S + r * WQ + q;
    const float2 v = *e;
    *e = make_float2(v.x * f.x - v.y * f.y, v.x * f.y + v.y * f.x);
  }
}

// out[x2][x1] = Re As[x2][x1] / (kaphat(x1/M) kaphat(x2/M))
__global__ void k_slice_out(const float2* __restrict__ As, float* __restrict__ out, const float* __restrict__ dx, int n) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n * n) return;
  const int x2 = i / n, x1 = i - x2 * n;
  out[i] = As[i].x * dx[x1] * dx[x2];
}

// ---------------------------------------------------------------------------------------------------------------
// x3 stage, one block per (x2, group of 2..8 x1): xi3 = k_v cos(phi)/h depends on k_v only (Eq. 6), so the planes
// A[p] are samples of a 1-D unequally spaced spectrum along x3 for every (x1, x2):
//   Gz[m3] = sum_p A[p] kap(t3(p) - m3),  t3 = M3 k_v cos(phi)/h;   vol[x3] = Re sum_m3 Gz[m3] e^{2 pi i x3 m3/M3}
//   divided by kaphat(x1/M) kaphat(x2/M) kaphat(x3/M3)  (PAPER.md:136 step 1, reversed per PAPER.md:140).
// The gridding is a banded matrix that is the same for every column.  Only the cells that some plane has a tap on
// are ACTIVE (about half of M3: the planes k_v >= 0 reach xi3 >= 0 only); for active cell j the planes with a tap on
// it are contiguous, [zlo[j], zlo[j] + zcnt[j]), with weights ztab[s][j]; the k_v = -h/2 plane (stored last) has its
// own weight zlast[j].  Three phases: (1) the block's columns of every plane are staged in shared memory (coalesced),
// (2) one thread per (active cell, column pair) accumulates the cell over its band: the weight is read once per tap
// and serves two columns, (3) the length-M3 inverse FFT (two columns per complex transform: only the real part is
// kept) reads the compact cells through the cell -> slot map zidx.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kZCb = 8, kZLog = 3;

struct ZArgs {
  const float2* A;       // [h/2+1][a_rows][n]: plane p, row x2 - a_x2_0 (in core: a_rows = n, a_x2_0 = 0; spilled: one slab)
  size_t a_pstride;      // plane stride of A in elements
  int a_x2_0;            // x2 index held by row 0 of A
  float* vol;            // output buffer; element (ix3, ix2, ix1) at vol[ix3*zstride + (ix2 - vol_x2_0)*n + ix1]
  size_t zstride;
  const float2* tw;      // length M3
  const float* ztab;     // [KZ][nact]
  const int* zlo;        // [nact] first plane with a tap on active cell j
  const int* zcnt;       // [nact] number of such planes (<= KZ)
  const float* zlast;    // [nact]
  const int* zidx;       // [M3] slot of cell i among the active cells, or -1
  const float* dx;       // [n]  1/kaphat(x/M)
  const float* dz;       // [nz] 1/kaphat(x3/M3)
  int n, nz, np, nact, lcb;  // 1 << lcb columns per block
  int x2_0;              // first x2 row of this launch
  int vol_x2_0;          // x2 index held by row 0 of the output buffer
};

// row pitch of the staged planes in float2: rows two or three planes apart (neighbouring cells) land in different
// 16-byte bank groups for the 128-bit reads of phase 2
__host__ __device__ constexpr int z_pitch(int cb) { return cb == 8 ? cb + 4 : cb; }  // 16 columns: one 128-byte row per quarter-warp, no padding needed

template <int LOGM3>
__global__ void __launch_bounds__(512, 2) k_zstage(ZArgs a) {
  constexpr int M3 = 1 << LOGM3;
  const int zlog = a.lcb, zcb = 1 << a.lcb, P = fft_tfast_pitch(M3, zcb >> 1), PA = z_pitch(zcb);
  extern __shared__ float2 sm[];
  float2* Ain = sm;                                           // [np][PA]; the FFT works in place of it afterwards
  const int fftsz = (zcb >> 1) * P, ainsz = a.np * PA;
  float2* Gz = sm + ((max(fftsz, ainsz) + 1) & ~1);           // [nact][zcb] compact active cells
  const int ix2 = a.x2_0 + blockIdx.y, c0 = blockIdx.x * zcb;
  const size_t nn = a.a_pstride;
  const float2* Ab = a.A + (size_t)(ix2 - a.a_x2_0) * a.n + c0;
  {  // phase 1: 16-byte loads, four in flight per thread before the first store (the loads are latency-bound otherwise);
     // the remainder that does not fill a round of 4 loads per thread goes one load at a time
    const int hlog = zlog - 1, total = a.np << hlog, round = 4 * blockDim.x, tmain = total - total % round;
    auto src = [&](int idx) { return reinterpret_cast<const float4*>(Ab + (size_t)(idx >> hlog) * nn + 2 * (idx & ((1 << hlog) - 1))); };
    auto dst = [&](int idx) { return reinterpret_cast<float4*>(Ain + (idx >> hlog) * PA + 2 * (idx & ((1 << hlog) - 1))); };
    for (int base = threadIdx.x; base < tmain; base += round) {
      float4 v[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) v[u] = __ldg(src(base + u * blockDim.x));
#pragma unroll
      for (int u = 0; u < 4; ++u) *dst(base + u * blockDim.x) = v[u];
    }
    if (tmain < total) {  // one more, partly filled round
      const int base = tmain + threadIdx.x;
      float4 v[4];
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (base + u * blockDim.x < total) v[u] = __ldg(src(base + u * blockDim.x));
#pragma unroll
      for (int u = 0; u < 4; ++u)
        if (base + u * blockDim.x < total) *dst(base + u * blockDim.x) = v[u];
    }
  }
  __syncthreads();
  {
    const int hc = zcb >> 1, last = (a.np - 1) * PA;
    for (int task = threadIdx.x; task < a.nact * hc; task += blockDim.x) {
      const int j = task / hc, c2 = (task - j * hc) * 2;
      const int lo = __ldg(&a.zlo[j]), cnt = __ldg(&a.zcnt[j]);
      const float wl = __ldg(&a.zlast[j]);
      const float4 v = *reinterpret_cast<const float4*>(Ain + last + c2);
      float4 acc = make_float4(v.x * wl, v.y * wl, v.z * wl, v.w * wl);
      const float2* ap = Ain + lo * PA + c2;
      const float* wt = a.ztab + j;
      for (int s = 0; s < cnt; ++s) {
        const float wv = __ldg(&wt[(size_t)s * a.nact]);
        const float4 x = *reinterpret_cast<const float4*>(ap + s * PA);
        acc.x = fmaf(x.x, wv, acc.x);
        acc.y = fmaf(x.y, wv, acc.y);
        acc.z = fmaf(x.z, wv, acc.z);
        acc.w = fmaf(x.w, wv, acc.w);
      }
      *reinterpret_cast<float4*>(Gz + j * zcb + c2) = acc;
    }
  }
  __syncthreads();
  // Only the real part of the x3 transform is kept, and Re IFFT(G) = IFFT(H) with H[m] = (G[m] + conj G[-m]) / 2.  Two
  // columns a, b are packed into ONE complex transform of H_a + i H_b (real part -> column a, imaginary part -> column
  // b), which halves the FFT work and its shared memory.  The factor 1/2 is applied at the store.
  auto ld = [&](int t, int i) -> float2 {
    const int k1 = __ldg(&a.zidx[i]), k2 = __ldg(&a.zidx[(M3 - i) & (M3 - 1)]);
    const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
    const float4 u = k1 >= 0 ? *reinterpret_cast<const float4*>(Gz + k1 * zcb + 2 * t) : z;
    const float4 v = k2 >= 0 ? *reinterpret_cast<const float4*>(Gz + k2 * zcb + 2 * t) : z;
    // H_a = (u.xy + conj v.xy), H_b = (u.zw + conj v.zw);  H_a + i H_b
    return make_float2((u.x + v.x) - (u.w - v.w), (u.y - v.y) + (u.z + v.z));
  };
  const float dx2 = 0.5f * a.dx[ix2];
  const int hz = a.nz / 2;
  float* vb = a.vol + (size_t)(ix2 - a.vol_x2_0) * a.n + c0;
  auto st = [&](int t, int k, float2 v) {
    int ix3 = k < hz ? k + hz : k - (M3 - hz);
    if (k >= hz && k < M3 - hz) return;
    const float sc = a.dz[ix3] * dx2;
    *reinterpret_cast<float2*>(vb + (size_t)ix3 * a.zstride + 2 * t) = make_float2(v.x * sc * a.dx[c0 + 2 * t], v.y * sc * a.dx[c0 + 2 * t + 1]);
  };
  block_fft<LOGM3, +1, true, true>(sm, zcb >> 1, zlog - 1, P, a.tw, ld, st);
}

// ---------------------------------------------------------------------------------------------------------------
// x3 stage, sm_100a form: a PERSISTENT block walks its share of the (x2, column group) work items; the planes of the
// NEXT item are fetched by TMA (one cp.async.bulk.tensor box [planes][cb columns] per <= 256 planes of the 3-D tensor
// A[p][x2][x1], completion on an mbarrier) into the second half of a double buffer while the current item is gridded,
// transformed and stored, so the global-memory latency of phase 1 is off the critical path.  The staged rows are dense
// (cb * 8 bytes); phase 2 keeps them conflict-free by giving the 8 lanes of a quarter-warp ONE cell: hc = cb/2 column
// pairs x E = 8/hc interleaved tap phases (taps s = e, e + E, ...), i.e. 8 consecutive 16-byte chunks of E consecutive
// rows; the E partial sums are combined with shuffles.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  unsigned ok;
  do {
    asm volatile("{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
  } while (!ok);
}
__device__ __forceinline__ void tma_load_3d(unsigned dst, const void* tmap, int c0, int c1, int c2, unsigned bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
               ::"r"(dst), "l"(reinterpret_cast<unsigned long long>(tmap)), "r"(c0), "r"(c1), "r"(c2), "r"(bar) : "memory");
}

struct ZTmaArgs {
  ZArgs z;
  int ngx;        // column groups per x2 row (n / cb)
  int nitems;     // work items of this launch: rows * ngx
  int nbox, pbox; // planes are fetched as nbox boxes of pbox planes (pbox <= 256; rows beyond np are zero-filled)
  int bufelems;   // float2 elements of one half of the double buffer (>= nbox*pbox*cb and >= the FFT scratch)
};

template <int LOGM3>
__global__ void __launch_bounds__(640) k_zstage_tma(const __grid_constant__ CUtensorMap tmap, ZTmaArgs t) {
  constexpr int M3 = 1 << LOGM3;
  const ZArgs& a = t.z;
  const int zlog = a.lcb, zcb = 1 << a.lcb, hlog = zlog - 1, P = fft_tfast_pitch(M3, zcb >> 1);
  extern __shared__ __align__(128) unsigned char smraw[];
  float2* buf[2] = {reinterpret_cast<float2*>(smraw), reinterpret_cast<float2*>(smraw) + t.bufelems};
  float2* Gz = reinterpret_cast<float2*>(smraw) + 2 * (size_t)t.bufelems;  // [nact][zcb]
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(Gz + (size_t)a.nact * zcb);
  const unsigned bar[2] = {smem_u32(&bars[0]), smem_u32(&bars[1])};
  const unsigned txbytes = (unsigned)t.nbox * t.pbox * zcb * 8u;
  auto issue = [&](int item, int b) {  // one thread
    const int r = item / t.ngx, gx = item - r * t.ngx;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // the buffer was last touched through the generic proxy
    mbar_expect_tx(bar[b], txbytes);
    for (int q = 0; q < t.nbox; ++q)
      tma_load_3d(smem_u32(buf[b] + (size_t)q * t.pbox * zcb), &tmap, gx * zcb, a.x2_0 + r, q * t.pbox, bar[b]);
  };
  if (threadIdx.x == 0) {
    mbar_init(bar[0], 1);
    mbar_init(bar[1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  if (threadIdx.x == 0 && (int)blockIdx.x < t.nitems) issue(blockIdx.x, 0);
  const int hc = zcb >> 1, E = 8 >> hlog;  // zcb <= 16; for zcb = 16: E = 1 and a quarter-warp is one row
  int it = 0;
  for (int item = blockIdx.x; item < t.nitems; item += gridDim.x, ++it) {
    const int b = it & 1;
    if (threadIdx.x == 0 && item + (int)gridDim.x < t.nitems) issue(item + gridDim.x, b ^ 1);
    mbar_wait(bar[b], (it >> 1) & 1);
    const float2* Ain = buf[b];
    const int r = item / t.ngx, gx = item - r * t.ngx;
    const int ix2 = a.x2_0 + r, c0 = gx * zcb;
    {  // phase 2: task = (cell j, tap phase e, column pair c2); lanes: c2 fastest, then e, then j
      const int total = a.nact << 3, lastrow = (a.np - 1) * zcb;
      for (int base = 0; base < total; base += blockDim.x) {
        const int task = base + threadIdx.x;
        const bool valid = task < total;
        const int j = valid ? task >> 3 : 0, sub = task & 7, c2 = (sub & (hc - 1)) * 2, e = sub >> hlog;
        const int lo = __ldg(&a.zlo[j]), cnt = valid ? __ldg(&a.zcnt[j]) : 0;
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        if (e == 0 && valid) {
          const float wl = __ldg(&a.zlast[j]);
          const float4 v = *reinterpret_cast<const float4*>(Ain + lastrow + c2);
          acc = make_float4(v.x * wl, v.y * wl, v.z * wl, v.w * wl);
        }
        const float2* ap = Ain + lo * zcb + c2;
        const float* wt = a.ztab + j;
#pragma unroll 4
        for (int s = e; s < cnt; s += E) {
          const float wv = __ldg(&wt[(size_t)s * a.nact]);
          const float4 x = *reinterpret_cast<const float4*>(ap + s * zcb);
          acc.x = fmaf(x.x, wv, acc.x);
          acc.y = fmaf(x.y, wv, acc.y);
          acc.z = fmaf(x.z, wv, acc.z);
          acc.w = fmaf(x.w, wv, acc.w);
        }
        for (int m = hc; m < 8; m <<= 1) {  // combine the E tap phases (lane bits hlog .. 2)
          acc.x += __shfl_xor_sync(0xffffffffu, acc.x, m);
          acc.y += __shfl_xor_sync(0xffffffffu, acc.y, m);
          acc.z += __shfl_xor_sync(0xffffffffu, acc.z, m);
          acc.w += __shfl_xor_sync(0xffffffffu, acc.w, m);
        }
        if (valid && e == 0) *reinterpret_cast<float4*>(Gz + j * zcb + c2) = acc;
      }
    }
    __syncthreads();
    auto ld = [&](int tt, int i) -> float2 {  // two columns per complex transform (see k_zstage)
      const int k1 = __ldg(&a.zidx[i]), k2 = __ldg(&a.zidx[(M3 - i) & (M3 - 1)]);
      const float4 z = make_float4(0.f, 0.f, 0.f, 0.f);
      const float4 u = k1 >= 0 ? *reinterpret_cast<const float4*>(Gz + k1 * zcb + 2 * tt) : z;
      const float4 v = k2 >= 0 ? *reinterpret_cast<const float4*>(Gz + k2 * zcb + 2 * tt) : z;
      return make_float2((u.x + v.x) - (u.w - v.w), (u.y - v.y) + (u.z + v.z));
    };
    const float dx2 = 0.5f * a.dx[ix2];
    const int hz = a.nz / 2;
    float* vb = a.vol + (size_t)(ix2 - a.vol_x2_0) * a.n + c0;
    auto st = [&](int tt, int k, float2 v) {
      int ix3 = k < hz ? k + hz : k - (M3 - hz);
      if (k >= hz && k < M3 - hz) return;
      const float sc = a.dz[ix3] * dx2;
      __stcs(reinterpret_cast<float2*>(vb + (size_t)ix3 * a.zstride + 2 * tt), make_float2(v.x * sc * a.dx[c0 + 2 * tt], v.y * sc * a.dx[c0 + 2 * tt + 1]));
    };
    block_fft<LOGM3, +1, true, true>(buf[b], zcb >> 1, zlog - 1, P, a.tw, ld, st);
    __syncthreads();  // buf[b] (FFT scratch) and Gz are free again
  }
}

}  // namespace lam
