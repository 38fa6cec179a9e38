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
__global__ void __launch_bounds__(256) k_rows(RowsArgs a) {
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
    if (c >= nc) return;
    int k = k0 + c;
    float2 cp = sm[c * P + fft_at<LOGH>(p)];
    float2 cm = sm[c * P + fft_at<LOGH>((h - p) & (h - 1))];
    cm.y = -cm.y;
    float2 pv = a.Pv[p];
    bool mid = p > 0 && p < h / 2;
    float wplus = mid ? (k < hw ? 2.f : 1.f) : (k < hw ? 1.f : 0.f);
    float wminus = mid ? (k < hw ? 2.f : 1.f) : 1.f;
    float2* Srow = a.S + ((size_t)p * a.ntheta + th) * a.WQ;
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
  auto ld = [&](int t, int i) -> float2 { return in[(size_t)t * M + i]; };
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
// x3 stage, one block per (x2, group of 2..8 x1): xi3 = k_v cos(phi)/h depends on k_v only (Eq. 6), so the planes
// A[p] are samples of a 1-D unequally spaced spectrum along x3 for every (x1, x2):
//   Gz[m3] = sum_p A[p] kap(t3(p) - m3),  t3 = M3 k_v cos(phi)/h;   vol[x3] = Re sum_m3 Gz[m3] e^{2 pi i x3 m3/M3}
//   divided by kaphat(x1/M) kaphat(x2/M) kaphat(x3/M3)  (PAPER.md:136 step 1, reversed per PAPER.md:140).
// The gridding is a banded matrix that is the same for every column.  Only the cells that some plane has a tap on
// are ACTIVE (about half of M3: the planes k_v >= 0 reach xi3 >= 0 only); for active cell j the planes with a tap on
// it are contiguous, [zlo[j], zlo[j] + zcnt[j]), with weights ztab[s][j]; the k_v = -h/2 plane (stored last) has its
// own weight zlast[j].  Three phases: (1) the block's columns of every plane are staged in shared memory (coalesced),
// (2) one thread per (active cell, column pair) accumulates the cell over its band: the weight is read once per tap
// and serves two columns, (3) the length-M3 inverse FFT reads the compact cells through the cell -> slot map zidx.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kZCb = 8, kZLog = 3;

struct ZArgs {
  const float2* A;       // [h/2+1][n][n]
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
__host__ __device__ constexpr int z_pitch(int cb) { return cb >= 8 ? cb + 4 : cb; }

template <int LOGM3>
__global__ void __launch_bounds__(512) k_zstage(ZArgs a) {
  constexpr int M3 = 1 << LOGM3;
  const int zlog = a.lcb, zcb = 1 << a.lcb, P = fft_tfast_pitch(M3, zcb), PA = z_pitch(zcb);
  extern __shared__ float2 sm[];
  float2* Ain = sm;                                           // [np][PA]; the FFT works in place of it afterwards
  const int fftsz = zcb * P, ainsz = a.np * PA;
  float2* Gz = sm + ((max(fftsz, ainsz) + 1) & ~1);           // [nact][zcb] compact active cells
  const int ix2 = a.x2_0 + blockIdx.y, c0 = blockIdx.x * zcb;
  const size_t nn = (size_t)a.n * a.n;
  const float2* Ab = a.A + (size_t)ix2 * a.n + c0;
  {  // phase 1: 16-byte loads, four in flight per thread before the first store (the loads are latency-bound otherwise)
    const int hlog = zlog - 1, total = a.np << hlog;
    for (int base = threadIdx.x; base < total; base += 4 * blockDim.x) {
      float4 v[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int idx = base + u * blockDim.x;
        if (idx < total) v[u] = __ldg(reinterpret_cast<const float4*>(Ab + (size_t)(idx >> hlog) * nn + 2 * (idx & ((1 << hlog) - 1))));
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int idx = base + u * blockDim.x;
        if (idx < total) *reinterpret_cast<float4*>(Ain + (idx >> hlog) * PA + 2 * (idx & ((1 << hlog) - 1))) = v[u];
      }
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
  auto ld = [&](int t, int i) -> float2 {
    const int k = __ldg(&a.zidx[i]);
    return k >= 0 ? Gz[k * zcb + t] : make_float2(0.f, 0.f);
  };
  const float dx2 = a.dx[ix2];
  const int hz = a.nz / 2;
  float* vb = a.vol + (size_t)(ix2 - a.vol_x2_0) * a.n + c0;
  auto st = [&](int t, int k, float2 v) {
    int ix3 = k < hz ? k + hz : k - (M3 - hz);
    if (k >= hz && k < M3 - hz) return;
    vb[(size_t)ix3 * a.zstride + t] = v.x * a.dz[ix3] * dx2 * a.dx[c0 + t];
  };
  block_fft<LOGM3, +1, true, true>(sm, zcb, zlog, P, a.tw, ld, st);
}

}  // namespace lam
