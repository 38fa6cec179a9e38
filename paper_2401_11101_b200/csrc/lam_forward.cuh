// lam_forward.cuh — kernels of lam_forward: proj = L vol, the exact transpose (over the reals) of lam_backproject
// with filter = none, stage by stage in reverse order (Eq. 5: L = F*_2D F_u3D; the USFFT steps of
// PAPER.md:136-138 in their forward order: division by the kernel transform, FFT, convolution-type interpolation).
// It serves the adjoint identity <L f, d> = <f, L* d> and is the forward model of lam_admm_tv.
//
//   k_zstage_T   (x3 stage)^T    vol * deapodisation -> zero-pad -> forward FFT along x3 -> interpolate at t3(k_v)
//   k_fft_x2_T   (k_ifft_x2)^T   zero-pad x2 (with the centring signs) -> forward FFT
//   k_fft_x1_T   (k_ifft_x1)^T   zero-pad x1 -> forward FFT                     -> fine-grid plane G^T
//   k_gather     (k_spread)^T    S^T[p][theta][q] = sum of W x W taps of G^T at the sample position (Eq. 6), tile-staged
//   k_cols_T     (k_cols)^T      un-fold the k_v >= 0 planes onto all h rows, inverse FFT along v
//   k_rows_T     (k_rows)^T      conj(Pu) * half spectrum -> inverse FFT along u -> real part
//
// Transposition rules used: a complex-linear map F becomes F^H (an unnormalised FFT of direction D becomes the
// unnormalised FFT of direction -D); y = Re(x) becomes x = y + 0i; g -> b conj(g) becomes s -> b conj(s); real
// weights stay.
#pragma once
#include "lam_kernels.cuh"
#include "lam_spread.cuh"

namespace lam {

struct ZTArgs {
  const float* vol;      // [nz][n][n]
  float2* A;             // [h/2+1][n][n]
  const float2* tw;      // length M3
  const float* wz;       // [h/2+1][W] tap weights of plane p
  const int* bz;         // [h/2+1] first tap m3 of plane p
  const float* dx;       // [n]
  const float* dz;       // [nz]
  int n, nz, np, W;
};

template <int LOGM3>
__global__ void __launch_bounds__(256) k_zstage_T(ZTArgs a) {
  constexpr int M3 = 1 << LOGM3, P = fft_tfast_pitch(M3, kZCb);
  extern __shared__ float2 sm[];
  const int ix2 = blockIdx.y, c0 = blockIdx.x * kZCb;
  const size_t nn = (size_t)a.n * a.n;
  const int hz = a.nz / 2;
  const float dx2 = a.dx[ix2];
  const float* vb = a.vol + (size_t)ix2 * a.n + c0;
  auto ld = [&](int t, int k) -> float2 {  // bin k of the zero-padded column: x3 = k (k < nz/2) or k - M3
    if (k >= hz && k < M3 - hz) return make_float2(0.f, 0.f);
    const int ix3 = k < hz ? k + hz : k - (M3 - hz);
    return make_float2(vb[(size_t)ix3 * nn + t] * a.dz[ix3] * dx2 * a.dx[c0 + t], 0.f);
  };
  block_fft<LOGM3, -1, true, false>(sm, kZCb, kZLog, P, a.tw, ld, [](int, int, float2) {});
  float2* Ab = a.A + (size_t)ix2 * a.n + c0;
  for (int idx = threadIdx.x; idx < a.np * kZCb; idx += blockDim.x) {
    const int p = idx >> kZLog, c = idx & (kZCb - 1);
    const int b = a.bz[p];
    float2 acc = make_float2(0.f, 0.f);
    for (int j = 0; j < a.W; ++j) {
      const float2 v = sm[c * P + fft_at<LOGM3>((b + j) & (M3 - 1))];
      const float wv = a.wz[p * a.W + j];
      acc.x = fmaf(v.x, wv, acc.x);
      acc.y = fmaf(v.y, wv, acc.y);
    }
    Ab[(size_t)p * nn + c] = acc;
  }
}

// (k_ifft_x2)^T: T^T[pl][i2][ix1] = sum_{kept k} e^{-2 pi i k i2/M} (-1)^k A^T[pl][ix(k)][ix1]
template <int LOGM>
__global__ void __launch_bounds__(512) k_fft_x2_T(IfftArgs a) {
  constexpr int M = 1 << LOGM;
  extern __shared__ float2 sm[];
  const int P = fft_tfast_pitch(M, a.nb);
  const int pl = blockIdx.y, c0 = blockIdx.x * a.nb;
  const int n = a.n, hn = a.n / 2;
  const float2* in = a.in + (size_t)pl * n * n + c0;   // A^T plane [n][n]
  float2* out = a.out + (size_t)pl * M * n + c0;       // T^T plane [M][n]
  auto ld = [&](int t, int k) -> float2 {
    if (k >= hn && k < M - hn) return make_float2(0.f, 0.f);
    const int ix = k < hn ? k + hn : k - (M - hn);
    float2 v = in[(size_t)ix * n + t];
    if (k & 1) { v.x = -v.x; v.y = -v.y; }
    return v;
  };
  auto st = [&](int t, int i, float2 v) { out[(size_t)i * n + t] = v; };
  block_fft<LOGM, -1, true, true>(sm, a.nb, a.lnb, P, a.tw, ld, st);
}

// (k_ifft_x1)^T: G^T[pl][i2][i1] = sum_{kept k} e^{-2 pi i k i1/M} (-1)^k T^T[pl][i2][ix(k)]
template <int LOGM>
__global__ void __launch_bounds__(256, 4) k_fft_x1_T(IfftArgs a) {
  constexpr int M = 1 << LOGM, P = fft_span(M);
  extern __shared__ float2 sm[];
  const int pl = blockIdx.y, r0 = blockIdx.x * a.nb;
  const int n = a.n, hn = a.n / 2;
  const float2* in = a.in + ((size_t)pl * M + r0) * n;   // T^T rows [M][n]
  float2* out = a.out + ((size_t)pl * M + r0) * M;       // G^T rows [M][M]
  auto ld = [&](int t, int k) -> float2 {
    if (k >= hn && k < M - hn) return make_float2(0.f, 0.f);
    const int ix = k < hn ? k + hn : k - (M - hn);
    float2 v = in[(size_t)t * n + ix];
    if (k & 1) { v.x = -v.x; v.y = -v.y; }
    return v;
  };
  auto st = [&](int t, int i, float2 v) { out[(size_t)t * M + i] = v; };
  block_fft<LOGM, -1, false, true>(sm, a.nb, 0, P, a.tw, ld, st);
}

// (k_spread)^T, tile-staged: the transpose of the gridding reads W x W cells of the fine-grid plane per sample.  The same
// work lists as k_spread are used (job = tile of plane p + the ranges of theta whose lines cross it): one warp stages the
// tile with its W - 1 halo on the high side in shared memory (coalesced rows of G^T, periodic wrap), clips every line of
// its ranges against the tile and lets lane = sample gather the samples whose FIRST tap cell lies inside the tile.  That
// cell comes from the absolute position in double, by the same formula in every tile, so every sample is owned by exactly
// one tile: plain stores, no atomics, and S^T needs no zeroing.  (The one-thread-per-sample form read its 36 taps from
// L2: 30 of the 57 ms of lam_forward on configs[2].)
struct GatherArgs {
  SpreadGeom g;
  KerPoly kp;
  const Job* jobs;   // the k_spread work list of this plane batch
  const float2* G;   // [planes in batch][M][M]
  float2* S;         // [h/2+1][ntheta][WQ]
  int WQ, p0;
};

template <int W>
__host__ __device__ constexpr int gather_pitch() { return ((kTS + W - 1) | 1); }  // odd pitch: rows start in different banks
template <int W>
__host__ __device__ constexpr size_t gather_smem() { return (size_t)(kTS + W - 1) * gather_pitch<W>() * sizeof(float2); }

template <int W>
__global__ void __launch_bounds__(32, 16) k_gather(GatherArgs a) {
  constexpr int TH = kTS + W - 1, TP = gather_pitch<W>();
  extern __shared__ float2 tile[];  // [TH][TP]
  const SpreadGeom& g = a.g;
  const int lane = threadIdx.x;
  const Job jb = a.jobs[blockIdx.x];
  const int tx = jb.w[0] & 0xff, ty = (jb.w[0] >> 8) & 0xff, p = (jb.w[0] >> 16) & 0x1fff;
  const int usex = jb.w[1] & 7, usey = (jb.w[1] >> 3) & 7, nranges = (jb.w[1] >> 6) & 7;
  if (nranges == 0) return;  // untouched tile: owns no sample
  const int kv = p == g.hh ? -g.hh : p;
  const double rho = g.rho_unit * kv;
  const int M = g.M, hw = g.w / 2;
  const int mx0 = tx * kTS - M / 2, my0 = ty * kTS - M / 2;
  {
    const float2* Gp = a.G + (size_t)(p - a.p0) * M * M;
    for (int i = lane; i < TH * TH; i += 32) {
      const int r = i / TH, c = i - r * TH;
      tile[r * TP + c] = __ldg(Gp + (size_t)((ty * kTS + r) & (M - 1)) * M + ((tx * kTS + c) & (M - 1)));
    }
  }
  __syncwarp();
  float2* Sp = a.S + (size_t)p * g.ntheta * a.WQ;
#pragma unroll 1
  for (int ri = 0; ri < nranges; ++ri) {
    const unsigned rw = jb.w[2 + ri];
    const int rs = rw & 0x3fff, rend = rs + (int)((rw >> 14) & 0x7ff);
    for (int tb = rs; tb < rend; tb += 32) {
      const int th = tb + lane;
      const bool tvalid = th < rend;
      const double2 cs = tvalid ? g.cs[th] : make_double2(1.0, 0.0);
#pragma unroll 1
      for (int sy = -1; sy <= 1; ++sy) {
        if (!(usey >> (sy + 1) & 1)) continue;
        const float oy = (float)(-rho * cs.x - my0 + (double)sy * M);
#pragma unroll 1
        for (int sx = -1; sx <= 1; ++sx) {
          if (!(usex >> (sx + 1) & 1)) continue;
          const float ox = (float)(rho * cs.y - mx0 + (double)sx * M);
          int ka = 1, kb = 0;
          if (tvalid) clip_box<W>(ox, oy, (float)cs.x, (float)cs.y, g.a1, hw, kTS, kTS, ka, kb);
          unsigned mask = __ballot_sync(0xffffffffu, ka <= kb);
          while (mask) {
            const int cur = __ffs(mask) - 1;
            mask &= mask - 1;
            const int thc = tb + cur, kac = __shfl_sync(0xffffffffu, ka, cur), kbc = __shfl_sync(0xffffffffu, kb, cur);
            const double cx = __shfl_sync(0xffffffffu, cs.x, cur), sn = __shfl_sync(0xffffffffu, cs.y, cur);
            for (int k = kac + lane; k <= kbc; k += 32) {
              const double u = (double)g.a1 * k;
              const double t1d = u * cx + rho * sn, t2d = u * sn - rho * cx;
              const double c1 = ceil(t1d - 0.5 * W), c2 = ceil(t2d - 0.5 * W);
              const int lx = ((int)c1 - mx0) & (M - 1), ly = ((int)c2 - my0) & (M - 1);
              if (lx >= kTS || ly >= kTS) continue;  // another tile owns this sample
              float w1[W], w2[W];
              kernel_weights<W>(a.kp, (float)(t1d - c1 - (0.5 * W - 0.5)), w1);
              kernel_weights<W>(a.kp, (float)(t2d - c2 - (0.5 * W - 0.5)), w2);
              const float2* t0 = tile + ly * TP + lx;
              float2 acc = make_float2(0.f, 0.f);
#pragma unroll
              for (int j2 = 0; j2 < W; ++j2) {
                float2 r = make_float2(0.f, 0.f);
#pragma unroll
                for (int j1 = 0; j1 < W; ++j1) r = __ffma2_rn(t0[j2 * TP + j1], make_float2(w1[j1], w1[j1]), r);
                acc = __ffma2_rn(r, make_float2(w2[j2], w2[j2]), acc);
              }
              Sp[(size_t)thc * a.WQ + hw + k] = acc;
            }
          }
        }
      }
    }
  }
}

// (k_cols)^T: for column k_u = k >= 0 of projection theta, C^T[p], p = 0..h-1, from the planes 0..h/2:
//   k_cols wrote  S[p][hw+k] = a_p C[p],  S[p][hw-k] = b_p conj(C[(h-p) mod h])  (k > 0),  a_p = Pv[p] wplus, b_p = Pv[p] wminus
//   so            C^T[p] = [p <= h/2] conj(a_p) S^T[p][hw+k] + [p' <= h/2, k > 0] b_p' conj(S^T[p'][hw-k]),  p' = (h-p) mod h
// then R^T[jv][k] = sum_p e^{+2 pi i p jv/h} C^T[p].
struct ColsTArgs {
  const float2* S;   // [h/2+1][ntheta][WQ]
  float2* R;         // [nth][h][WR]
  const float2* Pv;
  const float2* tw;
  int w, WR, WQ, ntheta, th0, lcb;
};

template <int LOGH>
__global__ void __launch_bounds__(512) k_cols_T(ColsTArgs a) {
  constexpr int h = 1 << LOGH;
  extern __shared__ float2 sm[];
  const int cb = 1 << a.lcb, P = fft_tfast_pitch(h, cb);
  const int thl = blockIdx.y, k0 = blockIdx.x * cb, hw = a.w / 2, th = a.th0 + thl;
  const int nc = min(cb, hw + 1 - k0);
  auto wts = [&](int p, int k, float& wplus, float& wminus) {
    const bool mid = p > 0 && p < h / 2;
    wplus = mid ? (k < hw ? 2.f : 1.f) : (k < hw ? 1.f : 0.f);
    wminus = mid ? (k < hw ? 2.f : 1.f) : 1.f;
  };
  auto ld = [&](int t, int p) -> float2 {
    float2 acc = make_float2(0.f, 0.f);
    if (t >= nc) return acc;
    const int k = k0 + t;
    if (p <= h / 2) {
      float wp, wm;
      wts(p, k, wp, wm);
      const float2 s = a.S[((size_t)p * a.ntheta + th) * a.WQ + hw + k], pv = a.Pv[p];
      const float2 ca = make_float2(pv.x * wp, -pv.y * wp);  // conj(a_p)
      acc = cmul(ca, s);
    }
    const int pp = (h - p) & (h - 1);
    if (pp <= h / 2 && k > 0) {
      float wp, wm;
      wts(pp, k, wp, wm);
      float2 s = a.S[((size_t)pp * a.ntheta + th) * a.WQ + hw - k];
      s.y = -s.y;
      const float2 pv = a.Pv[pp], b = make_float2(pv.x * wm, pv.y * wm);
      acc = cadd(acc, cmul(b, s));
    }
    return acc;
  };
  float2* Rb = a.R + (size_t)thl * h * a.WR + k0;
  auto st = [&](int t, int jv, float2 v) {
    if (t < nc) Rb[(size_t)jv * a.WR + t] = v;
  };
  block_fft<LOGH, +1, true, true>(sm, cb, a.lcb, P, a.tw, ld, st);
}

// (k_rows)^T: d^T[jv][ju] = Re sum_{k=0}^{w/2} conj(Pu[k]) R^T[jv][k] e^{+2 pi i k ju/w}
struct RowsTArgs {
  const float2* R;   // [nth][h][WR]
  float* proj;       // chunk base [nth][h][w]
  const float2* Pu;  // [w/2+1]
  const float2* tw;
  int h, WR, nb;     // nb rows per block
};

template <int LOGW>
__global__ void __launch_bounds__(256) k_rows_T(RowsTArgs a) {
  constexpr int w = 1 << LOGW, P = fft_span(w);
  extern __shared__ float2 sm[];
  const int th = blockIdx.y, r0 = blockIdx.x * a.nb;
  const float2* Rb = a.R + ((size_t)th * a.h + r0) * a.WR;
  float* out = a.proj + ((size_t)th * a.h + r0) * w;
  auto ld = [&](int t, int k) -> float2 {
    if (k > w / 2) return make_float2(0.f, 0.f);
    float2 pu = a.Pu[k];
    pu.y = -pu.y;
    return cmul(pu, Rb[(size_t)t * a.WR + k]);
  };
  auto st = [&](int t, int ju, float2 v) { out[(size_t)t * w + ju] = v.x; };
  block_fft<LOGW, +1, false, true>(sm, a.nb, 0, P, a.tw, ld, st);
}

}  // namespace lam
