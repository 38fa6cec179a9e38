// lam_kernels.cuh — sm_100a kernels of the laminographic back-projection (see include/lam.h for the operator).
//
// Stage map (S-numbers are SURVEY.md §8(a) rows):
//   k_rows     S0+S1  -log prep, row FFT along u of two real rows per complex transform, filter H[k_u] (Eq. 3)
//   k_cols     S1     column FFT along v, Hermitian fold onto the k_v >= 0 planes, centring phases
//   k_jobs_*   S2     work-list builder: which (tile, theta-range) pairs of a k_v plane hold samples (geometry only)
//   k_spread   S2     gridding in (xi1, xi2): width-W kernel scatter of every sample of Eq. 6 onto its plane
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

// Tuning constants of k_spread, each chosen by same-box A/B timings on configs[2].
constexpr int kTile = 32;         // gridding tile edge (fine-grid cells owned by a job)
constexpr int kTP = 32;           // float2 elements per storage row in shared memory (a multiple of 16)
constexpr int kNU = 1;            // samples a lane spreads per step (4*kNU concurrent slots per warp)
constexpr bool kHalo = false;     // storage tile with a kernel halo (no per-tap bounds tests) or without (more warps)
constexpr int kStage = 64;        // samples of one line segment parked in shared memory
constexpr int kJobSegs = 32;      // target segments (theta crossings) per job
constexpr int kJobMaxSpan = 1023;       // max theta span of one job (10 bits)
constexpr int kMaxW = 8;

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
// S2: gridding in (xi1, xi2).  Plane p (k_v fixed): sample (theta, k_u) sits at fine-grid position
//   t = a1 k_u (cos t, sin t) + rho (sin t, -cos t),  a1 = M/w,  rho = M k_v sin(phi)/h      (Eq. 6 times M)
// i.e. on a straight line per theta, tangent to the circle of radius rho.  The plane is cut into 32x32 tiles; a
// job = (tile, theta-range); a warp owns a private shared-memory tile, walks the theta-range, clips every line
// against the tile (+ kernel halo, + periodic images, reading Q7), and lets lane i deposit sample k_a + i.
// ---------------------------------------------------------------------------------------------------------------
struct SpreadGeom {
  const double2* cs;   // [ntheta] (cos, sin) in double
  double rho_unit;     // M sin(phi) / h
  float a1;            // M / w
  int M, nt, ntheta, w, hh /* h/2 */, kstride;
};

struct KerPoly {
  float E[kMaxW / 2][kPolyHalf];
  float O[kMaxW / 2][kPolyHalf];
};

// job word layout: x = tx[0:9) ty[9:18) th0[18:32);  y = nth[0:10) mx[10:13) my[13:16) flags[16:18) p[18:31) ydom[31]
constexpr unsigned kJobExclusive = 1u, kJobFirstMulti = 2u;

__device__ __forceinline__ uint2 job_pack(int tx, int ty, int th0, int nth, int mx, int my, unsigned fl, int p, int ydom) {
  return make_uint2((unsigned)tx | ((unsigned)ty << 9) | ((unsigned)th0 << 18),
                    (unsigned)nth | ((unsigned)mx << 10) | ((unsigned)my << 13) | (fl << 16) | ((unsigned)p << 18) |
                        ((unsigned)ydom << 31));
}

// ku range [ka, kb] of the samples of one line whose kernel footprint can reach the tile.
// (ox, oy): line origin relative to the tile's first cell; the sample k sits at (ox, oy) + a1 k (c, s).
// Footprint test is conservative (margin 0.02 cells >> fp32 error of ox, oy); exact clipping is per tap.
template <int W>
__device__ __forceinline__ void clip_line(float ox, float oy, float c, float s, float a1, int hw, int& ka, int& kb) {
  const float xl = -0.5f * W - 0.02f, xh = (float)(kTile - 1) + 0.5f * W + 0.02f;
  float lo = -a1 * hw, hi = a1 * hw;
  bool empty = false;
  if (fabsf(c) > 1e-6f) {
    float r = 1.0f / c, u0 = (xl - ox) * r, u1 = (xh - ox) * r;
    lo = fmaxf(lo, fminf(u0, u1));
    hi = fminf(hi, fmaxf(u0, u1));
  } else if (ox < xl || ox > xh) empty = true;
  if (fabsf(s) > 1e-6f) {
    float r = 1.0f / s, u0 = (xl - oy) * r, u1 = (xh - oy) * r;
    lo = fmaxf(lo, fminf(u0, u1));
    hi = fminf(hi, fmaxf(u0, u1));
  } else if (oy < xl || oy > xh) empty = true;
  float ia = 1.0f / a1;
  ka = max(-hw, (int)ceilf(lo * ia - 1e-3f));
  kb = min(hw, (int)floorf(hi * ia + 1e-3f));
  if (empty) { ka = 1; kb = 0; }
}

// which periodic images (shifts of -M, 0, +M per axis) of the sample cloud can reach the tile: bit sx+1 / sy+1
__device__ __forceinline__ void image_candidates(const SpreadGeom& g, double rho, int mx0, int my0, int W, int& candx,
                                                 int& candy) {
  float rmax = sqrtf((float)(0.25 * (double)g.M * g.M + rho * rho)) + 0.5f * W + 1.0f;
  candx = 0;
  candy = 0;
  for (int s = -1; s <= 1; ++s) {
    // the image shifted by s*M covers [s*M - rmax, s*M + rmax]; the tile covers [m0, m0 + 31]
    float lo = s * (float)g.M - rmax, hi = s * (float)g.M + rmax;
    if (hi >= mx0 && lo <= mx0 + kTile - 1) candx |= 1 << (s + 1);
    if (hi >= my0 && lo <= my0 + kTile - 1) candy |= 1 << (s + 1);
  }
}

struct JobsArgs {
  SpreadGeom g;
  int p0, np;            // planes [p0, p0+np)
  unsigned* count;       // [np][nt*nt]
  const unsigned* off;   // [np][nt*nt] exclusive offsets within the chunk's job array (fill pass)
  uint2* jobs;           // chunk job array (fill pass)
};

// FILL = false: count jobs per tile; FILL = true: write them.  One thread per (plane, tile).
template <int W, bool FILL>
__global__ void k_jobs(JobsArgs a) {
  const SpreadGeom& g = a.g;
  const int ntiles = g.nt * g.nt;
  long long gid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (gid >= (long long)a.np * ntiles) return;
  const int pl = (int)(gid / ntiles), tile = (int)(gid - (long long)pl * ntiles);
  const int p = a.p0 + pl, ty = tile / g.nt, tx = tile - ty * g.nt;
  const int kv = p == g.hh ? -g.hh : p;
  const double rho = g.rho_unit * kv;
  const int mx0 = tx * kTile - g.M / 2, my0 = ty * kTile - g.M / 2;
  int candx, candy;
  image_candidates(g, rho, mx0, my0, W, candx, candy);
  // pass A: which images are ever hit (so that all jobs of the tile carry the same masks)
  int usex = 0, usey = 0;
  for (int th = 0; th < g.ntheta; ++th) {
    double2 cs = g.cs[th];
    float c = (float)cs.x, s = (float)cs.y;
    for (int sy = -1; sy <= 1; ++sy) {
      if (!(candy >> (sy + 1) & 1)) continue;
      float oy = (float)(-rho * cs.x - my0 + (double)sy * g.M);
      for (int sx = -1; sx <= 1; ++sx) {
        if (!(candx >> (sx + 1) & 1)) continue;
        float ox = (float)(rho * cs.y - mx0 + (double)sx * g.M);
        int ka, kb;
        clip_line<W>(ox, oy, c, s, g.a1, g.w / 2, ka, kb);
        if (ka <= kb) { usex |= 1 << (sx + 1); usey |= 1 << (sy + 1); }
      }
    }
  }
  // pass B: emit jobs; a job holds lines of one orientation only (|cos| >= |sin|: x-dominant, else y-dominant)
  unsigned njobs = 0;
  int start = -1, last = -1, cnt = 0, ori = 0;
  uint2* out = FILL ? a.jobs + a.off[gid] : nullptr;
  const unsigned total = FILL ? a.count[gid] : 0;
  auto emit = [&](int t0, int t1) {
    if (FILL) {
      unsigned fl = total == 1 ? kJobExclusive : (njobs == 0 ? kJobFirstMulti : 0u);
      out[njobs] = job_pack(tx, ty, t0, t1 - t0, usex, usey, fl, p, ori);
    }
    ++njobs;
  };
  if (usex && usey) {
    for (int th = 0; th < g.ntheta; ++th) {
      double2 cs = g.cs[th];
      float c = (float)cs.x, s = (float)cs.y;
      const int o = fabsf(c) >= fabsf(s) ? 0 : 1;
      bool hit = false;
      for (int sy = -1; sy <= 1 && !hit; ++sy) {
        if (!(usey >> (sy + 1) & 1)) continue;
        float oy = (float)(-rho * cs.x - my0 + (double)sy * g.M);
        for (int sx = -1; sx <= 1 && !hit; ++sx) {
          if (!(usex >> (sx + 1) & 1)) continue;
          float ox = (float)(rho * cs.y - mx0 + (double)sx * g.M);
          int ka, kb;
          clip_line<W>(ox, oy, c, s, g.a1, g.w / 2, ka, kb);
          hit = ka <= kb;
        }
      }
      if (start >= 0 && (o != ori || (!hit && th - last > 32))) {
        emit(start, last + 1);
        start = -1;
        cnt = 0;
      }
      if (hit) {
        if (start < 0) { start = th; ori = o; }
        ++cnt;
        last = th;
        if (cnt == kJobSegs || th + 1 - start >= kJobMaxSpan) { emit(start, th + 1); start = -1; cnt = 0; }
      }
    }
    if (start >= 0) emit(start, last + 1);
  }
  if (njobs == 0) { ori = 0; emit(0, 0); }  // untouched tile: one exclusive job that stores zeros
  if (!FILL) a.count[gid] = njobs;
}

__device__ __forceinline__ float2 lds_v(unsigned addr) {
  float2 r;
  asm volatile("ld.volatile.shared.v2.f32 {%0,%1}, [%2];" : "=f"(r.x), "=f"(r.y) : "r"(addr) : "memory");
  return r;
}
__device__ __forceinline__ void sts_v(unsigned addr, float2 v) {
  asm volatile("st.volatile.shared.v2.f32 [%0], {%1,%2};" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
}

template <int W>
__device__ __forceinline__ void kernel_weights(const KerPoly& kp, float d, float (&wt)[W]) {
  float d2 = d * d;
#pragma unroll
  for (int j = 0; j < W / 2; ++j) {
    float e = kp.E[j][3], o = kp.O[j][3];
#pragma unroll
    for (int q = 2; q >= 0; --q) {
      e = fmaf(e, d2, kp.E[j][q]);
      o = fmaf(o, d2, kp.O[j][q]);
    }
    wt[j] = fmaf(d, o, e);
    wt[W - 1 - j] = fmaf(-d, o, e);
  }
}

template <int W>
__device__ __forceinline__ void kernel_weights_r(const float (&E)[W / 2][kPolyHalf], const float (&O)[W / 2][kPolyHalf], float d,
                                                 float (&wt)[W]) {
  float d2 = d * d;
#pragma unroll
  for (int j = 0; j < W / 2; ++j) {
    float e = E[j][3], o = O[j][3];
#pragma unroll
    for (int q = 2; q >= 0; --q) {
      e = fmaf(e, d2, E[j][q]);
      o = fmaf(o, d2, O[j][q]);
    }
    wt[j] = fmaf(d, o, e);
    wt[W - 1 - j] = fmaf(-d, o, e);
  }
}

struct SpreadArgs {
  SpreadGeom g;
  KerPoly kp;
  const uint2* jobs;   // jobs of this launch
  long long njobs;
  const float2* S;     // [h/2+1][ntheta][WQ]
  int WQ;
  float2* G;           // [planes in batch][M][M]
  int p0;              // first plane of the batch
  const unsigned* multi;  // tiles of the batch's planes that several jobs write (k_zero_tiles)
  long long nmulti;
};

// zero the tiles that receive atomic adds from several jobs: one warp per entry of the plan's list of such tiles
// (entry = plane << 18 | ty << 9 | tx, built once from the job counts)
__global__ void k_zero_tiles(SpreadArgs a) {
  const int lane = threadIdx.x & 31;
  long long j = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (j >= a.nmulti) return;
  const unsigned e = a.multi[j];
  const int M = a.g.M;
  int tx = e & 0x1ff, ty = (e >> 9) & 0x1ff, p = e >> 18;
  float2* Gp = a.G + (size_t)(p - a.p0) * M * M;
  const int x0 = tx * kTile, y0 = ty * kTile;
  for (int r = 0; r < kTile && y0 + r < M; ++r)
    for (int c = lane; c < kTile && x0 + c < M; c += 32) Gp[(size_t)(y0 + r) * M + x0 + c] = make_float2(0.f, 0.f);
}

// Spreading of one job.  The warp owns a private storage tile [kTile][kTP] in shared memory; a sample is visited
// iff its W x W footprint meets the kTile x kTile cells, and every tap is bounds-tested against the tile (the variant
// with a kernel halo around the tile and no tests, kHalo, halves the resident warps and is slower).
//
// Lane roles: half-warp h holds two slots of W lanes; lane j of a slot owns tap column j of the slot's current
// sample (along the MAJOR axis: x for x-dominant lines, y for y-dominant lines, whose jobs work on the transposed
// tile) and walks the W taps of the minor axis.  The four slots take samples q apart on the same line,
// q = ceil(W / sqrt 2): their footprints are disjoint (no lost update inside one instruction), and for W = 6 the
// two runs of 6 contiguous cells of a half-warp sit 7..10 columns apart in rows whose pitch is a multiple of 16:
// 12 distinct banks per 128-byte wavefront, no conflicts by construction.
template <int W>
__global__ void __launch_bounds__(32) k_spread(SpreadArgs a) {
  extern __shared__ float2 tile[];
  constexpr int H = kHalo ? W - 1 : 0;               // low-side halo of the storage (0: taps are bounds-tested)
  constexpr int ROWS = kHalo ? kTile + 2 * W - 2 : kTile;
  const SpreadGeom& g = a.g;
  const int Q = g.kstride;  // sample distance between slots (footprints disjoint)
  const int lane = threadIdx.x;
  const long long jid = blockIdx.x;
  const unsigned tile_addr = (unsigned)__cvta_generic_to_shared(tile);
  const uint2 jb = a.jobs[jid];
  const int tx = jb.x & 0x1ff, ty = (jb.x >> 9) & 0x1ff, th0 = jb.x >> 18;
  const int nth = jb.y & 0x3ff, usex = (jb.y >> 10) & 7, usey = (jb.y >> 13) & 7;
  const unsigned flags = (jb.y >> 16) & 3u;
  const int p = (jb.y >> 18) & 0x1fff;
  const bool ydom = (jb.y >> 31) != 0;
  const int kv = p == g.hh ? -g.hh : p;
  const double rho = g.rho_unit * kv;
  const int mx0 = tx * kTile - g.M / 2, my0 = ty * kTile - g.M / 2;
  const int hw = g.w / 2;

  // lane role
  const int hl = lane & 15, slot2 = hl / W, j1 = hl - slot2 * W;
  const bool role = slot2 < 2;
  const int sidx = 2 * (lane >> 4) + slot2;
  const int slot_lane0 = role ? lane - j1 : lane;  // first lane of this lane's slot
  float cE[kPolyHalf], cO[kPolyHalf];  // this lane's major-axis tap polynomial: E(d^2) + d O(d^2)
  {
    const int jj = role ? min(j1, W - 1 - j1) : 0;
    const float sg = j1 < W / 2 ? 1.f : -1.f;
#pragma unroll
    for (int q = 0; q < kPolyHalf; ++q) {
      cE[q] = a.kp.E[jj][q];
      cO[q] = sg * a.kp.O[jj][q];
    }
  }

  for (int i = lane; i < ROWS * kTP; i += 32) tile[i] = make_float2(0.f, 0.f);
  float2* stg = tile + ROWS * kTP;  // [2][kStage] samples of the current / next line
  int sb = 0;
  __syncwarp();

  const float2* Sp = a.S + (size_t)p * g.ntheta * a.WQ;
  for (int tb = th0; tb < th0 + nth; tb += 32) {
    const int th = tb + lane;
    const bool tvalid = th < th0 + nth;
    double2 cs = tvalid ? g.cs[th] : make_double2(1.0, 0.0);
    const float c = (float)cs.x, s = (float)cs.y;
    for (int sy = -1; sy <= 1; ++sy) {
      if (!(usey >> (sy + 1) & 1)) continue;
      const double oyd = -rho * cs.x - my0 + (double)sy * g.M;
      for (int sx = -1; sx <= 1; ++sx) {
        if (!(usex >> (sx + 1) & 1)) continue;
        const double oxd = rho * cs.y - mx0 + (double)sx * g.M;
        int ka = 1, kb = 0;
        if (tvalid) clip_line<W>((float)oxd, (float)oyd, c, s, g.a1, hw, ka, kb);
        // position of sample ka relative to the tile, in double (large terms cancel), then fp32
        const double u0 = (double)g.a1 * ka;
        const float p0x = (float)(oxd + u0 * cs.x), p0y = (float)(oyd + u0 * cs.y);
        // major / minor axes of this job
        const float lM0 = ydom ? p0y : p0x, lm0 = ydom ? p0x : p0y, lcM = ydom ? s : c, lcm = ydom ? c : s;
        unsigned mask = __ballot_sync(0xffffffffu, ka <= kb);
        if (!mask) continue;
        // lines of this batch, one after the other; the samples of the NEXT line are fetched into registers while
        // the current line is spread, then parked in the staging buffer (double-buffered)
        int src = __ffs(mask) - 1;
        int ska = __shfl_sync(0xffffffffu, ka, src), n = __shfl_sync(0xffffffffu, kb, src) - ska + 1;
        const float2* Srow = Sp + (size_t)(tb + src) * a.WQ + hw + ska;
        stg[sb * kStage + lane] = lane < n ? __ldg(&Srow[lane]) : make_float2(0.f, 0.f);
        stg[sb * kStage + lane + 32] = lane + 32 < n ? __ldg(&Srow[lane + 32]) : make_float2(0.f, 0.f);
        while (true) {
          const float aM = g.a1 * __shfl_sync(0xffffffffu, lcM, src), am = g.a1 * __shfl_sync(0xffffffffu, lcm, src);
          const float M0 = __shfl_sync(0xffffffffu, lM0, src), m0 = __shfl_sync(0xffffffffu, lm0, src);
          mask &= mask - 1;
          const bool more = mask != 0;
          int nsrc = 0, nska = 0, nn = 0;
          const float2* nSrow = Srow;
          float2 nv0 = make_float2(0.f, 0.f), nv1 = nv0;
          if (more) {
            nsrc = __ffs(mask) - 1;
            nska = __shfl_sync(0xffffffffu, ka, nsrc);
            nn = __shfl_sync(0xffffffffu, kb, nsrc) - nska + 1;
            nSrow = Sp + (size_t)(tb + nsrc) * a.WQ + hw + nska;
            if (lane < nn) nv0 = __ldg(&nSrow[lane]);
            if (lane + 32 < nn) nv1 = __ldg(&nSrow[lane + 32]);
          }
          __syncwarp();
          for (int seg = 0; seg < n; seg += kStage) {
            if (seg > 0) {  // long lines (small a1): later segments are fetched in place
              __syncwarp();
              stg[sb * kStage + lane] = seg + lane < n ? __ldg(&Srow[seg + lane]) : make_float2(0.f, 0.f);
              stg[sb * kStage + lane + 32] = seg + lane + 32 < n ? __ldg(&Srow[seg + lane + 32]) : make_float2(0.f, 0.f);
              __syncwarp();
            }
            const int nseg = min(n - seg, kStage);
            // 4*kNU slots (kNU per lane) take samples Qe apart; one sweep of Qe steps covers the segment
            const int Qe = max(Q, (nseg + 4 * kNU - 1) / (4 * kNU));
#pragma unroll 1
            for (int it = 0; it < Qe; ++it) {
              float2 acc[kNU][W];
              float wm[kNU][W];
              float2 vw[kNU];
              unsigned ad[kNU];
              bool ok[kNU];
              int rw0[kNU];
#pragma unroll
              for (int u = 0; u < kNU; ++u) {
                const int kk = (sidx + 4 * u) * Qe + it;
                const float fk = (float)(seg + kk);
                const float tM = fmaf(fk, aM, M0), tm = fmaf(fk, am, m0);
                const float cf = ceilf(tM - 0.5f * W), rf = ceilf(tm - 0.5f * W);
                const int col0 = (int)cf, row0 = (int)rf;
                ok[u] = role && kk < nseg && (unsigned)(col0 + W - 1) < (unsigned)(kTile + W - 1) &&
                        (unsigned)(row0 + W - 1) < (unsigned)(kTile + W - 1);
                if (!kHalo) ok[u] = ok[u] && (unsigned)(col0 + j1) < (unsigned)kTile;  // this lane's tap column
                rw0[u] = row0;
                const float2 v = stg[sb * kStage + (kk & (kStage - 1))];
                // this lane's tap polynomial at both offsets: its own major-axis weight, and minor-axis weight j1
                // of the slot's sample, which the W lanes of the slot then exchange
                const float dM = tM - cf - (0.5f * W - 0.5f), dm = tm - rf - (0.5f * W - 0.5f);
                const float dM2 = dM * dM, dm2 = dm * dm;
                float eM = cE[3], oM = cO[3], em = cE[3], om = cO[3];
#pragma unroll
                for (int q = 2; q >= 0; --q) {
                  eM = fmaf(eM, dM2, cE[q]);
                  oM = fmaf(oM, dM2, cO[q]);
                  em = fmaf(em, dm2, cE[q]);
                  om = fmaf(om, dm2, cO[q]);
                }
                const float wM = fmaf(dM, oM, eM), wmine = fmaf(dm, om, em);
#pragma unroll
                for (int j2 = 0; j2 < W; ++j2) wm[u][j2] = __shfl_sync(0xffffffffu, wmine, slot_lane0 + j2);
                vw[u] = make_float2(v.x * wM, v.y * wM);
                ad[u] = tile_addr + (unsigned)((row0 + H) * kTP + col0 + H + j1) * 8u;
              }
#pragma unroll
              for (int u = 0; u < kNU; ++u)
#pragma unroll
                for (int j2 = 0; j2 < W; ++j2)
                  if (ok[u] && (kHalo || (unsigned)(rw0[u] + j2) < (unsigned)kTile)) acc[u][j2] = lds_v(ad[u] + j2 * (kTP * 8));
#pragma unroll
              for (int u = 0; u < kNU; ++u)
#pragma unroll
                for (int j2 = 0; j2 < W; ++j2) {
                  acc[u][j2].x = fmaf(vw[u].x, wm[u][j2], acc[u][j2].x);
                  acc[u][j2].y = fmaf(vw[u].y, wm[u][j2], acc[u][j2].y);
                }
#pragma unroll
              for (int u = 0; u < kNU; ++u)
#pragma unroll
                for (int j2 = 0; j2 < W; ++j2)
                  if (ok[u] && (kHalo || (unsigned)(rw0[u] + j2) < (unsigned)kTile)) sts_v(ad[u] + j2 * (kTP * 8), acc[u][j2]);
            }
          }
          if (!more) break;
          sb ^= 1;
          stg[sb * kStage + lane] = nv0;
          stg[sb * kStage + lane + 32] = nv1;
          src = nsrc;
          ska = nska;
          n = nn;
          Srow = nSrow;
        }
        __syncwarp();
      }
    }
  }
  __syncwarp();
  // y-dominant jobs worked on the transposed tile: transpose the owned square in place (diagonal sweeps: lane i swaps
  // (i, i+r) with (i+r, i); both accesses of an instruction touch distinct banks)
  if (ydom) {
    for (int r = 1; r <= kTile / 2; ++r) {
      for (int i = lane; i < kTile; i += 32) {
        if (2 * r == kTile && i >= kTile / 2) continue;
        int j = i + r;
        if (j >= kTile) j -= kTile;
        const unsigned a1 = tile_addr + (unsigned)((i + H) * kTP + j + H) * 8u;
        const unsigned a2 = tile_addr + (unsigned)((j + H) * kTP + i + H) * 8u;
        float2 u = lds_v(a1), v = lds_v(a2);
        sts_v(a1, v);
        sts_v(a2, u);
      }
    }
    __syncwarp();
  }
  const int M = g.M, x0 = tx * kTile, y0 = ty * kTile;
  float2* Gp = a.G + (size_t)(p - a.p0) * M * M;
  if (flags & kJobExclusive) {
    for (int r = 0; r < kTile && y0 + r < M; ++r)
      for (int cc = lane; cc < kTile && x0 + cc < M; cc += 32)
        Gp[(size_t)(y0 + r) * M + x0 + cc] = lds_v(tile_addr + (unsigned)((r + H) * kTP + cc + H) * 8u);
  } else {
    for (int r = 0; r < kTile && y0 + r < M; ++r)
      for (int cc = lane; cc < kTile && x0 + cc < M; cc += 32) {
        float2 v = lds_v(tile_addr + (unsigned)((r + H) * kTP + cc + H) * 8u);
        if (v.x != 0.f || v.y != 0.f) atomicAdd(&Gp[(size_t)(y0 + r) * M + x0 + cc], v);
      }
  }
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
// The gridding is a banded matrix that is the same for every column: for grid cell i the planes with a tap on it
// are contiguous, [zlo[i], zlo[i] + KZ), with weights ztab[i][KZ] (zero padded); the k_v = -h/2 plane (stored
// last) has its own weight zlast[i].  Cell values are computed on the fly by the loader of the first FFT pass.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kZCb = 8, kZLog = 3;

struct ZArgs {
  const float2* A;       // [h/2+1][n][n]
  float* vol;            // output buffer; element (ix3, ix2, ix1) at vol[ix3*zstride + (ix2 - vol_x2_0)*n + ix1]
  size_t zstride;
  const float2* tw;      // length M3
  const float* ztab;     // [M3][KZ]
  const int* zlo;        // [M3] first plane with a tap on cell i
  const int* zcnt;       // [M3] number of such planes (<= KZ)
  const float* zlast;    // [M3]
  const float* dx;       // [n]  1/kaphat(x/M)
  const float* dz;       // [nz] 1/kaphat(x3/M3)
  int n, nz, np, KZ, lcb;  // 1 << lcb columns per block
  int x2_0;              // first x2 row of this launch
  int vol_x2_0;          // x2 index held by row 0 of the output buffer
};

template <int LOGM3>
__global__ void __launch_bounds__(512) k_zstage(ZArgs a) {
  constexpr int M3 = 1 << LOGM3;
  const int zlog = a.lcb, zcb = 1 << a.lcb, P = fft_tfast_pitch(M3, zcb);  // columns per block
  extern __shared__ float2 sm[];
  float2* Gz = sm;                                // [8][P]
  float2* Ain = sm + zcb * P;                    // [np + KZ][zcb], the KZ extra planes are zero
  const int ix2 = a.x2_0 + blockIdx.y, c0 = blockIdx.x * zcb;
  const size_t nn = (size_t)a.n * a.n;
  const float2* Ab = a.A + (size_t)ix2 * a.n + c0;
  for (int idx = threadIdx.x; idx < (a.np + a.KZ) * zcb; idx += blockDim.x) {
    int p = idx >> zlog, c = idx & (zcb - 1);
    Ain[idx] = p < a.np ? Ab[(size_t)p * nn + c] : make_float2(0.f, 0.f);
  }
  __syncthreads();
  const int KZ = a.KZ, last = (a.np - 1) * zcb;
  auto ld = [&](int t, int i) -> float2 {
    const float* wt = a.ztab + (size_t)i * KZ;
    const float2* ap = Ain + __ldg(&a.zlo[i]) * zcb + t;
    float wl = __ldg(&a.zlast[i]);
    float2 v = Ain[last + t];
    float2 acc = make_float2(v.x * wl, v.y * wl);
    const int cnt = __ldg(&a.zcnt[i]);
    for (int s = 0; s < cnt; ++s) {
      float wv = __ldg(&wt[s]);
      float2 x = ap[s * zcb];
      acc.x = fmaf(x.x, wv, acc.x);
      acc.y = fmaf(x.y, wv, acc.y);
    }
    return acc;
  };
  const float dx2 = a.dx[ix2];
  const int hz = a.nz / 2;
  float* vb = a.vol + (size_t)(ix2 - a.vol_x2_0) * a.n + c0;
  auto st = [&](int t, int k, float2 v) {
    int ix3 = k < hz ? k + hz : k - (M3 - hz);
    if (k >= hz && k < M3 - hz) return;
    vb[(size_t)ix3 * a.zstride + t] = v.x * a.dz[ix3] * dx2 * a.dx[c0 + t];
  };
  block_fft<LOGM3, +1, true, true>(Gz, zcb, zlog, P, a.tw, ld, st);
}

}  // namespace lam
