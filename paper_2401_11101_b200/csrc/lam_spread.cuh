// lam_spread.cuh — S2: gridding in (xi1, xi2) of one k_v plane.
//
// Plane p (k_v fixed): sample (theta, k_u) of Eq. 6, times M, sits at fine-grid position
//   t = a1 k_u (cos t, sin t) + rho (sin t, -cos t),   a1 = M/w,   rho = M k_v sin(phi)/h,
// i.e. on a straight equispaced line per theta, tangent to the circle of radius rho.  Every sample is spread with the
// separable width-W kernel onto the W x W cells around it (step 3 reversed), indices mod M
// (reading Q7).
//
// Work decomposition.  The plane is cut into kTS x kTS tiles.  A JOB is (tile, up to kJobRanges ranges of theta whose
// lines cross the tile); it is built once per plan from geometry alone (k_jobs).  One block of kSW warps owns the
// tile in shared memory.  A line is x-dominant (|cos| >= |sin|) or y-dominant; x-dominant lines are spread with
// "major axis" = x, y-dominant lines with major = y on the transposed tile (the tile is transposed in place between
// the two phases and back before the flush).
//
// Lane roles (the point of this kernel): lane L of warp w OWNS major-axis coordinate 32 w + L of the tile, i.e. one
// column of cells.  For the current line it walks the samples whose footprint covers its column (W/|a_M| = 3..5 of
// them), evaluates the major-axis weight of its column and the W minor-axis weights, and adds W taps into its own
// column with plain shared-memory read-modify-writes.  No two lanes ever touch the same cell, so there is nothing to
// synchronise inside a phase, no lane sits idle by construction, every (sample, column) pair is visited exactly once
// across the whole grid (only the minor axis has halo duplicates), and the 32 lanes of an instruction hit 32 distinct
// columns = distinct banks whatever rows they are in.  Tiles with one job are stored; tiles whose lines were split
// over several jobs (more than kJobMaxLines lines: the tiles around the xi3 axis, where every theta passes) are zeroed
// first (k_zero_tiles) and merged with red.global.add.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>

#include "lam_math.h"

namespace lam {

constexpr int kSW = 1;             // warps per job: one warp owns one 32 x 32 tile (wider jobs were measured slower)
constexpr int kTS = 32 * kSW;      // tile edge (fine-grid cells)
constexpr int kJobRanges = 6;      // theta ranges per job
constexpr int kJobMaxLines = 256;  // lines per job; a tile crossed by more lines is split over several jobs
constexpr int kRangeGap = 32;      // non-crossing thetas tolerated inside a range
constexpr int kRangeMaxLen = 2047; // 11 bits
constexpr int kMaxW = 8;

struct SpreadGeom {
  const double2* cs;   // [ntheta] (cos, sin) in double
  double rho_unit;     // M sin(phi) / h
  float a1;            // M / w
  int M, nt, ntheta, w, hh /* h/2 */;
};

// piecewise polynomial form of the gridding kernel (lam_math.h: kernel_poly)
struct KerPoly {
  float E[kMaxW / 2][kPolyHalf];
  float O[kMaxW / 2][kPolyHalf];
};

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

// job record, 32 bytes:
//   w[0] = tx | ty << 8 | p << 16 | multi << 29 | hasx << 30 | hasy << 31
//   w[1] = usex | usey << 3 | nranges << 6 | nlines << 9
//   w[2..7] = theta ranges: start | len << 14 | ydom << 25
struct Job {
  unsigned w[8];
};

// k range [ka, kb] of the samples of one line whose W x W footprint can reach the box [0, nM) x [0, nm) of cells.
// (oM, om): position of the k = 0 sample relative to the box's first cell; sample k sits at (oM, om) + a1 k (cM, cm).
// Conservative (margin 0.02 cells >> fp32 error of oM, om); exact clipping is per tap.
template <int W>
__device__ __forceinline__ void clip_box(float oM, float om, float cM, float cm, float a1, int hw, int nM, int nm, int& ka,
                                         int& kb) {
  const float lo0 = -0.5f * W - 0.02f, hiM = (float)(nM - 1) + 0.5f * W + 0.02f, him = (float)(nm - 1) + 0.5f * W + 0.02f;
  float lo = -a1 * hw, hi = a1 * hw;
  bool empty = false;
  if (fabsf(cM) > 1e-6f) {
    float r = 1.0f / cM, u0 = (lo0 - oM) * r, u1 = (hiM - oM) * r;
    lo = fmaxf(lo, fminf(u0, u1));
    hi = fminf(hi, fmaxf(u0, u1));
  } else if (oM < lo0 || oM > hiM) empty = true;
  if (fabsf(cm) > 1e-6f) {
    float r = 1.0f / cm, u0 = (lo0 - om) * r, u1 = (him - om) * r;
    lo = fmaxf(lo, fminf(u0, u1));
    hi = fminf(hi, fmaxf(u0, u1));
  } else if (om < lo0 || om > him) empty = true;
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
    float lo = s * (float)g.M - rmax, hi = s * (float)g.M + rmax;
    if (hi >= mx0 && lo <= mx0 + kTS - 1) candx |= 1 << (s + 1);
    if (hi >= my0 && lo <= my0 + kTS - 1) candy |= 1 << (s + 1);
  }
}

struct JobsArgs {
  SpreadGeom g;
  int p0, np;             // planes [p0, p0+np)
  unsigned* count;        // [np][nt*nt] jobs per tile (count pass: out; fill pass: in)
  unsigned* lines;        // [np][nt*nt] lines crossing the tile (count pass: out); bits 24..29: periodic images in use
  const unsigned* off;    // [np][nt*nt] first job of the tile in `jobs` (fill pass)
  Job* jobs;              // fill pass
};

// FILL = false: count jobs and lines per tile; FILL = true: write the job records.  One thread per (plane, tile).
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
  const int mx0 = tx * kTS - g.M / 2, my0 = ty * kTS - g.M / 2;
  int candx, candy;
  image_candidates(g, rho, mx0, my0, W, candx, candy);
  auto crosses = [&](int th, int mskx, int msky, int& hx, int& hy) {
    const double2 cs = g.cs[th];
    const float c = (float)cs.x, s = (float)cs.y;
    bool any = false;
    for (int sy = -1; sy <= 1; ++sy) {
      if (!(msky >> (sy + 1) & 1)) continue;
      const float oy = (float)(-rho * cs.x - my0 + (double)sy * g.M);
      for (int sx = -1; sx <= 1; ++sx) {
        if (!(mskx >> (sx + 1) & 1)) continue;
        const float ox = (float)(rho * cs.y - mx0 + (double)sx * g.M);
        // cheap exact-side rejection (99 % of all (tile, theta) pairs miss): the grown box of clip_box lies inside the
        // disc of radius sqrt(2) ((kTS - 1)/2 + W/2 + 0.02) around the tile centre; a line further away than that
        // (+0.05 for the fp32 rounding of ox, oy at |coordinates| <= 1e4) cannot have a sample in it
        constexpr float kHalf = 0.5f * (kTS - 1), kReach = 1.41421357f * (kHalf + 0.5f * W + 0.02f) + 0.05f;
        if (fabsf((kHalf - ox) * s - (kHalf - oy) * c) > kReach) continue;
        int ka, kb;
        clip_box<W>(ox, oy, c, s, g.a1, g.w / 2, kTS, kTS, ka, kb);
        if (ka <= kb) { hx |= 1 << (sx + 1); hy |= 1 << (sy + 1); any = true; }
      }
    }
    return any;
  };
  // which periodic images are ever hit (all jobs of the tile carry the same masks): the count pass tests every candidate
  // image and records the union in the top bits of `lines`; the fill pass reads it back and tests only those
  int usex = candx, usey = candy, seenx = 0, seeny = 0;
  if (FILL) {
    const unsigned m = a.lines[gid] >> 24;
    usex = m & 7;
    usey = (m >> 3) & 7;
  }
  // pass B: ranges of one orientation each, packed into jobs
  const unsigned total = FILL ? a.count[gid] : 0;
  Job* out = FILL ? a.jobs + a.off[gid] : nullptr;
  unsigned njobs = 0, nlines = 0;
  Job cur{};
  int nr = 0, jl = 0, hasx = 0, hasy = 0;
  auto emit_job = [&]() {
    if (FILL) {
      cur.w[0] = (unsigned)tx | (unsigned)ty << 8 | (unsigned)p << 16 | (total > 1 ? 1u << 29 : 0u) | (unsigned)hasx << 30 |
                 (unsigned)hasy << 31;
      cur.w[1] = (unsigned)usex | (unsigned)usey << 3 | (unsigned)nr << 6 | (unsigned)jl << 9;
      for (int i = nr; i < kJobRanges; ++i) cur.w[2 + i] = 0;
      out[njobs] = cur;
    }
    ++njobs;
    nr = 0; jl = 0; hasx = 0; hasy = 0;
  };
  int rs = -1, rlast = -1, ro = 0;
  auto close_range = [&]() {
    if (rs < 0) return;
    cur.w[2 + nr] = (unsigned)rs | (unsigned)(rlast + 1 - rs) << 14 | (unsigned)ro << 25;
    ++nr;
    if (ro) hasy = 1; else hasx = 1;
    rs = -1;
    if (nr == kJobRanges) emit_job();
  };
  if (usex && usey) {
    for (int th = 0; th < g.ntheta; ++th) {
      const double2 cs = g.cs[th];
      const int o = fabsf((float)cs.x) >= fabsf((float)cs.y) ? 0 : 1;
      const bool hit = crosses(th, usex, usey, seenx, seeny);
      if (rs >= 0 && (o != ro || (!hit && th - rlast > kRangeGap))) close_range();
      if (hit) {
        // a range may span up to kRangeGap misses between hits, so the length is checked BEFORE the hit is appended:
        // a length past the 11-bit field would spill into the ydom bit
        if (rs >= 0 && th + 1 - rs > kRangeMaxLen) close_range();
        if (rs < 0) { rs = th; ro = o; }
        rlast = th;
        ++jl;
        ++nlines;
        if (th + 1 - rs >= kRangeMaxLen) close_range();
        if (jl >= kJobMaxLines) { close_range(); if (nr > 0) emit_job(); }
      }
    }
    close_range();
    if (nr > 0) emit_job();
  }
  if (njobs == 0) emit_job();  // untouched tile: one job without ranges stores zeros
  if (!FILL) { a.count[gid] = njobs; a.lines[gid] = nlines | (unsigned)(seenx | seeny << 3) << 24; }
}

struct SpreadArgs {
  SpreadGeom g;
  KerPoly kp;
  const Job* jobs;        // jobs of this launch
  long long njobs;
  const float2* S;        // [h/2+1][ntheta][WQ]
  int WQ;
  float2* G;              // [planes in batch][M][M]
  int p0;                 // first plane of the batch
  const unsigned* multi;  // tiles of the batch's planes that several jobs write: p << 16 | ty << 8 | tx
  long long nmulti;
};

// zero the tiles that receive atomic adds from several jobs: one warp per entry
__global__ void k_zero_tiles(SpreadArgs a) {
  const int lane = threadIdx.x & 31;
  long long j = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  if (j >= a.nmulti) return;
  const unsigned e = a.multi[j];
  const int M = a.g.M;
  const int tx = e & 0xff, ty = (e >> 8) & 0xff, p = e >> 16;
  float4* Gp = reinterpret_cast<float4*>(a.G + (size_t)(p - a.p0) * M * M + (size_t)ty * kTS * M + tx * kTS);
  for (int i = lane; i < kTS * (kTS / 2); i += 32) {
    const int r = i / (kTS / 2), c = i - r * (kTS / 2);
    Gp[(size_t)r * (M / 2) + c] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
}

template <int OFF>
__device__ __forceinline__ float2 lds_f2(unsigned addr) {
  float2 r;
  asm volatile("ld.shared.v2.f32 {%0,%1}, [%2+%3];" : "=f"(r.x), "=f"(r.y) : "r"(addr), "n"(OFF) : "memory");
  return r;
}
template <int OFF>
__device__ __forceinline__ void sts_f2(unsigned addr, float2 v) {
  asm volatile("st.shared.v2.f32 [%0+%3], {%1,%2};" ::"r"(addr), "f"(v.x), "f"(v.y), "n"(OFF) : "memory");
}

template <int J, int N, class F>
__device__ __forceinline__ void static_for(F&& f) {
  if constexpr (J < N) {
    f(std::integral_constant<int, J>{});
    static_for<J + 1, N>(f);
  }
}

__host__ __device__ constexpr int j_off(int j) { return j * kTS * 8; }  // byte offset of tap row j in a tile column

struct LineParams {   // one line (theta, periodic image) clipped against a strip; 32 bytes
  float PM0, Pm0;     // position of sample ka relative to the strip's first cell (major, minor)
  float aM, am;       // step per sample
  float inv;          // 1 / aM
  int n;              // samples ka .. ka + n - 1
  int soff;           // index of sample ka inside the plane's spectra S[p]
  int pad;
};

// per-warp record of the <= 32 samples of the current line segment (what depends on the sample only, evaluated once
// per sample by lane = sample and read by the lanes = columns): value, minor-axis weights, first minor row + row mask
struct LineRec {
  float2 v[32];
  float wm[kMaxW][32];
  unsigned pk[32];   // (r0 & 0xff) | rowmask << 8
};

// dynamic shared memory of k_spread: tile + per-warp line parameters + per-warp sample records + kernel coefficients
constexpr size_t spread_smem() {
  return (size_t)kTS * kTS * 8 + (size_t)kSW * 32 * sizeof(LineParams) + (size_t)kSW * sizeof(LineRec) + 2 * (kMaxW / 2) * kPolyHalf * 4;
}

template <int W>
__global__ void __launch_bounds__(32 * kSW, 20) k_spread(SpreadArgs a) {
  extern __shared__ float2 smem[];
  float2* tile = smem;                                            // [kTS][kTS]: [minor][major]
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  LineParams* lp = reinterpret_cast<LineParams*>(smem + kTS * kTS) + wid * 32;
  LineRec* rec = reinterpret_cast<LineRec*>(reinterpret_cast<LineParams*>(smem + kTS * kTS) + kSW * 32) + wid;
  const SpreadGeom& g = a.g;
  const Job jb = a.jobs[blockIdx.x];
  const int tx = jb.w[0] & 0xff, ty = (jb.w[0] >> 8) & 0xff, p = (jb.w[0] >> 16) & 0x1fff;
  const bool multi = (jb.w[0] >> 29) & 1, hasx = (jb.w[0] >> 30) & 1, hasy = (jb.w[0] >> 31) & 1;
  const int usex = jb.w[1] & 7, usey = (jb.w[1] >> 3) & 7, nranges = (jb.w[1] >> 6) & 7;
  const int kv = p == g.hh ? -g.hh : p;
  const double rho = g.rho_unit * kv;
  const int mx0 = tx * kTS - g.M / 2, my0 = ty * kTS - g.M / 2;
  const int hw = g.w / 2;
  const int col = 32 * wid + lane;  // this lane's major-axis coordinate inside the tile
  const float fL = (float)lane;

  {
    float4* t4 = reinterpret_cast<float4*>(tile);
    for (int i = threadIdx.x; i < kTS * kTS / 2; i += 32 * kSW) t4[i] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  // polynomial coefficients (E_j[q], O_j[q]) of the kernel pieces, pinned in registers: read back from shared memory so
  // that the compiler cannot re-read the constant bank in every iteration
  float2 cEO[W / 2][kPolyHalf];
  {
    float* kps = reinterpret_cast<float*>(reinterpret_cast<LineRec*>(reinterpret_cast<LineParams*>(smem + kTS * kTS) + kSW * 32) + kSW);
    if (threadIdx.x < (kMaxW / 2) * kPolyHalf) {
      kps[threadIdx.x] = (&a.kp.E[0][0])[threadIdx.x];
      kps[(kMaxW / 2) * kPolyHalf + threadIdx.x] = (&a.kp.O[0][0])[threadIdx.x];
    }
    __syncthreads();
#pragma unroll
    for (int j = 0; j < W / 2; ++j)
#pragma unroll
      for (int q = 0; q < kPolyHalf; ++q)
        cEO[j][q] = make_float2(reinterpret_cast<volatile float*>(kps)[j * kPolyHalf + q],
                                reinterpret_cast<volatile float*>(kps)[(kMaxW / 2) * kPolyHalf + j * kPolyHalf + q]);
  }
  // (E_j(d^2), O_j(d^2)) of every half-tap j, packed: tap j has weight E_j + d O_j, tap W-1-j has E_j - d O_j
  auto pieces = [&](float d, float2 (&eo)[W / 2]) {
    const float d2 = d * d;
#pragma unroll
    for (int j = 0; j < W / 2; ++j) {
      eo[j] = cEO[j][kPolyHalf - 1];
#pragma unroll
      for (int q = kPolyHalf - 2; q >= 0; --q) eo[j] = __ffma2_rn(eo[j], make_float2(d2, d2), cEO[j][q]);
    }
  };

  const float2* Sp = a.S + (size_t)p * g.ntheta * a.WQ;
  const unsigned mycol_addr = (unsigned)__cvta_generic_to_shared(tile + col);

  for (int phase = 0; phase < 2; ++phase) {
    if (phase == 0 ? !hasx : !hasy) continue;
    const bool ydom = phase == 1;
    if (ydom && hasx) {  // transpose the tile in place: diagonal sweeps, both accesses of an instruction conflict-free
      __syncthreads();
      for (int r = 1; r <= kTS / 2; ++r) {
        const int i = threadIdx.x;
        if (2 * r == kTS && i >= kTS / 2) continue;
        int j = i + r;
        if (j >= kTS) j -= kTS;
        float2 u = tile[i * kTS + j], v = tile[j * kTS + i];
        tile[i * kTS + j] = v;
        tile[j * kTS + i] = u;
      }
      __syncthreads();
    }
#pragma unroll 1
    for (int ri = 0; ri < nranges; ++ri) {
      const unsigned rw = __ldg(&a.jobs[blockIdx.x].w[2 + ri]);
      if (((rw >> 25) & 1u) != (unsigned)phase) continue;
      const int rs = rw & 0x3fff, rend = rs + (int)((rw >> 14) & 0x7ff);
      for (int tb = rs; tb < rend; tb += 32) {
        const int th = tb + lane;
        const bool tvalid = th < rend;
        const double2 cs = tvalid ? g.cs[th] : make_double2(1.0, 0.0);
        const double cMd = ydom ? cs.y : cs.x, cmd = ydom ? cs.x : cs.y;
        const float cM = (float)cMd, cm = (float)cmd;
#pragma unroll 1
        for (int sy = -1; sy <= 1; ++sy) {
          if (!(usey >> (sy + 1) & 1)) continue;
          const double oyd = -rho * cs.x - my0 + (double)sy * g.M;
#pragma unroll 1
          for (int sx = -1; sx <= 1; ++sx) {
            if (!(usex >> (sx + 1) & 1)) continue;
            const double oxd = rho * cs.y - mx0 + (double)sx * g.M;
            const double oMd = (ydom ? oyd : oxd) - 32.0 * wid, omd = ydom ? oxd : oyd;
            int ka = 1, kb = 0;
            if (tvalid) clip_box<W>((float)oMd, (float)omd, cM, cm, g.a1, hw, 32, kTS, ka, kb);
            const bool hit = ka <= kb;
            // position of sample ka relative to the strip, in double (large terms cancel), then fp32
            const double u0 = (double)g.a1 * ka;
            const float aMl = g.a1 * cM;
            __syncwarp();
            reinterpret_cast<float4*>(lp + lane)[0] = make_float4((float)(oMd + u0 * cMd), (float)(omd + u0 * cmd), aMl, g.a1 * cm);
            reinterpret_cast<float4*>(lp + lane)[1] =
                make_float4(1.0f / aMl, __int_as_float(kb - ka + 1), __int_as_float(th * a.WQ + hw + ka), 0.f);
            unsigned mask = __ballot_sync(0xffffffffu, hit);
            __syncwarp();
            // lines of this batch one after the other.  Per line: (1) lane = sample evaluates what depends on the sample
            // only (minor-axis weights, rows) into the warp's record; (2) lane = column walks the samples covering its
            // column.  The samples of the NEXT line are fetched into a register while the current line is spread.
            int cur = -1;
            float2 vreg = make_float2(0.f, 0.f);
            if (mask) {
              cur = __ffs(mask) - 1;
              mask &= mask - 1;
              if (lane < lp[cur].n) vreg = __ldg(Sp + lp[cur].soff + lane);
            }
            while (cur >= 0) {
              const float4 q0 = reinterpret_cast<const float4*>(lp + cur)[0];
              const float4 q1 = reinterpret_cast<const float4*>(lp + cur)[1];
              const float PM0 = q0.x, Pm0 = q0.y, aM = q0.z, am = q0.w;
              const int n = __float_as_int(q1.y), soff = __float_as_int(q1.z);
              int nxt = -1;
              if (mask) {
                nxt = __ffs(mask) - 1;
                mask &= mask - 1;
              }
              const float uA = (fL - 0.5f * W - PM0) * q1.x, uB = (fL + 0.5f * W - PM0) * q1.x;
              const int is = max(0, (int)ceilf(fminf(uA, uB) - 1e-3f));
              const int ie = min(n - 1, (int)floorf(fmaxf(uA, uB) + 1e-3f));
              float2 vnext = make_float2(0.f, 0.f);
              for (int seg = 0; seg < n; seg += 32) {
                if (seg > 0) vreg = seg + lane < n ? __ldg(Sp + soff + seg + lane) : make_float2(0.f, 0.f);  // long runs (a1 < 2)
                __syncwarp();
                {  // (1) lane = sample seg + lane
                  const float Pm = fmaf((float)(seg + lane), am, Pm0);
                  const float xm = Pm - 0.5f * W, rf = ceilf(xm);
                  const int r0 = (int)rf;
                  float2 eo[W / 2];
                  const float dm = (xm - rf) + 0.5f;
                  pieces(dm, eo);
                  rec->v[lane] = vreg;
#pragma unroll
                  for (int j = 0; j < W / 2; ++j) {
                    rec->wm[j][lane] = fmaf(dm, eo[j].y, eo[j].x);
                    rec->wm[W - 1 - j][lane] = fmaf(-dm, eo[j].y, eo[j].x);
                  }
                  // bit j: row r0 + j is inside the tile (and the sample exists)
                  const int lo = min(max(-r0, 0), W), hi = min(max(kTS - r0, 0), W);
                  const unsigned rm = seg + lane < n ? ((1u << hi) - 1u) & ~((1u << lo) - 1u) : 0u;
                  rec->pk[lane] = ((unsigned)r0 & 0xffu) | rm << 8;
                }
                if (seg == 0 && nxt >= 0) vnext = lane < lp[nxt].n ? __ldg(Sp + lp[nxt].soff + lane) : make_float2(0.f, 0.f);
                __syncwarp();
                // (2) lane = column
                const int ls = max(is, seg), cnt = min(ie, seg + 31) - ls + 1;
                const int NI = __reduce_max_sync(0xffffffffu, cnt);
                if (NI <= 0) continue;
                auto prep = [&](int i, float2& vw, float (&wm)[W], unsigned& addr, unsigned& rm) {
                  const int k = min(ls - seg + i, 31);
                  const float PM = fmaf((float)(ls + i), aM, PM0);
                  const float xM = PM - 0.5f * W, cf = ceilf(xM);
                  const int j1 = lane - (int)cf;
                  const bool ok = i < cnt && (unsigned)j1 < (unsigned)W;
                  const float2 v = rec->v[k];
                  const unsigned pk = rec->pk[k];
#pragma unroll
                  for (int j = 0; j < W; ++j) wm[j] = rec->wm[j][k];
                  const float dM = (xM - cf) + 0.5f;
                  float2 eo[W / 2];
                  pieces(dM, eo);
                  // this lane's tap j1 of the sample
                  const int jj = j1 < W / 2 ? j1 : W - 1 - j1;
                  float2 es = eo[0];
#pragma unroll
                  for (int j = 1; j < W / 2; ++j) {
                    es.x = jj == j ? eo[j].x : es.x;
                    es.y = jj == j ? eo[j].y : es.y;
                  }
                  const float wM = fmaf(j1 < W / 2 ? dM : -dM, es.y, es.x);
                  vw = __fmul2_rn(v, make_float2(wM, wM));
                  const int r0 = (int)(signed char)(pk & 0xffu);
                  addr = mycol_addr + (unsigned)(r0 * (kTS * 8));
                  rm = ok ? pk >> 8 : 0u;
                };
#pragma unroll 1
                for (int i = 0; i < NI; ++i) {
                  float2 vw, c[W];
                  float wm[W];
                  unsigned addr, rm;
                  prep(i, vw, wm, addr, rm);
                  static_for<0, W>([&](auto J) {
                    if (rm >> J.value & 1u) c[J.value] = lds_f2<j_off(J.value)>(addr);
                  });
#pragma unroll
                  for (int j = 0; j < W; ++j) c[j] = __ffma2_rn(vw, make_float2(wm[j], wm[j]), c[j]);
                  static_for<0, W>([&](auto J) {
                    if (rm >> J.value & 1u) sts_f2<j_off(J.value)>(addr, c[J.value]);
                  });
                }
              }
              cur = nxt;
              vreg = vnext;
            }
            __syncwarp();
          }
        }
      }
    }
  }
  __syncthreads();
  if (hasy) {  // back to [y][x]
    for (int r = 1; r <= kTS / 2; ++r) {
      const int i = threadIdx.x;
      if (2 * r == kTS && i >= kTS / 2) continue;
      int j = i + r;
      if (j >= kTS) j -= kTS;
      float2 u = tile[i * kTS + j], v = tile[j * kTS + i];
      tile[i * kTS + j] = v;
      tile[j * kTS + i] = u;
    }
    __syncthreads();
  }
  const int M = g.M;
  float2* Gp = a.G + (size_t)(p - a.p0) * M * M + (size_t)ty * kTS * M + tx * kTS;
  if (!multi) {
    for (int r = 0; r < kTS; ++r) Gp[(size_t)r * M + threadIdx.x] = tile[r * kTS + threadIdx.x];
  } else {
    for (int r = 0; r < kTS; ++r) {
      const float2 v = tile[r * kTS + threadIdx.x];
      if (v.x != 0.f || v.y != 0.f) atomicAdd(&Gp[(size_t)r * M + threadIdx.x], v);
    }
  }
}

}  // namespace lam
