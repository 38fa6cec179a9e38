// lam_oracle.cpp — CPU double-precision ORACLE for the laminographic filtered back-projection
// of arxiv 2401.11101.  TEST INFRASTRUCTURE ONLY.
//
//   * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
//     build, load or call this file.  The product path (paper_2401_11101_b200/) never does.
//   * It shares no code, header, table or constant generator with the CUDA path.
//   * Everything is plain loops in fp64; OpenMP only distributes independent outer iterations.
//
// What is here (citations are PAPER.md lines):
//   path A  orc_fbp_nudft      exact non-uniform DFT adjoint  = Eq. 7 with the filter of
//                              Eq. 3, frequencies of Eq. 6.
//                              THE PARITY DEFINITION.
//           orc_fbp_brute      the same sum as a straight quintuple loop, naive DFTs (tiny sizes).
//           orc_forward_nudft  Eq. 5, exact NUDFT forward, tiny sizes (adjoint test).
//   path B  orc_fbp_direct / orc_fp_direct   direct discretisation of Eq. 4 / Eq. 1 with linear
//                              interpolation ("Linerec") — sanity + O(N^4) baseline.
//           orc_fp_ray         Eq. 1-2 sampled along the beam, trilinear (ray-driven forward).
//   path C  orc_fbp_gridded    USFFT of PAPER.md:130-142 (gridding, inverse 3D FFT, division by psi).
//   path C' orc_fbp_gridded_slice   Eq. 9: exact x3 transform + 2D USFFT, one slice.
//           orc_prep           dark/flat/-log, model of PAPER.md:99.
// Pins: tests/test_oracle_*.py.  Path B: orc_fp_ray is pinned to analytic blob line integrals (P9b); the
// voxel-driven pair is pinned as a transpose pair, by mass conservation and against A at the interpolation-error
// level (a few per cent by construction: linear against trigonometric interpolation).  B is never a parity gate.
//
// Conventions: voxel x_a = i_a - n_a/2, detector u = j_u - c_u, v = j_v - c_v,
// k_u in [-w/2,w/2), k_v in [-h/2,h/2), xi = (k_u/w) e_u + (k_v/h) e_v (cycles/voxel),
// e_u = (cos t, sin t, 0), e_v = (sin t sin p, -cos t sin p, cos p)  [Eq. 2, PAPER.md:97],
// F f(xi) = int f e^{-2 pi i x xi}  [PAPER.md:113].
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cd;
static const double PI = 3.14159265358979323846264338327950288;

extern "C" {
typedef struct {
  int n, nz, h, w, ntheta;
  double phi;           // tilt, radians; phi = 0 is tomography (Eq. 2)
  const double* theta;  // ntheta rotation angles, radians
  double cu, cv;        // rotation-axis position on the detector, pixels (default w/2, h/2)
  int filter;           // 0 none (pure adjoint L*), 1 ramp (Ram-Lak), 2 Shepp-Logan
  int dtype;            // projections: 0 = float64, 1 = float32, 2 = uint16 raw (needs dark/flat)
  const float* dark;    // h*w, dtype 2 only
  const float* flat;    // h*w, dtype 2 only
  double tmin;          // transmission clamp for -log
  int pad;              // rows edge-extended to pad*w samples before the filter (reading Q11b); 0 or 1: none
  double alpha;         // 2-D spectral multiplier 1/(1 + alpha ((k_u/w)^2 + (k_v/h)^2)) on the projections; 0: none
} orc_geom;
}

static int max_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

// ---------------------------------------------------------------------------------------------
// 1-D DFTs.  X[k] = sum_j x[j] e^{sign * 2 pi i j k / n}, unnormalised, standard (uncentred) order.
// ---------------------------------------------------------------------------------------------
static void dft_naive(const cd* in, cd* out, int n, int sign) {
  for (int k = 0; k < n; ++k) {
    cd s = 0;
    for (int j = 0; j < n; ++j) {
      double a = sign * 2.0 * PI * (double)(((long long)j * k) % n) / n;
      s += in[j] * cd(cos(a), sin(a));
    }
    out[k] = s;
  }
}

static bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

// textbook iterative radix-2 Cooley-Tukey; every twiddle comes from cos/sin directly (no recurrence)
static void fft_pow2(cd* a, int n, int sign) {
  for (int i = 1, j = 0; i < n; ++i) {
    int bit = n >> 1;
    for (; j & bit; bit >>= 1) j ^= bit;
    j ^= bit;
    if (i < j) std::swap(a[i], a[j]);
  }
  for (int len = 2; len <= n; len <<= 1) {
    for (int i = 0; i < n; i += len) {
      for (int k = 0; k < len / 2; ++k) {
        double ang = sign * 2.0 * PI * k / len;
        cd w(cos(ang), sin(ang));
        cd u = a[i + k], v = a[i + k + len / 2] * w;
        a[i + k] = u + v;
        a[i + k + len / 2] = u - v;
      }
    }
  }
}

static void dft1(cd* a, int n, int sign) {
  if (is_pow2(n)) { fft_pow2(a, n, sign); return; }
  std::vector<cd> t(n);
  dft_naive(a, t.data(), n, sign);
  memcpy(a, t.data(), sizeof(cd) * n);
}

extern "C" void orc_dft1d(const double* in_ri, double* out_ri, int n, int sign, int naive) {
  std::vector<cd> a(n), b(n);
  for (int i = 0; i < n; ++i) a[i] = cd(in_ri[2 * i], in_ri[2 * i + 1]);
  if (naive) dft_naive(a.data(), b.data(), n, sign);
  else { b = a; dft1(b.data(), n, sign); }
  for (int i = 0; i < n; ++i) { out_ri[2 * i] = b[i].real(); out_ri[2 * i + 1] = b[i].imag(); }
}

// ---------------------------------------------------------------------------------------------
// S0: projection theta as line integrals in double.  PAPER.md:99:  raw = e^{-d}(flat-dark)+dark
//   =>  d = -log( (raw-dark)/(flat-dark) ), with the clamps of DESIGN.md reading Q12.
// ---------------------------------------------------------------------------------------------
static void load_proj(const orc_geom& g, const void* proj, int th, double* out) {
  size_t npx = (size_t)g.h * g.w, off = (size_t)th * npx;
  if (g.dtype == 0) {
    const double* p = (const double*)proj + off;
    for (size_t i = 0; i < npx; ++i) out[i] = p[i];
  } else if (g.dtype == 1) {
    const float* p = (const float*)proj + off;
    for (size_t i = 0; i < npx; ++i) out[i] = (double)p[i];
  } else {
    const uint16_t* p = (const uint16_t*)proj + off;
    for (size_t i = 0; i < npx; ++i) {
      double den = (double)g.flat[i] - (double)g.dark[i];
      if (den < 1.0) den = 1.0;
      double t = ((double)p[i] - (double)g.dark[i]) / den;
      if (t < g.tmin) t = g.tmin;
      out[i] = -log(t);
    }
  }
}

extern "C" void orc_prep(const orc_geom* g, const void* proj, int th, double* out) {
  load_proj(*g, proj, th, out);
}

// ---------------------------------------------------------------------------------------------
// Filter W of Eq. 3: "a suitable scaled version of |sigma| cos(phi)".
// Reading Q3: H[k_u] = (pi cos(phi)/N_theta) * DFT_w(h)[k_u], h = the band-limited
// spatial ramp kernel at unit pitch (Ram-Lak: h[0]=1/4, h[odd j]=-1/(pi j)^2, h[even j]=0;
// Shepp-Logan: h[j] = -2/(pi^2 (4 j^2 - 1))), j in [-w/2, w/2).  filter 0: H = 1.
// Output Hk[k_u + w/2], real.
// ---------------------------------------------------------------------------------------------
static double ramp_kernel(int filter, int j) {
  if (filter == 1 || filter == 3) {
    if (j == 0) return 0.25;
    if (j % 2 == 0) return 0.0;
    return -1.0 / (PI * PI * (double)j * (double)j);
  }
  return -2.0 / (PI * PI * (4.0 * (double)j * (double)j - 1.0));
}

// Parzen (de la Vallee Poussin) window, "low pass filters (shepp-logan, parzen)"; reading Q15: the ramp
// response times P(x), x = |k_u| / (len/2) in [0, 1] (1 = Nyquist):
//   P(x) = 1 - 6 x^2 + 6 x^3  (x <= 1/2),   2 (1 - x)^3  (1/2 < x <= 1).
static double parzen(double x) {
  x = fabs(x);
  if (x <= 0.5) return 1.0 - 6.0 * x * x + 6.0 * x * x * x;
  if (x <= 1.0) return 2.0 * (1.0 - x) * (1.0 - x) * (1.0 - x);
  return 0.0;
}

// filter response for rows of `len` samples (len = w, or pad*w for padded rows): Hk[k + len/2], k in [-len/2, len/2)
static void make_filter_len(const orc_geom& g, int len, double* Hk) {
  if (g.filter == 0) { for (int i = 0; i < len; ++i) Hk[i] = 1.0; return; }
  double scale = PI * cos(g.phi) / g.ntheta;
  for (int ku = -len / 2; ku < len - len / 2; ++ku) {
    cd s = 0;
    for (int j = -len / 2; j < len - len / 2; ++j) {
      double a = -2.0 * PI * (double)(((long long)ku * j) % len) / len;
      s += ramp_kernel(g.filter, j) * cd(cos(a), sin(a));
    }
    Hk[ku + len / 2] = scale * s.real();
    if (g.filter == 3) Hk[ku + len / 2] *= parzen((double)ku / (0.5 * len));
  }
}

static void make_filter(const orc_geom& g, double* Hk) { make_filter_len(g, g.w, Hk); }

extern "C" void orc_filter(const orc_geom* g, double* Hk) { make_filter(*g, Hk); }

// ---------------------------------------------------------------------------------------------
// F_2D of Eq. 7 on one projection, centred in both domains, times the filter:
//   HD[k_v+h/2][k_u+w/2] = H[k_u] (1/(w h)) sum_{j_v,j_u} d[j_v][j_u] e^{-2 pi i (k_u u/w + k_v v/h)},
//   u = j_u - c_u, v = j_v - c_v.
// Rows then columns with the 1-D DFT above; the centring is the phase e^{+2 pi i k c / n}.
// ---------------------------------------------------------------------------------------------
// Reading Q11b (u-padding, PAPER.md is silent): with g.pad > 1 every detector row is extended to pad*w samples by
// replicating its two edge values ((pad-1) w / 2 samples on each side), filtered as a row of that length (the filter
// response of the longer row, so that the convolution with the ramp kernel no longer wraps around the detector) and
// cropped back to its w samples.  q[j_v][j_u], filter included.
static void filter_rows_padded(const orc_geom& g, const double* d, double* q) {
  int h = g.h, w = g.w, wp = g.pad * w, off = (wp - w) / 2;
  std::vector<double> Hp(wp);
  make_filter_len(g, wp, Hp.data());
#pragma omp parallel for schedule(static)
  for (int jv = 0; jv < h; ++jv) {
    std::vector<cd> row(wp);
    for (int j = 0; j < wp; ++j) {
      int ju = j - off;
      ju = ju < 0 ? 0 : (ju >= w ? w - 1 : ju);
      row[j] = d[(size_t)jv * w + ju];
    }
    dft1(row.data(), wp, -1);
    for (int k = -wp / 2; k < wp - wp / 2; ++k) row[(k + wp) % wp] *= Hp[k + wp / 2];
    dft1(row.data(), wp, +1);
    for (int ju = 0; ju < w; ++ju) q[(size_t)jv * w + ju] = row[ju + off].real() / wp;
  }
}

extern "C" void orc_filter_rows_padded(const orc_geom* g, const void* proj, int th, double* q) {
  std::vector<double> d((size_t)g->h * g->w);
  load_proj(*g, proj, th, d.data());
  filter_rows_padded(*g, d.data(), q);
}

static void spectrum(const orc_geom& g, const double* d_in, const double* Hk_in, cd* HD) {
  int h = g.h, w = g.w;
  std::vector<cd> tmp((size_t)h * w);
  // padded rows: the filter has been applied in the space domain already, the transform below runs with H = 1
  std::vector<double> qpad, ones;
  const double* d = d_in;
  const double* Hk = Hk_in;
  if (g.pad > 1 && g.filter != 0) {
    qpad.resize((size_t)h * w);
    filter_rows_padded(g, d_in, qpad.data());
    ones.assign(w, 1.0);
    d = qpad.data();
    Hk = ones.data();
  }
#pragma omp parallel for schedule(static)
  for (int jv = 0; jv < h; ++jv) {
    std::vector<cd> row(w);
    for (int ju = 0; ju < w; ++ju) row[ju] = d[(size_t)jv * w + ju];
    dft1(row.data(), w, -1);
    for (int ku = -w / 2; ku < w - w / 2; ++ku) {
      double a = 2.0 * PI * ku * g.cu / w;
      tmp[(size_t)jv * w + (ku + w / 2)] = row[(ku + w) % w] * cd(cos(a), sin(a)) * Hk[ku + w / 2];
    }
  }
#pragma omp parallel for schedule(static)
  for (int iu = 0; iu < w; ++iu) {
    std::vector<cd> col(h);
    for (int jv = 0; jv < h; ++jv) col[jv] = tmp[(size_t)jv * w + iu];
    dft1(col.data(), h, -1);
    for (int kv = -h / 2; kv < h - h / 2; ++kv) {
      double a = 2.0 * PI * kv * g.cv / h;
      HD[(size_t)(kv + h / 2) * w + iu] = col[(kv + h) % h] * cd(cos(a), sin(a)) / ((double)w * h);
    }
  }
  // 2-D spectral multiplier on the projection (PAPER.md:199, 279 name Paganin filtering as a pre-processing step; the
  // single-distance Paganin filter is the low-pass 1/(1 + alpha |k|^2); reading Q17: applied to the line integrals)
  if (g.alpha != 0.0) {
    for (int kv = -h / 2; kv < h - h / 2; ++kv)
      for (int ku = -w / 2; ku < w - w / 2; ++ku) {
        double fu = (double)ku / w, fv = (double)kv / h;
        HD[(size_t)(kv + h / 2) * w + (ku + w / 2)] /= 1.0 + g.alpha * (fu * fu + fv * fv);
      }
  }
}

extern "C" void orc_spectrum(const orc_geom* g, const void* proj, int th, double* HD_ri) {
  std::vector<double> d((size_t)g->h * g->w), Hk(g->w);
  load_proj(*g, proj, th, d.data());
  make_filter(*g, Hk.data());
  spectrum(*g, d.data(), Hk.data(), (cd*)HD_ri);
}

// ---------------------------------------------------------------------------------------------
// PATH A — exact NUDFT adjoint (the definition the GPU is compared with):
//   vol[x] = Re sum_theta sum_{k_v,k_u} HD[theta,k_v,k_u] e^{+2 pi i x . xi(theta,k_u,k_v)}     (Eq. 7)
// evaluated for a list of x3-columns (i1,i2).  With x.xi = k_u u'/w + k_v v'/h,
//   u' = x.e_u (independent of x3), v' = x.e_v = v0 + x3 cos(phi),
// the sum over k_u is done once per column and angle; the sum over k_v once per voxel.
// The phase table Z[x3][k_v] = e^{2 pi i x3 k_v cos(phi)/h} depends on neither theta nor the column.
// out_re / out_im: [ncols][nz]  (out_im may be NULL).
// ---------------------------------------------------------------------------------------------
extern "C" void orc_fbp_nudft(const orc_geom* gp, const void* proj, int ncols, const int* cols,
                              double* out_re, double* out_im) {
  const orc_geom& g = *gp;
  int h = g.h, w = g.w, nz = g.nz;
  std::vector<double> Hk(w), d((size_t)h * w);
  make_filter(g, Hk.data());
  std::vector<cd> HD((size_t)h * w), Z((size_t)nz * h), acc((size_t)ncols * nz, cd(0, 0));
  for (int i3 = 0; i3 < nz; ++i3)
    for (int kv = -h / 2; kv < h - h / 2; ++kv) {
      double a = 2.0 * PI * (i3 - nz / 2) * kv * cos(g.phi) / h;
      Z[(size_t)i3 * h + kv + h / 2] = cd(cos(a), sin(a));
    }
  for (int th = 0; th < g.ntheta; ++th) {
    load_proj(g, proj, th, d.data());
    spectrum(g, d.data(), Hk.data(), HD.data());
    double ct = cos(g.theta[th]), st = sin(g.theta[th]), sp = sin(g.phi);
#pragma omp parallel for schedule(dynamic, 4)
    for (int c = 0; c < ncols; ++c) {
      double x1 = cols[2 * c] - g.n / 2, x2 = cols[2 * c + 1] - g.n / 2;
      double up = x1 * ct + x2 * st;             // x . e_u
      double v0 = x1 * st * sp - x2 * ct * sp;   // x . e_v at x3 = 0
      std::vector<cd> pu(w), E(h);
      for (int ku = -w / 2; ku < w - w / 2; ++ku) {
        double a = 2.0 * PI * ku * up / w;
        pu[ku + w / 2] = cd(cos(a), sin(a));
      }
      for (int kv = -h / 2; kv < h - h / 2; ++kv) {
        cd s = 0;
        const cd* r = &HD[(size_t)(kv + h / 2) * w];
        for (int iu = 0; iu < w; ++iu) s += r[iu] * pu[iu];
        double a = 2.0 * PI * kv * v0 / h;
        E[kv + h / 2] = s * cd(cos(a), sin(a));
      }
      for (int i3 = 0; i3 < nz; ++i3) {
        cd s = 0;
        const cd* z = &Z[(size_t)i3 * h];
        for (int iv = 0; iv < h; ++iv) s += E[iv] * z[iv];
        acc[(size_t)c * nz + i3] += s;
      }
    }
  }
  for (size_t i = 0; i < acc.size(); ++i) {
    out_re[i] = acc[i].real();
    if (out_im) out_im[i] = acc[i].imag();
  }
}

// The same sum with nothing factored: naive 2-D DFT of every projection and one complex exponential
// per (voxel, angle, k_v, k_u), xi written exactly as Eq. 6.  Tiny sizes only.
// vol[i3][i2][i1].
extern "C" void orc_fbp_brute(const orc_geom* gp, const void* proj, double* vol) {
  const orc_geom& g = *gp;
  int h = g.h, w = g.w, n = g.n, nz = g.nz;
  std::vector<double> Hk(w), d((size_t)h * w);
  make_filter(g, Hk.data());
  std::vector<cd> HD((size_t)g.ntheta * h * w);
  for (int th = 0; th < g.ntheta; ++th) {
    load_proj(g, proj, th, d.data());
    for (int kv = -h / 2; kv < h - h / 2; ++kv)
      for (int ku = -w / 2; ku < w - w / 2; ++ku) {
        cd s = 0;
        for (int jv = 0; jv < h; ++jv)
          for (int ju = 0; ju < w; ++ju) {
            double a = -2.0 * PI * (ku * (ju - g.cu) / w + kv * (jv - g.cv) / h);
            s += d[(size_t)jv * w + ju] * cd(cos(a), sin(a));
          }
        HD[((size_t)th * h + kv + h / 2) * w + ku + w / 2] = Hk[ku + w / 2] * s / ((double)w * h);
      }
  }
#pragma omp parallel for collapse(2) schedule(static)
  for (int i3 = 0; i3 < nz; ++i3)
    for (int i2 = 0; i2 < n; ++i2)
      for (int i1 = 0; i1 < n; ++i1) {
        double x1 = i1 - n / 2, x2 = i2 - n / 2, x3 = i3 - nz / 2;
        cd s = 0;
        for (int th = 0; th < g.ntheta; ++th) {
          double ct = cos(g.theta[th]), st = sin(g.theta[th]), cp = cos(g.phi), sp = sin(g.phi);
          for (int kv = -h / 2; kv < h - h / 2; ++kv)
            for (int ku = -w / 2; ku < w - w / 2; ++ku) {
              double fu = (double)ku / w, fv = (double)kv / h;
              double xi1 = fu * ct + fv * st * sp;   // Eq. 6
              double xi2 = fu * st - fv * ct * sp;
              double xi3 = fv * cp;
              double a = 2.0 * PI * (x1 * xi1 + x2 * xi2 + x3 * xi3);
              s += HD[((size_t)th * h + kv + h / 2) * w + ku + w / 2] * cd(cos(a), sin(a));
            }
        }
        vol[((size_t)i3 * n + i2) * n + i1] = s.real();
      }
}

// Eq. 5 forward, exact NUDFT, no filter:
//   L f[theta,j_v,j_u] = Re (1/(w h)) sum_{k_u,k_v} e^{+2 pi i (k_u u/w + k_v v/h)} sum_x f[x] e^{-2 pi i x.xi}
// Tiny sizes only (cost n^2 nz w h N_theta).  proj[theta][j_v][j_u].
extern "C" void orc_forward_nudft(const orc_geom* gp, const double* vol, double* proj) {
  const orc_geom& g = *gp;
  int h = g.h, w = g.w, n = g.n, nz = g.nz;
#pragma omp parallel for schedule(dynamic, 1)
  for (int th = 0; th < g.ntheta; ++th) {
    double ct = cos(g.theta[th]), st = sin(g.theta[th]), cp = cos(g.phi), sp = sin(g.phi);
    std::vector<cd> F((size_t)h * w);
    for (int kv = -h / 2; kv < h - h / 2; ++kv)
      for (int ku = -w / 2; ku < w - w / 2; ++ku) {
        double fu = (double)ku / w, fv = (double)kv / h;
        double xi1 = fu * ct + fv * st * sp, xi2 = fu * st - fv * ct * sp, xi3 = fv * cp;
        cd s = 0;
        for (int i3 = 0; i3 < nz; ++i3)
          for (int i2 = 0; i2 < n; ++i2)
            for (int i1 = 0; i1 < n; ++i1) {
              double a = -2.0 * PI * ((i1 - n / 2) * xi1 + (i2 - n / 2) * xi2 + (i3 - nz / 2) * xi3);
              s += vol[((size_t)i3 * n + i2) * n + i1] * cd(cos(a), sin(a));
            }
        F[(size_t)(kv + h / 2) * w + ku + w / 2] = s;
      }
    for (int jv = 0; jv < h; ++jv)
      for (int ju = 0; ju < w; ++ju) {
        cd s = 0;
        for (int kv = -h / 2; kv < h - h / 2; ++kv)
          for (int ku = -w / 2; ku < w - w / 2; ++ku) {
            double a = 2.0 * PI * (ku * (ju - g.cu) / w + kv * (jv - g.cv) / h);
            s += F[(size_t)(kv + h / 2) * w + ku + w / 2] * cd(cos(a), sin(a));
          }
        proj[((size_t)th * h + jv) * w + ju] = s.real() / ((double)w * h);
      }
  }
}

// ---------------------------------------------------------------------------------------------
// PATH B — direct discretisation with linear interpolation ("Linerec").
// Filter: circular convolution of every detector row with (pi cos(phi)/N_theta) h[j]  (same H as
// above, applied in the space domain).  Back-projection, Eq. 4:
//   vol[x] = sum_theta q_theta( x.e_u + c_u , x.e_v + c_v ),  bilinear, zero outside the detector.
// ---------------------------------------------------------------------------------------------
static void filter_rows_space(const orc_geom& g, const double* d, double* q) {
  int h = g.h, w = g.w;
  if (g.filter == 0) { memcpy(q, d, sizeof(double) * (size_t)h * w); return; }
  double scale = PI * cos(g.phi) / g.ntheta;
  std::vector<double> hk(w);
  for (int j = -w / 2; j < w - w / 2; ++j) hk[j + w / 2] = scale * ramp_kernel(g.filter, j);
#pragma omp parallel for schedule(static)
  for (int jv = 0; jv < h; ++jv)
    for (int ju = 0; ju < w; ++ju) {
      double s = 0;
      for (int jp = 0; jp < w; ++jp) {
        int dj = ju - jp;                       // wrap the lag into [-w/2, w/2)
        if (dj >= w - w / 2) dj -= w;
        if (dj < -w / 2) dj += w;
        s += hk[dj + w / 2] * d[(size_t)jv * w + jp];
      }
      q[(size_t)jv * w + ju] = s;
    }
}

extern "C" void orc_fbp_direct(const orc_geom* gp, const void* proj, double* vol) {
  const orc_geom& g = *gp;
  int h = g.h, w = g.w, n = g.n, nz = g.nz;
  std::vector<double> d((size_t)h * w), q((size_t)h * w);
  memset(vol, 0, sizeof(double) * (size_t)n * n * nz);
  for (int th = 0; th < g.ntheta; ++th) {
    load_proj(g, proj, th, d.data());
    filter_rows_space(g, d.data(), q.data());
    double ct = cos(g.theta[th]), st = sin(g.theta[th]), cp = cos(g.phi), sp = sin(g.phi);
#pragma omp parallel for collapse(2) schedule(static)
    for (int i3 = 0; i3 < nz; ++i3)
      for (int i2 = 0; i2 < n; ++i2)
        for (int i1 = 0; i1 < n; ++i1) {
          double x1 = i1 - n / 2, x2 = i2 - n / 2, x3 = i3 - nz / 2;
          double pu = x1 * ct + x2 * st + g.cu;
          double pv = x1 * st * sp - x2 * ct * sp + x3 * cp + g.cv;
          double fu = floor(pu), fv = floor(pv);
          int ju = (int)fu, jv = (int)fv;
          double au = pu - fu, av = pv - fv, s = 0;
          for (int dv = 0; dv < 2; ++dv)
            for (int du = 0; du < 2; ++du) {
              int a = ju + du, b = jv + dv;
              if (a < 0 || a >= w || b < 0 || b >= h) continue;
              s += (du ? au : 1 - au) * (dv ? av : 1 - av) * q[(size_t)b * w + a];
            }
          vol[((size_t)i3 * n + i2) * n + i1] += s;
        }
  }
}

// exact transpose of orc_fbp_direct with filter = none: splat every voxel with the hat weights.
extern "C" void orc_fp_direct(const orc_geom* gp, const double* vol, double* proj) {
  const orc_geom& g = *gp;
  int h = g.h, w = g.w, n = g.n, nz = g.nz;
#pragma omp parallel for schedule(dynamic, 1)
  for (int th = 0; th < g.ntheta; ++th) {
    double* q = proj + (size_t)th * h * w;
    memset(q, 0, sizeof(double) * (size_t)h * w);
    double ct = cos(g.theta[th]), st = sin(g.theta[th]), cp = cos(g.phi), sp = sin(g.phi);
    for (int i3 = 0; i3 < nz; ++i3)
      for (int i2 = 0; i2 < n; ++i2)
        for (int i1 = 0; i1 < n; ++i1) {
          double x1 = i1 - n / 2, x2 = i2 - n / 2, x3 = i3 - nz / 2;
          double pu = x1 * ct + x2 * st + g.cu;
          double pv = x1 * st * sp - x2 * ct * sp + x3 * cp + g.cv;
          double fu = floor(pu), fv = floor(pv);
          int ju = (int)fu, jv = (int)fv;
          double au = pu - fu, av = pv - fv, f = vol[((size_t)i3 * n + i2) * n + i1];
          for (int dv = 0; dv < 2; ++dv)
            for (int du = 0; du < 2; ++du) {
              int a = ju + du, b = jv + dv;
              if (a < 0 || a >= w || b < 0 || b >= h) continue;
              q[(size_t)b * w + a] += (du ? au : 1 - au) * (dv ? av : 1 - av) * f;
            }
        }
  }
}

// Ray-driven forward projection: the line integral of Eq. 1-2 sampled along the beam.
// The two deltas of Eq. 2 fix (x.e_u, x.e_v) = (u, v); the line is x(t) = u e_u + v e_v + t e_b with the unit
// beam direction e_b = e_u x e_v = (sin(theta) cos(phi), -cos(theta) cos(phi), -sin(phi)).  The integral is the sum over
// unit steps t of mu(x(t)), mu trilinearly interpolated between voxel centres and zero outside the volume.
extern "C" void orc_fp_ray(const orc_geom* gp, const double* vol, double* proj) {
  const orc_geom& g = *gp;
  int h = g.h, w = g.w, n = g.n, nz = g.nz;
  const int T = (int)ceil(sqrt(0.5 * (double)n * n + 0.25 * (double)nz * nz)) + 2;
  auto mu = [&](int i1, int i2, int i3) -> double {
    if (i1 < 0 || i1 >= n || i2 < 0 || i2 >= n || i3 < 0 || i3 >= nz) return 0.0;
    return vol[((size_t)i3 * n + i2) * n + i1];
  };
#pragma omp parallel for schedule(dynamic, 1)
  for (int th = 0; th < g.ntheta; ++th) {
    double ct = cos(g.theta[th]), st = sin(g.theta[th]), cp = cos(g.phi), sp = sin(g.phi);
    const double eu[3] = {ct, st, 0.0}, ev[3] = {st * sp, -ct * sp, cp}, eb[3] = {st * cp, -ct * cp, -sp};
    for (int jv = 0; jv < h; ++jv)
      for (int ju = 0; ju < w; ++ju) {
        const double u = ju - g.cu, v = jv - g.cv;
        double s = 0;
        for (int t = -T; t <= T; ++t) {
          // voxel index coordinates of the point (x1 = i1 - n/2, ...)
          const double p1 = u * eu[0] + v * ev[0] + t * eb[0] + n / 2;
          const double p2 = u * eu[1] + v * ev[1] + t * eb[1] + n / 2;
          const double p3 = u * eu[2] + v * ev[2] + t * eb[2] + nz / 2;
          const double f1 = floor(p1), f2 = floor(p2), f3 = floor(p3);
          const int i1 = (int)f1, i2 = (int)f2, i3 = (int)f3;
          if (i1 < -1 || i1 >= n || i2 < -1 || i2 >= n || i3 < -1 || i3 >= nz) continue;
          const double a1 = p1 - f1, a2 = p2 - f2, a3 = p3 - f3;
          for (int d3 = 0; d3 < 2; ++d3)
            for (int d2 = 0; d2 < 2; ++d2)
              for (int d1 = 0; d1 < 2; ++d1)
                s += (d1 ? a1 : 1 - a1) * (d2 ? a2 : 1 - a2) * (d3 ? a3 : 1 - a3) * mu(i1 + d1, i2 + d2, i3 + d3);
        }
        proj[((size_t)th * h + jv) * w + ju] = s;
      }
  }
}

// ---------------------------------------------------------------------------------------------
// PATH C — USFFT, adjoint direction: convolution-type gridding onto an equally
// spaced grid oversampled by sigma, inverse 3-D FFT, division by psi in the space domain.
// The paper fixes only "a Gaussian function psi"; reading Q5 adds Kaiser-Bessel.
//   kernel 0 (KB):    kap(t) = I0(beta sqrt(1-(2t/W)^2))/I0(beta), |t|<=W/2 (grid units)
//                     kaphat(s) = (W/I0(beta)) sinh(a)/a, a = sqrt(beta^2 - (pi W s)^2)
//   kernel 1 (Gauss): kap(t) = exp(-t^2/(2 sg2)),  kaphat(s) = sqrt(2 pi sg2) exp(-2 pi^2 sg2 s^2)
// shape = beta or sg2.  Taps m = ceil(t - W/2) + j, j = 0..W-1, stored periodically (reading Q7).
// ---------------------------------------------------------------------------------------------
// Modified Bessel function I0 by its defining power series I0(x) = sum_k (x^2/4)^k / (k!)^2 (all terms positive, so
// no cancellation; it replaces std::cyl_bessel_i in the tap loops, where that routine cost ~1 us per tap and made
// the sliced path unusable at configs[2..4] sizes).  Pinned against scipy.special.i0 in tests/test_oracle_pins.py.
static double i0_series(double x) {
  static const struct InvK2 {   // 1/k^2, k = 1..255
    double v[256];
    InvK2() { v[0] = 0; for (int k = 1; k < 256; ++k) v[k] = 1.0 / ((double)k * (double)k); }
  } inv;
  double q = 0.25 * x * x, term = 1.0, sum = 1.0;
  for (int k = 1; k < 256; ++k) {
    term *= q * inv.v[k];
    sum += term;
    if (term < 1e-18 * sum) break;
  }
  return sum;
}

// kap with the constant I0(beta) handed in (it does not depend on t; the gridding loops evaluate it once)
static double kap_n(int kernel, int W, double shape, double i0b, double t) {
  if (kernel == 0) {
    double r = 1.0 - (2.0 * t / W) * (2.0 * t / W);
    if (r < 0) return 0.0;
    return i0_series(shape * sqrt(r)) / i0b;
  }
  if (fabs(t) > 0.5 * W) return 0.0;
  return exp(-t * t / (2.0 * shape));
}
static double kap(int kernel, int W, double shape, double t) {
  return kap_n(kernel, W, shape, kernel == 0 ? i0_series(shape) : 1.0, t);
}

static double kaphat(int kernel, int W, double shape, double s) {
  if (kernel == 0) {
    double q = shape * shape - (PI * W * s) * (PI * W * s);
    double i0 = i0_series(shape);
    if (q > 0) { double a = sqrt(q); return W / i0 * sinh(a) / a; }
    if (q < 0) { double a = sqrt(-q); return W / i0 * sin(a) / a; }
    return W / i0;
  }
  return sqrt(2.0 * PI * shape) * exp(-2.0 * PI * PI * shape * s * s);
}

extern "C" double orc_kap(int kernel, int W, double shape, double t) { return kap(kernel, W, shape, t); }
extern "C" double orc_kaphat(int kernel, int W, double shape, double s) { return kaphat(kernel, W, shape, s); }

static inline int wrapi(long long m, int M) { long long r = m % M; return (int)(r < 0 ? r + M : r); }

// centred unnormalised inverse DFT along one axis of a 3-D array a[n2][n1][n0] (n0 fastest):
// out[x] = sum_m a[m] e^{+2 pi i x m / N}, m and x in [-N/2, N/2), index = value + N/2.
static void centred_idft_axis(cd* a, size_t n0, size_t n1, size_t n2, int axis) {
  size_t N = axis == 0 ? n0 : axis == 1 ? n1 : n2;
  size_t stride = axis == 0 ? 1 : axis == 1 ? n0 : n0 * n1;
  size_t nlines = n0 * n1 * n2 / N;
#pragma omp parallel
  {
    std::vector<cd> t(N);
#pragma omp for schedule(static)
    for (long long l = 0; l < (long long)nlines; ++l) {
      size_t base;
      if (axis == 0) base = (size_t)l * n0;
      else if (axis == 1) base = ((size_t)l / n0) * n0 * n1 + (size_t)l % n0;
      else base = (size_t)l;
      for (size_t i = 0; i < N; ++i) t[(i + N - N / 2) % N] = a[base + i * stride];   // m = i - N/2
      dft1(t.data(), (int)N, +1);
      for (size_t i = 0; i < N; ++i) a[base + i * stride] = t[(i + N - N / 2) % N];   // x = i - N/2
    }
  }
}

extern "C" int orc_fbp_gridded(const orc_geom* gp, const void* proj, int kernel, int W, double sigma,
                               double shape, double* vol) {
  const orc_geom& g = *gp;
  int h = g.h, w = g.w, n = g.n, nz = g.nz;
  int M1 = (int)llround(sigma * n), M2 = M1, M3 = (int)llround(sigma * nz);
  std::vector<cd> G;
  try { G.assign((size_t)M1 * M2 * M3, cd(0, 0)); } catch (...) { return 1; }
  const double i0b = kernel == 0 ? i0_series(shape) : 1.0;
  std::vector<long long> B1((size_t)h * w), B2((size_t)h * w);
  std::vector<double> K1((size_t)h * w * W), K2((size_t)h * w * W);
  std::vector<double> Hk(w), d((size_t)h * w);
  std::vector<cd> HD((size_t)h * w);
  make_filter(g, Hk.data());
  for (int th = 0; th < g.ntheta; ++th) {
    load_proj(g, proj, th, d.data());
    spectrum(g, d.data(), Hk.data(), HD.data());
    double ct = cos(g.theta[th]), st = sin(g.theta[th]), cp = cos(g.phi), sp = sin(g.phi);
    // taps and weights of every sample along xi1, xi2 (they depend on the sample only): one pass, rows shared out
#pragma omp parallel for schedule(static)
    for (int kv = -h / 2; kv < h - h / 2; ++kv) {
      double fv = (double)kv / h;
      for (int ku = -w / 2; ku < w - w / 2; ++ku) {
        double fu = (double)ku / w;
        double t1 = M1 * (fu * ct + fv * st * sp);   // Eq. 6 in fine-grid units
        double t2 = M2 * (fu * st - fv * ct * sp);
        size_t si = (size_t)(kv + h / 2) * w + ku + w / 2;
        long long b1 = (long long)ceil(t1 - 0.5 * W), b2 = (long long)ceil(t2 - 0.5 * W);
        B1[si] = b1;
        B2[si] = b2;
        for (int j = 0; j < W; ++j) {
          K1[si * W + j] = kap_n(kernel, W, shape, i0b, t1 - (double)(b1 + j));
          K2[si * W + j] = kap_n(kernel, W, shape, i0b, t2 - (double)(b2 + j));
        }
      }
    }
    // each thread owns the fine planes m3 with (m3 mod nthreads) == tid, so no two threads write one cell
#pragma omp parallel
    {
#ifdef _OPENMP
      int tid = omp_get_thread_num(), nt = omp_get_num_threads();
#else
      int tid = 0, nt = 1;
#endif
      std::vector<double> k3(W);
      for (int kv = -h / 2; kv < h - h / 2; ++kv) {
        double fv = (double)kv / h;
        double t3 = M3 * (fv * cp);
        long long b3 = (long long)ceil(t3 - 0.5 * W);
        bool mine = false;
        for (int j = 0; j < W; ++j) mine = mine || wrapi(b3 + j + M3 / 2, M3) % nt == tid;
        if (!mine) continue;
        for (int j = 0; j < W; ++j) k3[j] = kap_n(kernel, W, shape, i0b, t3 - (double)(b3 + j));
        for (int ku = -w / 2; ku < w - w / 2; ++ku) {
          size_t si = (size_t)(kv + h / 2) * w + ku + w / 2;
          long long b1 = B1[si], b2 = B2[si];
          const double *k1 = &K1[si * W], *k2 = &K2[si * W];
          cd val = HD[si];
          for (int j3 = 0; j3 < W; ++j3) {
            int m3 = wrapi(b3 + j3 + M3 / 2, M3);
            if (m3 % nt != tid) continue;
            for (int j2 = 0; j2 < W; ++j2) {
              int m2 = wrapi(b2 + j2 + M2 / 2, M2);
              for (int j1 = 0; j1 < W; ++j1) {
                int m1 = wrapi(b1 + j1 + M1 / 2, M1);
                G[((size_t)m3 * M2 + m2) * M1 + m1] += val * (k1[j1] * k2[j2] * k3[j3]);
              }
            }
          }
        }
      }
    }
  }
  centred_idft_axis(G.data(), M1, M2, M3, 0);
  centred_idft_axis(G.data(), M1, M2, M3, 1);
  centred_idft_axis(G.data(), M1, M2, M3, 2);
  for (int i3 = 0; i3 < nz; ++i3)
    for (int i2 = 0; i2 < n; ++i2)
      for (int i1 = 0; i1 < n; ++i1) {
        double x1 = i1 - n / 2, x2 = i2 - n / 2, x3 = i3 - nz / 2;
        double den = kaphat(kernel, W, shape, x1 / M1) * kaphat(kernel, W, shape, x2 / M2) *
                     kaphat(kernel, W, shape, x3 / M3);
        cd v = G[((size_t)(i3 - nz / 2 + M3 / 2) * M2 + (i2 - n / 2 + M2 / 2)) * M1 + (i1 - n / 2 + M1 / 2)];
        vol[((size_t)i3 * n + i2) * n + i1] = v.real() / den;
      }
  return 0;
}

// ---------------------------------------------------------------------------------------------
// PATH C' — Eq. 9 for one slice i3: the x3 transform is done exactly
// (phase e^{2 pi i x3 k_v cos(phi)/h} on every sample), the (x1,x2) transform is a 2-D USFFT.
// Needs only an M2 x M1 double grid, so it runs at configs[3], [4] sizes.  slice[i2][i1].
// ---------------------------------------------------------------------------------------------
extern "C" int orc_fbp_gridded_slice(const orc_geom* gp, const void* proj, int kernel, int W, double sigma,
                                     double shape, int i3, double* slice) {
  const orc_geom& g = *gp;
  int h = g.h, w = g.w, n = g.n, nz = g.nz;
  int M1 = (int)llround(sigma * n), M2 = M1;
  std::vector<cd> G((size_t)M1 * M2, cd(0, 0));
  const double i0b = kernel == 0 ? i0_series(shape) : 1.0;
  std::vector<long long> B1((size_t)h * w), B2((size_t)h * w);
  std::vector<double> K1((size_t)h * w * W), K2((size_t)h * w * W);
  std::vector<double> Hk(w), d((size_t)h * w);
  std::vector<cd> HD((size_t)h * w);
  make_filter(g, Hk.data());
  double x3 = i3 - nz / 2;
  for (int th = 0; th < g.ntheta; ++th) {
    load_proj(g, proj, th, d.data());
    spectrum(g, d.data(), Hk.data(), HD.data());
    double ct = cos(g.theta[th]), st = sin(g.theta[th]), cp = cos(g.phi), sp = sin(g.phi);
    // taps and weights of every sample (they depend on the sample only): one pass, rows shared out
#pragma omp parallel for schedule(static)
    for (int kv = -h / 2; kv < h - h / 2; ++kv) {
      double fv = (double)kv / h;
      for (int ku = -w / 2; ku < w - w / 2; ++ku) {
        double fu = (double)ku / w;
        double t1 = M1 * (fu * ct + fv * st * sp);
        double t2 = M2 * (fu * st - fv * ct * sp);
        size_t si = (size_t)(kv + h / 2) * w + ku + w / 2;
        long long b1 = (long long)ceil(t1 - 0.5 * W), b2 = (long long)ceil(t2 - 0.5 * W);
        B1[si] = b1;
        B2[si] = b2;
        for (int j = 0; j < W; ++j) {
          K1[si * W + j] = kap_n(kernel, W, shape, i0b, t1 - (double)(b1 + j));
          K2[si * W + j] = kap_n(kernel, W, shape, i0b, t2 - (double)(b2 + j));
        }
      }
    }
    // each thread owns the grid rows m2 with (m2 mod nthreads) == tid, so no two threads write one cell
#pragma omp parallel
    {
#ifdef _OPENMP
      int tid = omp_get_thread_num(), nt = omp_get_num_threads();
#else
      int tid = 0, nt = 1;
#endif
      for (int kv = -h / 2; kv < h - h / 2; ++kv) {
        double fv = (double)kv / h;
        double a = 2.0 * PI * x3 * fv * cp;
        cd ph(cos(a), sin(a));
        for (int ku = -w / 2; ku < w - w / 2; ++ku) {
          size_t si = (size_t)(kv + h / 2) * w + ku + w / 2;
          long long b1 = B1[si], b2 = B2[si];
          const double *k1 = &K1[si * W], *k2 = &K2[si * W];
          cd val = HD[si] * ph;
          for (int j2 = 0; j2 < W; ++j2) {
            int m2 = wrapi(b2 + j2 + M2 / 2, M2);
            if (m2 % nt != tid) continue;
            for (int j1 = 0; j1 < W; ++j1) {
              int m1 = wrapi(b1 + j1 + M1 / 2, M1);
              G[(size_t)m2 * M1 + m1] += val * (k1[j1] * k2[j2]);
            }
          }
        }
      }
    }
  }
  centred_idft_axis(G.data(), M1, M2, 1, 0);
  centred_idft_axis(G.data(), M1, M2, 1, 1);
  for (int i2 = 0; i2 < n; ++i2)
    for (int i1 = 0; i1 < n; ++i1) {
      double x1 = i1 - n / 2, x2 = i2 - n / 2;
      double den = kaphat(kernel, W, shape, x1 / M1) * kaphat(kernel, W, shape, x2 / M2);
      cd v = G[(size_t)(i2 - n / 2 + M2 / 2) * M1 + (i1 - n / 2 + M1 / 2)];
      slice[(size_t)i2 * n + i1] = v.real() / den;
    }
  return 0;
}

extern "C" int orc_threads(void) { return max_threads(); }
