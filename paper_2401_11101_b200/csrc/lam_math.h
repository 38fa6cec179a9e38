// lam_math.h — host-side double-precision table makers for the CUDA path (gridding kernel, its transform, its
// piecewise-polynomial form, the ramp filter).  Product code: shares nothing with oracle/.
//
// Gridding kernel psi of the USFFT (PAPER.md:130 names "a Gaussian function psi"; reading Q5 adds Kaiser-Bessel):
//   KB:    kap(t) = I0(beta sqrt(1-(2t/W)^2)) / I0(beta), |t| <= W/2;  kaphat(s) = (W/I0(beta)) sinh(a)/a,
//          a = sqrt(beta^2 - (pi W s)^2)   (sin(a')/a' beyond the cut-off)
//   Gauss: kap(t) = exp(-t^2/(2 v)), truncated at |t| <= W/2;  kaphat(s) = sqrt(2 pi v) exp(-2 pi^2 v s^2)
// Filter W of Eq. 3, reading Q3: H[k] = (pi cos(phi)/N_theta) * DFT_w(h)[k], h the band-limited
// ramp (Ram-Lak) or Shepp-Logan spatial kernel at unit pitch.
#pragma once
#include <cmath>
#include <vector>

namespace lam {

static const double kPi = 3.141592653589793238462643383279502884;

// modified Bessel function I0 by its power series (all terms positive; converges for the beta <= 40 used here)
inline double bessel_i0(double x) {
  double q = 0.25 * x * x, term = 1.0, sum = 1.0;
  for (int k = 1; k < 500; ++k) {
    term *= q / ((double)k * (double)k);
    sum += term;
    if (term < 1e-17 * sum) break;
  }
  return sum;
}

struct GridKernel {
  int type;      // 0 KB, 1 Gauss
  int W;
  double shape;  // beta or variance
  double i0b;

  void init(int type_, int W_, double sigma, double shape_) {
    type = type_;
    W = W_;
    if (shape_ > 0) shape = shape_;
    else if (type == 0) shape = kPi * std::sqrt((W / sigma) * (W / sigma) * (sigma - 0.5) * (sigma - 0.5) - 0.8);
    else shape = sigma * (W / 2.0) / (2.0 * kPi * (sigma - 0.5));
    i0b = type == 0 ? bessel_i0(shape) : 1.0;
  }
  double kap(double t) const {
    if (std::fabs(t) > 0.5 * W) return 0.0;
    if (type == 0) {
      double r = 1.0 - (2.0 * t / W) * (2.0 * t / W);
      return bessel_i0(shape * std::sqrt(r < 0 ? 0 : r)) / i0b;
    }
    return std::exp(-t * t / (2.0 * shape));
  }
  double kaphat(double s) const {
    if (type == 0) {
      double q = shape * shape - (kPi * W * s) * (kPi * W * s);
      if (q > 1e-12) { double a = std::sqrt(q); return W / i0b * std::sinh(a) / a; }
      if (q < -1e-12) { double a = std::sqrt(-q); return W / i0b * std::sin(a) / a; }
      return W / i0b;
    }
    return std::sqrt(2.0 * kPi * shape) * std::exp(-2.0 * kPi * kPi * shape * s * s);
  }
};

// Piecewise polynomial form of the kernel.  With b = ceil(t - W/2), taps m = b + j (j = 0..W-1) and
// delta = t - b - (W/2 - 1/2) in [-1/2, 1/2):  kap(t - m) = p_j(delta), and p_{W-1-j}(delta) = p_j(-delta).
// For j < W/2 we store p_j = E_j(delta^2) + delta O_j(delta^2), degree 7: E, O have 4 coefficients each.
// Chebyshev interpolation on [-1/2, 1/2], converted to monomials; fit error ~1e-7 for KB W = 6 (fp32 level).
constexpr int kPolyHalf = 4;  // coefficients of E and of O

inline void kernel_poly(const GridKernel& gk, float* E /*[W/2][4]*/, float* O /*[W/2][4]*/) {
  const int D = 2 * kPolyHalf - 1, K = 48;
  for (int j = 0; j < gk.W / 2; ++j) {
    double cj = 0.5 * gk.W - 0.5 - j;
    // Chebyshev coefficients c_d = (2/K) sum_i f(x_i) T_d(x_i), x = 2 delta
    std::vector<double> c(D + 1, 0.0);
    for (int d = 0; d <= D; ++d) {
      double s = 0;
      for (int i = 0; i < K; ++i) {
        double th = kPi * (i + 0.5) / K, x = std::cos(th);
        s += gk.kap(0.5 * x + cj) * std::cos(d * th);
      }
      c[d] = (d == 0 ? 1.0 : 2.0) * s / K;
    }
    // T_d(x) -> monomials in x by the recurrence T_{d+1} = 2x T_d - T_{d-1}
    std::vector<std::vector<double>> T(D + 1, std::vector<double>(D + 1, 0.0));
    T[0][0] = 1.0;
    if (D >= 1) T[1][1] = 1.0;
    for (int d = 1; d < D; ++d)
      for (int m = 0; m <= D; ++m) {
        double v = -T[d - 1][m];
        if (m > 0) v += 2.0 * T[d][m - 1];
        T[d + 1][m] = v;
      }
    std::vector<double> mono(D + 1, 0.0);
    for (int d = 0; d <= D; ++d)
      for (int m = 0; m <= D; ++m) mono[m] += c[d] * T[d][m];
    // x = 2 delta
    double sc = 1.0;
    for (int m = 0; m <= D; ++m) { mono[m] *= sc; sc *= 2.0; }
    for (int q = 0; q < kPolyHalf; ++q) {
      E[j * kPolyHalf + q] = (float)mono[2 * q];
      O[j * kPolyHalf + q] = (float)mono[2 * q + 1];
    }
  }
}

inline double ramp_spatial(int filter, int j) {
  if (filter == 1 || filter == 3) {
    if (j == 0) return 0.25;
    if (j & 1) return -1.0 / (kPi * kPi * (double)j * (double)j);
    return 0.0;
  }
  return -2.0 / (kPi * kPi * (4.0 * (double)j * (double)j - 1.0));
}

// H[k], k = 0..w/2 (H is real and even in k).  filter 0: all ones.
inline void filter_response(int filter, int w, double phi, int ntheta, std::vector<double>& H) {
  H.assign(w / 2 + 1, 1.0);
  if (filter == 0) return;
  std::vector<double> hs(w);
  for (int j = -w / 2; j < w / 2; ++j) hs[j + w / 2] = ramp_spatial(filter, j);
  double scale = kPi * std::cos(phi) / ntheta;
  std::vector<double> cs(w);
  for (int m = 0; m < w; ++m) cs[m] = std::cos(2.0 * kPi * m / w);
  for (int k = 0; k <= w / 2; ++k) {
    double s = 0;
    for (int j = -w / 2; j < w / 2; ++j) {
      long long m = ((long long)k * j) % w;
      if (m < 0) m += w;
      s += hs[j + w / 2] * cs[m];
    }
    H[k] = scale * s;
    if (filter == 3) {  // Parzen window over the ramp: x = k / (w/2), 1 at DC, 0 at Nyquist
      const double x = (double)k / (0.5 * w);
      H[k] *= x <= 0.5 ? 1.0 - 6.0 * x * x * (1.0 - x) : 2.0 * (1.0 - x) * (1.0 - x) * (1.0 - x);
    }
  }
}

}  // namespace lam
