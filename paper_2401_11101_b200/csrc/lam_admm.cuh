// lam_admm.cuh — elementwise and reduction kernels of the TV-regularised reconstruction of PAPER.md Appendix A
// (Eqs. 10-20): ADMM with the splitting grad mu = psi (Eq. 12), the mu-subproblem (Eq. 17) by
// conjugate gradients with Dai-Yuan directions (Eq. 19) on the operators lam_forward (L) and lam_backproject with
// filter none (L^T), the psi-subproblem by the isotropic soft threshold (Eq. 20, re-derived: DESIGN.md reading Q18) and
// the multiplier update of Eq. 16.  The driver lam_admm_tv is in lam.cu.
//
// grad = forward differences with a zero last difference along each axis, div = -grad^T (reading Q20):
//   (grad mu)_c[i] = mu[i + e_c] - mu[i]  (i_c < N_c - 1),   (div q)[i] = sum_c q_c[i] [i_c < N_c - 1] - q_c[i - e_c] [i_c >= 1].
#pragma once
#include <cuda_runtime.h>

namespace lam {

struct TvDims {
  int n, nz;  // vol[nz][n][n]
};

__device__ __forceinline__ void tv_index(size_t i, const TvDims& d, int& i1, int& i2, int& i3) {
  i1 = (int)(i % d.n);
  const size_t r = i / d.n;
  i2 = (int)(r % d.n);
  i3 = (int)(r / d.n);
}

// out (+)= -rho div( grad x - psi + lam / rho ); psi = lam = nullptr: out (+)= -rho div grad x.     (Eq. 18, second term)
__global__ void k_tv_reggrad(const float* __restrict__ x, const float* __restrict__ psi, const float* __restrict__ lam, float rho,
                             float* __restrict__ out, int accumulate, TvDims d) {
  const size_t nvox = (size_t)d.nz * d.n * d.n;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nvox) return;
  int i1, i2, i3;
  tv_index(i, d, i1, i2, i3);
  const size_t st[3] = {1, (size_t)d.n, (size_t)d.n * d.n};
  const int idx[3] = {i1, i2, i3}, N[3] = {d.n, d.n, d.nz};
  const float irho = 1.0f / rho, xi = x[i];
  float dv = 0.f;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    if (idx[c] < N[c] - 1) {
      float q = x[i + st[c]] - xi;
      if (psi) q += -psi[c * nvox + i] + lam[c * nvox + i] * irho;
      dv += q;
    }
    if (idx[c] >= 1) {
      const size_t j = i - st[c];
      float q = xi - x[j];
      if (psi) q += -psi[c * nvox + j] + lam[c * nvox + j] * irho;
      dv -= q;
    }
  }
  const float v = -rho * dv;
  out[i] = accumulate ? out[i] + v : v;
}

// psi <- shrink(grad mu + lam / rho, alpha / rho)   (Eq. 15 / 20),   lam <- lam + rho (grad mu - psi)   (Eq. 16)
__global__ void k_tv_shrink(const float* __restrict__ mu, float* __restrict__ psi, float* __restrict__ lam, float alpha, float rho,
                            TvDims d) {
  const size_t nvox = (size_t)d.nz * d.n * d.n;
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= nvox) return;
  int i1, i2, i3;
  tv_index(i, d, i1, i2, i3);
  const size_t st[3] = {1, (size_t)d.n, (size_t)d.n * d.n};
  const int idx[3] = {i1, i2, i3}, N[3] = {d.n, d.n, d.nz};
  const float irho = 1.0f / rho, t = alpha * irho, xi = mu[i];
  float g[3], v[3], l[3];
  float nrm2 = 0.f;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    g[c] = idx[c] < N[c] - 1 ? mu[i + st[c]] - xi : 0.f;
    l[c] = lam[c * nvox + i];
    v[c] = g[c] + l[c] * irho;
    nrm2 += v[c] * v[c];
  }
  const float nrm = sqrtf(nrm2), sc = nrm > t ? 1.0f - t / nrm : 0.f;
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const float ps = v[c] * sc;
    psi[c * nvox + i] = ps;
    lam[c * nvox + i] = l[c] + rho * (g[c] - ps);
  }
}

// y <- a y + b x
__global__ void k_axpby(float* __restrict__ y, float a, const float* __restrict__ x, float b, size_t cnt) {
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < cnt; i += (size_t)gridDim.x * blockDim.x) y[i] = a * y[i] + b * x[i];
}

__device__ __forceinline__ void block_sum_to(double v, double* out) {
  __shared__ double sh[32];
  for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = v;
  __syncthreads();
  if (threadIdx.x < 32) {
    v = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    if (threadIdx.x == 0) atomicAdd(out, v);
  }
}

// out += <x, y> in double (products in double: the sums decide step lengths)
__global__ void k_dot(const float* __restrict__ x, const float* __restrict__ y, size_t cnt, double* out) {
  double acc = 0.0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < cnt; i += (size_t)gridDim.x * blockDim.x) acc += (double)x[i] * (double)y[i];
  block_sum_to(acc, out);
}

// out += || grad x ||^2
__global__ void k_tv_gradnorm2(const float* __restrict__ x, TvDims d, double* out) {
  const size_t nvox = (size_t)d.nz * d.n * d.n;
  double acc = 0.0;
  for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvox; i += (size_t)gridDim.x * blockDim.x) {
    int i1, i2, i3;
    tv_index(i, d, i1, i2, i3);
    const float xi = x[i];
    if (i1 < d.n - 1) { const float q = x[i + 1] - xi; acc += (double)q * q; }
    if (i2 < d.n - 1) { const float q = x[i + d.n] - xi; acc += (double)q * q; }
    if (i3 < d.nz - 1) { const float q = x[i + (size_t)d.n * d.n] - xi; acc += (double)q * q; }
  }
  block_sum_to(acc, out);
}

}  // namespace lam
