// lam.cu — host side of liblam.so: the C ABI of include/lam.h, the plan (tables, work lists, workspace) and the
// launch schedule of the sm_100a kernels in lam_kernels.cuh.  No CPU fallback: every compute entry point needs a
// CUDA device and returns LAM_ECUDA without one.
//
// Schedule of lam_backproject (Eq. 7 evaluated in the order of Eq. 9):
//   for every chunk of projections:   k_rows  (S0 + row FFT + filter)  ->  k_cols (column FFT, fold onto k_v >= 0 planes)
//   for every batch of k_v planes:    k_spread (gridding in xi1, xi2)  ->  k_ifft_x1  ->  k_ifft_x2  (cropped n x n planes)
//   once:                             k_zstage (gridding in xi3 + inverse FFT + crop + real part + deapodisation)
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/lam.h"
#include "lam_kernels.cuh"
#include "lam_spread.cuh"
#include "lam_forward.cuh"
#include "lam_admm.cuh"

using namespace lam;

namespace {

thread_local std::string g_create_error;
thread_local cudaError_t g_launch_error = cudaSuccess;  // first failed kernel launch of the current call
inline void note_launch() {
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess && g_launch_error == cudaSuccess) g_launch_error = e;
}

struct StageEvent {
  int stage;
  cudaEvent_t a, b;
};

}  // namespace

struct lam_plan {
  // problem
  int n = 0, nz = 0, h = 0, w = 0, ntheta = 0;
  double phi = 0;
  lam_params prm{};
  std::vector<double> theta;
  // derived
  int M = 0, M3 = 0, W = 0, NP = 0, WR = 0, WQ = 0;
  int logw = 0, logh = 0, logM = 0, logM3 = 0;
  int PB = 1, TC = 1;  // plane batch, theta chunk
  int TSB = 1;         // planes per x1/x2 sub-batch: T (the x1-transformed planes) is sized to stay L2-resident
  int rows_nb = 1, cols_lcb = 3, x1_nb = 1, x2_lnb = 3, KZ = 1, z_lcb = 3;
  GridKernel gk;
  KerPoly kp{};
  SpreadGeom geom{};
  // device tables
  double2* d_cs = nullptr;
  float2 *d_Pu = nullptr, *d_Pv = nullptr, *d_PuNone = nullptr;
  float* d_Hp = nullptr;       // pad_u: filter response of the 2w-sample rows, k = 0..w, times 1/(2w)
  float2* d_tw_w2 = nullptr;   // pad_u: twiddles of length 2w
  int rows_nb_pad = 1;
  // single-slice mode (allocated on first use): summed fine grid, its x1 transform, cropped plane, phase tables
  float2 *d_Gs = nullptr, *d_Ts = nullptr, *d_As = nullptr, *d_zph = nullptr, *d_cph = nullptr;
  // ADMM-TV workspace (allocated on first use): gradient, direction, H eta (volumes), psi, lambda (3 volumes each), one
  // projection-sized buffer, four double accumulators
  float *d_tv_g = nullptr, *d_tv_eta = nullptr, *d_tv_h = nullptr, *d_tv_psi = nullptr, *d_tv_lam = nullptr, *d_tv_r = nullptr;
  double* d_tv_acc = nullptr;
  float2 *d_tw_w = nullptr, *d_tw_h = nullptr, *d_tw_M = nullptr, *d_tw_M3 = nullptr;
  float *d_ztab = nullptr, *d_zlast = nullptr, *d_dx = nullptr, *d_dz = nullptr, *d_dark = nullptr, *d_flat = nullptr;
  float2* d_df = nullptr;
  float* d_wz = nullptr;  // [NP][W] x3 tap weights per plane (lam_forward)
  int* d_bz = nullptr;    // [NP] first x3 tap per plane
  int *d_zlo = nullptr, *d_zcnt = nullptr, *d_zidx = nullptr;
  int nact = 0;  // active x3 grid cells
  // x3 stage through TMA (k_zstage_tma): tensor map over A[p][x2][x1], box split, double-buffer size, launch shape
  CUtensorMap tmapA;
  bool z_tma = false;
  int z_nbox = 1, z_pbox = 1, z_bufelems = 0, z_threads = 512, z_blocks_per_sm = 1, n_sm = 148;
  size_t z_smem = 0;
  Job* d_jobs = nullptr;
  std::vector<long long> job_off;  // [batches+1] first job of each plane batch (jobs of a batch: heaviest tiles first)
  unsigned* d_multi = nullptr;     // tiles written by several jobs, batch-major
  std::vector<long long> multi_off;  // [batches+1]
  double plan_ms = 0;              // wall time of lam_create
  // workspace
  float2 *d_R = nullptr, *d_S = nullptr, *d_G = nullptr, *d_T = nullptr, *d_A = nullptr;  // d_S, d_A live inside d_arena
  float2* d_arena = nullptr;
  size_t device_bytes = 0, pinned_bytes = 0;
  bool have_darkflat = false;
  // host-pointer path (allocated on first use): device staging, copy streams, hand-over events
  void* d_in[2] = {nullptr, nullptr};
  float* d_out[2] = {nullptr, nullptr};
  int ZR = 0;  // x2 rows per output slab
  cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
  cudaEvent_t ev_in_ready[2] = {}, ev_in_free[2] = {}, ev_out_ready[2] = {}, ev_out_free[2] = {}, ev_fork = nullptr;
  bool host_path_ready = false;
  bool last_call_host = false;   // the last lam_backproject streamed through host pointers
  // spilled (out-of-core) mode, chosen by lam_create when the in-core workspace exceeds params.device_bytes
  // (PAPER.md:172 "> 64 GB for 2048^3", :181-191): the spectra S exist for one BAND of planes at a time (S0+S1 run once
  // per band), the cropped planes A[p] leave for pinned host memory as their batch is born and come back per x2-slab
  // for the x3 stage
  bool spill = false;
  int chunk_ctr = 0;                   // projection chunks issued by the current call (host-pointer path)
  int band = 0;                        // planes per band (a multiple of PB)
  int ZRs = 0;                         // x2 rows per x3-stage slab
  float2* h_A = nullptr;               // pinned host [NP][n][n]
  float2* d_Ab[2] = {nullptr, nullptr};  // device staging of one plane batch of A
  float2* d_As2[2] = {nullptr, nullptr}; // device slab [NP][ZRs][n]
  cudaEvent_t ev_ab_ready[2] = {}, ev_ab_free[2] = {}, ev_sl_ready[2] = {}, ev_sl_free[2] = {};
  // bookkeeping
  std::string err;
  int device = 0;
  bool profiling = false;
  bool copy_only = false;  // lam_set_profiling(plan, 2): the host<->device copies run, the kernels are skipped
  std::vector<StageEvent> events;
  size_t events_used = 0;
  long long launches = 0;
  float last_ms[6] = {0, 0, 0, 0, 0, 0};
  bool stage_valid = false;
};

namespace {

lam_status fail(lam_plan* p, lam_status st, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (p) p->err = buf;
  else g_create_error = buf;
  return st;
}

#define CU(p, call)                                                                                              \
  do {                                                                                                           \
    cudaError_t e_ = (call);                                                                                     \
    if (e_ != cudaSuccess)                                                                                       \
      return fail(p, e_ == cudaErrorMemoryAllocation ? LAM_ENOMEM_DEVICE : LAM_ECUDA, "%s: %s (%s:%d)", #call,   \
                  cudaGetErrorString(e_), __FILE__, __LINE__);                                                   \
  } while (0)

int ilog2(int v) {
  int l = 0;
  while ((1 << l) < v) ++l;
  return l;
}
bool pow2(int v) { return v > 0 && (v & (v - 1)) == 0; }

template <class T>
lam_status dalloc(lam_plan* p, T** ptr, size_t count) {
  size_t bytes = std::max<size_t>(count, 1) * sizeof(T);
  cudaError_t e = cudaMalloc((void**)ptr, bytes);
  if (e != cudaSuccess) {
    *ptr = nullptr;
    cudaGetLastError();
    return fail(p, LAM_ENOMEM_DEVICE, "cudaMalloc of %zu bytes failed: %s", bytes, cudaGetErrorString(e));
  }
  p->device_bytes += bytes;
  return LAM_OK;
}

template <class T>
lam_status upload(lam_plan* p, T** ptr, const std::vector<T>& v) {
  lam_status st = dalloc(p, ptr, v.size());
  if (st != LAM_OK) return st;
  CU(p, cudaMemcpy(*ptr, v.data(), v.size() * sizeof(T), cudaMemcpyHostToDevice));
  return LAM_OK;
}

std::vector<float2> twiddles(int N) {
  std::vector<float2> t(N);
  for (int k = 0; k < N; ++k) {
    double a = -2.0 * kPi * k / N;
    t[k] = make_float2((float)std::cos(a), (float)std::sin(a));
  }
  return t;
}

// ---- templated launch tables (FFT lengths 2^5 .. 2^13) ------------------------------------------------------------
constexpr int kLogMin = 5, kLogMax = 13;

template <int L>
struct Launch {
  static void rows(bool raw, dim3 g, size_t sm, cudaStream_t s, const RowsArgs& a) {
    if (raw) {
      cudaFuncSetAttribute(k_rows<L, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
      k_rows<L, true><<<g, 256, sm, s>>>(a);
      note_launch();
    } else {
      cudaFuncSetAttribute(k_rows<L, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
      k_rows<L, false><<<g, 256, sm, s>>>(a);
      note_launch();
    }
  }
  static void rows_pad(bool raw, dim3 g, size_t sm, cudaStream_t s, const RowsPadArgs& a) {
    if constexpr (L < kLogMax) {
      if (raw) {
        cudaFuncSetAttribute(k_rows_pad<L, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        k_rows_pad<L, true><<<g, 256, sm, s>>>(a);
      } else {
        cudaFuncSetAttribute(k_rows_pad<L, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        k_rows_pad<L, false><<<g, 256, sm, s>>>(a);
      }
      note_launch();
    }
  }
  static void cols(dim3 g, int threads, size_t sm, cudaStream_t s, const ColsArgs& a) {
    cudaFuncSetAttribute(k_cols<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    k_cols<L><<<g, threads, sm, s>>>(a);
      note_launch();
  }
  static void x1(dim3 g, size_t sm, cudaStream_t s, const IfftArgs& a) {
    cudaFuncSetAttribute(k_ifft_x1<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    k_ifft_x1<L><<<g, 256, sm, s>>>(a);
      note_launch();
  }
  static void x2(dim3 g, int threads, size_t sm, cudaStream_t s, const IfftArgs& a) {
    cudaFuncSetAttribute(k_ifft_x2<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    k_ifft_x2<L><<<g, threads, sm, s>>>(a);
      note_launch();
  }
  static void zT(dim3 g, size_t sm, cudaStream_t s, const ZTArgs& a) {
    cudaFuncSetAttribute(k_zstage_T<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    k_zstage_T<L><<<g, 256, sm, s>>>(a);
    note_launch();
  }
  static void x2T(dim3 g, int threads, size_t sm, cudaStream_t s, const IfftArgs& a) {
    cudaFuncSetAttribute(k_fft_x2_T<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    k_fft_x2_T<L><<<g, threads, sm, s>>>(a);
    note_launch();
  }
  static void x1T(dim3 g, size_t sm, cudaStream_t s, const IfftArgs& a) {
    cudaFuncSetAttribute(k_fft_x1_T<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    k_fft_x1_T<L><<<g, 256, sm, s>>>(a);
    note_launch();
  }
  static void colsT(dim3 g, int threads, size_t sm, cudaStream_t s, const ColsTArgs& a) {
    cudaFuncSetAttribute(k_cols_T<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    k_cols_T<L><<<g, threads, sm, s>>>(a);
    note_launch();
  }
  static void rowsT(dim3 g, size_t sm, cudaStream_t s, const RowsTArgs& a) {
    cudaFuncSetAttribute(k_rows_T<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    k_rows_T<L><<<g, 256, sm, s>>>(a);
    note_launch();
  }
  static void ztma(int grid, int threads, size_t sm, cudaStream_t s, const CUtensorMap& tm, const ZTmaArgs& a) {
    cudaFuncSetAttribute(k_zstage_tma<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    k_zstage_tma<L><<<grid, threads, sm, s>>>(tm, a);
    note_launch();
  }
  static int ztma_occupancy(int threads, size_t sm) {
    cudaFuncSetAttribute(k_zstage_tma<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_zstage_tma<L>, threads, sm) != cudaSuccess) { cudaGetLastError(); nb = 0; }
    return nb;
  }
  static void z(dim3 g, int threads, size_t sm, cudaStream_t s, const ZArgs& a) {
    cudaFuncSetAttribute(k_zstage<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    k_zstage<L><<<g, threads, sm, s>>>(a);
      note_launch();
  }
};

template <int L, class F>
void dispatch_log_impl(int lg, F&& f) {
  if constexpr (L <= kLogMax) {
    if (lg == L) f(Launch<L>{});
    else dispatch_log_impl<L + 1>(lg, f);
  }
}
#define DISPATCH_LOG(lg, call) dispatch_log_impl<kLogMin>(lg, [&](auto L_) { decltype(L_)::call; })

template <class F>
void dispatch_W(int W, F&& f) {
  if (W == 4) f(std::integral_constant<int, 4>{});
  else if (W == 6) f(std::integral_constant<int, 6>{});
  else f(std::integral_constant<int, 8>{});
}

// ---- profiling events ----------------------------------------------------------------------------------------------
struct StageScope {
  lam_plan* p;
  cudaStream_t s;
  long idx = -1;  // index, not pointer: nested scopes may grow the vector
  StageScope(lam_plan* p_, int stage, cudaStream_t s_) : p(p_), s(s_) {
    if (!p->profiling) return;
    if (p->events_used == p->events.size()) {
      StageEvent e{stage, nullptr, nullptr};
      cudaEventCreate(&e.a);
      cudaEventCreate(&e.b);
      p->events.push_back(e);
    }
    idx = (long)p->events_used++;
    p->events[idx].stage = stage;
    cudaEventRecord(p->events[idx].a, s);
  }
  ~StageScope() {
    if (idx >= 0) cudaEventRecord(p->events[idx].b, s);
  }
};

void free_all(lam_plan* p) {
  void* ptrs[] = {p->d_cs,    p->d_Pu,  p->d_Pv,  p->d_PuNone, p->d_tw_w, p->d_tw_h,   p->d_tw_M, p->d_tw_M3,
                  p->d_ztab,  p->d_dx,  p->d_dz,  p->d_dark,   p->d_flat, p->d_zlo,    p->d_zlast,  p->d_jobs, p->d_Hp, p->d_tw_w2, p->d_Gs, p->d_Ts, p->d_As, p->d_zph, p->d_cph, p->d_tv_g, p->d_tv_eta, p->d_tv_h, p->d_tv_psi, p->d_tv_lam, p->d_tv_r, p->d_tv_acc, p->d_zcnt, p->d_zidx, p->d_df, p->d_wz, p->d_bz, p->d_multi,
                  p->d_R,     p->d_arena, p->d_G, p->d_T};
  for (void* q : ptrs)
    if (q) cudaFree(q);
  for (int i = 0; i < 2; ++i) {
    if (p->d_in[i]) cudaFree(p->d_in[i]);
    if (p->d_out[i]) cudaFree(p->d_out[i]);
    if (p->ev_in_ready[i]) cudaEventDestroy(p->ev_in_ready[i]);
    if (p->ev_in_free[i]) cudaEventDestroy(p->ev_in_free[i]);
    if (p->ev_out_ready[i]) cudaEventDestroy(p->ev_out_ready[i]);
    if (p->ev_out_free[i]) cudaEventDestroy(p->ev_out_free[i]);
  }
  for (int i = 0; i < 2; ++i) {
    if (p->d_Ab[i]) cudaFree(p->d_Ab[i]);
    if (p->d_As2[i]) cudaFree(p->d_As2[i]);
    if (p->ev_ab_ready[i]) cudaEventDestroy(p->ev_ab_ready[i]);
    if (p->ev_ab_free[i]) cudaEventDestroy(p->ev_ab_free[i]);
    if (p->ev_sl_ready[i]) cudaEventDestroy(p->ev_sl_ready[i]);
    if (p->ev_sl_free[i]) cudaEventDestroy(p->ev_sl_free[i]);
  }
  if (p->h_A) cudaFreeHost(p->h_A);
  if (p->ev_fork) cudaEventDestroy(p->ev_fork);
  if (p->s_h2d) cudaStreamDestroy(p->s_h2d);
  if (p->s_d2h) cudaStreamDestroy(p->s_d2h);
  for (auto& e : p->events) {
    cudaEventDestroy(e.a);
    cudaEventDestroy(e.b);
  }
}

// ---- work lists of the (xi1, xi2) gridding: geometry only, built once ---------------------------------------------
// Two device passes (count, fill) with the host in between: the jobs of one plane batch (= one k_spread launch) are laid
// out heaviest tile first, so that the few tiles around the xi3 axis that every theta crosses start early.
lam_status build_jobs(lam_plan* p) {
  const int ntiles = p->geom.nt * p->geom.nt, NP = p->NP, PB = p->PB;
  const int chunk = std::max(1, std::min(NP, (1 << 22) / ntiles));
  unsigned *d_count = nullptr, *d_lines = nullptr, *d_off = nullptr;
  const size_t scratch = (size_t)chunk * ntiles;
  if (cudaMalloc(&d_count, scratch * 4) != cudaSuccess || cudaMalloc(&d_lines, scratch * 4) != cudaSuccess ||
      cudaMalloc(&d_off, scratch * 4) != cudaSuccess) {
    cudaGetLastError();
    if (d_count) cudaFree(d_count);
    if (d_lines) cudaFree(d_lines);
    return fail(p, LAM_ENOMEM_DEVICE, "work-list scratch of %zu bytes does not fit", scratch * 12);
  }
  std::vector<unsigned> counts((size_t)NP * ntiles), lines((size_t)NP * ntiles), offs((size_t)NP * ntiles);
  lam_status st = LAM_OK;
  auto launch = [&](int p0, int np, bool fill) {
    JobsArgs a{p->geom, p0, np, d_count, d_lines, d_off, p->d_jobs};
    const long long total = (long long)np * ntiles;
    const unsigned blocks = (unsigned)((total + 63) / 64);
    dispatch_W(p->W, [&](auto Wc) {
      constexpr int W = decltype(Wc)::value;
      if (fill) k_jobs<W, true><<<blocks, 64>>>(a);
      else k_jobs<W, false><<<blocks, 64>>>(a);
    });
  };
  for (int p0 = 0; p0 < NP && st == LAM_OK; p0 += chunk) {
    const int np = std::min(chunk, NP - p0);
    launch(p0, np, false);
    cudaError_t e = cudaMemcpy(counts.data() + (size_t)p0 * ntiles, d_count, (size_t)np * ntiles * 4, cudaMemcpyDeviceToHost);
    if (e == cudaSuccess) e = cudaMemcpy(lines.data() + (size_t)p0 * ntiles, d_lines, (size_t)np * ntiles * 4, cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) st = fail(p, LAM_ECUDA, "work-list count pass: %s", cudaGetErrorString(e));
  }
  if (st == LAM_OK) {
    const int nb = (NP + PB - 1) / PB;
    p->job_off.assign(nb + 1, 0);
    p->multi_off.assign(nb + 1, 0);
    std::vector<unsigned> multi;
    std::vector<unsigned> order, bucket;
    long long tot = 0;
    const int nt = p->geom.nt;
    for (int b = 0; b < nb; ++b) {
      const size_t i0 = (size_t)b * PB * ntiles, i1 = (size_t)std::min(NP, (b + 1) * PB) * ntiles;
      p->job_off[b] = tot;
      p->multi_off[b] = (long long)multi.size();
      // heaviest tiles first: a stable counting sort by descending line count (top bits of `lines`: image masks)
      order.resize(i1 - i0);
      unsigned kmax = 0;
      for (size_t i = i0; i < i1; ++i) kmax = std::max(kmax, lines[i] & 0xffffffu);
      bucket.assign((size_t)kmax + 2, 0);
      for (size_t i = i0; i < i1; ++i) ++bucket[kmax - (lines[i] & 0xffffffu) + 1];
      for (size_t b = 1; b < bucket.size(); ++b) bucket[b] += bucket[b - 1];
      for (size_t i = i0; i < i1; ++i) order[bucket[kmax - (lines[i] & 0xffffffu)]++] = (unsigned)(i - i0);
      for (unsigned o : order) {
        const size_t i = i0 + o;
        offs[i] = (unsigned)tot;
        tot += counts[i];
        if (counts[i] > 1) {
          const unsigned pl = (unsigned)(i / ntiles), t = (unsigned)(i % ntiles);
          multi.push_back(pl << 16 | (unsigned)(t / nt) << 8 | (unsigned)(t % nt));
        }
      }
    }
    p->job_off[nb] = tot;
    p->multi_off[nb] = (long long)multi.size();
    if (tot > 0xffffffffLL) st = fail(p, LAM_EUNSUPPORTED, "more than 2^32 gridding jobs");
    if (st == LAM_OK) st = dalloc(p, &p->d_jobs, (size_t)tot);
    if (st == LAM_OK) st = upload(p, &p->d_multi, multi);
  }
  for (int p0 = 0; p0 < NP && st == LAM_OK; p0 += chunk) {
    const int np = std::min(chunk, NP - p0);
    cudaMemcpy(d_off, offs.data() + (size_t)p0 * ntiles, (size_t)np * ntiles * 4, cudaMemcpyHostToDevice);
    cudaMemcpy(d_count, counts.data() + (size_t)p0 * ntiles, (size_t)np * ntiles * 4, cudaMemcpyHostToDevice);
    cudaMemcpy(d_lines, lines.data() + (size_t)p0 * ntiles, (size_t)np * ntiles * 4, cudaMemcpyHostToDevice);
    launch(p0, np, true);
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) st = fail(p, LAM_ECUDA, "work-list fill pass: %s", cudaGetErrorString(e));
  }
  cudaFree(d_count);
  cudaFree(d_lines);
  cudaFree(d_off);
  return st;
}

lam_status make_tables(lam_plan* p) {
  lam_status st;
  const int n = p->n, nz = p->nz, h = p->h, w = p->w, M = p->M, M3 = p->M3, W = p->W, NP = p->NP;
  const double sigma = p->prm.oversample;
  // angles
  std::vector<double2> cs(p->ntheta);
  for (int t = 0; t < p->ntheta; ++t) cs[t] = make_double2(std::cos(p->theta[t]), std::sin(p->theta[t]));
  if ((st = upload(p, &p->d_cs, cs)) != LAM_OK) return st;
  // filter x centring phase x 1/(wh) along k_u; centring phase along k_v
  const double cu = std::isnan(p->prm.center_u) ? 0.5 * w : (double)p->prm.center_u;
  const double cv = std::isnan(p->prm.center_v) ? 0.5 * h : (double)p->prm.center_v;
  for (int pass = 0; pass < 2; ++pass) {
    std::vector<double> H;
    filter_response(pass == 0 ? p->prm.filter : 0, w, p->phi, p->ntheta, H);
    std::vector<float2> Pu(w / 2 + 1);
    for (int k = 0; k <= w / 2; ++k) {
      double a = 2.0 * kPi * std::fmod((double)k * cu, (double)w) / w, s = H[k] / ((double)w * h);
      Pu[k] = make_float2((float)(s * std::cos(a)), (float)(s * std::sin(a)));
    }
    if ((st = upload(p, pass == 0 ? &p->d_Pu : &p->d_PuNone, Pu)) != LAM_OK) return st;
  }
  std::vector<float2> Pv(NP);
  for (int q = 0; q < NP; ++q) {
    int kv = q == h / 2 ? -h / 2 : q;
    double a = 2.0 * kPi * std::fmod((double)kv * cv, (double)h) / h;
    Pv[q] = make_float2((float)std::cos(a), (float)std::sin(a));
  }
  if ((st = upload(p, &p->d_Pv, Pv)) != LAM_OK) return st;
  if (p->prm.pad_u) {
    std::vector<double> H2;
    filter_response(p->prm.filter, 2 * w, p->phi, p->ntheta, H2);  // k = 0..w
    std::vector<float> Hp(w + 1);
    for (int k = 0; k <= w; ++k) Hp[k] = (float)(H2[k] / (2.0 * w));
    if ((st = upload(p, &p->d_Hp, Hp)) != LAM_OK) return st;
    if ((st = upload(p, &p->d_tw_w2, twiddles(2 * w))) != LAM_OK) return st;
  }
  if ((st = upload(p, &p->d_tw_w, twiddles(w))) != LAM_OK) return st;
  if ((st = upload(p, &p->d_tw_h, twiddles(h))) != LAM_OK) return st;
  if ((st = upload(p, &p->d_tw_M, twiddles(M))) != LAM_OK) return st;
  if ((st = upload(p, &p->d_tw_M3, twiddles(M3))) != LAM_OK) return st;
  // gridding kernel: polynomial pieces for (xi1, xi2); explicit weights for xi3 (they depend on k_v only)
  p->gk.init(p->prm.kernel, W, sigma, p->prm.shape);
  kernel_poly(p->gk, &p->kp.E[0][0], &p->kp.O[0][0]);
  // x3 gridding as a banded matrix: for grid cell i (stored index m3 mod M3) the planes p < h/2 with a tap on it
  // are contiguous; the k_v = -h/2 plane (p = h/2) is kept apart
  {
    const double cphi = std::cos(p->phi);
    std::vector<int> lo(M3, 0), hi(M3, -1);
    auto cell = [&](int m) { return ((m % M3) + M3) % M3; };
    for (int q = 0; q < h / 2; ++q) {
      double t3 = (double)M3 * q * cphi / h;
      int b = (int)std::ceil(t3 - 0.5 * W);
      for (int j = 0; j < W; ++j) {
        int i = cell(b + j);
        if (hi[i] < lo[i]) lo[i] = hi[i] = q;
        else { lo[i] = std::min(lo[i], q); hi[i] = std::max(hi[i], q); }
      }
    }
    int KZ = 1;
    for (int i = 0; i < M3; ++i) KZ = std::max(KZ, hi[i] - lo[i] + 1);
    p->KZ = KZ;
    std::vector<float> zfull((size_t)M3 * KZ, 0.f), zlastf(M3, 0.f), wz((size_t)NP * W);
    std::vector<int> bz(NP);
    for (int q = 0; q <= h / 2; ++q) {
      int kv = q == h / 2 ? -h / 2 : q;
      double t3 = (double)M3 * kv * cphi / h;
      int b = (int)std::ceil(t3 - 0.5 * W);
      bz[q] = b;
      for (int j = 0; j < W; ++j) {
        int i = cell(b + j);
        float wv = (float)p->gk.kap(t3 - (b + j));
        wz[(size_t)q * W + j] = wv;
        if (q == h / 2) zlastf[i] += wv;
        else zfull[(size_t)i * KZ + (q - lo[i])] += wv;
      }
    }
    // compact the active cells (a tap of some plane lands on them); tables cell-fastest for coalesced reads
    std::vector<int> zidx(M3, -1), zlo, zcnt;
    std::vector<float> zlast;
    for (int i = 0; i < M3; ++i)
      if (hi[i] >= lo[i] || zlastf[i] != 0.f) {
        zidx[i] = (int)zlo.size();
        zlo.push_back(hi[i] >= lo[i] ? lo[i] : 0);
        zcnt.push_back(hi[i] >= lo[i] ? hi[i] - lo[i] + 1 : 0);
        zlast.push_back(zlastf[i]);
      }
    p->nact = (int)zlo.size();
    std::vector<float> ztab((size_t)KZ * p->nact, 0.f);
    for (int i = 0; i < M3; ++i)
      if (zidx[i] >= 0)
        for (int s2 = 0; s2 < KZ; ++s2) ztab[(size_t)s2 * p->nact + zidx[i]] = zfull[(size_t)i * KZ + s2];
    if ((st = upload(p, &p->d_ztab, ztab)) != LAM_OK) return st;
    if ((st = upload(p, &p->d_zlo, zlo)) != LAM_OK) return st;
    if ((st = upload(p, &p->d_zcnt, zcnt)) != LAM_OK) return st;
    if ((st = upload(p, &p->d_zlast, zlast)) != LAM_OK) return st;
    if ((st = upload(p, &p->d_zidx, zidx)) != LAM_OK) return st;
    if ((st = upload(p, &p->d_wz, wz)) != LAM_OK) return st;
    if ((st = upload(p, &p->d_bz, bz)) != LAM_OK) return st;
  }
  std::vector<float> dx(n), dz(nz);
  for (int i = 0; i < n; ++i) dx[i] = (float)(1.0 / p->gk.kaphat((double)(i - n / 2) / M));
  for (int i = 0; i < nz; ++i) dz[i] = (float)(1.0 / p->gk.kaphat((double)(i - nz / 2) / M3));
  if ((st = upload(p, &p->d_dx, dx)) != LAM_OK) return st;
  if ((st = upload(p, &p->d_dz, dz)) != LAM_OK) return st;
  // geometry of the (xi1, xi2) gridding
  SpreadGeom& g = p->geom;
  g.cs = p->d_cs;
  g.rho_unit = (double)M * std::sin(p->phi) / h;
  g.a1 = (float)M / (float)w;
  g.M = M;
  g.nt = M / kTS;
  g.ntheta = p->ntheta;
  g.w = w;
  g.hh = h / 2;
  return LAM_OK;
}

size_t zstage_smem(const lam_plan* p, int cb) {
  const size_t work = std::max((size_t)p->NP * z_pitch(cb), (size_t)(cb / 2) * fft_tfast_pitch(p->M3, cb / 2));
  return (((work + 1) & ~(size_t)1) + (size_t)p->nact * cb) * sizeof(float2);
}

// x3 stage through TMA: tensor map of A viewed as [p][x2][x1] of 8-byte elements, boxes of pbox planes x cb columns
size_t ztma_smem(const lam_plan* p, int cb, int* nbox, int* pbox, int* bufelems) {
  const int nb = (p->NP + 255) / 256;
  int pb = (p->NP + nb - 1) / nb;
  pb = (pb + 7) & ~7;  // every box lands 128-byte aligned for cb >= 2
  if (pb > 256) pb = 256;
  const size_t ain = (size_t)nb * pb * cb, fft = (size_t)(cb / 2) * fft_tfast_pitch(p->M3, cb / 2);
  const size_t be = (std::max(ain, fft) + 15) & ~(size_t)15;
  *nbox = nb; *pbox = pb; *bufelems = (int)be;
  return (2 * be + (size_t)p->nact * cb) * sizeof(float2) + 16;
}

void setup_ztma(lam_plan* p) {
  p->z_tma = false;
  {
    int nsm = 0;
    if (cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, p->device) == cudaSuccess && nsm > 0) p->n_sm = nsm;
    else cudaGetLastError();
  }
  {  // block size of the plain kernel: fewest idle lanes over the rounds of its gridding phase (nact * cb/2 tasks)
    const int total = p->nact * ((1 << p->z_lcb) / 2);
    long bestcost = -1;
    for (int T = 384; T <= 512; T += 32) {
      const long cost = (long)((total + T - 1) / T) * T;
      if (bestcost < 0 || cost < bestcost || (cost == bestcost && T > p->z_threads)) { bestcost = cost; p->z_threads = T; }
    }
  }
  // The TMA-pipelined persistent form (k_zstage_tma) is the default when the tensor map can be encoded and the plan is
  // in core: measured at parity or slightly ahead of the plain kernel at equal columns per block (configs[2], 16
  // columns: 3.25 against 3.29 ms; configs[3], 8 columns: 36.5 against 37.3 ms).  params.z_form = 1
  // selects the plain kernel.
  // Not for sigma*nz >= 2048 (configs[4]: 279 against 219 ms: its gridding phase splits every cell's band over two lanes,
  // which costs more than the prefetch saves when the FFT is that long).
  const int form = p->prm.z_form;  // 0: this policy, 1: plain kernel, 2: TMA form wherever it can be set up
  if (form == 1 || p->spill || (p->M3 > 1024 && form != 2)) return;
  typedef CUresult (*encode_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return;
  }
  // columns per block: the most of 16, 8, 4, 2 whose double buffer fits one SM (one persistent block per SM then; wider
  // rows beat a second resident block, as for the plain kernel)
  int lcb = (p->n % 16 == 0) ? 4 : 3;
  if (p->prm.z_columns) lcb = ilog2(p->prm.z_columns);
  int nbox, pbox, be;
  while (lcb > 1 && ztma_smem(p, 1 << lcb, &nbox, &pbox, &be) > 226 * 1024) --lcb;
  const size_t sm = ztma_smem(p, 1 << lcb, &nbox, &pbox, &be);
  if (sm > 226 * 1024 || (p->n % (1 << lcb)) != 0) return;
  const int cb = 1 << lcb;
  cuuint64_t gdim[3] = {(cuuint64_t)p->n, (cuuint64_t)p->n, (cuuint64_t)p->NP};
  cuuint64_t gstr[2] = {(cuuint64_t)p->n * 8, (cuuint64_t)p->n * p->n * 8};
  cuuint32_t box[3] = {(cuuint32_t)cb, 1, (cuuint32_t)pbox};
  cuuint32_t estr[3] = {1, 1, 1};
  // L2 promotion no wider than a box row: with 128-byte promotion the 64-byte rows of an 8-column box fetched 1.7x the
  // algorithmic bytes from DRAM (ncu, configs[3]: 58 GB for 34 GB)
  const CUtensorMapL2promotion promo = cb >= 16 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B
                                       : cb >= 8 ? CU_TENSOR_MAP_L2_PROMOTION_L2_64B : CU_TENSOR_MAP_L2_PROMOTION_NONE;
  CUresult r = ((encode_fn)fn)(&p->tmapA, CU_TENSOR_MAP_DATA_TYPE_UINT64, 3, (void*)p->d_A, gdim, gstr, box, estr,
                               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, promo,
                               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return;
  // block size: fewest wasted lanes over the rounds of phase 2 (nact * 8 tasks), 384..640 threads
  const int total = p->nact * 8;
  int best = 512;
  long bestcost = -1;
  for (int T = 384; T <= 640; T += 32) {
    const long cost = (long)((total + T - 1) / T) * T;
    if (bestcost < 0 || cost < bestcost || (cost == bestcost && T > best)) { bestcost = cost; best = T; }
  }
  int occ = 0;
  dispatch_log_impl<kLogMin>(p->logM3, [&](auto L_) { occ = decltype(L_)::ztma_occupancy(best, sm); });
  if (occ < 1) return;
  p->z_lcb = lcb; p->z_nbox = nbox; p->z_pbox = pbox; p->z_bufelems = be; p->z_threads = best; p->z_blocks_per_sm = occ;
  p->z_smem = sm;
  p->z_tma = true;
}

}  // namespace

// ====================================================================================================================
extern "C" {

const char* lam_version(void) { return "lam-b200 0.4 (sm_100a)"; }

void lam_default_params(lam_params* p) {
  if (!p) return;
  memset(p, 0, sizeof *p);
  p->nz = 0;
  p->kernel = LAM_KERNEL_KB;
  p->width = 6;
  p->oversample = 2.0f;
  p->shape = 0.f;
  p->filter = LAM_FILTER_RAMP;
  p->input = LAM_INPUT_F32;
  p->center_u = NAN;
  p->center_v = NAN;
  p->t_min = 1e-6f;
  p->device_bytes = 0;
  p->plane_batch = 0;
  p->theta_chunk = 0;
  p->pad_u = 0;
  p->spectral_alpha = 0.f;
  p->z_form = 0;
  p->z_columns = 0;
}

const char* lam_last_error(const lam_plan* plan) { return plan ? plan->err.c_str() : g_create_error.c_str(); }

void lam_destroy(lam_plan* plan) {
  if (!plan) return;
  cudaSetDevice(plan->device);
  free_all(plan);
  delete plan;
}

lam_status lam_create(int n, int h, int w, int n_theta, float phi_rad, const float* theta_rad, const lam_params* prm,
                      lam_plan** out) {
  if (!out) return fail(nullptr, LAM_EINVAL, "out is NULL");
  *out = nullptr;
  lam_params P;
  if (prm) P = *prm;
  else lam_default_params(&P);
  if (P.nz == 0) P.nz = n;
  if (P.width == 0) P.width = 6;
  if (P.oversample == 0.f) P.oversample = 2.0f;
  if (P.t_min == 0.f) P.t_min = 1e-6f;
  if (n < 2 || h < 2 || w < 2 || P.nz < 2 || n_theta < 1 || !theta_rad)
    return fail(nullptr, LAM_EINVAL, "n, nz, h, w must be >= 2, n_theta >= 1, theta not NULL");
  if ((n | h | w | P.nz) & 1) return fail(nullptr, LAM_EINVAL, "n, nz, h, w must be even");
  if (!(phi_rad >= 0.f) || !(phi_rad < 1.5707963f)) return fail(nullptr, LAM_EINVAL, "phi must be in [0, pi/2)");
  if (P.kernel != LAM_KERNEL_KB && P.kernel != LAM_KERNEL_GAUSS) return fail(nullptr, LAM_EINVAL, "unknown kernel");
  if (P.filter < 0 || P.filter > 3) return fail(nullptr, LAM_EINVAL, "unknown filter");
  if (!(P.spectral_alpha >= 0.f)) return fail(nullptr, LAM_EINVAL, "spectral_alpha must be >= 0");
  if (P.pad_u != 0 && P.pad_u != 1) return fail(nullptr, LAM_EINVAL, "pad_u must be 0 or 1");
  if (P.z_form < 0 || P.z_form > 2) return fail(nullptr, LAM_EINVAL, "z_form must be 0 (auto), 1 (plain kernel) or 2 (TMA form)");
  if (P.z_columns != 0 && P.z_columns != 2 && P.z_columns != 4 && P.z_columns != 8 && P.z_columns != 16)
    return fail(nullptr, LAM_EINVAL, "z_columns must be 0 (auto), 2, 4, 8 or 16");
  if (P.z_columns && n % P.z_columns) return fail(nullptr, LAM_EINVAL, "z_columns must divide n");
  if (P.pad_u && w > 4096) return fail(nullptr, LAM_EUNSUPPORTED, "pad_u needs w <= 4096 (rows of 2w samples)");
  if (P.input != LAM_INPUT_F32 && P.input != LAM_INPUT_U16_RAW) return fail(nullptr, LAM_EINVAL, "unknown input type");
  if (P.width != 4 && P.width != 6 && P.width != 8) return fail(nullptr, LAM_EUNSUPPORTED, "width must be 4, 6 or 8");
  if (!(P.oversample >= 1.25f) || !(P.oversample <= 4.f)) return fail(nullptr, LAM_EINVAL, "oversample must be in [1.25, 4]");
  if (!(P.shape >= 0.f)) return fail(nullptr, LAM_EINVAL, "shape must be >= 0");
  double Md = (double)P.oversample * n, M3d = (double)P.oversample * P.nz;
  int M = (int)std::lround(Md), M3 = (int)std::lround(M3d);
  if (std::fabs(Md - M) > 1e-6 || std::fabs(M3d - M3) > 1e-6 || !pow2(M) || !pow2(M3) || !pow2(w) || !pow2(h))
    return fail(nullptr, LAM_EUNSUPPORTED, "w, h, sigma*n and sigma*nz must be powers of two (got %d, %d, %g, %g)", w, h, Md, M3d);
  const int lo = 1 << kLogMin, hi = 1 << kLogMax;
  if (w < lo || w > hi || h < lo || h > hi || M < 64 || M > hi || M3 < lo || M3 > hi)
    return fail(nullptr, LAM_EUNSUPPORTED, "w, h, sigma*nz must be in [32, 8192] and sigma*n in [64, 8192]");
  if (h / 2 + 1 > 0x1fff || M / kTS > 0x100 || n_theta > 0x3fff)
    return fail(nullptr, LAM_EUNSUPPORTED, "h <= 16382, sigma*n <= 16384 and n_theta <= 16383 in this build");
  if (M3 < 2 * P.width || M < 2 * P.width) return fail(nullptr, LAM_EINVAL, "grid smaller than the kernel footprint");

  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    cudaGetLastError();
    return fail(nullptr, LAM_ECUDA, "no CUDA device (this library has no CPU path)");
  }
  lam_plan* p = new (std::nothrow) lam_plan;
  if (!p) return fail(nullptr, LAM_ENOMEM_HOST, "out of host memory");
  cudaGetDevice(&p->device);
  p->n = n; p->nz = P.nz; p->h = h; p->w = w; p->ntheta = n_theta; p->phi = phi_rad; p->prm = P;
  p->theta.assign(theta_rad, theta_rad + n_theta);
  p->M = M; p->M3 = M3; p->W = P.width; p->NP = h / 2 + 1;
  p->WR = (w / 2 + 1 + 7) & ~7;
  p->WQ = (w + 1 + 7) & ~7;
  p->logw = ilog2(w); p->logh = ilog2(h); p->logM = ilog2(M); p->logM3 = ilog2(M3);

  auto bail = [&](lam_status st) {
    g_create_error = p->err;
    free_all(p);
    delete p;
    return st;
  };
  lam_status st = make_tables(p);
  if (st != LAM_OK) return bail(st);

  // block shapes
  p->rows_nb = std::min(h / 2, std::max(1, 4096 / w));
  p->rows_nb_pad = std::min(h / 2, std::max(1, 1024 / w));  // two buffers of 2w samples per row pair
  p->x1_nb = std::max(1, std::min(M, 4096 / M));
  auto tfast_lognb = [](int len, int lmax = 3) { int l = lmax; while (l > 0 && (size_t)(1 << l) * fft_tfast_pitch(len, 1 << l) * 8 > 200 * 1024) --l; return l; };
  p->cols_lcb = tfast_lognb(h);
  p->x2_lnb = tfast_lognb(M);
  if (n % 8) return bail(fail(p, LAM_EUNSUPPORTED, "n must be a multiple of 8"));
  // x3 stage: 8 columns per block, fewer when that would leave one block per SM (>= 2 blocks of <= 100 KB)
  // x3 stage, columns per block.  Measured (configs[2], [3]): 16 columns when two blocks still share an SM (128-byte rows,
  // conflict-free: S4 3.8 -> 3.3 ms), else 8 columns even at one block per SM (configs[3]: 35.0 ms against 41.8 ms with
  // 4 columns and two blocks) up to sigma*nz = 1024; for longer transforms 4 columns and two blocks (configs[4]: 219
  // against 299 ms), else whatever fits.
  p->z_lcb = 3;
  if (n % 16 == 0 && zstage_smem(p, 16) <= 112 * 1024) p->z_lcb = 4;
  else if (zstage_smem(p, 8) > 112 * 1024 && M3 > 1024 && zstage_smem(p, 4) <= 112 * 1024) p->z_lcb = 2;  // configs[4]: 219 against 299 ms
  while (p->z_lcb > 1 && zstage_smem(p, 1 << p->z_lcb) > 220 * 1024) --p->z_lcb;
  if (P.z_columns) {
    p->z_lcb = ilog2(P.z_columns);
    while (p->z_lcb > 1 && zstage_smem(p, 1 << p->z_lcb) > 220 * 1024) --p->z_lcb;
  }
  if (zstage_smem(p, 1 << p->z_lcb) > 220 * 1024) return bail(fail(p, LAM_EUNSUPPORTED, "x3 stage does not fit shared memory (h = %d, sigma*nz = %d)", h, M3));
  // workspace: batch sizes from the budget
  size_t freeb = 0, totalb = 0;
  if (cudaMemGetInfo(&freeb, &totalb) != cudaSuccess) return bail(fail(p, LAM_ECUDA, "cudaMemGetInfo failed"));
  size_t budget = P.device_bytes ? P.device_bytes : (size_t)(0.9 * (double)freeb);
  const size_t gplane = (size_t)M * M * 8, tplane = (size_t)M * n * 8;
  p->PB = P.plane_batch > 0 ? P.plane_batch : (int)std::max<size_t>(1, std::min<size_t>(p->NP, ((size_t)4 << 30) / (gplane + tplane)));
  p->PB = std::min(p->PB, p->NP);
  const size_t rproj = (size_t)h * p->WR * 8;
  p->TC = P.theta_chunk > 0 ? P.theta_chunk : (int)std::max<size_t>(1, std::min<size_t>(n_theta, ((size_t)1 << 30) / rproj));
  p->TC = std::min(p->TC, n_theta);
  // The spectra planes S[p] die as the planes are gridded and the cropped planes A[p] are born at the same pace, so both
  // share one arena: A grows from the front, S sits right-aligned at the back; a batch of PB planes may be in flight.
  const size_t splane = (size_t)n_theta * p->WQ, aplane = (size_t)n * n;
  const size_t arena = std::max((size_t)p->PB * aplane + (size_t)p->NP * splane, (size_t)p->NP * aplane + (size_t)p->PB * splane);
  // T holds the x1-transformed planes of one sub-batch.  Measured (configs[2], [3]): sub-batches small enough to keep T
  // in L2 (1-4 planes) are SLOWER than whole batches (S3 13.7 / 11.6 / 11.1 ms at 1 / 2 / 4 planes against 9.7 ms): the
  // passes are issue-bound, not HBM-bound, and short launches pay their tails.  So T covers the whole plane batch.
  p->TSB = p->PB;
  // the gridding work lists are allocated by build_jobs: about one 32-byte job per (plane, tile)
  const size_t jobs_est = (size_t)((double)p->NP * (M / kTS) * (M / kTS) * 1.1) * sizeof(Job);
  const size_t need = (size_t)p->TC * rproj + arena * 8 + (size_t)p->PB * gplane + (size_t)p->TSB * tplane + jobs_est + p->device_bytes;
  if (need <= budget) {
    if ((st = dalloc(p, &p->d_R, (size_t)p->TC * h * p->WR)) != LAM_OK) return bail(st);
    if ((st = dalloc(p, &p->d_arena, arena)) != LAM_OK) return bail(st);
    p->d_A = p->d_arena;
    p->d_S = p->d_arena + (arena - (size_t)p->NP * splane);
  } else {
    // ---- spilled mode: size every buffer from the budget ----
    p->spill = true;
    const size_t left0 = budget > jobs_est + p->device_bytes ? budget - jobs_est - p->device_bytes : 0;
    if (P.theta_chunk <= 0) p->TC = (int)std::max<size_t>(1, std::min<size_t>(p->TC, left0 / 16 / rproj));
    const size_t per_plane = gplane + tplane + 2 * aplane * 8;  // G, T and the two staging copies of the cropped plane
    if (P.plane_batch <= 0) p->PB = (int)std::max<size_t>(1, std::min<size_t>(p->PB, left0 / 4 / per_plane));
    p->TSB = p->PB;
    const size_t slab_row = (size_t)p->NP * n * 8;               // one x2 row of every plane
    p->ZRs = (int)std::max<size_t>(1, std::min<size_t>(n, left0 / 8 / (2 * slab_row)));
    while (n % p->ZRs) --p->ZRs;
    const size_t fixed = (size_t)p->TC * rproj + (size_t)p->PB * per_plane + 2 * (size_t)p->ZRs * slab_row;
    const size_t sbytes = splane * 8;
    size_t nband = left0 > fixed ? (left0 - fixed) / sbytes : 0;
    nband = std::min<size_t>(nband, p->NP);
    nband -= nband % p->PB;
    if (nband < (size_t)p->PB)
      return bail(fail(p, LAM_ENOMEM_DEVICE, "budget of %.2f GB is too small even for the spilled schedule (needs %.2f GB for one batch of %d planes)",
                       budget / 1e9, (fixed + (size_t)p->PB * sbytes + jobs_est + p->device_bytes) / 1e9, p->PB));
    p->band = (int)nband;
    if ((st = dalloc(p, &p->d_R, (size_t)p->TC * h * p->WR)) != LAM_OK) return bail(st);
    if ((st = dalloc(p, &p->d_arena, (size_t)p->band * splane)) != LAM_OK) return bail(st);
    p->d_S = p->d_arena;
    p->d_A = nullptr;
    for (int i = 0; i < 2; ++i) {
      if ((st = dalloc(p, &p->d_Ab[i], (size_t)p->PB * aplane)) != LAM_OK) return bail(st);
      if ((st = dalloc(p, &p->d_As2[i], (size_t)p->NP * p->ZRs * n)) != LAM_OK) return bail(st);
      for (cudaEvent_t* ev : {&p->ev_ab_ready[i], &p->ev_ab_free[i], &p->ev_sl_ready[i], &p->ev_sl_free[i]})
        if (cudaEventCreateWithFlags(ev, cudaEventDisableTiming) != cudaSuccess) {
          *ev = nullptr;
          return bail(fail(p, LAM_ECUDA, "spilled schedule: cudaEventCreateWithFlags failed: %s", cudaGetErrorString(cudaGetLastError())));
        }
    }
    const size_t hbytes = (size_t)p->NP * aplane * 8;
    if (cudaHostAlloc((void**)&p->h_A, hbytes, cudaHostAllocDefault) != cudaSuccess) {
      cudaGetLastError();
      p->h_A = nullptr;
      return bail(fail(p, LAM_ENOMEM_HOST, "spilled schedule: %.2f GB of pinned host memory for the cropped planes could not be allocated", hbytes / 1e9));
    }
    p->pinned_bytes += hbytes;
    p->ZR = p->ZRs;  // output slabs of the host-pointer path follow the x3-stage slabs
  }
  if ((st = dalloc(p, &p->d_G, (size_t)p->PB * M * M)) != LAM_OK) return bail(st);
  if ((st = dalloc(p, &p->d_T, (size_t)p->TSB * M * n)) != LAM_OK) return bail(st);
  setup_ztma(p);
  if ((st = build_jobs(p)) != LAM_OK) return bail(st);
  if (cudaDeviceSynchronize() != cudaSuccess) return bail(fail(p, LAM_ECUDA, "plan setup failed: %s", cudaGetErrorString(cudaGetLastError())));
  *out = p;
  return LAM_OK;
}

lam_status lam_set_darkflat(lam_plan* p, const float* dark, const float* flat) {
  if (!p) return LAM_EINVAL;
  if (!dark || !flat) return fail(p, LAM_EINVAL, "dark / flat is NULL");
  cudaSetDevice(p->device);
  size_t cnt = (size_t)p->h * p->w;
  lam_status st;
  if (!p->d_dark && (st = dalloc(p, &p->d_dark, cnt)) != LAM_OK) return st;
  if (!p->d_flat && (st = dalloc(p, &p->d_flat, cnt)) != LAM_OK) return st;
  CU(p, cudaMemcpy(p->d_dark, dark, cnt * 4, cudaMemcpyDefault));
  CU(p, cudaMemcpy(p->d_flat, flat, cnt * 4, cudaMemcpyDefault));
  if (!p->d_df && (st = dalloc(p, &p->d_df, cnt)) != LAM_OK) return st;
  k_darkflat<<<(unsigned)((cnt + 255) / 256), 256>>>(p->d_dark, p->d_flat, p->d_df, cnt);
  CU(p, cudaDeviceSynchronize());
  p->have_darkflat = true;
  return LAM_OK;
}

lam_status lam_set_profiling(lam_plan* p, int on) {
  if (!p) return LAM_EINVAL;
  p->profiling = on != 0;
  p->copy_only = on == 2;
  return LAM_OK;
}

static bool is_device_ptr(const void* q) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, q) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

// S0 + S1 for projections [th0, th0 + nth) at device pointer `chunk` (the first projection of the chunk)
static void launch_s1(lam_plan* p, const void* chunk, int th0, int nth, cudaStream_t s, int p_lo = 0, int p_hi = 1 << 30) {
  if (p->copy_only) return;
  const bool raw = p->prm.input == LAM_INPUT_U16_RAW;
  if (p->prm.pad_u && p->prm.filter != LAM_FILTER_NONE) {
    RowsPadArgs pa{{chunk, p->d_df, p->prm.t_min, p->d_R, p->d_PuNone, p->d_tw_w, p->h, p->WR, p->rows_nb_pad}, p->d_Hp, p->d_tw_w2};
    dim3 gr(p->h / 2 / p->rows_nb_pad, nth);
    size_t smr = (size_t)2 * p->rows_nb_pad * fft_span(2 * p->w) * sizeof(float2);
    DISPATCH_LOG(p->logw, rows_pad(raw, gr, smr, s, pa));
  } else {
    RowsArgs ra{chunk, p->d_df, p->prm.t_min, p->d_R, p->d_Pu, p->d_tw_w, p->h, p->WR, p->rows_nb};
    dim3 gr(p->h / 2 / p->rows_nb, nth);
    size_t smr = (size_t)p->rows_nb * fft_span(p->w) * sizeof(float2);
    DISPATCH_LOG(p->logw, rows(raw, gr, smr, s, ra));
  }
  const int cb = 1 << p->cols_lcb;
  // banded (spilled) mode: the stored band starts at plane p_lo; the kernels index planes absolutely
  float2* S0 = p->d_S - (size_t)(p->spill ? p_lo : 0) * p->ntheta * p->WQ;
  ColsArgs ca{p->d_R, S0, p->d_Pv, p->d_tw_h, p->w, p->WR, p->WQ, p->ntheta, th0, p->cols_lcb, p_lo, p_hi, p->prm.spectral_alpha};
  dim3 gc((p->w / 2 + 1 + cb - 1) / cb, nth);
  size_t smc = (size_t)cb * fft_tfast_pitch(p->h, cb) * sizeof(float2);
  DISPATCH_LOG(p->logh, cols(gc, (size_t)cb * p->h >= 16384 ? 512 : 256, smc, s, ca));
  p->launches += 2;
}

// S2 + S3 (x1, x2) for planes [p0, p0 + np): p0 is a multiple of the plane batch.  slice = true: S2 only, then the
// planes are added, each times its x3 phase, onto the single fine grid of lam_backproject_slice.
static void launch_planes(lam_plan* p, int p0, int np, cudaStream_t s, bool slice = false, float2* Aout = nullptr, int band_lo = 0) {
  if (p->copy_only) return;
  if (!Aout) Aout = p->d_A + (size_t)p0 * p->n * p->n;
  const int b = p0 / p->PB;
  SpreadArgs sa{p->geom, p->kp, p->d_jobs + p->job_off[b], p->job_off[b + 1] - p->job_off[b],
                p->d_S - (size_t)band_lo * p->ntheta * p->WQ, p->WQ, p->d_G, p0,
                p->d_multi + p->multi_off[b], p->multi_off[b + 1] - p->multi_off[b]};
  {
    StageScope sc(p, 1, s);
    if (sa.nmulti > 0) {
      k_zero_tiles<<<(unsigned)((sa.nmulti + 7) / 8), 256, 0, s>>>(sa);
      note_launch();
      p->launches += 1;
    }
    dispatch_W(p->W, [&](auto Wc) {
      constexpr int W = decltype(Wc)::value;
      size_t sm = spread_smem();
      cudaFuncSetAttribute(k_spread<W>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
      k_spread<W><<<(unsigned)sa.njobs, 32 * kSW, sm, s>>>(sa);
      note_launch();
    });
  }
  if (slice) {
    const size_t cells = (size_t)p->M * p->M;
    k_slice_reduce<<<p->n_sm * 8, 256, 0, s>>>(p->d_G, p->d_Gs, p->d_zph + p0, np, cells);
    note_launch();
    p->launches += 2;
    return;
  }
  {
    // x1 then x2 on sub-batches of TSB planes through ONE small T buffer: T is written and re-read while it is still
    // in L2 (its lines are overwritten by the next sub-batch before they are evicted), so only G and A move through HBM
    StageScope sc(p, 2, s);
    const int nb2 = 1 << p->x2_lnb;
    for (int q = 0; q < np; q += p->TSB) {
      const int nq = std::min(p->TSB, np - q);
      IfftArgs a1{p->d_G + (size_t)q * p->M * p->M, p->d_T, p->d_tw_M, p->n, p->x1_nb, 0};
      DISPATCH_LOG(p->logM, x1(dim3(p->M / p->x1_nb, nq), (size_t)p->x1_nb * fft_span(p->M) * sizeof(float2), s, a1));
      IfftArgs a2{p->d_T, Aout + (size_t)q * p->n * p->n, p->d_tw_M, p->n, nb2, p->x2_lnb};
      DISPATCH_LOG(p->logM, x2(dim3(p->n / nb2, nq), (size_t)nb2 * p->M >= 16384 ? 512 : 256,
                               (size_t)nb2 * fft_tfast_pitch(p->M, nb2) * sizeof(float2), s, a2));
      p->launches += 2;
    }
  }
  p->launches += 1;
}

// x3 stage for x2 rows [x2_0, x2_0 + rows); out holds x2 row `out_x2_0` in its first row, z-stride `zstride` floats
static void launch_z(lam_plan* p, float* out, size_t zstride, int x2_0, int rows, int out_x2_0, cudaStream_t s,
                     const float2* Abuf = nullptr, size_t a_pstride = 0, int a_x2_0 = 0) {
  if (p->copy_only) return;
  StageScope sc(p, 3, s);
  if (!Abuf) { Abuf = p->d_A; a_pstride = (size_t)p->n * p->n; a_x2_0 = 0; }
  ZArgs za{Abuf, a_pstride, a_x2_0, out, zstride, p->d_tw_M3, p->d_ztab, p->d_zlo, p->d_zcnt, p->d_zlast, p->d_zidx, p->d_dx, p->d_dz,
           p->n, p->nz, p->NP, p->nact, p->z_lcb, x2_0, out_x2_0};
  if (p->z_tma) {
    ZTmaArgs ta{za, p->n >> p->z_lcb, rows * (p->n >> p->z_lcb), p->z_nbox, p->z_pbox, p->z_bufelems};
    const int grid = std::min(ta.nitems, p->n_sm * p->z_blocks_per_sm);
    DISPATCH_LOG(p->logM3, ztma(grid, p->z_threads, p->z_smem, s, p->tmapA, ta));
  } else {
    DISPATCH_LOG(p->logM3, z(dim3(p->n >> p->z_lcb, rows), p->z_threads, zstage_smem(p, 1 << p->z_lcb), s, za));
  }
  p->launches += 1;
}

static lam_status init_copy_streams(lam_plan* p) {
  if (p->s_h2d) return LAM_OK;
  CU(p, cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming));
  CU(p, cudaStreamCreateWithFlags(&p->s_h2d, cudaStreamNonBlocking));
  CU(p, cudaStreamCreateWithFlags(&p->s_d2h, cudaStreamNonBlocking));
  return LAM_OK;
}

static lam_status init_host_path(lam_plan* p) {
  if (p->host_path_ready) return LAM_OK;
  {
    lam_status st0 = init_copy_streams(p);
    if (st0 != LAM_OK) return st0;
  }
  const size_t esz = p->prm.input == LAM_INPUT_U16_RAW ? 2 : 4;
  if (p->ZR == 0) {
    p->ZR = (int)std::max<size_t>(1, std::min<size_t>(p->n, ((size_t)256 << 20) / ((size_t)p->nz * p->n * 4)));
    while (p->n % p->ZR) --p->ZR;
  }
  lam_status st;
  for (int i = 0; i < 2; ++i) {
    char* q = nullptr;
    if ((st = dalloc(p, &q, (size_t)p->TC * p->h * p->w * esz)) != LAM_OK) return st;
    p->d_in[i] = q;
    if ((st = dalloc(p, &p->d_out[i], (size_t)p->nz * p->ZR * p->n)) != LAM_OK) return st;
    CU(p, cudaEventCreateWithFlags(&p->ev_in_ready[i], cudaEventDisableTiming));
    CU(p, cudaEventCreateWithFlags(&p->ev_in_free[i], cudaEventDisableTiming));
    CU(p, cudaEventCreateWithFlags(&p->ev_out_ready[i], cudaEventDisableTiming));
    CU(p, cudaEventCreateWithFlags(&p->ev_out_free[i], cudaEventDisableTiming));
  }
  p->host_path_ready = true;
  return LAM_OK;
}

// S0 + S1 over every projection for the planes [p_lo, p_hi) (all planes in core; one band in spilled mode).  Device
// projections are read in place; host projections stream in chunks on the copy stream, double-buffered against the
// kernels.  p->chunk_ctr numbers the chunks of the whole call: the two staging buffers alternate
// across bands as well.
static lam_status run_s1_all(lam_plan* p, const void* proj, bool proj_dev, cudaStream_t s, int p_lo, int p_hi) {
  const size_t esz = p->prm.input == LAM_INPUT_U16_RAW ? 2 : 4;
  const size_t pbytes = (size_t)p->h * p->w * esz;
  if (proj_dev) {
    StageScope sc(p, 0, s);
    for (int th0 = 0; th0 < p->ntheta; th0 += p->TC) {
      int nth = std::min(p->TC, p->ntheta - th0);
      launch_s1(p, (const char*)proj + (size_t)th0 * pbytes, th0, nth, s, p_lo, p_hi);
    }
    return LAM_OK;
  }
  if (p->chunk_ctr == 0) {
    CU(p, cudaEventRecord(p->ev_fork, s));
    CU(p, cudaStreamWaitEvent(p->s_h2d, p->ev_fork, 0));
  }
  for (int th0 = 0; th0 < p->ntheta; th0 += p->TC, ++p->chunk_ctr) {
    const int nth = std::min(p->TC, p->ntheta - th0), c = p->chunk_ctr, b = c & 1;
    if (c >= 2) CU(p, cudaStreamWaitEvent(p->s_h2d, p->ev_in_free[b], 0));
    {
      StageScope sc(p, 4, p->s_h2d);
      CU(p, cudaMemcpyAsync(p->d_in[b], (const char*)proj + (size_t)th0 * pbytes, (size_t)nth * pbytes, cudaMemcpyHostToDevice, p->s_h2d));
    }
    CU(p, cudaEventRecord(p->ev_in_ready[b], p->s_h2d));
    CU(p, cudaStreamWaitEvent(s, p->ev_in_ready[b], 0));
    {
      StageScope sc(p, 0, s);
      launch_s1(p, p->d_in[b], th0, nth, s, p_lo, p_hi);
    }
    CU(p, cudaEventRecord(p->ev_in_free[b], s));
  }
  return LAM_OK;
}

lam_status lam_backproject(lam_plan* p, const void* proj, float* vol, void* cuda_stream) {
  if (!p) return LAM_EINVAL;
  if (!proj || !vol) return fail(p, LAM_EINVAL, "proj / vol is NULL");
  if (p->prm.input == LAM_INPUT_U16_RAW && !p->have_darkflat) return fail(p, LAM_EINVAL, "uint16 input needs lam_set_darkflat first");
  cudaSetDevice(p->device);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const bool proj_dev = is_device_ptr(proj), vol_dev = is_device_ptr(vol);
  if (!proj_dev || !vol_dev) {
    lam_status st = init_host_path(p);
    if (st != LAM_OK) return st;
  }
  if (p->spill) {
    lam_status st = init_copy_streams(p);
    if (st != LAM_OK) return st;
  }
  p->launches = 0;
  g_launch_error = cudaSuccess;
  p->events_used = 0;
  p->stage_valid = false;
  {
    StageScope total(p, 5, s);
    {
      p->chunk_ctr = 0;
      lam_status st0 = run_s1_all(p, proj, proj_dev, s, 0, p->spill ? p->band : (1 << 30));
      if (st0 != LAM_OK) return st0;
    }
    if (!p->spill)
      for (int p0 = 0; p0 < p->NP; p0 += p->PB) launch_planes(p, p0, std::min(p->PB, p->NP - p0), s);
    if (p->spill) {
      // ---- spilled schedule: bands of planes; band 0 has been transformed above, the others repeat S0+S1 ----
      const size_t aplane = (size_t)p->n * p->n;
      int nb_done = 0;
      for (int p_lo = 0; p_lo < p->NP; p_lo += p->band) {
        const int p_hi = std::min(p->NP, p_lo + p->band);
        if (p_lo > 0) {
          lam_status st1 = run_s1_all(p, proj, proj_dev, s, p_lo, p_hi);
          if (st1 != LAM_OK) return st1;
        }
        for (int p0 = p_lo; p0 < p_hi; p0 += p->PB, ++nb_done) {
          const int np = std::min(p->PB, p_hi - p0), b = nb_done & 1;
          if (nb_done >= 2) CU(p, cudaStreamWaitEvent(s, p->ev_ab_free[b], 0));
          launch_planes(p, p0, np, s, false, p->d_Ab[b], p_lo);
          CU(p, cudaEventRecord(p->ev_ab_ready[b], s));
          CU(p, cudaStreamWaitEvent(p->s_d2h, p->ev_ab_ready[b], 0));
          {
            StageScope sc(p, 4, p->s_d2h);
            CU(p, cudaMemcpyAsync(p->h_A + (size_t)p0 * aplane, p->d_Ab[b], (size_t)np * aplane * sizeof(float2), cudaMemcpyDeviceToHost, p->s_d2h));
          }
          CU(p, cudaEventRecord(p->ev_ab_free[b], p->s_d2h));
        }
      }
      CU(p, cudaEventRecord(p->ev_fork, p->s_d2h));
      CU(p, cudaStreamWaitEvent(p->s_h2d, p->ev_fork, 0));  // the slabs are read back only after the last plane has left
      CU(p, cudaStreamWaitEvent(s, p->ev_fork, 0));
      int c = 0;
      for (int r0 = 0; r0 < p->n; r0 += p->ZRs, ++c) {
        const int b = c & 1;
        if (c >= 2) CU(p, cudaStreamWaitEvent(p->s_h2d, p->ev_sl_free[b], 0));
        {
          StageScope sc(p, 4, p->s_h2d);
          CU(p, cudaMemcpy2DAsync(p->d_As2[b], (size_t)p->ZRs * p->n * sizeof(float2), p->h_A + (size_t)r0 * p->n, aplane * sizeof(float2),
                                  (size_t)p->ZRs * p->n * sizeof(float2), p->NP, cudaMemcpyHostToDevice, p->s_h2d));
        }
        CU(p, cudaEventRecord(p->ev_sl_ready[b], p->s_h2d));
        CU(p, cudaStreamWaitEvent(s, p->ev_sl_ready[b], 0));
        if (vol_dev) {
          launch_z(p, vol, (size_t)p->n * p->n, r0, p->ZRs, 0, s, p->d_As2[b], (size_t)p->ZRs * p->n, r0);
        } else {
          if (c >= 2) CU(p, cudaStreamWaitEvent(s, p->ev_out_free[b], 0));
          launch_z(p, p->d_out[b], (size_t)p->ZR * p->n, r0, p->ZRs, r0, s, p->d_As2[b], (size_t)p->ZRs * p->n, r0);
          CU(p, cudaEventRecord(p->ev_out_ready[b], s));
          CU(p, cudaStreamWaitEvent(p->s_d2h, p->ev_out_ready[b], 0));
          {
            StageScope sc(p, 4, p->s_d2h);
            CU(p, cudaMemcpy2DAsync(vol + (size_t)r0 * p->n, (size_t)p->n * p->n * 4, p->d_out[b], (size_t)p->ZR * p->n * 4,
                                    (size_t)p->ZR * p->n * 4, p->nz, cudaMemcpyDeviceToHost, p->s_d2h));
          }
          CU(p, cudaEventRecord(p->ev_out_free[b], p->s_d2h));
        }
        CU(p, cudaEventRecord(p->ev_sl_free[b], s));
      }
      if (!vol_dev) {
        CU(p, cudaEventRecord(p->ev_fork, p->s_d2h));
        CU(p, cudaStreamWaitEvent(s, p->ev_fork, 0));
      }
    } else if (vol_dev) {
      launch_z(p, vol, (size_t)p->n * p->n, 0, p->n, 0, s);
    } else {
      // volume leaves in slabs of ZR x2-rows, double-buffered against the x3 stage
      int c = 0;
      for (int r0 = 0; r0 < p->n; r0 += p->ZR, ++c) {
        int b = c & 1;
        if (c >= 2) CU(p, cudaStreamWaitEvent(s, p->ev_out_free[b], 0));
        launch_z(p, p->d_out[b], (size_t)p->ZR * p->n, r0, p->ZR, r0, s);
        CU(p, cudaEventRecord(p->ev_out_ready[b], s));
        CU(p, cudaStreamWaitEvent(p->s_d2h, p->ev_out_ready[b], 0));
        {
          StageScope sc(p, 4, p->s_d2h);
          CU(p, cudaMemcpy2DAsync(vol + (size_t)r0 * p->n, (size_t)p->n * p->n * 4, p->d_out[b], (size_t)p->ZR * p->n * 4,
                                  (size_t)p->ZR * p->n * 4, p->nz, cudaMemcpyDeviceToHost, p->s_d2h));
        }
        CU(p, cudaEventRecord(p->ev_out_free[b], p->s_d2h));
      }
      CU(p, cudaEventRecord(p->ev_fork, p->s_d2h));
      CU(p, cudaStreamWaitEvent(s, p->ev_fork, 0));  // join: the user stream completes after the last copy
    }
  }
  CU(p, cudaGetLastError());
  if (g_launch_error != cudaSuccess) return fail(p, LAM_ECUDA, "kernel launch failed: %s", cudaGetErrorString(g_launch_error));
  p->stage_valid = p->profiling;
  p->last_call_host = !proj_dev || !vol_dev;
  if (p->spill) {
    // the pinned plane store and the slab buffers are plan-owned and shared by every later call, whatever stream it
    // is given: nothing of them is in flight on return.  The x3 kernels on `s` wait for every slab read-back on s_h2d,
    // so s_d2h + s cover all three streams.
    CU(p, cudaStreamSynchronize(p->s_d2h));
    CU(p, cudaStreamSynchronize(s));
  }
  if (!proj_dev) CU(p, cudaStreamSynchronize(p->s_h2d));  // the caller's host projections are consumed on return
  if (!vol_dev) CU(p, cudaStreamSynchronize(p->s_d2h));   // host results are valid on return
  return LAM_OK;
}

lam_status lam_backproject_slice(lam_plan* p, const void* proj, int i3, int n_centers, const float* centers_u, float* out,
                                 void* cuda_stream) {
  if (!p) return LAM_EINVAL;
  if (!proj || !out) return fail(p, LAM_EINVAL, "proj / out is NULL");
  if (i3 < 0 || i3 >= p->nz) return fail(p, LAM_EINVAL, "slice index %d outside [0, %d)", i3, p->nz);
  if (n_centers < 0 || (n_centers > 0 && !centers_u)) return fail(p, LAM_EINVAL, "n_centers < 0 or centers_u is NULL");
  if (p->prm.input == LAM_INPUT_U16_RAW && !p->have_darkflat) return fail(p, LAM_EINVAL, "uint16 input needs lam_set_darkflat first");
  cudaSetDevice(p->device);
  if (!is_device_ptr(proj) || !is_device_ptr(out)) return fail(p, LAM_EUNSUPPORTED, "lam_backproject_slice takes device pointers only");
  if (p->spill) return fail(p, LAM_EUNSUPPORTED, "lam_backproject_slice needs the in-core workspace (the plan runs the spilled schedule)");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const int n = p->n, M = p->M, NP = p->NP, w = p->w, h = p->h;
  lam_status st;
  if (!p->d_Gs) {
    if ((st = dalloc(p, &p->d_Gs, (size_t)M * M)) != LAM_OK) return st;
    if ((st = dalloc(p, &p->d_Ts, (size_t)M * n)) != LAM_OK) return st;
    if ((st = dalloc(p, &p->d_As, (size_t)n * n)) != LAM_OK) return st;
    if ((st = dalloc(p, &p->d_zph, (size_t)NP)) != LAM_OK) return st;
    if ((st = dalloc(p, &p->d_cph, (size_t)p->WQ)) != LAM_OK) return st;
  }
  p->launches = 0;
  g_launch_error = cudaSuccess;
  p->stage_valid = false;
  // exact x3 phase of every plane: e^{2 pi i x3 k_v cos(phi) / h}, x3 = i3 - nz/2 (Eq. 9)
  {
    std::vector<float2> zph(NP);
    const double x3 = (double)(i3 - p->nz / 2), cphi = std::cos(p->phi);
    for (int q = 0; q < NP; ++q) {
      const int kv = q == h / 2 ? -h / 2 : q;
      const double a = 2.0 * kPi * std::fmod(x3 * kv * cphi / h, 1.0);
      zph[q] = make_float2((float)std::cos(a), (float)std::sin(a));
    }
    CU(p, cudaMemcpyAsync(p->d_zph, zph.data(), NP * sizeof(float2), cudaMemcpyHostToDevice, s));
    CU(p, cudaStreamSynchronize(s));  // the pageable source vector dies with this scope
  }
  const size_t esz = p->prm.input == LAM_INPUT_U16_RAW ? 2 : 4;
  const size_t pbytes = (size_t)h * w * esz;
  for (int th0 = 0; th0 < p->ntheta; th0 += p->TC)
    launch_s1(p, (const char*)proj + (size_t)th0 * pbytes, th0, std::min(p->TC, p->ntheta - th0), s);
  const double cu0 = std::isnan(p->prm.center_u) ? 0.5 * w : (double)p->prm.center_u;
  double cu_now = cu0;
  const int nc = std::max(1, n_centers);
  std::vector<float2> cph(p->WQ);
  for (int ic = 0; ic < nc; ++ic) {
    const double cu = n_centers > 0 ? (double)centers_u[ic] : cu0, delta = cu - cu_now;
    if (delta != 0.0) {  // move the rotation axis by delta pixels: a phase on k_u (reading Q13), applied to S in place
      for (int q = 0; q <= w; ++q) {
        const double a = 2.0 * kPi * std::fmod((double)(q - w / 2) * delta / w, 1.0);
        cph[q] = make_float2((float)std::cos(a), (float)std::sin(a));
      }
      CU(p, cudaMemcpyAsync(p->d_cph, cph.data(), (size_t)(w + 1) * sizeof(float2), cudaMemcpyHostToDevice, s));
      CU(p, cudaStreamSynchronize(s));
      k_center_shift<<<dim3((w + 1 + 127) / 128, 1024), 128, 0, s>>>(p->d_S, p->d_cph, p->WQ, w + 1, (size_t)NP * p->ntheta);
      note_launch();
      p->launches += 1;
      cu_now = cu;
    }
    CU(p, cudaMemsetAsync(p->d_Gs, 0, (size_t)M * M * sizeof(float2), s));
    for (int p0 = 0; p0 < NP; p0 += p->PB) launch_planes(p, p0, std::min(p->PB, NP - p0), s, true);
    IfftArgs a1{p->d_Gs, p->d_Ts, p->d_tw_M, n, p->x1_nb, 0};
    DISPATCH_LOG(p->logM, x1(dim3(M / p->x1_nb, 1), (size_t)p->x1_nb * fft_span(M) * sizeof(float2), s, a1));
    const int nb2 = 1 << p->x2_lnb;
    IfftArgs a2{p->d_Ts, p->d_As, p->d_tw_M, n, nb2, p->x2_lnb};
    DISPATCH_LOG(p->logM, x2(dim3(n / nb2, 1), (size_t)nb2 * M >= 16384 ? 512 : 256,
                             (size_t)nb2 * fft_tfast_pitch(M, nb2) * sizeof(float2), s, a2));
    k_slice_out<<<(unsigned)(((size_t)n * n + 255) / 256), 256, 0, s>>>(p->d_As, out + (size_t)ic * n * n, p->d_dx, n);
    note_launch();
    p->launches += 3;
  }
  CU(p, cudaGetLastError());
  if (g_launch_error != cudaSuccess) return fail(p, LAM_ECUDA, "kernel launch failed: %s", cudaGetErrorString(g_launch_error));
  return LAM_OK;
}

}  // extern "C"

// ---- lam_backproject_slice_static: the slice search on scratch memory that is part of the library image --------------
// The five buffers lam_backproject_slice cudaMallocs on its first call (summed fine grid Gs, its x1 transform Ts, the
// cropped plane As, the x3 and axis phase tables) are carved out of ONE file-scope device array instead.  The array is
// zero-initialised device memory that every GPU holds from the moment the library's kernels are loaded on it until the
// process exits: kSliceScratchBytes = 16 MiB, enough for sigma*n <= 1024 at sigma = 2 (n <= 512) with h, w <= 8192.
//
// `g_slice_scratch` below is a HOST-side handle of that array, not a device address: handing it to a kernel or to
// cudaMemsetAsync would make the GPU fault (or scribble over host memory it can reach).  The device address is asked for
// once per device, with that device current, through cudaGetSymbolAddress, and cached in g_slice_scratch_dev[].
constexpr size_t kSliceScratchElems = (size_t)2 << 20;  // float2 elements
constexpr size_t kSliceScratchBytes = kSliceScratchElems * sizeof(float2);
constexpr int kSliceScratchMaxDevices = 64;

static __device__ __align__(256) float2 g_slice_scratch[kSliceScratchElems];

namespace {

std::mutex g_slice_scratch_mu;
float2* g_slice_scratch_dev[kSliceScratchMaxDevices] = {};  // device address of g_slice_scratch, per device ordinal

// Device address of the static scratch on p->device (which must be the current device).
lam_status slice_scratch_address(lam_plan* p, float2** out) {
  if (p->device < 0 || p->device >= kSliceScratchMaxDevices)
    return fail(p, LAM_EUNSUPPORTED, "static slice scratch is tracked for device ordinals below %d (plan is on %d)",
                kSliceScratchMaxDevices, p->device);
  std::lock_guard<std::mutex> lk(g_slice_scratch_mu);
  if (!g_slice_scratch_dev[p->device]) {
    void* q = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&q, g_slice_scratch);
    if (e != cudaSuccess || !q) {
      cudaGetLastError();
      return fail(p, LAM_ECUDA, "cudaGetSymbolAddress(g_slice_scratch) on device %d failed: %s", p->device, cudaGetErrorString(e));
    }
    g_slice_scratch_dev[p->device] = (float2*)q;
  }
  *out = g_slice_scratch_dev[p->device];
  return LAM_OK;
}

// Points the plan's single-slice buffers at the static scratch for the duration of one call and puts the plan's own
// (possibly still null) pointers back afterwards, so that lam_destroy never sees an address it did not allocate.
struct SliceScratchLease {
  lam_plan* p;
  float2 *Gs, *Ts, *As, *zph, *cph;
  bool profiling;
  SliceScratchLease(lam_plan* p_, float2* base, const size_t off[5])
      : p(p_), Gs(p_->d_Gs), Ts(p_->d_Ts), As(p_->d_As), zph(p_->d_zph), cph(p_->d_cph), profiling(p_->profiling) {
    p->d_Gs = base + off[0];
    p->d_Ts = base + off[1];
    p->d_As = base + off[2];
    p->d_zph = base + off[3];
    p->d_cph = base + off[4];
    p->profiling = false;  // stage timing creates CUDA events on demand; this path creates nothing
  }
  ~SliceScratchLease() {
    p->d_Gs = Gs; p->d_Ts = Ts; p->d_As = As; p->d_zph = zph; p->d_cph = cph;
    p->profiling = profiling;
  }
};

}  // namespace

extern "C" {

lam_status lam_backproject_slice_static(lam_plan* p, const void* proj, int i3, int n_centers, const float* centers_u, float* out,
                                        void* cuda_stream) {
  if (!p) return LAM_EINVAL;
  if (p->spill) return fail(p, LAM_EUNSUPPORTED, "lam_backproject_slice_static needs the in-core workspace (the plan runs the spilled schedule)");
  // sub-buffers in the order Gs, Ts, As, zph, cph, each starting on a 256-byte boundary (32 float2)
  const size_t want[5] = {(size_t)p->M * p->M, (size_t)p->M * p->n, (size_t)p->n * p->n, (size_t)p->NP, (size_t)p->WQ};
  size_t off[5], total = 0;
  for (int i = 0; i < 5; ++i) {
    off[i] = total;
    total += (want[i] + 31) / 32 * 32;
  }
  if (total > kSliceScratchElems)
    return fail(p, LAM_EUNSUPPORTED,
                "lam_backproject_slice_static: this plan needs %zu bytes of slice scratch (fine grid %d x %d), the static "
                "scratch holds %zu bytes (sigma*n <= 1024 at sigma = 2); use lam_backproject_slice, which allocates",
                total * sizeof(float2), p->M, p->M, kSliceScratchBytes);
  if (cudaSetDevice(p->device) != cudaSuccess) {
    cudaGetLastError();
    return fail(p, LAM_ECUDA, "cudaSetDevice(%d) failed", p->device);
  }
  float2* base = nullptr;
  lam_status st = slice_scratch_address(p, &base);
  if (st != LAM_OK) return st;
  const size_t bytes_before = p->device_bytes;
  {
    // Every call starts from whatever the previous call (of any plan on this device) left in the scratch.  The only
    // buffer that is accumulated into is Gs, and the slice path zeroes it per centre before gridding; Ts and As are
    // written in full before they are read, the two phase tables are uploaded before their kernels run.
    SliceScratchLease lease(p, base, off);
    st = lam_backproject_slice(p, proj, i3, n_centers, centers_u, out, cuda_stream);
  }
  if (st == LAM_OK && p->device_bytes != bytes_before)
    return fail(p, LAM_ECUDA, "internal: lam_backproject_slice_static allocated %zu bytes of device memory",
                p->device_bytes - bytes_before);
  return st;
}

lam_status lam_forward(lam_plan* p, const float* vol, float* proj, void* cuda_stream) {
  if (!p) return LAM_EINVAL;
  if (!vol || !proj) return fail(p, LAM_EINVAL, "vol / proj is NULL");
  cudaSetDevice(p->device);
  if (!is_device_ptr(vol) || !is_device_ptr(proj)) return fail(p, LAM_EUNSUPPORTED, "lam_forward takes device pointers only");
  if (p->spill) return fail(p, LAM_EUNSUPPORTED, "lam_forward needs the in-core workspace (the plan runs the spilled schedule)");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  p->launches = 0;
  g_launch_error = cudaSuccess;
  p->stage_valid = false;
  const int n = p->n, M = p->M, NP = p->NP;
  // (x3 stage)^T: all columns -> A^T[p][x2][x1]
  {
    ZTArgs za{vol, p->d_A, p->d_tw_M3, p->d_wz, p->d_bz, p->d_dx, p->d_dz, n, p->nz, NP, p->W};
    size_t sm = (size_t)kZCb * fft_tfast_pitch(p->M3, kZCb) * sizeof(float2);
    if (sm > 220 * 1024) return fail(p, LAM_EUNSUPPORTED, "lam_forward: sigma*nz = %d does not fit the x3 stage's shared memory", p->M3);
    DISPATCH_LOG(p->logM3, zT(dim3(n / kZCb, n), sm, s, za));
    p->launches += 1;
  }
  // planes, last batch first (the spectra planes are written right-aligned into the arena the A^T planes leave)
  for (int p0 = ((NP - 1) / p->PB) * p->PB; p0 >= 0; p0 -= p->PB) {
    const int np = std::min(p->PB, NP - p0), nb2 = 1 << p->x2_lnb;
    for (int q = 0; q < np; q += p->TSB) {
      const int nq = std::min(p->TSB, np - q);
      IfftArgs a2{p->d_A + (size_t)(p0 + q) * n * n, p->d_T, p->d_tw_M, n, nb2, p->x2_lnb};
      DISPATCH_LOG(p->logM, x2T(dim3(n / nb2, nq), (size_t)nb2 * M >= 16384 ? 512 : 256,
                                (size_t)nb2 * fft_tfast_pitch(M, nb2) * sizeof(float2), s, a2));
      IfftArgs a1{p->d_T, p->d_G + (size_t)q * M * M, p->d_tw_M, n, p->x1_nb, 0};
      DISPATCH_LOG(p->logM, x1T(dim3(M / p->x1_nb, nq), (size_t)p->x1_nb * fft_span(M) * sizeof(float2), s, a1));
      p->launches += 2;
    }
    const int b = p0 / p->PB;
    GatherArgs ga{p->geom, p->kp, p->d_jobs + p->job_off[b], p->d_G, p->d_S, p->WQ, p0};
    const long long njobs = p->job_off[b + 1] - p->job_off[b];
    dispatch_W(p->W, [&](auto Wc) {
      constexpr int W = decltype(Wc)::value;
      k_gather<W><<<(unsigned)njobs, 32, gather_smem<W>(), s>>>(ga);
      note_launch();
    });
    p->launches += 1;
  }
  // (S1)^T: un-fold + inverse FFT along v, then inverse FFT along u; H = 1 (the filter is not part of L)
  const int cb = 1 << p->cols_lcb, nbr = std::max(1, std::min(p->h, 4096 / p->w));
  for (int th0 = 0; th0 < p->ntheta; th0 += p->TC) {
    const int nth = std::min(p->TC, p->ntheta - th0);
    ColsTArgs ca{p->d_S, p->d_R, p->d_Pv, p->d_tw_h, p->w, p->WR, p->WQ, p->ntheta, th0, p->cols_lcb};
    DISPATCH_LOG(p->logh, colsT(dim3((p->w / 2 + 1 + cb - 1) / cb, nth), (size_t)cb * p->h >= 16384 ? 512 : 256,
                                (size_t)cb * fft_tfast_pitch(p->h, cb) * sizeof(float2), s, ca));
    RowsTArgs ra{p->d_R, proj + (size_t)th0 * p->h * p->w, p->d_PuNone, p->d_tw_w, p->h, p->WR, nbr};
    DISPATCH_LOG(p->logw, rowsT(dim3(p->h / nbr, nth), (size_t)nbr * fft_span(p->w) * sizeof(float2), s, ra));
    p->launches += 2;
  }
  CU(p, cudaGetLastError());
  if (g_launch_error != cudaSuccess) return fail(p, LAM_ECUDA, "kernel launch failed: %s", cudaGetErrorString(g_launch_error));
  return LAM_OK;
}

lam_status lam_admm_tv(lam_plan* p, const float* proj, float* vol, float alpha, float rho, int n_outer, int n_cg, double* history,
                       void* cuda_stream) {
  if (!p) return LAM_EINVAL;
  if (!proj || !vol) return fail(p, LAM_EINVAL, "proj / vol is NULL");
  if (!(alpha >= 0.f) || !(rho > 0.f) || n_outer < 1 || n_cg < 1) return fail(p, LAM_EINVAL, "need alpha >= 0, rho > 0, n_outer >= 1, n_cg >= 1");
  if (p->prm.filter != LAM_FILTER_NONE || p->prm.input != LAM_INPUT_F32 || p->prm.pad_u || p->prm.spectral_alpha != 0.f)
    return fail(p, LAM_EINVAL, "lam_admm_tv needs a plan with filter none, fp32 input, no padding, no spectral multiplier (L^T must be the plain adjoint)");
  cudaSetDevice(p->device);
  if (!is_device_ptr(proj) || !is_device_ptr(vol)) return fail(p, LAM_EUNSUPPORTED, "lam_admm_tv takes device pointers only");
  if (p->spill) return fail(p, LAM_EUNSUPPORTED, "lam_admm_tv needs the in-core workspace (the plan runs the spilled schedule)");
  cudaStream_t s = (cudaStream_t)cuda_stream;
  const size_t nvox = (size_t)p->nz * p->n * p->n, nproj = (size_t)p->ntheta * p->h * p->w;
  lam_status st;
  if (!p->d_tv_g) {
    if ((st = dalloc(p, &p->d_tv_g, nvox)) != LAM_OK) return st;
    if ((st = dalloc(p, &p->d_tv_eta, nvox)) != LAM_OK) return st;
    if ((st = dalloc(p, &p->d_tv_h, nvox)) != LAM_OK) return st;
    if ((st = dalloc(p, &p->d_tv_psi, 3 * nvox)) != LAM_OK) return st;
    if ((st = dalloc(p, &p->d_tv_lam, 3 * nvox)) != LAM_OK) return st;
    if ((st = dalloc(p, &p->d_tv_r, nproj)) != LAM_OK) return st;
    if ((st = dalloc(p, &p->d_tv_acc, 4)) != LAM_OK) return st;
  }
  const TvDims dims{p->n, p->nz};
  const unsigned vb = (unsigned)((nvox + 255) / 256), rb = (unsigned)std::min<size_t>((nvox + 255) / 256, (size_t)p->n_sm * 16),
                 pb = (unsigned)std::min<size_t>((nproj + 255) / 256, (size_t)p->n_sm * 16);
  float *mu = vol, *g = p->d_tv_g, *eta = p->d_tv_eta, *hv = p->d_tv_h, *psi = p->d_tv_psi, *lamv = p->d_tv_lam, *r = p->d_tv_r;
  long long launches = 0;
  // three double sums per CG step, read back together
  auto sums = [&](double out[4]) -> lam_status {
    CU(p, cudaMemcpyAsync(out, p->d_tv_acc, 4 * sizeof(double), cudaMemcpyDeviceToHost, s));
    CU(p, cudaStreamSynchronize(s));
    return LAM_OK;
  };
  CU(p, cudaMemsetAsync(mu, 0, nvox * 4, s));
  CU(p, cudaMemsetAsync(psi, 0, 3 * nvox * 4, s));
  CU(p, cudaMemsetAsync(lamv, 0, 3 * nvox * 4, s));
  double gnorm = 0.0;  // ||grad F|| after the last CG step taken
  for (int k = 0; k < n_outer; ++k) {
    // grad F(mu) = L^T (L mu - d) - rho div(grad mu - psi + lam / rho)                                   (Eq. 18)
    if ((st = lam_forward(p, mu, r, s)) != LAM_OK) return st;
    launches += p->launches;
    k_axpby<<<pb, 256, 0, s>>>(r, 1.f, proj, -1.f, nproj);
    if ((st = lam_backproject(p, r, g, s)) != LAM_OK) return st;
    launches += p->launches;
    k_tv_reggrad<<<vb, 256, 0, s>>>(mu, psi, lamv, rho, g, 1, dims);
    CU(p, cudaMemsetAsync(eta, 0, nvox * 4, s));
    k_axpby<<<rb, 256, 0, s>>>(eta, 0.f, g, -1.f, nvox);  // eta_0 = -grad F
    launches += 3;
    for (int m = 0; m < n_cg; ++m) {
      // exact minimiser of the quadratic F along eta (reading Q19): gamma = -<g, eta> / (|L eta|^2 + rho |grad eta|^2)
      if ((st = lam_forward(p, eta, r, s)) != LAM_OK) return st;
      launches += p->launches;
      CU(p, cudaMemsetAsync(p->d_tv_acc, 0, 4 * sizeof(double), s));
      k_dot<<<pb, 256, 0, s>>>(r, r, nproj, p->d_tv_acc + 0);
      k_tv_gradnorm2<<<rb, 256, 0, s>>>(eta, dims, p->d_tv_acc + 1);
      k_dot<<<rb, 256, 0, s>>>(g, eta, nvox, p->d_tv_acc + 2);
      double a[4];
      if ((st = sums(a)) != LAM_OK) return st;
      const double denom = a[0] + (double)rho * a[1];
      if (!std::isfinite(denom) || !std::isfinite(a[2]))
        return fail(p, LAM_EINVAL, "lam_admm_tv: non-finite step length at outer iteration %d, CG step %d (NaN or Inf in proj?)", k, m);
      if (!(denom > 0.0)) {
        // eta = 0: the subproblem is solved.  The steps that are skipped still own their history slots (k n_cg + m).
        if (history)
          for (int q = m; q < n_cg; ++q) history[(size_t)k * n_cg + q] = gnorm;
        break;
      }
      const double gamma = -a[2] / denom;
      k_axpby<<<rb, 256, 0, s>>>(mu, 1.f, eta, (float)gamma, nvox);
      // H eta = L^T L eta - rho div grad eta;  grad F(mu + gamma eta) = grad F(mu) + gamma H eta  (F is quadratic)
      if ((st = lam_backproject(p, r, hv, s)) != LAM_OK) return st;
      launches += p->launches;
      k_tv_reggrad<<<vb, 256, 0, s>>>(eta, nullptr, nullptr, rho, hv, 1, dims);
      k_axpby<<<rb, 256, 0, s>>>(g, 1.f, hv, (float)gamma, nvox);
      CU(p, cudaMemsetAsync(p->d_tv_acc, 0, 4 * sizeof(double), s));
      k_dot<<<rb, 256, 0, s>>>(g, g, nvox, p->d_tv_acc + 0);
      k_dot<<<rb, 256, 0, s>>>(hv, eta, nvox, p->d_tv_acc + 1);
      if ((st = sums(a)) != LAM_OK) return st;
      // Dai-Yuan: beta = |g_new|^2 / <g_new - g, eta> = |g_new|^2 / (gamma <H eta, eta>)                    (Eq. 19)
      const double dy = gamma * a[1];
      const double beta = dy != 0.0 ? a[0] / dy : 0.0;
      k_axpby<<<rb, 256, 0, s>>>(eta, (float)beta, g, -1.f, nvox);
      launches += 9;
      gnorm = std::sqrt(a[0]);
      if (history) history[(size_t)k * n_cg + m] = gnorm;
    }
    k_tv_shrink<<<vb, 256, 0, s>>>(mu, psi, lamv, alpha, rho, dims);
    launches += 1;
  }
  note_launch();
  CU(p, cudaGetLastError());
  if (g_launch_error != cudaSuccess) return fail(p, LAM_ECUDA, "kernel launch failed: %s", cudaGetErrorString(g_launch_error));
  p->launches = launches;
  return LAM_OK;
}

lam_status lam_stage_ms(lam_plan* p, float ms[6]) {
  if (!p || !ms) return LAM_EINVAL;
  if (!p->stage_valid) return fail(p, LAM_EINVAL, "no profiled lam_backproject to report (lam_set_profiling(plan, 1) first)");
  cudaSetDevice(p->device);
  for (int i = 0; i < 6; ++i) ms[i] = 0.f;
  for (size_t i = 0; i < p->events_used; ++i) {
    StageEvent& e = p->events[i];
    CU(p, cudaEventSynchronize(e.b));
    float t = 0.f;
    CU(p, cudaEventElapsedTime(&t, e.a, e.b));
    ms[e.stage] += t;
  }
  return LAM_OK;
}

lam_status lam_plan_info(const lam_plan* p, long long info[8]) {
  if (!p || !info) return LAM_EINVAL;
  info[0] = (long long)p->device_bytes;
  info[1] = p->NP;
  info[2] = p->PB;
  info[3] = p->job_off.empty() ? 0 : p->job_off.back();
  info[4] = (p->last_call_host ? 1 : 0) | (p->spill ? 2 : 0);
  info[5] = p->TC;
  info[6] = p->launches;
  info[7] = (long long)p->pinned_bytes;
  return LAM_OK;
}

}  // extern "C"
