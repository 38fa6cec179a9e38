/* lam.h — C ABI of the B200 (sm_100a) laminography filtered back-projection library (liblam.so).
 *
 * What is computed (citations are /root/reference/PAPER.md lines; readings Q1..Q16 are in DESIGN.md):
 *
 *   lam_backproject:  vol = W L*_phi d                                    Eq. 3
 *                     L*_phi = F*_u3D F_2D                                Eq. 7
 *     with the unequally spaced frequencies of Eq. 6
 *         xi = (k_u/w) e_u(theta) + (k_v/h) e_v(theta),
 *         e_u = (cos t, sin t, 0), e_v = (sin t sin phi, -cos t sin phi, cos phi)      Eq. 2
 *     F*_u3D evaluated as a USFFT: convolution-type gridding with a width-W kernel onto a
 *     grid oversampled by sigma, inverse FFT, division by the kernel transform; in the order of Eq. 9
 *     (PAPER.md:174-179): 2-D USFFT in (x1,x2) per detector-frequency row k_v, then 1-D USFFT in x3.
 *     In formulas:  vol[x] = Re sum_theta sum_{k_v,k_u} H[k_u] D[theta,k_v,k_u] e^{+2 pi i x.xi},
 *         D = (1/(w h)) sum_{j_v,j_u} d[theta,j_v,j_u] e^{-2 pi i (k_u u/w + k_v v/h)},  u = j_u-c_u, v = j_v-c_v,
 *         H = (pi cos(phi)/N_theta) DFT_w(band-limited ramp kernel)   (reading Q3 of "a suitable scaled version
 *         of |sigma| cos(phi)"), its Shepp-Logan or Parzen-windowed low-pass variants,
 *         or H = 1 (pure adjoint L*).
 *   lam_forward:      proj = L_phi vol = F*_2D F_u3D vol                   Eq. 5; the exact transpose
 *                     of lam_backproject with filter = LAM_FILTER_NONE (adjoint test <L f, d> = <f, L* d>).
 *   raw 16-bit input: d = -log( max( (raw-dark)/max(flat-dark,1), t_min ) ), the inverse of the detector model
 *                     raw = e^{-d}(flat-dark)+dark of PAPER.md:99, fused into the first FFT pass.
 *
 * Layouts (all C-contiguous, last index fastest):
 *   proj  [n_theta][h][w]   float32 line integrals, or uint16 raw counts (params.input = 1)
 *   vol   [nz][n][n]        float32, voxel (i3,i2,i1) <-> x = (i1-n/2, i2-n/2, i3-nz/2)
 *   dark, flat [h][w]       float32
 *
 * Pointers: proj / vol may be DEVICE pointers or HOST pointers (detected with cudaPointerGetAttributes), each on its
 * own.  With a host pointer the library streams chunks of projections in / slabs of the volume out with
 * cudaMemcpyAsync between the CALLER'S buffer and two plan-owned DEVICE staging buffers per direction, on plan-owned
 * copy streams that overlap the compute stream (Figs. 6-7: three streams, 2 + 2 buffers).  There
 * is no plan-owned pinned host staging: PINNED caller buffers (cudaHostAlloc / cudaHostRegister / torch pin_memory)
 * give asynchronous, overlapped copies; PAGEABLE buffers are accepted and give the same result, but the CUDA runtime
 * then stages every copy through its own bounce buffer and the copies do not overlap the kernels.
 *
 * Workspace: params.device_bytes decides the schedule (PAPER.md:172 "> 64 GB for 2048^3", :181-191).  When the in-core
 * workspace (all intermediates in device memory) fits the budget, it is used, whatever the pointer kinds are.  When it
 * does not, lam_create plans the SPILLED schedule instead of failing: the projection spectra exist for one band of k_v
 * planes at a time (the filter/FFT stage runs once per band over every projection), the cropped intermediate planes
 * leave for a plan-owned PINNED HOST store ((h/2+1) n^2 complex64, reported by lam_plan_info; LAM_ENOMEM_HOST if it
 * cannot be allocated) as they are produced and come back per slab of x2 rows for the x3 stage, all double-buffered on
 * the copy streams.  lam_backproject gives the same result either way (to fp32 rounding); lam_forward,
 * lam_backproject_slice and lam_admm_tv need the in-core workspace (LAM_EUNSUPPORTED on a spilled plan).  A budget too
 * small even for one plane batch of every buffer gives LAM_ENOMEM_DEVICE.
 * The caller owns proj and vol; the plan owns every workspace.
 *
 * All work of lam_backproject / lam_forward is enqueued on `cuda_stream` (a cudaStream_t, may be NULL = the
 * legacy default stream) and on plan-owned streams forked from / joined to it with events; the calls return
 * without synchronising when both pointers are device pointers and the plan is in core (a spilled plan returns when
 * all of the call's work has finished on the device: its plan-owned pinned store and slab buffers are then free for
 * the next call, on whatever stream that is issued).  With a host proj the call returns after the last
 * host->device copy has completed (the caller may reuse proj), with a host vol after the last device->host copy
 * (vol is complete on return).
 *
 * Errors: no exception or abort crosses this boundary.  Every function returns a lam_status; lam_last_error()
 * gives a plan-owned (or, for lam_create failures, thread-local) message.  There is NO CPU fallback: without a
 * CUDA device every compute entry point returns LAM_ECUDA.
 */
#ifndef LAM_H_
#define LAM_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lam_plan lam_plan; /* opaque; owns all device/host workspace */

typedef enum {
  LAM_OK = 0,
  LAM_EINVAL = 1,        /* bad argument (see lam_last_error)                              */
  LAM_ENOMEM_DEVICE = 2, /* not even the spilled schedule fits params.device_bytes / a cudaMalloc failed */
  LAM_ENOMEM_HOST = 3,   /* host allocation failed: the plan object, or the pinned store of a spilled plan */
  LAM_ECUDA = 4,         /* CUDA runtime error, or no device                                */
  LAM_EUNSUPPORTED = 5   /* valid request outside what this build implements                */
} lam_status;

enum { LAM_KERNEL_KB = 0, LAM_KERNEL_GAUSS = 1 };
enum { LAM_FILTER_NONE = 0, LAM_FILTER_RAMP = 1, LAM_FILTER_SHEPP_LOGAN = 2, LAM_FILTER_PARZEN = 3 };
enum { LAM_INPUT_F32 = 0, LAM_INPUT_U16_RAW = 1 };

typedef struct {
  int nz;              /* volume thickness in x3; 0 -> n                                                   */
  int kernel;          /* LAM_KERNEL_KB (default) or LAM_KERNEL_GAUSS  (PAPER.md:130 names a Gaussian psi) */
  int width;           /* W, taps per axis: 4, 6 or 8; 0 -> 6                                               */
  float oversample;    /* sigma; 0 -> 2.0; sigma*n and sigma*nz must be powers of two                       */
  float shape;         /* KB beta or Gaussian variance s_g^2 in grid cells; 0 -> Beatty / Dutt-Rokhlin rule */
  int filter;          /* LAM_FILTER_*                                                                      */
  int input;           /* LAM_INPUT_*                                                                       */
  float center_u;      /* rotation-axis column on the detector, pixels; NaN -> w/2                          */
  float center_v;      /* detector row hit by the ray through the origin; NaN -> h/2                        */
  float t_min;         /* transmission clamp before -log; 0 -> 1e-6                                         */
  size_t device_bytes; /* workspace budget; 0 -> 90 % of the free device memory at lam_create; decides in-core
                          against spilled schedule (header comment).  It covers what lam_create allocates.  Outside
                          it, allocated on first use: the host-pointer staging (2 theta chunks of input + 2 output
                          slabs), the slice buffers of lam_backproject_slice (8 (M^2 + M n + n^2) bytes) and the
                          lam_admm_tv workspace (9 volumes + 1 projection set); leave room for the ones you use   */
  int plane_batch;     /* k_v planes gridded + transformed per launch; 0 -> as many as fit 4 GB of fine grid  */
  int theta_chunk;     /* projections per filter/FFT launch (and per host->device copy); 0 -> auto          */
  int pad_u;           /* 1: every detector row is extended to 2w samples by replicating its edge values before the
                          filter and cropped after it, so that the ramp convolution does not wrap around the detector
                          (reading Q11b; w <= 4096); 0: none (the circular filter of the definition)              */
  float spectral_alpha;/* alpha >= 0 of the 2-D low-pass 1/(1 + alpha ((k_u/w)^2 + (k_v/h)^2)) applied to every
                          projection spectrum: the single-distance Paganin multiplier named as pre-processing in
                          PAPER.md:199, 279, applied to the line integrals (reading Q17); 0: none                 */
  int z_form;          /* form of the x3 stage: 0 -> the library's policy (TMA-fed persistent kernel below
                          sigma*nz = 2048 on an in-core plan, plain kernel otherwise); 1: plain kernel; 2: TMA form
                          wherever its tensor map and buffers can be set up (never on a spilled plan).  Both forms
                          compute the same sums in a different order; tests compare them                          */
  int z_columns;       /* x2-columns per block of the x3 stage: 0 -> policy; 2, 4, 8 or 16 (must divide n; reduced
                          if the block would not fit shared memory)                                               */
} lam_params;

/* Fill *p with the defaults (KB, W = 6, sigma = 2, ramp filter, fp32 input, centred axis). */
void lam_default_params(lam_params* p);

/* Build a plan.  n: lateral volume size (n x n x nz voxels); h, w: detector rows, columns; n_theta angles
 * theta_rad[] (HOST pointer, copied; any values, quadrature weight 2 pi/n_theta as for a uniform full circle,
 * PAPER.md:154-156); phi_rad: tilt of the rotation axis, 0 <= phi < pi/2, phi = 0 is tomography (Eq. 2).
 * Requirements: n, nz, h, w even; w, h, sigma*n, sigma*nz powers of two in [32, 8192]; sigma*n >= 64.
 * Allocates all tables and the gridding work lists (they depend on geometry only).  *out is NULL on error. */
lam_status lam_create(int n, int h, int w, int n_theta, float phi_rad, const float* theta_rad,
                      const lam_params* p, lam_plan** out);

/* dark, flat: h*w float32 each, host or device pointers, copied into the plan.  Needed before lam_backproject
 * when params.input == LAM_INPUT_U16_RAW. */
lam_status lam_set_darkflat(lam_plan* plan, const float* dark, const float* flat);

/* vol <- W L* proj (overwrites vol).  proj: float32 or uint16 per params.input.  See the header comment for
 * pointer kinds and stream semantics. */
lam_status lam_backproject(lam_plan* plan, const void* proj, float* vol, void* cuda_stream);

/* One x3-slice of lam_backproject for a list of rotation-axis positions: the `try` search of PAPER.md:254-270 ("run
 * reconstruction of 1 slice for different rotation axes"); with plans created for different phi it is the
 * `try-lamino` search.  out[c][i2][i1] (device, n_centers x n x n float32; n_centers = 0: one slice
 * at the plan's own axis, centers_u may be NULL) is slice i3 (0 <= i3 < nz) of the volume lam_backproject would return
 * with params.center_u = centers_u[c] (HOST array, pixels).  Evaluated as Eq. 9 with the x3
 * transform done exactly: every k_v plane is gridded in (xi1, xi2), multiplied by e^{2 pi i x3 k_v cos(phi)/h} and
 * added onto one fine grid, then one 2-D inverse FFT, crop and division by the kernel transform in x1, x2 (no x3
 * gridding, so the slice differs from the full volume's by the x3 gridding error only, ~1e-5).  The axis position
 * is a phase on the k_u spectra (reading Q13), re-applied per centre.  Device pointers only; asynchronous on
 * cuda_stream except for two small table uploads; cost per centre ~ one S2 stage. */
lam_status lam_backproject_slice(lam_plan* plan, const void* proj, int i3, int n_centers, const float* centers_u,
                                 float* out, void* cuda_stream);

/* lam_backproject_slice for callers that must not touch the device allocator at call time.  Same arguments, same result
 * (evaluated as Eq. 9); the difference is where the slice scratch lives.
 *
 * Who needs it: lam_backproject_slice calls cudaMalloc five times on its first use per plan.  That is a problem for a
 * program that creates its plans while it is starting up and afterwards has no allocator left to call: a beamline
 * preview service that runs the axis search between detector frames and cannot afford cudaMalloc's device-wide
 * synchronisation and unbounded latency there; a host application (a PyTorch or CuPy process) whose memory pool took all
 * remaining device memory after start-up, so a late cudaMalloc from this library simply fails; code that runs where the
 * CUDA runtime forbids allocation calls altogether.  For those callers this entry point allocates and frees NO device
 * memory, creates no streams or events, and calls no allocating library routine (on the host it uses a few short-lived
 * std::vector tables, as lam_backproject_slice does).
 *
 * How: the summed fine grid, its x1 transform, the cropped plane and the two phase tables live in a 16 MiB array that is
 * part of liblam.so's device image.  Every GPU on which the library's kernels are loaded holds those 16 MiB until the
 * process exits, whether or not this function is ever called.  Limit: the plan's slice scratch,
 * 8 (M^2 + M n + n^2 + (h/2+1) + (w+8)) bytes with M = sigma*n, must fit, i.e. sigma*n <= 1024 at sigma = 2 (n <= 512)
 * for any supported h, w; a larger plan gets LAM_EUNSUPPORTED and a message that names both sizes (use
 * lam_backproject_slice there).  Spilled plans: LAM_EUNSUPPORTED, as for lam_backproject_slice.
 *
 * First call per device: looks up the device address of that array (cudaGetSymbolAddress, which may also make the
 * runtime load the library's device code).  Make that first call during set-up, before any stream capture is begun.
 * Later calls only read the cached address.
 *
 * Sharing: there is ONE such array per device, shared by every plan and every call in the process, and it keeps whatever
 * the previous call left in it.  The function clears what has to start at zero (the summed grid, once per centre) and
 * overwrites the rest before reading it, so calls that follow one another on a device, on any streams, need nothing
 * from the caller as long as each has finished on the GPU before the next starts.  Two calls that overlap on the GPU
 * (different streams or threads, same device) race on the array and both results are garbage: serialise them, or give
 * the second caller lam_backproject_slice.  Per-stage profiling (lam_set_profiling) records nothing for this call. */
lam_status lam_backproject_slice_static(lam_plan* plan, const void* proj, int i3, int n_centers, const float* centers_u,
                                        float* out, void* cuda_stream);

/* proj <- L vol (overwrites proj, float32): Eq. 5 as the exact transpose, stage by stage in reverse
 * order, of lam_backproject with filter none (the plan's filter setting is ignored; an input plan of type uint16
 * still yields float32 line integrals).  Device pointers only (host pointers: LAM_EUNSUPPORTED); asynchronous on
 * cuda_stream.  <L f, d> = <f, L* d> holds to fp32 rounding (about 1e-6 relative).  Needs the
 * in-core workspace (LAM_EUNSUPPORTED on a spilled plan).  About the cost of one lam_backproject. */
lam_status lam_forward(lam_plan* plan, const float* vol, float* proj, void* cuda_stream);

/* TV-regularised reconstruction of PAPER.md Appendix A (Eqs. 10-20):
 *     minimise over mu   1/2 || L mu - d ||^2 + alpha || |grad mu| ||_1                                   (Eq. 10-11)
 * by ADMM on the splitting grad mu = psi (Eqs. 12-16), starting from zeros: n_outer iterations of
 *   (14) n_cg conjugate-gradient steps on F(mu) = 1/2 ||L mu - d||^2 + rho/2 ||grad mu - psi + lambda/rho||^2 (Eq. 17,
 *        gradient Eq. 18) with Dai-Yuan directions (Eq. 19) and the exact step along each direction (F is quadratic),
 *   (15) psi = shrink(grad mu + lambda/rho, alpha/rho), the isotropic soft threshold (Eq. 20 re-derived from Eq. 13:
 *        the printed factors 2 do not satisfy the optimality condition; reading Q18),
 *   (16) lambda += rho (grad mu - psi).
 * L = lam_forward, L^T = lam_backproject of THIS plan, which must have been created with LAM_FILTER_NONE, fp32 input,
 * no padding and no spectral multiplier (else LAM_EINVAL).  grad: forward differences, zero at the far faces.
 * proj: the data d, [n_theta][h][w] float32; vol: the result mu (overwritten); both DEVICE pointers.
 * history: NULL, or a HOST array of n_outer * n_cg doubles; entry k*n_cg + m receives ||grad F|| after CG step m of
 * outer iteration k.  When a direction has no curvature left (the subproblem is solved early), the remaining entries of
 * that outer iteration repeat the last norm taken.  NaN or Inf in proj: LAM_EINVAL at the first step that sees it.
 * The call synchronises cuda_stream twice per CG step (the step lengths are host scalars). */
lam_status lam_admm_tv(lam_plan* plan, const float* proj, float* vol, float alpha, float rho, int n_outer, int n_cg,
                       double* history, void* cuda_stream);

/* Per-stage device times of the LAST lam_backproject, milliseconds, measured with CUDA events on the plan's
 * streams when profiling is on (lam_set_profiling(plan, 1); it adds event records but no synchronisation inside
 * the call; this function synchronises).  ms[0] prep + filter + 2-D FFT (S0+S1), ms[1] gridding in (xi1,xi2)
 * (S2), ms[2] inverse FFT passes in x1 and x2 (S3), ms[3] fused x3 stage: gridding in xi3 + inverse FFT +
 * deapodise/crop/real part (S2 z-part + S3 + S4), ms[4] host<->device copies (host-pointer path), ms[5] whole call. */
lam_status lam_stage_ms(lam_plan* plan, float ms[6]);
/* on = 0: off; 1: per-stage events; 2: per-stage events AND a copy-only dry run: the following lam_backproject calls
 * issue exactly their host<->device copies but skip every kernel (vol then holds no result): the t_copy_only leg of the
 * overlap measurement of the host-pointer path. */
lam_status lam_set_profiling(lam_plan* plan, int on);

/* Workspace facts of a plan, for benchmarks and tests:
 * info[0] device bytes allocated, info[1] k_v planes, info[2] plane batch, info[3] gridding work items (jobs),
 * info[4] bit 0: the last lam_backproject streamed through host pointers, bit 1: the plan runs the spilled schedule,
 * info[5] theta chunk,
 * info[6] kernel launches of the last lam_backproject, info[7] pinned host bytes. */
lam_status lam_plan_info(const lam_plan* plan, long long info[8]);

/* Message of the last error on this plan (plan == NULL: of the last failed lam_create on this thread). */
const char* lam_last_error(const lam_plan* plan);

void lam_destroy(lam_plan* plan);

/* Library version string, e.g. "lam-b200 0.4 (sm_100a)". */
const char* lam_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LAM_H_ */
