"""Thin ctypes binding of liblam.so (include/lam.h).  Argument marshalling only: every step of the path runs
in the CUDA kernels behind the C ABI.  There is no CPU path: if the library is missing this module raises.

Names mirror the C entry points: lam_create, lam_set_darkflat, lam_backproject, lam_forward, lam_stage_ms,
lam_set_profiling, lam_plan_info, lam_last_error, lam_destroy, lam_version, lam_default_params.
`Plan` is a small convenience wrapper that owns a lam_plan* and takes torch tensors (device memory and
streams are PyTorch's; nothing else of torch is used).
"""
import ctypes as C
import math
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
LIB_PATH = os.environ.get("LAM_LIB") or os.path.join(_HERE, "liblam.so")
INCLUDE = os.path.join(os.path.dirname(_HERE), "include")

LAM_OK, LAM_EINVAL, LAM_ENOMEM_DEVICE, LAM_ENOMEM_HOST, LAM_ECUDA, LAM_EUNSUPPORTED = range(6)
STATUS_NAMES = ["LAM_OK", "LAM_EINVAL", "LAM_ENOMEM_DEVICE", "LAM_ENOMEM_HOST", "LAM_ECUDA", "LAM_EUNSUPPORTED"]
KERNELS = {"kb": 0, "gauss": 1}
FILTERS = {"none": 0, "ramp": 1, "shepp-logan": 2, "parzen": 3}
INPUTS = {"f32": 0, "u16": 1}

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


class lam_params(C.Structure):
    _fields_ = [("nz", C.c_int), ("kernel", C.c_int), ("width", C.c_int), ("oversample", C.c_float),
                ("shape", C.c_float), ("filter", C.c_int), ("input", C.c_int), ("center_u", C.c_float),
                ("center_v", C.c_float), ("t_min", C.c_float), ("device_bytes", C.c_size_t),
                ("plane_batch", C.c_int), ("theta_chunk", C.c_int), ("pad_u", C.c_int), ("spectral_alpha", C.c_float),
                ("z_form", C.c_int), ("z_columns", C.c_int)]


class LamError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS_NAMES[status] if 0 <= status < 6 else status}: {msg}")
        self.status = status


def sources():
    return [os.path.join(_CSRC, f) for f in sorted(os.listdir(_CSRC))] + [os.path.join(INCLUDE, "lam.h")]


def build(force=False, verbose=False):
    """Compile csrc/lam.cu for sm_100a into liblam.so (in-tree).  nvcc cross-compiles without a GPU."""
    if not force and os.path.exists(LIB_PATH):
        mt = os.path.getmtime(LIB_PATH)
        if all(os.path.getmtime(s) <= mt for s in sources()):
            return LIB_PATH
    cmd = ["nvcc"] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", LIB_PATH, os.path.join(_CSRC, "lam.cu")]
    subprocess.check_call(cmd)
    return LIB_PATH


_lib = None


def lib():
    global _lib
    if _lib is not None:
        return _lib
    if not os.environ.get("LAM_LIB"):
        build()             # rebuilds when a source is newer than the library (a stale .so is never loaded silently)
    L = C.CDLL(LIB_PATH)
    P = C.c_void_p
    L.lam_version.restype = C.c_char_p
    L.lam_last_error.restype = C.c_char_p
    L.lam_last_error.argtypes = [P]
    L.lam_default_params.restype = None
    L.lam_default_params.argtypes = [C.POINTER(lam_params)]
    L.lam_create.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_float, C.POINTER(C.c_float),
                             C.POINTER(lam_params), C.POINTER(P)]
    L.lam_set_darkflat.argtypes = [P, P, P]
    L.lam_backproject.argtypes = [P, P, P, P]
    L.lam_forward.argtypes = [P, P, P, P]
    L.lam_backproject_slice.argtypes = [P, P, C.c_int, C.c_int, C.POINTER(C.c_float), P, P]
    L.lam_backproject_slice_static.argtypes = [P, P, C.c_int, C.c_int, C.POINTER(C.c_float), P, P]
    L.lam_admm_tv.argtypes = [P, P, P, C.c_float, C.c_float, C.c_int, C.c_int, C.POINTER(C.c_double), P]
    L.lam_stage_ms.argtypes = [P, C.POINTER(C.c_float)]
    L.lam_set_profiling.argtypes = [P, C.c_int]
    L.lam_plan_info.argtypes = [P, C.POINTER(C.c_longlong)]
    L.lam_destroy.restype = None
    L.lam_destroy.argtypes = [P]
    _lib = L
    return L


EXPORTS = ["lam_version", "lam_default_params", "lam_create", "lam_set_darkflat", "lam_backproject", "lam_forward",
           "lam_backproject_slice", "lam_backproject_slice_static", "lam_admm_tv",
           "lam_stage_ms", "lam_set_profiling", "lam_plan_info", "lam_last_error", "lam_destroy"]


# ---- 1:1 wrappers ---------------------------------------------------------------------------------------------------
def lam_version():
    return lib().lam_version().decode()


def lam_default_params():
    p = lam_params()
    lib().lam_default_params(C.byref(p))
    return p


def lam_last_error(plan=None):
    return lib().lam_last_error(plan).decode()


def _check(st, plan=None):
    if st != LAM_OK:
        raise LamError(st, lam_last_error(plan))


def lam_create(n, h, w, theta, phi, params=None):
    """theta: sequence of angles in radians (host).  Returns the opaque lam_plan* (c_void_p)."""
    th = (C.c_float * len(theta))(*[float(t) for t in theta])
    out = C.c_void_p()
    st = lib().lam_create(int(n), int(h), int(w), len(theta), C.c_float(phi), th,
                          C.byref(params) if params is not None else None, C.byref(out))
    _check(st)
    return out


def lam_set_darkflat(plan, dark_ptr, flat_ptr):
    _check(lib().lam_set_darkflat(plan, C.c_void_p(dark_ptr), C.c_void_p(flat_ptr)), plan)


def lam_backproject(plan, proj_ptr, vol_ptr, stream=0):
    _check(lib().lam_backproject(plan, C.c_void_p(proj_ptr), C.c_void_p(vol_ptr), C.c_void_p(stream)), plan)


def lam_backproject_slice(plan, proj_ptr, i3, centers, out_ptr, stream=0):
    """centers: sequence of rotation-axis positions (pixels, host) or None / empty for the plan's own axis."""
    nc = len(centers) if centers is not None else 0
    arr = (C.c_float * nc)(*[float(c) for c in centers]) if nc else None
    _check(lib().lam_backproject_slice(plan, C.c_void_p(proj_ptr), int(i3), nc, arr, C.c_void_p(out_ptr), C.c_void_p(stream)), plan)


def lam_backproject_slice_static(plan, proj_ptr, i3, centers, out_ptr, stream=0):
    """lam_backproject_slice on the scratch array built into liblam.so: for callers that may not allocate device memory
    once their plans exist (include/lam.h has the limit, sigma*n <= 1024, and the sharing rules)."""
    nc = len(centers) if centers is not None else 0
    arr = (C.c_float * nc)(*[float(c) for c in centers]) if nc else None
    _check(lib().lam_backproject_slice_static(plan, C.c_void_p(proj_ptr), int(i3), nc, arr, C.c_void_p(out_ptr),
                                              C.c_void_p(stream)), plan)


def lam_admm_tv(plan, proj_ptr, vol_ptr, alpha, rho, n_outer, n_cg, stream=0):
    """Returns the list of ||grad F|| after every CG step (Appendix A)."""
    hist = (C.c_double * (n_outer * n_cg))()
    _check(lib().lam_admm_tv(plan, C.c_void_p(proj_ptr), C.c_void_p(vol_ptr), C.c_float(alpha), C.c_float(rho), int(n_outer),
                             int(n_cg), hist, C.c_void_p(stream)), plan)
    return list(hist)


def lam_forward(plan, vol_ptr, proj_ptr, stream=0):
    _check(lib().lam_forward(plan, C.c_void_p(vol_ptr), C.c_void_p(proj_ptr), C.c_void_p(stream)), plan)


def lam_set_profiling(plan, on):
    _check(lib().lam_set_profiling(plan, int(on)), plan)


def lam_stage_ms(plan):
    ms = (C.c_float * 6)()
    _check(lib().lam_stage_ms(plan, ms), plan)
    return list(ms)


def lam_plan_info(plan):
    info = (C.c_longlong * 8)()
    _check(lib().lam_plan_info(plan, info), plan)
    keys = ["device_bytes", "planes", "plane_batch", "jobs", "out_of_core", "theta_chunk", "launches", "pinned_bytes"]
    return dict(zip(keys, list(info)))


def lam_destroy(plan):
    lib().lam_destroy(plan)


# ---- convenience wrapper over torch tensors --------------------------------------------------------------------------
class Plan:
    def __init__(self, n, h, w, theta, phi, nz=None, kernel="kb", width=6, oversample=2.0, shape=0.0, filter="ramp",
                 input="f32", center_u=None, center_v=None, t_min=1e-6, device_bytes=0, plane_batch=0, theta_chunk=0,
                 pad_u=False, spectral_alpha=0.0, z_form=0, z_columns=0):
        p = lam_default_params()
        p.nz = int(nz or n)
        p.kernel, p.width, p.oversample, p.shape = KERNELS[kernel], int(width), float(oversample), float(shape)
        p.filter, p.input = FILTERS[filter], INPUTS[input]
        p.center_u = math.nan if center_u is None else float(center_u)
        p.center_v = math.nan if center_v is None else float(center_v)
        p.t_min, p.device_bytes = float(t_min), int(device_bytes)
        p.plane_batch, p.theta_chunk = int(plane_batch), int(theta_chunk)
        p.pad_u, p.spectral_alpha = int(bool(pad_u)), float(spectral_alpha)
        p.z_form, p.z_columns = int(z_form), int(z_columns)
        self.n, self.nz, self.h, self.w, self.ntheta = int(n), p.nz, int(h), int(w), len(theta)
        self.input = input
        self._plan = lam_create(n, h, w, theta, phi, p)

    def set_darkflat(self, dark, flat):
        assert dark.is_contiguous() and flat.is_contiguous() and dark.numel() == self.h * self.w == flat.numel()
        lam_set_darkflat(self._plan, dark.data_ptr(), flat.data_ptr())

    def backproject(self, proj, vol=None, stream=None):
        import torch
        assert proj.is_contiguous() and tuple(proj.shape) == (self.ntheta, self.h, self.w)
        assert proj.dtype == (torch.uint16 if self.input == "u16" else torch.float32)
        if vol is None:
            vol = torch.empty((self.nz, self.n, self.n), dtype=torch.float32, device=proj.device)
        assert vol.is_contiguous() and vol.dtype == torch.float32 and tuple(vol.shape) == (self.nz, self.n, self.n)
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        lam_backproject(self._plan, proj.data_ptr(), vol.data_ptr(), stream)
        return vol

    def backproject_slice(self, proj, i3, centers=None, out=None, stream=None, static_scratch=False):
        """Slice i3 for each rotation-axis position in `centers` (the `try` search) -> [nc][n][n].
        static_scratch=True goes through lam_backproject_slice_static (no device allocation inside the library; pass
        `out` as well if torch must not allocate either)."""
        import torch
        assert proj.is_contiguous() and tuple(proj.shape) == (self.ntheta, self.h, self.w) and proj.is_cuda
        nc = len(centers) if centers is not None and len(centers) else 1
        if out is None:
            out = torch.empty((nc, self.n, self.n), dtype=torch.float32, device=proj.device)
        assert out.is_contiguous() and out.dtype == torch.float32 and tuple(out.shape) == (nc, self.n, self.n)
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        call = lam_backproject_slice_static if static_scratch else lam_backproject_slice
        call(self._plan, proj.data_ptr(), i3, centers, out.data_ptr(), stream)
        return out

    def admm_tv(self, proj, alpha, rho, n_outer, n_cg, vol=None, stream=None):
        """TV-regularised reconstruction (Appendix A) -> (vol, ||grad F|| history)."""
        import torch
        assert proj.is_contiguous() and proj.dtype == torch.float32 and tuple(proj.shape) == (self.ntheta, self.h, self.w)
        if vol is None:
            vol = torch.empty((self.nz, self.n, self.n), dtype=torch.float32, device=proj.device)
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        hist = lam_admm_tv(self._plan, proj.data_ptr(), vol.data_ptr(), alpha, rho, n_outer, n_cg, stream)
        return vol, hist

    def forward(self, vol, proj=None, stream=None):
        import torch
        assert vol.is_contiguous() and vol.dtype == torch.float32 and tuple(vol.shape) == (self.nz, self.n, self.n)
        if proj is None:
            proj = torch.empty((self.ntheta, self.h, self.w), dtype=torch.float32, device=vol.device)
        if stream is None:
            stream = torch.cuda.current_stream().cuda_stream
        lam_forward(self._plan, vol.data_ptr(), proj.data_ptr(), stream)
        return proj

    def set_profiling(self, on=True):
        lam_set_profiling(self._plan, on)

    def stage_ms(self):
        return lam_stage_ms(self._plan)

    def info(self):
        return lam_plan_info(self._plan)

    def close(self):
        if self._plan is not None:
            lam_destroy(self._plan)
            self._plan = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
