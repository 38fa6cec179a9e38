"""ctypes front end of the CPU fp64 oracle (oracle/lam_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
The product package paper_2401_11101_b200 never does, and this module never imports the product.
Every function cites the PAPER.md passage it follows in lam_oracle.cpp.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lam_oracle.cpp")
_LIB = os.path.join(_HERE, "liblam_oracle.so")


def build(force=False):
    """Compile the oracle with g++ (no fast-math).  Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["g++", "-O3", "-std=c++17", "-fopenmp", "-fPIC", "-shared",
                               "-o", _LIB, _SRC])
    return _LIB


class _Geom(C.Structure):
    _fields_ = [("n", C.c_int), ("nz", C.c_int), ("h", C.c_int), ("w", C.c_int), ("ntheta", C.c_int),
                ("phi", C.c_double), ("theta", C.POINTER(C.c_double)),
                ("cu", C.c_double), ("cv", C.c_double),
                ("filter", C.c_int), ("dtype", C.c_int),
                ("dark", C.POINTER(C.c_float)), ("flat", C.POINTER(C.c_float)),
                ("tmin", C.c_double), ("pad", C.c_int), ("alpha", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_kap.restype = C.c_double
        _lib.orc_kap.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double]
        _lib.orc_kaphat.restype = C.c_double
        _lib.orc_kaphat.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double]
        _lib.orc_fbp_gridded.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_void_p]
        _lib.orc_fbp_gridded_slice.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double,
                                               C.c_int, C.c_void_p]
    return _lib


FILTERS = {"none": 0, "ramp": 1, "shepp-logan": 2, "parzen": 3}
KERNELS = {"kb": 0, "gauss": 1}


class Geometry:
    """Scan geometry (Eq. 2 / Eq. 6) + filter choice + input encoding."""

    def __init__(self, n, h, w, theta, phi, nz=None, filter="ramp", cu=None, cv=None,
                 dark=None, flat=None, tmin=1e-6, pad=1, alpha=0.0):
        self.n, self.h, self.w = int(n), int(h), int(w)
        self.nz = int(nz) if nz else int(n)
        self.theta = np.ascontiguousarray(theta, dtype=np.float64)
        self.ntheta = len(self.theta)
        self.phi = float(phi)
        self.filter = filter
        self.cu = self.w / 2 if cu is None else float(cu)
        self.cv = self.h / 2 if cv is None else float(cv)
        self.dark = None if dark is None else np.ascontiguousarray(dark, dtype=np.float32)
        self.flat = None if flat is None else np.ascontiguousarray(flat, dtype=np.float32)
        self.tmin = float(tmin)
        self.pad = int(pad)        # rows edge-extended to pad*w before the filter (reading Q11b)
        self.alpha = float(alpha)  # 2-D spectral multiplier 1/(1 + alpha |k|^2) (reading Q17)

    def _c(self, proj):
        g = _Geom()
        g.n, g.nz, g.h, g.w, g.ntheta = self.n, self.nz, self.h, self.w, self.ntheta
        g.phi = self.phi
        g.theta = self.theta.ctypes.data_as(C.POINTER(C.c_double))
        g.cu, g.cv = self.cu, self.cv
        g.filter = FILTERS[self.filter]
        g.tmin = self.tmin
        g.pad, g.alpha = self.pad, self.alpha
        if proj is None:
            g.dtype = 0
        else:
            assert proj.flags["C_CONTIGUOUS"] and proj.shape == (self.ntheta, self.h, self.w), proj.shape
            g.dtype = {np.dtype(np.float64): 0, np.dtype(np.float32): 1, np.dtype(np.uint16): 2}[proj.dtype]
            if g.dtype == 2:
                assert self.dark is not None and self.flat is not None
                g.dark = self.dark.ctypes.data_as(C.POINTER(C.c_float))
                g.flat = self.flat.ctypes.data_as(C.POINTER(C.c_float))
        return g


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def threads():
    return int(lib().orc_threads())


def dft1d(x, sign, naive=False):
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    lib().orc_dft1d(_p(x), _p(out), C.c_int(len(x)), C.c_int(sign), C.c_int(int(naive)))
    return out


def filter_response(geom):
    """H[k_u + w/2] of Eq. 3, reading Q3."""
    out = np.empty(geom.w)
    g = geom._c(None)
    lib().orc_filter(C.byref(g), _p(out))
    return out


def prep(geom, proj, th):
    """-log((raw-dark)/(flat-dark)) of PAPER.md:99 for projection th -> float64 [h][w]."""
    out = np.empty((geom.h, geom.w))
    g = geom._c(proj)
    lib().orc_prep(C.byref(g), _p(proj), C.c_int(th), _p(out))
    return out


def filter_rows_padded(geom, proj, th):
    """Rows of projection th filtered after edge extension to pad*w samples (reading Q11b) -> float64 [h][w]."""
    assert geom.pad > 1
    out = np.empty((geom.h, geom.w))
    g = geom._c(proj)
    lib().orc_filter_rows_padded(C.byref(g), _p(proj), C.c_int(th), _p(out))
    return out


def spectrum(geom, proj, th):
    """Filtered centred 2-D spectrum HD[k_v+h/2][k_u+w/2] of projection th (F_2D of Eq. 7)."""
    out = np.empty((geom.h, geom.w), dtype=np.complex128)
    g = geom._c(proj)
    lib().orc_spectrum(C.byref(g), _p(proj), C.c_int(th), _p(out))
    return out


def fbp_nudft(geom, proj, cols=None, return_imag=False):
    """Path A.  cols: int array [ncols][2] of (i1, i2); None = every column -> vol[nz][n][n]."""
    full = cols is None
    if full:
        i2, i1 = np.meshgrid(np.arange(geom.n), np.arange(geom.n), indexing="ij")
        cols = np.stack([i1.ravel(), i2.ravel()], axis=1)
    cols = np.ascontiguousarray(cols, dtype=np.int32)
    re = np.empty((len(cols), geom.nz))
    im = np.empty((len(cols), geom.nz))
    g = geom._c(proj)
    lib().orc_fbp_nudft(C.byref(g), _p(proj), C.c_int(len(cols)), _p(cols), _p(re), _p(im))
    if full:
        re = np.ascontiguousarray(re.reshape(geom.n, geom.n, geom.nz).transpose(2, 0, 1))
        im = np.ascontiguousarray(im.reshape(geom.n, geom.n, geom.nz).transpose(2, 0, 1))
    return (re, im) if return_imag else re


def fbp_brute(geom, proj):
    vol = np.empty((geom.nz, geom.n, geom.n))
    g = geom._c(proj)
    lib().orc_fbp_brute(C.byref(g), _p(proj), _p(vol))
    return vol


def forward_nudft(geom, vol):
    vol = np.ascontiguousarray(vol, dtype=np.float64)
    assert vol.shape == (geom.nz, geom.n, geom.n)
    out = np.empty((geom.ntheta, geom.h, geom.w))
    g = geom._c(None)
    lib().orc_forward_nudft(C.byref(g), _p(vol), _p(out))
    return out


def fbp_direct(geom, proj):
    vol = np.empty((geom.nz, geom.n, geom.n))
    g = geom._c(proj)
    lib().orc_fbp_direct(C.byref(g), _p(proj), _p(vol))
    return vol


def fp_direct(geom, vol):
    vol = np.ascontiguousarray(vol, dtype=np.float64)
    out = np.empty((geom.ntheta, geom.h, geom.w))
    g = geom._c(None)
    lib().orc_fp_direct(C.byref(g), _p(vol), _p(out))
    return out


def fp_ray(geom, vol):
    """Ray-driven forward projection (Eq. 1-2): unit steps along the beam, trilinear."""
    vol = np.ascontiguousarray(vol, dtype=np.float64)
    assert vol.shape == (geom.nz, geom.n, geom.n)
    out = np.empty((geom.ntheta, geom.h, geom.w))
    g = geom._c(None)
    lib().orc_fp_ray(C.byref(g), _p(vol), _p(out))
    return out


def default_shape(kernel, W, sigma):
    """KB: Beatty's beta = pi sqrt((W/sigma)^2 (sigma-1/2)^2 - 0.8); Gauss: sg2 = sigma (W/2)/(2 pi (sigma-1/2))."""
    if kernel == "kb":
        return float(np.pi * np.sqrt((W / sigma) ** 2 * (sigma - 0.5) ** 2 - 0.8))
    return float(sigma * (W / 2) / (2 * np.pi * (sigma - 0.5)))


def kap(kernel, W, shape, t):
    return lib().orc_kap(KERNELS[kernel], W, shape, float(t))


def kaphat(kernel, W, shape, s):
    return lib().orc_kaphat(KERNELS[kernel], W, shape, float(s))


def fbp_gridded(geom, proj, kernel="kb", W=6, sigma=2.0, shape=None):
    """Path C -> vol[nz][n][n]."""
    shape = default_shape(kernel, W, sigma) if shape is None else shape
    vol = np.empty((geom.nz, geom.n, geom.n))
    g = geom._c(proj)
    rc = lib().orc_fbp_gridded(C.byref(g), _p(proj), KERNELS[kernel], W, sigma, shape, _p(vol))
    if rc:
        raise MemoryError("oracle path C: fine grid does not fit host memory")
    return vol


def fbp_gridded_slice(geom, proj, i3, kernel="kb", W=6, sigma=2.0, shape=None):
    """Path C' -> slice[n][n] at x3 index i3."""
    shape = default_shape(kernel, W, sigma) if shape is None else shape
    out = np.empty((geom.n, geom.n))
    g = geom._c(proj)
    lib().orc_fbp_gridded_slice(C.byref(g), _p(proj), KERNELS[kernel], W, sigma, shape, int(i3), _p(out))
    return out
