"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-types the oracle's own formula: each compares it with an analytic closed form, a textbook
special case, an invariant, a library routine (numpy FFT) used on a different formulation, or brute force.
"""
import math

import numpy as np
import pytest

from oracle import lam_oracle as O


def rel(a, b):
    return float(np.linalg.norm(np.asarray(a) - np.asarray(b)) / np.linalg.norm(np.asarray(b)))


def unit_vectors(theta, phi):
    """Normals of the two delta functions of Eq. 2, written out by hand."""
    e_u = np.array([math.cos(theta), math.sin(theta), 0.0])
    e_v = np.array([math.sin(theta) * math.sin(phi), -math.cos(theta) * math.sin(phi), math.cos(phi)])
    return e_u, e_v


def blob_projection(c, s, A, theta, phi, h, w):
    """Line integral of A exp(-|x-c|^2/(2s^2)) along the line of Eq. 2: the two deltas fix (x.e_u, x.e_v),
    e_u and e_v are orthonormal, so the integral is over the third orthonormal direction and equals
    A s sqrt(2 pi) exp(-((u-c.e_u)^2+(v-c.e_v)^2)/(2 s^2))."""
    e_u, e_v = unit_vectors(theta, phi)
    u = np.arange(w) - w / 2
    v = np.arange(h) - h / 2
    return A * s * math.sqrt(2 * math.pi) * np.exp(-((u[None, :] - c @ e_u) ** 2 + (v[:, None] - c @ e_v) ** 2) / (2 * s * s))


# ------------------------------------------------------------------ P0: the oracle's own FFT
@pytest.mark.parametrize("n", [2, 8, 64, 12, 30])
@pytest.mark.parametrize("sign", [-1, 1])
def test_fft_against_naive_dft_and_numpy(n, sign):
    rng = np.random.default_rng(n)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    fast, slow = O.dft1d(x, sign), O.dft1d(x, sign, naive=True)
    ref = np.fft.fft(x) if sign < 0 else np.fft.ifft(x) * n
    assert rel(fast, ref) < 1e-13 and rel(slow, ref) < 1e-13


# ------------------------------------------------------------------ P1: Fourier-slice identity (Eqs. 5-6)
@pytest.mark.parametrize("phi_deg", [0.0, 20.0, 35.0])
def test_P1_fourier_slice_of_analytic_blob(phi_deg):
    """(1/(wh)) DFT2 of the analytic blob projection = (1/(wh)) * analytic 3-D transform of the blob,
    A (2 pi)^{3/2} s^3 exp(-2 pi^2 s^2 |xi|^2) e^{-2 pi i c.xi}, at xi of Eq. 6.  Pins the signs of Eq. 6,
    the sign of the transform, the centring and the 1/(wh) normalisation."""
    h = w = 64
    phi = math.radians(phi_deg)
    c, s, A = np.array([3.0, -5.0, 2.0]), 2.0, 0.8
    theta = np.array([0.3, 1.9, 4.0])
    geom = O.Geometry(n=64, h=h, w=w, theta=theta, phi=phi, filter="none")
    proj = np.stack([blob_projection(c, s, A, t, phi, h, w) for t in theta])
    for i, t in enumerate(theta):
        D = O.spectrum(geom, proj, i)
        ku = (np.arange(w) - w // 2)[None, :] / w
        kv = (np.arange(h) - h // 2)[:, None] / h
        xi1 = ku * math.cos(t) + kv * math.sin(t) * math.sin(phi)      # Eq. 6
        xi2 = ku * math.sin(t) - kv * math.cos(t) * math.sin(phi)
        xi3 = kv * math.cos(phi) + 0 * ku
        ana = A * (2 * math.pi) ** 1.5 * s ** 3 * np.exp(-2 * math.pi ** 2 * s * s * (xi1 ** 2 + xi2 ** 2 + xi3 ** 2)) \
            * np.exp(-2j * math.pi * (c[0] * xi1 + c[1] * xi2 + c[2] * xi3)) / (w * h)
        assert rel(D, ana) < 1e-7


# ------------------------------------------------------------------ P2 / P3: adjoint = Eq. 4
def test_P2_P3_adjoint_is_backprojection_integral():
    """Path A without filter on band-limited blob projections equals Eq. 4:
    sum_theta d_analytic(theta, x.e_u, x.e_v) at any voxel, and on the axis the closed form
    N_theta A s sqrt(2 pi) exp(-x3^2 cos^2(phi)/(2 s^2)) for a centred blob."""
    n, h, w, nth = 32, 64, 64, 48
    phi = math.radians(20.0)
    theta = 2 * np.pi * np.arange(nth) / nth
    s, A = 2.5, 0.7
    geom = O.Geometry(n=n, h=h, w=w, theta=theta, phi=phi, filter="none")
    # P3: centred blob, column through the axis
    proj = np.stack([blob_projection(np.zeros(3), s, A, t, phi, h, w) for t in theta])
    col = O.fbp_nudft(geom, proj, cols=[[n // 2, n // 2]])[0]
    x3 = np.arange(n) - n / 2
    closed = nth * A * s * math.sqrt(2 * math.pi) * np.exp(-x3 ** 2 * math.cos(phi) ** 2 / (2 * s * s))
    assert rel(col, closed) < 1e-8
    # P2: off-centre blob, arbitrary voxels
    c = np.array([4.0, -3.0, 2.0])
    proj = np.stack([blob_projection(c, s, A, t, phi, h, w) for t in theta])
    cols = np.array([[10, 20], [16, 16], [25, 7], [20, 13]])
    got = O.fbp_nudft(geom, proj, cols=cols)
    want = np.zeros_like(got)
    for ci, (i1, i2) in enumerate(cols):
        for i3 in range(n):
            x = np.array([i1 - n / 2, i2 - n / 2, i3 - n / 2])
            for t in theta:
                e_u, e_v = unit_vectors(t, phi)
                want[ci, i3] += A * s * math.sqrt(2 * math.pi) * math.exp(
                    -((x @ e_u - c @ e_u) ** 2 + (x @ e_v - c @ e_v) ** 2) / (2 * s * s))
    assert rel(got, want) < 1e-8


# ------------------------------------------------------------------ P4: phi = 0 is tomography
@pytest.mark.parametrize("filt,tol", [("ramp", 1e-6), ("shepp-logan", 3e-2)])
def test_P4_tomography_limit_reproduces_blob(filt, tol):
    """At phi = 0 Eq. 1 is the Radon transform and FBP (Eq. 3) with the textbook constant
    f = (1/2) int_0^{2 pi} (d * ramp)(x.e_u) dtheta must return the object: pins the filter constant
    pi/N_theta and the Ram-Lak discretisation.  (Shepp-Logan is a low-pass: percent-level only.)"""
    n, h, w, nth = 32, 64, 64, 96
    theta = 2 * np.pi * np.arange(nth) / nth
    c, s, A = np.array([5.0, -3.0, 2.0]), 2.0, 0.9
    geom = O.Geometry(n=n, h=h, w=w, theta=theta, phi=0.0, filter=filt)
    proj = np.stack([blob_projection(c, s, A, t, 0.0, h, w) for t in theta])
    vol = O.fbp_nudft(geom, proj)
    x = np.arange(n) - n / 2
    X3, X2, X1 = np.meshgrid(x, x, x, indexing="ij")
    blob = A * np.exp(-((X1 - c[0]) ** 2 + (X2 - c[1]) ** 2 + (X3 - c[2]) ** 2) / (2 * s * s))
    assert rel(vol, blob) < tol


# ------------------------------------------------------------------ P4b: filter responses in closed form
@pytest.mark.parametrize("w", [64, 1024])
@pytest.mark.parametrize("filt", ["ramp", "shepp-logan"])
def test_P4b_filter_response_closed_form(filt, w):
    """Reading Q3: H = (pi cos(phi)/N_theta) DFT_w(h).  The DTFT of the infinite band-limited ramp kernel
    (h[0] = 1/4, h[odd j] = -1/(pi j)^2) is |f| on |f| <= 1/2, and that of the Shepp-Logan kernel
    h[j] = -2/(pi^2 (4 j^2 - 1)) is |sin(pi f)|/pi (both textbook).  Cutting the kernels to w taps changes every
    bin by at most the dropped tail, sum_{|j| >= w/2} |h[j]| <= 2/(pi^2 w) (1 + O(1/w)).  A wrong constant, a
    wrong kernel entry or a swapped ramp/Shepp-Logan branch is off by far more than that."""
    phi, nth = 0.3, 10
    geom = O.Geometry(n=w, h=w, w=w, theta=np.arange(float(nth)), phi=phi, filter=filt)
    H = O.filter_response(geom)
    f = (np.arange(w) - w // 2) / w
    c = math.pi * math.cos(phi) / nth
    want = c * (np.abs(f) if filt == "ramp" else np.abs(np.sin(math.pi * f)) / math.pi)
    bound = 2.0 / (math.pi ** 2 * w) * (1.0 + 4.0 / w)
    assert np.abs(H - want).max() <= c * bound
    assert np.abs(H - want).max() >= c * 0.5 * bound          # the bound is sharp: the test has teeth
    other = c * (np.abs(np.sin(math.pi * f)) / math.pi if filt == "ramp" else np.abs(f))
    assert np.abs(H - other).max() > 20 * c * bound           # the two filters are told apart


# ------------------------------------------------------------------ P5: phi > 0, missing cone
@pytest.mark.parametrize("phi_deg", [20.0, 30.0])
def test_P5_missing_cone_closed_form(phi_deg):
    """By Eq. 6 the frequencies with |xi3| tan(phi) > |(xi1,xi2)| are never sampled, every other one is hit
    twice with Jacobian |k_u| cos(phi); so FBP (Eq. 3) returns the inverse 3-D transform of
    ghat(xi) 1[|xi3| tan(phi) < |(xi1,xi2)|].  The reference is numpy's FFT of the ANALYTIC ghat on a large
    grid.  Pins the cos(phi) in the filter constant and the geometry at phi > 0.  (Limited by the reference's
    own discretisation of the cone edge: 1e-3 level.)"""
    phi = math.radians(phi_deg)
    n, h, w, nth = 32, 64, 64, 128
    theta = 2 * np.pi * np.arange(nth) / nth
    c, s, A = np.array([2.0, -1.0, 1.0]), 2.0, 1.0
    geom = O.Geometry(n=n, h=h, w=w, theta=theta, phi=phi, filter="ramp")
    proj = np.stack([blob_projection(c, s, A, t, phi, h, w) for t in theta])
    vol = O.fbp_nudft(geom, proj)
    NF = 256
    f = np.fft.fftfreq(NF)
    F3, F2, F1 = np.meshgrid(f, f, f, indexing="ij")
    ghat = A * (2 * math.pi) ** 1.5 * s ** 3 * np.exp(-2 * math.pi ** 2 * s * s * (F1 ** 2 + F2 ** 2 + F3 ** 2)) \
        * np.exp(-2j * math.pi * (c[0] * F1 + c[1] * F2 + c[2] * F3))
    rho, z = np.sqrt(F1 ** 2 + F2 ** 2), np.abs(F3) * math.tan(phi)
    mask = (z < rho).astype(float) + 0.5 * (z == rho)
    ref = np.fft.ifftn(ghat * mask).real          # sum_xi ghat e^{+2 pi i x xi} dxi^3, dxi = 1/NF
    idx = (np.arange(n) - n // 2) % NF
    ref = ref[np.ix_(idx, idx, idx)]
    assert rel(vol, ref) < 4e-3
    x = np.arange(n) - n / 2
    X3, X2, X1 = np.meshgrid(x, x, x, indexing="ij")
    blob = A * np.exp(-((X1 - c[0]) ** 2 + (X2 - c[1]) ** 2 + (X3 - c[2]) ** 2) / (2 * s * s))
    assert rel(vol, blob) > 0.05                  # the test has teeth: the raw blob is far away


# ------------------------------------------------------------------ P6: transposes
def test_P6_adjoint_identity_exact_operators():
    """<L f, d> = <f, L* d> to 1e-10 (north_star) for the NUDFT pair (Eq. 5 / Eq. 7) and the direct pair."""
    rng = np.random.default_rng(5)
    n, nz, h, w, nth = 8, 6, 10, 12, 5
    theta = rng.uniform(0, 2 * np.pi, nth)
    geom = O.Geometry(n=n, nz=nz, h=h, w=w, theta=theta, phi=math.radians(25.0), filter="none", cu=5.7, cv=5.2)
    f = rng.standard_normal((nz, n, n))
    d = rng.standard_normal((nth, h, w))
    lhs = np.vdot(O.forward_nudft(geom, f), d)
    rhs = np.vdot(f, O.fbp_nudft(geom, d))
    assert abs(lhs - rhs) / abs(lhs) < 1e-10
    lhs = np.vdot(O.fp_direct(geom, f), d)
    rhs = np.vdot(f, O.fbp_direct(geom, d))
    assert abs(lhs - rhs) / abs(lhs) < 1e-10


def test_P6b_forward_nudft_matches_analytic_projection():
    """Eq. 5 on a sampled band-limited blob returns its analytic line integrals (Eq. 1): pins O1 itself."""
    n, h, w = 24, 24, 24
    phi = math.radians(20.0)
    theta = np.array([0.4, 2.2])
    c, s, A = np.array([1.0, -2.0, 0.5]), 2.0, 1.0
    x = np.arange(n) - n / 2
    X3, X2, X1 = np.meshgrid(x, x, x, indexing="ij")
    blob = A * np.exp(-((X1 - c[0]) ** 2 + (X2 - c[1]) ** 2 + (X3 - c[2]) ** 2) / (2 * s * s))
    geom = O.Geometry(n=n, h=h, w=w, theta=theta, phi=phi, filter="none")
    got = O.forward_nudft(geom, blob)
    want = np.stack([blob_projection(c, s, A, t, phi, h, w) for t in theta])
    assert rel(got, want) < 1e-5


# ------------------------------------------------------------------ P7: brute force on tiny inputs
def test_P7_brute_force_16():
    rng = np.random.default_rng(7)
    n, nz, h, w, nth = 16, 8, 16, 16, 6
    theta = rng.uniform(0, 2 * np.pi, nth)
    d = rng.standard_normal((nth, h, w))
    for filt in ("none", "ramp"):
        geom = O.Geometry(n=n, nz=nz, h=h, w=w, theta=theta, phi=math.radians(20.0), filter=filt, cu=8.3)
        a = O.fbp_nudft(geom, d)
        b = O.fbp_brute(geom, d)
        assert rel(a, b) < 1e-12
        cgrid = O.fbp_gridded(geom, d, kernel="kb", W=8, sigma=2.0)
        assert rel(cgrid, a) < 1e-6      # random (non band-limited) data: high-frequency corners dominate


def test_nonpow2_sizes_use_naive_dft():
    rng = np.random.default_rng(8)
    geom = O.Geometry(n=6, nz=4, h=6, w=10, theta=[0.5, 3.0], phi=0.3, filter="ramp")
    d = rng.standard_normal((2, 6, 10))
    assert rel(O.fbp_nudft(geom, d), O.fbp_brute(geom, d)) < 1e-12


# ------------------------------------------------------------------ kernels of path C
@pytest.mark.parametrize("kernel", ["kb", "gauss"])
def test_kernel_transform_pair_by_quadrature(kernel):
    """kaphat is the continuous Fourier transform of kap: check the closed form by numerical quadrature of
    kap itself (Gauss: up to the truncation at |t| = W/2)."""
    W, sigma = 6, 2.0
    shape = O.default_shape(kernel, W, sigma)
    t = np.linspace(-W / 2, W / 2, 20001)
    k = np.array([O.kap(kernel, W, shape, x) for x in t])
    for s in [0.0, 0.05, 0.125, 0.25]:
        num = np.trapezoid(k * np.cos(2 * np.pi * s * t), t)
        ana = O.kaphat(kernel, W, shape, s)
        assert abs(num - ana) / ana < (1e-6 if kernel == "kb" else 2e-3)
    assert abs(O.default_shape("kb", 6, 2.0) - 13.8551) < 1e-3
    assert O.kap(kernel, W, shape, 0.0) == pytest.approx(1.0)
    assert O.kap("kb", W, O.default_shape("kb", W, sigma), W / 2 + 1e-9) == 0.0


# ------------------------------------------------------------------ P8: path C against path A
def _tiny_case(filter="ramp", n=32, nth=24, seed=3):
    """configs[0]-like: band-limited blobs in a thin slab, phi = 20 deg."""
    rng = np.random.default_rng(seed)
    h = w = n
    phi = math.radians(20.0)
    theta = 2 * np.pi * np.arange(nth) / nth
    proj = np.zeros((nth, h, w))
    for _ in range(6):
        r, a = 0.3 * n * math.sqrt(rng.uniform()), rng.uniform(0, 2 * np.pi)
        c = np.array([r * math.cos(a), r * math.sin(a), rng.uniform(-n / 16, n / 16)])
        s, A = rng.uniform(1.5, 3.0), rng.uniform(0.5, 1.0)
        proj += np.stack([blob_projection(c, s, A, t, phi, h, w) for t in theta])
    return O.Geometry(n=n, h=h, w=w, theta=theta, phi=phi, filter=filter), proj


def test_P8_gridded_path_matches_nudft():
    geom, proj = _tiny_case()
    a = O.fbp_nudft(geom, proj)
    assert rel(O.fbp_gridded(geom, proj, kernel="kb"), a) < 1e-5          # KB, W=6, sigma=2
    g = rel(O.fbp_gridded(geom, proj, kernel="gauss"), a)
    assert 5e-5 < g < 2e-3                                                # reading Q5: Gaussian misses 2e-4 at W=6
    assert rel(O.fbp_gridded(geom, proj, kernel="gauss", W=12), a) < 1e-5
    # float32 input goes through the same path
    assert rel(O.fbp_gridded(geom, proj.astype(np.float32)), O.fbp_nudft(geom, proj.astype(np.float32))) < 1e-5


def test_P8b_slice_path_matches_full_gridded_and_nudft():
    geom, proj = _tiny_case(nth=12)
    a = O.fbp_nudft(geom, proj)
    for i3 in (3, 16, 29):
        sl = O.fbp_gridded_slice(geom, proj, i3)
        rms = np.linalg.norm(a) / math.sqrt(geom.nz)             # error relative to the volume's slice RMS
        assert np.linalg.norm(sl - a[i3]) / rms < 1e-5


def test_Q7_out_of_band_samples_wrap():
    """|xi1| reaches (1/2) sqrt(1+sin^2 phi) > 1/2: those samples must alias periodically (e^{2 pi i x xi} has
    period 1 in xi on integer voxels).  A delta-like projection makes the corners matter."""
    n = 16
    theta = np.array([math.pi / 4, 2.0])
    geom = O.Geometry(n=n, h=n, w=n, theta=theta, phi=math.radians(40.0), filter="none")
    d = np.zeros((2, n, n)); d[:, n // 2 + 1, n // 2 - 2] = 1.0
    a = O.fbp_nudft(geom, d)
    assert rel(O.fbp_gridded(geom, d, W=10), a) < 1e-7


def test_kaiser_bessel_kernel_against_library_bessel():
    """orc_kap evaluates I0 by its power series; scipy.special.i0 (a library routine on another algorithm) must
    agree to rounding over the whole support, for several widths."""
    from scipy.special import i0
    for W, sigma in ((4, 2.0), (6, 2.0), (8, 2.0), (6, 1.5)):
        beta = O.default_shape("kb", W, sigma)
        for t in np.linspace(-W / 2, W / 2, 41):
            want = i0(beta * math.sqrt(max(0.0, 1 - (2 * t / W) ** 2))) / i0(beta)
            assert abs(O.kap("kb", W, beta, t) - want) <= 1e-13 * max(want, 1e-3)


# ------------------------------------------------------------------ P9: path B ("Linerec")
def test_P9_direct_path_agrees_at_interpolation_level():
    """B differs from A only by the interpolation of the filtered projections (linear against trigonometric).
    Linear interpolation multiplies the spectrum by sinc^2(k_u/w) sinc^2(k_v/h) (plus weak images): path A fed
    with projections weighted that way must be CLOSER to B than path A itself is."""
    geom, proj = _tiny_case()
    a, b = O.fbp_nudft(geom, proj), O.fbp_direct(geom, proj)
    ku, kv = np.fft.fftfreq(geom.w), np.fft.fftfreq(geom.h)
    wt = (np.sinc(kv) ** 2)[:, None] * (np.sinc(ku) ** 2)[None, :]
    pb = np.ascontiguousarray(np.real(np.fft.ifft2(np.fft.fft2(proj, axes=(1, 2)) * wt, axes=(1, 2))))
    a2 = O.fbp_nudft(geom, pb)
    m = slice(4, -4)
    e_plain, e_weighted = rel(b[m, m, m], a[m, m, m]), rel(b[m, m, m], a2[m, m, m])
    assert e_plain < 0.04
    assert e_weighted < 0.6 * e_plain


def _blob_volume(c, s, A, n, nz):
    x, z = np.arange(n) - n / 2, np.arange(nz) - nz / 2
    X3, X2, X1 = np.meshgrid(z, x, x, indexing="ij")
    return A * np.exp(-((X1 - c[0]) ** 2 + (X2 - c[1]) ** 2 + (X3 - c[2]) ** 2) / (2 * s * s))


@pytest.mark.parametrize("s,tol", [(2.0, 3e-3), (3.0, 1e-3)])
def test_P9b_ray_driven_forward_matches_analytic_line_integrals(s, tol):
    """Eq. 1-2 sampled along the beam with trilinear interpolation.  Trilinear interpolation of a
    sampled band-limited blob is the blob convolved with the unit hat in each axis; the hat has variance 1/6, so
    to second order in 1/s the interpolated volume is the Gaussian of variance s^2 + 1/6 and amplitude
    A (s/s')^3, whose line integral is closed form.  The remainder is the hat's fourth cumulant, O(s^-4).
    Against the unblurred blob the same projection is off by several per cent (checked: the pin has teeth)."""
    n, nz, h, w = 48, 32, 64, 64
    phi = math.radians(25.0)
    theta = np.array([0.4, 2.2, 3.9])
    c, A = np.array([3.0, -4.0, 1.5]), 1.0
    geom = O.Geometry(n=n, h=h, w=w, theta=theta, phi=phi, nz=nz, filter="none")
    got = O.fp_ray(geom, _blob_volume(c, s, A, n, nz))
    s2 = math.sqrt(s * s + 1.0 / 6.0)
    want = np.stack([blob_projection(c, s2, A * (s / s2) ** 3, t, phi, h, w) for t in theta])
    raw = np.stack([blob_projection(c, s, A, t, phi, h, w) for t in theta])
    assert rel(got, want) < tol
    assert rel(got, raw) > 4 * tol


def test_P9c_voxel_driven_forward_conserves_mass_and_is_percent_accurate():
    """orc_fp_direct (the exact transpose of the bilinear back-projector, pinned as such by P6) splats every voxel
    with hat weights that sum to one: each projection's total equals the volume's total exactly, whatever the
    angle, and that total is the blob's A (2 pi)^{3/2} s^3.  Pointwise the voxel-driven splat carries the known
    few-per-cent moire of hat footprints on a tilted lattice, so it is pinned at that level only."""
    n, nz, h, w = 48, 32, 64, 64
    phi = math.radians(25.0)
    theta = np.array([0.0, 0.4, 2.2])
    c, s, A = np.array([3.0, -4.0, 1.5]), 3.0, 1.0
    f = _blob_volume(c, s, A, n, nz)
    geom = O.Geometry(n=n, h=h, w=w, theta=theta, phi=phi, nz=nz, filter="none")
    got = O.fp_direct(geom, f)
    assert np.allclose(got.sum(axis=(1, 2)), f.sum(), rtol=1e-12)
    assert abs(f.sum() / (A * (2 * math.pi) ** 1.5 * s ** 3) - 1) < 1e-4
    want = np.stack([blob_projection(c, s, A, t, phi, h, w) for t in theta])
    assert rel(got, want) < 0.05


# ------------------------------------------------------------------ P10: S0
def test_P10_prep_inverts_detector_model():
    rng = np.random.default_rng(10)
    h, w = 8, 12
    d = rng.uniform(0.0, 2.0, (3, h, w))
    dark = (100 + rng.standard_normal((h, w))).astype(np.float32)
    flat = (30000 * (1 + 0.01 * rng.standard_normal((h, w)))).astype(np.float32)
    raw = np.exp(-d) * (flat.astype(float) - dark) + dark
    raw16 = np.round(raw).astype(np.uint16)
    geom = O.Geometry(n=8, h=h, w=w, theta=[0, 1, 2], phi=0.3, dark=dark, flat=flat)
    for th in range(3):
        got = O.prep(geom, raw16, th)
        assert np.all(np.abs(got - d[th]) <= 0.5 / (raw[th] - dark) * 1.0001 + 1e-12)
    z = np.zeros((3, h, w), dtype=np.uint16)                     # raw < dark: clamp at tmin
    assert np.allclose(O.prep(geom, z, 0), -math.log(1e-6))


# ------------------------------------------------------------------ P11: real part and Nyquist bins (reading Q8)
def test_P11_imaginary_part_comes_from_nyquist_bins_only():
    geom, proj = _tiny_case(n=16, nth=8)
    re, im = O.fbp_nudft(geom, proj, return_imag=True)
    assert 1e-5 < np.linalg.norm(im) / np.linalg.norm(re)        # a naive Hermitian shortcut would be wrong
    # remove the Nyquist row and column of every projection spectrum -> imaginary part vanishes
    h = w = 16
    F = np.fft.fft2(proj, axes=(1, 2)); F[:, h // 2, :] = 0; F[:, :, w // 2] = 0
    re2, im2 = O.fbp_nudft(geom, np.ascontiguousarray(np.fft.ifft2(F, axes=(1, 2)).real), return_imag=True)
    assert np.linalg.norm(im2) / np.linalg.norm(re2) < 1e-13


# ------------------------------------------------------------------ stored values (written by tests/golden/make_golden.py)
def test_golden_nudft_tiny16_is_reproduced():
    import importlib.util
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "make_golden.py"))
    mg = importlib.util.module_from_spec(spec); spec.loader.exec_module(mg)
    geom, d = mg.case()
    want = np.loadtxt(os.path.join(here, "nudft_tiny16.txt")).reshape(geom.nz, geom.n, geom.n)
    assert rel(O.fbp_nudft(geom, d), want) < 1e-13
    assert rel(O.fbp_brute(geom, d), want) < 1e-12


def test_paper_table1_gain_column_is_consistent():
    """'Gain' = Linerec / Fourierrec time (the fixture is the paper's own print-out)."""
    import os
    t = np.loadtxt(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "paper_table1.txt"))
    assert np.all(np.abs(t[:, 4] / t[:, 3] - t[:, 5]) < 0.06)


# ---- f4: Parzen window, u-padding, 2-D spectral multiplier -----------------------------------------
def test_P12_parzen_window_is_the_fourfold_box_convolution():
    """PAPER.md:109 names the Parzen low-pass.  The Parzen window is, independently of its piecewise-cubic formula,
    the four-fold self-convolution of a box (cubic B-spline) normalised to 1 at the origin: checked on a fine grid,
    plus the exact values P(0) = 1, P(1/2) = 1/4, P(1) = 0."""
    w = 64
    g_r = O.Geometry(32, 16, w, np.linspace(0, 2 * np.pi, 8, endpoint=False), 0.3, filter="ramp")
    g_p = O.Geometry(32, 16, w, np.linspace(0, 2 * np.pi, 8, endpoint=False), 0.3, filter="parzen")
    Hr, Hp = O.filter_response(g_r), O.filter_response(g_p)
    k = np.arange(-w // 2, w // 2)
    ratio = Hp[k != 0] / Hr[k != 0]
    m = 4000                                   # samples per box; box width 1/2 so that the 4-fold convolution spans [-1, 1]
    box = np.ones(m)
    b4 = np.convolve(np.convolve(box, box), np.convolve(box, box)).astype(np.float64)
    b4 /= b4.max()
    xs = (np.arange(len(b4)) - (len(b4) - 1) / 2) / (2.0 * m)   # total support 4 m samples = 2 units
    ref = np.interp(np.abs(k[k != 0]) / (w / 2), xs, b4)
    assert np.abs(ratio - ref).max() < 2e-3
    assert abs(Hp[w // 2 + w // 4] / Hr[w // 2 + w // 4] - 0.25) < 1e-12   # x = 1/2
    assert abs(Hp[0]) < 1e-15                                              # x = 1 (Nyquist)
    assert abs(Hp[w // 2 + 1] / Hr[w // 2 + 1] - (1 - 6 * (2 / w) ** 2 + 6 * (2 / w) ** 3)) < 1e-12


def test_P13_padded_rows_are_a_linear_convolution_with_the_ramp_kernel():
    """Reading Q11b: after edge extension to 2w samples the filter is the LINEAR convolution of the extended row with
    the band-limited ramp kernel h_RL (h[0] = 1/4, h[odd j] = -1/(pi j)^2), truncated to |j| <= w: numpy.convolve of
    the closed-form kernel samples is the library routine it must reduce to."""
    rng = np.random.default_rng(5)
    n, h, w, nth, phi = 16, 8, 32, 6, 0.35
    theta = np.linspace(0, 2 * np.pi, nth, endpoint=False)
    proj = rng.normal(size=(nth, h, w))
    g = O.Geometry(n, h, w, theta, phi, filter="ramp", pad=2)
    q = O.filter_rows_padded(g, proj, 2)
    wp, off = 2 * w, w // 2
    j = np.arange(-wp // 2, wp // 2)
    hk = np.where(j == 0, 0.25, np.where(j % 2 == 0, 0.0, -1.0 / (np.pi * np.maximum(np.abs(j), 1)) ** 2))
    scale = np.pi * np.cos(phi) / nth
    for jv in (0, 3, 7):
        ext = np.concatenate([np.full(off, proj[2, jv, 0]), proj[2, jv], np.full(off, proj[2, jv, -1])])
        # circular convolution of length 2w == linear convolution wrapped once; written as the full linear
        # convolution folded back modulo 2w (kernel index j = -w .. w-1)
        lin = np.convolve(ext, hk)                       # index i <-> position i + j[0]
        circ = np.zeros(wp)
        for i, v in enumerate(lin):
            circ[(i + j[0]) % wp] += v
        assert np.abs(q[jv] - scale * circ[off:off + w]).max() < 1e-12
    # and the point of padding: a constant row is filtered to (nearly) zero instead of wrapping edge to edge
    gc = O.Geometry(n, h, w, theta, phi, filter="ramp", pad=2)
    ramp = np.tile(np.linspace(0.0, 1.0, w), (nth, h, 1))
    qp = O.filter_rows_padded(gc, ramp, 0)
    g1 = O.Geometry(n, h, w, theta, phi, filter="ramp")
    q1 = np.fft.ifft(np.fft.fft(ramp[0, 0]) * np.fft.ifftshift(O.filter_response(g1))).real
    assert np.abs(qp[0]).max() < 0.25 * np.abs(q1).max()   # the unpadded filter sees the 1 -> 0 jump at the wrap


def test_P14_spectral_multiplier_scales_a_plane_wave_exactly():
    """Reading Q17: the 2-D multiplier 1/(1 + alpha ((k_u/w)^2 + (k_v/h)^2)).  A projection that is one plane wave
    cos(2 pi (a u/w + b v/h)) has the two spectral bins (b, a) and (-b, -a) only; each must come out as
    H[a] / 2 / (1 + alpha (a^2/w^2 + b^2/h^2)), and alpha = 0 must change nothing."""
    n, h, w, nth, phi = 16, 16, 32, 4, 0.3
    theta = np.linspace(0, 2 * np.pi, nth, endpoint=False)
    a, b, alpha = 5, -3, 37.0
    ju, jv = np.meshgrid(np.arange(w) - w / 2, np.arange(h) - h / 2)
    proj = np.tile(np.cos(2 * np.pi * (a * ju / w + b * jv / h)), (nth, 1, 1))
    g0 = O.Geometry(n, h, w, theta, phi, filter="ramp")
    g1 = O.Geometry(n, h, w, theta, phi, filter="ramp", alpha=alpha)
    H = O.filter_response(g0)
    s0, s1 = O.spectrum(g0, proj, 1), O.spectrum(g1, proj, 1)
    mult = 1.0 / (1.0 + alpha * ((a / w) ** 2 + (b / h) ** 2))
    assert abs(s0[b + h // 2, a + w // 2] - 0.5 * H[a + w // 2]) < 1e-13
    assert abs(s1[b + h // 2, a + w // 2] - 0.5 * H[a + w // 2] * mult) < 1e-13
    assert abs(s1[-b + h // 2, -a + w // 2] - 0.5 * H[-a + w // 2] * mult) < 1e-13
    mask = np.ones((h, w), bool)
    mask[b + h // 2, a + w // 2] = mask[-b + h // 2, -a + w // 2] = False
    assert np.abs(s1[mask]).max() < 1e-13
