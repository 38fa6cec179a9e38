"""ADMM-TV reconstruction of PAPER.md Appendix A (Eqs. 10-20) in plain numpy fp64.
TEST INFRASTRUCTURE ONLY (same rules as lam_oracle.py: only tests/, smoke() and bench.py's CPU legs may import it;
it shares nothing with the CUDA path).

Follows the paper step by step, in its notation:
  Eq. 10-11  minimise  1/2 ||L mu - d||^2 + alpha || |grad mu| ||_1      (isotropic TV)
  Eq. 12-13  split grad mu = psi, augmented Lagrangian A_rho(mu, psi, lambda)
  Eq. 14     mu-update: a few conjugate-gradient steps on F(mu) of Eq. 17 with the gradient of Eq. 18,
             directions by the Dai-Yuan formula Eq. 19
  Eq. 15     psi-update: soft threshold
  Eq. 16     lambda <- lambda + rho (grad mu - psi)
L and L^T are the oracle's exact NUDFT pair (orc_forward_nudft, orc_fbp_nudft with filter none; Eqs. 5, 7).

Readings:
  Q18  Eq. 20 as printed has 2 lambda / rho and 2 alpha / rho; minimising Eq. 13 over psi gives
       psi = shrink(grad mu + lambda / rho, alpha / rho), shrink(v, t) = v / |v| * max(0, |v| - t) with |v| the
       Euclidean norm over the three gradient components (Eq. 11).  The factors 2 do not follow from Eqs. 13, 17
       (SURVEY.md 8(f) f2 flags them); the re-derived form is used, and pinned by the optimality condition of Eq. 15.
  Q19  "gamma_m is a step length computed by a line-search procedure": F is quadratic, so the exact minimiser along
       eta is used, gamma = -<grad F, eta> / <eta, H eta>, H = L^T L - rho div grad.
  Q20  grad = forward differences with a zero last difference (Neumann), div = -grad^T exactly.
"""
import numpy as np

from . import lam_oracle as O


def grad(mu):
    """(3, nz, n, n): forward differences along x1 (last axis), x2, x3; zero at the far face."""
    g = np.zeros((3,) + mu.shape)
    g[0, :, :, :-1] = mu[:, :, 1:] - mu[:, :, :-1]
    g[1, :, :-1, :] = mu[:, 1:, :] - mu[:, :-1, :]
    g[2, :-1, :, :] = mu[1:, :, :] - mu[:-1, :, :]
    return g


def div(q):
    """div = -grad^T (PAPER.md: "the divergence operator div is the adjoint to -grad"):
    (grad^T q)[i] = q[i-1] - q[i] along each axis (q of the far face is never used), so div q[i] = q[i] - q[i-1]."""
    d = np.zeros(q.shape[1:])
    d[:, :, :-1] += q[0, :, :, :-1]
    d[:, :, 1:] -= q[0, :, :, :-1]
    d[:, :-1, :] += q[1, :, :-1, :]
    d[:, 1:, :] -= q[1, :, :-1, :]
    d[:-1, :, :] += q[2, :-1, :, :]
    d[1:, :, :] -= q[2, :-1, :, :]
    return d


def shrink(v, t):
    """isotropic soft threshold: v / |v| max(0, |v| - t), |v| over the component axis 0 (Eq. 20, reading Q18)."""
    nrm = np.sqrt((v ** 2).sum(axis=0))
    scale = np.where(nrm > t, 1.0 - t / np.maximum(nrm, 1e-300), 0.0)
    return v * scale[None]


def lagrangian(Lmu_minus_d, gmu, psi, lam, alpha, rho):
    """Eq. 13."""
    return (0.5 * float((Lmu_minus_d ** 2).sum()) + alpha * float(np.sqrt((psi ** 2).sum(axis=0)).sum())
            + float((lam * (gmu - psi)).sum()) + 0.5 * rho * float(((gmu - psi) ** 2).sum()))


def admm_tv(geom, d, alpha, rho, n_outer, n_cg, L=None, LT=None, track=True):
    """geom: O.Geometry with filter "none".  d: projections [ntheta][h][w] (float64).
    Returns mu and a history dict (||grad F|| after every CG step, psi, lam; with track: F before/after every CG step and
    the Lagrangian per outer iteration, which cost one more application of L each)."""
    assert geom.filter == "none"
    if L is None:
        L = lambda f: O.forward_nudft(geom, f)
    if LT is None:
        LT = lambda r: O.fbp_nudft(geom, np.ascontiguousarray(r))
    mu = np.zeros((geom.nz, geom.n, geom.n))
    psi = np.zeros((3,) + mu.shape)
    lam = np.zeros_like(psi)
    hist = {"F": [], "lagr": [], "gradF_norm": []}

    def F(mu_):  # Eq. 17
        return 0.5 * float(((L(mu_) - d) ** 2).sum()) + 0.5 * rho * float(((grad(mu_) - psi + lam / rho) ** 2).sum())

    def gradF(mu_):  # Eq. 18
        return LT(L(mu_) - d) - rho * div(grad(mu_) - psi + lam / rho)

    for k in range(n_outer):
        g = gradF(mu)
        eta = -g
        if track:
            hist["F"].append(F(mu))
        for m in range(n_cg):
            Leta, Geta = L(eta), grad(eta)
            gamma = -float((g * eta).sum()) / (float((Leta ** 2).sum()) + rho * float((Geta ** 2).sum()))  # reading Q19
            mu = mu + gamma * eta
            g_new = gradF(mu)
            beta = float((g_new ** 2).sum()) / float(((g_new - g) * eta).sum())                             # Eq. 19
            eta = -g_new + beta * eta
            g = g_new
            hist.setdefault("gnorm_steps", []).append(float(np.sqrt((g ** 2).sum())))
            if track:
                hist["F"].append(F(mu))
        hist["gradF_norm"].append(float(np.sqrt((g ** 2).sum())))
        gmu = grad(mu)
        psi = shrink(gmu + lam / rho, alpha / rho)    # Eq. 15 / 20 (reading Q18)
        lam = lam + rho * (gmu - psi)                 # Eq. 16
        if track:
            hist["lagr"].append(lagrangian(L(mu) - d, gmu, psi, lam, alpha, rho))
    hist["psi"], hist["lam"] = psi, lam
    return mu, hist
