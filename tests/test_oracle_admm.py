"""Pins of the ADMM-TV oracle (oracle/admm_tv.py; Appendix A, Eqs. 10-20).  None of them re-types the
algorithm: they are the optimality conditions and invariants the paper's formulas imply."""
import numpy as np

from oracle import admm_tv as A
from oracle import lam_oracle as O


def _setup(n=12, nz=6, h=12, w=12, nth=8, phi=0.4, seed=0):
    rng = np.random.default_rng(seed)
    theta = np.linspace(0, 2 * np.pi, nth, endpoint=False)
    g = O.Geometry(n, h, w, theta, phi, nz=nz, filter="none")
    mu_true = np.zeros((nz, n, n))
    mu_true[2:4, 3:8, 4:9] = 1.0          # a piecewise-constant block: what TV favours
    d = O.forward_nudft(g, mu_true) + 0.02 * rng.normal(size=(nth, h, w))
    return g, d, mu_true


def test_div_is_minus_the_adjoint_of_grad():
    rng = np.random.default_rng(1)
    mu, q = rng.normal(size=(5, 6, 7)), rng.normal(size=(3, 5, 6, 7))
    assert abs((A.grad(mu) * q).sum() + (mu * A.div(q)).sum()) < 1e-12


def test_shrink_solves_the_psi_subproblem_of_eq15():
    """psi = argmin alpha |psi| - lam.psi + rho/2 |g - psi|^2 (Eq. 13 in psi).  Optimality: for psi != 0,
    alpha psi/|psi| - lam - rho (g - psi) = 0; for psi = 0, |lam + rho g| <= alpha.  Also better than the paper's
    printed factors (2 lam/rho, 2 alpha/rho), which do NOT satisfy it: reading Q18 has teeth."""
    rng = np.random.default_rng(2)
    g, lam = rng.normal(size=(3, 4, 5, 6)), 0.3 * rng.normal(size=(3, 4, 5, 6))
    alpha, rho = 0.7, 1.3
    psi = A.shrink(g + lam / rho, alpha / rho)
    nrm = np.sqrt((psi ** 2).sum(0))
    nz = nrm > 0
    res = alpha * psi / np.maximum(nrm, 1e-300) - lam - rho * (g - psi)
    assert np.abs(res[:, nz]).max() < 1e-12
    assert (np.sqrt(((lam + rho * g) ** 2).sum(0))[~nz] <= alpha + 1e-12).all()
    assert nz.any() and (~nz).any()
    obj = lambda p: (alpha * np.sqrt((p ** 2).sum(0)) - (lam * p).sum(0) + 0.5 * rho * ((g - p) ** 2).sum(0)).sum()
    printed = A.shrink(g + 2 * lam / rho, 2 * alpha / rho)
    assert obj(psi) < obj(printed) - 1e-6
    for _ in range(20):   # and no random perturbation does better
        assert obj(psi) <= obj(psi + 1e-3 * rng.normal(size=psi.shape)) + 1e-12


def test_cg_steps_decrease_F_and_reach_the_optimality_condition_of_eq17():
    g, d, _ = _setup()
    mu, hist = A.admm_tv(g, d, alpha=0.05, rho=0.5, n_outer=1, n_cg=40)
    F = np.array(hist["F"])
    assert (np.diff(F) <= 1e-12 * F[0]).all()          # exact line search on a quadratic: monotone
    # after many CG steps grad F (Eq. 18) vanishes: L^T(L mu - d) - rho div(grad mu - psi0 + lam0/rho) = 0 with psi0 = lam0 = 0
    gF = O.fbp_nudft(g, O.forward_nudft(g, mu) - d) - 0.5 * A.div(A.grad(mu))
    g0 = O.fbp_nudft(g, -d)
    assert np.linalg.norm(gF) < 1e-6 * np.linalg.norm(g0)


def test_admm_iterations_behave_like_admm():
    """Over the outer iterations the constraint residual |grad mu - psi| shrinks, the data term stays bounded, and the
    TV-regularised result is closer to the piecewise-constant truth than the unregularised least-squares solution."""
    g, d, mu_true = _setup()
    mu, hist = A.admm_tv(g, d, alpha=0.15, rho=1.0, n_outer=12, n_cg=4)
    r_first = None
    mu1, h1 = A.admm_tv(g, d, alpha=0.15, rho=1.0, n_outer=1, n_cg=4)
    r1 = np.linalg.norm(A.grad(mu1) - h1["psi"])
    r12 = np.linalg.norm(A.grad(mu) - hist["psi"])
    assert r12 < 0.5 * r1
    ls, _ = A.admm_tv(g, d, alpha=0.0, rho=1e-9, n_outer=1, n_cg=48)   # plain least squares by CG
    tv = lambda x: np.sqrt((A.grad(x) ** 2).sum(0)).sum()
    assert tv(mu) < 0.8 * tv(ls)
    assert np.linalg.norm(mu - mu_true) < np.linalg.norm(ls - mu_true)
