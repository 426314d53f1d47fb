"""Pins of the oracle's exact Lagrangian Hessian path (Eq. 5, Eq. 24-25)."""
import numpy as np
import torch

import oracle as O
import workloads as W


def _case(**kw):
    wl = W.make_workload(6, **kw)
    return wl, wl.u_hat[0].numpy(), wl.cdata[0].numpy(), wl.params


def test_hessian_matches_finite_differences_of_the_lagrangian_gradient():
    """W v = I v + d/d eps [ J(u + eps v)^T lam ] on the free levels (central differences; the constraints are at most
    quadratic there, so the difference quotient is exact up to rounding)."""
    wl, uh, u0, p = _case(batch=1, nx=16, nt=9)
    K, F, E = O.fluxk_counts(p, wl.nt)
    g = np.random.default_rng(1)
    lam = np.zeros(O.num_rows(wl.kind, wl.nx, 1, wl.nt, p))
    sl = O.row_slices(wl.kind, wl.nx, 1, wl.nt, p)
    lam[sl["energy"]] = 0.3 * g.standard_normal(E)                    # small enough for every level to pass the safeguard
    lam[sl["mass"]] = g.standard_normal(F)
    Wm = O.lagrangian_hessian(wl.kind, uh, lam, p)
    assert abs(Wm - Wm.T).max() == 0.0
    v = np.zeros_like(uh)
    v[K + 1:] = g.standard_normal(v[K + 1:].shape)                    # free levels only (pinned levels: W = I by R22)
    eps = 1e-3
    gp = O.jacobian(wl.kind, uh + eps * v, p).T @ lam
    gm = O.jacobian(wl.kind, uh - eps * v, p).T @ lam
    fd = v.ravel() + (gp - gm) / (2 * eps)
    free = np.zeros(uh.shape, dtype=bool)
    free[K + 1:] = True
    np.testing.assert_allclose((Wm @ v.ravel())[free.ravel()], fd[free.ravel()], rtol=0, atol=1e-11)
    # the Hessian of the energy rows also reaches the pinned level K (role "earlier level" of row E_0); it is left out there
    assert np.abs((Wm @ np.ones(Wm.shape[0]))[: (K + 1) * wl.nx] - 1.0).max() == 0.0


def test_one_newton_step_equals_a_dense_solve_of_the_kkt_matrix():
    wl, uh, u0, p = _case(batch=1, nx=8, nt=6, params=dict(flux_steps=2))
    g = np.random.default_rng(2)
    lam0 = 0.2 * g.standard_normal(O.num_rows(wl.kind, wl.nx, 1, wl.nt, p))
    u = uh + 0.01 * g.standard_normal(uh.shape)
    J = O.jacobian(wl.kind, u, p)
    h = O.residual(wl.kind, u, u0, p)
    Wm = O.lagrangian_hessian(wl.kind, u, lam0, p)
    du, lam = O.solve_kkt_sparse_lu(Wm, J, (u - uh).ravel(), h)
    n, m = Wm.shape[0], J.shape[0]
    Kd = np.block([[Wm.toarray(), J.toarray().T], [J.toarray(), np.zeros((m, m))]])
    x = np.linalg.solve(Kd, -np.concatenate([(u - uh).ravel(), h]))
    np.testing.assert_allclose(du, x[:n], rtol=0, atol=1e-12)
    np.testing.assert_allclose(lam, x[n:], rtol=0, atol=1e-11)


def test_both_hessians_share_the_kkt_point_and_the_exact_one_converges_faster():
    """Same KKT point (the limit does not depend on W); Gauss-Newton contracts linearly on this row set, Newton with the
    exact Hessian quadratically: ||d|| falls at least like its square once it is small."""
    wl, uh, u0, p = _case(batch=1, nx=64, nt=96, noise=0.3)     # noise 0.3: Gauss-Newton needs 12 solves here, Newton 6
    gn_hist, ex_hist = [], []
    a = O.project(wl.kind, uh, u0, dict(p, hessian=0), history=gn_hist)
    b = O.project(wl.kind, uh, u0, dict(p, hessian=1), history=ex_hist)
    assert a["status"] == 0 and b["status"] == 0
    assert a["iters"] >= 10 and b["iters"] <= 7, (a["iters"], b["iters"])
    np.testing.assert_allclose(b["u"], a["u"], rtol=0, atol=2e-9)       # Gauss-Newton stops RMS(d) <= 1e-10 short of the limit (R18)
    np.testing.assert_allclose(b["lam"], a["lam"], rtol=0, atol=1e-7 * max(1.0, np.abs(a["lam"]).max()))
    J = O.jacobian(wl.kind, b["u"], p)
    stat = (b["u"] - uh).ravel() + J.T @ b["lam"]
    assert np.abs(stat).max() <= 1e-11 * max(1.0, np.abs(b["lam"]).max())    # quadratic rate: P4's bound holds again
    assert np.abs(O.residual(wl.kind, b["u"], u0, p)).max() < 1e-12


def test_safeguard_falls_back_to_gauss_newton_levels():
    """Multipliers that make a level's W_k indefinite: that level uses I; the iteration still reaches the KKT point."""
    wl, uh, u0, p = _case(batch=1, nx=16, nt=9)
    K, F, E = O.fluxk_counts(p, wl.nt)
    sl = O.row_slices(wl.kind, wl.nx, 1, wl.nt, p)
    lam = np.zeros(O.num_rows(wl.kind, wl.nx, 1, wl.nt, p))
    lam[sl["energy"]] = np.where(np.arange(E) % 2 == 0, -200.0, 200.0)      # a = 1 + dx (lam_f - lam_{f+1}) far below 0 on every other level
    Wm = O.lagrangian_hessian(wl.kind, uh, lam, p)
    d = Wm.diagonal().reshape(wl.nt, wl.nx)
    assert (d[: K + 1] == 1.0).all()
    assert (d[K + 1:] == 1.0).any() and (d[K + 1:] >= O.HESS_SAFEGUARD).all()
    ev = np.linalg.eigvalsh(Wm.toarray())
    assert ev.min() >= O.HESS_SAFEGUARD - 1e-12
