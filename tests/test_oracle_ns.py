"""Pins of the oracle for kind 6, NS2D_VORT_ENST (Eq. 20: IC + total vorticity + enstrophy) -- CPU only."""
import numpy as np

import oracle as O
import workloads as W


def _closed_form(wl, b):
    """Projection of every level k >= 1 onto {sum w = sum w_IC} n {sum w^2 = sum w_IC^2}: a sphere inside a hyperplane.
    The nearest point keeps the direction of the deviation from the mean and takes the mean and the radius of the IC;
    multipliers from the stationarity condition w* - w_hat + lam_V a 1 + lam_Z 2 a w* = 0 split into mean and deviation."""
    uh, u0, p = wl.u_hat[b].numpy(), wl.cdata[b].numpy(), wl.params
    a = p["dx"] * p["dy"]
    m, r = u0.mean(), np.linalg.norm(u0 - u0.mean())
    u = np.empty_like(uh)
    u[0] = u0
    lamV, lamZ = [], []
    for k in range(1, wl.nt):
        mh = uh[k].mean()
        dev = uh[k] - mh
        s = np.linalg.norm(dev) / r
        u[k] = m + dev / s
        lamZ.append((s - 1.0) / (2.0 * a))
        lamV.append((mh - s * m) / a)
    lam = np.concatenate([(uh[0] - u0).ravel(), lamV, lamZ])
    return u, lam


def test_generic_newton_kkt_route_equals_the_sphere_hyperplane_projection():
    wl = W.make_workload(9, batch=2, nx=8, ny=6, nt=7)
    for b in range(wl.batch):
        u_cf, lam_cf = _closed_form(wl, b)
        for hz in (0, 1):
            o = O.project(wl.kind, wl.u_hat[b].numpy(), wl.cdata[b].numpy(), dict(wl.params, hessian=hz))
            assert o["status"] == 0
            np.testing.assert_allclose(o["u"], u_cf, rtol=0, atol=1e-11)
            np.testing.assert_allclose(o["lam"], lam_cf, rtol=0, atol=1e-9 * max(1.0, np.abs(lam_cf).max()))
            assert np.abs(O.residual(wl.kind, o["u"], wl.cdata[b].numpy(), wl.params)).max() < 1e-12


def test_jacobian_matches_finite_differences_and_rows_are_independent():
    wl = W.make_workload(9, batch=1, nx=6, ny=4, nt=4)
    u, u0, p = wl.u_hat[0].numpy(), wl.cdata[0].numpy(), wl.params
    J = O.jacobian(wl.kind, u, p).toarray()
    assert J.shape == (O.num_rows(wl.kind, wl.nx, wl.ny, wl.nt, p), u.size)
    eps = 1e-6
    for j in np.random.default_rng(0).choice(u.size, 12, replace=False):
        e = np.zeros(u.size); e[j] = eps
        fd = (O.residual(wl.kind, u + e.reshape(u.shape), u0, p) - O.residual(wl.kind, u - e.reshape(u.shape), u0, p)) / (2 * eps)
        np.testing.assert_allclose(J[:, j], fd, rtol=0, atol=1e-9)
    assert np.linalg.matrix_rank(J) == J.shape[0]
    assert O.full_rank_rows(wl.kind, wl.nx, wl.ny, wl.nt, p).all()


def test_feasible_field_and_invariants():
    """A periodically shifted IC keeps sum w and sum w^2: feasible, returned unchanged with zero multipliers; the result of a
    noisy input satisfies the KKT conditions (P4) and is idempotent."""
    wl = W.make_workload(9, batch=1, nx=8, ny=8, nt=6)
    u0, p = wl.cdata[0].numpy(), wl.params
    ut = wl.u_true[0].numpy()
    assert np.abs(O.residual(wl.kind, ut, u0, p)).max() < 1e-14
    o = O.project(wl.kind, ut, u0, p)
    np.testing.assert_array_equal(o["u"], ut)
    assert np.abs(o["lam"]).max() < 1e-12
    o = O.project(wl.kind, wl.u_hat[0].numpy(), u0, dict(p, hessian=1))
    J = O.jacobian(wl.kind, o["u"], p)
    stat = (o["u"] - wl.u_hat[0].numpy()).ravel() + J.T @ o["lam"]
    assert np.abs(stat).max() <= 1e-11 * max(1.0, np.abs(o["lam"]).max())
    again = O.project(wl.kind, o["u"], u0, p)
    np.testing.assert_allclose(again["u"], o["u"], rtol=0, atol=1e-13)
