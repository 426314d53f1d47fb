"""Pins for the oracle's kind 5, BURGERS1D_FLUXK: the paper's "IC, Mass, Flux(k)"
row set (Eq. 14, Table XVIII) with the energy-evolution row of Eq. 11 (L336, L512-527, L603-607)
and the Godunov flux (L555).  As for the other kinds the oracle is checked against things other than itself: the
paper's min/max definition of the flux by brute force, hand-written scalar formulas, central differences, closed forms
(the affine levels reduce to the heat formula P1; one free level with an energy row is the nearest point on a
sphere-hyperplane intersection), dense LU of the full KKT matrix, and the KKT invariants.  CPU only."""
import math

import numpy as np
import pytest

import oracle as O
import workloads as W
from oracle import constraints as C

K5 = C.BURGERS1D_FLUXK


def _wl(cfg=6, **kw):
    return W.make_workload(cfg, **kw)


def test_godunov_flux_equals_the_papers_min_max_definition():
    """L555: F(a,b) = min_{u in [a,b]} u^2/2 if a <= b, max_{u in [b,a]} u^2/2 otherwise -- brute force on a fine grid."""
    rng = np.random.default_rng(0)
    ab = rng.uniform(-2, 2, size=(400, 2))
    ab = np.vstack([ab, [[0.0, 0.0], [-1.0, 1.0], [1.0, -1.0], [0.5, 0.5], [-0.3, 0.0], [0.0, 0.7]]])
    for a, b in ab:
        grid = np.linspace(min(a, b), max(a, b), 20001)
        f = 0.5 * grid * grid
        want = f.min() if a <= b else f.max()
        assert abs(float(O.godunov_flux(a, b)) - want) <= 1e-8 * max(1.0, want)
    # gradient element vs one-sided differences away from the kinks
    for a, b in ab[:200]:
        fa, fb = 0.5 * max(a, 0) ** 2, 0.5 * min(b, 0) ** 2
        if abs(fa - fb) < 1e-3 or abs(a) < 1e-3 or abs(b) < 1e-3:
            continue
        da, db = O.godunov_flux_grad(a, b)
        e = 1e-6
        assert abs((O.godunov_flux(a + e, b) - O.godunov_flux(a - e, b)) / (2 * e) - da) < 1e-6
        assert abs((O.godunov_flux(a, b + e) - O.godunov_flux(a, b - e)) / (2 * e) - db) < 1e-6


def test_row_counts_and_layout():
    wl = _wl(batch=1, nx=6, nt=7, params=dict(flux_steps=2))
    p = wl.params
    assert O.fluxk_counts(p, wl.nt) == (2, 4, 4)
    assert O.num_rows(K5, 6, 1, 7, p) == 3 * 6 + 4 + 4 == wl.m
    sl = O.row_slices(K5, 6, 1, 7, p)
    assert (sl["ic"], sl["pde"], sl["mass"], sl["energy"]) == (slice(0, 6), slice(6, 18), slice(18, 22), slice(22, 26))
    p2 = dict(p, energy_rows=0)
    assert O.num_rows(K5, 6, 1, 7, p2) == 18 + 4
    assert O.full_rank_rows(K5, 6, 1, 7, p).all()
    J = O.jacobian(K5, wl.u_hat[0].numpy(), p).toarray()
    assert np.linalg.matrix_rank(J) == J.shape[0] < J.shape[1]          # wide, full row rank: no redundant rows
    # the omitted mass rows of levels 0..K really are implied by IC + conservative flux rows (L493 practice)
    u = wl.u_hat[0].numpy()
    h = O.residual(K5, u, wl.cdata[0].numpy(), p)
    dx = p["dx"]
    M0 = dx * wl.cdata[0].numpy().sum()
    for k in range(3):
        implied = dx * h[:(k + 1) * 6].sum()                            # dx (sum IC rows + flux rows of steps < k)
        assert abs((dx * u[k].sum() - M0) - implied) < 1e-13


@pytest.mark.parametrize("flux_kind", [0, 1])
def test_residual_matches_handwritten_scalar_formulas(flux_kind):
    wl = _wl(batch=1, nx=7, nt=6, params=dict(flux_steps=2, flux_kind=flux_kind))
    p = wl.params
    u, u0 = wl.u_hat[0].numpy(), wl.cdata[0].numpy()
    nx, nt, K = 7, 6, 2
    dx, dt, nu, al = p["dx"], p["dt"], p["nu"], p["alpha"]
    h = O.residual(K5, u, u0, p)

    def flux(a, b):
        if flux_kind == 0:
            return 0.5 * (0.5 * a * a + 0.5 * b * b) - 0.5 * al * (b - a)
        lo, hi = min(a, b), max(a, b)
        if a <= b:
            return 0.0 if lo <= 0.0 <= hi else 0.5 * min(lo * lo, hi * hi)
        return 0.5 * max(lo * lo, hi * hi)

    for i in range(nx):
        assert h[i] == u[0, 0, i] - u0[0, i]
    for k in range(K):
        v = u[k, 0]
        for i in range(nx):
            Fr, Fl = flux(v[i], v[(i + 1) % nx]), flux(v[i - 1], v[i])
            want = u[k + 1, 0, i] - (v[i] - dt / dx * (Fr - Fl)) - nu * dt / dx ** 2 * (v[(i + 1) % nx] - 2 * v[i] + v[i - 1])
            assert abs(h[(k + 1) * nx + i] - want) < 1e-14
    loc = (K + 1) * nx
    F = nt - 1 - K
    M0 = dx * math.fsum(u0[0])
    for f in range(F):
        assert abs(h[loc + f] - (dx * math.fsum(u[K + 1 + f, 0]) - M0)) < 1e-14
    for f in range(F):
        k = K + f
        v, w = u[k, 0], u[k + 1, 0]
        E1, E0 = 0.5 * dx * sum(x * x for x in w), 0.5 * dx * sum(x * x for x in v)
        D0 = dx * sum(((v[(i + 1) % nx] - v[i]) / dx) ** 2 for i in range(nx))
        assert abs(h[loc + F + f] - (E1 - E0 + dt * nu * D0)) < 1e-13


@pytest.mark.parametrize("flux_kind,energy", [(0, 1), (0, 0), (1, 0), (1, 1)])
def test_p5_jacobian_vs_central_differences(flux_kind, energy):
    wl = _wl(batch=1, nx=6, nt=5, params=dict(flux_steps=2, flux_kind=flux_kind, energy_rows=energy))
    p = wl.params
    u, u0 = wl.u_hat[0].numpy(), wl.cdata[0].numpy()
    J = O.jacobian(K5, u, p).toarray()
    e = 1e-6
    Jfd = np.zeros_like(J)
    for c in range(u.size):
        d = np.zeros(u.size)
        d[c] = e
        Jfd[:, c] = (O.residual(K5, (u.ravel() + d).reshape(u.shape), u0, p)
                     - O.residual(K5, (u.ravel() - d).reshape(u.shape), u0, p)) / (2 * e)
    assert np.abs(J - Jfd).max() < 1e-8      # generic random u: no cell sits on a kink of the Godunov flux


def test_p1_without_energy_rows_the_free_levels_have_the_heat_closed_form():
    """energy_rows = 0 is exactly Eq. 14: levels 0..K are the scheme's forward solution (P2), every later level
    carries one mass row and projects like the heat kind: u*[k] = u_hat[k] - mean + M0/(nx dx), lam = P1's."""
    for flux_kind in (0, 1):
        wl = _wl(batch=2, nx=16, nt=12, params=dict(flux_steps=3, energy_rows=0, flux_kind=flux_kind))
        p = wl.params
        K, dx, nx = 3, p["dx"], 16
        for b in range(2):
            uh, u0 = wl.u_hat[b].numpy(), wl.cdata[b].numpy()
            o = O.project(K5, uh, u0, p)
            assert o["status"] == 0
            np.testing.assert_allclose(o["u"][:K + 1], wl.u_true[b].numpy()[:K + 1], rtol=0, atol=1e-12)
            M0 = dx * u0.sum()
            for k in range(K + 1, 12):
                want = uh[k, 0] - uh[k, 0].mean() + M0 / (nx * dx)
                np.testing.assert_allclose(o["u"][k, 0], want, rtol=0, atol=1e-13)
                lam_k = (dx * uh[k, 0].sum() - M0) / (nx * dx * dx)
                assert abs(o["lam"][(K + 1) * nx + (k - K - 1)] - lam_k) < 1e-12
            # the result depends on u_hat (unlike the square kinds 1-4, R5)
            o2 = O.project(K5, uh + 0.01 * np.cos(np.arange(uh.size)).reshape(uh.shape), u0, p)
            assert np.abs(o2["u"][K + 1:] - o["u"][K + 1:]).max() > 1e-3
            np.testing.assert_allclose(o2["u"][:K + 1], o["u"][:K + 1], rtol=0, atol=1e-12)


def test_one_free_level_with_an_energy_row_is_the_nearest_point_on_a_sphere_hyperplane_intersection():
    """nt = K + 2: the only free level v = u[K+1] must satisfy  dx sum v = M0  and  1/2 dx |v|^2 = E*  with
    E* = E(u[K]) - dt nu D(u[K]) fixed by the pinned levels.  Nearest point to w = u_hat[K+1]:
    v = mbar 1 + r (w - mean(w)) / |w - mean(w)|,  mbar = M0/(nx dx),  r^2 = 2 E*/dx - nx mbar^2."""
    wl = _wl(batch=3, nx=12, nt=5, params=dict(flux_steps=3, energy_rows=1))
    p = wl.params
    dx, dt, nu, nx, K = p["dx"], p["dt"], p["nu"], 12, 3
    for b in range(3):
        uh, u0 = wl.u_hat[b].numpy(), wl.cdata[b].numpy()
        o = O.project(K5, uh, u0, p)
        assert o["status"] == 0
        uK = wl.u_true[b].numpy()[K, 0]
        np.testing.assert_allclose(o["u"][K, 0], uK, rtol=0, atol=1e-12)
        Estar = 0.5 * dx * (uK ** 2).sum() - dt * nu * ((np.roll(uK, -1) - uK) ** 2).sum() / dx
        mbar = dx * u0.sum() / (nx * dx)
        w = uh[K + 1, 0]
        dev = w - w.mean()
        r = math.sqrt(2.0 * Estar / dx - nx * mbar ** 2)
        want = mbar + r * dev / np.linalg.norm(dev)
        np.testing.assert_allclose(o["u"][K + 1, 0], want, rtol=0, atol=1e-11)


@pytest.mark.parametrize("flux_kind,energy", [(0, 1), (1, 0), (0, 0)])
def test_p3_one_gauss_newton_step_equals_dense_lu_of_the_full_kkt_matrix(flux_kind, energy):
    wl = _wl(batch=1, nx=4, nt=4, params=dict(flux_steps=1, flux_kind=flux_kind, energy_rows=energy))
    p = wl.params
    uh, u0 = wl.u_hat[0].numpy(), wl.cdata[0].numpy()
    rng = np.random.default_rng(5)
    u = uh + 0.1 * rng.standard_normal(uh.shape)            # a point with u != u_hat
    J = O.jacobian(K5, u, p)
    h = O.residual(K5, u, u0, p)
    w = (u - uh).ravel()
    d, lam = O.solve_kkt_dense_lu(J, w, h)
    Jd = J.toarray()
    lam_s = O.solve_schur_dense_cholesky(Jd @ Jd.T, h - Jd @ w)
    np.testing.assert_allclose(lam, lam_s, rtol=0, atol=1e-11 * max(1, np.abs(lam).max()))
    np.testing.assert_allclose(u.ravel() + d, uh.ravel() - Jd.T @ lam_s, rtol=0, atol=1e-12)
    # the oracle's own iteration takes that step first: its history starts at ||h(u_hat)||_inf
    hist = []
    O.project(K5, uh, u0, p, history=hist)
    assert hist[0] == np.abs(O.residual(K5, uh, u0, p)).max()


@pytest.mark.parametrize("cfg,kw", [(6, dict(batch=2, nx=24, nt=20)), (7, dict(batch=2, nx=24, nt=20)),
                                    (6, dict(batch=1, nx=32, nt=12, params=dict(flux_steps=0))),
                                    (6, dict(batch=1, nx=16, nt=9, params=dict(flux_steps=8)))])
def test_p4_kkt_invariants_and_dependence_on_the_input(cfg, kw):
    wl = _wl(cfg, **kw)
    p = wl.params
    for b in range(wl.batch):
        uh, u0 = wl.u_hat[b].numpy(), wl.cdata[b].numpy()
        o = O.project(K5, uh, u0, p)
        assert o["status"] == 0
        assert np.abs(O.residual(K5, o["u"], u0, p)).max() < 1e-12
        J = O.jacobian(K5, o["u"], p)
        stat = (o["u"] - uh).ravel() + J.T @ o["lam"]
        # wide J, W = I: stationarity is first order in the last step, |stat| <~ |lam| |grad^2 h| |d_last|, and the stop
        # rule bounds only ||h||_inf (< 1e-10, then one polish step) -- hence 1e-10 here against P4's 1e-11
        assert np.abs(stat).max() < 1e-10 * max(1.0, np.abs(o["lam"]).max())
        K = int(p["flux_steps"])
        np.testing.assert_allclose(o["u"][:K + 1], wl.u_true[b].numpy()[:K + 1], rtol=0, atol=1e-11)   # P2 on pinned levels
        again = O.project(K5, o["u"], u0, p)                          # P7 idempotence
        assert again["steps"] == 0
        np.testing.assert_array_equal(again["u"], o["u"])


def test_gauss_newton_converges_linearly_with_energy_rows_and_the_line_search_is_live():
    """With W = I and non-linear border rows on a wide J the contraction is linear, visibly so on
    a far input; both penalty rules reach the same point (R2)."""
    wl = _wl(batch=1, nx=24, nt=12, noise=1.0)
    uh, u0 = wl.u_hat[0].numpy(), wl.cdata[0].numpy()
    hist = []
    a = O.project(K5, uh, u0, dict(wl.params, max_iter=400), history=hist)   # contraction ~0.93 per step this far out
    assert a["status"] == 0 and len(hist) >= 50
    # linear, not quadratic: feasibility arrives early (h -> rounding) but the tangential step shrinks by a constant
    # factor per solve, so stationarity takes > 50 solves here where Newton would need a handful
    J = O.jacobian(K5, a["u"], wl.params)
    stat = (a["u"] - uh).ravel() + J.T @ a["lam"]
    assert np.abs(stat).max() < 1e-9 * max(1.0, np.abs(a["lam"]).max())    # the step criterion (R18) bounds stationarity
    assert a["backtracks"] > 0                    # and the Armijo test rejects full steps on the way
    # (this far out the lam_inf rule takes > 50 un-damped steps at contraction ~0.93: the regime NEXT-2's exact W is for)
    wl = _wl(batch=1, nx=24, nt=12, noise=0.3)
    uh, u0 = wl.u_hat[0].numpy(), wl.cdata[0].numpy()
    a = O.project(K5, uh, u0, wl.params)
    b = O.project(K5, uh, u0, dict(wl.params, mu_rule="lam_inf"))
    assert a["status"] == 0 and b["status"] == 0
    np.testing.assert_allclose(a["u"], b["u"], rtol=0, atol=1e-11)


def test_p7_shift_equivariance():
    wl = _wl(batch=1, nx=16, nt=10)
    uh, u0 = wl.u_hat[0].numpy(), wl.cdata[0].numpy()
    a = O.project(K5, uh, u0, wl.params)
    b = O.project(K5, np.roll(uh, 3, -1), np.roll(u0, 3, -1), wl.params)
    np.testing.assert_allclose(np.roll(a["u"], 3, -1), b["u"], rtol=0, atol=1e-12)
    sl = O.row_slices(K5, 16, 1, 10, wl.params)
    np.testing.assert_allclose(a["lam"][sl["mass"]], b["lam"][sl["mass"]], rtol=0, atol=1e-10)
    np.testing.assert_allclose(a["lam"][sl["energy"]], b["lam"][sl["energy"]], rtol=0, atol=1e-10)
