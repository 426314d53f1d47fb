"""Pins of the oracle's PCFM step (oracle/flow.py; Eq. 1-3) -- all CPU, `-m "not gpu"`."""
import numpy as np
import torch

import oracle as O
import workloads as W


def _prior(wl, seed):
    g = torch.Generator().manual_seed(seed)
    return torch.randn(wl.u_hat.shape, generator=g, dtype=torch.float64)


def test_shooting_onto_the_schemes_solution_gives_the_closed_form():
    """v = (u_true - u_tau) / (1 - tau) shoots exactly onto the feasible point (P2: u_true is the unique feasible point of
    the square kinds), so Eq. 2 returns it and Eq. 3 is the straight line from the prior sample: nothing of the
    projection's arithmetic is needed to state the expected result."""
    for cfg, kw in ((2, dict(batch=2, nx=24, nt=10)), (3, dict(batch=2, nx=16, nt=8)), (4, dict(batch=1, nx=8, ny=8, nt=4))):
        wl = W.make_workload(cfg, **kw)
        u_true = wl.u_true.numpy().reshape(wl.u_hat.shape)
        u0p = _prior(wl, 11).numpy()
        for tau, taun in ((0.0, 0.1), (0.3, 0.5), (0.9, 1.0)):
            u_tau = u0p + tau * (u_true - u0p)                       # on the OT line
            vel = (u_true - u_tau) / (1.0 - tau)
            for b in range(wl.batch):
                o = O.flow_step(wl.kind, u_tau[b], vel[b], u0p[b], tau, taun, wl.cdata[b].numpy(), wl.params)
                assert o["status"] == 0
                np.testing.assert_allclose(o["u_hat"], u_true[b], rtol=0, atol=1e-13)
                np.testing.assert_allclose(o["u1"], u_true[b], rtol=0, atol=1e-11)
                np.testing.assert_allclose(o["u_next"], u0p[b] + taun * (u_true[b] - u0p[b]), rtol=0, atol=1e-11)


def test_heat_step_matches_the_closed_form_projection():
    """Affine constraints (kind 0): Eq. 2 has the closed form P1, so the whole step is closed form."""
    wl = W.make_workload(1, batch=2, nx=12, nt=7)
    p = wl.params
    g = torch.Generator().manual_seed(5)
    vel = torch.randn(wl.u_hat.shape, generator=g, dtype=torch.float64).numpy()
    u0p = _prior(wl, 6).numpy()
    u_tau = wl.u_hat.numpy()
    tau, taun = 0.25, 0.5
    nx, dx = wl.nx, p["dx"]
    for b in range(wl.batch):
        u0 = wl.cdata[b].numpy()
        o = O.flow_step(wl.kind, u_tau[b], vel[b], u0p[b], tau, taun, u0, p)
        uh = u_tau[b] + 0.75 * vel[b]
        M0 = dx * u0.sum()
        u1 = uh - uh.mean(axis=2, keepdims=True) + M0 / (nx * dx)     # P1: levels k >= 1
        u1[0] = u0                                                    # level 0 = the IC
        np.testing.assert_allclose(o["u1"], u1, rtol=0, atol=1e-12)
        np.testing.assert_allclose(o["u_next"], u0p[b] + taun * (u1 - u0p[b]), rtol=0, atol=1e-12)


def test_interpolant_end_points_and_linearity():
    wl = W.make_workload(5, batch=1, nx=16, nt=8)
    g = torch.Generator().manual_seed(3)
    vel = 0.1 * torch.randn(wl.u_hat.shape, generator=g, dtype=torch.float64).numpy()[0]
    u0p = _prior(wl, 4).numpy()[0]
    u_tau, u0 = wl.u_hat.numpy()[0], wl.cdata[0].numpy()
    a = O.flow_step(wl.kind, u_tau, vel, u0p, 0.4, 1.0, u0, wl.params)
    np.testing.assert_array_equal(a["u_next"], u0p + 1.0 * (a["u1"] - u0p))
    np.testing.assert_allclose(a["u_next"], a["u1"], rtol=0, atol=1e-15)          # tau' = 1: the sample itself
    b = O.flow_step(wl.kind, u_tau, vel, u0p, 0.4, 0.0, u0, wl.params)
    np.testing.assert_array_equal(b["u_next"], u0p)                                # tau' = 0: the prior sample
    c = O.flow_step(wl.kind, u_tau, vel, u0p, 0.4, 0.5, u0, wl.params)
    np.testing.assert_allclose(c["u_next"], 0.5 * (a["u_next"] + b["u_next"]), rtol=0, atol=1e-15)
    np.testing.assert_array_equal(a["u1"], c["u1"])                                # the projection does not see tau'
    # Eq. 1 at tau = 1 leaves the state untouched
    d = O.flow_step(wl.kind, u_tau, vel, u0p, 1.0, 1.0, u0, wl.params)
    np.testing.assert_array_equal(d["u_hat"], u_tau)
