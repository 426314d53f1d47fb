"""Oracle: one PCFM sampling step around the projection (§III-A).

TEST INFRASTRUCTURE (see oracle/__init__.py).  For a flow time tau -> tau' the sampler performs, per sample,

    u_hat_1 = u_tau + (1 - tau) v_theta(u_tau, tau)              (Eq. 1: one-step extrapolation to tau = 1)
    u_1     = argmin_u 1/2 ||u - u_hat_1||^2  s.t.  h(u) = 0     (Eq. 2: the projection, oracle/project.py)
    u_tau'  = u_0 + tau' (u_1 - u_0)                             (Eq. 3: optimal-transport interpolant back to tau')

The velocity field v_theta is the pretrained flow model (not in the container); its VALUES are an input
here, exactly as the projection's u_hat is.  The penalised correction of [4] is omitted, as in the paper (L56).
Pins (tests/test_oracle_flow.py): closed forms of Eq. 1 / Eq. 3 on inputs whose projection is known exactly (a velocity that
shoots onto the scheme's own solution; the affine heat kind, pin P1), tau' = 1 returns u_1, linearity in (u_0, u_1).
"""
from __future__ import annotations

import numpy as np

from .project import project


def flow_step(kind: int, u_tau: np.ndarray, vel: np.ndarray, u_prior: np.ndarray, tau: float, tau_next: float,
              u0: np.ndarray, p: dict, backend: str = "auto") -> dict:
    """One sample.  u_tau, vel, u_prior: [nt, ny, nx]; u0: [ny, nx] (the sample's constraint data).
    Returns u_hat (Eq. 1), u1 (Eq. 2), u_next (Eq. 3), lam, iters, status."""
    u_tau = np.asarray(u_tau, dtype=np.float64)
    vel = np.asarray(vel, dtype=np.float64)
    u_prior = np.asarray(u_prior, dtype=np.float64)
    u_hat = u_tau + (1.0 - tau) * vel
    out = project(kind, u_hat, u0, p, backend=backend)
    u1 = out["u"]
    u_next = u_prior + tau_next * (u1 - u_prior)
    return {"u_hat": u_hat, "u1": u1, "u_next": u_next, "lam": out["lam"], "iters": out["iters"], "status": out["status"]}
