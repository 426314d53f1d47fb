"""Oracle: Gauss-Newton / Newton-KKT projection of one sample (and a plain loop over a batch).

TEST INFRASTRUCTURE (see oracle/__init__.py).  Follows SURVEY.md §8(c) "Algorithm, step by
step" in that order and notation:

    u <- u_hat ; mu <- 0
    repeat
       h <- h(u) ; J <- J(u)                       (explicit sparse matrix)
       r <- h - J (u - u_hat)
       lam+ <- solve (J J^T) lam+ = r              (Schur form of Eq. 24 L468 with W = I)
       u_full <- u_hat - J^T lam+ ;  d <- u_full - u
       if ||h||_inf < tol:  polish (R4) and return
       mu <- max(mu, 1e-3, ((u - u_hat)^T d + 1/2 ||d||^2) / ((1 - rho) ||h||_1)),  rho = 1/2
                                                   (mu_rule "nw18_36", default: N&W Eq. 18.36 with sigma = 1,
                                                    Hessian of f = I; ref [15] L275)
         or  mu <- max(mu, 1.1 ||lam+||_inf + 1e-3)     (mu_rule "lam_inf": SURVEY.md §8(c) algorithm listing)
       -- the paper fixes no merit rule (only "filter line search", ref [29] L289); both are textbook choices
          for the l1 exact penalty and tests/test_oracle_pins.py pins that the limit point is the same.
       Armijo back-tracking on phi(v) = 1/2 ||v - u_hat||^2 + mu ||h(v)||_1     (N&W ch. 18, ref [15] L275)
       u <- u + alpha d

Rank-deficient row sets (R6): the solve uses the full-rank row subset (redundant multipliers 0,
"basic solution"); the returned multiplier is the minimum-norm one unless lambda_mode = 1.
"""
from __future__ import annotations

import os
from typing import Optional

import numpy as np

from . import constraints as C
from . import linsolve as L

STATUS_OK = 0
STATUS_MAXITER = -1
STATUS_LINESEARCH = -2
STATUS_NONFINITE = -3
STATUS_PCG = -4

MU_RHO = 0.5               # N&W Eq. 18.36: fraction of the constraint decrease kept in the model
MU_FLOOR = 1e-3
POLISH_SKIP_FACTOR = 1e-3   # skip the polish step when ||h||_inf <= 1e-3 * tol (R4 "adaptive variant")


def _solve_basic(J, w, h, keep, backend, cg_state):
    """lam+ with redundant multipliers pinned to 0 (R6 "basic solution"): the Newton-KKT system
    restricted to the kept rows J_k, i.e. (J_k J_k^T) lam_k = h_k - J_k w with w = u - u_hat."""
    Jk = J[keep] if not keep.all() else J
    if backend == "dense":
        _, lam_k = L.solve_kkt_dense_lu(Jk, w, h[keep])      # full (n+m)x(n+m) KKT matrix, LU
        lam = np.zeros(J.shape[0])
        lam[keep] = lam_k
        return lam
    rk = h[keep] - Jk @ w
    if backend == "banded":
        lam_k = L.solve_schur_banded_cholesky((Jk @ Jk.T).tocsr(), rk)
    elif backend == "dense_chol":
        lam_k = L.solve_schur_dense_cholesky((Jk @ Jk.T).toarray(), rk)
    elif backend == "cg":
        lam_k, its = L.solve_schur_cg((Jk @ Jk.T).tocsr(), rk, rtol=cg_state["rtol"], maxiter=cg_state["maxiter"])
        cg_state["iters"] += its
    else:
        raise ValueError(backend)
    lam = np.zeros(J.shape[0])
    lam[keep] = lam_k
    return lam


def project(kind: int, u_hat: np.ndarray, u0: np.ndarray, p: dict, backend: str = "auto",
            history: Optional[list] = None) -> dict:
    """Project one sample.  u_hat: [nt, ny, nx]; u0: [ny, nx].  Returns a dict with
    u [nt,ny,nx], lam [m], iters (linear solves, or the negative status), status, steps, hinf."""
    u_hat = np.asarray(u_hat, dtype=np.float64)
    u0 = np.asarray(u0, dtype=np.float64)
    nt, ny, nx = u_hat.shape
    if backend == "auto":
        # kind 5: few rows (m ~ (K+1) nx + 2 nt) with dense border rows: dense Cholesky of the assembled J J^T
        backend = {C.ALLENCAHN2D_IE: "cg", C.BURGERS1D_FLUXK: "dense_chol", C.NS2D_VORT_ENST: "banded"}.get(kind, "banded")
    keep = C.full_rank_rows(kind, nx, ny, nt, p)
    tol = p.get("tol", 1e-10)
    max_iter = int(p.get("max_iter", 50))
    polish = int(p.get("polish", 1))
    c1 = p.get("ls_c1", 1e-4)
    shrink = p.get("ls_shrink", 0.5)
    ls_max = int(p.get("ls_max", 20))
    mu_rule = p.get("mu_rule", "nw18_36")
    if mu_rule not in ("nw18_36", "lam_inf"):
        raise ValueError(f"unknown mu_rule {mu_rule!r}")
    # hessian = 1: exact Lagrangian Hessian W = I + sum lam_i grad^2 h_i at the multipliers of the previous solve
    # (Eq. 5 / 25); 0: Gauss-Newton, W = I (R1).  Same KKT points, different rate.
    exact_w = int(p.get("hessian", 0)) == 1
    cg_state = {"rtol": 1e-13, "maxiter": 20000, "iters": 0}
    uh = u_hat.ravel()
    shape = u_hat.shape

    def h_of(v):
        return C.residual(kind, v.reshape(shape), u0, p)

    W_cur = [None]      # Hessian of the last linearisation (exact_w only): for the step and the model term d^T W d

    def lin(v, lam_prev=None):
        h = h_of(v)
        J = C.jacobian(kind, v.reshape(shape), p)
        try:
            with np.errstate(all="ignore"):
                if exact_w:
                    W = C.lagrangian_hessian(kind, v.reshape(shape), lam_prev, p)
                    W_cur[0] = W
                    Jk = J[keep] if not keep.all() else J
                    _, lam_k = L.solve_kkt_sparse_lu(W, Jk, v - uh, h[keep])
                    lam = np.zeros(J.shape[0])
                    lam[keep] = lam_k
                else:
                    lam = _solve_basic(J, v - uh, h, keep, backend, cg_state)
        except (np.linalg.LinAlgError, ValueError, RuntimeError):     # overflowed / singular / non-SPD system (R16)
            lam = np.full(J.shape[0], np.nan)
        return h, J, lam

    def full_step(v, J, lam):
        """u + du of the Newton-KKT step: W du = -(u - u_hat) - J^T lam+   (W = I: u_hat - J^T lam+)."""
        if not exact_w:
            return uh - J.T @ lam
        import scipy.sparse.linalg as spla
        return v - spla.spsolve(W_cur[0].tocsc(), (v - uh) + J.T @ lam)

    u = uh.copy()
    mu = 0.0
    solves = 0
    steps = 0
    backtracks = 0
    status = STATUS_OK
    lam = np.zeros(C.num_rows(kind, nx, ny, nt, p))
    J = None
    while True:
        h, J, lam = lin(u, lam)
        solves += 1
        hinf = float(np.abs(h).max())
        if history is not None:
            history.append(hinf)
        if not (np.isfinite(hinf) and np.all(np.isfinite(lam))):
            status = STATUS_NONFINITE          # R16: leave u* = u_hat
            u = uh.copy()
            lam[:] = 0.0
            break
        u_full = full_step(u, J, lam)
        # Wide J (kind 5): Gauss-Newton with W = I contracts only linearly and ||h|| alone says nothing about
        # stationarity, so convergence also asks for a small step, RMS(d) <= tol (R18).  For the square
        # kinds d = -J^-1 h and the paper's/north_star's rule ||h||_inf < tol stands alone.
        small_step = True
        if kind in (C.BURGERS1D_FLUXK, C.NS2D_VORT_ENST):
            d0 = u_full - u
            small_step = float(d0 @ d0) <= d0.size * tol * tol
        if hinf < tol and small_step:
            if hinf > POLISH_SKIP_FACTOR * tol:
                for _ in range(polish):        # R4: full step(s), then the multiplier at the polished point
                    u = u_full
                    h, J, lam = lin(u, lam)
                    solves += 1
                    u_full = full_step(u, J, lam)
                    hinf = float(np.abs(h).max())
                    if history is not None:
                        history.append(hinf)
            break
        if steps >= max_iter:
            status = STATUS_MAXITER
            break
        if hinf < tol:
            # feasible to tolerance but the step is not small yet (wide J only, R18): full Gauss-Newton steps without
            # a merit test, like polish steps (R4) -- merit differences are below rounding here
            u = u_full
            steps += 1
            continue
        d = u_full - u
        h1 = float(np.abs(h).sum())
        if mu_rule == "nw18_36":
            # penalty parameter from the predicted decrease of the quadratic model (N&W Eq. 18.36, sigma = 1):
            # needs no multiplier, so an implementation may postpone the multiplier solve (R2)
            # (exact Hessian: the model term is d^T W d, N&W Eq. 18.36 with sigma = 1 where it is positive)
            quad = float(d @ (W_cur[0] @ d)) if exact_w else float(d @ d)
            mu = max(mu, MU_FLOOR, (float((u - uh) @ d) + 0.5 * max(quad, 0.0)) / ((1.0 - MU_RHO) * h1))
        else:
            # mu >= 1.1 ||lam+||_inf (+ floor) makes the l1 penalty exact (N&W Thm 17.3)
            mu = max(mu, 1.1 * float(np.abs(lam).max()) + MU_FLOOR)
        phi0 = 0.5 * float((u - uh) @ (u - uh)) + mu * h1
        Dphi = float((u - uh) @ d) - mu * h1
        alpha = 1.0
        tries = 0
        while True:
            ut = u + alpha * d
            ht = h_of(ut)
            phit = 0.5 * float((ut - uh) @ (ut - uh)) + mu * float(np.abs(ht).sum())
            if np.isfinite(phit) and phit <= phi0 + c1 * alpha * Dphi:
                break
            tries += 1
            if tries > ls_max:
                status = STATUS_LINESEARCH
                break
            alpha *= shrink
            backtracks += 1
        if status != STATUS_OK:
            break
        u = ut
        steps += 1

    if status in (STATUS_OK, STATUS_MAXITER, STATUS_LINESEARCH) and int(p.get("lambda_mode", 0)) == 0 \
            and not keep.all():
        lam = L.min_norm_multiplier(J, lam)
    return {"u": u.reshape(shape), "lam": lam, "iters": solves if status == STATUS_OK else status,
            "status": status, "solves": solves, "steps": steps, "hinf": hinf, "cg_iters": cg_state["iters"],
            "backtracks": backtracks}


def _one(args):
    kind, uh, u0, p, backend = args
    try:
        from threadpoolctl import threadpool_limits
        with threadpool_limits(limits=1):
            return project(kind, uh, u0, p, backend)
    except ImportError:
        return project(kind, uh, u0, p, backend)


def project_batch(kind: int, u_hat: np.ndarray, cdata: np.ndarray, p: dict, backend: str = "auto",
                  workers: int = 1) -> dict:
    """Samples are independent blocks: a plain loop (or a process pool of
    `workers`, one BLAS thread each) over `project`.  u_hat: [B, nt, ny, nx], cdata: [B, ny, nx]."""
    u_hat = np.asarray(u_hat, dtype=np.float64)
    cdata = np.asarray(cdata, dtype=np.float64)
    B = u_hat.shape[0]
    jobs = [(kind, u_hat[b], cdata[b], p, backend) for b in range(B)]
    if workers > 1 and B > 1:
        import multiprocessing as mp
        with mp.get_context("fork").Pool(min(workers, B)) as pool:
            outs = pool.map(_one, jobs)
    else:
        outs = [project(*j) for j in jobs]
    return {"u": np.stack([o["u"] for o in outs]), "lam": np.stack([o["lam"] for o in outs]),
            "iters": np.array([o["iters"] for o in outs], dtype=np.int32),
            "solves": np.array([o["solves"] for o in outs], dtype=np.int32),
            "steps": np.array([o["steps"] for o in outs], dtype=np.int32),
            "hinf": np.array([o["hinf"] for o in outs]), "workers": min(max(workers, 1), B),
            "cpu_count": os.cpu_count()}
