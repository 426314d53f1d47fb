"""Oracle: constraint residual h(u) and explicit sparse Jacobian J(u) per kind.

TEST INFRASTRUCTURE (see oracle/__init__.py).  fp64, numpy/scipy, no blocking or fusion.

Layout (time-major, x fastest).  One sample:
    u[k][j][i],  k = 0..nt-1 (time), j = 0..ny-1, i = 0..nx-1;  unknown index (k*ny + j)*nx + i.
Constraint rows (the lambda layout of include/snap.h):
    local block  [nt][ny][nx] : level 0 = initial-condition rows u[0] - u0   (Eq. 10, Eq. 14)
                                level k>=1 = one-step scheme residual between levels k-1 and k (L549, L561)
                  (kind HEAT1D_IC_MASS has only level 0: nx rows)
    mass block   [nt]         : dx * sum_i u[k][i] - M0,  M0 = dx * sum_i u0[i]   (L573-575; kinds 0 and 4)
The paper orders IC, mass, then flux rows (L374, L499); the order of rows does not change
the projection, only the order of the multipliers.
"""
from __future__ import annotations

import math

import numpy as np
import scipy.sparse as sp

HEAT1D_IC_MASS = 0
BURGERS1D_LF = 1
FISHER1D_IE = 2
ALLENCAHN2D_IE = 3
BURGERS1D_LF_MASS = 4
BURGERS1D_FLUXK = 5
NS2D_VORT_ENST = 6

_HAS_MASS = (HEAT1D_IC_MASS, BURGERS1D_LF_MASS)

# Kind 5, BURGERS1D_FLUXK — the paper's own Burgers constraint set "IC, Mass, Flux(k)" (Eq. 14,
# Table XVIII) with the energy-evolution row of Eq. 11 (L336, Appendix D) as an option:
#   local block  [K+1][nx] : level 0 = IC rows; level k = 1..K = one-step finite-volume residual of step k-1 -> k
#                            (L549, L561), K = p["flux_steps"]; numerical flux p["flux_kind"]: 0 Lax-Friedrichs (as
#                            kinds 1, 4), 1 Godunov (L555, non-smooth: an element of the generalised Jacobian is used)
#   mass block   [F]       : levels k = K+1..nt-1 (F = nt-1-K):  dx sum_i u[k][i] - M0   (L573-575).  The rows of
#                            levels 0..K are implied by IC + conservative periodic flux rows and are OMITTED, as the
#                            paper omits its implied first row ("the constraint at the first timestep is omitted", L493)
#   energy block [F]       : steps k = K..nt-2, only if p["energy_rows"]:
#                            E(u[k+1]) - E(u[k]) + dt nu D(u[k]),   E(v) = 1/2 dx sum_i v_i^2   (Eq. 7),
#                            D(v) = dx sum_i ((v_{i+1} - v_i)/dx)^2 (periodic)  — Eq. 11's  d/dt 1/2 int u^2 + alpha int u_x^2
#                            discretised as L603-607 (Riemann sums, forward difference in time, un-divided by dt like
#                            the other rows, R11), dissipation explicit at level k (R8), alpha = nu.
# Levels 0..K are pinned by square local rows (unique, as kinds 1/4); levels K+1.. are free up to 1-2 global rows
# each, so J is wide, u* depends on u_hat, and with energy rows the border Schur complement is a banded SPD matrix
# (each energy row couples two consecutive levels) and Gauss-Newton with W = I converges only linearly.


# Kind 6, NS2D_VORT_ENST — the paper's Navier-Stokes constraint set (Eq. 20; Table row "IC | Mass | Enstrophy" L684):
#   IC block        [ny][nx] : w[0] - w_IC
#   vorticity block [nt-1]   : dx dy sum w[k] - dx dy sum w_IC            (total vorticity, "vorticity-mass", k = 1..nt-1)
#   enstrophy block [nt-1]   : dx dy sum w[k]^2 - dx dy sum w_IC^2        (Eq. 20 as printed: no factor 1/2)
# Riemann sums over all nodes (R7); the rows of level 0 are implied by the IC rows and omitted as the paper omits its
# implied first row (L493).  No local PDE rows: every level k >= 1 is constrained only by its two global rows, so the
# levels decouple and the projection of one level is the projection onto a sphere inside a hyperplane:
#     w* = m + (r / ||dev||) dev ,  m = mean(w_IC), r = ||w_IC - m||_2, dev = w_hat - mean(w_hat)
# (tests/test_oracle_ns.py pins the generic Newton-KKT route against this closed form).


def fluxk_counts(p: dict, nt: int):
    """(K, F, E): flux steps, free levels, energy rows of kind 5."""
    K = int(p.get("flux_steps", 0))
    if not 0 <= K <= nt - 1:
        raise ValueError(f"flux_steps {K} outside [0, nt-1]")
    F = nt - 1 - K
    return K, F, (F if int(p.get("energy_rows", 0)) else 0)


def num_rows(kind: int, nx: int, ny: int, nt: int, p: dict = None) -> int:
    if kind == HEAT1D_IC_MASS:
        return nx + nt
    if kind == BURGERS1D_FLUXK:
        K, F, E = fluxk_counts(p, nt)
        return (K + 1) * nx + F + E
    if kind == NS2D_VORT_ENST:
        return nx * ny + 2 * (nt - 1)
    n = nx * ny * nt
    return n + nt if kind == BURGERS1D_LF_MASS else n


def row_slices(kind: int, nx: int, ny: int, nt: int, p: dict = None):
    """{'ic': slice, 'pde': slice, 'mass': slice[, 'energy': slice]} into the row vector (empty where absent)."""
    lvl = nx * ny
    if kind == HEAT1D_IC_MASS:
        return {"ic": slice(0, nx), "pde": slice(nx, nx), "mass": slice(nx, nx + nt)}
    if kind == BURGERS1D_FLUXK:
        K, F, E = fluxk_counts(p, nt)
        loc = (K + 1) * nx
        return {"ic": slice(0, nx), "pde": slice(nx, loc), "mass": slice(loc, loc + F), "energy": slice(loc + F, loc + F + E)}
    if kind == NS2D_VORT_ENST:       # "mass" = total-vorticity rows, "energy" = enstrophy rows
        return {"ic": slice(0, lvl), "pde": slice(lvl, lvl), "mass": slice(lvl, lvl + nt - 1),
                "energy": slice(lvl + nt - 1, lvl + 2 * (nt - 1))}
    n = lvl * nt
    mass = slice(n, n + nt) if kind == BURGERS1D_LF_MASS else slice(n, n)
    return {"ic": slice(0, lvl), "pde": slice(lvl, n), "mass": mass}


def full_rank_rows(kind: int, nx: int, ny: int, nt: int, p: dict = None) -> np.ndarray:
    """Boolean mask of a maximal linearly independent row subset.

    kind 0: the t=0 mass row is implied by the nx IC rows (the paper omits it, L493).
    kind 4: every mass row is implied by IC + conservative periodic finite-volume rows
            (sum_i h^P_{k,i} dx = mass_{k+1} - mass_k identically).
    tests/test_oracle_pins.py verifies both statements by numerical rank on tiny grids."""
    m = num_rows(kind, nx, ny, nt, p)
    keep = np.ones(m, dtype=bool)
    if kind in (BURGERS1D_FLUXK, NS2D_VORT_ENST):
        return keep                      # implied rows are not part of these kinds' row sets
    s = row_slices(kind, nx, ny, nt)["mass"]
    if kind == HEAT1D_IC_MASS:
        keep[s.start] = False
    elif kind == BURGERS1D_LF_MASS:
        keep[s] = False
    return keep


# ------------------------------------------------------------------------------------------
# residual
# ------------------------------------------------------------------------------------------

def _lf_flux(a, b, alpha):
    """Lax-Friedrichs numerical flux for f(u) = u^2/2 through the interface between
    a = u_i and b = u_{i+1} (smooth stand-in for the Godunov flux of L555)."""
    return 0.5 * (0.5 * a * a + 0.5 * b * b) - 0.5 * alpha * (b - a)


def godunov_flux(a, b):
    """Godunov numerical flux for f(u) = u^2/2: min of f over [a, b] if a <= b, max over [b, a]
    otherwise.  For this convex f both cases equal  max(f(max(a, 0)), f(min(b, 0)))  (the textbook closed form;
    tests/test_oracle_pins.py checks it against the min/max definition by brute force)."""
    return np.maximum(0.5 * np.maximum(a, 0.0) ** 2, 0.5 * np.minimum(b, 0.0) ** 2)


def godunov_flux_grad(a, b):
    """(dF/da, dF/db): an element of the generalised Jacobian of the piecewise-smooth flux; where the two
    branches tie (incl. a <= 0 <= b, F = 0) the first branch is taken: dF/da = max(a, 0), dF/db = 0."""
    fa, fb = 0.5 * np.maximum(a, 0.0) ** 2, 0.5 * np.minimum(b, 0.0) ** 2
    first = fa >= fb
    return np.where(first, np.maximum(a, 0.0), 0.0), np.where(first, 0.0, np.minimum(b, 0.0))


def _fv_step_residual(v, w, p):
    """One conservative finite-volume update residual  w - [v - dt/dx (F_{i+1/2} - F_{i-1/2})] - viscous term
    (L561; R8) between consecutive levels v = u[k], w = u[k+1]; periodic."""
    dx, dt = p["dx"], p["dt"]
    s = dt / dx
    c = p["nu"] * dt / dx ** 2
    vp, vm = np.roll(v, -1), np.roll(v, 1)
    if int(p.get("flux_kind", 0)) == 1:
        F_r, F_l = godunov_flux(v, vp), godunov_flux(vm, v)
    else:
        F_r, F_l = _lf_flux(v, vp, p["alpha"]), _lf_flux(vm, v, p["alpha"])
    return w - v + s * (F_r - F_l) - c * (vp - 2.0 * v + vm)


def _energy(v, dx):
    return 0.5 * dx * math.fsum((v * v).tolist())


def _dissipation(v, dx):
    d = np.roll(v, -1) - v
    return math.fsum((d * d).tolist()) / dx


def _mass_rows(u, u0, dx):
    nt = u.shape[0]
    M0 = dx * math.fsum(u0.ravel().tolist())
    return np.array([dx * math.fsum(u[k].ravel().tolist()) - M0 for k in range(nt)])


def residual(kind: int, u: np.ndarray, u0: np.ndarray, p: dict) -> np.ndarray:
    """h(u) as one vector in the row layout above.  u: [nt, ny, nx], u0: [ny, nx]."""
    u = np.asarray(u, dtype=np.float64)
    u0 = np.asarray(u0, dtype=np.float64)
    nt, ny, nx = u.shape
    dx, dt = p["dx"], p["dt"]
    ic = (u[0] - u0).ravel()
    if kind == HEAT1D_IC_MASS:
        return np.concatenate([ic, _mass_rows(u, u0, dx)])
    if kind == NS2D_VORT_ENST:
        a = dx * p["dy"]
        s1, s2 = math.fsum(u0.ravel().tolist()), math.fsum((u0 * u0).ravel().tolist())
        vort = [a * (math.fsum(u[k].ravel().tolist()) - s1) for k in range(1, nt)]
        enst = [a * (math.fsum((u[k] * u[k]).ravel().tolist()) - s2) for k in range(1, nt)]
        return np.concatenate([ic, np.array(vort, dtype=np.float64), np.array(enst, dtype=np.float64)])
    if kind == BURGERS1D_FLUXK:
        K, F, E = fluxk_counts(p, nt)
        loc = [ic] + [_fv_step_residual(u[k, 0], u[k + 1, 0], p) for k in range(K)]
        mass = _mass_rows(u, u0, dx)[K + 1:]
        en = [_energy(u[k + 1, 0], dx) - _energy(u[k, 0], dx) + dt * p["nu"] * _dissipation(u[k, 0], dx)
              for k in range(K, nt - 1)] if E else []
        return np.concatenate(loc + [mass, np.array(en, dtype=np.float64)])

    loc = np.empty_like(u)
    loc[0] = u[0] - u0
    if kind in (BURGERS1D_LF, BURGERS1D_LF_MASS):
        s = dt / dx
        c = p["nu"] * dt / dx ** 2
        al = p["alpha"]
        for k in range(nt - 1):
            v = u[k, 0]
            vp = np.roll(v, -1)       # u_{i+1}
            vm = np.roll(v, 1)        # u_{i-1}
            F_r = _lf_flux(v, vp, al)     # F_{i+1/2}
            F_l = _lf_flux(vm, v, al)     # F_{i-1/2}
            # R^(k) = u^{k+1} - [u^k - dt/dx (F_{i+1/2} - F_{i-1/2})]  (L561) with explicit viscosity (R8)
            loc[k + 1, 0] = u[k + 1, 0] - v + s * (F_r - F_l) - c * (vp - 2.0 * v + vm)
    elif kind == FISHER1D_IE:
        D, rho = p["D"], p["rho"]
        for k in range(nt - 1):
            w = u[k + 1, 0]
            lap = np.empty(nx)
            lap[1:-1] = (w[2:] - 2.0 * w[1:-1] + w[:-2]) / dx ** 2
            lap[0] = (w[1] - w[0]) / dx ** 2            # ghost-cell Neumann (R10, L577-587)
            lap[-1] = (w[-2] - w[-1]) / dx ** 2
            loc[k + 1, 0] = w - u[k, 0] - dt * (D * lap + rho * w * (1.0 - w))
    elif kind == ALLENCAHN2D_IE:
        dy, eps = p["dy"], p["eps"]
        for k in range(nt - 1):
            w = u[k + 1]
            lap = ((np.roll(w, -1, 1) - 2.0 * w + np.roll(w, 1, 1)) / dx ** 2
                   + (np.roll(w, -1, 0) - 2.0 * w + np.roll(w, 1, 0)) / dy ** 2)
            loc[k + 1] = w - u[k] - dt * (eps ** 2 * lap - w ** 3 + w)
    else:
        raise ValueError(f"unknown kind {kind}")
    if kind == BURGERS1D_LF_MASS:
        return np.concatenate([loc.ravel(), _mass_rows(u, u0, dx)])
    return loc.ravel()


def residual_norms(kind: int, u: np.ndarray, u0: np.ndarray, p: dict) -> np.ndarray:
    """[ ||h||_inf, ||h_IC||_2, ||h_PDE||_2, ||h_mass||_2 ]  — the per-type Euclidean norms
    are the per-sample terms of the paper's constraint-error metric (Eq. 27)."""
    nt, ny, nx = np.asarray(u).shape
    h = residual(kind, u, u0, p)
    sl = row_slices(kind, nx, ny, nt, p)
    out = [np.abs(h).max() if h.size else 0.0,
           np.linalg.norm(h[sl["ic"]]), np.linalg.norm(h[sl["pde"]]), np.linalg.norm(h[sl["mass"]])]
    if "energy" in sl:
        out.append(np.linalg.norm(h[sl["energy"]]))
    return np.array(out)


# ------------------------------------------------------------------------------------------
# Jacobian (explicit sparse matrix; fixed pattern)
# ------------------------------------------------------------------------------------------

def jacobian(kind: int, u: np.ndarray, p: dict) -> sp.csr_matrix:
    """J(u) = dh/du as an explicit CSR matrix, rows in the layout above."""
    u = np.asarray(u, dtype=np.float64)
    nt, ny, nx = u.shape
    lvl = nx * ny
    n = lvl * nt
    m = num_rows(kind, nx, ny, nt, p)
    dx, dt = p["dx"], p["dt"]
    rows, cols, vals = [], [], []

    def add(r, c, v):
        rows.append(np.asarray(r).ravel())
        cols.append(np.asarray(c).ravel())
        vals.append(np.broadcast_to(np.asarray(v, dtype=np.float64), np.asarray(r).shape).ravel())

    cell = np.arange(lvl)
    add(cell, cell, 1.0)                                 # IC rows: d(u[0]-u0)/du[0] = I

    if kind in (BURGERS1D_LF, BURGERS1D_LF_MASS, BURGERS1D_FLUXK):
        s = dt / dx
        c = p["nu"] * dt / dx ** 2
        al = p["alpha"]
        i = np.arange(nx)
        ip = (i + 1) % nx
        im = (i - 1) % nx
        godunov = kind == BURGERS1D_FLUXK and int(p.get("flux_kind", 0)) == 1
        steps = fluxk_counts(p, nt)[0] if kind == BURGERS1D_FLUXK else nt - 1
        for k in range(steps):
            v = u[k, 0]
            r = (k + 1) * nx + i
            if godunov:
                dFr_di, dFr_dip = godunov_flux_grad(v[i], v[ip])
                dFl_dim, dFl_di = godunov_flux_grad(v[im], v[i])
            else:
                # dF_{i+1/2}/du_i = u_i/2 + alpha/2 ; dF_{i+1/2}/du_{i+1} = u_{i+1}/2 - alpha/2
                dFr_di, dFr_dip = 0.5 * v[i] + 0.5 * al, 0.5 * v[ip] - 0.5 * al
                dFl_dim, dFl_di = 0.5 * v[im] + 0.5 * al, 0.5 * v[i] - 0.5 * al
            add(r, (k + 1) * nx + i, 1.0)
            add(r, k * nx + i, -1.0 + s * (dFr_di - dFl_di) + 2.0 * c)
            add(r, k * nx + ip, s * dFr_dip - c)
            add(r, k * nx + im, -s * dFl_dim - c)
    elif kind == FISHER1D_IE:
        D, rho = p["D"], p["rho"]
        a = dt * D / dx ** 2
        i = np.arange(nx)
        for k in range(nt - 1):
            w = u[k + 1, 0]
            r = (k + 1) * nx + i
            nnb = np.full(nx, 2.0)
            nnb[0] = 1.0
            nnb[-1] = 1.0                                  # number of neighbours (Neumann ends)
            add(r, k * nx + i, -1.0)
            add(r, (k + 1) * nx + i, 1.0 + a * nnb - dt * rho * (1.0 - 2.0 * w))
            add(r[1:], (k + 1) * nx + i[:-1], -a)
            add(r[:-1], (k + 1) * nx + i[1:], -a)
    elif kind == ALLENCAHN2D_IE:
        dy, eps = p["dy"], p["eps"]
        ax = dt * eps ** 2 / dx ** 2
        ay = dt * eps ** 2 / dy ** 2
        jj, ii = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
        here = (jj * nx + ii).ravel()
        xp = (jj * nx + (ii + 1) % nx).ravel()
        xm = (jj * nx + (ii - 1) % nx).ravel()
        yp = (((jj + 1) % ny) * nx + ii).ravel()
        ym = (((jj - 1) % ny) * nx + ii).ravel()
        for k in range(nt - 1):
            w = u[k + 1].ravel()
            r = (k + 1) * lvl + here
            base = (k + 1) * lvl
            add(r, k * lvl + here, -1.0)
            add(r, base + here, 1.0 + 2.0 * ax + 2.0 * ay + dt * (3.0 * w * w - 1.0))
            add(r, base + xp, -ax)
            add(r, base + xm, -ax)
            add(r, base + yp, -ay)
            add(r, base + ym, -ay)
    elif kind == NS2D_VORT_ENST:
        a = dx * p["dy"]
        for k in range(1, nt):
            add(np.full(lvl, lvl + (k - 1)), k * lvl + cell, a)                          # total vorticity: a 1
            add(np.full(lvl, lvl + (nt - 1) + (k - 1)), k * lvl + cell, 2.0 * a * u[k].ravel())   # enstrophy: 2 a w
    elif kind != HEAT1D_IC_MASS:
        raise ValueError(f"unknown kind {kind}")

    if kind == BURGERS1D_FLUXK:
        K, F, E = fluxk_counts(p, nt)
        i = np.arange(nx)
        ip, im = (i + 1) % nx, (i - 1) % nx
        m0 = (K + 1) * nx
        for f in range(F):                                   # mass rows of the free levels k = K+1..nt-1
            add(np.full(nx, m0 + f), (K + 1 + f) * nx + i, dx)
        for f in range(E):                                   # energy row of step k = K+f: levels k and k+1
            k = K + f
            v, w = u[k, 0], u[k + 1, 0]
            add(np.full(nx, m0 + F + f), (k + 1) * nx + i, dx * w)
            add(np.full(nx, m0 + F + f), k * nx + i,
                -dx * v + dt * p["nu"] * (2.0 / dx) * (2.0 * v - v[ip] - v[im]))
    if kind in _HAS_MASS:
        m0 = nx if kind == HEAT1D_IC_MASS else n
        i = np.arange(nx)
        for k in range(nt):
            add(np.full(nx, m0 + k), k * nx + i, dx)

    J = sp.coo_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))), shape=(m, n))
    return J.tocsr()        # duplicates (tiny periodic grids where i+1 == i-1) are summed


HESS_SAFEGUARD = 0.1     # a free level's W_k is used only if its smallest eigenvalue a - 2|b| is at least this (else I)


def lagrangian_hessian(kind: int, u: np.ndarray, lam: np.ndarray, p: dict) -> sp.csr_matrix:
    """W = d^2/du^2 [ 1/2 ||u - u_hat||^2 + lam^T h(u) ] = I + sum_i lam_i grad^2 h_i(u)   (Eq. 5, Eq. 25)
    restricted to where it can change the Newton-KKT step (R22):

    * kinds whose local rows are square (1-4) and the pinned levels 0..K of kind 5: the step is fixed by J_loc du = -h
      whatever W is, so W = I there (kind 0 is affine: W = I exactly);
    * kind 5, free level k = K+1+f: only the energy rows are non-linear.  Row E_f = E(u[k]) - E(u[k-1]) + dt nu D(u[k-1])
      has grad^2 = dx I on level k and -dx I + dt nu (2/dx) L on level k-1 (E = dx/2 sum u^2, D = sum (u_{i+1}-u_i)^2 / dx,
      L = periodic second difference 2, -1, -1), so
          W_k = (1 + dx lam_E[f] - dx lam_E[f+1]) I + dt nu (2/dx) lam_E[f+1] L      (lam_E[F] := 0),
      a symmetric circulant tridiagonal with eigenvalues in [a - 2|b|, a + 2|b|], a = diagonal, b = off-diagonal.
      Inertia safeguard: if a - 2|b| < HESS_SAFEGUARD the level uses W_k = I (a Gauss-Newton level).
    Mass rows are linear.  Returns an n x n CSR matrix."""
    u = np.asarray(u, dtype=np.float64)
    nt, ny, nx = u.shape
    n = nt * ny * nx
    if kind == NS2D_VORT_ENST:       # enstrophy row of level k: grad^2 = 2 dx dy I on that level => W_k = (1 + 2 a lam_Z[k]) I
        a = p["dx"] * p["dy"]
        lamZ = np.asarray(lam, dtype=np.float64)[row_slices(kind, nx, ny, nt, p)["energy"]]
        diag = np.ones(n)
        for k in range(1, nt):
            wk = 1.0 + 2.0 * a * lamZ[k - 1]
            if wk >= HESS_SAFEGUARD:
                diag[k * ny * nx:(k + 1) * ny * nx] = wk
        return sp.diags(diag, format="csr")
    if kind != BURGERS1D_FLUXK:
        return sp.identity(n, format="csr")
    K, F, E = fluxk_counts(p, nt)
    if E == 0:
        return sp.identity(n, format="csr")
    lamE = np.concatenate([np.asarray(lam, dtype=np.float64)[row_slices(kind, nx, ny, nt, p)["energy"]], [0.0]])
    dx, cD = p["dx"], p["dt"] * p["nu"] * 2.0 / p["dx"]
    diag = np.ones(n)
    rows, cols, vals = [], [], []
    i = np.arange(nx)
    for f in range(F):
        k = K + 1 + f
        a = 1.0 + dx * (lamE[f] - lamE[f + 1]) + 2.0 * cD * lamE[f + 1]
        b = -cD * lamE[f + 1]
        if a - 2.0 * abs(b) < HESS_SAFEGUARD:
            continue                                 # W_k = I
        diag[k * nx:(k + 1) * nx] = a
        if b != 0.0:
            for sh in (1, -1):
                rows.append(k * nx + i)
                cols.append(k * nx + (i + sh) % nx)
                vals.append(np.full(nx, b))
    W = sp.diags(diag, format="csr")
    if rows:
        W = W + sp.coo_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))), shape=(n, n)).tocsr()
    return W


def paper_example_jacobian(nx: int, nt: int) -> np.ndarray:
    """The paper's own worked example (Appendix C, Eq. 26): IC rows first, then for
    k = 2..nt the left-Riemann mass row  sum_{i<nx} u_i^(k) - sum_{i<nx} u_i^(1)  (no dx weight,
    last node excluded, first time step omitted).  Dense (nx + nt - 1) x (nx nt)."""
    J = np.zeros((nx + nt - 1, nx * nt))
    for i in range(nx):
        J[i, i] = 1.0
    for k in range(1, nt):
        for i in range(nx - 1):
            J[nx + k - 1, i] = -1.0
            J[nx + k - 1, k * nx + i] = 1.0
    return J
