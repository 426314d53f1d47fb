"""Seeded input generators for the five BASELINE.json configs.

Everything here is *input manufacture*: grids, initial conditions, the scheme's
own forward solution `u_true` (written in time-stepping "update" form), and the
noisy field `u_hat` handed to the projection.  No projection, residual-vector,
Jacobian or KKT arithmetic lives here.  The paper's datasets and pretrained flow
models are not available, so these
synthetic fields stand in for them; shapes follow the paper's experiments E1/E4/E5/E6
and values follow BASELINE.json `configs`.

All tensors are torch fp64.  A `torch.Generator` on the requested device is seeded
per config; per-sample parameters are drawn first, then the noise in C order.  The
CPU and CUDA generators produce different streams: whoever generates the tensors
hands *the same tensors* (host copy) to the oracle, so no RNG parity is involved.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Dict, Optional

import torch

KIND_HEAT1D_IC_MASS = 0
KIND_BURGERS1D_LF = 1
KIND_FISHER1D_IE = 2
KIND_ALLENCAHN2D_IE = 3
KIND_BURGERS1D_LF_MASS = 4
KIND_BURGERS1D_FLUXK = 5
KIND_NS2D_VORT_ENST = 6
KIND_NAMES = {
    0: "HEAT1D_IC_MASS", 1: "BURGERS1D_LF", 2: "FISHER1D_IE",
    3: "ALLENCAHN2D_IE", 4: "BURGERS1D_LF_MASS", 5: "BURGERS1D_FLUXK", 6: "NS2D_VORT_ENST",
}

# cfg -> (kind, batch, nx, ny, nt, seed)   (BASELINE.json configs[0..4] = cfg 1..5)
CONFIG_SHAPES = {
    1: (KIND_HEAT1D_IC_MASS, 4, 64, 1, 64, 1001),
    2: (KIND_BURGERS1D_LF, 32, 128, 1, 128, 1002),
    3: (KIND_FISHER1D_IE, 256, 128, 1, 128, 1003),
    4: (KIND_ALLENCAHN2D_IE, 64, 64, 64, 32, 1004),
    5: (KIND_BURGERS1D_LF_MASS, 1024, 256, 1, 256, 1005),
    # SURVEY.md §8(f) NEXT-1 / NEXT-4 (not BASELINE.json configs): the paper's "IC, Mass, Flux(k = 5)" row set
    # (Eq. 14, Table XVIII) at the scale of cfg 5.
    6: (KIND_BURGERS1D_FLUXK, 1024, 256, 1, 256, 1006),   # Lax-Friedrichs flux rows + energy-evolution rows (Eq. 11)
    7: (KIND_BURGERS1D_FLUXK, 1024, 256, 1, 256, 1007),   # Godunov flux rows (L555), inviscid, no energy rows
    8: (KIND_BURGERS1D_FLUXK, 1024, 256, 1, 256, 1006),   # config 6 (same inputs) with the exact Lagrangian Hessian (NEXT-2)
    # the paper's Navier-Stokes row set (Eq. 20: IC + total vorticity + enstrophy) at the paper's grid 16 x 16 x 50
    # (L398); the paper samples 2 fields, here a batch of 256
    9: (KIND_NS2D_VORT_ENST, 256, 16, 16, 50, 1009),
}
CONFIG_EXTRA = {6: dict(flux_steps=5, energy_rows=1, flux_kind=0),
                7: dict(flux_steps=5, energy_rows=0, flux_kind=1, nu=0.0),
                8: dict(flux_steps=5, energy_rows=1, flux_kind=0, hessian=1)}

F64 = torch.float64


def default_params(kind: int, nx: int, ny: int, nt: int) -> Dict[str, float]:
    """Grid steps and physical constants per kind, plus the
    solver knobs of `snap_params` at their defaults."""
    p = dict(dx=1.0, dy=1.0, dt=1.0, nu=0.0, alpha=1.0, D=0.0, rho=0.0, eps=0.0,
             tol=1e-10, max_iter=50, polish=1, ls_c1=1e-4, ls_shrink=0.5, ls_max=20,
             pcg_rtol=1e-13, pcg_max=200, precond=2, lambda_mode=0)
    if kind == KIND_HEAT1D_IC_MASS:
        p.update(dx=1.0 / (nx - 1), dt=1.0 / max(nt - 1, 1), nu=0.1)
    elif kind in (KIND_BURGERS1D_LF, KIND_BURGERS1D_LF_MASS, KIND_BURGERS1D_FLUXK):
        p.update(dx=2.0 * math.pi / nx, dt=1e-3, nu=0.01, alpha=1.0)
        if kind == KIND_BURGERS1D_FLUXK:
            p.update(flux_steps=min(5, nt - 1), energy_rows=1, flux_kind=0)
    elif kind == KIND_FISHER1D_IE:
        p.update(dx=1.0 / nx, dt=1.0 / max(nt - 1, 1), D=0.01, rho=1.0)
    elif kind == KIND_ALLENCAHN2D_IE:
        p.update(dx=1.0 / nx, dy=1.0 / ny, dt=1e-3, eps=0.05)
    elif kind == KIND_NS2D_VORT_ENST:
        p.update(dx=1.0 / nx, dy=1.0 / ny, dt=1.0)       # Omega = [0, 1]^2, unit time step (Eq. 19)
    else:
        raise ValueError(f"unknown kind {kind}")
    return p


@dataclass
class Workload:
    cfg: int
    kind: int
    batch: int
    nx: int
    ny: int
    nt: int
    params: Dict[str, float]
    cdata: torch.Tensor            # [B, ny, nx]      per-sample IC target u0
    u_true: torch.Tensor           # [B, nt, ny, nx]  clean field
    u_hat: Optional[torch.Tensor]  # [B, nt, ny, nx]  noisy input (None for cfg 5: use burgers_tau_input)
    seed: int = 0
    meta: Dict[str, object] = field(default_factory=dict)

    @property
    def n(self) -> int:
        return self.nx * self.ny * self.nt

    @property
    def m(self) -> int:
        """Number of constraint rows per sample, in the lambda layout of include/snap.h."""
        if self.kind == KIND_HEAT1D_IC_MASS:
            return self.nx + self.nt
        if self.kind == KIND_BURGERS1D_LF_MASS:
            return self.n + self.nt
        if self.kind == KIND_BURGERS1D_FLUXK:
            K = int(self.params["flux_steps"])
            F = self.nt - 1 - K
            return (K + 1) * self.nx + F * (2 if int(self.params["energy_rows"]) else 1)
        if self.kind == KIND_NS2D_VORT_ENST:
            return self.nx * self.ny + 2 * (self.nt - 1)
        return self.n


# ----------------------------------------------------------------------------------------
# scheme forward solvers (update form u[k+1] = Phi(u[k])), batched over the leading axis
# ----------------------------------------------------------------------------------------

def _burgers_lf_step(v: torch.Tensor, dx: float, dt: float, nu: float, alpha: float) -> torch.Tensor:
    """One finite-volume step with Lax-Friedrichs flux F=(f(a)+f(b))/2 - alpha/2 (b-a),
    f=u^2/2, explicit central viscosity, periodic (BASELINE.json configs 2, 5)."""
    vp = torch.roll(v, -1, -1)
    vm = torch.roll(v, 1, -1)
    f = 0.5 * v * v
    F_right = 0.5 * (f + torch.roll(f, -1, -1)) - 0.5 * alpha * (vp - v)   # F_{i+1/2}
    F_left = torch.roll(F_right, 1, -1)                                    # F_{i-1/2}
    return v - (dt / dx) * (F_right - F_left) + (nu * dt / dx ** 2) * (vp - 2.0 * v + vm)


def _burgers_godunov_step(v: torch.Tensor, dx: float, dt: float, nu: float) -> torch.Tensor:
    """One finite-volume step with the Godunov flux of f = u^2/2 and optional explicit
    central viscosity, periodic."""
    vp = torch.roll(v, -1, -1)
    vm = torch.roll(v, 1, -1)
    F_right = torch.maximum(0.5 * v.clamp_min(0.0) ** 2, 0.5 * vp.clamp_max(0.0) ** 2)   # F(u_i, u_{i+1})
    F_left = torch.roll(F_right, 1, -1)
    return v - (dt / dx) * (F_right - F_left) + (nu * dt / dx ** 2) * (vp - 2.0 * v + vm)


def _thomas_batched(lo: torch.Tensor, di: torch.Tensor, up: torch.Tensor, rhs: torch.Tensor) -> torch.Tensor:
    """Tridiagonal solve along the last axis, vectorised over leading axes
    (lo[...,0] and up[...,-1] unused)."""
    n = di.shape[-1]
    c = torch.empty_like(di)
    d = torch.empty_like(rhs)
    c[..., 0] = up[..., 0] / di[..., 0]
    d[..., 0] = rhs[..., 0] / di[..., 0]
    for i in range(1, n):
        den = di[..., i] - lo[..., i] * c[..., i - 1]
        c[..., i] = up[..., i] / den
        d[..., i] = (rhs[..., i] - lo[..., i] * d[..., i - 1]) / den
    x = torch.empty_like(rhs)
    x[..., -1] = d[..., -1]
    for i in range(n - 2, -1, -1):
        x[..., i] = d[..., i] - c[..., i] * x[..., i + 1]
    return x


def _lap1d_neumann(v: torch.Tensor, dx: float) -> torch.Tensor:
    """Cell-centred 3-point Laplacian with ghost-cell Neumann ends (R10)."""
    out = torch.empty_like(v)
    out[..., 1:-1] = v[..., 2:] - 2.0 * v[..., 1:-1] + v[..., :-2]
    out[..., 0] = v[..., 1] - v[..., 0]
    out[..., -1] = v[..., -2] - v[..., -1]
    return out / dx ** 2


def _fisher_ie_step(v: torch.Tensor, dx: float, dt: float, D: float, rho: float, newton: int = 8) -> torch.Tensor:
    """Implicit Euler step of u_t = D u_xx + rho u (1-u): solve
    w - v - dt (D Lap w + rho w (1-w)) = 0 for w by Newton with tridiagonal solves."""
    w = v.clone()
    nx = v.shape[-1]
    a = dt * D / dx ** 2
    off = torch.full_like(v, -a)
    for _ in range(newton):
        g = w - v - dt * (D * _lap1d_neumann(w, dx) + rho * w * (1.0 - w))
        diag = 1.0 + 2.0 * a - dt * rho * (1.0 - 2.0 * w)
        diag[..., 0] -= a
        diag[..., nx - 1] -= a
        w = w - _thomas_batched(off, diag, off, g)
    return w


def _lap2d_periodic(v: torch.Tensor, dx: float, dy: float) -> torch.Tensor:
    return ((torch.roll(v, -1, -1) - 2.0 * v + torch.roll(v, 1, -1)) / dx ** 2
            + (torch.roll(v, -1, -2) - 2.0 * v + torch.roll(v, 1, -2)) / dy ** 2)


def _allencahn_ie_step(v: torch.Tensor, dx: float, dy: float, dt: float, eps: float,
                       newton: int = 6, cg_iters: int = 40) -> torch.Tensor:
    """Implicit Euler step of u_t = eps^2 Lap u - u^3 + u (periodic): Newton on
    w - v - dt (eps^2 Lap w - w^3 + w) = 0, inner linear solves by batched CG
    (the Newton matrix is SPD with condition number ~1.1)."""
    w = v.clone()

    def dot(a, b):
        return (a * b).sum((-1, -2), keepdim=True)

    for _ in range(newton):
        g = w - v - dt * (eps ** 2 * _lap2d_periodic(w, dx, dy) - w ** 3 + w)
        c = 1.0 + dt * (3.0 * w * w - 1.0)

        def T(x):
            return c * x - dt * eps ** 2 * _lap2d_periodic(x, dx, dy)

        x = torch.zeros_like(g)
        r = g.clone()
        p = r.clone()
        rr = dot(r, r)
        for _ in range(cg_iters):
            if float(rr.max()) == 0.0:
                break
            q = T(p)
            al = rr / dot(p, q).clamp_min(1e-300)
            x = x + al * p
            r = r - al * q
            rr_new = dot(r, r)
            p = r + (rr_new / rr.clamp_min(1e-300)) * p
            rr = rr_new
            if float(rr.max()) < 1e-36:
                break
        w = w - x
    return w


# ----------------------------------------------------------------------------------------
# the five configs
# ----------------------------------------------------------------------------------------

def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def make_workload(cfg: int, batch: Optional[int] = None, nx: Optional[int] = None,
                  ny: Optional[int] = None, nt: Optional[int] = None, seed: Optional[int] = None,
                  device="cpu", noise: Optional[float] = None, with_u_hat: bool = True,
                  params: Optional[Dict[str, float]] = None) -> Workload:
    """Build config `cfg` (1..5) of BASELINE.json, optionally at reduced batch/grid
    (same recipe, same seeds) for tests.  For cfg 5 `u_hat` is the tau_j = j/50, j=25
    input unless `with_u_hat=False`; use `burgers_tau_input` for the 50-tau sequence."""
    kind, B0, nx0, ny0, nt0, seed0 = CONFIG_SHAPES[cfg]
    B = B0 if batch is None else int(batch)
    nx = nx0 if nx is None else int(nx)
    ny = ny0 if ny is None else int(ny)
    nt = nt0 if nt is None else int(nt)
    seed = seed0 if seed is None else int(seed)
    dev = torch.device(device)
    g = _gen(seed, dev)
    p = default_params(kind, nx, ny, nt)
    if cfg in CONFIG_EXTRA:
        p.update(CONFIG_EXTRA[cfg])
        p["flux_steps"] = min(int(p["flux_steps"]), nt - 1)
    if params:
        p.update(params)
    meta: Dict[str, object] = {}

    if kind == KIND_HEAT1D_IC_MASS:
        x = torch.arange(nx, dtype=F64, device=dev) * p["dx"]
        t = torch.arange(nt, dtype=F64, device=dev) * p["dt"]
        u0 = torch.sin(math.pi * x).expand(B, 1, nx).contiguous()
        clean = (torch.sin(math.pi * x)[None, None, :]
                 * torch.exp(-math.pi ** 2 * p["nu"] * t)[None, :, None]).expand(B, nt, nx)
        u_true = clean.reshape(B, nt, 1, nx).contiguous()
        sigma = 0.1 if noise is None else noise
    elif kind in (KIND_BURGERS1D_LF, KIND_BURGERS1D_LF_MASS, KIND_BURGERS1D_FLUXK):
        x = torch.arange(nx, dtype=F64, device=dev) * p["dx"]
        phi = torch.rand(B, generator=g, dtype=F64, device=dev) * (2.0 * math.pi)
        meta["phi"] = phi
        u0 = (torch.sin(x)[None, :] + 0.5 * torch.sin(2.0 * x[None, :] + phi[:, None])).reshape(B, 1, nx)
        u_true = torch.empty(B, nt, 1, nx, dtype=F64, device=dev)
        u_true[:, 0] = u0
        godunov = kind == KIND_BURGERS1D_FLUXK and int(p.get("flux_kind", 0)) == 1
        for k in range(nt - 1):
            if godunov:
                u_true[:, k + 1] = _burgers_godunov_step(u_true[:, k], p["dx"], p["dt"], p["nu"])
            else:
                u_true[:, k + 1] = _burgers_lf_step(u_true[:, k], p["dx"], p["dt"], p["nu"], p["alpha"])
        sigma = 0.05 if noise is None else noise
    elif kind == KIND_FISHER1D_IE:
        x = (torch.arange(nx, dtype=F64, device=dev) + 0.5) * p["dx"]
        amp = 0.2 + 0.6 * torch.rand(B, generator=g, dtype=F64, device=dev)
        meta["amp"] = amp
        u0 = (amp[:, None] * torch.exp(-(x[None, :] - 0.5) ** 2 / (2.0 * 0.1 ** 2))).reshape(B, 1, nx)
        u_true = torch.empty(B, nt, 1, nx, dtype=F64, device=dev)
        u_true[:, 0] = u0
        for k in range(nt - 1):
            u_true[:, k + 1] = _fisher_ie_step(u_true[:, k], p["dx"], p["dt"], p["D"], p["rho"])
        sigma = 0.05 if noise is None else noise
    elif kind == KIND_ALLENCAHN2D_IE:
        x = torch.arange(nx, dtype=F64, device=dev) * p["dx"]
        y = torch.arange(ny, dtype=F64, device=dev) * p["dy"]
        modes = [(kx, ky) for kx in range(-4, 5) for ky in range(-4, 5)
                 if 0 < kx * kx + ky * ky <= 16]
        coef = torch.randn(B, len(modes), 2, generator=g, dtype=F64, device=dev)
        u0 = torch.zeros(B, ny, nx, dtype=F64, device=dev)
        for mi, (kx, ky) in enumerate(modes):
            ph = 2.0 * math.pi * (kx * x[None, :] + ky * y[:, None])
            u0 += coef[:, mi, 0, None, None] * torch.cos(ph)[None] + coef[:, mi, 1, None, None] * torch.sin(ph)[None]
        u0 = u0 / u0.abs().amax((-1, -2), keepdim=True)
        u_true = torch.empty(B, nt, ny, nx, dtype=F64, device=dev)
        u_true[:, 0] = u0
        for k in range(nt - 1):
            u_true[:, k + 1] = _allencahn_ie_step(u_true[:, k], p["dx"], p["dy"], p["dt"], p["eps"])
        sigma = 0.05 if noise is None else noise
    elif kind == KIND_NS2D_VORT_ENST:
        # IC: a random Fourier field as for cfg 4 plus a non-zero mean; clean field: the IC advected by one cell per
        # step (a periodic shift keeps sum w and sum w^2, so it is feasible for Eq. 20 whatever the flow is)
        x = torch.arange(nx, dtype=F64, device=dev) * p["dx"]
        y = torch.arange(ny, dtype=F64, device=dev) * p["dy"]
        modes = [(kx, ky) for kx in range(-3, 4) for ky in range(-3, 4) if 0 < kx * kx + ky * ky <= 9]
        coef = torch.randn(B, len(modes), 2, generator=g, dtype=F64, device=dev)
        mean = 0.2 * torch.randn(B, 1, 1, generator=g, dtype=F64, device=dev)
        u0 = torch.zeros(B, ny, nx, dtype=F64, device=dev)
        for mi, (kx, ky) in enumerate(modes):
            ph = 2.0 * math.pi * (kx * x[None, :] + ky * y[:, None])
            u0 += coef[:, mi, 0, None, None] * torch.cos(ph)[None] + coef[:, mi, 1, None, None] * torch.sin(ph)[None]
        u0 = u0 / u0.abs().amax((-1, -2), keepdim=True) + mean
        u_true = torch.stack([torch.roll(u0, shifts=(k % ny, (2 * k) % nx), dims=(-2, -1)) for k in range(nt)], dim=1)
        sigma = 0.05 if noise is None else noise
    else:
        raise ValueError(kind)

    cdata = u0.reshape(B, ny, nx).contiguous()
    u_hat = None
    if cfg == 5:
        wl = Workload(cfg, kind, B, nx, ny, nt, p, cdata, u_true, None, seed, meta)
        if with_u_hat:
            wl.u_hat = burgers_tau_input(wl, 25)
        return wl
    if with_u_hat:
        u_hat = u_true + sigma * torch.randn(u_true.shape, generator=g, dtype=F64, device=dev)
    return Workload(cfg, kind, B, nx, ny, nt, p, cdata, u_true, u_hat, seed, meta)


def burgers_tau_input(wl: Workload, j: int, n_tau: int = 50, out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """Config 5 input at flow time tau_j = j/n_tau (j = 1..n_tau):
    u_hat_j = tau_j u_true + (1 - tau_j) N(0,1), fresh noise seeded 5000 + j."""
    tau = float(j) / float(n_tau)
    g = _gen(5000 + j, wl.u_true.device)
    if out is None:
        out = torch.empty_like(wl.u_true)
    out.normal_(generator=g)
    out.mul_(1.0 - tau).add_(wl.u_true, alpha=tau)
    return out
