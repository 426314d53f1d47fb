"""ctypes binding of include/snap.h — argument marshalling only (same names as the C ABI)."""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional

HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(HERE, "libsnap.so")

HEAT1D_IC_MASS, BURGERS1D_LF, FISHER1D_IE, ALLENCAHN2D_IE, BURGERS1D_LF_MASS, BURGERS1D_FLUXK, NS2D_VORT_ENST = range(7)
# include/snap.h SNAP_STAT_* (slots of one sample's work-counter record) and SNAP_VAR_* (kernel variants)
(STAT_LINEARISATIONS, STAT_PASSES, STAT_ROWS_READ, STAT_ROWS_WRITTEN, STAT_VARIANT, STAT_INNER, STAT_ROW_DOUBLES,
 STAT_BACKTRACKS, STAT_COUNT) = range(9)
(VAR_NONE, VAR_HEAT_CLOSED_FORM, VAR_CLASSIC_BULK, VAR_CLASSIC_PLAIN, VAR_FUSED_TMA, VAR_PCG2D, VAR_DIRECT2D,
 VAR_FLUXK_BAND, VAR_NS_CLOSED_FORM) = range(9)

EXPORTS = [
    "snap_params_default", "snap_problem_create", "snap_problem_destroy", "snap_num_unknowns", "snap_num_rows",
    "snap_workspace_bytes", "snap_project", "snap_project_host", "snap_residual", "snap_schur_apply",
    "snap_project_stats", "snap_launch_count", "snap_strerror", "snap_flow_step", "snap_project_f32",
    "snap_schur_apply_static", "snap_static_scratch_bytes", "snap_static_scratch_init",
]


class SnapError(RuntimeError):
    pass


class SnapParams(C.Structure):
    """Mirror of `snap_params` (include/snap.h); field order and types must match."""
    _fields_ = [
        ("dx", C.c_double), ("dy", C.c_double), ("dt", C.c_double),
        ("nu", C.c_double), ("alpha", C.c_double),
        ("D", C.c_double), ("rho", C.c_double),
        ("eps", C.c_double),
        ("tol", C.c_double),
        ("max_iter", C.c_int), ("polish", C.c_int),
        ("ls_c1", C.c_double), ("ls_shrink", C.c_double),
        ("ls_max", C.c_int),
        ("pcg_rtol", C.c_double),
        ("pcg_max", C.c_int), ("precond", C.c_int), ("lambda_mode", C.c_int), ("gn_fuse", C.c_int),
        ("flux_steps", C.c_int), ("energy_rows", C.c_int), ("flux_kind", C.c_int), ("hessian", C.c_int),
    ]


_lib = None


def library_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen libsnap.so; raises SnapError if it is missing (no fallback of any kind)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise SnapError(f"{_LIB_PATH} not found: build it with `python -m paper_2607_00095_b200.build` "
                        "(or __graft_entry__.build()); there is no CPU fallback")
    lib = C.CDLL(_LIB_PATH)
    vp, dp, ip = C.c_void_p, C.c_void_p, C.c_void_p
    lib.snap_params_default.argtypes = [C.POINTER(SnapParams)]
    lib.snap_params_default.restype = None
    lib.snap_problem_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(SnapParams)]
    lib.snap_problem_create.restype = C.c_int
    lib.snap_problem_destroy.argtypes = [vp]
    lib.snap_problem_destroy.restype = C.c_int
    lib.snap_num_unknowns.argtypes = [vp]
    lib.snap_num_unknowns.restype = C.c_size_t
    lib.snap_num_rows.argtypes = [vp]
    lib.snap_num_rows.restype = C.c_size_t
    lib.snap_workspace_bytes.argtypes = [vp, C.c_int]
    lib.snap_workspace_bytes.restype = C.c_size_t
    lib.snap_project.argtypes = [vp, C.c_int, dp, dp, dp, dp, ip, C.c_int, vp, C.c_size_t, vp]
    lib.snap_project.restype = C.c_int
    lib.snap_flow_step.argtypes = [vp, C.c_int, dp, dp, dp, C.c_double, C.c_double, dp, dp, dp, dp, ip, vp, C.c_size_t, vp]
    lib.snap_flow_step.restype = C.c_int
    lib.snap_project_f32.argtypes = [vp, C.c_int, vp, vp, vp, ip, C.c_float, vp, C.c_size_t, vp]
    lib.snap_project_f32.restype = C.c_int
    lib.snap_project_host.argtypes = [vp, C.c_int, dp, dp, dp, dp, ip, C.c_int, vp]
    lib.snap_project_host.restype = C.c_int
    lib.snap_residual.argtypes = [vp, C.c_int, dp, dp, dp, dp, vp]
    lib.snap_residual.restype = C.c_int
    lib.snap_schur_apply.argtypes = [vp, C.c_int, dp, dp, dp, vp, C.c_size_t, vp]
    lib.snap_schur_apply.restype = C.c_int
    lib.snap_schur_apply_static.argtypes = [vp, C.c_int, dp, dp, dp, vp]
    lib.snap_schur_apply_static.restype = C.c_int
    lib.snap_static_scratch_bytes.argtypes = []
    lib.snap_static_scratch_bytes.restype = C.c_size_t
    lib.snap_static_scratch_init.argtypes = []
    lib.snap_static_scratch_init.restype = C.c_int
    lib.snap_project_stats.argtypes = [vp, C.c_int, vp, C.c_size_t, vp, vp]
    lib.snap_project_stats.restype = C.c_int
    lib.snap_launch_count.argtypes = [vp]
    lib.snap_launch_count.restype = C.c_longlong
    lib.snap_strerror.argtypes = [C.c_int]
    lib.snap_strerror.restype = C.c_char_p
    _lib = lib
    return lib


def exported_symbols() -> Dict[str, bool]:
    lib = load_library()
    return {name: hasattr(lib, name) for name in EXPORTS}


def snap_strerror(code: int) -> str:
    return load_library().snap_strerror(int(code)).decode()


def _check(rc: int, what: str):
    if rc != 0:
        raise SnapError(f"{what} failed: {rc} ({snap_strerror(rc)})")


def make_params(params: Optional[dict] = None) -> SnapParams:
    p = SnapParams()
    load_library().snap_params_default(C.byref(p))
    names = {f[0] for f in SnapParams._fields_}
    for k, v in (params or {}).items():
        if k not in names:
            raise SnapError(f"unknown snap_params field {k!r}")
        setattr(p, k, v)
    return p


def snap_problem_create(kind: int, nx: int, ny: int, nt: int, params: Optional[dict] = None) -> "Problem":
    return Problem(kind, nx, ny, nt, params)


def snap_problem_destroy(p: "Problem"):
    p.destroy()


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _nbytes(t) -> int:
    return 0 if t is None else int(t.numel() * t.element_size())


def _stream_handle(stream) -> Optional[C.c_void_p]:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return C.c_void_p(int(stream.cuda_stream))


class Problem:
    """Opaque `snap_problem*` plus its sizes."""

    def __init__(self, kind: int, nx: int, ny: int, nt: int, params: Optional[dict] = None):
        lib = load_library()
        self._h = C.c_void_p()
        self.kind, self.nx, self.ny, self.nt = int(kind), int(nx), int(ny), int(nt)
        self.cparams = make_params(params)
        rc = lib.snap_problem_create(C.byref(self._h), self.kind, self.nx, self.ny, self.nt, C.byref(self.cparams))
        if rc != 0:
            self._h = C.c_void_p()
            _check(rc, "snap_problem_create")
        self.n = int(lib.snap_num_unknowns(self._h))
        self.m = int(lib.snap_num_rows(self._h))

    @property
    def handle(self):
        return self._h

    def launch_count(self) -> int:
        return int(load_library().snap_launch_count(self._h))

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load_library().snap_problem_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def snap_workspace_bytes(p: Problem, batch: int) -> int:
    return int(load_library().snap_workspace_bytes(p.handle, int(batch)))


def _need(t, shape_numel: int, name: str, dtype):
    if t.dtype != dtype or not t.is_contiguous() or t.numel() < shape_numel:
        raise SnapError(f"{name}: need a contiguous {dtype} tensor with >= {shape_numel} elements")


def snap_project(p: Problem, batch: int, u_hat, cdata, u_star, lam, iters, warm: bool = False, workspace=None,
                 stream=None):
    """Enqueue the batched projection on `stream` (torch CUDA tensors in, results written in place)."""
    import torch
    for name, t, ne, dt in (("u_hat", u_hat, batch * p.n, torch.float64), ("cdata", cdata, batch * p.nx * p.ny, torch.float64),
                            ("u_star", u_star, batch * p.n, torch.float64), ("lambda", lam, batch * p.m, torch.float64),
                            ("iters", iters, batch, torch.int32)):
        if t is None and name == "lambda":
            continue                      # multiplier-free call (include/snap.h)
        _need(t, ne, name, dt)
        if not t.is_cuda:
            raise SnapError(f"{name} must be a CUDA tensor (use snap_project_host for host buffers)")
    if workspace is None:
        workspace = torch.empty(snap_workspace_bytes(p, batch), dtype=torch.uint8, device=u_hat.device)
    # the size check is the library's (SNAP_ENOMEM), not the binding's
    rc = load_library().snap_project(p.handle, int(batch), _ptr(u_hat), _ptr(cdata), _ptr(u_star), _ptr(lam), _ptr(iters),
                                     int(bool(warm)), _ptr(workspace), _nbytes(workspace), _stream_handle(stream))
    _check(rc, "snap_project")
    return workspace


def snap_flow_step(p: Problem, batch: int, u_tau, vel, u_prior, tau: float, tau_next: float, cdata, u1, u_next, lam, iters,
                   workspace=None, stream=None):
    """Enqueue one PCFM step (Eq. 1 shoot, Eq. 2 projection, Eq. 3 pull-back; include/snap.h).  `u_tau` is overwritten
    by u_hat_1; `lam` may be None (multiplier-free step)."""
    import torch
    for name, t, ne, dt in (("u_tau", u_tau, batch * p.n, torch.float64), ("vel", vel, batch * p.n, torch.float64),
                            ("u_prior", u_prior, batch * p.n, torch.float64), ("cdata", cdata, batch * p.nx * p.ny, torch.float64),
                            ("u1", u1, batch * p.n, torch.float64), ("u_next", u_next, batch * p.n, torch.float64),
                            ("lambda", lam, batch * p.m, torch.float64), ("iters", iters, batch, torch.int32)):
        if t is None and name == "lambda":
            continue
        _need(t, ne, name, dt)
        if not t.is_cuda:
            raise SnapError(f"{name} must be a CUDA tensor")
    if workspace is None:
        workspace = torch.empty(snap_workspace_bytes(p, batch), dtype=torch.uint8, device=u_tau.device)
    rc = load_library().snap_flow_step(p.handle, int(batch), _ptr(u_tau), _ptr(vel), _ptr(u_prior), float(tau), float(tau_next),
                                       _ptr(cdata), _ptr(u1), _ptr(u_next), _ptr(lam), _ptr(iters), _ptr(workspace),
                                       _nbytes(workspace), _stream_handle(stream))
    _check(rc, "snap_flow_step")
    return workspace


def snap_project_f32(p: Problem, batch: int, u_hat, cdata, u_star, iters, tol: float = 1e-5, workspace=None, stream=None):
    """Float32 mode (include/snap.h): multiplier-free projection of the Burgers kinds in fp32; torch.float32 CUDA tensors."""
    import torch
    for name, t, ne, dt in (("u_hat", u_hat, batch * p.n, torch.float32), ("cdata", cdata, batch * p.nx * p.ny, torch.float32),
                            ("u_star", u_star, batch * p.n, torch.float32), ("iters", iters, batch, torch.int32)):
        _need(t, ne, name, dt)
        if not t.is_cuda:
            raise SnapError(f"{name} must be a CUDA tensor")
    if workspace is None:
        workspace = torch.empty(snap_workspace_bytes(p, batch), dtype=torch.uint8, device=u_hat.device)
    rc = load_library().snap_project_f32(p.handle, int(batch), _ptr(u_hat), _ptr(cdata), _ptr(u_star), _ptr(iters), float(tol),
                                         _ptr(workspace), _nbytes(workspace), _stream_handle(stream))
    _check(rc, "snap_project_f32")
    return workspace


def snap_project_host(p: Problem, batch: int, u_hat, cdata, u_star, lam, iters, warm: bool = False, stream=None):
    """Same with HOST tensors (pinned or pageable); returns after the results are in the host buffers."""
    import torch
    for name, t, ne, dt in (("u_hat", u_hat, batch * p.n, torch.float64), ("cdata", cdata, batch * p.nx * p.ny, torch.float64),
                            ("u_star", u_star, batch * p.n, torch.float64), ("lambda", lam, batch * p.m, torch.float64),
                            ("iters", iters, batch, torch.int32)):
        if t is None and name == "lambda":
            continue
        _need(t, ne, name, dt)
        if t.is_cuda:
            raise SnapError(f"{name} must be a host tensor")
    rc = load_library().snap_project_host(p.handle, int(batch), _ptr(u_hat), _ptr(cdata), _ptr(u_star), _ptr(lam),
                                          _ptr(iters), int(bool(warm)), _stream_handle(stream))
    _check(rc, "snap_project_host")


def snap_residual(p: Problem, batch: int, u, cdata, h=None, norms=None, stream=None):
    rc = load_library().snap_residual(p.handle, int(batch), _ptr(u), _ptr(cdata), _ptr(h), _ptr(norms),
                                      _stream_handle(stream))
    _check(rc, "snap_residual")


def snap_schur_apply(p: Problem, batch: int, u, x, out, workspace, stream=None):
    rc = load_library().snap_schur_apply(p.handle, int(batch), _ptr(u), _ptr(x), _ptr(out), _ptr(workspace),
                                         _nbytes(workspace), _stream_handle(stream))
    _check(rc, "snap_schur_apply")


def snap_static_scratch_bytes() -> int:
    return int(load_library().snap_static_scratch_bytes())


def snap_static_scratch_init():
    """Resolve the static scratch array on the current device (once per device, at set-up; include/snap.h)."""
    _check(load_library().snap_static_scratch_init(), "snap_static_scratch_init")


def snap_schur_apply_static(p: Problem, batch: int, u, x, out, stream=None):
    """snap_schur_apply without a workspace: the scratch is the library's static device array (include/snap.h)."""
    rc = load_library().snap_schur_apply_static(p.handle, int(batch), _ptr(u), _ptr(x), _ptr(out), _stream_handle(stream))
    _check(rc, "snap_schur_apply_static")


def snap_project_stats(p: Problem, batch: int, workspace, stats, stream=None):
    """Copy the per-sample work counters of the last snap_project that used `workspace` into
    `stats` (CUDA int64 tensor [batch][STAT_COUNT], slots STAT_* = include/snap.h SNAP_STAT_*)."""
    import torch
    _need(stats, STAT_COUNT * batch, "stats", torch.int64)
    rc = load_library().snap_project_stats(p.handle, int(batch), _ptr(workspace), _nbytes(workspace), _ptr(stats),
                                           _stream_handle(stream))
    _check(rc, "snap_project_stats")
