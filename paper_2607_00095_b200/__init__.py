"""B200-native batched constraint projection (SNAP-FM hot path, arxiv/paper_2607_00095).

Thin Python binding over the C-ABI CUDA library `libsnap.so` (include/snap.h).  PyTorch is used
only for device memory and streams; every step of the path runs in the library's kernels.
There is no CPU fallback: loading fails loudly if the library has not been built.
"""
from .binding import (  # noqa: F401
    SnapError, SnapParams, Problem, load_library, library_path, exported_symbols,
    snap_problem_create, snap_problem_destroy, snap_workspace_bytes, snap_project, snap_project_host,
    snap_residual, snap_schur_apply, snap_strerror, snap_project_stats, snap_flow_step, snap_project_f32,
    snap_schur_apply_static, snap_static_scratch_bytes, snap_static_scratch_init,
    HEAT1D_IC_MASS, BURGERS1D_LF, FISHER1D_IE, ALLENCAHN2D_IE, BURGERS1D_LF_MASS, BURGERS1D_FLUXK, NS2D_VORT_ENST,
    STAT_LINEARISATIONS, STAT_PASSES, STAT_ROWS_READ, STAT_ROWS_WRITTEN, STAT_VARIANT, STAT_INNER, STAT_ROW_DOUBLES,
    STAT_BACKTRACKS, STAT_COUNT,
    VAR_NONE, VAR_HEAT_CLOSED_FORM, VAR_CLASSIC_BULK, VAR_CLASSIC_PLAIN, VAR_FUSED_TMA, VAR_PCG2D, VAR_DIRECT2D, VAR_FLUXK_BAND, VAR_NS_CLOSED_FORM,
)
