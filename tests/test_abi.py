"""CPU-only checks of the C-ABI boundary: the library builds, loads and exports every symbol
include/snap.h declares; argument validation that needs no GPU."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2607_00095_b200 import build as B
    B.build()
    import paper_2607_00095_b200 as S
    return S


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "snap.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(snap_[a-z0-9_]+)\s*\(", src)))


def test_header_declares_and_library_exports_every_symbol(lib):
    declared = _declared_functions()
    assert {"snap_problem_create", "snap_project", "snap_residual", "snap_workspace_bytes",
            "snap_project_host", "snap_schur_apply"} <= set(declared)
    dll = C.CDLL(lib.library_path())
    for name in declared:
        assert hasattr(dll, name), f"{name} declared in snap.h but not exported"
    assert all(lib.exported_symbols().values())


def test_params_struct_matches_header_order(lib):
    src = open(os.path.join(ROOT, "include", "snap.h")).read()
    body = src[src.index("typedef struct {"):src.index("} snap_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in re.findall(r"(?:double|int)\s+([^;]+);", body):
        names += [n.strip() for n in decl.split(",")]
    assert names == [f[0] for f in lib.SnapParams._fields_]


def test_create_validates_arguments(lib):
    ok = dict(dx=0.1, dt=1e-3)
    p = lib.snap_problem_create(lib.BURGERS1D_LF, 32, 1, 16, ok)
    assert (p.n, p.m) == (512, 512)
    assert lib.snap_workspace_bytes(p, 4) >= 2 * 4 * 512 * 8
    p.destroy()
    p = lib.snap_problem_create(lib.BURGERS1D_LF_MASS, 32, 1, 16, ok)
    assert p.m == 512 + 16
    p = lib.snap_problem_create(lib.HEAT1D_IC_MASS, 32, 1, 16, ok)
    assert (p.n, p.m) == (512, 48)
    for bad in [dict(kind=7, nx=32, ny=1, nt=16), dict(kind=1, nx=32, ny=2, nt=16), dict(kind=1, nx=1, ny=1, nt=16),
                dict(kind=1, nx=1024, ny=1, nt=16), dict(kind=1, nx=32, ny=1, nt=1), dict(kind=3, nx=128, ny=64, nt=4)]:
        with pytest.raises(lib.SnapError):
            lib.snap_problem_create(bad["kind"], bad["nx"], bad["ny"], bad["nt"], ok)
    for badp in [dict(dx=0.0, dt=1e-3), dict(dx=0.1, dt=-1.0), dict(dx=0.1, dt=1e-3, tol=0.0),
                 dict(dx=0.1, dt=1e-3, ls_shrink=1.5), dict(dx=0.1, dt=1e-3, lambda_mode=3),
                 dict(dx=0.1, dt=1e-3, gn_fuse=-2), dict(dx=0.1, dt=1e-3, gn_fuse=65)]:
        with pytest.raises(lib.SnapError):
            lib.snap_problem_create(lib.BURGERS1D_LF, 32, 1, 16, badp)
    for fuse in (-1, 0, 1, 3):                 # classic path, default, capped
        lib.snap_problem_create(lib.BURGERS1D_LF, 32, 1, 16, dict(ok, gn_fuse=fuse)).destroy()
    # the workspace carries the per-sample work counters of snap_project_stats
    p = lib.snap_problem_create(lib.FISHER1D_IE, 64, 1, 16, ok)
    assert lib.snap_workspace_bytes(p, 3) >= 2 * 3 * p.n * 8 + 3 * 2 * 16 * 8 + 3 * 8 * lib.STAT_COUNT
    p.destroy()
    assert "invalid" in lib.snap_strerror(-1)


def test_short_workspace_is_refused_by_the_library_itself(lib):
    """SNAP_ENOMEM comes from the C entry points (not from the Python binding): call them through raw ctypes
    with a workspace one byte short.  The size check precedes every CUDA call, so no GPU is needed and the
    (never dereferenced) dummy pointers are safe."""
    p = lib.snap_problem_create(lib.BURGERS1D_LF_MASS, 64, 1, 16, dict(dx=0.1, dt=1e-3))
    dll = lib.load_library()
    need = lib.snap_workspace_bytes(p, 5)
    fake = C.c_void_p(0x1000)
    assert dll.snap_project(p.handle, 5, fake, fake, fake, fake, fake, 0, fake, need - 1, None) == -3
    assert dll.snap_project(p.handle, 5, fake, fake, fake, fake, fake, 0, fake, 0, None) == -3
    assert dll.snap_project(p.handle, 5, fake, fake, fake, fake, fake, 0, None, need, None) == -1   # NULL workspace
    assert dll.snap_project_stats(p.handle, 5, fake, need - 1, fake, None) == -3
    assert dll.snap_schur_apply(p.handle, 5, fake, fake, fake, fake, 5 * p.n * 8 - 1, None) == -3
    assert dll.snap_project(p.handle, 0, None, None, None, None, None, 0, None, 0, None) == 0       # empty batch
    assert "workspace" in lib.snap_strerror(-3)
    p.destroy()


def test_missing_library_fails_loudly(lib, monkeypatch):
    from paper_2607_00095_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "_LIB_PATH", "/nonexistent/libsnap.so")
    with pytest.raises(binding.SnapError):
        binding.load_library()


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2607_00095_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith(".py"):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2607_00095_b200" not in txt.replace("`paper_2607_00095_b200/`", ""), f
