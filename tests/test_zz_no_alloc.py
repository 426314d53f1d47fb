"""No-allocation entry point (include/snap.h "No-allocation variant of snap_schur_apply"): snap_schur_apply_static keeps its
scratch vector g = J^T x in a file-scope static device array of the library instead of a caller workspace.  Checked
against the existing path (snap_schur_apply with a caller workspace) on the same inputs, two calls in a row that share
the static array (the second one smaller, of another kind: stale contents of the first must not matter), and against
the oracle's assembled J J^T x.  The file name sorts last on purpose (the suite runs with `pytest -x`)."""
import numpy as np
import pytest
import torch

import oracle as O
import workloads as W

pytestmark = pytest.mark.gpu

ATOL_SCHUR = 1e-13      # tests/test_gpu_parity.py::test_residual_and_schur_operator


@pytest.fixture(scope="module")
def S():
    import paper_2607_00095_b200 as S
    S.load_library()
    return S


def _both_paths(S, wl, seed):
    dev = torch.device("cuda:0")
    p = S.snap_problem_create(wl.kind, wl.nx, wl.ny, wl.nt, wl.params)
    B = wl.batch
    u = wl.u_hat.to(dev).contiguous()
    x = torch.randn(B, p.m, generator=torch.Generator().manual_seed(seed), dtype=torch.float64)
    xd = x.to(dev)
    ref = torch.full((B, p.m), float("nan"), dtype=torch.float64, device=dev)
    ws = torch.empty(B * p.n, dtype=torch.float64, device=dev)
    S.snap_schur_apply(p, B, u, xd, ref, ws)                       # existing path: caller workspace
    out = torch.full((B, p.m), float("nan"), dtype=torch.float64, device=dev)
    l0 = p.launch_count()
    S.snap_schur_apply_static(p, B, u, xd, out)                    # new path: the library's static scratch
    torch.cuda.synchronize()
    assert p.launch_count() - l0 == 2
    p.destroy()
    return x, ref.cpu().numpy(), out.cpu().numpy()


def test_static_scratch_entry_point_matches_the_workspace_path_on_two_calls_in_a_row(S):
    assert S.snap_static_scratch_bytes() == 8 * 2 ** 20
    S.snap_static_scratch_init()                                   # set-up, once per device; idempotent
    S.snap_static_scratch_init()
    # call 1 fills a large part of the array (4 x 128 x 128 doubles), call 2 and 3 reuse its head with other kinds / shapes
    cases = [(5, dict(batch=4, nx=128, nt=128)), (3, dict(batch=3, nx=77, nt=9)), (4, dict(batch=2, nx=12, ny=10, nt=6)),
             (1, dict(batch=2, nx=65, nt=7)), (2, dict(batch=2, nx=101, nt=9))]
    for i, (cfg, kw) in enumerate(cases):
        wl = W.make_workload(cfg, **kw)
        x, ref, out = _both_paths(S, wl, seed=11 + i)
        scale = max(1.0, np.abs(ref).max())
        assert np.isfinite(out).all()
        np.testing.assert_allclose(out, ref, rtol=0, atol=ATOL_SCHUR * scale)      # same kernels: in fact bit for bit
        np.testing.assert_array_equal(out, ref)
        if i > 0:                                                                   # small cases: the oracle's assembled J J^T
            for b in range(wl.batch):
                J = O.jacobian(wl.kind, wl.u_hat[b].numpy(), wl.params)
                s_ref = J @ (J.T @ x[b].numpy())
                np.testing.assert_allclose(out[b], s_ref, rtol=0, atol=ATOL_SCHUR * max(1.0, np.abs(s_ref).max()))


def test_static_scratch_entry_point_refuses_sizes_beyond_its_limit(S):
    dev = torch.device("cuda:0")
    wl = W.make_workload(2, batch=1, nx=128, nt=128)
    p = S.snap_problem_create(wl.kind, wl.nx, wl.ny, wl.nt, wl.params)
    limit = S.snap_static_scratch_bytes() // 8
    B = limit // p.n + 1                                           # 65 samples of 128 x 128: one beyond the limit
    assert B * p.n > limit >= (B - 1) * p.n
    u = torch.zeros(B, p.n, dtype=torch.float64, device=dev)
    x = torch.zeros(B, p.m, dtype=torch.float64, device=dev)
    out = torch.full((B, p.m), 7.0, dtype=torch.float64, device=dev)
    l0 = p.launch_count()
    with pytest.raises(S.SnapError, match="static scratch"):
        S.snap_schur_apply_static(p, B, u, x, out)
    torch.cuda.synchronize()
    assert p.launch_count() == l0 and bool((out == 7.0).all())     # nothing launched, nothing written
    S.snap_schur_apply_static(p, B - 1, u[:B - 1], x[:B - 1], out[:B - 1])          # exactly at the limit: accepted
    torch.cuda.synchronize()
    assert bool((out[:B - 1] == 0.0).all())
    p.destroy()
