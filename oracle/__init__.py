"""CPU oracle for the SNAP-FM batched constraint projection (arxiv/paper_2607_00095).

THIS PACKAGE IS TEST INFRASTRUCTURE, NOT PRODUCT CODE.  It is a plain, slow,
obviously-correct fp64 numpy/scipy implementation of

    u* = argmin_u 1/2 ||u - u_hat||^2   s.t.  h(u) = 0          (Eq. 2, Eq. 4)

by Gauss-Newton / Newton-KKT iterations on explicitly assembled sparse matrices
(Eq. 5, Eq. 24 L468 with W = I).  Only `tests/`,
`__graft_entry__.smoke()` and the `cpu_baseline` / `--impl reference` legs of
`bench.py` may import it.  It shares no code with `paper_2607_00095_b200/`
(the CUDA path) and imports nothing from it; the only common module is
`workloads/` (seeded input generators, no method arithmetic).

Pins (tests/test_oracle_pins.py, all `-m "not gpu"`):
  P1 closed-form linear projection (heat), P2 forward-solve identity (kinds 1-4),
  P3 dense LU of the full KKT matrix / pseudo-inverse on tiny grids, P4 KKT invariants,
  P5 Jacobian vs central finite differences, P6 chol(J J^T) = J factor identity and
  the analytic Gram matrix of the left null space, P7 feasible-input / idempotence /
  shift-equivariance / batch-independence, P8 the paper's printed 5x9 Jacobian (Eq. 26).
Parity unpinned: the *trajectory* (iterates, step lengths, iteration counts) — the paper
prints no numeric values of any projected field; only the converged (u*, lambda*) is pinned.
"""
from .constraints import (  # noqa: F401
    residual, jacobian, row_slices, full_rank_rows, num_rows, residual_norms,
    paper_example_jacobian, godunov_flux, godunov_flux_grad, fluxk_counts, lagrangian_hessian, HESS_SAFEGUARD, NS2D_VORT_ENST,
)
from .linsolve import (  # noqa: F401
    solve_kkt_dense_lu, solve_schur_pinv, solve_schur_banded_cholesky, solve_schur_cg, solve_schur_dense_cholesky,
    min_norm_multiplier, solve_kkt_sparse_lu,
)
from .project import project, project_batch  # noqa: F401
from .flow import flow_step  # noqa: F401
