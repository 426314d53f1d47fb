"""Oracle linear algebra back ends for the Newton-KKT step (Eq. 5, Eq. 24).

TEST INFRASTRUCTURE (see oracle/__init__.py).  Every routine works on explicitly
assembled matrices and calls a generic library factorisation (LAPACK through
numpy/scipy); nothing here knows the block structure the CUDA path exploits.

With f(u) = 1/2 ||u - u_hat||^2 and W = I (Gauss-Newton) system (24) is
    [ I  J^T ] [ d    ]     [ u - u_hat ]
    [ J  0   ] [ lam+ ] = - [ h         ]
whose Schur form is  (J J^T) lam+ = h - J (u - u_hat) =: r ,  d = -(u - u_hat) - J^T lam+ .
"""
from __future__ import annotations

import numpy as np
import scipy.linalg as sla
import scipy.sparse as sp


def solve_kkt_dense_lu(J, w: np.ndarray, h: np.ndarray):
    """Tiny grids: assemble the full dense (n+m) x (n+m) KKT matrix [I J^T; J 0] and solve it
    by LU with partial pivoting (LAPACK gesv).  Needs full row rank.  Returns (d, lam)."""
    Jd = J.toarray() if sp.issparse(J) else np.asarray(J)
    m, n = Jd.shape
    K = np.zeros((n + m, n + m))
    K[:n, :n] = np.eye(n)
    K[:n, n:] = Jd.T
    K[n:, :n] = Jd
    sol = np.linalg.solve(K, -np.concatenate([w, h]))
    return sol[:n], sol[n:]


def solve_schur_pinv(J, r: np.ndarray) -> np.ndarray:
    """Tiny grids, rank-deficient J: minimum-norm solution lam = (J J^T)^+ r via the SVD-based
    pseudo-inverse."""
    Jd = J.toarray() if sp.issparse(J) else np.asarray(J)
    return np.linalg.pinv(Jd @ Jd.T, rcond=1e-12, hermitian=True) @ r


def _to_upper_banded(S: sp.spmatrix):
    """Upper banded storage ab[bw + i - j, j] = S[i, j] (i <= j) for LAPACK pbtrf."""
    Sd = sp.dia_matrix(S)
    offs = Sd.offsets
    bw = int(max(offs.max(), 0))
    n = S.shape[0]
    ab = np.zeros((bw + 1, n))
    for off, row in zip(offs, Sd.data):
        if off >= 0:
            ab[bw - off, off:] = row[off:n]
    return ab


def solve_schur_banded_cholesky(S: sp.spmatrix, r: np.ndarray, refine: int = 1) -> np.ndarray:
    """1D at size: explicit S = J J^T (SPD, half-bandwidth 2 nx - 1 in time-major order) ->
    banded Cholesky (LAPACK pbtrf/pbtrs) + `refine` steps of iterative refinement."""
    ab = _to_upper_banded(S)
    cb = sla.cholesky_banded(ab, lower=False, check_finite=False)
    x = sla.cho_solve_banded((cb, False), r, check_finite=False)
    for _ in range(refine):
        x = x + sla.cho_solve_banded((cb, False), r - S @ x, check_finite=False)
    return x


def solve_schur_dense_cholesky(S: np.ndarray, r: np.ndarray, refine: int = 1) -> np.ndarray:
    """Few rows with dense border rows (kind 5): explicit dense S = J J^T (SPD) -> LAPACK potrf/potrs + `refine`
    steps of iterative refinement."""
    cf = sla.cho_factor(S, lower=True, check_finite=False)
    x = sla.cho_solve(cf, r, check_finite=False)
    for _ in range(refine):
        x = x + sla.cho_solve(cf, r - S @ x, check_finite=False)
    return x


def solve_schur_cg(S: sp.spmatrix, r: np.ndarray, x0=None, rtol: float = 1e-13, maxiter: int = 20000):
    """2D at size: plain un-preconditioned conjugate gradients on explicit S to relative
    residual ||r - S x|| / ||r|| <= rtol.  Returns (x, iterations)."""
    x = np.zeros_like(r) if x0 is None else np.array(x0, dtype=np.float64)
    res = r - S @ x
    p = res.copy()
    rr = float(res @ res)
    bnorm = float(np.linalg.norm(r))
    if bnorm == 0.0:
        return np.zeros_like(r), 0
    it = 0
    while np.sqrt(rr) > rtol * bnorm and it < maxiter:
        q = S @ p
        a = rr / float(p @ q)
        x += a * p
        res -= a * q
        rr_new = float(res @ res)
        p = res + (rr_new / rr) * p
        rr = rr_new
        it += 1
    return x, it


def min_norm_multiplier(J: sp.spmatrix, lam_any: np.ndarray) -> np.ndarray:
    """Minimum-norm multiplier: among all lam with J^T lam = J^T lam_any
    return the one of least Euclidean norm, lam = (J^T)^+ (J^T lam_any).

    * few rows (m <= 4096): dense SVD least squares (LAPACK gelsd) — works for any rank;
    * otherwise J must have full column rank (kind 4: J_loc is square nonsingular), then
      (J^T)^+ = J (J^T J)^{-1} and J^T J (n x n, banded) is factored by banded Cholesky."""
    g = J.T @ lam_any
    m, n = J.shape
    if m <= 4096:
        lam, *_ = np.linalg.lstsq(J.T.toarray(), g, rcond=1e-12)
        return lam
    N = (J.T @ J).tocsr()
    z = solve_schur_banded_cholesky(N, g, refine=1)
    return J @ z


def solve_kkt_sparse_lu(W: sp.spmatrix, J: sp.spmatrix, w: np.ndarray, h: np.ndarray):
    """Newton-KKT step with a general (symmetric) Lagrangian Hessian W (Eq. 24):
        [ W  J^T ] [ du  ]   [ -w ]
        [ J   0  ] [ lam ] = [ -h ]
    by sparse LU (SuperLU) of the full (n+m) x (n+m) matrix -- the paper's own formulation (sparse LDL^T of the KKT
    matrix, L114-116), no Schur complement.  One step of iterative refinement.  Returns (du, lam)."""
    import scipy.sparse.linalg as spla
    n, m = W.shape[0], J.shape[0]
    Kmat = sp.bmat([[W, J.T], [J, None]], format="csc")
    rhs = -np.concatenate([w, h])
    lu = spla.splu(Kmat)
    x = lu.solve(rhs)
    x += lu.solve(rhs - Kmat @ x)
    return x[:n], x[n:]

