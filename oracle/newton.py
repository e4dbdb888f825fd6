"""ORACLE — test infrastructure only.  SURVEY.md §8(f) NEXT-1: the steps around the element evaluation in one global
Newton iteration, written out plainly in numpy / scipy (fp64).  Only tests/ may import this; it shares nothing with the
CUDA path and imports nothing from paper_2606_17390_b200.

  spmv            y = K x                                     definition of the CSR matrix-vector product
  dirichlet       identity rows for constrained DOFs          PAPER.md:298 ("zero off-diagonal entries and reset the
                                                              diagonal to unity"), Alg. E1 steps 6-11 :1048-1053
  linear_solve    x = K^-1 b by a sparse direct factorisation the result of the paper's linear solve (Eq.(39) :279) has a
                                                              plain definition, so the oracle is that definition, not a
                                                              Krylov iteration (PAPER.md:304 lists direct solvers too)
  newton_solve    K dd = -R, d <- d + dd until ||rhs|| is small Eq.(39), in the paper's order

Pins (tests/test_oracle_newton.py): homogeneous-deformation patch solution, Hencky uniaxial closed form
(lateral log strain = -nu x axial log strain), identity-row invariants, quadratic convergence of the residual.
"""
import numpy as np
import scipy.sparse as sp
import scipy.sparse.linalg as spla

from . import assemble as _assemble


def csr(row_ptr, col_idx, vals):
    n = len(row_ptr) - 1
    return sp.csr_matrix((np.asarray(vals, dtype=np.float64), np.asarray(col_idx), np.asarray(row_ptr)), shape=(n, n))


def spmv(row_ptr, col_idx, vals, x):
    """y_r = sum_j vals[j] x[col_idx[j]] over row r, written out (no library call): the definition."""
    y = np.zeros(len(row_ptr) - 1)
    prod = np.asarray(vals, dtype=np.float64) * np.asarray(x, dtype=np.float64)[np.asarray(col_idx)]
    np.add.at(y, np.repeat(np.arange(len(row_ptr) - 1), np.diff(row_ptr)), prod)
    return y


def dirichlet(row_ptr, col_idx, vals, rhs, bc_dofs, bc_rhs=None):
    """Alg. E1 steps 6-11: each constrained row becomes the identity row; rhs[d] = bc_rhs (0 if None).  Columns untouched.
    Returns new (vals, rhs)."""
    vals = np.array(vals, dtype=np.float64, copy=True)
    rhs = None if rhs is None else np.array(rhs, dtype=np.float64, copy=True)
    for i, d in enumerate(np.asarray(bc_dofs)):
        a, b = row_ptr[d], row_ptr[d + 1]
        vals[a:b] = 0.0
        for j in range(a, b):
            if col_idx[j] == d:
                vals[j] = 1.0
        if rhs is not None:
            rhs[d] = 0.0 if bc_rhs is None else bc_rhs[i]
    return vals, rhs


def linear_solve(row_ptr, col_idx, vals, b):
    """x with K x = b (sparse LU)."""
    return spla.spsolve(csr(row_ptr, col_idx, vals).tocsc(), np.asarray(b, dtype=np.float64))


def newton_solve(coords, conn, u0, hist_in, mat, row_ptr, col_idx, bc_dofs, bc_vals, fbar=0, rtol=1e-9, atol=1e-10,
                 max_newton=25):
    """One load increment (Eq.(39)): repeat { R, K = assemble(u); rhs = -R; constrained rows: identity, rhs = prescribed - u;
    stop if ||rhs||_2 <= atol or <= rtol ||rhs_0||_2; dd = K^-1 rhs; u += dd }.
    Returns dict(u, hist_out, newton_iters, converged, norms)."""
    u = np.array(u0, dtype=np.float64, copy=True).reshape(-1, 3)
    bc_dofs = np.asarray(bc_dofs)
    bc_vals = np.asarray(bc_vals, dtype=np.float64)
    norms, out, converged, it = [], None, False, 0
    while True:
        out = _assemble(coords, conn, u, hist_in, mat, row_ptr, col_idx, fbar=fbar)
        vals, rhs = dirichlet(row_ptr, col_idx, out["csr_vals"], -out["residual"], bc_dofs, bc_vals - u.ravel()[bc_dofs])
        nrm = float(np.linalg.norm(rhs))
        norms.append(nrm)
        if nrm <= atol or nrm <= rtol * norms[0]:
            converged = True
            break
        if it >= max_newton or not np.isfinite(nrm):
            break
        dd = linear_solve(row_ptr, col_idx, vals, rhs)
        u = u + dd.reshape(-1, 3)
        it += 1
    return dict(u=u, hist_out=out["hist_out"], newton_iters=it, converged=converged, norms=norms, stats=out["stats"])
