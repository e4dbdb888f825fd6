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
  load_path       adaptive load stepping around newton_solve   PAPER.md:306 (step in [dt_min, dt_max], cut back on failure,
                                                              extrapolated initial guess), benchmark protocol :485

Pins (tests/test_oracle_newton.py): homogeneous-deformation patch solution, Hencky uniaxial closed form
(lateral log strain = -nu x axial log strain), identity-row invariants, quadratic convergence of the residual;
load_path: for proportional loading of an isotropic material the backward-Euler return map is exact for any step
size, so the stepped path must end in the state of a single increment, whatever the schedule and the cut-backs.
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


def load_path(coords, conn, hist0, mat, row_ptr, col_idx, bc_dofs, bc_full, fbar=0, dt0=1e-3, dt_min=1e-5, dt_max=5e-2, grow=1.5,
              cut=0.5, grow_below=5, max_steps=10000, extrapolate=1, rtol=1e-8, atol=1e-10, max_newton=12):
    """The paper's load stepping from load fraction t = 0 to 1 of the prescribed displacement bc_full:
    repeat { dt = min(dt, 1 - t); guess = u + (u - u_prev) dt/dt_prev (extrapolate = 1; the parabola through the last
    three converged states for 2; u for 0); newton_solve at t + dt; accepted when it converged and the balanced state
    shows no local non-convergence and no det F <= 0: t += dt, history carried over, dt *= grow (capped at dt_max) if
    it took <= grow_below iterations; otherwise the state stays and dt *= cut; give up when dt < dt_min }.
    Returns dict(u, hist, ts (accepted load fractions), steps, rejected, t, completed, newton_iters_total)."""
    bc_dofs = np.asarray(bc_dofs)
    bc_full = np.asarray(bc_full, dtype=np.float64)
    u = np.zeros_like(np.asarray(coords, dtype=np.float64))
    u_prev, u_pp = u.copy(), u.copy()
    hist = np.array(hist0, dtype=np.float64, copy=True)
    t, dt, dt_prev, dt_pp = 0.0, min(dt0, dt_max), 0.0, 0.0
    ts, rejected, newton_total = [], 0, 0
    while t < 1.0 - 1e-12:
        if len(ts) + rejected >= max_steps:
            break
        dt = min(dt, 1.0 - t)
        if extrapolate == 2 and dt_pp > 0.0:
            t0, t1, t2, t3 = -(dt_prev + dt_pp), -dt_prev, 0.0, dt
            l0 = (t3 - t1) * (t3 - t2) / ((t0 - t1) * (t0 - t2))
            l1 = (t3 - t0) * (t3 - t2) / ((t1 - t0) * (t1 - t2))
            l2 = (t3 - t0) * (t3 - t1) / ((t2 - t0) * (t2 - t1))
            guess = l2 * u + l1 * u_prev + l0 * u_pp
        else:
            r = dt / dt_prev if (extrapolate and dt_prev > 0.0) else 0.0
            guess = (1.0 + r) * u - r * u_prev
        res = newton_solve(coords, conn, guess, hist, mat, row_ptr, col_idx, bc_dofs, bc_full * (t + dt), fbar=fbar, rtol=rtol,
                           atol=atol, max_newton=max_newton)
        newton_total += res["newton_iters"]
        trouble = res["stats"]["n_nonconverged"] > 0 or res["stats"]["n_detF_nonpos"] > 0
        if res["converged"] and not trouble:
            t += dt
            ts.append(t)
            u_pp, u_prev, u = u_prev, u, res["u"]
            hist = res["hist_out"]
            dt_pp, dt_prev = dt_prev, dt
            if res["newton_iters"] <= grow_below:
                dt = min(dt * grow, dt_max)
        else:
            rejected += 1
            dt *= cut
            if dt < dt_min:
                break
    return dict(u=u, hist=hist, ts=ts, steps=len(ts), rejected=rejected, t=t, completed=t >= 1.0 - 1e-12,
                newton_iters_total=newton_total)
