"""Pins of oracle/newton.py against what mechanics and linear algebra fix, not against itself:
dense brute force for the Dirichlet rows and y = K x, the homogeneous-deformation patch solution, the Hencky uniaxial
closed form, the Lankford ratio of the plastic lateral strains, and quadratic convergence of the global Newton loop."""
import numpy as np
import pytest

import oracle
import oracle.newton as onw
import synth
from synth import mesh


def _problem(nx, ny, nz, L=(1.0, 1.0, 1.0), desc=None):
    coords, conn = mesh.structured_hex_mesh(nx, ny, nz, *L)
    ne = conn.shape[0]
    mat = oracle.mat_from_desc(dict(synth.configs.SWIFT) if desc is None else desc, ne)
    row_ptr, col_idx, _ = oracle.pattern(coords.shape[0], conn, with_slots=False)
    return coords, conn, mat, row_ptr, col_idx, np.zeros((ne, 8, 7))


def _dense(row_ptr, col_idx, vals):
    n = len(row_ptr) - 1
    K = np.zeros((n, n))
    for r in range(n):
        for j in range(row_ptr[r], row_ptr[r + 1]):
            K[r, col_idx[j]] += vals[j]
    return K


def test_spmv_and_dirichlet_against_dense_brute_force():
    coords, conn, mat, rp, ci, h0 = _problem(2, 2, 1)
    rng = np.random.default_rng(3)
    u = 1e-3 * rng.normal(size=coords.shape)
    out = oracle.assemble(coords, conn, u, h0, mat, rp, ci)
    K = _dense(rp, ci, out["csr_vals"])
    x = rng.normal(size=K.shape[0])
    assert np.allclose(onw.spmv(rp, ci, out["csr_vals"], x), K @ x, rtol=1e-13, atol=1e-9)
    bc = np.array([0, 4, 5, 17, 26])
    g = rng.normal(size=bc.size)
    vals, rhs = onw.dirichlet(rp, ci, out["csr_vals"], -out["residual"], bc, g)
    Kd = K.copy()
    Kd[bc, :] = 0.0
    Kd[bc, bc] = 1.0
    assert np.array_equal(_dense(rp, ci, vals), Kd)           # rows replaced, columns untouched
    r2 = -out["residual"].copy(); r2[bc] = g
    assert np.array_equal(rhs, r2)
    xs = onw.linear_solve(rp, ci, vals, rhs)
    assert np.allclose(xs, np.linalg.solve(Kd, r2), rtol=1e-9, atol=1e-14)
    assert np.allclose(xs[bc], g, rtol=1e-12, atol=0)            # identity rows pin the constrained values


def test_patch_solution_homogeneous_deformation():
    """All boundary nodes follow u = A X; the homogeneous field is the exact discrete solution for a homogeneous material,
    elastic or plastic, so Newton from a zero interior guess must return A X at the interior nodes."""
    coords, conn, mat, rp, ci, h0 = _problem(3, 3, 3)
    A = np.array([[0.02, 0.01, -0.004], [0.003, -0.012, 0.006], [-0.005, 0.002, 0.015]])
    exact = coords @ A.T
    on_b = np.any((np.abs(coords) < 1e-12) | (np.abs(coords - 1.0) < 1e-12), axis=1)
    bc = (3 * np.flatnonzero(on_b)[:, None] + np.arange(3)).ravel()
    res = onw.newton_solve(coords, conn, np.zeros_like(coords), h0, mat, rp, ci, bc, exact.ravel()[bc])
    assert res["converged"] and res["stats"]["n_plastic"] == 8 * conn.shape[0]
    assert np.abs(res["u"] - exact).max() < 1e-10


def _uniaxial(delta, desc=None):
    coords, conn, mat, rp, ci, h0 = _problem(2, 2, 2, desc=desc)
    nid = np.arange(coords.shape[0])
    bc, val = [], []
    for sel, comp, v in ((np.abs(coords[:, 0]) < 1e-12, 0, 0.0), (np.abs(coords[:, 0] - 1) < 1e-12, 0, delta),
                         (np.abs(coords[:, 1]) < 1e-12, 1, 0.0), (np.abs(coords[:, 2]) < 1e-12, 2, 0.0)):
        bc += list(3 * nid[sel] + comp); val += [v] * int(sel.sum())
    res = onw.newton_solve(coords, conn, np.zeros_like(coords), h0, mat, rp, ci, np.array(bc), np.array(val))
    assert res["converged"]
    u = res["u"]
    top_y, top_z = np.abs(coords[:, 1] - 1) < 1e-12, np.abs(coords[:, 2] - 1) < 1e-12
    return res, np.log1p(delta), np.log1p(u[top_y, 1]), np.log1p(u[top_z, 2])


def test_hencky_uniaxial_elastic_closed_form():
    """Below yield T = E : ln U, so free lateral faces give ln(lambda_lat) = -nu ln(lambda_ax) exactly (Eq.(7)-(8) :108-113)."""
    res, e_ax, e_y, e_z = _uniaxial(5e-4)
    assert res["stats"]["n_plastic"] == 0
    assert np.allclose(e_y, -0.33 * e_ax, rtol=1e-9) and np.allclose(e_z, -0.33 * e_ax, rtol=1e-9)


def test_plastic_uniaxial_lateral_strains_follow_lankford_r0():
    """Uniaxial tension along material axis 1 beyond yield: the plastic width / thickness strain ratio is the Lankford
    value r0 that produced the Hill ratios (associative flow Eq.(13) :141 + the Lankford conversion, D2)."""
    res, e_ax, e_y, e_z = _uniaxial(0.03)
    assert res["stats"]["n_plastic"] == 64
    h = res["hist_out"].reshape(-1, 7)
    ep = h.mean(axis=0)
    assert np.ptp(h[:, 0]) < 1e-10                                   # homogeneous state
    assert abs(ep[1] / ep[2] - 0.7) < 1e-9                           # eps_p22 / eps_p33 = r0
    sig = 70000.0 * (e_ax - ep[0])                                   # uniaxial stress from the elastic axial log strain
    assert np.allclose(e_y, -0.33 * sig / 70000.0 + ep[1], rtol=1e-8)
    assert np.allclose(e_z, -0.33 * sig / 70000.0 + ep[2], rtol=1e-8)
    # Swift flow stress reached: sigma11 = r11 * sigma_flow(alpha) with r11 = 1 (G2)
    assert abs(sig - 500.0 * (0.01 + h[0, 6]) ** 0.2) < 1e-6 * sig


def clamped_shear_problem():
    """3^3 cube, face x = 0 clamped, face x = 1 displaced by (0.02, 0.01, 0): the paper's benchmark loading (PAPER.md:485,
    left face fixed, right face moved in x and y), inhomogeneous and fully plastic."""
    coords, conn, mat, rp, ci, h0 = _problem(3, 3, 3)
    nid = np.arange(coords.shape[0])
    lf, rt = np.abs(coords[:, 0]) < 1e-12, np.abs(coords[:, 0] - 1) < 1e-12
    bc = np.concatenate([(3 * nid[lf][:, None] + np.arange(3)).ravel(), (3 * nid[rt][:, None] + np.arange(3)).ravel()])
    val = np.concatenate([np.zeros(3 * lf.sum()), np.tile([0.02, 0.01, 0.0], rt.sum())])
    return coords, conn, mat, rp, ci, h0, bc, val


def test_global_newton_converges_quadratically():
    """With the consistent tangent (Eq.(40) :294) the residual norm squares from one iteration to the next once it is small."""
    coords, conn, mat, rp, ci, h0, bc, val = clamped_shear_problem()
    res = onw.newton_solve(coords, conn, np.zeros_like(coords), h0, mat, rp, ci, bc, val)
    n = res["norms"]
    assert res["converged"] and res["stats"]["n_plastic"] > 0.9 * 8 * conn.shape[0]
    k = next(i for i in range(1, len(n)) if n[i] < 1e-2)
    assert n[k + 1] < 1e-4 * n[k], n
    # equilibrium: the internal force of the returned state vanishes on the free DOFs
    out = oracle.assemble(coords, conn, res["u"], h0, mat, rp, ci)
    free = np.setdiff1d(np.arange(3 * coords.shape[0]), bc)
    assert np.abs(out["residual"][free]).max() < 1e-9 * np.abs(out["residual"][bc]).max()
    assert np.allclose(res["u"].ravel()[bc], val, rtol=0, atol=1e-15)


def test_load_path_is_step_size_independent_for_proportional_loading():
    """Pin of oracle.newton.load_path.  Isotropic material (all r = 1), homogeneous isochoric-free uniaxial
    stretch of a patch with lateral faces free: the loading is proportional in fixed principal axes, N is constant along
    the path, and backward Euler is then exact for any step size - so the adaptively stepped path, with whatever
    schedule and cut-backs it takes, must end in the state of one single increment (displacement and history)."""
    desc = dict(synth.configs.SWIFT, r0=1.0, r45=1.0, r90=1.0)
    coords, conn, mat, rp, ci, h0 = _problem(2, 2, 2, desc=desc)
    nid = np.arange(coords.shape[0])
    x0, x1 = np.abs(coords[:, 0]) < 1e-12, np.abs(coords[:, 0] - 1) < 1e-12
    bc = [3 * nid[x0], 3 * nid[x1]]                                   # u_x on both x faces
    bc += [np.array([3 * n + 1]) for n in nid[np.abs(coords[:, 1]) < 1e-12]]   # symmetry planes y = 0, z = 0
    bc += [np.array([3 * n + 2]) for n in nid[np.abs(coords[:, 2]) < 1e-12]]
    bc = np.concatenate(bc)
    full = np.zeros(bc.size)
    full[x0.sum():x0.sum() + x1.sum()] = 0.04                          # 4 % stretch: well into the plastic range
    one = onw.newton_solve(coords, conn, np.zeros_like(coords), h0, mat, rp, ci, bc, full, max_newton=30)
    assert one["converged"] and one["stats"]["n_plastic"] == 8 * conn.shape[0]
    # a schedule that starts too ambitiously for 3 Newton iterations: it must cut back, then grow again
    path = onw.load_path(coords, conn, h0, mat, rp, ci, bc, full, dt0=1.0, dt_min=1e-3, dt_max=0.4, grow=1.5, cut=0.5, grow_below=4,
                         max_newton=3, extrapolate=1)
    assert path["completed"] and path["rejected"] >= 1 and path["steps"] >= 3
    assert np.all(np.diff(path["ts"]) > 0) and abs(path["ts"][-1] - 1.0) < 1e-12
    assert np.allclose(path["u"], one["u"], rtol=0, atol=1e-9 * np.abs(one["u"]).max())
    assert np.allclose(path["hist"], one["hist_out"], rtol=0, atol=1e-9 * np.abs(one["hist_out"]).max())
    # no extrapolation and quadratic extrapolation reach the same state
    for ex in (0, 2):
        p2 = onw.load_path(coords, conn, h0, mat, rp, ci, bc, full, dt0=0.2, dt_min=1e-3, dt_max=0.3, extrapolate=ex, max_newton=12)
        assert p2["completed"] and np.allclose(p2["u"], one["u"], rtol=0, atol=1e-9 * np.abs(one["u"]).max())
    # a path that cannot be completed reports where it stopped
    p3 = onw.load_path(coords, conn, h0, mat, rp, ci, bc, full, dt0=1.0, dt_min=0.6, dt_max=1.0, max_newton=1)
    assert not p3["completed"] and p3["t"] == 0.0 and p3["rejected"] == 1
