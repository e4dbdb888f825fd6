"""GPU parity of SURVEY.md §8(f) NEXT-1 (fem_spmv, fem_apply_dirichlet, fem_bicgstab, fem_newton_solve) against
oracle/newton.py on the same seeded inputs.  Tolerances: Dirichlet rows bit-exact (pure placement); y = K x relative L2
<= 1e-13 (summation order differs); linear solve: relative L2 against the direct solve <= 1e-7 with rtol = 1e-12
(cond(K) of these meshes ~1e4 times the residual tolerance); Newton: converged displacement <= 1e-8 relative."""
import numpy as np
import pytest

import synth
from parity_util import rel_l2
from test_oracle_newton import clamped_shear_problem, _problem

pytestmark = pytest.mark.gpu


def _ctx(coords, conn, fbar=0):
    import torch
    import paper_2606_17390_b200 as fem
    dev = torch.device("cuda:0")
    ctx = fem.FemContext(torch.from_numpy(coords).to(dev), torch.from_numpy(conn).to(dev), fbar=fbar)
    ctx.build_csr_pattern()
    return ctx, dev


def _assembled(cfg, fbar=0):
    import torch
    import paper_2606_17390_b200 as fem
    import oracle
    ctx, dev = _ctx(cfg["coords"], cfg["conn"], fbar)
    ne = cfg["conn"].shape[0]
    mat = torch.from_numpy(fem.mat_from_desc(cfg["matdesc"], ne).ravel()).to(dev)
    res, vals, hout, _ = ctx.assemble(torch.from_numpy(cfg["u"].ravel()).to(dev), torch.from_numpy(cfg["hist_in"].ravel()).to(dev), mat)
    rp, ci, _ = oracle.pattern(cfg["coords"].shape[0], cfg["conn"], with_slots=False)
    return ctx, dev, res, vals, rp, ci


@pytest.mark.parametrize("fbar", [0, 1])
def test_spmv_and_dirichlet_match_oracle(fbar):
    import torch
    import oracle.newton as onw
    cfg = synth.make_config(4, n=10)              # irregular connectivity, ragged neighbour counts
    ctx, dev, res, vals, rp, ci = _assembled(cfg, fbar)
    rng = np.random.default_rng(11)
    x = rng.normal(size=ctx.n_rows)
    y = ctx.spmv(vals, torch.from_numpy(x).to(dev))
    v_np = vals.cpu().numpy()
    assert rel_l2(y.cpu().numpy(), onw.spmv(rp, ci, v_np, x)) <= 1e-13
    bc = np.unique(rng.integers(0, ctx.n_rows, size=300)).astype(np.int32)
    g = rng.normal(size=bc.size)
    rhs = -res.clone()
    ctx.apply_dirichlet(torch.from_numpy(bc).to(dev), vals, rhs, torch.from_numpy(g).to(dev))
    ov, orhs = onw.dirichlet(rp, ci, v_np, -res.cpu().numpy(), bc, g)
    assert np.array_equal(vals.cpu().numpy(), ov) and np.array_equal(rhs.cpu().numpy(), orhs)
    # rhs = NULL and bc_rhs = NULL variants
    vals2 = torch.from_numpy(v_np).to(dev)
    ctx.apply_dirichlet(torch.from_numpy(bc).to(dev), vals2)
    assert np.array_equal(vals2.cpu().numpy(), ov)


@pytest.mark.parametrize("case", ["elastic", "plastic", "plastic-fbar"])
def test_bicgstab_against_direct_solve(case):
    """elastic: the linear-elastic stiffness of a cube clamped on one face (the workload of Table F1);
    plastic: the consistent tangent of a homogeneous, fully plastic equilibrium state u = A X, both x faces constrained.
    (The tangent of the raw config-3 displacement field, which is no equilibrium state, has a negative eigenvalue; neither
    this solver nor SciPy's BiCGSTAB converges on it, so it is no test case.)"""
    import torch
    import oracle.newton as onw
    cfg = synth.make_config(3, n=14)
    if case == "elastic":
        cfg = dict(cfg, u=np.zeros_like(cfg["u"]))
    else:
        A = np.array([[0.02, 0.01, -0.004], [0.003, -0.012, 0.006], [-0.005, 0.002, 0.015]])
        cfg = dict(cfg, u=cfg["coords"] @ A.T)
    ctx, dev, res, vals, rp, ci = _assembled(cfg, 1 if case.endswith("fbar") else 0)
    coords = cfg["coords"]
    sel = np.abs(coords[:, 0]) < 1e-12
    if case != "elastic":
        sel |= np.abs(coords[:, 0] - 1) < 1e-12
    bc = (3 * np.flatnonzero(sel)[:, None] + np.arange(3)).ravel().astype(np.int32)
    rhs = torch.from_numpy(np.random.default_rng(5).normal(size=ctx.n_rows)).to(dev)
    ctx.apply_dirichlet(torch.from_numpy(bc).to(dev), vals, rhs)
    x, iters, relres, ok = ctx.bicgstab(vals, rhs, rtol=1e-12, max_iter=20000)
    assert ok and relres <= 1e-10, (iters, relres)
    xo = onw.linear_solve(rp, ci, vals.cpu().numpy(), rhs.cpu().numpy())
    assert rel_l2(x.cpu().numpy(), xo) <= 1e-7, (iters, relres)
    x2, it2, _, _ = ctx.bicgstab(vals, rhs, rtol=1e-12, max_iter=20000)
    assert it2 == iters and torch.equal(x, x2)                       # fixed reduction order: bit-identical
    if not case.endswith("fbar"):
        # CG on the symmetric reduced system: the guess carries the prescribed values on the constrained DOFs
        xg = torch.zeros_like(rhs)
        xg[torch.from_numpy(bc.astype(np.int64)).to(dev)] = rhs[torch.from_numpy(bc.astype(np.int64)).to(dev)]
        xc, itc, rrc, okc = ctx.pcg(vals, rhs, x=xg.clone(), rtol=1e-12, max_iter=20000)
        assert okc and rrc <= 1e-10 and rel_l2(xc.cpu().numpy(), xo) <= 1e-7, (itc, rrc)
        xc2, itc2, _, _ = ctx.pcg(vals, rhs, x=xg.clone(), rtol=1e-12, max_iter=20000)
        assert itc2 == itc and torch.equal(xc, xc2)
        # mixed precision: fp32 copy of K inside the iteration, fp64 residuals + refinement: same acceptance test, same solution
        ctx.set_mixed_precision(True)
        xm, itm, rrm, okm = ctx.pcg(vals, rhs, x=xg.clone(), rtol=1e-12, max_iter=20000)
        assert okm and rrm <= 1e-12 and rel_l2(xm.cpu().numpy(), xo) <= 1e-7, (itm, rrm)
        assert itm <= 2 * itc, (itm, itc)
        xm2, itm2, _, _ = ctx.pcg(vals, rhs, x=xg.clone(), rtol=1e-12, max_iter=20000)
        assert itm2 == itm and torch.equal(xm, xm2)
        xl, itl, rrl, okl = ctx.pcg(vals, rhs, x=xg.clone(), rtol=1e-4, max_iter=20000)     # loose tolerance: one round
        assert okl and rrl <= 1e-4 and itl < itm
        ctx.set_mixed_precision(False)
    # zero right-hand side and iteration cap
    x0, it0, rr0, ok0 = ctx.bicgstab(vals, torch.zeros_like(rhs), x=torch.ones_like(rhs))
    assert ok0 and it0 == 0 and float(x0.abs().max()) == 0.0
    _, it1, _, ok1 = ctx.bicgstab(vals, rhs, rtol=1e-12, max_iter=3)
    assert (not ok1) and it1 == 3


@pytest.mark.parametrize("fbar,solver", [(0, 0), (0, 1), (1, 0)])
def test_newton_solve_matches_oracle(fbar, solver):
    import torch
    import paper_2606_17390_b200 as fem
    import oracle.newton as onw
    coords, conn, omat, rp, ci, h0, bc, val = clamped_shear_problem()
    ctx, dev = _ctx(coords, conn, fbar)
    ne = conn.shape[0]
    mat = torch.from_numpy(fem.mat_from_desc(dict(synth.configs.SWIFT), ne).ravel()).to(dev)
    u = torch.zeros(coords.size, dtype=torch.float64, device=dev)
    u, hout, rep = ctx.newton_solve(u, torch.from_numpy(h0.ravel()).to(dev), mat, torch.from_numpy(bc.astype(np.int32)).to(dev),
                                    torch.from_numpy(val).to(dev), lin_rtol=1e-12, linear_solver=solver)
    o = onw.newton_solve(coords, conn, np.zeros_like(coords), h0, omat, rp, ci, bc, val, fbar=fbar)
    assert rep["converged"] and o["converged"] and rep["lin_failures"] == 0
    assert rep["newton_iters"] == o["newton_iters"], (rep, o["norms"])
    assert rel_l2(u.cpu().numpy(), o["u"]) <= 1e-8
    assert rel_l2(hout.cpu().numpy(), o["hist_out"]) <= 1e-7
    assert rep["last_stats"]["n_plastic"] == o["stats"]["n_plastic"]
    assert np.array_equal(u.cpu().numpy()[bc], val)                 # prescribed values hit exactly


def test_newton_patch_solution_and_error_paths():
    import torch
    import paper_2606_17390_b200 as fem
    coords, conn, omat, rp, ci, h0 = _problem(4, 3, 3)
    ctx, dev = _ctx(coords, conn)
    ne = conn.shape[0]
    A = np.array([[0.02, 0.01, -0.004], [0.003, -0.012, 0.006], [-0.005, 0.002, 0.015]])
    exact = coords @ A.T
    on_b = np.any((np.abs(coords) < 1e-12) | (np.abs(coords - 1.0) < 1e-12), axis=1)
    bc = (3 * np.flatnonzero(on_b)[:, None] + np.arange(3)).ravel().astype(np.int32)
    mat = torch.from_numpy(fem.mat_from_desc(dict(synth.configs.SWIFT), ne).ravel()).to(dev)
    hin = torch.zeros(56 * ne, dtype=torch.float64, device=dev)
    u = torch.zeros(coords.size, dtype=torch.float64, device=dev)
    u, _, rep = ctx.newton_solve(u, hin, mat, torch.from_numpy(bc).to(dev), torch.from_numpy(exact.ravel()[bc]).to(dev))
    assert rep["converged"] and np.abs(u.cpu().numpy() - exact.ravel()).max() < 1e-9   # homogeneous-deformation patch solution
    # a failed increment (iteration cap) leaves u at its entry value
    u_in = torch.from_numpy(1e-3 * np.random.default_rng(2).normal(size=coords.size)).to(dev)
    u2, _, rep2 = ctx.newton_solve(u_in.clone(), hin, mat, torch.from_numpy(bc).to(dev), torch.from_numpy(exact.ravel()[bc]).to(dev),
                                   max_newton=1)
    assert not rep2["converged"] and rep2["newton_iters"] == 1 and torch.equal(u2, u_in)
    w = ctx.lincomb(2.0, u_in, -0.5, u)
    assert torch.equal(w, torch.addcmul(-0.5 * u, u_in, torch.full_like(u_in, 2.0))) or rel_l2(w.cpu().numpy(), (2.0 * u_in - 0.5 * u).cpu().numpy()) <= 1e-16
    bad = torch.tensor([0, 3 * coords.shape[0]], dtype=torch.int32, device=dev)      # DOF out of range
    with pytest.raises(fem.FemError):
        ctx.newton_solve(u, hin, mat, bad, torch.zeros(2, dtype=torch.float64, device=dev))
    with pytest.raises(fem.FemError):
        ctx.apply_dirichlet(bad, torch.zeros(ctx.nnz, dtype=torch.float64, device=dev))


def test_load_path_with_history_matches_oracle():
    """Three load steps on the clamped cube, converged state and history carried from step to step (the protocol of the
    paper's benchmark): displacement and history after the last step against the oracle's own path."""
    import torch
    import paper_2606_17390_b200 as fem
    import oracle.newton as onw
    coords, conn, omat, rp, ci, h0, bc, val = clamped_shear_problem()
    ctx, dev = _ctx(coords, conn)
    ne = conn.shape[0]
    mat = torch.from_numpy(fem.mat_from_desc(dict(synth.configs.SWIFT), ne).ravel()).to(dev)
    bc_d = torch.from_numpy(bc.astype(np.int32)).to(dev)
    u = torch.zeros(coords.size, dtype=torch.float64, device=dev)
    h_a = torch.zeros(56 * ne, dtype=torch.float64, device=dev)
    uo, ho = np.zeros_like(coords), h0.copy()
    for frac in (0.3, 0.7, 1.0):
        u, h_b, rep = ctx.newton_solve(u, h_a, mat, bc_d, torch.from_numpy(val * frac).to(dev), lin_rtol=1e-12)
        assert rep["converged"]
        h_a = h_b
        o = onw.newton_solve(coords, conn, uo, ho, omat, rp, ci, bc, val * frac)
        assert o["converged"]
        uo, ho = o["u"], o["hist_out"]
    assert rel_l2(u.cpu().numpy(), uo) <= 1e-8 and rel_l2(h_a.cpu().numpy(), ho) <= 1e-7
    assert float(h_a.view(-1, 7)[:, 6].max()) > 0.01          # the path is well into the plastic range


@pytest.mark.parametrize("fbar,extrapolate", [(0, 1), (0, 2), (1, 1)])
def test_fem_load_path_matches_oracle_loop(fbar, extrapolate):
    """fem_load_path (the adaptive load stepping of PAPER.md:306 behind one C-ABI call) against the same loop written with
    oracle functions only (oracle.newton.load_path): a schedule that starts too ambitiously for the Newton cap, so it has
    to cut back and grow again.  Same accepted load fractions, same number of rejected steps, same final state."""
    import torch
    import paper_2606_17390_b200 as fem
    import oracle.newton as onw
    coords, conn, omat, rp, ci, h0, bc, val = clamped_shear_problem()
    ctx, dev = _ctx(coords, conn, fbar)
    ne = conn.shape[0]
    mat = torch.from_numpy(fem.mat_from_desc(dict(synth.configs.SWIFT), ne).ravel()).to(dev)
    u = torch.zeros(coords.size, dtype=torch.float64, device=dev)
    hist = torch.zeros(56 * ne, dtype=torch.float64, device=dev)
    kw = dict(dt0=0.7, dt_min=1e-3, dt_max=0.5, grow=1.5, cut=0.5, grow_below=5, extrapolate=extrapolate)
    rc, rep, ts = ctx.load_path(u, hist, mat, torch.from_numpy(bc.astype(np.int32)).to(dev), torch.from_numpy(val).to(dev),
                                newton=dict(rtol=1e-8, atol=1e-10, max_newton=4, lin_rtol=1e-12, lin_max_iter=20000), **kw)
    o = onw.load_path(coords, conn, h0, omat, rp, ci, bc, val, fbar=fbar, rtol=1e-8, atol=1e-10, max_newton=4, **kw)
    assert rc == 0 and o["completed"] and rep["t_reached"] == 1.0
    assert rep["rejected"] == o["rejected"] >= 1 and rep["steps"] == o["steps"] >= 3
    assert np.allclose(ts, o["ts"], rtol=0, atol=1e-15)
    assert rep["newton_iters_total"] == o["newton_iters_total"]
    assert rel_l2(u.cpu().numpy(), o["u"]) <= 1e-8 and rel_l2(hist.cpu().numpy(), o["hist"]) <= 1e-7
    assert float(hist.view(-1, 7)[:, 6].max()) > 0.01
    # a second path on the same context (workspace reuse) from the same start gives the same bits
    u2 = torch.zeros_like(u); hist2 = torch.zeros_like(hist)
    rc2, rep2, ts2 = ctx.load_path(u2, hist2, mat, torch.from_numpy(bc.astype(np.int32)).to(dev), torch.from_numpy(val).to(dev),
                                   newton=dict(rtol=1e-8, atol=1e-10, max_newton=4, lin_rtol=1e-12, lin_max_iter=20000), **kw)
    assert rc2 == 0 and ts2 == ts and torch.equal(u2, u) and torch.equal(hist2, hist)


def test_balanced_state_with_local_nonconvergence_is_rejected():
    """an increment whose balanced state holds local solves that hit kmax is no root of the discrete problem.
    With the local iteration cap at 1 the return map is cut short at every plastic point: fem_newton_solve must report
    physics trouble, return FEM_ERR_NOCONV and restore u; fem_load_path must cut back and finally give up, leaving the
    last accepted state.  Overlapping history buffers are refused."""
    import torch
    import paper_2606_17390_b200 as fem
    coords, conn, omat, rp, ci, h0, bc, val = clamped_shear_problem()
    dev = torch.device("cuda:0")
    ne = conn.shape[0]
    ctx = fem.FemContext(torch.from_numpy(coords).to(dev), torch.from_numpy(conn).to(dev), kmax=1)
    ctx.build_csr_pattern()
    mat = torch.from_numpy(fem.mat_from_desc(dict(synth.configs.SWIFT), ne).ravel()).to(dev)
    bc_d, val_d = torch.from_numpy(bc.astype(np.int32)).to(dev), torch.from_numpy(val).to(dev)
    hin = torch.zeros(56 * ne, dtype=torch.float64, device=dev)
    u_in = torch.zeros(coords.size, dtype=torch.float64, device=dev)
    u, _, rep = ctx.newton_solve(u_in.clone(), hin, mat, bc_d, val_d, lin_rtol=1e-12, rtol=1e-7, max_newton=40)
    assert rep["last_stats"]["n_nonconverged"] > 0
    assert rep["physics_trouble"] and not rep["converged"] and torch.equal(u, u_in)
    rc, prep, ts = ctx.load_path(u_in.clone(), hin.clone(), mat, bc_d, val_d, dt0=0.5, dt_min=0.2, dt_max=0.5,
                                 newton=dict(lin_rtol=1e-12, rtol=1e-7, max_newton=40))
    assert rc == -11 and prep["rejected_physics"] >= 1 and prep["steps"] == 0 and prep["t_reached"] == 0.0
    with pytest.raises(fem.FemError) as ei:            # hist_out overlapping hist_in (offset view of the same buffer)
        big = torch.zeros(56 * ne + 8, dtype=torch.float64, device=dev)
        ctx.newton_solve(u_in.clone(), big[:56 * ne], mat, bc_d, val_d, hist_out=big[8:])
    assert ei.value.code == -9
    ctx.close()


def test_barlat_exponent_outside_the_supported_set_is_reported():
    """an exponent m that is not an even integer in 2..16 must not index past the coefficient tables: it is clamped
    inside the call and the call reports FEM_ERR_ARG when statistics are requested."""
    import torch
    import paper_2606_17390_b200 as fem
    cfg = synth.make_config(1)
    dev = torch.device("cuda:0")
    ctx = fem.FemContext(torch.from_numpy(cfg["coords"]).to(dev), torch.from_numpy(cfg["conn"]).to(dev))
    ctx.build_csr_pattern()
    mat = torch.tensor([70000.0, 0.33, 1, 1, 1, 1, 1, 1, 1.0, 500.0, 0.01, 0.2, 1.0, 0.0, 0.0, 0.0], dtype=torch.float64, device=dev)
    u = torch.from_numpy(cfg["u"].ravel()).to(dev); h = torch.from_numpy(cfg["hist_in"].ravel()).to(dev)
    good = torch.tensor([1.0] * 18 + [8.0, 0.0], dtype=torch.float64, device=dev)
    r8, v8, _, st = ctx.assemble(u, h, mat, want_stats=True, barlat=good)
    assert st["n_nonfinite"] == 0
    for m in (40.0, 7.0, 0.0, float("nan")):
        bad = good.clone(); bad[18] = m
        with pytest.raises(fem.FemError) as ei:
            ctx.assemble(u, h, mat, want_stats=True, barlat=bad)
        assert ei.value.code == -2
        r, v, _, _ = ctx.assemble(u, h, mat, barlat=bad)         # without statistics: clamped, finite, no fault
        torch.cuda.synchronize()
        assert bool(torch.isfinite(v).all())
    ctx.close()
