"""GPU parity of fem_assemble_vjp against oracle/sens.py on the same seeded inputs, through the C ABI.

Tolerances: the VJPs are products of the quantities the north_star bounds at 1e-10 (tangent, history) with
the cotangents, so g_u and g_hist_in are held to rel. L2 <= 1e-9; g_mat is a sum over all Gauss points with cancellation, so
every entry is held to 1e-9 of the sum of |element contributions| the oracle reports (g_mat_abs).  Properties that hold at
any size (K lambda, linearity, elastic history leg, determinism) are checked at config 3's full size."""
import numpy as np
import pytest

from parity_util import rel_l2

pytestmark = pytest.mark.gpu

TOL = 1e-9


def _small_problem(seed=5, n=(3, 2, 2), per_elem=False, voce=False, amp=0.006, hist=True):
    import oracle
    import synth
    from synth import mesh
    coords, conn = mesh.structured_hex_mesh(*n)
    rng = np.random.default_rng(seed)
    coords = coords + 0.04 * rng.uniform(-1, 1, size=coords.shape) / max(n)
    ne = conn.shape[0]
    base = oracle.mat_from_desc(dict(synth.configs.SWIFT), 1)[0]
    nm = ne if per_elem else 1
    mat = np.tile(base, (nm, 1))
    if voce:
        mat[:, 8], mat[:, 9], mat[:, 10], mat[:, 11] = 0.0, 200.0, 150.0, 12.0
    if per_elem:
        mat[:, 2:8] *= 1 + 0.1 * rng.uniform(-1, 1, size=(nm, 6))
        mat[:, 9] *= 1 + 0.1 * rng.uniform(-1, 1, size=nm)
        q = rng.normal(size=(nm, 4)); mat[:, 12:16] = q / np.linalg.norm(q, axis=1)[:, None]
    A = rng.normal(size=(3, 3)); A *= amp / np.linalg.norm(A)
    u = (coords @ A.T) * (0.15 + coords[:, :1]) + 2e-4 * rng.normal(size=coords.shape)
    h = np.zeros((ne, 8, 7))
    if hist:
        h[..., 6] = 0.01 * rng.uniform(size=(ne, 8))
        d = rng.normal(size=(ne, 8, 6)) * 2e-4
        d[..., :3] -= d[..., :3].mean(axis=-1, keepdims=True)
        h[..., :6] = d
    lam = rng.normal(size=coords.shape)
    mu = rng.normal(size=(ne, 8, 7)) * np.array([1e3] * 6 + [1e2])
    return dict(coords=coords, conn=conn, mat=mat, u=u, h=h, lam=lam, mu=mu)


def _ctx(coords, conn):
    import torch
    import paper_2606_17390_b200 as fem
    dev = torch.device("cuda:0")
    ctx = fem.FemContext(torch.from_numpy(np.ascontiguousarray(coords)).to(dev), torch.from_numpy(np.ascontiguousarray(conn)).to(dev))
    ctx.build_csr_pattern()
    return ctx


def _gpu_vjp(ctx, p, lam=True, mu=True, **kw):
    import torch
    dev = ctx.device
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).ravel()).to(dev)
    g_u, g_h, g_m = ctx.assemble_vjp(t(p["u"]), t(p["h"]), t(p["mat"]), t(p["lam"]) if lam else None, t(p["mu"]) if mu else None, **kw)
    torch.cuda.synchronize()
    c = lambda x: None if x is None else x.cpu().numpy()
    return c(g_u), c(g_h), c(g_m)


def _check_mat(g_m, o):
    scale = np.maximum(o["g_mat_abs"], 1e-300)
    err = np.abs(g_m - o["g_mat"]) / scale
    err[o["g_mat_abs"] == 0.0] = np.abs(g_m)[o["g_mat_abs"] == 0.0]
    assert err.max() <= TOL, err.max()


@pytest.mark.parametrize("variant", ["uniform_swift", "per_elem_rotated_voce", "uniform_voce_virgin"])
def test_vjp_small_meshes(variant):
    import oracle.sens as osn
    p = _small_problem(per_elem=variant == "per_elem_rotated_voce", voce=variant != "uniform_swift", hist=variant != "uniform_voce_virgin")
    ctx = _ctx(p["coords"], p["conn"])
    o = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], p["mu"])
    g_u, g_h, g_m = _gpu_vjp(ctx, p)
    assert rel_l2(g_u, o["g_u_full"]) <= TOL
    assert rel_l2(g_h, o["g_hist_in"]) <= TOL
    _check_mat(g_m, o)
    assert np.all(g_m[:, [8, 12, 13, 14, 15]] == 0.0)
    # history leg alone (lam = NULL) and residual leg alone (mu = NULL)
    g_u2, g_h2, g_m2 = _gpu_vjp(ctx, p, lam=False)
    assert rel_l2(g_u2, o["g_u"]) <= TOL
    o3 = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], None)
    g_u3, g_h3, g_m3 = _gpu_vjp(ctx, p, mu=False)
    assert rel_l2(g_u3, o3["g_u_full"]) <= TOL and rel_l2(g_h3, o3["g_hist_in"]) <= TOL
    _check_mat(g_m3, o3)
    # outputs may be skipped one by one
    a, b, c = _gpu_vjp(ctx, p, want_u=False, want_mat=False)
    assert a is None and c is None and np.array_equal(b, g_h)
    a, b, c = _gpu_vjp(ctx, p, want_hist=False)
    assert b is None and np.array_equal(a, g_u) and np.array_equal(c, g_m)
    ctx.close()


def test_vjp_config1_and_config2():
    """Configs 1 (whole mesh) and 2 (plate, ~50 % plastic, non-zero history): g_u and g_mat need every element, so config 2 is
    compared on a 12x12x4 corner of the plate cut out as its own mesh (same field, same history), plus sampled elements of
    the whole plate for g_hist_in."""
    import oracle
    import oracle.sens as osn
    import synth
    for k in (1, 2):
        cfg = synth.make_config(k)
        ne = cfg["conn"].shape[0]
        rng = np.random.default_rng(100 + k)
        p = dict(coords=cfg["coords"], conn=cfg["conn"], u=cfg["u"], h=cfg["hist_in"].reshape(ne, 8, 7),
                 mat=oracle.mat_from_desc(cfg["matdesc"], ne), lam=rng.normal(size=cfg["coords"].shape),
                 mu=rng.normal(size=(ne, 8, 7)) * np.array([1e3] * 6 + [1e2]))
        ctx = _ctx(p["coords"], p["conn"])
        g_u, g_h, g_m = _gpu_vjp(ctx, p)
        if k == 1:
            o = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], p["mu"])
            assert rel_l2(g_u, o["g_u_full"]) <= TOL and rel_l2(g_h, o["g_hist_in"]) <= TOL
            _check_mat(g_m, o)
        else:
            el = np.sort(rng.choice(ne, 160, replace=False))
            o = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], p["mu"], elems=el)
            assert rel_l2(g_h.reshape(ne, 8, 7)[el], o["g_hist_in"][el]) <= TOL
            # sub-mesh: elements with ix, iy < 12 of the 40x40x4 plate (element id = ix + 40 iy + 1600 iz)
            ids = np.array([ix + 40 * iy + 1600 * iz for iz in range(4) for iy in range(12) for ix in range(12)])
            nodes, inv = np.unique(cfg["conn"][ids], return_inverse=True)
            sp = dict(coords=p["coords"][nodes], conn=inv.reshape(-1, 8).astype(np.int32), u=p["u"].reshape(-1, 3)[nodes],
                      h=p["h"][ids], mat=p["mat"], lam=p["lam"][nodes], mu=p["mu"][ids])
            sctx = _ctx(sp["coords"], sp["conn"])
            s_u, s_h, s_m = _gpu_vjp(sctx, sp)
            so = osn.assemble_vjp(sp["coords"], sp["conn"], sp["u"], sp["h"], sp["mat"], sp["lam"], sp["mu"])
            assert rel_l2(s_u, so["g_u_full"]) <= TOL and rel_l2(s_h, so["g_hist_in"]) <= TOL
            _check_mat(s_m, so)
            sctx.close()
        ctx.close()


def test_vjp_large_strain_levels():
    """Strain sweep of config 5's form on a small mesh: peak strain up to 0.3 (divided differences far from the series
    branch, many return-map iterations) and 1e-5 (all-elastic, eigenvalues of C within 1e-5 of each other)."""
    import oracle
    import oracle.sens as osn
    for amp, seed in ((0.3, 21), (0.05, 22), (1e-5, 23)):
        p = _small_problem(seed=seed, n=(2, 2, 2), amp=amp, hist=amp > 1e-4)
        if amp <= 1e-4:
            p["u"] = p["u"] * 0 + (p["coords"] @ (amp * np.array([[1.0, 0.2, 0], [0, -0.4, 0.1], [0.3, 0, 0.5]])).T)
        ctx = _ctx(p["coords"], p["conn"])
        o = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], p["mu"])
        g_u, g_h, g_m = _gpu_vjp(ctx, p)
        assert rel_l2(g_u, o["g_u_full"]) <= TOL, amp
        assert rel_l2(g_h, o["g_hist_in"]) <= TOL, amp
        _check_mat(g_m, o)
        ctx.close()


def test_vjp_errors_and_edge_cases():
    import torch
    import paper_2606_17390_b200 as fem
    p = _small_problem(n=(2, 2, 2))
    dev = torch.device("cuda:0")
    ctx = fem.FemContext(torch.from_numpy(p["coords"]).to(dev), torch.from_numpy(p["conn"]).to(dev))
    with pytest.raises(fem.FemError):      # no pattern yet
        _gpu_vjp(ctx, p)
    ctx.close()
    ctx = _ctx(p["coords"], p["conn"])
    with pytest.raises(fem.FemError):      # constrained DOF out of range
        t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).ravel()).to(dev)
        ctx.adjoint_step(t(p["u"]), t(p["h"]), t(p["mat"]), torch.full((3,), 10 ** 6, dtype=torch.int32, device=dev))
    ctx.close()
    # zero cotangents give zero gradients; zero displacement and virgin history (repeated eigenvalues of C, all elastic)
    ctx = _ctx(p["coords"], p["conn"])
    g_u, g_h, g_m = _gpu_vjp(ctx, p, lam=False, mu=False)
    assert not g_u.any() and not g_h.any() and not g_m.any()
    p0 = dict(p, u=np.zeros_like(p["u"]), h=np.zeros_like(p["h"]))
    import oracle.sens as osn
    o = osn.assemble_vjp(p0["coords"], p0["conn"], p0["u"], p0["h"], p0["mat"], p0["lam"], p0["mu"])
    g_u, g_h, g_m = _gpu_vjp(ctx, p0)
    assert rel_l2(g_u, o["g_u_full"]) <= TOL and rel_l2(g_h, o["g_hist_in"]) <= TOL
    _check_mat(g_m, o)
    ctx.close()


def test_vjp_full_size_properties_and_samples():
    """Config 3 (1M elements) in one call: K lambda from the library's own tangent (K symmetric), linearity in
    the cotangents, the history leg at elastic points, bit-identical repeats, and sampled elements / nodes against the oracle."""
    import torch
    import oracle
    import oracle.sens as osn
    import synth
    import paper_2606_17390_b200 as fem
    cfg = synth.make_config(3)
    ne, nn = cfg["conn"].shape[0], cfg["coords"].shape[0]
    dev = torch.device("cuda:0")
    ctx = _ctx(cfg["coords"], cfg["conn"])
    g = torch.Generator(device="cpu"); g.manual_seed(3)
    lam = torch.randn(3 * nn, dtype=torch.float64, generator=g).to(dev)
    mu = (torch.randn(ne, 8, 7, dtype=torch.float64, generator=g) * torch.tensor([1e3] * 6 + [1e2], dtype=torch.float64)).reshape(-1).to(dev)
    u = torch.from_numpy(cfg["u"].ravel()).to(dev); h = torch.from_numpy(cfg["hist_in"].ravel()).to(dev)
    mat1 = torch.from_numpy(fem.mat_from_desc(cfg["matdesc"], ne).ravel()).to(dev)
    res, vals, hout, _ = ctx.assemble(u, h, mat1)
    a_u, a_h, a_m = ctx.assemble_vjp(u, h, mat1, lam, None)
    Kl = ctx.spmv(vals, lam)
    assert float(torch.linalg.norm(a_u - Kl) / torch.linalg.norm(Kl)) <= 1e-10
    b_u, b_h, b_m = ctx.assemble_vjp(u, h, mat1, None, mu)
    c_u, c_h, c_m = ctx.assemble_vjp(u, h, mat1, lam, mu)
    for x, y, z in ((a_u, b_u, c_u), (a_h, b_h, c_h)):
        assert float(torch.linalg.norm(x + y - z) / torch.linalg.norm(z)) <= 1e-12
    assert float(torch.max(torch.abs(a_m + b_m - c_m) / (torch.abs(a_m) + torch.abs(b_m) + 1e-300))) <= 1e-9
    elastic = (hout.view(ne, 8, 7)[..., 6] == h.view(ne, 8, 7)[..., 6])
    assert 0.2 < float(elastic.double().mean()) < 0.4
    assert float(torch.max(torch.abs(b_h.view(ne, 8, 7)[elastic] - mu.view(ne, 8, 7)[elastic]))) <= 1e-9 * 1e3
    d_u, d_h, d_m = ctx.assemble_vjp(u, h, mat1, lam, mu)
    assert torch.equal(c_u, d_u) and torch.equal(c_h, d_h) and torch.equal(c_m, d_m)
    # dR/dE = R/E at any state (E scales the stress at fixed nu only where every point is elastic) -> instead: Euler's relation
    # for the degree-1 homogeneity of R in (E, h0) for Swift: R(sE, sK) = s R  =>  E dR/dE + K dR/dK = R
    m0 = fem.mat_from_desc(cfg["matdesc"], ne).ravel()
    assert abs(float(a_m[0, 0] * m0[0] + a_m[0, 9] * m0[9]) - float(res @ lam)) <= 1e-9 * float(torch.abs(res) @ torch.abs(lam))
    # samples against the oracle: per-element material records (n_mat = n_elems) so that g_mat is per element
    rng = np.random.default_rng(7)
    el = np.sort(rng.choice(ne, 48, replace=False))
    matn = torch.from_numpy(np.tile(m0, (ne, 1)).ravel()).to(dev)
    e_u, e_h, e_m = ctx.assemble_vjp(u, h, matn, lam, mu)
    assert torch.equal(e_u, c_u) and torch.equal(e_h, c_h)
    lam_n, mu_n = lam.cpu().numpy().reshape(nn, 3), mu.cpu().numpy().reshape(ne, 8, 7)
    o = osn.assemble_vjp(cfg["coords"], cfg["conn"], cfg["u"], cfg["hist_in"], np.tile(m0, (ne, 1)), lam_n, mu_n, elems=el)
    assert rel_l2(e_h.cpu().numpy().reshape(ne, 8, 7)[el], o["g_hist_in"][el]) <= TOL
    gm = e_m.cpu().numpy()[el]
    assert np.max(np.abs(gm - o["g_mat"][el]) / np.maximum(o["g_mat_abs"][el].max(axis=0), 1e-300)) <= TOL
    # the uniform-material gradient is the sum of the per-element ones
    assert float(torch.max(torch.abs(e_m.sum(dim=0) - c_m[0]) / (torch.abs(e_m).sum(dim=0) + 1e-300))) <= 1e-12
    # sampled nodes: g_u of a node needs its (up to 8) elements
    nodes = rng.choice(nn, 12, replace=False)
    els = np.unique(np.flatnonzero(np.isin(cfg["conn"], nodes).any(axis=1)))
    o2 = osn.assemble_vjp(cfg["coords"], cfg["conn"], cfg["u"], cfg["hist_in"], m0.reshape(1, 16), lam_n, mu_n, elems=els)
    gu = c_u.cpu().numpy().reshape(nn, 3)[nodes]
    assert rel_l2(gu, o2["g_u_full"][nodes]) <= TOL
    ctx.close()


@pytest.mark.parametrize("fbar", [0, 1])
def test_adjoint_gradient_of_load_path_matches_oracle(fbar):
    """Alg. 1 end to end on the GPU: two load increments with fem_newton_solve, then backwards per step
    Eq.(51) K^T lam = -(dJ/du)^T - (dh/du)^T mu by fem_pcg on the row-eliminated tangent, Eq.(49) by fem_assemble_vjp with the
    history cotangent carried from step to step (reading G17), J = sum_n |u^n - u_gt^n|^2.  Expected values: the same loop
    written with oracle/ functions only (oracle.newton + oracle.sens, itself pinned to central differences of J)."""
    import torch
    import oracle
    import oracle.sens as osn
    import oracle.newton as onw
    import paper_2606_17390_b200 as fem
    from synth import mesh
    p = _small_problem(seed=4, n=(2, 2, 2), hist=False)
    coords, conn, mat = p["coords"], p["conn"], p["mat"]
    nn, ne = coords.shape[0], conn.shape[0]
    X0 = mesh.structured_hex_mesh(2, 2, 2)[0]
    x0, x1 = np.isclose(X0[:, 0], 0.0), np.isclose(X0[:, 0], 1.0)
    bn = np.flatnonzero(x0 | x1)
    bc = (3 * bn[:, None] + np.arange(3)).ravel()
    free = np.setdiff1d(np.arange(3 * nn), bc)

    def target(s):
        t = np.zeros((nn, 3)); t[x1, 0] = 0.012 * s; t[x1, 1] = 0.006 * s
        return t.ravel()[bc]
    targets = [target(0.5), target(1.0)]
    rng = np.random.default_rng(0)
    ugt = [0.01 * rng.normal(size=(nn, 3)) for _ in targets]
    # ---- oracle side
    rp, ci, _ = oracle.pattern(nn, conn, with_slots=False)
    uo, ho, states = np.zeros_like(coords), np.zeros((ne, 8, 7)), []
    for t in targets:
        r = onw.newton_solve(coords, conn, uo, ho, mat, rp, ci, bc, t, rtol=1e-13, atol=1e-9, fbar=fbar)
        assert r["converged"]
        states.append((r["u"].copy(), ho.copy()))
        uo, ho = r["u"], r["hist_out"]
    grad_o, mu_o = np.zeros(16), None
    for (u, h), g in zip(reversed(states), reversed(ugt)):
        out = oracle.assemble(coords, conn, u, h, mat, rp, ci, fbar=fbar)
        rhs = -2.0 * (u - g).ravel()
        if mu_o is not None:
            rhs -= osn.assemble_vjp(coords, conn, u, h, mat, None, mu_o, fbar=fbar)["g_u"].ravel()
        K = onw.csr(rp, ci, out["csr_vals"]).toarray()
        lam = np.zeros(3 * nn)
        lam[free] = np.linalg.solve(K[np.ix_(free, free)].T, rhs[free])
        v = osn.assemble_vjp(coords, conn, u, h, mat, lam, mu_o, fbar=fbar)
        grad_o += v["g_mat"][0]
        mu_o = v["g_hist_in"]
    # ---- GPU side
    ctx = _ctx_fbar(coords, conn)[0] if fbar else _ctx(coords, conn)
    dev = ctx.device
    t64 = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).ravel()).to(dev)
    mat_d, bc_d = t64(mat), torch.from_numpy(bc.astype(np.int32)).to(dev)
    u_d = torch.zeros(3 * nn, dtype=torch.float64, device=dev)
    h_d = torch.zeros(56 * ne, dtype=torch.float64, device=dev)
    gstates = []
    for t in targets:
        u_d, h_new, rep = ctx.newton_solve(u_d, h_d, mat_d, bc_d, t64(t), rtol=1e-13, atol=1e-9, lin_rtol=1e-13)
        assert rep["converged"]
        gstates.append((u_d.clone(), h_d))
        h_d = h_new
    idx = list(osn.THETA_IDX)
    gg = None
    if not fbar:      # composed from the single calls (CG on the symmetric reduced tangent)
        grad_g, mu_d = torch.zeros(16, dtype=torch.float64, device=dev), None
        for (u, h), g in zip(reversed(gstates), reversed(ugt)):
            _, vals, _, _ = ctx.assemble(u, h, mat_d)
            rhs = -2.0 * (u - t64(g))
            if mu_d is not None:
                rhs = rhs - ctx.assemble_vjp(u, h, mat_d, None, mu_d, want_hist=False, want_mat=False)[0]
            ctx.apply_dirichlet(bc_d, vals, rhs)                         # identity rows, lam = 0 on the constrained DOFs
            lam, _, _, ok = ctx.pcg(vals, rhs, rtol=1e-13, max_iter=5000)
            assert ok
            _, mu_new, g_m = ctx.assemble_vjp(u, h, mat_d, lam, mu_d, want_u=False)
            grad_g += g_m[0]
            mu_d = mu_new
        gg = grad_g.cpu().numpy()
        assert np.max(np.abs(gg[idx] - grad_o[idx]) / np.maximum(np.abs(grad_o[idx]), 1e-6 * np.abs(grad_o[idx]).max())) <= 1e-6
        assert rel_l2(mu_d.cpu().numpy(), mu_o) <= 1e-6
    # the same backward sweep through fem_adjoint_step (one C-ABI call per load step)
    grad_s, mu_s = torch.zeros(16, dtype=torch.float64, device=dev), None
    for (u, h), g in zip(reversed(gstates), reversed(ugt)):
        lam_s, mu_s, g_m, its = ctx.adjoint_step(u, h, mat_d, bc_d, dJdu=2.0 * (u - t64(g)), mu_in=mu_s, lin_rtol=1e-13)
        assert its > 0 and float(torch.abs(lam_s[bc_d.long()]).max()) == 0.0
        grad_s += g_m[0]
    gs = grad_s.cpu().numpy()
    if gg is not None:
        assert np.max(np.abs(gs[idx] - gg[idx]) / np.maximum(np.abs(gg[idx]), 1e-6 * np.abs(gg[idx]).max())) <= 1e-9
    assert np.max(np.abs(gs[idx] - grad_o[idx]) / np.maximum(np.abs(grad_o[idx]), 1e-6 * np.abs(grad_o[idx]).max())) <= 1e-6
    assert rel_l2(mu_s.cpu().numpy(), mu_o) <= 1e-6
    with pytest.raises(fem.FemError):      # mu_out must not alias hist_in: checked by the library
        import ctypes as C
        L = fem.lib()
        rc = L.fem_adjoint_step(ctx._h, u.data_ptr(), h.data_ptr(), mat_d.data_ptr(), 1, bc_d.numel(), bc_d.data_ptr(), None, None,
                                lam_s.data_ptr(), h.data_ptr(), g_m.data_ptr(), 1e-10, 100, None, None)
        if rc != 0:
            raise fem.FemError(rc, "fem_adjoint_step")
    ctx.close()


def test_vjp_config4_and_config5_samples():
    """Config 4 (void-mask mesh, shuffled element order, per-element Hill ratios and Swift K: irregular gather, nodes with fewer
    than 8 elements, n_mat = n_elems) and the top strain level of config 5 (peak strain 0.3): sampled elements (g_hist_in,
    per-element g_mat) and sampled nodes (g_u) against the oracle; K lam against the library's own tangent."""
    import torch
    import oracle
    import oracle.sens as osn
    import synth
    import paper_2606_17390_b200 as fem
    dev = torch.device("cuda:0")
    for label, cfg in (("config4", synth.make_config(4)), ("config5s3", synth.make_config(5, sweep="strain", level=3))):
        ne, nn = cfg["conn"].shape[0], cfg["coords"].shape[0]
        mat_np = np.ascontiguousarray(fem.mat_from_desc(cfg["matdesc"], ne))
        omat = np.ascontiguousarray(oracle.mat_from_desc(cfg["matdesc"], ne))
        ctx = _ctx(cfg["coords"], cfg["conn"])
        g = torch.Generator(device="cpu"); g.manual_seed(11)
        lam = torch.randn(3 * nn, dtype=torch.float64, generator=g).to(dev)
        mu = (torch.randn(ne, 8, 7, dtype=torch.float64, generator=g) * torch.tensor([1e3] * 6 + [1e2], dtype=torch.float64)).reshape(-1).to(dev)
        u = torch.from_numpy(cfg["u"].ravel()).to(dev); h = torch.from_numpy(cfg["hist_in"].ravel()).to(dev)
        mat = torch.from_numpy(mat_np.ravel()).to(dev)
        _, vals, _, _ = ctx.assemble(u, h, mat)
        a_u, _, _ = ctx.assemble_vjp(u, h, mat, lam, None, want_hist=False, want_mat=False)
        Kl = ctx.spmv(vals, lam)
        assert float(torch.linalg.norm(a_u - Kl) / torch.linalg.norm(Kl)) <= 1e-10, label
        c_u, c_h, c_m = ctx.assemble_vjp(u, h, mat, lam, mu)
        lam_n, mu_n = lam.cpu().numpy().reshape(nn, 3), mu.cpu().numpy().reshape(ne, 8, 7)
        rng = np.random.default_rng(12)
        el = np.sort(rng.choice(ne, 40, replace=False))
        o = osn.assemble_vjp(cfg["coords"], cfg["conn"], cfg["u"], cfg["hist_in"], omat, lam_n, mu_n, elems=el)
        assert rel_l2(c_h.cpu().numpy().reshape(ne, 8, 7)[el], o["g_hist_in"][el]) <= TOL, label
        if omat.shape[0] == ne:
            gm = c_m.cpu().numpy()[el]
            assert np.max(np.abs(gm - o["g_mat"][el]) / np.maximum(o["g_mat_abs"][el].max(axis=0), 1e-300)) <= TOL, label
        nodes = rng.choice(nn, 10, replace=False)
        els = np.unique(np.flatnonzero(np.isin(cfg["conn"], nodes).any(axis=1)))
        o2 = osn.assemble_vjp(cfg["coords"], cfg["conn"], cfg["u"], cfg["hist_in"], omat, lam_n, mu_n, elems=els)
        assert rel_l2(c_u.cpu().numpy().reshape(nn, 3)[nodes], o2["g_u_full"][nodes]) <= TOL, label
        ctx.close()


def _ctx_fbar(coords, conn):
    import torch
    import paper_2606_17390_b200 as fem
    dev = torch.device("cuda:0")
    ctx = fem.FemContext(torch.from_numpy(np.ascontiguousarray(coords)).to(dev), torch.from_numpy(np.ascontiguousarray(conn)).to(dev), fbar=1)
    rp, ci, _ = ctx.build_csr_pattern()
    return ctx, rp.cpu().numpy(), ci.cpu().numpy()


@pytest.mark.parametrize("variant", ["uniform_swift", "per_elem_rotated_voce", "large_strain"])
def test_vjp_fbar_small_meshes(variant):
    """F-bar element (Eq.(31)-(32) PAPER.md:237-243): the 8 Gauss points of an element are coupled through Jbar."""
    import oracle.sens as osn
    p = _small_problem(per_elem=variant == "per_elem_rotated_voce", voce=variant == "per_elem_rotated_voce",
                       amp=0.2 if variant == "large_strain" else 0.006, seed=31)
    ctx, _, _ = _ctx_fbar(p["coords"], p["conn"])
    o = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], p["mu"], fbar=1)
    g_u, g_h, g_m = _gpu_vjp(ctx, p)
    assert rel_l2(g_u, o["g_u_full"]) <= TOL and rel_l2(g_h, o["g_hist_in"]) <= TOL
    _check_mat(g_m, o)
    g_u2, _, _ = _gpu_vjp(ctx, p, lam=False)
    assert rel_l2(g_u2, o["g_u"]) <= TOL
    # and it differs from the standard element (the coupling is not a no-op on this field)
    o0 = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], p["mu"], fbar=0)
    assert rel_l2(g_u, o0["g_u_full"]) > 1e-6
    ctx.close()


def test_vjp_fbar_config2_transposed_tangent_and_samples():
    """Config 2 with F-bar: g_u(lam, 0) = K^T lam with the library's own (unsymmetric) F-bar tangent — K lam must not match —
    and sampled elements / nodes against the oracle."""
    import torch
    import scipy.sparse as sp
    import oracle
    import oracle.sens as osn
    import synth
    import paper_2606_17390_b200 as fem
    cfg = synth.make_config(2)
    ne, nn = cfg["conn"].shape[0], cfg["coords"].shape[0]
    ctx, rp, ci = _ctx_fbar(cfg["coords"], cfg["conn"])
    dev = ctx.device
    rng = np.random.default_rng(41)
    lam_n = rng.normal(size=(nn, 3)); mu_n = rng.normal(size=(ne, 8, 7)) * np.array([1e3] * 6 + [1e2])
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64).ravel()).to(dev)
    u, h, lam, mu = t(cfg["u"]), t(cfg["hist_in"]), t(lam_n), t(mu_n)
    mat = t(fem.mat_from_desc(cfg["matdesc"], ne))
    _, vals, _, _ = ctx.assemble(u, h, mat)
    a_u, _, _ = ctx.assemble_vjp(u, h, mat, lam, None, want_hist=False, want_mat=False)
    K = sp.csr_matrix((vals.cpu().numpy(), ci, rp), shape=(3 * nn, 3 * nn))
    Ktl, Kl = K.T @ lam_n.ravel(), K @ lam_n.ravel()
    assert rel_l2(a_u.cpu().numpy(), Ktl) <= 1e-10
    assert rel_l2(a_u.cpu().numpy(), Kl) > 1e-6
    c_u, c_h, c_m = ctx.assemble_vjp(u, h, mat, lam, mu)
    omat = oracle.mat_from_desc(cfg["matdesc"], ne)
    el = np.sort(rng.choice(ne, 60, replace=False))
    o = osn.assemble_vjp(cfg["coords"], cfg["conn"], cfg["u"], cfg["hist_in"], omat, lam_n, mu_n, elems=el, fbar=1)
    assert rel_l2(c_h.cpu().numpy().reshape(ne, 8, 7)[el], o["g_hist_in"][el]) <= TOL
    nodes = rng.choice(nn, 10, replace=False)
    els = np.unique(np.flatnonzero(np.isin(cfg["conn"], nodes).any(axis=1)))
    o2 = osn.assemble_vjp(cfg["coords"], cfg["conn"], cfg["u"], cfg["hist_in"], omat, lam_n, mu_n, elems=els, fbar=1)
    assert rel_l2(c_u.cpu().numpy().reshape(nn, 3)[nodes], o2["g_u_full"][nodes]) <= TOL
    d_u, d_h, d_m = ctx.assemble_vjp(u, h, mat, lam, mu)
    assert torch.equal(c_u, d_u) and torch.equal(c_h, d_h) and torch.equal(c_m, d_m)
    ctx.close()
