"""Pins of oracle/sens.py against what is fixed outside it: central finite differences of the C
oracle's own `assemble` (the paper's check, Eq.(52)), the assembled tangent K (g_u_full(lambda, 0) = K lambda),
elastic closed forms, linearity, and the adjoint gradient of a short load path against central differences of J (Table 6)."""
import numpy as np
import pytest

import oracle
import oracle.sens as osn
import oracle.newton as onw
import synth
from synth import mesh


def _problem(seed=5, n=(2, 2, 2), per_elem=False, voce=False, amp=0.006, hist=True):
    coords, conn = mesh.structured_hex_mesh(*n)
    rng = np.random.default_rng(seed)
    coords = coords + 0.04 * rng.uniform(-1, 1, size=coords.shape) / max(n)
    ne = conn.shape[0]
    base = oracle.mat_from_desc(dict(synth.configs.SWIFT), 1)[0]
    nm = ne if per_elem else 1
    mat = np.tile(base, (nm, 1))
    if voce:
        mat[:, 8], mat[:, 9], mat[:, 10], mat[:, 11] = 0.0, 200.0, 150.0, 12.0     # sigma0, Q, b
    if per_elem:
        mat[:, 2:8] *= 1 + 0.1 * rng.uniform(-1, 1, size=(nm, 6))
        mat[:, 9] *= 1 + 0.1 * rng.uniform(-1, 1, size=nm)
        q = rng.normal(size=(nm, 4)); mat[:, 12:16] = q / np.linalg.norm(q, axis=1)[:, None]
    A = rng.normal(size=(3, 3)); A *= amp / np.linalg.norm(A)
    # the x-dependent factor leaves part of the mesh elastic
    u = (coords @ A.T) * (0.15 + coords[:, :1]) + 2e-4 * rng.normal(size=coords.shape)
    h = np.zeros((ne, 8, 7))
    if hist:
        h[..., 6] = 0.01 * rng.uniform(size=(ne, 8))
        d = rng.normal(size=(ne, 8, 6)) * 2e-4
        d[..., :3] -= d[..., :3].mean(axis=-1, keepdims=True)
        h[..., :6] = d
    rp, ci, _ = oracle.pattern(coords.shape[0], conn, with_slots=False)
    lam = rng.normal(size=coords.shape)
    mu = rng.normal(size=(ne, 8, 7)) * np.array([1e3] * 6 + [1e2])
    return dict(coords=coords, conn=conn, mat=mat, u=u, h=h, rp=rp, ci=ci, lam=lam, mu=mu)


def _psi(p, u=None, h=None, mat=None):
    out = oracle.assemble(p["coords"], p["conn"], p["u"] if u is None else u, p["h"] if h is None else h,
                          p["mat"] if mat is None else mat, p["rp"], p["ci"])
    return float(np.dot(out["residual"], p["lam"].ravel()) + np.dot(out["hist_out"].ravel(), p["mu"].ravel())), out


def _fd(f, x, idx, step):
    g = np.zeros(len(idx))
    for n, k in enumerate(idx):
        xp, xm = x.copy(), x.copy()
        xp.flat[k] += step(x.flat[k]); xm.flat[k] -= step(x.flat[k])
        g[n] = (f(xp) - f(xm)) / (xp.flat[k] - xm.flat[k])
    return g


@pytest.mark.parametrize("variant", ["uniform_swift", "per_elem_rotated_voce"])
def test_vjp_against_central_differences_of_assemble(variant):
    p = _problem(per_elem=variant != "uniform_swift", voce=variant != "uniform_swift")
    _, out = _psi(p)
    npl = out["stats"]["n_plastic"]
    assert 8 < npl < 8 * p["conn"].shape[0] - 8          # both branches of Alg. C1 are exercised
    v = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], p["mu"])
    rng = np.random.default_rng(1)
    # d psi / d u  = K^T lambda + (dh_out/du)^T mu
    idx = rng.choice(p["u"].size, 24, replace=False)
    g = _fd(lambda x: _psi(p, u=x)[0], p["u"], idx, lambda x: 1e-7)
    assert np.allclose(v["g_u_full"].ravel()[idx], g, rtol=2e-6, atol=1e-6 * np.abs(g).max())
    # d psi / d hist_in
    idx = rng.choice(p["h"].size, 40, replace=False)
    g = _fd(lambda x: _psi(p, h=x)[0], p["h"], idx, lambda x: 1e-7)
    assert np.allclose(v["g_hist_in"].ravel()[idx], g, rtol=2e-6, atol=1e-6 * np.abs(g).max())
    # d psi / d theta (every record, every differentiated parameter)
    nm = p["mat"].shape[0]
    idx = [m * 16 + k for m in (range(nm) if nm == 1 else (0, nm - 1)) for k in osn.THETA_IDX]
    g = _fd(lambda x: _psi(p, mat=x)[0], p["mat"], idx, lambda x: 1e-6 * abs(x))
    ref = v["g_mat"].ravel()[idx]
    assert np.allclose(ref, g, rtol=5e-6, atol=1e-7 * v["g_mat_abs"].ravel()[idx].max())
    assert np.all(v["g_mat"][:, [8, 12, 13, 14, 15]] == 0.0)


def test_history_leg_only_and_linearity():
    """g_u holds the mu leg alone; the lambda leg of g_u_full is K lambda (K symmetric for fbar = 0)."""
    p = _problem(seed=9)
    a = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], None)
    b = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], None, p["mu"])
    c = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], p["mu"])
    assert np.all(a["g_u"] == 0.0)
    out = oracle.assemble(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["rp"], p["ci"])
    Kl = onw.csr(p["rp"], p["ci"], out["csr_vals"]).T @ p["lam"].ravel()
    assert np.allclose(a["g_u_full"].ravel(), Kl, rtol=1e-10, atol=1e-10 * np.abs(Kl).max())
    assert np.allclose(b["g_u_full"], b["g_u"], rtol=1e-12, atol=1e-12 * np.abs(b["g_u"]).max())
    for k in ("g_u", "g_hist_in", "g_mat"):
        assert np.allclose(a[k] + b[k], c[k], rtol=1e-12, atol=1e-12 * np.abs(c[k]).max())
    # the mu leg vanishes at elastic points: hist_out = hist_in there (Alg. C1 steps 3-5 :898-902)
    el = np.isclose(out["hist_out"][..., 6], p["h"][..., 6], rtol=0, atol=0)
    assert el.any() and (~el).any()
    assert np.allclose(b["g_hist_in"][el], p["mu"][el], rtol=1e-13)


def test_elastic_closed_forms():
    """All-elastic state: R is linear in E (dR/dE = R/E), independent of the Hill ratios and hardening constants, and
    g_hist_in = -(dR/d eps)^T lambda has no alpha component."""
    p = _problem(seed=2, amp=1e-3, hist=False)
    _, out = _psi(p)
    assert out["stats"]["n_plastic"] == 0
    v = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], None)
    assert np.isclose(v["g_mat"][0, 0], np.dot(out["residual"], p["lam"].ravel()) / p["mat"][0, 0], rtol=1e-10)
    assert np.all(v["g_mat"][0, 2:] == 0.0)
    assert np.all(v["g_hist_in"][..., 6] == 0.0)


def _load_path(theta_mat, p, bc, targets, want_states=False):
    u = np.zeros_like(p["coords"]); h = np.zeros_like(p["h"]); states = []
    for t in targets:
        res = onw.newton_solve(p["coords"], p["conn"], u, h, theta_mat, p["rp"], p["ci"], bc, t, rtol=1e-13, atol=1e-9)
        assert res["converged"]
        states.append((res["u"].copy(), h.copy()))
        u, h = res["u"], res["hist_out"]
    return states


def test_adjoint_gradient_against_central_differences():
    """Alg. 1 on a two-step load path with the exact history recursion (reading G17), checked as the
    paper checks it: central differences of J (Eq.(52) :412; Table 6 :531-545 reports < 0.2 % — here the discrete adjoint is
    exact, so the agreement is limited by the difference quotient only)."""
    p = _problem(seed=4, hist=False)
    coords, conn, rp, ci = p["coords"], p["conn"], p["rp"], p["ci"]
    nn = coords.shape[0]
    x0 = np.isclose(mesh.structured_hex_mesh(2, 2, 2)[0][:, 0], 0.0)
    x1 = np.isclose(mesh.structured_hex_mesh(2, 2, 2)[0][:, 0], 1.0)
    bn = np.flatnonzero(x0 | x1)
    bc = (3 * bn[:, None] + np.arange(3)).ravel()
    def target(s):
        t = np.zeros((nn, 3)); t[x1, 0] = 0.012 * s; t[x1, 1] = 0.006 * s
        return t.ravel()[bc]
    targets = [target(0.5), target(1.0)]
    rng = np.random.default_rng(0)
    ugt = [0.01 * rng.normal(size=(nn, 3)) for _ in targets]
    free = np.setdiff1d(np.arange(3 * nn), bc)

    def J(mat):
        st = _load_path(mat, p, bc, targets)
        return sum(float(np.sum((s[0] - g) ** 2)) for s, g in zip(st, ugt))

    mat = p["mat"]
    states = _load_path(mat, p, bc, targets)
    assert oracle.assemble(coords, conn, states[-1][0], states[-1][1], mat, rp, ci)["stats"]["n_plastic"] > 16
    grad = np.zeros(16)
    mu = None
    for (u, h), g in zip(reversed(states), reversed(ugt)):
        out = oracle.assemble(coords, conn, u, h, mat, rp, ci)
        rhs = -2.0 * (u - g).ravel()                                # -(dJ^n/du^n)^T
        if mu is not None:
            rhs -= osn.assemble_vjp(coords, conn, u, h, mat, None, mu)["g_u"].ravel()   # -(dR^{n+1}/du^n)^T lambda^{n+1}
        K = onw.csr(rp, ci, out["csr_vals"]).toarray()
        lam = np.zeros(3 * nn)
        lam[free] = np.linalg.solve(K[np.ix_(free, free)].T, rhs[free])                # Eq.(51) on the free DOFs
        v = osn.assemble_vjp(coords, conn, u, h, mat, lam, mu)
        grad += v["g_mat"][0]                                                          # Eq.(49)
        mu = v["g_hist_in"]
    idx = list(osn.THETA_IDX)
    fd = _fd(J, mat, idx, lambda x: 1e-5 * abs(x))
    assert np.allclose(grad[idx], fd, rtol=2e-4, atol=1e-6 * np.abs(fd).max())


def test_fbar_vjp_against_central_differences_and_transposed_tangent():
    """F-bar element (Eq.(31)-(32) PAPER.md:237-243, reading G12): the element-level coupling through Jbar is part of the VJP.
    Pins: central differences of the C oracle's F-bar assemble (Eq.(52) :412) in u, hist_in and theta, and g_u_full(lambda, 0) =
    K^T lambda with the oracle's assembled F-bar tangent — which is unsymmetric, so K lambda must NOT match (a transposed
    operand fails here)."""
    p = _problem(seed=5)

    def psi(u=None, h=None, mat=None):
        out = oracle.assemble(p["coords"], p["conn"], p["u"] if u is None else u, p["h"] if h is None else h,
                              p["mat"] if mat is None else mat, p["rp"], p["ci"], fbar=1)
        return float(np.dot(out["residual"], p["lam"].ravel()) + np.dot(out["hist_out"].ravel(), p["mu"].ravel())), out
    _, out = psi()
    assert 8 < out["stats"]["n_plastic"] < 8 * p["conn"].shape[0] - 8
    v = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], p["mu"], fbar=1)
    rng = np.random.default_rng(1)
    idx = rng.choice(p["u"].size, 16, replace=False)
    g = _fd(lambda x: psi(u=x)[0], p["u"], idx, lambda x: 1e-7)
    assert np.allclose(v["g_u_full"].ravel()[idx], g, rtol=2e-6, atol=1e-6 * np.abs(g).max())
    idx = rng.choice(p["h"].size, 24, replace=False)
    g = _fd(lambda x: psi(h=x)[0], p["h"], idx, lambda x: 1e-7)
    assert np.allclose(v["g_hist_in"].ravel()[idx], g, rtol=2e-6, atol=1e-6 * np.abs(g).max())
    idx = list(osn.THETA_IDX)
    g = _fd(lambda x: psi(mat=x)[0], p["mat"], idx, lambda x: 1e-6 * abs(x))
    assert np.allclose(v["g_mat"].ravel()[idx], g, rtol=5e-6, atol=1e-7 * v["g_mat_abs"].ravel()[idx].max())
    a = osn.assemble_vjp(p["coords"], p["conn"], p["u"], p["h"], p["mat"], p["lam"], None, fbar=1)
    K = onw.csr(p["rp"], p["ci"], out["csr_vals"])
    Ktl, Kl = K.T @ p["lam"].ravel(), K @ p["lam"].ravel()
    assert np.allclose(a["g_u_full"].ravel(), Ktl, rtol=1e-10, atol=1e-10 * np.abs(Ktl).max())
    assert np.abs(a["g_u_full"].ravel() - Kl).max() > 1e-5 * np.abs(Kl).max()
    # the standard element is the fbar = 0 branch of the same function; on an affine field both coincide (J_q = Jbar)
    A = np.array([[0.004, 0.001, 0.0], [0.0, -0.003, 0.002], [0.001, 0.0, 0.002]])
    ua = p["coords"] @ A.T
    s0 = osn.assemble_vjp(p["coords"], p["conn"], ua, p["h"] * 0, p["mat"], p["lam"], p["mu"], fbar=0)
    s1 = osn.assemble_vjp(p["coords"], p["conn"], ua, p["h"] * 0, p["mat"], p["lam"], p["mu"], fbar=1)
    assert np.allclose(s0["g_hist_in"], s1["g_hist_in"], rtol=1e-9, atol=1e-9 * np.abs(s0["g_hist_in"]).max())
    assert np.allclose(s0["g_mat"], s1["g_mat"], rtol=1e-9, atol=1e-9 * np.abs(s0["g_mat_abs"]).max())
