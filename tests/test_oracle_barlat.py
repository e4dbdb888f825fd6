"""Pins for the Yld2004-18p oracle (Eq.(12), App. A.2 :808-830, App. B :836-881).
Each compares with something the oracle does not compute itself: the value the paper prints for its line-search
example, the reductions the paper states (:828), Hershey closed forms, the eigenvalue definition, homogeneity,
finite differences, a brute-force closest-point search, or the independently pinned Hill-48 solver."""
import os
import numpy as np
import pytest
import oracle

MW = np.array([1, 1, 1, np.sqrt(2), np.sqrt(2), np.sqrt(2)])
HERE = os.path.dirname(__file__)


def sym(v):
    return np.array([[v[0], v[3], v[5]], [v[3], v[1], v[4]], [v[5], v[4], v[2]]])


def vec(A):
    return np.array([A[0, 0], A[1, 1], A[2, 2], A[0, 1], A[1, 2], A[0, 2]])


def hooke_strain(E, nu, sig):
    S = sym(sig)
    return vec((1 + nu) / E * S - nu / E * np.trace(S) * np.eye(3))


def hooke_stress(E, nu, eps):
    mu, la = E / (2 * (1 + nu)), E * nu / ((1 + nu) * (1 - 2 * nu))
    e = sym(eps)
    return vec(la * np.trace(e) * np.eye(3) + 2 * mu * e)


def read_golden():
    g = {}
    for line in open(os.path.join(HERE, "golden", "barlat_linesearch.txt")):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        g[k] = [float(x) for x in v]
    return g


TAB2 = oracle.barlat_record()                       # Table 2, m = 8
ISO8 = oracle.barlat_record([1] * 9, [1] * 9, 8)


def perfect_mat(E=1000.0, nu=0.3, s0=1.0, quat=(1, 0, 0, 0)):
    return oracle.mat_record(E, nu, [1] * 6, 0, s0, 0.0, 1.0, quat)   # Voce with Q = 0


def swift_mat(quat=(1, 0, 0, 0)):
    return oracle.mat_record(70000.0, 0.33, [1] * 6, 1, 500.0, 0.01, 0.2, quat)


# ------------------------------------------------------------------ the paper's printed example
def test_paper_linesearch_example():
    g = read_golden()
    E, nu = g["E"][0], g["nu"][0]
    Ttr = np.array(g["trial_principal_stress"] + [0, 0, 0])
    assert abs(Ttr[:3].sum()) < 1e-12                                    # "deviatoric trial stress state"
    r = oracle.return_map_gen(perfect_mat(E, nu, g["sigma0"][0]), TAB2, hooke_strain(E, nu, Ttr), np.zeros(6), 0.0,
                              beta=g["beta"][0], eta=g["eta"][0])
    tr = r["trace"]
    k = int(g["linesearch_iteration"][0]) - 1
    assert np.all(tr[:k, 2] == 1.0)                                      # "the first two iterations are similar"
    assert tr[k, 1] > tr[k, 0]                                           # "zeta = 1 increases the merit function"
    assert abs(tr[k, 2] - g["zeta"][0]) < 5e-4                           # "selects zeta = 0.363"
    assert r["plastic"] and not r["nonconv"] and r["iters"] <= 12        # line search "leads to robust convergence"
    phi, _, _ = oracle.yield_eval(perfect_mat(E, nu), TAB2, r["T"])
    assert abs(phi - 1.0) < 1e-13


def test_table2_normalisation():
    # Fig. A1 caption :830: "normalized such that the yield stress in uniaxial tension along the first principal axis is 1"
    assert abs(oracle.barlat_phi_eig(TAB2, [1, 0, 0, 0, 0, 0]) - 1.0) < 1e-3


# ------------------------------------------------------------------ reductions and closed forms
@pytest.mark.parametrize("m", [2, 4])
def test_isotropic_reduces_to_von_mises(m):
    # :828 "when all 18 parameters are set to unity and m=2 or m=4, the Barlat model reduces to the von Mises criterion"
    rng = np.random.default_rng(m)
    bar = oracle.barlat_record([1] * 9, [1] * 9, m)
    for _ in range(20):
        T = rng.normal(size=6) * 100
        s = sym(T) - np.trace(sym(T)) / 3 * np.eye(3)
        vm = np.sqrt(1.5 * np.sum(s * s))
        phi, N, H = oracle.barlat_derivs(bar, T * MW)
        assert abs(phi / vm - 1) < 1e-13
        assert abs(oracle.barlat_phi_eig(bar, T * MW) / vm - 1) < 1e-13
        assert np.allclose(N, 1.5 * vec(s) * MW / vm, rtol=1e-12, atol=1e-14)      # textbook J2 flow direction
        Pd = np.eye(6); Pd[:3, :3] -= 1 / 3
        assert np.allclose(H, (1.5 * Pd - np.outer(N, N)) / vm, atol=1e-12 / vm * 100)


@pytest.mark.parametrize("m", [6, 8, 12])
def test_hershey_closed_forms(m):
    bar = oracle.barlat_record([1] * 9, [1] * 9, m)
    # uniaxial tension in any direction: phi = sigma ; pure shear: s = (tau, -tau, 0) -> phi = tau (2^(m-1) + 1)^(1/m)
    rng = np.random.default_rng(m)
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    for T, ref in ((Q @ np.diag([3.0, 0, 0]) @ Q.T, 3.0), (Q @ np.diag([2.0, -2.0, 0]) @ Q.T, 2.0 * (2 ** (m - 1) + 1) ** (1 / m)),
                   (Q @ np.diag([5.0, 5.0, 1.0]) @ Q.T, 4.0)):   # hydrostatic part drops out: (4,4,0) = balanced biaxial
        Tm = vec(T) * MW
        assert abs(oracle.barlat_phi_eig(bar, Tm) / ref - 1) < 1e-13
        assert abs(oracle.barlat_derivs(bar, Tm)[0] / ref - 1) < 1e-12


def hill_ratios_from_map(bar):
    """C' = C'': sum_ij (a_i - a_j)^2 = 6 |dev s'|^2, so phi^2 = 3/2 |dev(C':s)|^2 = 3/2 T:(L^T P L):T -> the paper's Hill
    tensor H = L^T P L and its yield ratios (Eq.(A3)-(A5): H1111 = 2/(3 r11^2), 2 H1212 = 1/r12^2)."""
    c = np.asarray(bar[:9])
    Cm = np.zeros((6, 6))
    Cm[0, 1], Cm[0, 2], Cm[1, 0], Cm[1, 2], Cm[2, 0], Cm[2, 1] = -c[:6]
    Cm[3, 3], Cm[4, 4], Cm[5, 5] = c[6:9]
    P = np.eye(6); P[:3, :3] -= 1 / 3
    L = Cm @ P
    H = L.T @ P @ L
    r = [np.sqrt(2 / (3 * H[i, i])) for i in range(3)] + [1 / np.sqrt(H[i, i]) for i in (3, 4, 5)]
    return H, r


@pytest.mark.parametrize("m", [2, 4])
def test_equal_transformations_reduce_to_hill48(m):
    # :828 "With C'=C'' and m=2 or m=4, it reduces to the Hill-48 model" — ties the new code to the pinned Hill-48 oracle
    # through the whole return map (same T, eps_p, alpha, C_ep), including the W / sqrt(2/3) conventions (reading G2)
    rng = np.random.default_rng(10 + m)
    cp = 1.0 + 0.3 * rng.uniform(-1, 1, size=9)
    bar = oracle.barlat_record(cp, cp, m)
    H, r = hill_ratios_from_map(bar)
    quat = rng.normal(size=4)
    matB = oracle.mat_record(70000.0, 0.33, [1] * 6, 1, 500.0, 0.01, 0.2, quat)
    matH = oracle.mat_record(70000.0, 0.33, r, 1, 500.0, 0.01, 0.2, quat)
    assert np.allclose(oracle.hill_mandel(oracle.mat_record(1, 0.3, r, 0, 1, 0, 1)), H, atol=1e-13)
    nplastic = 0
    for _ in range(12):
        eps = rng.normal(size=6) * 0.006
        epn = rng.normal(size=6) * 0.002; epn[:3] -= epn[:3].mean()
        an = rng.uniform(0, 0.02)
        phiB, NB, _ = oracle.yield_eval(matB, bar, hooke_stress(70000.0, 0.33, eps))
        phiH, NH, _ = oracle.yield_eval(matH, None, hooke_stress(70000.0, 0.33, eps))
        assert abs(phiB / (np.sqrt(1.5) * phiH) - 1) < 1e-12
        a = oracle.return_map_gen(matB, bar, eps, epn, an)
        b = oracle.return_map(matH, eps, epn, an)
        assert a["plastic"] == b["plastic"] and not a["nonconv"]
        nplastic += a["plastic"]
        assert np.allclose(a["T"], b["T"], rtol=1e-11, atol=1e-9)
        assert np.allclose(a["ep"], b["ep"], rtol=1e-10, atol=1e-14)
        assert abs(a["alpha"] - b["alpha"]) < 1e-13
        assert np.allclose(a["Cep"], b["Cep"], rtol=1e-8, atol=1e-6)
    assert nplastic >= 6


def test_generic_solver_equals_hill_solver():
    rng = np.random.default_rng(5)
    r = oracle.hill_from_lankford(0.7, 0.6, 0.8)
    mat = oracle.mat_record(70000.0, 0.33, r, 1, 500.0, 0.01, 0.2, rng.normal(size=4))
    for _ in range(10):
        eps = rng.normal(size=6) * 0.01
        a = oracle.return_map_gen(mat, None, eps, np.zeros(6), 0.003)
        b = oracle.return_map(mat, eps, np.zeros(6), 0.003)
        assert a["plastic"] == b["plastic"]
        assert np.allclose(a["T"], b["T"], rtol=1e-11, atol=1e-9) and abs(a["alpha"] - b["alpha"]) < 1e-13
        assert np.allclose(a["Cep"], b["Cep"], rtol=1e-8, atol=1e-6)


# ------------------------------------------------------------------ derivatives
@pytest.mark.parametrize("m", [6, 8])
def test_power_sum_form_equals_eigenvalue_definition(m):
    rng = np.random.default_rng(m)
    bar = oracle.barlat_record(oracle.TABLE2_CP, oracle.TABLE2_CPP, m)
    for _ in range(50):
        Tm = rng.normal(size=6) * 300
        assert abs(oracle.barlat_derivs(bar, Tm, hess=False)[0] / oracle.barlat_phi_eig(bar, Tm) - 1) < 2e-13


def test_gradient_and_hessian():
    rng = np.random.default_rng(0)
    for _ in range(10):
        Tm = rng.normal(size=6) * 200
        phi, N, H = oracle.barlat_derivs(TAB2, Tm)
        # Euler: phi is homogeneous of degree 1 -> N.T = phi, H T = 0 ; H symmetric, positive semi-definite (convex phi)
        assert abs(N @ Tm / phi - 1) < 1e-12
        assert np.linalg.norm(H @ Tm) < 1e-11 * np.linalg.norm(H) * np.linalg.norm(Tm)
        assert np.allclose(H, H.T, atol=1e-15 + 1e-13 * np.abs(H).max())
        assert np.linalg.eigvalsh(H).min() > -1e-12 * np.abs(H).max()
        # pressure-insensitive: N is deviatoric
        assert abs(N[:3].sum()) < 1e-13
        # central differences of the DEFINITION (eigenvalues) and of N
        h = 1e-4 * np.linalg.norm(Tm)
        Nfd = np.array([(oracle.barlat_phi_eig(TAB2, Tm + h * e) - oracle.barlat_phi_eig(TAB2, Tm - h * e)) / (2 * h) for e in np.eye(6)])
        assert np.allclose(N, Nfd, atol=1e-7)
        Hfd = np.array([(oracle.barlat_derivs(TAB2, Tm + h * e, hess=False)[1] - oracle.barlat_derivs(TAB2, Tm - h * e, hess=False)[1]) / (2 * h)
                        for e in np.eye(6)])
        assert np.allclose(H, Hfd, atol=1e-6 * np.abs(H).max())


def test_material_rotation():
    rng = np.random.default_rng(3)
    q = rng.normal(size=4); q /= np.linalg.norm(q)
    w, x, y, z = q
    Th = np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                   [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                   [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])   # textbook quaternion -> rotation
    mat = swift_mat(q)
    T = rng.normal(size=6) * 200
    phi, N, H = oracle.yield_eval(mat, TAB2, T)
    Tmat = Th.T @ sym(T) @ Th                                    # Eq.(A1) :774, Theta columns = material axes (reading G4)
    assert abs(phi / oracle.barlat_phi_eig(TAB2, vec(Tmat) * MW) - 1) < 1e-13
    _, Nm, _ = oracle.barlat_derivs(TAB2, vec(Tmat) * MW)
    assert np.allclose(sym(N / MW), Th @ sym(Nm / MW) @ Th.T, atol=1e-13)
    assert np.linalg.norm(H @ (T * MW)) < 1e-10 * np.linalg.norm(H) * np.linalg.norm(T)


# ------------------------------------------------------------------ return map
def test_return_map_invariants_and_tangent():
    rng = np.random.default_rng(7)
    E, nu = 70000.0, 0.33
    for trial in range(8):
        mat = swift_mat(rng.normal(size=4))
        eps = rng.normal(size=6) * 0.01
        epn = rng.normal(size=6) * 0.003; epn[:3] -= epn[:3].mean()
        an = rng.uniform(0, 0.05)
        r = oracle.return_map_gen(mat, TAB2, eps, epn, an)
        if not r["plastic"]:
            continue
        assert not r["nonconv"]
        phi, N, _ = oracle.yield_eval(mat, TAB2, r["T"])
        sf, _ = oracle.flow(mat, r["alpha"])
        assert abs(phi / sf - 1) < 1e-12                                         # Eq.(21), W = 1: f = phi - sigma_flow
        assert abs(r["alpha"] - an - r["dgam"]) < 1e-15 and r["dgam"] > 0         # Eq.(20), W = 1 (:145)
        assert np.allclose((r["ep"] - epn) * MW, r["dgam"] * N, atol=1e-14)       # Eq.(19)
        assert np.allclose(r["T"], hooke_stress(E, nu, eps - r["ep"]), rtol=1e-12, atol=1e-9)   # Eq.(22)
        # C_ep (App. D) against central differences of the return map itself
        Cfd = np.zeros((6, 6))
        for b in range(6):
            d = np.zeros(6); d[b] = 1e-7
            Tp = oracle.return_map_gen(mat, TAB2, eps + d, epn, an)["T"]
            Tn = oracle.return_map_gen(mat, TAB2, eps - d, epn, an)["T"]
            Cfd[:, b] = (Tp - Tn) / 2e-7 * MW / MW[b]
        assert np.allclose(r["Cep"], Cfd, atol=2e-6 * np.abs(Cfd).max())
        assert np.allclose(r["Cep"], r["Cep"].T, atol=1e-9 * np.abs(Cfd).max())


def test_closest_point_property_brute_force():
    # perfect plasticity: T_{n+1} is the point of the yield surface closest to T_tr in the energy norm (Fig. C1 :885);
    # brute force: no radially projected neighbour of the solution is closer
    rng = np.random.default_rng(11)
    E, nu = 1000.0, 0.3
    mat = perfect_mat(E, nu)
    for _ in range(5):
        Ttr = rng.normal(size=6) * 2.0
        r = oracle.return_map_gen(mat, TAB2, hooke_strain(E, nu, Ttr), np.zeros(6), 0.0)
        if not r["plastic"]:
            continue
        dist = lambda T: (Ttr - T) @ (hooke_strain(E, nu, Ttr - T) * MW * MW)      # (Ttr-T):E^-1:(Ttr-T)
        d0 = dist(r["T"])
        for _ in range(300):
            Tc = r["T"] + rng.normal(size=6) * 10 ** rng.uniform(-3, -0.5)
            Tc[:3] += (Ttr[:3].sum() - Tc[:3].sum()) / 3                         # same pressure as the trial state
            s = vec(sym(Tc) - np.trace(sym(Tc)) / 3 * np.eye(3))
            s = s / oracle.yield_eval(mat, TAB2, s)[0]                             # deviator scaled onto phi = sigma0 = 1
            Tc = s + np.array([1, 1, 1, 0, 0, 0]) * Tc[:3].sum() / 3
            assert dist(Tc) >= d0 * (1 - 1e-12)


def test_line_search_converges_for_far_trial_states():
    # App. B :879: trial states between the yield surface and a 30 times larger similar surface; with the line search
    # "converges for all sampled points" (40-iteration cap in the paper)
    rng = np.random.default_rng(2)
    E, nu = 1000.0, 0.3
    mat = perfect_mat(E, nu)
    worst = 0
    for _ in range(300):
        th = rng.uniform(0, 2 * np.pi)
        d = np.array([np.cos(th), np.cos(th - 2 * np.pi / 3), np.cos(th + 2 * np.pi / 3), 0, 0, 0])   # pi-plane direction
        d /= oracle.yield_eval(mat, TAB2, d)[0]
        Ttr = d * rng.uniform(1.0, 30.0)
        r = oracle.return_map_gen(mat, TAB2, hooke_strain(E, nu, Ttr), np.zeros(6), 0.0, tol=1e-12, kmax=40)
        assert r["plastic"] and not r["nonconv"]
        worst = max(worst, r["iters"])
    assert worst <= 40


# ------------------------------------------------------------------ element level
def test_Ke_vs_central_fd_barlat():
    rng = np.random.default_rng(4)
    X = np.array([[0, 0, 0], [1, 0, 0], [1, 1, 0], [0, 1, 0], [0, 0, 1], [1, 0, 1], [1, 1, 1], [0, 1, 1]], float)
    X = X + rng.normal(size=X.shape) * 0.05
    Gd = rng.normal(size=(3, 3)) * 0.012
    u = X @ Gd.T + rng.normal(size=X.shape) * 2e-4
    hin = np.zeros((8, 7))
    mat = swift_mat(rng.normal(size=4))
    Re, Ke, hout, st = oracle.element(X, u, hin, mat, 0, bar=TAB2)
    assert st[0] >= 4                       # plastic points present
    h = 1e-7
    Kfd = np.zeros((24, 24))
    for b in range(24):
        du = np.zeros(24); du[b] = h
        Rp = oracle.element(X, u + du.reshape(8, 3), hin, mat, 0, bar=TAB2)[0]
        Rn = oracle.element(X, u - du.reshape(8, 3), hin, mat, 0, bar=TAB2)[0]
        Kfd[:, b] = (Rp - Rn) / (2 * h)
    assert np.allclose(Ke, Kfd, atol=2e-6 * np.abs(Ke).max())
    assert np.allclose(Ke, Ke.T, atol=1e-9 * np.abs(Ke).max())
    assert np.linalg.norm(Ke @ np.tile(np.eye(3), (8, 1))) < 1e-9 * np.abs(Ke).max()     # rigid translations in the null space
