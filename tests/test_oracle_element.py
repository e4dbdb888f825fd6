"""Pins for the element- and mesh-level oracle."""
import numpy as np
import pytest
import oracle
import synth
from synth import mesh as smesh

XI = np.array([[-1, -1, -1], [1, -1, -1], [1, 1, -1], [-1, 1, -1], [-1, -1, 1], [1, -1, 1], [1, 1, 1], [-1, 1, 1]], float)


def rnd_rot(rng):
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    return Q * np.sign(np.linalg.det(Q))


def distorted_hex(rng, amp=0.15):
    return 0.5 * (XI + 1.0) + amp * rng.uniform(-1, 1, size=(8, 3))


def textbook_linear_Ke(X, E, nu):
    """Textbook small-strain hex8 stiffness sum_q w B^T D B, written independently (Voigt, engineering shear)."""
    lam, mu = E * nu / ((1 + nu) * (1 - 2 * nu)), E / (2 * (1 + nu))
    D = np.zeros((6, 6)); D[:3, :3] = lam; D[np.arange(3), np.arange(3)] += 2 * mu; D[np.arange(3, 6), np.arange(3, 6)] = mu
    g = 1 / np.sqrt(3)
    K = np.zeros((24, 24))
    for kz in (-g, g):
        for ky in (-g, g):
            for kx in (-g, g):
                xi = np.array([kx, ky, kz])
                dN = np.array([[XI[I, d] * np.prod([1 + xi[m] * XI[I, m] for m in range(3) if m != d]) / 8 for d in range(3)]
                               for I in range(8)])
                J = X.T @ dN
                G = dN @ np.linalg.inv(J)
                B = np.zeros((6, 24))
                for I in range(8):
                    gx, gy, gz = G[I]
                    B[:, 3 * I:3 * I + 3] = [[gx, 0, 0], [0, gy, 0], [0, 0, gz], [gy, gx, 0], [0, gz, gy], [gz, 0, gx]]
                K += np.linalg.det(J) * B.T @ D @ B
    return K


def test_shape_gradients_partition_and_linear_field():
    rng = np.random.default_rng(0)
    X = distorted_hex(rng)
    vol = 0.0
    for q in range(8):
        G, w = oracle.shape_grad(X, q)
        assert w > 0
        assert np.abs(G.sum(axis=0)).max() < 1e-14              # sum_I grad N_I = 0
        assert np.allclose(X.T @ G, np.eye(3), atol=1e-14)      # grad of the field X itself is I
        vol += w
    # volume of the distorted hex by the 2x2x2 rule equals the exact trilinear volume (integrand degree <= 2 per axis)
    from itertools import product
    gl = np.polynomial.legendre.leggauss(4)
    v4 = 0.0
    for (a, wa), (b, wb), (c, wc) in product(zip(*gl), repeat=3):
        xi = np.array([a, b, c])
        dN = np.array([[XI[I, d] * np.prod([1 + xi[m] * XI[I, m] for m in range(3) if m != d]) / 8 for d in range(3)] for I in range(8)])
        v4 += wa * wb * wc * np.linalg.det(X.T @ dN)
    assert abs(vol - v4) < 1e-14


def test_elastic_limit_equals_textbook_linear_stiffness(swift_mat):          # P2
    rng = np.random.default_rng(1)
    X = distorted_hex(rng)
    Re, Ke, hout, st = oracle.element(X, np.zeros((8, 3)), np.zeros((8, 7)), swift_mat, 0)
    Kref = textbook_linear_Ke(X, swift_mat[0], swift_mat[1])
    assert np.abs(Re).max() == 0.0
    assert np.abs(Ke - Kref).max() < 1e-13 * np.abs(Kref).max()
    assert st[0] == 0 and np.abs(hout).max() == 0


@pytest.mark.parametrize("fbar", [0, 1])
def test_rigid_body(fbar, swift_mat):                                         # P3
    rng = np.random.default_rng(2)
    X = distorted_hex(rng)
    u = 0.03 * rng.normal(size=(8, 3))
    hin = np.zeros((8, 7))
    Re, Ke, _, st = oracle.element(X, u, hin, swift_mat, fbar)
    assert st[0] > 0                                                          # a plastic state
    sc = np.abs(Ke).max()
    for d in range(3):
        t = np.zeros((8, 3)); t[:, d] = 1.0
        assert np.abs(Ke @ t.ravel()).max() < 1e-12 * sc                      # K t = 0 at any state
    assert np.abs(Re.reshape(8, 3).sum(axis=0)).max() < 1e-12 * np.abs(Re).max()
    Q = rnd_rot(rng)
    Re, Ke, _, _ = oracle.element(X, X @ Q.T - X, hin, swift_mat, fbar)       # u = (Q-I)X
    assert np.abs(Re).max() < 1e-10
    # stress-free state: 6 zero eigenvalues (3 translations + 3 infinitesimal rotations)
    ev = np.linalg.eigvalsh(0.5 * (Ke + Ke.T))
    assert np.sum(np.abs(ev) < 1e-9 * ev.max()) == 6


@pytest.mark.parametrize("fbar", [0, 1])
@pytest.mark.parametrize("state", ["plastic", "elastic"])
def test_Ke_vs_central_fd(fbar, state, swift_mat):                            # P11, P14
    rng = np.random.default_rng(3)
    X = distorted_hex(rng)
    amp = 0.04 if state == "plastic" else 3e-4
    u = amp * rng.normal(size=(8, 3))
    hin = np.zeros((8, 7))
    if state == "plastic":
        hin[:, 6] = 0.01 * rng.random(8)
    Re, Ke, _, st = oracle.element(X, u, hin, swift_mat, fbar)
    assert (st[0] == 8) if state == "plastic" else (st[0] == 0)
    sc = np.abs(Ke).max()
    errs = {}
    for h in (1e-4, 1e-5, 1e-6, 1e-7, 1e-9):
        fd = np.empty((24, 24))
        for b in range(24):
            d = np.zeros(24); d[b] = h
            Rp = oracle.element(X, u + d.reshape(8, 3), hin, swift_mat, fbar)[0]
            Rm = oracle.element(X, u - d.reshape(8, 3), hin, swift_mat, fbar)[0]
            fd[:, b] = (Rp - Rm) / (2 * h)
        errs[h] = np.abs(fd - Ke).max() / sc
    assert errs[1e-6] < 1e-8, errs
    assert errs[1e-9] > errs[1e-6] and errs[1e-4] > errs[1e-6] * 0.5, errs   # V-shaped curve
    asym = np.abs(Ke - Ke.T).max() / sc
    if fbar == 0:
        assert asym < 1e-13
    elif state == "plastic":
        assert asym > 1e-6                                                    # F-bar tangent is unsymmetric


def test_fbar_equals_standard_on_affine_field(swift_mat):                     # P1 (second half)
    rng = np.random.default_rng(4)
    X = distorted_hex(rng)
    A = 0.03 * rng.normal(size=(3, 3))
    u = X @ A.T
    r0 = oracle.element(X, u, np.zeros((8, 7)), swift_mat, 0)
    r1 = oracle.element(X, u, np.zeros((8, 7)), swift_mat, 1)
    assert np.allclose(r0[0], r1[0], rtol=1e-12, atol=1e-10)
    assert np.allclose(r0[2], r1[2], rtol=1e-12, atol=1e-16)


def test_objectivity(swift_mat):                                              # P17
    rng = np.random.default_rng(5)
    X = distorted_hex(rng)
    u = 0.03 * rng.normal(size=(8, 3))
    hin = np.zeros((8, 7)); hin[:, 6] = 0.005
    Q = rnd_rot(rng)
    for fbar in (0, 1):
        Re, Ke, ho, _ = oracle.element(X, u, hin, swift_mat, fbar)
        u2 = (X + u) @ Q.T - X
        Re2, Ke2, ho2, _ = oracle.element(X, u2, hin, swift_mat, fbar)
        QQ = np.kron(np.eye(8), Q)
        assert np.allclose(Re2, QQ @ Re, rtol=1e-11, atol=1e-9)
        assert np.abs(Ke2 - QQ @ Ke @ QQ.T).max() < 1e-11 * np.abs(Ke).max()
        assert np.allclose(ho2, ho, rtol=1e-11, atol=1e-15)


# ------------------------------------------------------------------ mesh level
def test_patch_test(swift_mat):                                               # P1
    coords, conn = smesh.structured_hex_mesh(3, 3, 3)
    interior = np.all((coords > 1e-9) & (coords < 1 - 1e-9), axis=1)
    coords = coords + 0.08 * interior[:, None] * (2 * synth.rng.uniform(5, 12, np.arange(coords.size)).reshape(-1, 3) - 1)
    rng = np.random.default_rng(6)
    A = 0.03 * rng.normal(size=(3, 3))
    u = coords @ A.T
    rp, ci, _ = oracle.pattern(coords.shape[0], conn)
    out = oracle.assemble(coords, conn, u, np.zeros((27, 8, 7)), swift_mat, rp, ci, 0)
    R = out["residual"].reshape(-1, 3)
    assert out["stats"]["n_plastic"] == 27 * 8
    assert np.abs(R[interior]).max() < 1e-12 * np.abs(R[~interior]).max()
    h = out["hist_out"].reshape(-1, 7)
    assert np.abs(h - h[0]).max() < 1e-14                                     # same state at every point
    out1 = oracle.assemble(coords, conn, u, np.zeros((27, 8, 7)), swift_mat, rp, ci, 1)
    assert np.allclose(out1["residual"], out["residual"], rtol=1e-11, atol=1e-10)


def test_pattern_closed_form_and_dense_boolean():                             # P13
    for (nx, ny, nz) in ((1, 1, 1), (2, 3, 1), (4, 4, 4), (5, 2, 3)):
        coords, conn = smesh.structured_hex_mesh(nx, ny, nz)
        nn = coords.shape[0]
        rp, ci, sl = oracle.pattern(nn, conn)
        assert ci.size == 9 * (3 * nx + 1) * (3 * ny + 1) * (3 * nz + 1)
        lens = np.diff(rp)
        assert set(lens.tolist()) <= {24, 36, 54, 81}
        dense = np.zeros((3 * nn, 3 * nn), dtype=bool)
        for e in conn:
            d = (3 * e[:, None] + np.arange(3)).ravel()
            dense[np.ix_(d, d)] = True
        r, c = np.nonzero(dense)                                              # row-major => sorted by (row, col)
        assert np.array_equal(ci, c.astype(np.int32))
        assert np.array_equal(rp, np.concatenate([[0], np.cumsum(dense.sum(1))]).astype(np.int32))
        d = (3 * conn[:, :, None] + np.arange(3)).reshape(-1, 24)
        rows = np.repeat(d, 24, axis=1).reshape(-1, 576); cols = np.tile(d, (1, 24))
        assert np.array_equal(ci[sl], cols)
        assert np.all((rp[rows] <= sl) & (sl < rp[rows + 1]))


def test_assembly_brute_force_and_order_invariance(swift_mat):               # P15
    c = synth.make_config(1)
    coords, conn, u, hin = c["coords"], c["conn"], c["u"], c["hist_in"]
    nn = coords.shape[0]
    rp, ci, sl = oracle.pattern(nn, conn)
    out = oracle.assemble(coords, conn, u, hin, swift_mat, rp, ci, 0)
    Kd = np.zeros((3 * nn, 3 * nn)); Rd = np.zeros(3 * nn)
    for e in range(conn.shape[0]):
        Re, Ke, _, _ = oracle.element(coords[conn[e]], u[conn[e]], hin[e], swift_mat, 0)
        d = (3 * conn[e][:, None] + np.arange(3)).ravel()
        Kd[np.ix_(d, d)] += Ke; Rd[d] += Re
    from scipy.sparse import csr_matrix
    Kc = csr_matrix((out["csr_vals"], ci, rp), shape=(3 * nn, 3 * nn)).toarray()
    assert np.abs(Kc - Kd).max() < 1e-14 * np.abs(Kd).max()
    assert np.abs(out["residual"] - Rd).max() < 1e-13 * np.abs(Rd).max()
    assert np.abs(Kc - Kc.T).max() < 1e-13 * np.abs(Kd).max()                 # P14: global symmetry, fbar=0
    perm = synth.rng.permutation(3, 10, conn.shape[0])
    rp2, ci2, _ = oracle.pattern(nn, conn[perm])
    assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2)
    out2 = oracle.assemble(coords, conn[perm], u, hin[perm], swift_mat, rp2, ci2, 0)
    assert np.abs(out2["csr_vals"] - out["csr_vals"]).max() < 1e-14 * np.abs(out["csr_vals"]).max()
    assert np.allclose(out2["hist_out"], out["hist_out"][perm], rtol=0, atol=0)
    # sampled-row path agrees with the full assemble
    node_elems = {n: np.nonzero((conn == n).any(axis=1))[0].tolist() for n in (0, 31, 62, 124)}
    rows, _ = oracle.assemble_rows(coords, conn, u, hin, swift_mat, rp, ci, list(node_elems), node_elems, 0)
    for n, (res, rws) in rows.items():
        assert np.allclose(res, out["residual"][3 * n:3 * n + 3], rtol=1e-14, atol=1e-12)
        for i in range(3):
            assert np.allclose(rws[i], out["csr_vals"][rp[3 * n + i]:rp[3 * n + i + 1]], rtol=1e-14, atol=1e-9)
