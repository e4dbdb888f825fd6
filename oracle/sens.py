"""ORACLE — test infrastructure only.  SURVEY.md §8(f) NEXT-3: parameter sensitivities of the element path.

What is computed.  One call of the path is the map  Phi : (u, hist_in, theta) -> (R, hist_out)  (Eq.(34)-(35) PAPER.md:253-257
with Alg. C1 :889-918 at every Gauss point).  Alg. 1 needs its vector-Jacobian products: with lambda the
adjoint of Eq.(51) :366 and mu a cotangent on hist_out,

    g_theta   = (dR/dtheta)^T lambda + (dhist_out/dtheta)^T mu          Eq.(49) :355   "(dR^n/dtheta)^T lambda^n"
    g_hist_in = (dR/dhist_in)^T lambda + (dhist_out/dhist_in)^T mu      the history leg of (dR^{n+1}/du^n)^T lambda^{n+1}
    g_u       = (dhist_out/du)^T mu                                     the displacement leg of the same term, Eq.(50)-(51)
    (g_u_full = g_u + K^T lambda, K = dR/du the tangent of Eq.(39); returned too because it is a strong pin: = K lambda)

Reading G17: the paper writes R^n(u^n, u^{n-1}, theta) with the internal variables "implicitly accounted for"
(:323).  R^{n+1} depends on u^n only through the history h^n = hist_out of step n, which also depends on h^{n-1}; the exact
discrete adjoint therefore carries mu backwards:  mu^{n-1} = g_hist_in(lambda^n, mu^n).  `adjoint_gradient` below does that;
it is checked against central differences of J (Eq.(52) :412, Table 6 :531-545) in tests/test_oracle_sens.py.

How.  The definition of a VJP is J^T cot with J the Jacobian of the map, so the oracle forms the Jacobian of the point map
(F, hist_in, theta) -> (P, hist_out) explicitly as a dense 16 x 27 matrix by the chain rule, each factor a plain matrix:
dC/dF, d eps/dC = P_L/2, the return map by App. D (Eq.(D4)-(D7) :1002-1019: J_y dy = -dG/dz dz on the
paper's 8 unknowns y = [T, alpha, dgam], G of Eq.(19)-(24) :176-196), dS = P_L:dT + (T:L_L):dC/2 (Eq.(25) :204), dP = dF S + F dS
(Eq.(26) :208), and multiplies its transpose with the cotangent.  theta = (E, nu, r11, r22, r33, r12, r23, r13, h0, h1, h2)
(Tables 3/5: the identified parameters are Hill ratios and hardening constants); the orientation quaternion and the
law switch are not differentiated (their gradient entries are 0).  Hill-48 only; standard element and F-bar (fbar = 1: the
relative-volume coupling of the 8 Gauss points, Eq.(31)-(32) :237-243, is differentiated at element level in `element_vjp`).

Pins (tests/test_oracle_sens.py, -m "not gpu"): central differences of lambda.R + mu.hist_out computed with the C oracle's
assemble (the paper's own check, Eq.(52)); g_u_full(lambda, 0) = K lambda with the oracle's assembled K; elastic closed
forms dT/dE = T/E; the adjoint gradient of a two-step load path against central differences of J.
The fbar = 1 branch inherits reading G12 of the forward path (literal Eq.(35): no external value pins that reading, 'parity
unpinned' there); its derivative is pinned by central differences of the F-bar assemble and by K^T lambda with the assembled
unsymmetric tangent.
Shares nothing with the CUDA path; imports nothing from paper_2606_17390_b200.
"""
import numpy as np

from . import NPAR, shape_grad, logstrain, hill_mandel, flow, return_map, divdiff, postprocess

W = np.sqrt(2.0 / 3.0)
VI = (0, 1, 2, 0, 1, 0)  # (11,22,33,12,23,13)
VJ = (0, 1, 2, 1, 2, 2)
MW = np.array([1.0, 1.0, 1.0, np.sqrt(2.0), np.sqrt(2.0), np.sqrt(2.0)])
THETA_IDX = (0, 1, 2, 3, 4, 5, 6, 7, 9, 10, 11)  # positions of theta in the 16-double material record
NTH = len(THETA_IDX)
M1 = np.array([1.0, 1.0, 1.0, 0.0, 0.0, 0.0])


def t4_to_mandel(T4):
    M = np.empty((6, 6))
    for a in range(6):
        for b in range(6):
            M[a, b] = MW[a] * MW[b] * T4[VI[a], VJ[a], VI[b], VJ[b]]
    return M


def quat_to_rot(q):
    w, x, y, z = np.asarray(q, dtype=np.float64) / np.linalg.norm(q)
    return np.array([[1 - 2 * (y * y + z * z), 2 * (x * y - w * z), 2 * (x * z + w * y)],
                     [2 * (x * y + w * z), 1 - 2 * (x * x + z * z), 2 * (y * z - w * x)],
                     [2 * (x * z - w * y), 2 * (y * z + w * x), 1 - 2 * (x * x + y * y)]])


def hill_basis(quat):
    """Six Mandel matrices M_k with H = sum_k s_k M_k, s_k = 1/r_k^2, k over (11,22,33,12,23,13): Eq.(A2)-(A5) PAPER.md:779-801
    are linear in the s_k (p1 = 2/3 s11, p7 = s12, p4 = (p3-p1-p2)/2, ...), rotated by Eq.(A1) :774."""
    Th = quat_to_rot(quat)
    out = []
    for k in range(6):
        s = np.zeros(6); s[k] = 1.0
        p1, p2, p3, p7, p8, p9 = 2 * s[0] / 3, 2 * s[1] / 3, 2 * s[2] / 3, s[3], s[4], s[5]
        p4, p5, p6 = 0.5 * (p3 - p1 - p2), 0.5 * (p1 - p2 - p3), 0.5 * (p2 - p1 - p3)
        L = np.zeros((3, 3, 3, 3))
        L[0, 0, 0, 0], L[1, 1, 1, 1], L[2, 2, 2, 2] = p1, p2, p3
        L[0, 0, 1, 1] = L[1, 1, 0, 0] = p4
        L[1, 1, 2, 2] = L[2, 2, 1, 1] = p5
        L[0, 0, 2, 2] = L[2, 2, 0, 0] = p6
        for (i, j, p) in ((0, 1, p7), (1, 2, p8), (0, 2, p9)):
            L[i, j, i, j] = L[i, j, j, i] = L[j, i, i, j] = L[j, i, j, i] = 0.5 * p
        G = np.einsum('ia,jb,kc,ld,abcd->ijkl', Th, Th, Th, Th, L)
        out.append(t4_to_mandel(G))
    return out


def elast(E, nu):
    """Mandel matrices of E (Eq.(8), isotropic) and of dE/dE, dE/dnu."""
    mu, la = E / (2 * (1 + nu)), E * nu / ((1 + nu) * (1 - 2 * nu))
    dmu = -E / (2 * (1 + nu) ** 2)
    dla = E * (1 + 2 * nu * nu) / ((1 + nu) ** 2 * (1 - 2 * nu) ** 2)
    I6, mm = np.eye(6), np.outer(M1, M1)
    return la * mm + 2 * mu * I6, (la * mm + 2 * mu * I6) / E, dla * mm + 2 * dmu * I6


def flow_param_derivs(mat, alpha):
    """d sigma_flow / d(h0,h1,h2) at alpha: Voce sigma0+Q(1-exp(-b a)) (Eq.(10) :121), Swift K(eps0+a)^n (BASELINE configs)."""
    h0, h1, h2 = mat[9], mat[10], mat[11]
    if mat[8] == 0.0:
        e = np.exp(-h2 * alpha)
        return np.array([1.0, 1.0 - e, h1 * alpha * e])
    b = h1 + alpha
    return np.array([b ** h2, h0 * h2 * b ** (h2 - 1), h0 * b ** h2 * np.log(b)])


def return_map_jacobian(mat, eps, hin):
    """D(T, ep_out, alpha_out) / D(eps, ep_n, alpha_n, theta): 13 x 24, tensors as Mandel vectors.  App. D :1002-1019."""
    mat = np.asarray(mat, dtype=np.float64)
    rm = return_map(mat, eps, hin[:6], hin[6])
    E6, dE_E, dE_nu = elast(mat[0], mat[1])
    Tm = rm['T'] * MW
    ee = np.linalg.solve(E6, Tm)            # elastic strain eps - ep_{n+1}
    J = np.zeros((13, 13 + NTH))
    if not rm['plastic']:
        J[0:6, 0:6] = E6
        J[0:6, 6:12] = -E6
        J[0:6, 13 + 0] = dE_E @ ee
        J[0:6, 13 + 1] = dE_nu @ ee
        J[6:12, 6:12] = np.eye(6)
        J[12, 12] = 1.0
        return J, rm
    dg, al = rm['dgam'], rm['alpha']
    H6 = hill_mandel(mat)
    r = mat[2:8]
    Mk = hill_basis(mat[12:16])
    dH = [-2.0 / r[k] ** 3 * Mk[k] for k in range(6)]          # dH/dr_k, s_k = 1/r_k^2
    phi = np.sqrt(Tm @ H6 @ Tm)
    N = H6 @ Tm / phi                                           # Eq.(13) :141
    dNdT = (H6 - np.outer(N, N)) / phi
    sf, dsf = flow(mat, al)
    dsy = W * dsf                                               # sigma_y = sqrt(2/3) sigma_flow (reading G2)
    # J_y on y = [T(6), alpha, dgam]  (Eq.(D4))
    Jy = np.zeros((8, 8))
    Jy[0:6, 0:6] = np.eye(6) + dg * E6 @ dNdT
    Jy[0:6, 7] = E6 @ N
    Jy[6, 6], Jy[6, 7] = 1.0, -W
    Jy[7, 0:6], Jy[7, 6] = N, -dsy
    # dG/dz, z = [eps(6), ep_n(6), alpha_n, theta(11)]
    Gz = np.zeros((8, 13 + NTH))
    Gz[0:6, 0:6] = -E6
    Gz[0:6, 6:12] = E6
    Gz[6, 12] = -1.0
    Gz[0:6, 13 + 0] = -dE_E @ ee
    Gz[0:6, 13 + 1] = -dE_nu @ ee
    dphi_r, dN_r = np.zeros(6), np.zeros((6, 6))
    for k in range(6):
        dphi_r[k] = Tm @ dH[k] @ Tm / (2 * phi)
        dN_r[:, k] = dH[k] @ Tm / phi - N * dphi_r[k] / phi
        Gz[0:6, 13 + 2 + k] = dg * E6 @ dN_r[:, k]
        Gz[7, 13 + 2 + k] = dphi_r[k]
    Gz[7, 13 + 8:13 + 11] = -W * flow_param_derivs(mat, al)
    dy = -np.linalg.solve(Jy, Gz)                               # Eq.(D7)
    J[0:6] = dy[0:6]
    J[12] = dy[6]
    # ep_{n+1} = ep_n + dgam N(T, r)   (Eq.(20) :180)
    J[6:12] = np.outer(N, dy[7]) + dg * dNdT @ dy[0:6]
    J[6:12, 6:12] += np.eye(6)
    J[6:12, 13 + 2:13 + 8] += dg * dN_r
    return J, rm


def point_jacobian(mat, F, hin):
    """D(P[9 row-major iJ], hist_out[7]) / D(F[9], hist_in[7], theta[11]) as a dense 16 x 27 matrix."""
    F = np.asarray(F, dtype=np.float64).reshape(3, 3)
    hin = np.asarray(hin, dtype=np.float64)
    eps, lam, R = logstrain(F)
    th, _ = divdiff(lam)
    PL4 = np.einsum('ab,ia,jb,ka,lb->ijkl', 2 * th, R, R, R, R)     # (P_L:A)^_ab = 2 g[a,b] A^_ab
    PL4 = 0.5 * (PL4 + PL4.transpose(0, 1, 3, 2))
    PL = t4_to_mandel(PL4)
    Jrm, rm = return_map_jacobian(mat, eps, hin)
    S6, CL = postprocess(lam, R, rm['T'], rm['Cep'])
    CLgeo = CL - PL @ rm['Cep'] @ PL                                 # T : L_L alone
    S = np.zeros((3, 3))
    for m in range(6):
        S[VI[m], VJ[m]] = S[VJ[m], VI[m]] = S6[m]
    # dC_m / dF  (C = F^T F)
    MCF = np.zeros((6, 9))
    for m in range(6):
        K, L = VI[m], VJ[m]
        for i in range(3):
            MCF[m, i * 3 + K] += MW[m] * F[i, L]
            MCF[m, i * 3 + L] += MW[m] * F[i, K]
    # z = [eps, ep_n, alpha_n, theta] as a function of x = [F, hist_in, theta]
    Z = np.zeros((13 + NTH, 9 + 7 + NTH))
    Z[0:6, 0:9] = 0.5 * PL @ MCF
    Z[6:12, 9:15] = np.diag(MW)
    Z[12, 15] = 1.0
    Z[13:, 16:] = np.eye(NTH)
    D = Jrm @ Z                                                      # d(T_m, ep_m, alpha)/dx
    dS = PL @ D[0:6]
    dS[:, 0:9] += 0.5 * CLgeo @ MCF
    J = np.zeros((16, 9 + 7 + NTH))
    for i in range(3):
        for Jc in range(3):
            row = i * 3 + Jc
            for K in range(3):
                J[row, i * 3 + K] += S[K, Jc]                        # dF_iK S_KJ
                m = [a for a in range(6) if (VI[a], VJ[a]) in ((K, Jc), (Jc, K))][0]
                J[row] += F[i, K] * dS[m] / MW[m]
    J[9:15] = D[6:12] / MW[:, None]
    J[15] = D[12]
    return J, rm


def element_vjp(X, u, hin, mat, lam_e, mu_e, fbar=0):
    """VJPs of one element: X[8,3], u[8,3], hin[8,7], lam_e[8,3], mu_e[8,7] ->
    g_u[8,3] (history leg only), g_u_full[8,3], g_hist[8,7], g_theta[11].
    fbar = 1 (Eq.(31)-(32) PAPER.md:237-243, reading G12: R^e contracts P(Fbar) with grad_0 N): the point map is evaluated at
    Fbar_q = c_q F_q, c_q = (Jbar/J_q)^(1/3), Jbar = sum_p w_p J_p / V, and the cotangent on Fbar_q is taken back to the F_p by
    dFbar_q = c_q dF_q + F_q c_q/3 (dJbar/Jbar - dJ_q/J_q), dJ_p = J_p F_p^-T : dF_p."""
    X, u, hin = np.asarray(X, dtype=np.float64), np.asarray(u, dtype=np.float64), np.asarray(hin, dtype=np.float64)
    g_u, g_uf, g_h, g_t = np.zeros((8, 3)), np.zeros((8, 3)), np.zeros((8, 7)), np.zeros(NTH)
    Gs, ws, Fs = [], [], []
    for q in range(8):
        G, w = shape_grad(X, q)
        Gs.append(G); ws.append(w); Fs.append(np.eye(3) + u.T @ G)                # Eq.(30) :228
    if fbar:
        V = sum(ws)
        Js = [np.linalg.det(F) for F in Fs]
        Jbar = sum(w * J for w, J in zip(ws, Js)) / V                          # Eq.(31) :237
        cs = [(Jbar / J) ** (1.0 / 3.0) for J in Js]                              # Eq.(32) :243
    else:
        cs = [1.0] * 8
    gFb_full, gFb_hist = [], []
    for q in range(8):
        J, _ = point_jacobian(mat, cs[q] * Fs[q], hin[q])
        Pbar = ws[q] * (lam_e.T @ Gs[q])                                          # R^e_Ii = sum_q w P_iJ G_IJ (Eq.(35) :257)
        cot = np.concatenate([Pbar.ravel(), mu_e[q]])
        g = J.T @ cot
        gFb_full.append(g[0:9].reshape(3, 3))
        gFb_hist.append((J[9:, 0:9].T @ mu_e[q]).reshape(3, 3))
        g_h[q] = g[9:16]
        g_t += g[16:]
    for gFb, out in ((gFb_full, g_uf), (gFb_hist, g_u)):
        if fbar:
            s = [cs[q] / 3.0 * float(np.sum(gFb[q] * Fs[q])) for q in range(8)]
            S = sum(s)
        for q in range(8):
            gF = cs[q] * gFb[q]
            if fbar:
                FiT = np.linalg.inv(Fs[q]).T
                gF = gF - s[q] * FiT + (S / Jbar) * (ws[q] * Js[q] / V) * FiT
            out += (gF @ Gs[q].T).T
    return g_u, g_uf, g_h, g_t


def assemble_vjp(coords, conn, u, hist_in, mat, lam, mu, elems=None, fbar=0):
    """Mesh level, elements in ascending id.  mat [n_mat,16] (n_mat = 1 or n_elems).  Returns dict with g_u, g_u_full [n_nodes,3],
    g_hist_in [n_elems,8,7], g_mat [n_mat,16] and g_mat_abs (sum of |element contributions|, the scale a tolerance refers to).
    `elems` restricts the work to a subset of elements (the other entries stay 0)."""
    coords, u = np.asarray(coords, dtype=np.float64), np.asarray(u, dtype=np.float64).reshape(-1, 3)
    conn = np.asarray(conn)
    mat = np.asarray(mat, dtype=np.float64).reshape(-1, NPAR)
    ne = conn.shape[0]
    lam = np.zeros_like(u) if lam is None else np.asarray(lam, dtype=np.float64).reshape(-1, 3)
    mu = np.zeros((ne, 8, 7)) if mu is None else np.asarray(mu, dtype=np.float64).reshape(ne, 8, 7)
    hist_in = np.asarray(hist_in, dtype=np.float64).reshape(ne, 8, 7)
    g_u, g_uf = np.zeros_like(u), np.zeros_like(u)
    g_h = np.zeros((ne, 8, 7))
    g_m, g_ma = np.zeros((mat.shape[0], NPAR)), np.zeros((mat.shape[0], NPAR))
    for e in (range(ne) if elems is None else elems):
        c = conn[e].astype(np.int64)
        m = 0 if mat.shape[0] == 1 else e
        a, b, g_h[e], t = element_vjp(coords[c], u[c], hist_in[e], mat[m], lam[c], mu[e], fbar=fbar)
        for I in range(8):
            g_u[c[I]] += a[I]
            g_uf[c[I]] += b[I]
        g_m[m, list(THETA_IDX)] += t
        g_ma[m, list(THETA_IDX)] += np.abs(t)
    return dict(g_u=g_u, g_u_full=g_uf, g_hist_in=g_h, g_mat=g_m, g_mat_abs=g_ma)
