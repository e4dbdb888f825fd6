"""Seeded displacement and history fields.  Closed-form
analytic fields only; "peak strain" is measured on the analytic gradient at
element centroids, no FEM arithmetic here."""
import numpy as np
from . import rng

S = rng.STREAM


def affine_matrix(seed, norm):
    A = rng.normal(seed, S["affine"], np.arange(9)).reshape(3, 3)
    return norm * A / np.linalg.norm(A)


def _modes(seed, nmodes=3):
    """Random unit amplitude vectors a_k, wave vectors kappa_k in {1,2}^3, phases."""
    a = rng.normal(seed, S["field_dir"], np.arange(3 * nmodes)).reshape(nmodes, 3)
    a /= np.linalg.norm(a, axis=1, keepdims=True)
    kap = 1.0 + np.floor(2.0 * rng.uniform(seed, S["field_k"], np.arange(3 * nmodes))).reshape(nmodes, 3)
    ph = 2.0 * np.pi * rng.uniform(seed, S["field_phase"], np.arange(nmodes))
    return a, kap, ph


def smooth_field(seed, X, L, xc=None, width=0.05):
    """s(X)=sum_k a_k sin(2 pi kappa_k.Xhat + phi_k), optionally times the
    envelope m(xhat)=0.5(1-tanh((xhat-xc)/width)).  Returns (u, grad_u) with
    grad_u[n,i,J] = d u_i / d X_J, both for unit amplitude."""
    a, kap, ph = _modes(seed)
    Xh = X / L
    u = np.zeros_like(X)
    g = np.zeros(X.shape + (3,))
    for k in range(a.shape[0]):
        arg = 2.0 * np.pi * (Xh @ kap[k]) + ph[k]
        u += np.sin(arg)[:, None] * a[k]
        g += (np.cos(arg)[:, None, None] * a[k][None, :, None]) * (2.0 * np.pi * kap[k] / L)[None, None, :]
    if xc is not None:
        th = np.tanh((Xh[:, 0] - xc) / width)
        m = 0.5 * (1.0 - th)
        dm = -0.5 * (1.0 - th * th) / (width * L[0])
        g = m[:, None, None] * g
        g[:, :, 0] += u * dm[:, None]
        u = m[:, None] * u
    return u, g


def scaled_smooth_displacement(seed, coords, conn, L, peak_strain, xc=None, affine=None):
    """u = scale*(affine X + s(X)) with scale such that max over element
    centroids of ||sym grad u||_F equals peak_strain."""
    cen = coords[conn.astype(np.int64)].mean(axis=1)
    _, gc = smooth_field(seed, cen, L, xc)
    if affine is not None:
        gc = gc + affine[None]
    sym = 0.5 * (gc + np.swapaxes(gc, 1, 2))
    peak = np.sqrt((sym * sym).sum(axis=(1, 2))).max()
    scale = peak_strain / peak
    u, _ = smooth_field(seed, coords, L, xc)
    if affine is not None:
        u = u + coords @ affine.T
    return scale * u


def history_random(seed, n_qp, alpha_max=0.02):
    """alpha~U[0,alpha_max]; eps_p = alpha*0.1*sqrt(3/2)*D/||D||_F, D random
    trace-free symmetric ("Fp near identity").  Layout [n_qp,7] =
    (ep11,ep22,ep33,ep12,ep23,ep13,alpha)."""
    q = np.arange(n_qp, dtype=np.uint64)
    alpha = alpha_max * rng.uniform(seed, S["alpha"], q)
    d = rng.normal(seed, S["ep_dir"], np.arange(6 * n_qp)).reshape(n_qp, 6)
    tr = d[:, :3].mean(axis=1, keepdims=True)
    d[:, :3] -= tr
    nrm = np.sqrt((d[:, :3] ** 2).sum(1) + 2.0 * (d[:, 3:] ** 2).sum(1))
    h = np.empty((n_qp, 7))
    h[:, :6] = d * (alpha * 0.1 * np.sqrt(1.5) / nrm)[:, None]
    h[:, 6] = alpha
    return h


def material_fields(seed, cen, n_fields=4, amp=0.05, lo=0.85, hi=1.15):
    """clip(1+amp*g_j(centroid), lo, hi), g_j unit-variance sums of 8 cosines."""
    out = np.empty((cen.shape[0], n_fields))
    for j in range(n_fields):
        g = np.zeros(cen.shape[0])
        for k in range(8):
            base = 1000 * j + 10 * k
            kk = 1.0 + np.floor(3.0 * rng.uniform(seed, S["mat"], np.arange(3) + base))
            ph = 2.0 * np.pi * rng.uniform(seed, S["mat"], np.array([base + 5]))[0]
            g += np.cos(2.0 * np.pi * (cen @ kk) + ph)
        g *= np.sqrt(2.0 / 8.0)
        out[:, j] = np.clip(1.0 + amp * g, lo, hi)
    return out
