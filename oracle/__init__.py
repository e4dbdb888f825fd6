"""ORACLE — test infrastructure only (see fem_oracle.c header).

ctypes wrapper around oracle/fem_oracle.c.  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / `--impl reference` leg may import this package.
It imports nothing from paper_2606_17390_b200.
"""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fem_oracle.c")
_LIB = os.path.join(_HERE, "libfem_oracle.so")
NPAR = 16


def build(force=False):
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int)
_lp = C.POINTER(C.c_longlong)


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_shape_grad.restype = C.c_double
        L.orc_shape_grad.argtypes = [_dp, C.c_int, _dp]
        L.orc_logstrain.argtypes = [_dp] * 4
        L.orc_hill_mandel.argtypes = [_dp, _dp]
        L.orc_flow.argtypes = [_dp, C.c_double, _dp, _dp]
        L.orc_return_map.restype = C.c_int
        L.orc_return_map.argtypes = [_dp, _dp, _dp, C.c_double, _dp, _dp, _dp, _dp, _dp, _ip, _ip]
        L.orc_return_map_c2.restype = C.c_int
        L.orc_return_map_c2.argtypes = [_dp, _dp, _dp, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double,
                                        _dp, _dp, _dp, _dp, _ip]
        L.orc_cep_implicit.argtypes = [_dp, _dp, C.c_double, C.c_double, _dp]
        L.orc_divdiff.argtypes = [_dp, _dp, _dp]
        L.orc_postprocess.argtypes = [_dp] * 6
        L.orc_point.restype = C.c_int
        L.orc_point.argtypes = [_dp] * 9 + [_ip]
        L.orc_element.restype = C.c_int
        L.orc_element.argtypes = [_dp, _dp, _dp, _dp, C.c_int, _dp, _dp, _dp, _lp]
        L.orc_pattern.restype = C.c_longlong
        L.orc_pattern.argtypes = [C.c_longlong, C.c_longlong, _ip, _ip, _ip, _ip]
        L.orc_assemble.restype = C.c_int
        L.orc_assemble.argtypes = [C.c_longlong, _dp, C.c_longlong, _ip, C.c_int, _dp, _dp, _dp, C.c_longlong, _ip, _ip,
                                   _dp, _dp, _dp, _lp]
        L.orc_num_threads.restype = C.c_int
        L.orc_barlat_phi_eig.restype = C.c_double
        L.orc_barlat_phi_eig.argtypes = [_dp, _dp]
        L.orc_barlat_derivs.argtypes = [_dp] * 5
        L.orc_yield_eval.argtypes = [_dp] * 6
        L.orc_return_map_gen.restype = C.c_int
        L.orc_return_map_gen.argtypes = [_dp, _dp, _dp, _dp, C.c_double, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double,
                                         _dp, _dp, _dp, _dp, _dp, _ip, _ip, _dp]
        L.orc_point_yld.restype = C.c_int
        L.orc_point_yld.argtypes = [_dp] * 10 + [_ip]
        L.orc_element_yld.restype = C.c_int
        L.orc_element_yld.argtypes = [_dp, _dp, _dp, _dp, _dp, C.c_int, _dp, _dp, _dp, _lp]
        L.orc_assemble_yld.restype = C.c_int
        L.orc_assemble_yld.argtypes = [C.c_longlong, _dp, C.c_longlong, _ip, C.c_int, _dp, _dp, _dp, C.c_longlong, _dp, _ip,
                                       _ip, _dp, _dp, _dp, _lp]
        L.orc_hill_from_lankford.argtypes = [C.c_double] * 3 + [_dp]
        _lib = L
    return _lib


def _f(a):
    return np.ascontiguousarray(a, dtype=np.float64)


# ---------------------------------------------------------------- materials
def hill_from_lankford(r0, r45, r90):
    out = np.empty(6)
    lib().orc_hill_from_lankford(float(r0), float(r45), float(r90), _d(out))
    return out


def mat_record(E, nu, r, law, h0, h1, h2, quat=(1.0, 0.0, 0.0, 0.0)):
    """One 16-double record: E,nu,r11,r22,r33,r12,r23,r13,law(0 Voce,1 Swift),h0,h1,h2,q0..q3."""
    return np.array([E, nu, *r, law, h0, h1, h2, *quat], dtype=np.float64)


def mat_from_desc(desc, n_elems):
    """matdesc (synth.configs) -> [n_mat,16] records using the oracle's own Lankford helper."""
    per_elem = any(np.ndim(v) > 0 for v in desc.values())
    n = n_elems if per_elem else 1
    g = lambda k: np.broadcast_to(np.asarray(desc[k], dtype=np.float64), (n,))
    out = np.empty((n, NPAR))
    for e in range(n):
        r = hill_from_lankford(g("r0")[e], g("r45")[e], g("r90")[e])
        out[e] = mat_record(g("E")[e], g("nu")[e], r, g("law")[e], g("h0")[e], g("h1")[e], g("h2")[e])
    return out


# ---------------------------------------------------------------- point-level pieces
def shape_grad(X, q):
    X = _f(X); G = np.empty((8, 3))
    w = lib().orc_shape_grad(_d(X), int(q), _d(G))
    return G, w


def logstrain(F):
    F = _f(F); eps = np.empty(6); lam = np.empty(3); R = np.empty((3, 3))
    lib().orc_logstrain(_d(F), _d(eps), _d(lam), _d(R))
    return eps, lam, R


def hill_mandel(mat):
    mat = _f(mat); H = np.empty((6, 6))
    lib().orc_hill_mandel(_d(mat), _d(H))
    return H


def flow(mat, alpha):
    mat = _f(mat); s = C.c_double(); d = C.c_double()
    lib().orc_flow(_d(mat), float(alpha), C.byref(s), C.byref(d))
    return s.value, d.value


def return_map(mat, eps, epn, alphan):
    mat, eps, epn = _f(mat), _f(eps), _f(epn)
    T = np.empty(6); ep = np.empty(6); Cep = np.empty((6, 6))
    a = C.c_double(); dg = C.c_double(); it = C.c_int(); nc = C.c_int()
    pl = lib().orc_return_map(_d(mat), _d(eps), _d(epn), float(alphan), _d(T), _d(ep), C.byref(a), C.byref(dg), _d(Cep),
                              C.byref(it), C.byref(nc))
    return dict(plastic=bool(pl), T=T, ep=ep, alpha=a.value, dgam=dg.value, Cep=Cep, iters=it.value, nonconv=nc.value)


def return_map_c2(mat, eps, epn, alphan, tol=1e-12, kmax=60, jmax=10, beta=1e-4, eta=0.1):
    mat, eps, epn = _f(mat), _f(eps), _f(epn)
    T = np.empty(6); a = C.c_double(); dg = C.c_double(); res = np.full(kmax + 1, np.nan); nls = C.c_int()
    k = lib().orc_return_map_c2(_d(mat), _d(eps), _d(epn), float(alphan), tol, kmax, jmax, beta, eta, _d(T), C.byref(a),
                                C.byref(dg), _d(res), C.byref(nls))
    return dict(iters=k, T=T, alpha=a.value, dgam=dg.value, resnorms=res, n_linesearch=nls.value)


def cep_implicit(mat, T, alpha, dgam):
    mat, T = _f(mat), _f(T); Cep = np.empty((6, 6))
    lib().orc_cep_implicit(_d(mat), _d(T), float(alpha), float(dgam), _d(Cep))
    return Cep


def divdiff(lam):
    lam = _f(lam); th = np.empty((3, 3)); ga = np.empty((3, 3, 3))
    lib().orc_divdiff(_d(lam), _d(th), _d(ga))
    return th, ga


def postprocess(lam, R, T, Cep):
    lam, R, T, Cep = _f(lam), _f(R), _f(T), _f(Cep)
    S = np.empty(6); CL = np.empty((6, 6))
    lib().orc_postprocess(_d(lam), _d(R), _d(T), _d(Cep), _d(S), _d(CL))
    return S, CL


def _bar(bar):
    return None if bar is None else _f(bar)


def point(mat, F, hin, bar=None):
    mat, F, hin, bar = _f(mat), _f(F), _f(hin), _bar(bar)
    P = np.empty((3, 3)); A = np.empty((3, 3, 3, 3)); hout = np.empty(7); S = np.empty(6); T = np.empty(6); CL = np.empty((6, 6))
    it = C.c_int()
    fl = lib().orc_point_yld(_d(mat), None if bar is None else _d(bar), _d(F), _d(hin), _d(P), _d(A), _d(hout), _d(S), _d(T),
                             _d(CL), C.byref(it))
    return dict(flags=fl, P=P, A=A, hist=hout, S=S, T=T, CL=CL, iters=it.value)


def element(X, u, hin, mat, fbar=0, bar=None):
    X, u, hin, mat, bar = _f(X), _f(u), _f(hin), _f(mat), _bar(bar)
    Re = np.empty(24); Ke = np.empty((24, 24)); hout = np.empty((8, 7)); st = np.zeros(4, dtype=np.int64)
    lib().orc_element_yld(_d(X), _d(u), _d(hin), _d(mat), None if bar is None else _d(bar), int(fbar), _d(Re), _d(Ke), _d(hout),
                          st.ctypes.data_as(_lp))
    return Re, Ke, hout, st


# ---------------------------------------------------------------- Yld2004-18p
NBAR = 20
# PAPER.md:471-477 Table 2: c'12,c'13,c'21,c'23,c'31,c'32,c'44,c'55,c'66 ; the same nine for C'' ; m
TABLE2_CP = (-0.069888, 0.936408, 0.079143, 1.003060, 0.524741, 1.363180, 1.023770, 1.069060, 0.954322)
TABLE2_CPP = (0.981171, 0.476741, 0.575316, 0.866827, 1.145010, -0.079294, 1.051660, 1.147100, 1.404620)


def barlat_record(cp=TABLE2_CP, cpp=TABLE2_CPP, m=8):
    """One 20-double record: c' (9), c'' (9), m, 0."""
    return np.array([*cp, *cpp, float(m), 0.0], dtype=np.float64)


def barlat_phi_eig(bar, Tm):
    """Eq.(12) by its definition (eigenvalues); Tm = material-frame stress, Mandel 6-vector."""
    bar, Tm = _f(bar), _f(Tm)
    return lib().orc_barlat_phi_eig(_d(bar), _d(Tm))


def barlat_derivs(bar, Tm, hess=True):
    bar, Tm = _f(bar), _f(Tm)
    phi = C.c_double(); N = np.empty(6); H = np.empty((6, 6))
    lib().orc_barlat_derivs(_d(bar), _d(Tm), C.byref(phi), _d(N), _d(H) if hess else None)
    return phi.value, N, (H if hess else None)


def yield_eval(mat, bar, T6):
    """Global frame, T6 tensor components -> phi, N (Mandel), dN/dT (6x6 Mandel); bar None = Hill-48."""
    mat, T6, bar = _f(mat), _f(T6), _bar(bar)
    phi = C.c_double(); N = np.empty(6); H = np.empty((6, 6))
    lib().orc_yield_eval(_d(mat), None if bar is None else _d(bar), _d(T6), C.byref(phi), _d(N), _d(H))
    return phi.value, N, H


def return_map_gen(mat, bar, eps, epn, alphan, tol=1e-14, kmax=100, jmax=20, beta=1e-4, eta=0.1):
    """Alg. C1/C2 step by step (8 unknowns, line search of App. B) for either yield function."""
    mat, eps, epn, bar = _f(mat), _f(eps), _f(epn), _bar(bar)
    T = np.empty(6); ep = np.empty(6); Cep = np.empty((6, 6)); tr = np.empty((kmax + 1, 3))
    a = C.c_double(); dg = C.c_double(); it = C.c_int(); nc = C.c_int()
    pl = lib().orc_return_map_gen(_d(mat), None if bar is None else _d(bar), _d(eps), _d(epn), float(alphan), tol, kmax, jmax,
                                  beta, eta, _d(T), _d(ep), C.byref(a), C.byref(dg), _d(Cep), C.byref(it), C.byref(nc), _d(tr))
    return dict(plastic=bool(pl), T=T, ep=ep, alpha=a.value, dgam=dg.value, Cep=Cep, iters=it.value, nonconv=nc.value, trace=tr)


# ---------------------------------------------------------------- mesh-level
def pattern(n_nodes, conn, with_slots=True):
    conn = np.ascontiguousarray(conn, dtype=np.int32)
    ne = conn.shape[0]
    row_ptr = np.empty(3 * n_nodes + 1, dtype=np.int32)
    nnz = lib().orc_pattern(n_nodes, ne, _i(conn), _i(row_ptr), None, None)
    col_idx = np.empty(nnz, dtype=np.int32)
    slots = np.empty((ne, 576), dtype=np.int32) if with_slots else None
    lib().orc_pattern(n_nodes, ne, _i(conn), _i(row_ptr), _i(col_idx), _i(slots) if with_slots else None)
    return row_ptr, col_idx, slots


def assemble(coords, conn, u, hist_in, mat, row_ptr, col_idx, fbar=0, bar=None):
    coords, u, hist_in, mat = _f(coords), _f(u), _f(hist_in), _f(mat).reshape(-1, NPAR)
    if bar is not None:
        bar = _f(bar).reshape(-1, NBAR)
        assert bar.shape[0] == mat.shape[0]
    conn = np.ascontiguousarray(conn, dtype=np.int32)
    nn, ne = coords.shape[0], conn.shape[0]
    res = np.empty(3 * nn); vals = np.empty(col_idx.shape[0]); hout = np.empty((ne, 8, 7)); st = np.zeros(4, dtype=np.int64)
    rc = lib().orc_assemble_yld(nn, _d(coords), ne, _i(conn), int(fbar), _d(u), _d(hist_in), _d(mat), mat.shape[0],
                                None if bar is None else _d(bar), _i(row_ptr), _i(col_idx), _d(res), _d(vals), _d(hout),
                                st.ctypes.data_as(_lp))
    if rc != 0:
        raise MemoryError("orc_assemble")
    return dict(residual=res, csr_vals=vals, hist_out=hout,
                stats=dict(n_plastic=int(st[0]), n_nonconverged=int(st[1]), n_detF_nonpos=int(st[2]), max_local_iters=int(st[3])))


def assemble_rows(coords, conn, u, hist_in, mat, row_ptr, col_idx, nodes, node_elems, fbar=0, bar=None):
    """Sampled check at full size: rows 3n..3n+2 of K and R for each node n in `nodes`, summing the incident
    elements (node_elems[n], ascending) one by one.  Returns {node: (res[3], rows list of 3 arrays)} and the
    hist_out of every touched element."""
    mat = _f(mat).reshape(-1, NPAR)
    if bar is not None:
        bar = _f(bar).reshape(-1, NBAR)
    out, hist = {}, {}
    cache = {}
    for n in nodes:
        res = np.zeros(3, dtype=np.longdouble)
        rows = [np.zeros(row_ptr[3 * n + i + 1] - row_ptr[3 * n + i], dtype=np.longdouble) for i in range(3)]
        for e in sorted(node_elems[n]):
            if e not in cache:
                c = conn[e].astype(np.int64)
                cache[e] = element(coords[c], u[c], hist_in[e], mat[0 if mat.shape[0] == 1 else e], fbar,
                                   bar=None if bar is None else bar[0 if bar.shape[0] == 1 else e])
            Re, Ke, ho, _ = cache[e]
            hist[e] = ho
            I = int(np.where(conn[e] == n)[0][0])
            for i in range(3):
                res[i] += Re[3 * I + i]
                cols = col_idx[row_ptr[3 * n + i]:row_ptr[3 * n + i + 1]]
                for K in range(8):
                    for k in range(3):
                        j = np.searchsorted(cols, 3 * conn[e][K] + k)
                        rows[i][j] += Ke[3 * I + i, 3 * K + k]
        out[n] = (res.astype(np.float64), [r.astype(np.float64) for r in rows])
    return out, hist


def num_threads():
    return lib().orc_num_threads()
