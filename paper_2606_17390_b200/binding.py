"""ctypes binding with the same names as include/fem.h.  Argument marshalling only."""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
NPAR = 16
NBARLAT = 20

ABI_SYMBOLS = ["fem_default_options", "fem_setup", "fem_build_csr_pattern", "fem_assemble", "fem_assemble_barlat", "fem_assemble_host",
               "fem_last_kernel_ms", "fem_launches_per_assemble", "fem_probe_fp64_peak", "fem_destroy", "fem_strerror",
               "fem_last_cuda_error", "fem_hill_from_lankford", "fem_spmv", "fem_apply_dirichlet", "fem_bicgstab", "fem_pcg", "fem_lincomb",
               "fem_default_newton_options", "fem_newton_solve", "fem_assemble_vjp", "fem_adjoint_step", "fem_set_mixed_precision",
               "fem_default_path_options", "fem_load_path", "fem_assemble_static_prepare", "fem_assemble_static"]
STATIC_MAX_ELEMS = 4096          # FEM_STATIC_MAX_ELEMS of include/fem.h
STATIC_SCRATCH_BYTES = 20710144  # FEM_STATIC_SCRATCH_BYTES


class FemOptions(C.Structure):
    _fields_ = [("fbar", C.c_int), ("quad_order", C.c_int), ("tol", C.c_double), ("kmax", C.c_int), ("jmax", C.c_int),
                ("beta", C.c_double), ("eta", C.c_double), ("assembly_mode", C.c_int)]


class FemStats(C.Structure):
    _fields_ = [("n_plastic", C.c_longlong), ("n_nonconverged", C.c_longlong), ("n_detF_nonpos", C.c_longlong),
                ("n_nonfinite", C.c_longlong), ("max_local_iters", C.c_int), ("iter_hist", C.c_longlong * 64)]

    def as_dict(self):
        return dict(n_plastic=self.n_plastic, n_nonconverged=self.n_nonconverged, n_detF_nonpos=self.n_detF_nonpos,
                    n_nonfinite=self.n_nonfinite, max_local_iters=self.max_local_iters, iter_hist=list(self.iter_hist))


class FemNewtonOptions(C.Structure):
    _fields_ = [("rtol", C.c_double), ("atol", C.c_double), ("max_newton", C.c_int), ("lin_rtol", C.c_double),
                ("lin_max_iter", C.c_int), ("linear_solver", C.c_int)]


class FemNewtonReport(C.Structure):
    _fields_ = [("newton_iters", C.c_int), ("converged", C.c_int), ("lin_iters_total", C.c_int), ("lin_failures", C.c_int),
                ("rhs_norm0", C.c_double), ("rhs_norm", C.c_double), ("last_stats", FemStats), ("physics_trouble", C.c_int)]

    def as_dict(self):
        return dict(newton_iters=self.newton_iters, converged=bool(self.converged), lin_iters_total=self.lin_iters_total,
                    lin_failures=self.lin_failures, rhs_norm0=self.rhs_norm0, rhs_norm=self.rhs_norm,
                    last_stats=self.last_stats.as_dict(), physics_trouble=bool(self.physics_trouble))


class FemPathOptions(C.Structure):
    _fields_ = [("dt0", C.c_double), ("dt_min", C.c_double), ("dt_max", C.c_double), ("grow", C.c_double), ("cut", C.c_double),
                ("grow_below", C.c_int), ("max_steps", C.c_int), ("extrapolate", C.c_int), ("newton", FemNewtonOptions)]


class FemPathReport(C.Structure):
    _fields_ = [("steps", C.c_int), ("rejected", C.c_int), ("rejected_physics", C.c_int), ("newton_iters_total", C.c_int),
                ("lin_iters_total", C.c_int), ("t_reached", C.c_double), ("last", FemNewtonReport)]

    def as_dict(self):
        return dict(steps=self.steps, rejected=self.rejected, rejected_physics=self.rejected_physics,
                    newton_iters_total=self.newton_iters_total, lin_iters_total=self.lin_iters_total, t_reached=self.t_reached,
                    last=self.last.as_dict())


class FemError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        msg = lib().fem_strerror(code).decode()
        if code == -6:
            msg += ": " + lib().fem_last_cuda_error().decode()
        super().__init__("%s failed (%d): %s" % (where, code, msg))


_lib = None


def lib_path():
    return os.path.join(_HERE, "libfem_b200.so")


def lib():
    """Loads libfem_b200.so (built in-tree by build.py).  Fails loudly when it is missing: no fallback exists."""
    global _lib
    if _lib is None:
        p = lib_path()
        from . import build as _b
        if _b.needs_build():          # stale or missing: rebuild in-tree (nvcc); a failure is loud, there is no fallback
            try:
                _b.build()
            except Exception as ex:
                if not os.path.exists(p):
                    raise FileNotFoundError(p + " not built and nvcc failed (%s); run `python -m paper_2606_17390_b200.build`"
                                            " — there is no CPU fallback" % (ex,))
                raise
        L = C.CDLL(p)
        vp, ll, dp = C.c_void_p, C.c_longlong, C.POINTER(C.c_double)
        L.fem_default_options.argtypes = [C.POINTER(FemOptions)]
        L.fem_default_options.restype = None
        L.fem_setup.argtypes = [C.POINTER(vp), ll, vp, ll, vp, C.POINTER(FemOptions)]
        L.fem_build_csr_pattern.argtypes = [vp, C.POINTER(ll), C.POINTER(ll), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
        L.fem_assemble.argtypes = [vp, vp, vp, vp, ll, vp, vp, vp, C.POINTER(FemStats), vp]
        L.fem_assemble_barlat.argtypes = [vp, vp, vp, vp, vp, ll, vp, vp, vp, C.POINTER(FemStats), vp]
        L.fem_assemble_static_prepare.argtypes = [vp]
        L.fem_assemble_static.argtypes = [vp, vp, vp, vp, ll, vp, vp, vp, C.POINTER(FemStats), vp]
        L.fem_assemble_host.argtypes = [vp, vp, vp, vp, ll, vp, vp, vp, C.POINTER(FemStats)]
        L.fem_last_kernel_ms.argtypes = [vp, dp]
        L.fem_launches_per_assemble.argtypes = [vp]
        L.fem_probe_fp64_peak.argtypes = [C.c_double, dp, vp]
        L.fem_destroy.argtypes = [vp]
        L.fem_destroy.restype = None
        L.fem_strerror.argtypes = [C.c_int]
        L.fem_strerror.restype = C.c_char_p
        L.fem_last_cuda_error.restype = C.c_char_p
        L.fem_hill_from_lankford.argtypes = [C.c_double] * 3 + [dp]
        L.fem_spmv.argtypes = [vp, vp, vp, vp, vp]
        L.fem_apply_dirichlet.argtypes = [vp, ll, vp, vp, vp, vp, vp]
        L.fem_bicgstab.argtypes = [vp, vp, vp, vp, C.c_double, C.c_int, C.POINTER(C.c_int), dp, vp]
        L.fem_pcg.argtypes = [vp, vp, vp, vp, C.c_double, C.c_int, C.POINTER(C.c_int), dp, vp]
        L.fem_lincomb.argtypes = [vp, C.c_double, vp, C.c_double, vp, vp, vp]
        L.fem_default_newton_options.argtypes = [C.POINTER(FemNewtonOptions)]
        L.fem_default_newton_options.restype = None
        L.fem_newton_solve.argtypes = [vp, vp, vp, vp, ll, ll, vp, vp, vp, C.POINTER(FemNewtonOptions),
                                       C.POINTER(FemNewtonReport), vp]
        L.fem_default_path_options.argtypes = [C.POINTER(FemPathOptions)]
        L.fem_default_path_options.restype = None
        L.fem_load_path.argtypes = [vp, vp, vp, vp, ll, ll, vp, vp, C.POINTER(FemPathOptions), C.POINTER(FemPathReport),
                                    C.POINTER(C.c_double), C.c_int, vp]
        L.fem_assemble_vjp.argtypes = [vp, vp, vp, vp, ll, vp, vp, vp, vp, vp, vp]
        L.fem_set_mixed_precision.argtypes = [vp, C.c_int]
        L.fem_adjoint_step.argtypes = [vp, vp, vp, vp, ll, ll, vp, vp, vp, vp, vp, vp, C.c_double, C.c_int, C.POINTER(C.c_int), vp]
        _lib = L
    return _lib


def _check(rc, where):
    if rc != 0:
        raise FemError(rc, where)


def hill_from_lankford(r0, r45, r90):
    out = (C.c_double * 6)()
    _check(lib().fem_hill_from_lankford(float(r0), float(r45), float(r90), out), "fem_hill_from_lankford")
    return np.array(out[:], dtype=np.float64)


def mat_record(E, nu, r, law, h0, h1, h2, quat=(1.0, 0.0, 0.0, 0.0)):
    """One FEM_NPAR record: E,nu,r11,r22,r33,r12,r23,r13,law(0 Voce,1 Swift),h0,h1,h2,q0..q3."""
    return np.array([E, nu, *r, law, h0, h1, h2, *quat], dtype=np.float64)


def barlat_record(cp, cpp, m):
    """One FEM_NBARLAT record: c'12,c'13,c'21,c'23,c'31,c'32,c'44,c'55,c'66, the same nine of C'', m, 0 (PAPER.md:471-477 order)."""
    return np.array([*cp, *cpp, float(m), 0.0], dtype=np.float64)


def mat_from_desc(desc, n_elems):
    """Material description (synth.configs matdesc) -> [n_mat,16] records via the library's own Lankford helper."""
    per_elem = any(np.ndim(v) > 0 for v in desc.values())
    n = n_elems if per_elem else 1
    g = {k: np.broadcast_to(np.asarray(v, dtype=np.float64), (n,)) for k, v in desc.items()}
    out = np.empty((n, NPAR))
    for e in range(n):
        r = hill_from_lankford(g["r0"][e], g["r45"][e], g["r90"][e])
        out[e] = mat_record(g["E"][e], g["nu"][e], r, g["law"][e], g["h0"][e], g["h1"][e], g["h2"][e])
    return out


def _torch():
    import torch
    return torch


def _stream_ptr():
    torch = _torch()
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t, dtype, numel=None, name="tensor"):
    torch = _torch()
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError("%s must be a CUDA torch tensor" % name)
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError("%s must be contiguous %s" % (name, dtype))
    if numel is not None and t.numel() != numel:
        raise ValueError("%s has %d elements, expected %d" % (name, t.numel(), numel))
    return C.c_void_p(t.data_ptr())


class FemContext:
    """fem_setup + fem_build_csr_pattern + fem_assemble on torch CUDA tensors (device memory and streams only)."""

    def __init__(self, coords, conn, fbar=0, tol=None, kmax=None, assembly_mode=None):
        torch = _torch()
        L = lib()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_17390_b200 needs a CUDA device: there is no CPU fallback")
        self.n_nodes, self.n_elems = int(coords.shape[0]), int(conn.shape[0])
        opt = FemOptions()
        L.fem_default_options(C.byref(opt))
        opt.fbar = int(fbar)
        if tol is not None:
            opt.tol = float(tol)
        if kmax is not None:
            opt.kmax = int(kmax)
        if assembly_mode is not None:
            opt.assembly_mode = int(assembly_mode)
        self._h = C.c_void_p()
        _check(L.fem_setup(C.byref(self._h), self.n_nodes, _ptr(coords, torch.float64, 3 * self.n_nodes, "coords"),
                           self.n_elems, _ptr(conn, torch.int32, 8 * self.n_elems, "conn"), C.byref(opt)), "fem_setup")
        self.device = coords.device
        self.n_rows = 3 * self.n_nodes
        self.nnz = None

    def build_csr_pattern(self, want_elem_slot=False):
        """Returns (row_ptr, col_idx, elem_slot or None) as torch tensors (copies of the library-owned arrays)."""
        torch = _torch()
        L = lib()
        nr, nnz = C.c_longlong(), C.c_longlong()
        rp, ci, es = C.c_void_p(), C.c_void_p(), C.c_void_p()
        _check(L.fem_build_csr_pattern(self._h, C.byref(nr), C.byref(nnz), C.byref(rp), C.byref(ci),
                                       C.byref(es) if want_elem_slot else None), "fem_build_csr_pattern")
        self.n_rows, self.nnz = nr.value, nnz.value

        def copy(ptr, n):
            out = torch.empty(n, dtype=torch.int32, device=self.device)
            rc = _cudart().cudaMemcpy(C.c_void_p(out.data_ptr()), ptr, C.c_size_t(4 * n), 3)
            if rc != 0:
                raise RuntimeError("cudaMemcpy failed: %d" % rc)
            return out
        row_ptr, col_idx = copy(rp, self.n_rows + 1), copy(ci, self.nnz)
        elem_slot = copy(es, 576 * self.n_elems).view(self.n_elems, 576) if want_elem_slot else None
        return row_ptr, col_idx, elem_slot

    def assemble(self, u, hist_in, mat, residual=None, csr_vals=None, hist_out=None, want_stats=False, barlat=None):
        """One fem_assemble call (fem_assemble_barlat when `barlat` records are given) on the current torch stream.
        Returns (residual, csr_vals, hist_out, stats|None)."""
        torch = _torch()
        if self.nnz is None:
            raise FemError(-7, "fem_assemble")
        f64 = torch.float64
        n_mat = mat.numel() // NPAR
        if residual is None:
            residual = torch.empty(self.n_rows, dtype=f64, device=self.device)
        if csr_vals is None:
            csr_vals = torch.empty(self.nnz, dtype=f64, device=self.device)
        if hist_out is None:
            hist_out = torch.empty(self.n_elems * 56, dtype=f64, device=self.device)
        st = FemStats() if want_stats else None
        if barlat is not None:
            _check(lib().fem_assemble_barlat(self._h, _ptr(u, f64, self.n_rows, "u"), _ptr(hist_in, f64, 56 * self.n_elems, "hist_in"),
                                             _ptr(mat, f64, None, "mat"), _ptr(barlat, f64, NBARLAT * n_mat, "barlat"), n_mat,
                                             _ptr(residual, f64, self.n_rows, "residual"), _ptr(csr_vals, f64, self.nnz, "csr_vals"),
                                             _ptr(hist_out, f64, 56 * self.n_elems, "hist_out"),
                                             C.byref(st) if want_stats else None, _stream_ptr()), "fem_assemble_barlat")
            return residual, csr_vals, hist_out, (st.as_dict() if want_stats else None)
        _check(lib().fem_assemble(self._h, _ptr(u, f64, self.n_rows, "u"), _ptr(hist_in, f64, 56 * self.n_elems, "hist_in"),
                                  _ptr(mat, f64, None, "mat"), n_mat, _ptr(residual, f64, self.n_rows, "residual"),
                                  _ptr(csr_vals, f64, self.nnz, "csr_vals"), _ptr(hist_out, f64, 56 * self.n_elems, "hist_out"),
                                  C.byref(st) if want_stats else None, _stream_ptr()), "fem_assemble")
        return residual, csr_vals, hist_out, (st.as_dict() if want_stats else None)

    def assemble_static_prepare(self):
        """fem_assemble_static_prepare: the set-up step of assemble_static (device address of the library's static scratch)."""
        _check(lib().fem_assemble_static_prepare(self._h), "fem_assemble_static_prepare")

    def assemble_static(self, u, hist_in, mat, residual, csr_vals, hist_out, want_stats=False):
        """fem_assemble_static: fem_assemble with its scratch in the library's file-scope device array; the call allocates
        nothing, so the caller passes every output.  At most STATIC_MAX_ELEMS elements.  Returns stats|None."""
        f64 = _torch().float64
        n_mat = mat.numel() // NPAR
        st = FemStats() if want_stats else None
        _check(lib().fem_assemble_static(self._h, _ptr(u, f64, self.n_rows, "u"), _ptr(hist_in, f64, 56 * self.n_elems, "hist_in"),
                                         _ptr(mat, f64, None, "mat"), n_mat, _ptr(residual, f64, self.n_rows, "residual"),
                                         _ptr(csr_vals, f64, self.nnz, "csr_vals"),
                                         _ptr(hist_out, f64, 56 * self.n_elems, "hist_out"),
                                         C.byref(st) if want_stats else None, _stream_ptr()), "fem_assemble_static")
        return st.as_dict() if want_stats else None

    def assemble_host(self, u, hist_in, mat, residual, csr_vals, hist_out, want_stats=False):
        """fem_assemble_host on HOST buffers (numpy arrays or pinned CPU torch tensors); copies are inside the call."""
        def hp(a, n, name):
            if hasattr(a, "data_ptr"):
                if a.is_cuda or a.dtype != _torch().float64 or not a.is_contiguous() or a.numel() != n:
                    raise TypeError("%s must be a contiguous float64 host tensor of %d elements" % (name, n))
                return C.c_void_p(a.data_ptr())
            if a.dtype != np.float64 or not a.flags["C_CONTIGUOUS"] or a.size != n:
                raise TypeError("%s must be a contiguous float64 array of %d elements" % (name, n))
            return C.c_void_p(a.ctypes.data)
        n_mat = (mat.numel() if hasattr(mat, "numel") else mat.size) // NPAR
        st = FemStats() if want_stats else None
        _check(lib().fem_assemble_host(self._h, hp(u, self.n_rows, "u"), hp(hist_in, 56 * self.n_elems, "hist_in"),
                                       hp(mat, NPAR * n_mat, "mat"), n_mat, hp(residual, self.n_rows, "residual"),
                                       hp(csr_vals, self.nnz, "csr_vals"), hp(hist_out, 56 * self.n_elems, "hist_out"),
                                       C.byref(st) if want_stats else None), "fem_assemble_host")
        return st.as_dict() if want_stats else None

    def spmv(self, csr_vals, x, y=None):
        """fem_spmv: y = K x on the context's pattern."""
        torch = _torch()
        if y is None:
            y = torch.empty(self.n_rows, dtype=torch.float64, device=self.device)
        _check(lib().fem_spmv(self._h, _ptr(csr_vals, torch.float64, self.nnz, "csr_vals"), _ptr(x, torch.float64, self.n_rows, "x"),
                              _ptr(y, torch.float64, self.n_rows, "y"), _stream_ptr()), "fem_spmv")
        return y

    def apply_dirichlet(self, bc_dofs, csr_vals, rhs=None, bc_rhs=None):
        """fem_apply_dirichlet: identity rows for bc_dofs (int32 CUDA tensor), rhs[d] = bc_rhs (0 if None).  In place."""
        torch = _torch()
        nbc = bc_dofs.numel()
        _check(lib().fem_apply_dirichlet(self._h, nbc, _ptr(bc_dofs, torch.int32, None, "bc_dofs"),
                                         None if bc_rhs is None else _ptr(bc_rhs, torch.float64, nbc, "bc_rhs"),
                                         _ptr(csr_vals, torch.float64, self.nnz, "csr_vals"),
                                         None if rhs is None else _ptr(rhs, torch.float64, self.n_rows, "rhs"), _stream_ptr()),
               "fem_apply_dirichlet")

    def bicgstab(self, csr_vals, b, x=None, rtol=1e-10, max_iter=10000):
        """fem_bicgstab: returns (x, iters, relres, converged)."""
        torch = _torch()
        if x is None:
            x = torch.zeros(self.n_rows, dtype=torch.float64, device=self.device)
        it, rr = C.c_int(0), C.c_double(0.0)
        rc = lib().fem_bicgstab(self._h, _ptr(csr_vals, torch.float64, self.nnz, "csr_vals"), _ptr(b, torch.float64, self.n_rows, "b"),
                                _ptr(x, torch.float64, self.n_rows, "x"), float(rtol), int(max_iter), C.byref(it), C.byref(rr),
                                _stream_ptr())
        if rc not in (0, -11):
            _check(rc, "fem_bicgstab")
        return x, it.value, rr.value, rc == 0

    def lincomb(self, a, x, b, y, out=None):
        """fem_lincomb: out = a x + b y on DOF vectors."""
        torch = _torch()
        if out is None:
            out = torch.empty(self.n_rows, dtype=torch.float64, device=self.device)
        _check(lib().fem_lincomb(self._h, float(a), _ptr(x, torch.float64, self.n_rows, "x"), float(b), _ptr(y, torch.float64, self.n_rows, "y"),
                                 _ptr(out, torch.float64, self.n_rows, "out"), _stream_ptr()), "fem_lincomb")
        return out

    def pcg(self, csr_vals, b, x=None, rtol=1e-10, max_iter=10000):
        """fem_pcg: returns (x, iters, relres, converged).  x must hold b[d] on Dirichlet DOFs d (see include/fem.h)."""
        torch = _torch()
        if x is None:
            x = torch.zeros(self.n_rows, dtype=torch.float64, device=self.device)
        it, rr = C.c_int(0), C.c_double(0.0)
        rc = lib().fem_pcg(self._h, _ptr(csr_vals, torch.float64, self.nnz, "csr_vals"), _ptr(b, torch.float64, self.n_rows, "b"),
                           _ptr(x, torch.float64, self.n_rows, "x"), float(rtol), int(max_iter), C.byref(it), C.byref(rr), _stream_ptr())
        if rc not in (0, -11):
            _check(rc, "fem_pcg")
        return x, it.value, rr.value, rc == 0

    def newton_solve(self, u, hist_in, mat, bc_dofs, bc_vals, hist_out=None, rtol=None, atol=None, max_newton=None,
                     lin_rtol=None, lin_max_iter=None, linear_solver=None):
        """fem_newton_solve: one load increment; u is updated in place.  Returns (u, hist_out, report dict)."""
        torch = _torch()
        f64 = torch.float64
        if hist_out is None:
            hist_out = torch.empty(self.n_elems * 56, dtype=f64, device=self.device)
        opt = FemNewtonOptions()
        lib().fem_default_newton_options(C.byref(opt))
        for k, v in (("rtol", rtol), ("atol", atol), ("max_newton", max_newton), ("lin_rtol", lin_rtol), ("lin_max_iter", lin_max_iter),
                     ("linear_solver", linear_solver)):
            if v is not None:
                setattr(opt, k, v)
        rep = FemNewtonReport()
        nbc = bc_dofs.numel()
        rc = lib().fem_newton_solve(self._h, _ptr(u, f64, self.n_rows, "u"), _ptr(hist_in, f64, 56 * self.n_elems, "hist_in"),
                                    _ptr(mat, f64, None, "mat"), mat.numel() // NPAR, nbc, _ptr(bc_dofs, torch.int32, None, "bc_dofs"),
                                    _ptr(bc_vals, f64, nbc, "bc_vals"), _ptr(hist_out, f64, 56 * self.n_elems, "hist_out"),
                                    C.byref(opt), C.byref(rep), _stream_ptr())
        if rc not in (0, -11):
            _check(rc, "fem_newton_solve")
        return u, hist_out, rep.as_dict()

    def load_path(self, u, hist, mat, bc_dofs, bc_full, newton=None, **path):
        """fem_load_path: adaptive load stepping from t = 0 to 1; u and hist are updated in place.
        `path`: dt0, dt_min, dt_max, grow, cut, grow_below, max_steps, extrapolate; `newton`: dict of fem_newton_options fields.
        Returns (return code, report dict, accepted load fractions)."""
        torch = _torch()
        f64 = torch.float64
        opt = FemPathOptions()
        lib().fem_default_path_options(C.byref(opt))
        for k, v in path.items():
            setattr(opt, k, v)
        for k, v in (newton or {}).items():
            setattr(opt.newton, k, v)
        rep = FemPathReport()
        cap = int(opt.max_steps)
        ts = (C.c_double * cap)()
        nbc = bc_dofs.numel()
        rc = lib().fem_load_path(self._h, _ptr(u, f64, self.n_rows, "u"), _ptr(hist, f64, 56 * self.n_elems, "hist"),
                                 _ptr(mat, f64, None, "mat"), mat.numel() // NPAR, nbc, _ptr(bc_dofs, torch.int32, None, "bc_dofs"),
                                 _ptr(bc_full, f64, nbc, "bc_full"), C.byref(opt), C.byref(rep), ts, cap, _stream_ptr())
        if rc not in (0, -11):
            _check(rc, "fem_load_path")
        return rc, rep.as_dict(), list(ts[:rep.steps])

    def assemble_vjp(self, u, hist_in, mat, lam=None, mu=None, want_u=True, want_hist=True, want_mat=True):
        """fem_assemble_vjp: (g_u, g_hist_in, g_mat) for the cotangents lam on the residual and mu on hist_out (None = zero);
        outputs not wanted are None."""
        torch = _torch()
        f64 = torch.float64
        n_mat = mat.numel() // NPAR
        g_u = torch.empty(self.n_rows, dtype=f64, device=self.device) if want_u else None
        g_h = torch.empty(self.n_elems * 56, dtype=f64, device=self.device) if want_hist else None
        g_m = torch.empty(n_mat * NPAR, dtype=f64, device=self.device) if want_mat else None
        opt = lambda t, n, name: None if t is None else _ptr(t, f64, n, name)
        _check(lib().fem_assemble_vjp(self._h, _ptr(u, f64, self.n_rows, "u"), _ptr(hist_in, f64, 56 * self.n_elems, "hist_in"),
                                      _ptr(mat, f64, None, "mat"), n_mat, opt(lam, self.n_rows, "lam"), opt(mu, 56 * self.n_elems, "mu"),
                                      opt(g_u, self.n_rows, "g_u"), opt(g_h, 56 * self.n_elems, "g_hist_in"),
                                      opt(g_m, n_mat * NPAR, "g_mat"), _stream_ptr()), "fem_assemble_vjp")
        return g_u, g_h, (g_m.view(n_mat, NPAR) if g_m is not None else None)

    def adjoint_step(self, u, hist_in, mat, bc_dofs, dJdu=None, mu_in=None, lin_rtol=1e-10, lin_max_iter=10000):
        """fem_adjoint_step: one step of the backward sweep of Alg. 1.  Returns (lam, mu_out, g_mat, lin_iters)."""
        torch = _torch()
        f64 = torch.float64
        n_mat = mat.numel() // NPAR
        lam = torch.empty(self.n_rows, dtype=f64, device=self.device)
        mu_out = torch.empty(self.n_elems * 56, dtype=f64, device=self.device)
        g_m = torch.empty(n_mat * NPAR, dtype=f64, device=self.device)
        it = C.c_int(0)
        opt = lambda t, n, name: None if t is None else _ptr(t, f64, n, name)
        _check(lib().fem_adjoint_step(self._h, _ptr(u, f64, self.n_rows, "u"), _ptr(hist_in, f64, 56 * self.n_elems, "hist_in"),
                                      _ptr(mat, f64, None, "mat"), n_mat, bc_dofs.numel(), _ptr(bc_dofs, torch.int32, None, "bc_dofs"),
                                      opt(dJdu, self.n_rows, "dJdu"), opt(mu_in, 56 * self.n_elems, "mu_in"),
                                      _ptr(lam, f64, self.n_rows, "lam"), _ptr(mu_out, f64, 56 * self.n_elems, "mu_out"),
                                      _ptr(g_m, f64, n_mat * NPAR, "g_mat"), float(lin_rtol), int(lin_max_iter), C.byref(it),
                                      _stream_ptr()), "fem_adjoint_step")
        return lam, mu_out, g_m.view(n_mat, NPAR), it.value

    def set_mixed_precision(self, on=True):
        """fem_set_mixed_precision: fp32 copy of K inside the CG iteration, fp64 residuals and refinement."""
        _check(lib().fem_set_mixed_precision(self._h, 1 if on else 0), "fem_set_mixed_precision")

    def last_kernel_ms(self):
        ms = (C.c_double * 3)()
        _check(lib().fem_last_kernel_ms(self._h, ms), "fem_last_kernel_ms")
        return dict(element=ms[0], gather=ms[1], mat_prep=ms[2])

    def launches_per_assemble(self):
        return int(lib().fem_launches_per_assemble(self._h))

    def close(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().fem_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


_crt = None


def _cudart():
    """The CUDA runtime already loaded by torch (used only to copy library-owned pattern arrays into torch tensors)."""
    global _crt
    if _crt is None:
        import glob
        torch = _torch()
        cands = glob.glob(os.path.join(os.path.dirname(torch.__file__), "lib", "libcudart*.so*")) + \
            glob.glob("/usr/local/cuda/lib64/libcudart.so*")
        for c in cands:
            try:
                _crt = C.CDLL(c)
                break
            except OSError:
                continue
        if _crt is None:
            raise RuntimeError("libcudart not found")
        _crt.cudaMemcpy.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t, C.c_int]
    return _crt


def probe_fp64_peak(ms_target=50.0):
    out = C.c_double()
    _check(lib().fem_probe_fp64_peak(float(ms_target), C.byref(out), _stream_ptr()), "fem_probe_fp64_peak")
    return out.value
