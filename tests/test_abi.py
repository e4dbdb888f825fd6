"""Host-side checks (no GPU): the C-ABI library builds, loads, and exports every symbol include/fem.h declares;
host helpers and argument checks behave as the header says."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def header_symbols():
    src = open(os.path.join(ROOT, "include", "fem.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fem_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import paper_2606_17390_b200 as fem
    L = fem.lib()
    syms = header_symbols()
    assert len(syms) >= 12
    for s in syms:
        assert hasattr(L, s), s
    assert set(fem.ABI_SYMBOLS) == set(syms)


def test_strerror_and_defaults():
    import paper_2606_17390_b200 as fem
    L = fem.lib()
    assert L.fem_strerror(0) == b"ok"
    for code in range(-11, 0):
        assert L.fem_strerror(code) not in (b"ok", b"unknown error code")
    opt = fem.FemOptions()
    L.fem_default_options(C.byref(opt))
    assert (opt.fbar, opt.quad_order, opt.kmax, opt.assembly_mode) == (0, 2, 60, 0)
    assert opt.tol == 1e-10 and opt.beta == 1e-4 and opt.eta == 0.1      # beta, eta: PAPER.md:871


def test_null_and_argument_errors_without_device_work():
    import paper_2606_17390_b200 as fem
    L = fem.lib()
    h = C.c_void_p()
    assert L.fem_setup(C.byref(h), 10, None, 1, None, None) == -1          # FEM_ERR_NULL
    assert L.fem_setup(None, 10, None, 1, None, None) == -1
    assert L.fem_build_csr_pattern(None, None, None, None, None, None) == -1
    assert L.fem_assemble(None, None, None, None, 1, None, None, None, None, None) == -1
    assert L.fem_launches_per_assemble(None) == 0
    assert L.fem_spmv(None, None, None, None, None) == -1
    assert L.fem_apply_dirichlet(None, 0, None, None, None, None, None) == -1
    assert L.fem_bicgstab(None, None, None, None, 1e-8, 10, None, None, None) == -1
    assert L.fem_newton_solve(None, None, None, None, 1, 0, None, None, None, None, None, None) == -1
    no = fem.FemNewtonOptions()
    L.fem_default_newton_options(C.byref(no))
    assert (no.rtol, no.atol, no.max_newton, no.lin_rtol, no.lin_max_iter, no.linear_solver) == (1e-9, 1e-10, 25, 1e-10, 10000, 0)
    assert L.fem_pcg(None, None, None, None, 1e-8, 10, None, None, None) == -1
    assert L.fem_lincomb(None, 1.0, None, 1.0, None, None, None) == -1
    assert L.fem_assemble_vjp(None, None, None, None, 1, None, None, None, None, None, None) == -1
    assert L.fem_adjoint_step(None, None, None, None, 1, 0, None, None, None, None, None, None, 1e-8, 10, None, None) == -1


def test_lankford_helper_matches_closed_form():
    """SURVEY.md §8(c) 'Lankford -> paper parameters' values for (0.7, 0.6, 0.8); (1,1,1) -> all ratios 1 (von Mises)."""
    import paper_2606_17390_b200 as fem
    r = fem.hill_from_lankford(0.7, 0.6, 0.8)
    assert np.allclose(r, [1.0, 1.0389249632986395, 0.9521904571390466, 1.1119188982851387, 1.0, 1.0], rtol=1e-15)
    assert np.allclose(fem.hill_from_lankford(1, 1, 1), 1.0, rtol=1e-15)
    out = (C.c_double * 6)()
    assert fem.lib().fem_hill_from_lankford(-1.0, 1.0, 1.0, out) == -2
    assert fem.lib().fem_hill_from_lankford(1.0, 1.0, 1.0, None) == -1


def test_product_path_does_not_import_oracle():
    """The oracle is test infrastructure: nothing under paper_2606_17390_b200/ or synth/ may reference it."""
    for pkg in ("paper_2606_17390_b200", "synth"):
        for dp, _, fs in os.walk(os.path.join(ROOT, pkg)):
            for f in fs:
                if f.endswith((".py", ".cu", ".h")):
                    txt = open(os.path.join(dp, f)).read()
                    assert "import oracle" not in txt and "from oracle" not in txt and "fem_oracle" not in txt, f


def test_no_cuda_device_is_a_loud_error():
    import torch
    import paper_2606_17390_b200 as fem
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        fem.FemContext(torch.zeros(8, 3, dtype=torch.float64), torch.zeros(1, 8, dtype=torch.int32))
