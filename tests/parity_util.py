"""Shared helpers of the GPU parity tests: run the CUDA path and the oracle on the same seeded inputs and compare.
Tolerances are BASELINE.json north_star's: rel. L2 <= 1e-11 residual, <= 1e-10 CSR values and history, pattern exact."""
import numpy as np

TOL_RES, TOL_VALS, TOL_HIST = 1e-11, 1e-10, 1e-10


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64).ravel(); b = np.asarray(b, dtype=np.float64).ravel()
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / nb if nb > 0 else np.linalg.norm(a)


def run_gpu(cfg, fbar=0, want_elem_slot=False, mat=None, assembly_mode=None, barlat=None):
    import torch
    import paper_2606_17390_b200 as fem
    dev = torch.device("cuda:0")
    ne = cfg["conn"].shape[0]
    if mat is None:
        mat = fem.mat_from_desc(cfg["matdesc"], ne)
    ctx = fem.FemContext(torch.from_numpy(cfg["coords"]).to(dev), torch.from_numpy(cfg["conn"]).to(dev), fbar=fbar,
                         assembly_mode=assembly_mode)
    row_ptr, col_idx, slots = ctx.build_csr_pattern(want_elem_slot=want_elem_slot)
    res, vals, hout, stats = ctx.assemble(torch.from_numpy(cfg["u"].ravel()).to(dev), torch.from_numpy(cfg["hist_in"].ravel()).to(dev),
                                          torch.from_numpy(np.ascontiguousarray(mat).ravel()).to(dev), want_stats=True,
                                          barlat=None if barlat is None else torch.from_numpy(np.ascontiguousarray(barlat).ravel()).to(dev))
    torch.cuda.synchronize()
    out = dict(row_ptr=row_ptr.cpu().numpy(), col_idx=col_idx.cpu().numpy(),
               elem_slot=None if slots is None else slots.cpu().numpy(), residual=res.cpu().numpy(), csr_vals=vals.cpu().numpy(),
               hist_out=hout.cpu().numpy().reshape(ne, 8, 7), stats=stats, ctx=ctx)
    return out


def run_oracle(cfg, fbar=0, with_slots=False, mat=None, barlat=None):
    import oracle
    ne = cfg["conn"].shape[0]
    if mat is None:
        mat = oracle.mat_from_desc(cfg["matdesc"], ne)
    row_ptr, col_idx, slots = oracle.pattern(cfg["coords"].shape[0], cfg["conn"], with_slots=with_slots)
    out = oracle.assemble(cfg["coords"], cfg["conn"], cfg["u"], cfg["hist_in"], mat, row_ptr, col_idx, fbar=fbar, bar=barlat)
    out.update(row_ptr=row_ptr, col_idx=col_idx, elem_slot=slots)
    return out


def compare(g, o, label=""):
    """Returns dict of errors; asserts the north_star tolerances."""
    assert g["row_ptr"].dtype == np.int32 and g["col_idx"].dtype == np.int32
    assert np.array_equal(g["row_ptr"], o["row_ptr"]), label + " row_ptr differs"
    assert np.array_equal(g["col_idx"], o["col_idx"]), label + " col_idx differs"
    if g.get("elem_slot") is not None and o.get("elem_slot") is not None:
        assert np.array_equal(g["elem_slot"], o["elem_slot"]), label + " elem_slot differs"
    err = dict(res=rel_l2(g["residual"], o["residual"]), vals=rel_l2(g["csr_vals"], o["csr_vals"]),
               hist=rel_l2(g["hist_out"], o["hist_out"]))
    assert g["stats"]["n_plastic"] == o["stats"]["n_plastic"], (label, g["stats"]["n_plastic"], o["stats"]["n_plastic"])
    assert g["stats"]["n_nonconverged"] == 0 and o["stats"]["n_nonconverged"] == 0, label
    assert err["res"] <= TOL_RES, (label, err)
    assert err["vals"] <= TOL_VALS, (label, err)
    assert err["hist"] <= TOL_HIST, (label, err)
    return err
