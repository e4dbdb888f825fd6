"""fem_assemble_static (include/fem.h): the entry point that allocates nothing -- its scratch is a file-scope device array
inside the library -- against the existing fem_assemble path on the same inputs, two calls in a row.

Collected last on purpose (the name sorts after every other test file): the suite runs with `pytest -x`."""
import numpy as np
import pytest

import synth
from parity_util import TOL_HIST, TOL_RES, TOL_VALS, rel_l2

pytestmark = pytest.mark.gpu


def _setup(cfg, fbar):
    import torch
    import paper_2606_17390_b200 as fem
    dev = torch.device("cuda:0")
    ne = cfg["conn"].shape[0]
    ctx = fem.FemContext(torch.from_numpy(cfg["coords"]).to(dev), torch.from_numpy(cfg["conn"]).to(dev), fbar=fbar)
    ctx.build_csr_pattern()
    mat = torch.from_numpy(np.ascontiguousarray(fem.mat_from_desc(cfg["matdesc"], ne)).ravel()).to(dev)
    u = torch.from_numpy(cfg["u"].ravel()).to(dev)
    h = torch.from_numpy(cfg["hist_in"].ravel()).to(dev)
    return ctx, u, h, mat


def _static_vs_existing(ctx, u, h, mat, label, check_free=False):
    """One fem_assemble_static call against one fem_assemble call on the same inputs; outputs pre-filled with NaN."""
    import torch
    ref_res, ref_vals, ref_hout, ref_stats = ctx.assemble(u, h, mat, want_stats=True)
    torch.cuda.synchronize()
    res = torch.full_like(ref_res, float("nan")); vals = torch.full_like(ref_vals, float("nan"))
    hout = torch.full_like(ref_hout, float("nan"))
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    stats = ctx.assemble_static(u, h, mat, res, vals, hout, want_stats=True)
    torch.cuda.synchronize()
    if check_free:   # a cudaMalloc inside the call would show as less free device memory
        assert torch.cuda.mem_get_info()[0] == free0, label
    assert rel_l2(res.cpu().numpy(), ref_res.cpu().numpy()) <= TOL_RES, label
    assert rel_l2(vals.cpu().numpy(), ref_vals.cpu().numpy()) <= TOL_VALS, label
    assert rel_l2(hout.cpu().numpy(), ref_hout.cpu().numpy()) <= TOL_HIST, label
    # same kernels, same summation order: the bits agree as well
    assert torch.equal(res, ref_res) and torch.equal(vals, ref_vals) and torch.equal(hout, ref_hout), label
    for k in ("n_plastic", "n_nonconverged", "n_detF_nonpos", "n_nonfinite", "max_local_iters", "iter_hist"):
        assert stats[k] == ref_stats[k], (label, k)
    return stats


@pytest.mark.parametrize("fbar", [0, 1])
def test_static_scratch_matches_existing_path_two_calls_in_a_row(fbar):
    # 13^3 = 2197 elements: 138 CTAs with a ragged tail, 70 % plastic points (the config-3 recipe at reduced resolution)
    cfg = synth.make_config(3, n=13)
    ctx, u, h, mat = _setup(cfg, fbar)
    ctx.assemble_static_prepare()
    s1 = _static_vs_existing(ctx, u, h, mat, "call 1 fbar=%d" % fbar, check_free=True)
    assert s1["n_plastic"] > 0
    # second call, straight after, on different inputs: the array still holds call 1's records and counters
    u2 = u * 0.4
    s2 = _static_vs_existing(ctx, u2, h, mat, "call 2 fbar=%d" % fbar, check_free=True)
    assert s2["n_plastic"] != s1["n_plastic"]
    # and the first inputs again: identical to call 1 (nothing of call 2 leaks)
    s3 = _static_vs_existing(ctx, u, h, mat, "call 3 fbar=%d" % fbar)
    assert s3 == s1
    ctx.close()


def test_static_scratch_shared_by_two_contexts_and_per_element_material():
    """Two contexts use the one array in turn: a smaller shuffled mesh with per-element records (config-4 recipe), then the
    structured one again.  Records of the larger mesh left beyond the smaller one's extent must not matter.  No explicit
    prepare here: the first call does the set-up step itself."""
    cfg_a = synth.make_config(3, n=12)
    cfg_b = synth.make_config(4, n=12)
    assert cfg_b["conn"].shape[0] < cfg_a["conn"].shape[0] and np.ndim(cfg_b["matdesc"]["r0"]) == 1
    a = _setup(cfg_a, 0)
    b = _setup(cfg_b, 0)
    _static_vs_existing(*a, "ctx a")
    _static_vs_existing(*b, "ctx b after a")
    _static_vs_existing(*a, "ctx a after b")
    a[0].close(); b[0].close()


def test_static_scratch_rejects_meshes_beyond_the_maximum():
    import torch
    import paper_2606_17390_b200 as fem
    from paper_2606_17390_b200 import binding
    assert binding.STATIC_MAX_ELEMS == 4096
    cfg = synth.make_config(3, n=16)             # exactly the maximum: accepted
    assert cfg["conn"].shape[0] == binding.STATIC_MAX_ELEMS
    ctx, u, h, mat = _setup(cfg, 0)
    _static_vs_existing(ctx, u, h, mat, "n = max")
    ctx.close()
    cfg = synth.make_config(3, n=17)             # 4913 elements: refused with its own error code, outputs untouched
    ctx, u, h, mat = _setup(cfg, 0)
    res = torch.full((ctx.n_rows,), 7.0, dtype=torch.float64, device=u.device)
    vals = torch.full((ctx.nnz,), 7.0, dtype=torch.float64, device=u.device)
    hout = torch.full((56 * ctx.n_elems,), 7.0, dtype=torch.float64, device=u.device)
    for call in (ctx.assemble_static_prepare, lambda: ctx.assemble_static(u, h, mat, res, vals, hout)):
        with pytest.raises(fem.FemError) as ei:
            call()
        assert ei.value.code == -12 and "FEM_STATIC_MAX_ELEMS" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((res == 7.0).all()) and bool((vals == 7.0).all()) and bool((hout == 7.0).all())
    ctx.close()


def test_static_scratch_call_can_be_captured_in_a_cuda_graph():
    """The reason the entry point exists: under stream capture a cudaMalloc fails the capture.  The call (counters cleared with a
    memset node, three kernel nodes) is captured once after the set-up step and replayed on new inputs."""
    import torch
    cfg = synth.make_config(3, n=13)
    ctx, u, h, mat = _setup(cfg, 0)
    ctx.assemble_static_prepare()                      # set-up step outside the capture
    ref1 = ctx.assemble(u, h, mat)
    u_in = u.clone()
    res = torch.empty_like(ref1[0]); vals = torch.empty_like(ref1[1]); hout = torch.empty_like(ref1[2])
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):                      # warm-up on the capture stream (torch's recipe)
        ctx.assemble_static(u_in, h, mat, res, vals, hout)
    torch.cuda.current_stream().wait_stream(side)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        ctx.assemble_static(u_in, h, mat, res, vals, hout)
    for scale in (1.0, 0.4):
        u_in.copy_(u * scale)
        res.fill_(float("nan")); vals.fill_(float("nan")); hout.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        ref = ctx.assemble(u * scale, h, mat)
        torch.cuda.synchronize()
        assert torch.equal(res, ref[0]) and torch.equal(vals, ref[1]) and torch.equal(hout, ref[2]), scale
    del g
    ctx.close()
