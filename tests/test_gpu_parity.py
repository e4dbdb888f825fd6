"""GPU parity: the CUDA path (through the C ABI) against the oracle, element by element, on the same seeded inputs.
Sizes: configs 1, 2 at full size; 3, 4, 5 at reduced resolution spanning several CTAs with a ragged tail (the recipe
is unchanged); full-size config 3 is covered by test_gpu_fullsize.py on sampled rows."""
import numpy as np
import pytest

import synth
from parity_util import compare, run_gpu, run_oracle, rel_l2

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("fbar", [0, 1])
def test_config1_cube4(fbar):
    cfg = synth.make_config(1)
    g, o = run_gpu(cfg, fbar, want_elem_slot=True), run_oracle(cfg, fbar, with_slots=True)
    err = compare(g, o, "cfg1")
    assert g["stats"]["n_detF_nonpos"] == 0 and g["stats"]["n_nonfinite"] == 0
    assert err["vals"] < 1e-13


@pytest.mark.parametrize("fbar", [0, 1])
def test_config2_plate(fbar):
    cfg = synth.make_config(2)
    g, o = run_gpu(cfg, fbar), run_oracle(cfg, fbar)
    compare(g, o, "cfg2")
    frac = g["stats"]["n_plastic"] / (8.0 * cfg["conn"].shape[0])
    assert 0.3 < frac < 0.7, frac       # "~50 % of quad points yield"


@pytest.mark.parametrize("n", [13, 22])   # 13^3 = 2197 elements: ragged tail of the 16-element CTAs and 4-element warps
def test_config3_reduced(n):
    cfg = synth.make_config(3, n=n)
    compare(run_gpu(cfg), run_oracle(cfg), "cfg3@%d" % n)


@pytest.mark.parametrize("fbar", [0, 1])
def test_config4_void_mask_per_element_material(fbar):
    cfg = synth.make_config(4, n=18)
    g, o = run_gpu(cfg, fbar, want_elem_slot=True), run_oracle(cfg, fbar, with_slots=True)
    compare(g, o, "cfg4@18")


@pytest.mark.parametrize("level", [0, 1, 2, 3, 4])
def test_config5_fraction_sweep(level):
    cfg = synth.make_config(5, n=14, level=level, sweep="fraction")
    g, o = run_gpu(cfg), run_oracle(cfg)
    compare(g, o, "cfg5 fraction %d" % level)
    if level == 0:
        assert g["stats"]["n_plastic"] == 0
        assert np.array_equal(g["hist_out"], cfg["hist_in"])      # elastic step: history copied bit for bit


@pytest.mark.parametrize("level", [0, 1, 2, 3])
def test_config5_strain_sweep(level):
    cfg = synth.make_config(5, n=14, level=level, sweep="strain")
    g, o = run_gpu(cfg), run_oracle(cfg)
    compare(g, o, "cfg5 strain %d" % level)
    assert g["stats"]["max_local_iters"] <= 30


def test_voce_and_rotated_material():
    """Voce hardening (Table 3 :493-495) and a non-identity material orientation (Eq.(A1) :774)."""
    import oracle
    cfg = synth.make_config(3, n=9)
    ne = cfg["conn"].shape[0]
    q = np.array([0.9, 0.2, -0.3, 0.25]); q /= np.linalg.norm(q)
    rec = [219000.0, 0.3, 1.5449, 1.0666, 1.0, 1.0307, 0.95, 1.1, 0.0, 138.0, 410.0, 3.8, *q]
    mat = np.tile(np.array(rec), (ne, 1))
    mat[:, 9] *= 1.0 + 0.1 * np.sin(np.arange(ne))            # per-element sigma0
    g, o = run_gpu(cfg, 0, mat=mat), run_oracle(cfg, 0, mat=mat)
    compare(g, o, "voce+rotation")
    assert g["stats"]["n_plastic"] > 0


def test_history_from_previous_increment_two_steps():
    """Two increments: hist_out of the first call is hist_in of the second (caller swaps buffers)."""
    import torch
    import oracle
    import paper_2606_17390_b200 as fem
    cfg = synth.make_config(5, n=8, level=3, sweep="fraction")
    ne = cfg["conn"].shape[0]
    g1, o1 = run_gpu(cfg), run_oracle(cfg)
    compare(g1, o1, "step 1")
    cfg2 = dict(cfg); cfg2["u"] = 1.5 * cfg["u"]; cfg2["hist_in"] = o1["hist_out"]
    g2, o2 = run_gpu(cfg2), run_oracle(cfg2)
    compare(g2, o2, "step 2")


def test_determinism_bitwise():
    import torch
    import paper_2606_17390_b200 as fem
    cfg = synth.make_config(4, n=16)
    g1 = run_gpu(cfg)
    g2 = run_gpu(cfg)
    for k in ("residual", "csr_vals", "hist_out"):
        assert np.array_equal(g1[k], g2[k]), k
    ctx = g1["ctx"]
    dev = torch.device("cuda:0")
    ne = cfg["conn"].shape[0]
    mat = torch.from_numpy(fem.mat_from_desc(cfg["matdesc"], ne).ravel()).to(dev)
    u = torch.from_numpy(cfg["u"].ravel()).to(dev); h = torch.from_numpy(cfg["hist_in"].ravel()).to(dev)
    r3, v3, h3, _ = ctx.assemble(u, h, mat)
    torch.cuda.synchronize()
    assert np.array_equal(v3.cpu().numpy(), g1["csr_vals"]) and np.array_equal(r3.cpu().numpy(), g1["residual"])


def test_host_buffer_call_matches_device_call():
    import paper_2606_17390_b200 as fem
    cfg = synth.make_config(2)
    g = run_gpu(cfg)
    ctx = g["ctx"]
    ne = cfg["conn"].shape[0]
    mat = fem.mat_from_desc(cfg["matdesc"], ne)
    res = np.empty(ctx.n_rows); vals = np.empty(ctx.nnz); hout = np.empty(56 * ne)
    st = ctx.assemble_host(np.ascontiguousarray(cfg["u"].ravel()), np.ascontiguousarray(cfg["hist_in"].ravel()),
                           np.ascontiguousarray(mat.ravel()), res, vals, hout, want_stats=True)
    assert np.array_equal(res, g["residual"]) and np.array_equal(vals, g["csr_vals"])
    assert np.array_equal(hout.reshape(ne, 8, 7), g["hist_out"]) and st["n_plastic"] == g["stats"]["n_plastic"]


def test_error_codes_on_device():
    import torch
    import paper_2606_17390_b200 as fem
    dev = torch.device("cuda:0")
    cfg = synth.make_config(1)
    coords = torch.from_numpy(cfg["coords"]).to(dev)
    bad = cfg["conn"].copy(); bad[3, 2] = 10_000
    with pytest.raises(fem.FemError) as ei:
        fem.FemContext(coords, torch.from_numpy(bad).to(dev))
    assert ei.value.code == -4
    inv = cfg["conn"].copy(); inv[5] = inv[5][[1, 0, 3, 2, 5, 4, 7, 6]]     # mirrored element: det J_ref < 0
    with pytest.raises(fem.FemError) as ei:
        fem.FemContext(coords, torch.from_numpy(inv).to(dev))
    assert ei.value.code == -5
    ctx = fem.FemContext(coords, torch.from_numpy(cfg["conn"]).to(dev))
    u = torch.zeros(375, dtype=torch.float64, device=dev); h = torch.zeros(64 * 56, dtype=torch.float64, device=dev)
    mat = torch.from_numpy(fem.mat_from_desc(cfg["matdesc"], 64).ravel()).to(dev)
    with pytest.raises(fem.FemError) as ei:       # pattern not built
        ctx.assemble(u, h, mat)
    assert ei.value.code == -7
    ctx.build_csr_pattern()
    with pytest.raises(fem.FemError) as ei:       # hist_out aliases hist_in
        ctx.assemble(u, h, mat, hist_out=h)
    assert ei.value.code == -9
    with pytest.raises(fem.FemError) as ei:       # n_mat neither 1 nor n_elems
        ctx.assemble(u, h, torch.cat([mat, mat]))
    assert ei.value.code == -10
    r, v, ho, st = ctx.assemble(u, h, mat, want_stats=True)   # u = 0: R = 0, nothing plastic
    assert float(r.abs().max()) == 0.0 and st["n_plastic"] == 0


@pytest.mark.parametrize("fbar", [0, 1])
@pytest.mark.parametrize("cfgid,n", [(3, 22), (4, 27)])
def test_fused_gather_equals_separate_gather(cfgid, n, fbar):
    """assembly_mode 2 gathers node quads inside the element launch (a second warpgroup of chunks launched one wave later
    reads the records back from L2, completion flags, bounded polling) and finishes the rest in k_gather_list;
    assembly_mode 1 runs the element kernel and the stand-alone gather kernel one after the other.  Both sum in ascending element id: the two
    must agree bit for bit, with the oracle within tolerance, and with themselves on a second call.  Sizes: more than
    3*148+64 chunks of 16 elements, so that part of the quads really is gathered in-kernel."""
    cfg = synth.make_config(cfgid, n=n)
    assert cfg["conn"].shape[0] > 16 * (3 * 148 + 64)
    g = run_gpu(cfg, fbar, assembly_mode=2)
    compare(g, run_oracle(cfg, fbar), "fused cfg%d" % cfgid)
    g1 = run_gpu(cfg, fbar, assembly_mode=1)
    assert np.array_equal(g["csr_vals"], g1["csr_vals"]) and np.array_equal(g["residual"], g1["residual"])
    assert np.array_equal(g["hist_out"], g1["hist_out"])
    g2 = run_gpu(cfg, fbar, assembly_mode=2)
    assert np.array_equal(g["csr_vals"], g2["csr_vals"]) and np.array_equal(g["residual"], g2["residual"])


def test_fused_gather_repeated_calls_and_isolated_node():
    """The chunk flags carry the epoch of the call: repeated calls on one context stay correct; a node that belongs to no
    element gets a zero residual."""
    import torch
    import paper_2606_17390_b200 as fem
    cfg = synth.make_config(3, n=22)
    coords = np.vstack([cfg["coords"], [[5.0, 5.0, 5.0]]])          # one extra, unreferenced node
    u = np.vstack([cfg["u"], [[0.0, 0.0, 0.0]]])
    cfg2 = dict(cfg, coords=coords, u=u)
    o = run_oracle(cfg2)
    dev = torch.device("cuda:0")
    ne = cfg2["conn"].shape[0]
    ctx = fem.FemContext(torch.from_numpy(coords).to(dev), torch.from_numpy(cfg2["conn"]).to(dev), assembly_mode=2)
    ctx.build_csr_pattern()
    mat = torch.from_numpy(fem.mat_from_desc(cfg2["matdesc"], ne).ravel()).to(dev)
    ud, hd = torch.from_numpy(u.ravel()).to(dev), torch.from_numpy(cfg2["hist_in"].ravel()).to(dev)
    prev = None
    for rep in range(4):
        uu = ud if rep != 2 else 0.5 * ud                            # a different state in between: stale records must not leak
        res, vals, hout, _ = ctx.assemble(uu, hd, mat, want_stats=True)
        torch.cuda.synchronize()
        if rep == 2:
            continue
        assert rel_l2(res.cpu().numpy(), o["residual"]) <= 1e-11 and rel_l2(vals.cpu().numpy(), o["csr_vals"]) <= 1e-10
        assert np.all(res.cpu().numpy()[-3:] == 0.0)
        if prev is not None:
            assert torch.equal(prev, vals)
        prev = vals.clone()


def _pinwheel_mesh(nsec=12, layers=2):
    """nsec hexes around the z-axis share the axis edge: axis nodes belong to nsec (> 8) elements per layer pair; they take
    the general path of the gather kernel, all other nodes of the same mesh the fast table path."""
    nodes, idx = [], {}

    def nid(key, xyz):
        if key not in idx:
            idx[key] = len(nodes); nodes.append(xyz)
        return idx[key]
    conn = []
    for L in range(layers):
        for j in range(nsec):
            t0, t1 = 2 * np.pi * j / nsec, 2 * np.pi * (j + 1) / nsec
            tm = 0.5 * (t0 + t1)
            quad = [("a",), ("p", j % nsec), ("q", j), ("p", (j + 1) % nsec)]
            xy = [(0.0, 0.0), (np.cos(t0), np.sin(t0)), (1.5 * np.cos(tm), 1.5 * np.sin(tm)), (np.cos(t1), np.sin(t1))]
            el = []
            for z in (L, L + 1):
                for key, (x, y) in zip(quad, xy):
                    el.append(nid(key + (z,), (x, y, 0.7 * z)))
            conn.append(el)
    return np.array(nodes, dtype=np.float64), np.array(conn, dtype=np.int32)


def _mini_cfg(coords, conn, seed=5, amp=0.03):
    rng = np.random.default_rng(seed)
    A = rng.normal(size=(3, 3)); A *= amp / np.linalg.norm(A)
    u = coords @ A.T + 2e-3 * rng.normal(size=coords.shape)
    return dict(coords=coords, conn=conn, u=u, hist_in=np.zeros((conn.shape[0], 8, 7)), matdesc=dict(synth.configs.SWIFT))


def test_high_valence_mesh_uses_general_gather():
    coords, conn = _pinwheel_mesh()
    cfg = _mini_cfg(coords, conn)
    g = run_gpu(cfg, 0, want_elem_slot=True)
    compare(g, run_oracle(cfg, 0, with_slots=True), "pinwheel")
    assert g["stats"]["n_plastic"] > 0


def test_node_with_more_than_32_neighbours_takes_the_two_kernel_schedule():
    """Eight hexes that share ONLY the centre node (a non-conforming mesh: every element has its own copies of the other
    seven nodes): the centre node has 8 elements but 57 neighbours, more than one warp holds one position per lane for.
    Even with the fused schedule requested the result must be the oracle's."""
    nodes, conn = [[0.0, 0.0, 0.0]], []
    for sx in (-1, 1):
        for sy in (-1, 1):
            for sz in (-1, 1):
                loc = {}
                for (i, j, k) in [(0, 0, 0), (1, 0, 0), (1, 1, 0), (0, 1, 0), (0, 0, 1), (1, 0, 1), (1, 1, 1), (0, 1, 1)]:
                    if (i, j, k) == (0, 0, 0):
                        loc[(i, j, k)] = 0
                    else:
                        loc[(i, j, k)] = len(nodes); nodes.append([sx * i * 1.0, sy * j * 0.9, sz * k * 1.1])
                # hex8 node order (-,-,-),(+,-,-),(+,+,-),(-,+,-),(-,-,+),... in the element's own axes; mirrored octants are
                # re-ordered so that det J_ref > 0
                order = [(0, 0, 0), (1, 0, 0), (1, 1, 0), (0, 1, 0), (0, 0, 1), (1, 0, 1), (1, 1, 1), (0, 1, 1)]
                el = [loc[o] for o in order]
                if sx * sy * sz < 0:
                    el = [el[0], el[3], el[2], el[1], el[4], el[7], el[6], el[5]]
                conn.append(el)
    coords, conn = np.array(nodes), np.array(conn, dtype=np.int32)
    assert coords.shape[0] == 57
    # the star comes first in a mesh large enough for the fused schedule to gather its nodes inside the element launch
    cube = synth.make_config(3, n=22)
    coords = np.vstack([coords + np.array([5.0, 5.0, 5.0]), cube["coords"]])
    conn = np.vstack([conn, cube["conn"] + 57]).astype(np.int32)
    assert conn.shape[0] > 16 * (3 * 148 + 64)
    cfg = _mini_cfg(coords, conn, seed=11)
    o = run_oracle(cfg, 0)
    assert np.diff(o["row_ptr"]).max() == 3 * 57
    for mode in (2, 1, 0):
        g = run_gpu(cfg, 0, assembly_mode=mode)
        compare(g, o, "star mesh mode %d" % mode)


def test_collapsed_hex_wedge_elements():
    """A wedge written as a hex with two node pairs repeated (collapsed element): the same node appears twice in an
    element, so several local (I,K) pairs map to one CSR block; assembly must add them all (mode falls back to 0)."""
    base = np.array([[0, 0, 0], [1, 0, 0], [0, 1, 0], [1, 1, 0.0]])
    coords = np.vstack([np.c_[base[:, :2], np.full(4, z)] for z in (0.0, 0.8, 1.7)])
    def wedge(a, b, c, off):   # triangle a,b,c extruded: hex nodes a,b,c,c / top
        return [a + off, b + off, c + off, c + off, a + off + 4, b + off + 4, c + off + 4, c + off + 4]
    conn = np.array([wedge(0, 1, 2, 0), wedge(1, 3, 2, 0), wedge(0, 1, 2, 4), wedge(1, 3, 2, 4)], dtype=np.int32)
    cfg = _mini_cfg(coords, conn, seed=9)
    g = run_gpu(cfg, 0, want_elem_slot=True)                      # collapsed elements: the general gather kernel
    assert g["ctx"].launches_per_assemble() == 3
    compare(g, run_oracle(cfg, 0, with_slots=True), "wedge")


@pytest.mark.parametrize("fbar", [0, 1])
def test_zero_and_rigid_displacement(fbar):
    """u = 0 (C = I exactly: every Jacobi rotation is the degenerate d = a_pq = 0 case) gives the linear-elastic stiffness
    and a zero residual; a rigid translation gives the same matrix."""
    cfg = synth.make_config(3, n=7)
    cfg0 = dict(cfg, u=np.zeros_like(cfg["u"]))
    g, o = run_gpu(cfg0, fbar), run_oracle(cfg0, fbar)
    compare(g, o, "u=0")
    assert np.abs(g["residual"]).max() <= 1e-9 and g["stats"]["n_plastic"] == 0
    cfg1 = dict(cfg, u=np.tile(np.array([0.3, -0.2, 0.1]), (cfg["u"].shape[0], 1)))
    g1 = run_gpu(cfg1, fbar)
    assert rel_l2(g1["csr_vals"], o["csr_vals"]) <= 1e-10 and np.abs(g1["residual"]).max() <= 1e-6


@pytest.mark.parametrize("world", [2, 3])
def test_sharded_rows_equal_single_gpu_rows(world):
    """row-ownership slabs with recomputed ghost elements, run one after the other on this GPU (no rank
    waits for another); the union of the owned rows is the single-GPU matrix bit for bit."""
    import torch
    import paper_2606_17390_b200 as fem
    from paper_2606_17390_b200 import shard
    cfg = synth.make_config(4, n=14)
    g = run_gpu(cfg)
    dev = torch.device("cuda:0")
    ne = cfg["conn"].shape[0]
    gmat = fem.mat_from_desc(cfg["matdesc"], ne)
    vals, res, rowlen, cols = [], [], [], []
    for rank in range(world):
        sh = shard.ShardedFem(cfg["coords"], cfg["conn"], world, rank, dev)
        p = sh.part
        u_local = torch.from_numpy(cfg["u"][p["lnodes"]].ravel().copy()).to(dev)
        r, v, h = sh.assemble(None, torch.from_numpy(cfg["hist_in"][p["elems"]].ravel().copy()).to(dev),
                              torch.from_numpy(np.ascontiguousarray(gmat[p["elems"]]).ravel()).to(dev), u_local=u_local)
        vals.append(v.cpu().numpy()); res.append(r.cpu().numpy()); cols.append(sh.col_idx.cpu().numpy())
        rowlen.append(np.diff(sh.row_ptr.cpu().numpy()))
        assert np.array_equal(h.cpu().numpy().reshape(-1, 8, 7), g["hist_out"][p["elems"]])
        sh.ctx.close()
    assert np.array_equal(np.concatenate(rowlen), np.diff(g["row_ptr"]))
    assert np.array_equal(np.concatenate(cols), g["col_idx"])
    assert np.array_equal(np.concatenate(vals), g["csr_vals"]) and np.array_equal(np.concatenate(res), g["residual"])
