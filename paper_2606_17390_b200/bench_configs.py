"""Throughput of fem_assemble on the five BASELINE.json workloads at full size ("reported per config").

    python -m paper_2606_17390_b200.bench_configs [--steps 10] [--only 3,4,5f,5s]

Prints one markdown table row per case: mesh sizes, plastic fraction, local-iteration histogram, ms per call
(CUDA events around K calls after 3 warm-ups, inputs resident in HBM), per-kernel times and element-evals/s.
bench.py stays the driver's contract (config 3); this script is the per-config report kept in profiles/.
"""
import argparse
import sys
import os

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


# PAPER.md:471-477 Table 2 (c' , c'' , m = 8): the paper's Yld2004-18p coefficients
TABLE2 = [-0.069888, 0.936408, 0.079143, 1.003060, 0.524741, 1.363180, 1.023770, 1.069060, 0.954322,
          0.981171, 0.476741, 0.575316, 0.866827, 1.145010, -0.079294, 1.051660, 1.147100, 1.404620, 8.0, 0.0]


def run_case(label, cfg, steps, fbar=0, mode=None, barlat=None):
    import torch
    import paper_2606_17390_b200 as fem
    dev = torch.device("cuda:0")
    ne, nn = cfg["conn"].shape[0], cfg["coords"].shape[0]
    mat_np = fem.mat_from_desc(cfg["matdesc"], ne)
    ctx = fem.FemContext(torch.from_numpy(cfg["coords"]).to(dev), torch.from_numpy(cfg["conn"]).to(dev), fbar=fbar,
                         assembly_mode=mode)
    ctx.build_csr_pattern()
    u = torch.from_numpy(cfg["u"].ravel()).to(dev)
    hin = torch.from_numpy(cfg["hist_in"].ravel()).to(dev)
    mat = torch.from_numpy(np.ascontiguousarray(mat_np).ravel()).to(dev)
    if barlat is not None:   # fem_assemble_barlat: same elastic constants and hardening, r-values ignored
        barlat = torch.from_numpy(np.tile(np.asarray(barlat, dtype=np.float64), (mat_np.shape[0], 1)).ravel()).to(dev)
    res = torch.empty(3 * nn, dtype=torch.float64, device=dev)
    vals = torch.empty(ctx.nnz, dtype=torch.float64, device=dev)
    hout = torch.empty(56 * ne, dtype=torch.float64, device=dev)
    for _ in range(3):
        ctx.assemble(u, hin, mat, res, vals, hout, barlat=barlat)
    _, _, _, st = ctx.assemble(u, hin, mat, res, vals, hout, want_stats=True, barlat=barlat)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(steps):
        ctx.assemble(u, hin, mat, res, vals, hout, barlat=barlat)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    k = dict(element=0.0, gather=0.0)
    for _ in range(steps):
        ctx.assemble(u, hin, mat, res, vals, hout, barlat=barlat)
        km = ctx.last_kernel_ms()
        for key in k:
            k[key] += km[key] / steps
    hist = {i: int(c) for i, c in enumerate(st["iter_hist"]) if c}
    finite = bool(torch.isfinite(res).all().item() and torch.isfinite(vals).all().item())
    print("| %s | %d | %d | %d | %.3f | %s | %d | %.3f | %.3f | %.3f | %.1f | %s |" % (
        label, ne, 3 * nn, ctx.nnz, st["n_plastic"] / (8.0 * ne), hist, st["n_nonconverged"], ms, k["element"], k["gather"],
        ne / ms / 1e3, "yes" if finite else "NO"), flush=True)
    ctx.close()
    del u, hin, mat, res, vals, hout
    torch.cuda.empty_cache()


def main():
    import synth
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--only", default="1,2,3,3fbar,4,5f,5s,e4")
    args = ap.parse_args()
    only = set(args.only.split(","))
    print("| case | elements | DOF | nnz | plastic fraction | local iterations (count per iteration number) | non-converged | "
          "ms/call | element ms | gather ms | M element-evals/s | finite |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|")
    if "1" in only:
        run_case("config 1 (4^3)", synth.make_config(1), args.steps)
    if "2" in only:
        run_case("config 2 (40x40x4 plate, history)", synth.make_config(2), args.steps)
    if "3" in only:
        run_case("config 3 (100^3)", synth.make_config(3), args.steps)
    if "3fbar" in only:
        run_case("config 3, fbar=1", synth.make_config(3), args.steps, fbar=1)
    if "3b" in only:
        run_case("config 3, Yld2004-18p (Table 2, m=8)", synth.make_config(3), args.steps, barlat=TABLE2)
    if "3bfbar" in only:
        run_case("config 3, Yld2004-18p, fbar=1", synth.make_config(3), args.steps, fbar=1, barlat=TABLE2)
    if "5sb" in only:
        for lv in range(4):
            run_case("config 5 strain level %d (64^3), Yld2004-18p" % lv, synth.make_config(5, level=lv, sweep="strain"), args.steps,
                     barlat=TABLE2)
    if "4" in only:
        run_case("config 4 (100^3 void mask, shuffled, per-element material)", synth.make_config(4), args.steps)
    if "e4" in only:
        # the paper's largest case: 250 x 150 x 120 elements (13,758,063 DOF by its mesh; "~11.2 M" in the text),
        # config-3 recipe (same field, peak strain 0.1, x_c = 0.62) on the unit cube
        from synth import mesh, fields
        from synth.configs import BASE_SEED, SWIFT, XC
        coords, conn = mesh.structured_hex_mesh(250, 150, 120)
        u = fields.scaled_smooth_displacement(BASE_SEED + 3, coords, conn, np.ones(3), 0.1, xc=XC[3])
        run_case("E4 size (250x150x120), config-3 recipe", dict(coords=np.ascontiguousarray(coords), conn=np.ascontiguousarray(conn), u=u,
                                                                hist_in=np.zeros((conn.shape[0], 8, 7)), matdesc=dict(SWIFT)), max(2, args.steps // 2))
    if "5f" in only:
        for lv in range(5):
            run_case("config 5 fraction level %d (64^3)" % lv, synth.make_config(5, level=lv, sweep="fraction"), args.steps)
    if "5s" in only:
        for lv in range(4):
            run_case("config 5 strain level %d (64^3)" % lv, synth.make_config(5, level=lv, sweep="strain"), args.steps)


if __name__ == "__main__":
    main()
