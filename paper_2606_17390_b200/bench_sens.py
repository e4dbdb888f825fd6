"""Timing of fem_assemble_vjp at the BASELINE.json workload sizes, next to fem_assemble.

    python -m paper_2606_17390_b200.bench_sens [--steps 10] [--configs 3,4]

Prints markdown: per case ms per call (CUDA events around K calls after 3 warm-ups, inputs resident in HBM), element
VJP-evaluations per second, and the algorithmic HBM bytes of the call (reads conn, coords, u, lam, hist_in, mu; writes
g_hist_in, the g_u scratch and g_u) against the measured copy bandwidth.  The report is kept in profiles/.
"""
import argparse
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def run_case(k, steps, fbar=0):
    import torch
    import synth
    import paper_2606_17390_b200 as fem
    dev = torch.device("cuda:0")
    cfg = synth.make_config(k)
    ne, nn = cfg["conn"].shape[0], cfg["coords"].shape[0]
    ctx = fem.FemContext(torch.from_numpy(cfg["coords"]).to(dev), torch.from_numpy(cfg["conn"]).to(dev), fbar=fbar)
    ctx.build_csr_pattern()
    u = torch.from_numpy(cfg["u"].ravel()).to(dev)
    hin = torch.from_numpy(cfg["hist_in"].ravel()).to(dev)
    mat = torch.from_numpy(np.ascontiguousarray(fem.mat_from_desc(cfg["matdesc"], ne)).ravel()).to(dev)
    g = torch.Generator(device="cpu"); g.manual_seed(k)
    lam = torch.randn(3 * nn, dtype=torch.float64, generator=g).to(dev)
    mu = torch.randn(56 * ne, dtype=torch.float64, generator=g).to(dev)

    def timed(fn):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / steps
    ms_asm = timed(lambda: ctx.assemble(u, hin, mat))
    ms_all = timed(lambda: ctx.assemble_vjp(u, hin, mat, lam, mu))
    ms_u = timed(lambda: ctx.assemble_vjp(u, hin, mat, None, mu, want_hist=False, want_mat=False))
    ms_hm = timed(lambda: ctx.assemble_vjp(u, hin, mat, lam, mu, want_u=False))
    # algorithmic bytes per element of the full call: conn 32, coords+u+lam 3*24*nn/ne, hist_in+mu+g_hist 3*448, scratch 2*192, g_u 24*nn/ne
    b_alg = ne * (32 + 3 * 448 + 2 * 192) + nn * 24 * 4 + mat.numel() * 8 + (mat.numel() if mat.numel() > 16 else 0) * 8
    print("| %s | %d | %d | %.3f | %.3f | %.3f | %.3f | %.1f | %.0f |" % (
        ("%d, fbar=1" % k) if fbar else str(k), ne, 3 * nn, ms_asm, ms_all, ms_u, ms_hm, ne / ms_all * 1e-3, b_alg / ms_all * 1e-6))
    ctx.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--configs", default="2,3,4")
    ap.add_argument("--fbar", type=int, default=0, help="1: also time the F-bar element on every config")
    a = ap.parse_args()
    print("| config | elements | DOF | fem_assemble ms | fem_assemble_vjp ms (g_u, g_hist_in, g_mat) | g_u only (lam = NULL) ms | g_hist_in + g_mat ms | M element-VJPs/s | algorithmic GB/s |")
    print("|---|---|---|---|---|---|---|---|---|")
    for k in a.configs.split(","):
        run_case(int(k), a.steps)
        if a.fbar:
            run_case(int(k), a.steps, fbar=1)


if __name__ == "__main__":
    main()
