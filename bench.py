#!/usr/bin/env python
"""bench.py — element residual+tangent+CSR-assembly evaluations per second at 3M DOF, fp64 (BASELINE.json metric).

A "step" is one fem_assemble call (all rows of SURVEY.md §8(a): material pre-pass, element kernel, gather kernel) on
BASELINE.json config 3: 100x100x100 hex8 cube, 1,000,000 elements, 3,090,903 DOF, 8M Gauss points, Hill-48 + Swift,
seeded smooth displacement with peak strain 0.1.  The CSR pattern is built once, outside the timed region.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--n 100]

One JSON line on stdout (rank 0).  Keys beyond the driver's contract: roofline (dominant kernel vs the FP64 ALU
roofline), cpu_baseline (the oracle timed on this box's host cores on a bounded sample), e2e (same metric through
fem_assemble_host with host buffers), kernels_ms, plastic_fraction.
"""
import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "element residual+tangent+CSR-assembly evals/s at 3M DOF fp64"
UNIT = "element-evals/s"

# Frozen algorithmic work model: FP64 flops per Gauss point
# (FMA = 2) in the cheapest known formulation, and bytes per element that must cross HBM.
FLOPS_ELASTIC_POINT = 6850.0
FLOPS_PLASTIC_EXTRA = 1600.0
FLOPS_ELEMENT_EXTRA = 600.0
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 FP64 FMA lanes x 2 x 1.965 GHz = 37.2


def alg_flops_per_element(plastic_fraction):
    return 8.0 * (FLOPS_ELASTIC_POINT + FLOPS_PLASTIC_EXTRA * plastic_fraction) + FLOPS_ELEMENT_EXTRA


def alg_bytes_per_element(n_nodes, n_elems, nnz, per_elem_mat):
    # conn + coords,u (once per node) + hist in/out + csr values + residual + compressed slot map (+ material records)
    b = 32.0 + 2 * 24.0 * n_nodes / n_elems + 896.0 + 8.0 * nnz / n_elems + 24.0 * n_nodes / n_elems + 256.0
    return b + (128.0 if per_elem_mat else 0.0)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d.get("hbm_gbs", 6650.0)), "measured"
    return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks line of B200_PROFILING.md, sampled during the timed region."""

    def __init__(self, index):
        self.path = os.path.join("/tmp", "bench_clocks_%d_%d.csv" % (os.getpid(), index))
        self.proc = None
        self.index = index

    def start(self):
        q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + q, "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.f.close()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                c = [x.strip() for x in line.split(",")]
                if len(c) < 9:
                    continue
                try:
                    sm.append(float(c[1])); mx.append(float(c[2]))
                except ValueError:
                    continue
                for nm, v in zip(names, c[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            os.remove(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


def aggregate_over_ranks(ms_local, n_units_per_rank, world, device=None):
    """max-over-ranks step time and whole-job throughput (units of all ranks / slowest rank's time); weak scaling:
    every rank processes its own replica, no data-path collective.  Works with any torch.distributed backend."""
    ms = float(ms_local)
    if world > 1:
        import torch
        import torch.distributed as dist
        t = torch.tensor([ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    return ms, world * n_units_per_rank / (ms * 1e-3)


def slab_sample(cfg, n, layers):
    """First `layers` z-layers of the n^3 mesh as a self-contained sub-mesh (nodes are lexicographic, so contiguous)."""
    ne, nn = layers * n * n, (layers + 1) * (n + 1) * (n + 1)
    return dict(coords=cfg["coords"][:nn], conn=cfg["conn"][:ne], u=cfg["u"][:nn], hist_in=cfg["hist_in"][:ne],
                matdesc=cfg["matdesc"])


def time_oracle(sample, repeats=1):
    """Seconds per oracle assemble (O1-O13, pattern build excluded) on the host cores."""
    import oracle
    ne = sample["conn"].shape[0]
    mat = oracle.mat_from_desc(sample["matdesc"], ne)
    rp, ci, _ = oracle.pattern(sample["coords"].shape[0], sample["conn"], with_slots=False)
    ts = []
    for _ in range(repeats):
        t = time.perf_counter()
        oracle.assemble(sample["coords"], sample["conn"], sample["u"], sample["hist_in"], mat, rp, ci, fbar=0)
        ts.append(time.perf_counter() - t)
    return ts, oracle.num_threads()


def run_reference(args):
    """--impl reference: the oracle, as it stands, on host cores; each step a bounded slab sample of config 3."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import synth
    n = args.n
    cfg = synth.make_config(3, n=n)
    t1, cores = time_oracle(slab_sample(cfg, n, 1))           # calibration: one layer
    rate = n * n / t1[0]
    layers = int(max(1, min(10, n, round(4.0 * rate / (n * n)))))  # about 4 s per step
    sample = slab_sample(cfg, n, layers)
    ne = sample["conn"].shape[0]
    time_oracle(sample, max(0, args.warmup - 1)) if args.warmup > 1 else None
    ts, cores = time_oracle(sample, args.steps)
    tot = float(np.sum(ts))
    val = ne * args.steps / tot
    desc = "first %d z-layers of the %d^3 mesh (%d elements) per step" % (layers, n, ne)
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "config3 cube%d hex8 Hill-48+Swift, oracle on a bounded sample" % n, "sample": desc},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def run_gpu(args):
    import torch
    import synth
    import paper_2606_17390_b200 as fem

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    fem.lib()  # fail loudly when the extension is missing

    n = args.n
    cfg = synth.make_config(3, n=n)   # every rank: its own replica of the workload (weak scaling, no data-path collective)
    ne, nn = cfg["conn"].shape[0], cfg["coords"].shape[0]
    mat_np = fem.mat_from_desc(cfg["matdesc"], ne)
    t0 = time.perf_counter()
    ctx = fem.FemContext(torch.from_numpy(cfg["coords"]).to(dev), torch.from_numpy(cfg["conn"]).to(dev), fbar=args.fbar, assembly_mode=args.mode)
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t0
    t0 = time.perf_counter()
    ctx.build_csr_pattern()
    torch.cuda.synchronize()
    t_pattern = time.perf_counter() - t0
    nnz = ctx.nnz
    u = torch.from_numpy(cfg["u"].ravel()).to(dev)
    hin = torch.from_numpy(cfg["hist_in"].ravel()).to(dev)
    mat = torch.from_numpy(mat_np.ravel()).to(dev)
    res = torch.empty(3 * nn, dtype=torch.float64, device=dev)
    vals = torch.empty(nnz, dtype=torch.float64, device=dev)
    hout = torch.empty(56 * ne, dtype=torch.float64, device=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    peak_tf = fem.probe_fp64_peak(30.0)
    for _ in range(max(args.warmup, 3)):
        ctx.assemble(u, hin, mat, res, vals, hout)
    _, _, _, stats = ctx.assemble(u, hin, mat, res, vals, hout, want_stats=True)
    pfrac = stats["n_plastic"] / (8.0 * ne)

    # ---- timed region: exactly K steps, device events on the launching (current) stream
    clocks = ClockSampler(local)
    clocks.start()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        ctx.assemble(u, hin, mat, res, vals, hout)
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    # per-kernel durations (library events on the same stream), same launches, K more steps
    kms = dict(element=0.0, gather=0.0, mat_prep=0.0)
    for _ in range(args.steps):
        ctx.assemble(u, hin, mat, res, vals, hout)
        k = ctx.last_kernel_ms()
        for key in kms:
            kms[key] += k[key] / args.steps
    clk = clocks.stop()
    ms_step, value = aggregate_over_ranks(ms_total / args.steps, ne, world, dev)

    # ---- end-to-end: host buffers through fem_assemble_host, copies inside the timed region
    e2e_steps = max(1, min(args.steps, 5))
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a).ravel()).pin_memory()
    hu, hh, hm = pin(cfg["u"]), pin(cfg["hist_in"]), pin(mat_np)
    hres = torch.empty(3 * nn, dtype=torch.float64).pin_memory()
    hvals = torch.empty(nnz, dtype=torch.float64).pin_memory()
    hhout = torch.empty(56 * ne, dtype=torch.float64).pin_memory()
    ctx.assemble_host(hu, hh, hm, hres, hvals, hhout)   # warm-up (allocates the staging buffers)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ctx.assemble_host(hu, hh, hm, hres, hvals, hhout)
    torch.cuda.synchronize()
    t_e2e = (time.perf_counter() - t0) / e2e_steps
    if world > 1:
        t = torch.tensor([t_e2e], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        t_e2e = float(t.item())
    h2d = 8 * (hu.numel() + hh.numel() + hm.numel())
    d2h = 8 * (hres.numel() + hvals.numel() + hhout.numel())
    e2e_ok = bool(np.isfinite(hres.numpy()).all())

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (element kernel): FP64 ALU bound
    fl_el = alg_flops_per_element(pfrac)
    by_el = alg_bytes_per_element(nn, ne, nnz, mat_np.shape[0] > 1)
    hbm_gbs, hbm_src = measured_peaks()
    dom = max(("element", "gather"), key=lambda k: kms[k])
    ach_tf = fl_el * ne / (kms["element"] * 1e-3) / 1e12
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.csv")   # per-launch DRAM bytes from the committed ncu --set full capture
    if os.path.exists(tp):
        try:
            for line in open(tp):
                c = line.split(",")
                if c[0] == "k_element":
                    traffic = float(c[1])
        except Exception:
            traffic = None
    roofline = {"bound": "alu", "kernel": "k_element", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": ach_tf / peak_tf, "traffic": traffic,
                "peak_source": "DFMA probe kernel measured live in this run (nominal %.1f)" % NOMINAL_FP64_TFLOPS,
                "alg_flops_per_element": fl_el, "alg_bytes_per_element": by_el,
                "whole_step_frac": max(fl_el * ne / (peak_tf * 1e12), by_el * ne / (hbm_gbs * 1e9)) / (ms_step * 1e-3),
                "hbm_peak_gbs": hbm_gbs, "hbm_peak_source": hbm_src,
                "gather_alg_gbs": (8.0 * nnz + 4608.0 * ne) / (kms["gather"] * 1e-3) / 1e9, "dominant": dom}

    # ---- CPU baseline: the oracle on a bounded slab sample of the same workload
    cpu = None
    if not args.no_cpu:
        try:
            t1, cores = time_oracle(slab_sample(cfg, n, 1))
            rate = n * n / t1[0]
            layers = int(max(1, min(n, round(15.0 * rate / (n * n)))))
            ts, cores = time_oracle(slab_sample(cfg, n, layers))
            cpu = {"value": layers * n * n / ts[0], "unit": UNIT, "cores": cores, "kind": "oracle",
                   "sample": "first %d z-layers of the %d^3 mesh (%d elements), one oracle assemble, %.1f s" % (
                       layers, n, layers * n * n, ts[0])}
        except Exception as ex:  # the oracle is test infrastructure: its absence must not hide the GPU number
            cpu = {"value": None, "unit": UNIT, "cores": None, "kind": "oracle", "sample": "failed: %r" % (ex,)}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": "config3: %dx%dx%d hex8 cube, %d elements, %d DOF, 2x2x2 Gauss, Hill-48 (Lankford 0.7/0.6/0.8) + Swift, "
                               "smooth displacement peak strain 0.1, zero initial history" % (n, n, n, ne, 3 * nn),
                   "fbar": args.fbar, "replicas": world, "l2_policy": "inputs+outputs per step (%.1f GB) exceed the 126 MB L2"
                   % ((by_el * ne) / 1e9), "nnz": nnz},
        "clocks": {"sm_mhz": clk["sm_mhz"], "sm_max_mhz": clk["sm_max_mhz"], "reasons": clk["reasons"], "samples": clk["samples"]},
        "e2e": {"value": world * ne / t_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": 1e3 * t_e2e, "steps": e2e_steps, "finite": e2e_ok},
        "gpu_launches": args.steps * ctx.launches_per_assemble(),
        "roofline": roofline, "cpu_baseline": cpu,
        "kernels_ms": kms, "plastic_fraction": pfrac, "stats": {k: stats[k] for k in ("n_plastic", "n_nonconverged",
                                                                                    "n_detF_nonpos", "n_nonfinite", "max_local_iters")},
        "setup_s": t_setup, "pattern_s": t_pattern, "fp64_peak_probe_tflops": peak_tf,
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=100, help="mesh resolution (100 = BASELINE.json config 3)")
    ap.add_argument("--fbar", type=int, default=0)
    ap.add_argument("--mode", type=int, default=None, help="fem_options.assembly_mode (default: the library's default)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
