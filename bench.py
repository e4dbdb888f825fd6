#!/usr/bin/env python
"""bench.py — element residual+tangent+CSR-assembly evaluations per second at 3M DOF, fp64 (BASELINE.json metric).

A "step" is one fem_assemble call (all rows of SURVEY.md §8(a): material pre-pass, element kernel, gather kernel) on
BASELINE.json config 3: 100x100x100 hex8 cube, 1,000,000 elements, 3,090,903 DOF, 8M Gauss points, Hill-48 + Swift,
seeded smooth displacement with peak strain 0.1.  The CSR pattern is built once, outside the timed region.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
                  [--workload config1..config5|e4] [--level L] [--sweep fraction|strain] [--fbar 0|1] [--mode 0|1] [--barlat]

N = 1: every step is timed with its own CUDA-event pair inside ONE barrier-bracketed region; `ms_per_step` is the
median of the K steps, `ms_per_step_mean` the mean.  N > 1 (torchrun): the SURVEY.md §8(e)
partition - the ONE problem is cut into N node slabs (paper_2606_17390_b200/shard.py), a step is the all-gather of the
owned displacement slabs (NCCL) followed by the rank's fem_assemble; `value` = elements of the whole problem / the slowest
rank's median step time ("scaling": "strong").

One JSON line on stdout (rank 0).  Keys beyond the driver's contract: roofline (dominant kernel vs the FP64 ALU
roofline), cpu_baseline (the oracle timed on this box's host cores on a bounded sample), e2e (same metric through
fem_assemble_host with host buffers), kernels_ms, plastic_fraction.
"""
import argparse
import hashlib
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


# fem_assemble_barlat, frozen in round 2 (FMA = 2): elastic point 12,050 (trial evaluation of phi, N, H
# included), plastic point 13,000 + 4,800 per Newton iteration of the return map (6x6 Cholesky, two solves, evaluation with
# Hessian, hardening law, merit); the iteration count is the measured one (stats.iter_hist of the same call).
FLOPS_BAR_ELASTIC_POINT = 12050.0
FLOPS_BAR_PLASTIC_POINT = 13000.0
FLOPS_BAR_ITERATION = 4800.0


def alg_flops_per_element_barlat(plastic_fraction, iter_hist):
    n_pl = float(sum(iter_hist))
    mean_it = sum(k * v for k, v in enumerate(iter_hist)) / n_pl if n_pl > 0 else 0.0
    return 8.0 * ((1.0 - plastic_fraction) * FLOPS_BAR_ELASTIC_POINT +
                  plastic_fraction * (FLOPS_BAR_PLASTIC_POINT + FLOPS_BAR_ITERATION * mean_it)) + FLOPS_ELEMENT_EXTRA


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


KERNEL_SOURCES = ["fem_assemble.cu", "fem_device.cuh", "fem_barlat.cuh", "fem_internal.h"]


def kernel_sha16():
    """Identifies the kernel sources a DRAM-traffic capture belongs to."""
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        with open(os.path.join(ROOT, "paper_2606_17390_b200", "csrc", f), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def recorded_traffic(workload, mode):
    """dram__bytes_read + dram__bytes_write per launch of the step's kernels from the `ncu --set full` capture recorded in
    profiles/r02_traffic.json - only if that capture was taken from the kernel sources of THIS build (same sha16), so the
    number can never go stale; otherwise None."""
    p = os.path.join(ROOT, "profiles", "r02_traffic.json")
    try:
        with open(p) as f:
            d = json.load(f)
        if d.get("kernel_sha16") != kernel_sha16():
            return None
        e = d.get("%s/mode%d" % (workload, mode))
        if e is None:
            return None
        return dict(e, kernel_sha16=d["kernel_sha16"], commit=d.get("commit"))
    except Exception:
        return None


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


def aggregate_over_ranks(ms_local, n_units_total, world, device=None):
    """max-over-ranks step time and whole-job throughput: the units of the WHOLE job (all ranks together) divided by the
    slowest rank's time.  Works with any torch.distributed backend."""
    ms = float(ms_local)
    if world > 1:
        import torch
        import torch.distributed as dist
        t = torch.tensor([ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    return ms, n_units_total / (ms * 1e-3)


def make_workload(args):
    """The seeded synthetic inputs of the named workload and a description for `config.workload`."""
    import synth
    w = args.workload
    if w == "e4":     # the paper's largest mesh, config-3 recipe
        from synth import mesh, fields
        coords, conn = mesh.structured_hex_mesh(250, 150, 120)
        seed = synth.configs.BASE_SEED + 3
        u = fields.scaled_smooth_displacement(seed, coords, conn, np.ones(3), 0.1, xc=synth.configs.XC[3])
        cfg = dict(coords=np.ascontiguousarray(coords), conn=np.ascontiguousarray(conn), u=u,
                   hist_in=np.zeros((conn.shape[0], 8, 7)), matdesc=dict(synth.configs.SWIFT))
        return cfg, "e4: 250x150x120 hex8 (PAPER.md:489), config-3 recipe"
    k = int(w.replace("config", ""))
    if k == 3:
        cfg = synth.make_config(3, n=args.n)
        n = args.n
        return cfg, ("config3: %dx%dx%d hex8 cube, %d elements, %d DOF, 2x2x2 Gauss, Hill-48 (Lankford 0.7/0.6/0.8) + Swift, "
                     "smooth displacement peak strain 0.1, zero initial history" % (n, n, n, cfg["conn"].shape[0], 3 * cfg["coords"].shape[0]))
    if k == 5:
        cfg = synth.make_config(5, level=args.level, sweep=args.sweep)
        return cfg, "config5: 64^3 hex8 cube, %s sweep level %d" % (args.sweep, args.level)
    cfg = synth.make_config(k)
    names = {1: "config1: 4x4x4 cube, affine + noise", 2: "config2: 40x40x4 plate, history from a prior increment",
             4: "config4: 100^3 minus 30 % void mask, shuffled element order, per-element Hill/Swift records"}
    return cfg, names[k]


TABLE2_BARLAT = [-0.069888, 0.936408, 0.079143, 1.003060, 0.524741, 1.363180, 1.023770, 1.069060, 0.954322,
                 0.981171, 0.476741, 0.575316, 0.866827, 1.145010, -0.079294, 1.051660, 1.147100, 1.404620, 8.0, 0.0]


def step_times_ms(events):
    return [events[i].elapsed_time(events[i + 1]) for i in range(len(events) - 1)]


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
    import paper_2606_17390_b200 as fem
    from paper_2606_17390_b200 import shard

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    fem.lib()  # fail loudly when the extension is missing

    cfg, wl_desc = make_workload(args)
    ne_g, nn_g = cfg["conn"].shape[0], cfg["coords"].shape[0]
    mat_g = fem.mat_from_desc(cfg["matdesc"], ne_g)
    mode = 0 if args.mode is None else args.mode
    bar = torch.tensor(TABLE2_BARLAT, dtype=torch.float64, device=dev) if args.barlat else None
    t_part = 0.0
    t0 = time.perf_counter()
    if world > 1:
        # node slabs own whole CSR rows, the one-element ghost layer is recomputed, ONE all-gather of the
        # owned displacement slabs precedes the kernels (shard.py).  Host partitioning is setup, timed separately.
        part = shard.partition(nn_g, cfg["conn"], world, rank)
        t_part = time.perf_counter() - t0
        t0 = time.perf_counter()
        lcoords = np.ascontiguousarray(cfg["coords"][part["lnodes"]])
        ctx = fem.FemContext(torch.from_numpy(lcoords).to(dev), torch.from_numpy(part["lconn"]).to(dev), fbar=args.fbar, assembly_mode=mode)
        u_owned = torch.from_numpy(cfg["u"][part["n0"]:part["n1"]].ravel().copy()).to(dev)
        hin = torch.from_numpy(np.ascontiguousarray(cfg["hist_in"][part["elems"]]).ravel()).to(dev)
        mat_np = mat_g if mat_g.shape[0] == 1 else np.ascontiguousarray(mat_g[part["elems"]])
        plan = shard.exchange_plan(part, dev)
        ne, nn = part["lconn"].shape[0], part["lnodes"].shape[0]
    else:
        part = plan = u_owned = None
        ctx = fem.FemContext(torch.from_numpy(cfg["coords"]).to(dev), torch.from_numpy(cfg["conn"]).to(dev), fbar=args.fbar, assembly_mode=mode)
        hin = torch.from_numpy(cfg["hist_in"].ravel()).to(dev)
        mat_np = mat_g
        ne, nn = ne_g, nn_g
    torch.cuda.synchronize()
    t_setup = time.perf_counter() - t0
    t0 = time.perf_counter()
    row_ptr, _, _ = ctx.build_csr_pattern()
    torch.cuda.synchronize()
    t_pattern = time.perf_counter() - t0
    nnz = ctx.nnz
    nnz_g = nnz
    if world > 1:    # nnz of the whole problem = sum of the owned rows' entries over the ranks
        t = torch.tensor([float(shard.owned_nnz(row_ptr, part))], dtype=torch.float64, device=dev)
        dist.all_reduce(t)
        nnz_g = int(t.item())
    u = torch.from_numpy(cfg["u"].ravel()).to(dev) if world == 1 else shard.exchange_u(u_owned, part, plan=plan)
    mat = torch.from_numpy(np.ascontiguousarray(mat_np).ravel()).to(dev)
    res = torch.empty(3 * nn, dtype=torch.float64, device=dev)
    vals = torch.empty(nnz, dtype=torch.float64, device=dev)
    hout = torch.empty(56 * ne, dtype=torch.float64, device=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    vjp_in = None
    if args.vjp:   # time fem_assemble_vjp (all three products) with seeded cotangents instead
        g = torch.Generator(device=dev).manual_seed(17390)
        vjp_in = (torch.randn(3 * nn, dtype=torch.float64, device=dev, generator=g),
                  1e3 * torch.randn(56 * ne, dtype=torch.float64, device=dev, generator=g))

    def step():
        if vjp_in is not None:
            ctx.assemble_vjp(u, hin, mat, lam=vjp_in[0], mu=vjp_in[1])
            return
        if world > 1:     # the one collective of the sharded path, then the rank's kernels
            ul = shard.exchange_u(u_owned, part, plan=plan)
            ctx.assemble(ul, hin, mat, res, vals, hout, barlat=bar)
        else:
            ctx.assemble(u, hin, mat, res, vals, hout, barlat=bar)

    peak_tf = fem.probe_fp64_peak(30.0)
    n_warm = max(args.warmup, 3)
    for _ in range(n_warm):
        step()
    _, _, _, stats = ctx.assemble(u, hin, mat, res, vals, hout, want_stats=True, barlat=bar)
    pfrac = stats["n_plastic"] / (8.0 * ne)

    # ---- timed region: exactly K steps between two barriers; one CUDA event between consecutive steps on the launching
    #      (current) stream, so that every step has its own duration: median = ms_per_step, total / K = the mean
    clocks = ClockSampler(local)
    clocks.start()
    barrier()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record()
    for i in range(args.steps):
        step()
        ev[i + 1].record()
    barrier()
    per_step = step_times_ms(ev)
    ms_median_local, ms_mean_local = float(np.median(per_step)), float(np.mean(per_step))
    # per-kernel durations (library events on the same stream), same launches, K more steps: medians
    ksamples = dict(element=[], gather=[], mat_prep=[])
    for _ in range(args.steps):
        ctx.assemble(u, hin, mat, res, vals, hout, barlat=bar)
        k = ctx.last_kernel_ms()
        for key in ksamples:
            ksamples[key].append(k[key])
    kms = {key: float(np.median(v)) for key, v in ksamples.items()}
    clk = clocks.stop()
    ms_step, value = aggregate_over_ranks(ms_median_local, ne_g, world, dev)
    ms_mean, _ = aggregate_over_ranks(ms_mean_local, ne_g, world, dev)

    # ---- end-to-end: host buffers through fem_assemble_host, copies inside the timed region (N = 1 only: the sharded arm's
    #      host path would need the collective on host buffers)
    e2e = None
    if world == 1 and not args.no_e2e and not args.barlat and not args.vjp:
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
        e2e = {"value": ne / t_e2e, "unit": UNIT, "h2d_bytes_per_step": 8 * (hu.numel() + hh.numel() + hm.numel()),
               "d2h_bytes_per_step": 8 * (hres.numel() + hvals.numel() + hhout.numel()), "ms_per_step": 1e3 * t_e2e,
               "steps": e2e_steps, "finite": bool(np.isfinite(hres.numpy()).all())}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (element kernel): FP64 ALU bound
    fl_el = alg_flops_per_element_barlat(pfrac, stats["iter_hist"]) if args.barlat else alg_flops_per_element(pfrac)
    by_el = alg_bytes_per_element(nn_g, ne_g, nnz_g, mat_np.shape[0] > 1)
    hbm_gbs, hbm_src = measured_peaks()
    dom = max(("element", "gather"), key=lambda k: kms[k])
    ach_tf = fl_el * ne / (kms["element"] * 1e-3) / 1e12
    tr = recorded_traffic(args.workload, mode) if (world == 1 and not args.barlat and not args.fbar) else None
    roofline = {"bound": "alu", "kernel": "k_element", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                "frac": ach_tf / peak_tf, "traffic": None if tr is None else tr.get("k_element_bytes"),
                "traffic_step": None if tr is None else tr.get("step_bytes"), "traffic_source": tr,
                "peak_source": "DFMA probe kernel measured live in this run (nominal %.1f)" % NOMINAL_FP64_TFLOPS,
                "alg_flops_per_element": fl_el, "alg_bytes_per_element": by_el,
                "whole_step_frac": max(fl_el * ne_g / world / (peak_tf * 1e12), by_el * ne_g / world / (hbm_gbs * 1e9)) / (ms_step * 1e-3),
                "hbm_peak_gbs": hbm_gbs, "hbm_peak_source": hbm_src, "dominant": dom}

    # ---- CPU baseline: the oracle on a bounded slab sample of the same workload (config 3, N = 1 only)
    cpu = None
    if not args.no_cpu and world == 1 and args.workload == "config3" and not args.barlat:
        try:
            n = args.n
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
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": n_warm,
        "warmup_requested": args.warmup, "ms_per_step": ms_step, "ms_per_step_mean": ms_mean, "higher_is_better": True,
        "scaling": "weak" if world == 1 else "strong", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl_desc, "call": "fem_assemble_vjp (g_u, g_hist_in, g_mat)" if args.vjp else ("fem_assemble_barlat" if args.barlat else "fem_assemble"),
                   "fbar": args.fbar, "assembly_mode": mode, "yield": "Yld2004-18p (Table 2)" if args.barlat else "Hill-48",
                   "partition": "single GPU" if world == 1 else "%d node slabs, ghost elements recomputed, one all-gather of u per step" % world,
                   "l2_policy": "inputs+outputs per step (%.1f GB) exceed the 126 MB L2" % ((by_el * ne_g) / 1e9), "nnz": nnz},
        "clocks": {"sm_mhz": clk["sm_mhz"], "sm_max_mhz": clk["sm_max_mhz"], "reasons": clk["reasons"], "samples": clk["samples"]},
        "e2e": e2e,
        "gpu_launches": args.steps * (ctx.launches_per_assemble() + (1 if args.barlat else 0)),
        "roofline": roofline, "cpu_baseline": cpu,
        "kernels_ms": kms, "plastic_fraction": pfrac, "stats": {k: stats[k] for k in ("n_plastic", "n_nonconverged",
                                                                                    "n_detF_nonpos", "n_nonfinite", "max_local_iters")},
        "iter_hist": {str(k): int(v) for k, v in enumerate(stats["iter_hist"]) if v},
        "setup_s": t_setup, "pattern_s": t_pattern, "partition_s": t_part, "fp64_peak_probe_tflops": peak_tf,
        "local_elems_rank0": ne, "kernel_sha16": kernel_sha16(),
    }
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1, help="number of ranks the driver launches (informative: the ranks come from torchrun's environment)")
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config3", choices=["config1", "config2", "config3", "config4", "config5", "e4"])
    ap.add_argument("--level", type=int, default=2, help="config5 sweep level")
    ap.add_argument("--sweep", default="fraction", choices=["fraction", "strain"])
    ap.add_argument("--n", type=int, default=100, help="mesh resolution of config3 (100 = BASELINE.json)")
    ap.add_argument("--fbar", type=int, default=0)
    ap.add_argument("--mode", type=int, default=None, help="fem_options.assembly_mode (default: the library's default)")
    ap.add_argument("--barlat", action="store_true", help="time fem_assemble_barlat with the Table 2 coefficients instead")
    ap.add_argument("--vjp", action="store_true", help="time fem_assemble_vjp (NEXT-3) instead of fem_assemble")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg")
    args = ap.parse_args()
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus != world and int(os.environ.get("RANK", "0")) == 0 and args.impl == "ours":
        print("bench.py: --gpus %d but WORLD_SIZE=%d: launch with torch.distributed.run --nproc-per-node %d" % (args.gpus, world, args.gpus),
              file=sys.stderr)
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
