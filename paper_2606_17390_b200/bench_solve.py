"""Measurements of SURVEY.md §8(f) NEXT-1 on the paper's unit-cube benchmark (Table 3 :493-495,
Table F1 :1064-1073), 100^3 hex8 = 3,090,903 DOF, one B200:

    python -m paper_2606_17390_b200.bench_solve [--n 100] [--lin-rtol 1e-8]

  1. fem_spmv: ms and achieved GB/s (algorithmic bytes: 8 nnz values + 4 bytes per 3x3 block index + x read + y written).
  2. fem_bicgstab on the linear-elastic stiffness (Table F1's workload: "linear elastic problem on a unit-cube domain";
     left face fixed, right face displaced): iterations, seconds, ms per iteration.  Paper, H100: JAX-BiCGSTAB 11.21 s,
     AMGX-BiCGSTAB 1.96 s at 3,090,903 DOF (tolerance not stated; context, other hardware).
  3. fem_newton_solve: one load increment of the elastoplastic benchmark (Hill-48 + Voce, Table 3; right face moved by
     dt * (0.2, 0.1, 0) mm, dt = 0.05 = the paper's largest step): Newton iterations, BiCGSTAB iterations, seconds.
     Paper, H100: 31 load steps / 111 Newton iterations in 2030 s = 18.3 s per Newton iteration (context).
Prints markdown; kept in profiles/.  Inputs are synthetic (structured unit cube, seeded nothing: the problem is fully
specified by the paper's text).
"""
import argparse
import os
import sys
import time

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def main():
    import torch
    import paper_2606_17390_b200 as fem
    from synth import mesh
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=100)
    ap.add_argument("--fbar", type=int, default=0, help="1: F-bar element (unsymmetric tangent, BiCGSTAB)")
    ap.add_argument("--mesh", default="", help="nx x ny x nz elements on the unit cube, e.g. 250x150x120 (the paper's largest case, :489); overrides --n")
    ap.add_argument("--lin-rtol", type=float, default=1e-8)
    ap.add_argument("--dt", default="0.002,0.005", help="load fractions of the Newton runs, each from the undeformed state")
    ap.add_argument("--path", default="0.002x8", help="load path: step size x number of steps, history and displacement carried over")
    ap.add_argument("--full", type=float, default=0.0, help="if > 0: run the whole benchmark loading (right face to 0.2, 0.1 mm) with "
                    "adaptive stepping (the paper's dt_initial 1e-3, dt_max 5e-2, cut-back on failure, :485) for at most this many seconds")
    ap.add_argument("--extrapolate", type=int, default=1, help="initial guess of a step: 0 last state, 1 linear, 2 quadratic extrapolation")
    ap.add_argument("--adjoint", type=int, default=0, help="1: after the load path, run the backward sweep of Alg. 1 (fem_adjoint_step per step) "
                    "for J = 1/2 sum_n |u^n|^2 on the free DOFs and check dJ/d(sigma0) against a central difference of two more forward paths")
    ap.add_argument("--mixed", type=int, default=0, help="1: fem_set_mixed_precision (fp32 copy of K inside CG, fp64 residuals)")
    ap.add_argument("--grow-below", type=int, default=6, help="grow the step after a step with at most this many Newton iterations")
    args = ap.parse_args()
    n = args.n
    dev = torch.device("cuda:0")
    nx, ny, nz = (int(v) for v in args.mesh.split("x")) if args.mesh else (n, n, n)
    coords, conn = mesh.structured_hex_mesh(nx, ny, nz)
    nn, ne = coords.shape[0], conn.shape[0]
    ctx = fem.FemContext(torch.from_numpy(coords).to(dev), torch.from_numpy(conn).to(dev), fbar=args.fbar)
    ctx.build_csr_pattern()
    if args.mixed:
        ctx.set_mixed_precision(True)
    nnz, nr = ctx.nnz, 3 * nn
    # Table 3: E = 219 GPa, Voce sigma0 = 138, Q = 410, b = 3.8, ratios r11..r23; nu is not printed: 0.3
    rec = fem.mat_record(219000.0, 0.3, [1.5449, 1.0666, 1.0, 1.0307, 1.0, 1.0], 0.0, 138.0, 410.0, 3.8)
    mat = torch.from_numpy(rec).to(dev)
    nid = np.arange(nn)
    lf, rt = np.abs(coords[:, 0]) < 1e-12, np.abs(coords[:, 0] - 1.0) < 1e-12
    bc = np.concatenate([(3 * nid[lf][:, None] + np.arange(3)).ravel(), (3 * nid[rt][:, None] + np.arange(3)).ravel()]).astype(np.int32)
    full = np.concatenate([np.zeros(3 * int(lf.sum())), np.tile([0.2, 0.1, 0.0], int(rt.sum()))])
    bc_d = torch.from_numpy(bc).to(dev)
    hin = torch.zeros(56 * ne, dtype=torch.float64, device=dev)
    u0 = torch.zeros(nr, dtype=torch.float64, device=dev)
    print("# NEXT-1 on the unit-cube benchmark, %d x %d x %d elements, %d DOF, nnz %d\n" % (nx, ny, nz, nr, nnz))

    # ---- 1. SpMV
    res, vals, _, _ = ctx.assemble(u0, hin, mat)
    x = torch.from_numpy(np.random.default_rng(1).normal(size=nr)).to(dev)
    y = torch.empty_like(x)
    for _ in range(3):
        ctx.spmv(vals, x, y)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 20
    e0.record()
    for _ in range(reps):
        ctx.spmv(vals, x, y)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    byts = 8.0 * nnz + 4.0 * nnz / 9 + 16.0 * nr
    print("| fem_spmv | %.3f ms | %.0f GB/s algorithmic (values + block indices + x + y = %.2f GB) |" % (ms, byts / ms / 1e6, byts / 1e9))

    # ---- 2. BiCGSTAB on the linear-elastic stiffness (Table F1 workload)
    rhs = torch.zeros(nr, dtype=torch.float64, device=dev)
    ctx.apply_dirichlet(bc_d, vals, rhs, torch.from_numpy(full * 0.05).to(dev))
    torch.cuda.synchronize()
    for rtol in (1e-6, args.lin_rtol):
        t0 = time.perf_counter()
        xs, its, rr, ok = ctx.bicgstab(vals, rhs, rtol=rtol, max_iter=20000)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        print("| fem_bicgstab, linear elastic, rtol %.0e | %d iterations | %.3f s | %.3f ms/iteration | explicit relres %.2e | converged %s |"
              % (rtol, its, dt, 1e3 * dt / max(its, 1), rr, ok))

    # ---- 3. one elastoplastic load increment from the undeformed state, for several increment sizes
    for dts in [d for d in args.dt.split(",") if d]:
        dtf = float(dts)
        u = torch.zeros(nr, dtype=torch.float64, device=dev)
        t0 = time.perf_counter()
        u, hout, rep = ctx.newton_solve(u, hin, mat, bc_d, torch.from_numpy(full * dtf).to(dev), lin_rtol=args.lin_rtol,
                                        lin_max_iter=5000, rtol=1e-8, max_newton=12)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        st = rep["last_stats"]
        print("| fem_newton_solve, load fraction %.3g (right face %.3g, %.3g mm), Table 3 material | %d Newton iterations | %d linear "
              "iterations | %.2f s total = %.2f s per Newton iteration | plastic fraction %.3f | rhs norm %.2e -> %.2e | converged %s, "
              "linear failures %d |" % (dtf, 0.2 * dtf, 0.1 * dtf, rep["newton_iters"], rep["lin_iters_total"], dt,
                                        dt / max(rep["newton_iters"], 1), st["n_plastic"] / (8.0 * ne), rep["rhs_norm0"], rep["rhs_norm"],
                                        rep["converged"], rep["lin_failures"]), flush=True)

    # ---- 4. a load path: equal steps, converged state and history carried from step to step (the paper's protocol, :485-487,
    #         without its adaptive step control; initial guess = last converged displacement)
    step, nsteps = args.path.split("x")
    step, nsteps = float(step), int(nsteps)
    u = torch.zeros(nr, dtype=torch.float64, device=dev)
    h_a = torch.zeros(56 * ne, dtype=torch.float64, device=dev)
    h_b = torch.empty_like(h_a)
    tot_newton = tot_lin = 0
    t_path = time.perf_counter()
    for k in range(1, nsteps + 1):
        t0 = time.perf_counter()
        u, h_b, rep = ctx.newton_solve(u, h_a, mat, bc_d, torch.from_numpy(full * (step * k)).to(dev), hist_out=h_b,
                                       lin_rtol=args.lin_rtol, lin_max_iter=10000, rtol=1e-8, max_newton=12)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        st = rep["last_stats"]
        print("| path step %d, load fraction %.4g | %d Newton iterations | %d linear iterations | %.2f s | plastic fraction %.3f | "
              "rhs norm %.2e -> %.2e | converged %s, linear failures %d |" % (k, step * k, rep["newton_iters"], rep["lin_iters_total"], dt,
                                                                            st["n_plastic"] / (8.0 * ne), rep["rhs_norm0"], rep["rhs_norm"],
                                                                            rep["converged"], rep["lin_failures"]), flush=True)
        if not rep["converged"]:
            break
        tot_newton += rep["newton_iters"]; tot_lin += rep["lin_iters_total"]
        h_a, h_b = h_b, h_a
    dt = time.perf_counter() - t_path
    print("| path total | %d Newton iterations | %d linear iterations | %.2f s = %.2f s per Newton iteration |"
          % (tot_newton, tot_lin, dt, dt / max(tot_newton, 1)))

    # ---- 4b. NEXT-3: the discrete adjoint of that path (Alg. 1) and the paper's own check of it (Eq.(52) :412)
    if args.adjoint and nsteps > 0:
        free = torch.ones(nr, dtype=torch.float64, device=dev)
        free[bc_d.long()] = 0.0

        def forward(mat_t, keep):
            u = torch.zeros(nr, dtype=torch.float64, device=dev)
            h_a = torch.zeros(56 * ne, dtype=torch.float64, device=dev)
            states, J = [], 0.0
            for k in range(1, nsteps + 1):
                u, h_b, rep = ctx.newton_solve(u, h_a, mat_t, bc_d, torch.from_numpy(full * (step * k)).to(dev),
                                               lin_rtol=1e-10, lin_max_iter=20000, rtol=1e-9, atol=1e-8, max_newton=15)
                assert rep["converged"], rep
                J += 0.5 * float(((u * free) ** 2).sum())
                if keep:
                    states.append((u.clone(), h_a))
                h_a = h_b
            return J, states
        torch.cuda.synchronize(); t0 = time.perf_counter()
        J0, states = forward(mat, True)
        torch.cuda.synchronize(); t_fwd = time.perf_counter() - t0
        t0 = time.perf_counter()
        grad = torch.zeros(16, dtype=torch.float64, device=dev)
        mu, its_tot = None, 0
        for (u_n, h_nm1) in reversed(states):
            lam, mu, g_m, its = ctx.adjoint_step(u_n, h_nm1, mat, bc_d, dJdu=u_n * free, mu_in=mu, lin_rtol=1e-10, lin_max_iter=20000)
            grad += g_m[0]; its_tot += its
        torch.cuda.synchronize(); t_bwd = time.perf_counter() - t0
        g = grad.cpu().numpy()
        print("\n| adjoint of the %d-step path (J = 1/2 sum |u^n|^2 on the free DOFs = %.6e) | forward %.2f s (Newton rtol 1e-9, linear 1e-10) | backward sweep %.2f s "
              "= %.2f s per step, %d CG iterations |" % (nsteps, J0, t_fwd, t_bwd, t_bwd / nsteps, its_tot))
        names = ["E", "nu", "r11", "r22", "r33", "r12", "r23", "r13", "law", "sigma0", "Q", "b"]
        print("| dJ/dtheta | " + " | ".join("%s %.6e" % (names[i], g[i]) for i in (0, 1, 2, 3, 4, 5, 6, 7, 9, 10, 11)) + " |")
        for idx, rel in ((9, 1e-3), (3, 1e-3)):
            mp, mm = mat.clone(), mat.clone()
            hstep = rel * float(mat[idx])
            mp[idx] += hstep; mm[idx] -= hstep
            fd = (forward(mp, False)[0] - forward(mm, False)[0]) / (2 * hstep)
            print("| central difference d J / d %s (Eq.(52), h = %.0e theta) | %.6e | adjoint %.6e | relative difference %.2e |"
                  % (names[idx], rel, fd, g[idx], abs(fd - g[idx]) / abs(fd)), flush=True)

    # ---- 5. the whole benchmark loading with the paper's adaptive stepping parameters (host control flow)
    if args.full > 0:
        t, dt, dt_max, dt_min = 0.0, 1e-3, 5e-2, 1e-5
        u = torch.zeros(nr, dtype=torch.float64, device=dev)
        h_a = torch.zeros(56 * ne, dtype=torch.float64, device=dev)
        h_b = torch.empty_like(h_a)
        steps = newton = lin = rejected = 0
        ts = []                               # accepted load fractions (the schedule the adjoint run below repeats)
        u_try = torch.empty_like(u)
        u_prev = torch.zeros_like(u)          # converged states one and two steps back ("linear or quadratic extrapolation")
        u_pp = torch.zeros_like(u)
        dt_prev = dt_pp = 0.0
        t_start = time.perf_counter()
        print("\n| step | load fraction | dt | Newton iterations | linear iterations | s | plastic fraction | result |")
        print("|---|---|---|---|---|---|---|---|")
        while t < 1.0 - 1e-12 and time.perf_counter() - t_start < args.full:
            dt = min(dt, 1.0 - t)
            t0 = time.perf_counter()
            if args.extrapolate == 2 and dt_pp > 0:      # quadratic (Lagrange) through the last three converged states
                t0_, t1_, t2_, t3_ = -(dt_prev + dt_pp), -dt_prev, 0.0, dt
                l0 = (t3_ - t1_) * (t3_ - t2_) / ((t0_ - t1_) * (t0_ - t2_))
                l1 = (t3_ - t0_) * (t3_ - t2_) / ((t1_ - t0_) * (t1_ - t2_))
                l2 = (t3_ - t0_) * (t3_ - t1_) / ((t2_ - t0_) * (t2_ - t1_))
                ctx.lincomb(l2, u, l1, u_prev, u_try)
                ctx.lincomb(1.0, u_try, l0, u_pp, u_try)
            else:
                r = dt / dt_prev if (dt_prev > 0 and args.extrapolate) else 0.0
                ctx.lincomb(1.0 + r, u, -r, u_prev, u_try)                  # u + (u - u_prev) dt / dt_prev
            u_try, h_b, rep = ctx.newton_solve(u_try, h_a, mat, bc_d, torch.from_numpy(full * (t + dt)).to(dev), hist_out=h_b,
                                               lin_rtol=args.lin_rtol, lin_max_iter=20000, rtol=1e-8, max_newton=12)
            torch.cuda.synchronize()
            el = time.perf_counter() - t0
            st = rep["last_stats"]
            ok = rep["converged"] and rep["lin_failures"] == 0
            print("| %d | %.5f | %.2e | %d | %d | %.2f | %.3f | %s |" % (steps + 1, t + dt, dt, rep["newton_iters"], rep["lin_iters_total"], el,
                                                                  st["n_plastic"] / (8.0 * ne), "ok" if ok else "rejected"), flush=True)
            newton += rep["newton_iters"]; lin += rep["lin_iters_total"]
            if ok:
                t += dt; steps += 1; ts.append(t)
                h_a, h_b = h_b, h_a
                u_pp, u_prev, u, u_try = u_prev, u, u_try, u_pp
                dt_pp, dt_prev = dt_prev, dt
                if rep["newton_iters"] <= args.grow_below:
                    dt = min(dt * 1.5, dt_max)
            else:
                rejected += 1
                dt *= 0.5
                if dt < dt_min:
                    break
        tot = time.perf_counter() - t_start
        print("| total | reached %.4f of the load | | %d (incl. rejected steps) | %d | %.1f | | %d steps accepted, %d rejected |"
              % (t, newton, lin, tot, steps, rejected))

        # ---- 5b. NEXT-3 on the whole benchmark: forward over the accepted schedule with the states kept, backward sweep of Alg. 1,
        #          and the paper's check (Eq.(52) :412) of dJ/d(sigma0) by two more forward runs over the same schedule
        if args.adjoint and t >= 1.0 - 1e-12:
            free = torch.ones(nr, dtype=torch.float64, device=dev)
            free[bc_d.long()] = 0.0

            def run_schedule(mat_t, keep):
                u = torch.zeros(nr, dtype=torch.float64, device=dev)
                u_prev = torch.zeros_like(u)
                h_a = torch.zeros(56 * ne, dtype=torch.float64, device=dev)
                states, J, t_prev, dt_prev, nwt = [], 0.0, 0.0, 0.0, 0
                for tn in ts:
                    r = (tn - t_prev) / dt_prev if dt_prev > 0 else 0.0
                    u_try = ctx.lincomb(1.0 + r, u, -r, u_prev)
                    u_try, h_b, rep = ctx.newton_solve(u_try, h_a, mat_t, bc_d, torch.from_numpy(full * tn).to(dev),
                                                       lin_rtol=1e-10, lin_max_iter=40000, rtol=1e-9, atol=1e-8, max_newton=20)
                    assert rep["converged"], (tn, rep)
                    nwt += rep["newton_iters"]
                    J += 0.5 * float(((u_try * free) ** 2).sum())
                    if keep:
                        states.append((u_try.clone(), h_a))
                    u_prev, u = u, u_try
                    dt_prev, t_prev = tn - t_prev, tn
                    h_a = h_b
                return J, states, nwt
            torch.cuda.synchronize(); t0 = time.perf_counter()
            J0, states, nwt = run_schedule(mat, True)
            torch.cuda.synchronize(); t_fwd = time.perf_counter() - t0
            t0 = time.perf_counter()
            grad = torch.zeros(16, dtype=torch.float64, device=dev)
            mu, its_tot = None, 0
            for (u_n, h_nm1) in reversed(states):
                lam, mu, g_m, its = ctx.adjoint_step(u_n, h_nm1, mat, bc_d, dJdu=u_n * free, mu_in=mu, lin_rtol=1e-10, lin_max_iter=40000)
                grad += g_m[0]; its_tot += its
            torch.cuda.synchronize(); t_bwd = time.perf_counter() - t0
            g = grad.cpu().numpy()
            print("\n| adjoint of the whole benchmark (%d steps, J = 1/2 sum |u^n|^2 on the free DOFs = %.6e) | forward %.1f s, %d Newton iterations "
                  "(Newton rtol 1e-9, linear 1e-10) | backward sweep %.1f s = %.2f s per step, %d Krylov iterations |"
                  % (len(ts), J0, t_fwd, nwt, t_bwd, t_bwd / len(ts), its_tot), flush=True)
            names = ["E", "nu", "r11", "r22", "r33", "r12", "r23", "r13", "law", "sigma0", "Q", "b"]
            print("| dJ/dtheta | " + " | ".join("%s %.6e" % (names[i], g[i]) for i in (0, 1, 2, 3, 4, 5, 6, 7, 9, 10, 11)) + " |", flush=True)
            if args.adjoint > 1:
                idx, rel = 9, 1e-3
                mp, mm = mat.clone(), mat.clone()
                hstep = rel * float(mat[idx])
                mp[idx] += hstep; mm[idx] -= hstep
                fd = (run_schedule(mp, False)[0] - run_schedule(mm, False)[0]) / (2 * hstep)
                print("| central difference d J / d %s (Eq.(52), h = %.0e theta, same schedule) | %.6e | adjoint %.6e | relative difference %.2e |"
                      % (names[idx], rel, fd, g[idx], abs(fd - g[idx]) / abs(fd)), flush=True)


if __name__ == "__main__":
    main()
