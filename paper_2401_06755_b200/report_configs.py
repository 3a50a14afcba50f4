"""Run the five BASELINE.json configurations on cuda:0 and print a markdown report.

    python -m paper_2401_06755_b200.report_configs > gpurun_out/configs.md

Config 1: solve to 1e-8 (fp32 mixed precision and fp64).  Config 2: solve to 1e-7.  Config 3: 20 fixed cycles with
the residual history, per-level time and algorithmic bytes.  Config 4: V(nu, nu) cycles for nu = 1..4, 10 cycles each.
Config 5: full time steps.  Inputs are the seeded synthetic workloads of workloads/configs.py; every number is a
CUDA-event time on the solver's stream after warm-up.  Nothing here touches the oracle.
"""
from __future__ import annotations

import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import paper_2401_06755_b200 as mg          # noqa: E402
from workloads import configs                # noqa: E402


def f32(a):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()


def timed(fn, reps):
    fn()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(reps):
        out = fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps, out


def rhs_from_velocity(w):
    b = torch.empty(w.shape, device="cuda")
    mg.pressure_rhs(f32(w.fields["u"]), f32(w.fields["v"]), f32(w.fields["w"]), w.h, 1.0, b)
    return b


def solver_for(w, dtype=None, **params):
    s = mg.mg_create((w.nx, w.ny, w.nz, w.h), w.levels, w.bc, dtype if dtype is not None else mg.MG_F32)
    p = dict(nu_pre=w.nu_pre, nu_post=w.nu_post, coarse_sweeps=w.coarse_sweeps, sweeps_per_pass=1, omega=w.omega, mixed_precision=1)
    p.update(params)
    mg.mg_set_params(s, **p)
    return s


def collapsing_column(n=64):
    """SURVEY 8(f) next 3, "a real collapsing-column run can be sanity-checked qualitatively": the four-stage step on a water column
    (a = 0.25 wide, H = 0.5 high, unit box, free-slip walls, open top) released from rest, to T* = t sqrt(2 g / a) = 3.5."""
    import time
    levels = int(np.log2(n)) - 1
    w = configs.config5(n, levels)
    h, grav, sig, a, H = w.h, 9.81, 0.0728, 0.25, 0.5
    dt = 0.1 * h / 3.0
    xs = (np.arange(n) + 0.5) * h
    print("\n### A collapsing water column with the four-stage step (%d^3, %d levels, dt = %.2e s = Courant 0.1 at 3 m/s; a = %.2f, H = %.2f; "
          "sqrt(g H) = %.2f, sqrt(2 g H) = %.2f m/s)\n" % (n, levels, dt, a, H, np.sqrt(grav * H), np.sqrt(2 * grav * H)))
    for ps, name in ((0, "plain V(2,2) cycles (mg_solve)"), (1, "V-cycle-preconditioned CG (mg_pcg_solve)")):
        s_hs, s_nh = solver_for(w, cycles_per_defect=0), solver_for(w, cycles_per_defect=0)
        C = f32(w.fields["alpha"])
        u, v, ww = (torch.zeros_like(C) for _ in range(3))
        phs, pnh = torch.zeros_like(C), torch.zeros_like(C)
        vol0 = float(C.double().sum())
        t, step, cycles, nxt, worst = 0.0, 0, 0, 0.5, 0
        print("stage 3 by %s:\n" % name)
        print("| T* | t s | front x/a | column height / H | liquid volume drift | min C | max C | max liquid speed m/s | max speed m/s | cycles per step |")
        print("|---|---|---|---|---|---|---|---|---|---|")
        torch.cuda.synchronize(); t0 = time.perf_counter()
        while t * np.sqrt(2 * grav / a) < 3.5:
            st, cyc, rel = mg.flow_time_step_full_ex(s_hs, s_nh, C, u, v, ww, phs, pnh, w.rho_l, w.rho_g, w.mu_l, w.mu_g, grav, sig, dt,
                                                     1e-6, 100, 0.0, 20, (1, 1, 1, 1, 1, 0), ps)
            t += dt; step += 1; cycles += cyc; worst = max(worst, st)
            ts = t * np.sqrt(2 * grav / a)
            if ts >= nxt:
                Cb, Cw = C[0, n // 2, :].cpu().numpy(), C[:, n // 2, 0].cpu().numpy()
                wet, col = np.where(Cb > 0.5)[0], np.where(Cw > 0.5)[0]
                sp = torch.sqrt(u * u + v * v + ww * ww)
                print("| %.2f | %.4f | %.2f | %.2f | %+.1e | %.3f | %.3f | %.2f | %.2f | %.1f |" % (
                    ts, t, xs[wet.max()] / a if wet.size else 0.0, xs[col.max()] / H if col.size else 0.0,
                    float(C.double().sum()) / vol0 - 1, float(C.min()), float(C.max()), float((sp * (C > 0.5)).max()), float(sp.max()),
                    cycles / step))
                nxt += 0.5
        torch.cuda.synchronize()
        print("\n%d steps, %.2f ms per step (wall clock, host loop included), worst stage-3 status %d\n" % (step, (time.perf_counter() - t0) / step * 1e3, worst))
        mg.mg_destroy(s_hs); mg.mg_destroy(s_nh)
    print("Without the limit on C in the material mixtures (DESIGN.md reading C7) the same run ends at T* = 0.7 (at 32^3: 0.9): C undershoots to -0.003 in the thin tongue at the front, rho = 1000 C + (1 - C) turns negative there, the stage-3 operator loses definiteness and both solvers diverge within twenty steps.")


def main():
    torch.cuda.set_device(0)
    print("# The five BASELINE.json configurations on one B200 (%s)\n" % mg.mg_version())
    print("Made by `python -m paper_2401_06755_b200.report_configs`; CUDA-event times, fp32 unless noted.\n")

    # ---- config 1 ----
    w = configs.config1()
    print("## Config 1: 32^3, constant coefficient, Dirichlet, 4 levels, solve to 1e-8\n")
    print("| dtype | status | cycles | relative residual | ms per solve |\n|---|---|---|---|---|")
    for name, dt, tdt in (("fp32 + fp64 defect correction", mg.MG_F32, torch.float32), ("fp64", mg.MG_F64, torch.float64)):
        s = solver_for(w, dt)
        b = torch.from_numpy(w.fields["b"]).to(tdt).cuda()
        x = torch.zeros_like(b)

        def run():
            x.zero_()
            return mg.mg_solve(s, x, b, w.tol, 100)
        ms, (st, cyc, rel) = timed(run, 5)
        print("| %s | %d | %d | %.2e | %.3f |" % (name, st, cyc, rel, ms))
        mg.mg_destroy(s)

    # ---- config 2 ----
    w = configs.config2()
    print("\n## Config 2: 128^3 water column (rho 1000:1), 6 levels, solve to 1e-7\n")
    s = solver_for(w)
    mg.mg_set_coefficient_from_vof(s, f32(w.fields["alpha"]), w.rho_l, w.rho_g)
    b = rhs_from_velocity(w)
    x = torch.zeros_like(b)

    def run2():
        x.zero_()
        return mg.mg_solve(s, x, b, w.tol, 100)
    ms, (st, cyc, rel) = timed(run2, 5)
    print("status %d, %d cycles, relative residual %.2e, %.3f ms per solve (%.3f ms per cycle including the fp64 residual)\n"
          % (st, cyc, rel, ms, ms / max(cyc, 1)))
    print("history: " + ", ".join("%.2e" % h for h in mg.mg_get_history(s)))
    mg.mg_destroy(s)

    # ---- config 3 ----
    w = configs.config3()
    print("\n## Config 3: 256^3 rising bubble, 7 levels, 20 fixed V(2,2) cycles (P:429)\n")
    s = solver_for(w)
    mg.mg_set_coefficient_from_vof(s, f32(w.fields["alpha"]), w.rho_l, w.rho_g)
    b = rhs_from_velocity(w)
    x = torch.zeros_like(b)

    def run3():
        x.zero_()
        return mg.mg_solve(s, x, b, 0.0, 20)
    ms, (st, cyc, rel) = timed(run3, 3)
    print("20 cycles with fp64 residuals: %.3f ms (%.1f V-cycles/s); final relative residual %.2e\n" % (ms, 20e3 / ms, rel))
    print("history: " + ", ".join("%.2e" % h for h in mg.mg_get_history(s)) + "\n")
    mg.mg_set_params(s, nu_pre=w.nu_pre, nu_post=w.nu_post, coarse_sweeps=w.coarse_sweeps, sweeps_per_pass=1, omega=w.omega,
                     mixed_precision=1, cycles_per_defect=0)
    ms, (st, cyc, rel) = timed(run3, 3)
    print("the same with cycles_per_defect = 0 (fp64 defects after cycles %s): %.3f ms (%.1f V-cycles/s); final relative residual %.2e\n"
          % (mg.mg_get_history_cycles(s), ms, 20e3 / ms, rel))
    mg.mg_set_params(s, nu_pre=w.nu_pre, nu_post=w.nu_post, coarse_sweeps=w.coarse_sweeps, sweeps_per_pass=1, omega=w.omega,
                     mixed_precision=1, cycles_per_defect=1)
    def run3p():
        x.zero_()
        return mg.mg_pcg_solve(s, x, b, 1e-7, 100)
    ms, (st, its, rel) = timed(run3p, 3)
    print("V-cycle-preconditioned CG (mg_pcg_solve, not in the paper) to 1e-7: status %d, %d iterations, relative residual %.2e, %.2f ms\n"
          % (st, its, rel, ms))
    print("history: " + ", ".join("%.2e" % h for h in mg.mg_get_history(s)) + "\n")
    msc, _ = timed(lambda: mg.mg_vcycle(s, x, b), 200)
    print("one V-cycle (CUDA graph): %.1f us = %.0f V-cycles/s\n" % (msc * 1e3, 1e3 / msc))
    dn = np.zeros(w.levels); up = np.zeros(w.levels)
    for _ in range(20):
        a, c = mg.mg_vcycle_timed(s, x, b)
        dn += a; up += c
    dn /= 20; up /= 20
    print("| level | grid | points | down leg us | up leg us | algorithmic MB per cycle (77.5 B/point as launched) |\n|---|---|---|---|---|---|")
    for l in range(w.levels):
        n, (nx, ny, nz) = mg.mg_level_info(s, l)
        print("| %d | %dx%dx%d | %d | %.1f | %.1f | %.1f |" % (l, nx, ny, nz, n, dn[l] * 1e3, up[l] * 1e3, n * 77.5e-6))
    print("\n(per-level times are taken outside the graph, with events between the launches: their sum exceeds the graph's cycle time;"
          " the levels from 16^3 down run as one cluster kernel, timed under level 4)")
    r3 = torch.empty_like(b)
    msr, _ = timed(lambda: mg.mg_residual(s, x, b, r3), 50)
    msa, _ = timed(lambda: mg.mg_apply_operator(s, x, r3), 50)
    print("\nmg_residual (r = b - A x, 16 B/point): %.1f us = %.0f GB/s; mg_apply_operator (y = A x, 12 B/point): %.1f us = %.0f GB/s"
          " (streaming kernel, MODE_RES)" % (msr * 1e3, 16.0 * w.n / msr * 1e-6, msa * 1e3, 12.0 * w.n / msa * 1e-6))
    del r3
    mg.mg_destroy(s)

    # ---- what bounds the smoother: sweep time against the footprint, and the wave kernel ----
    print("\n### What bounds the fine-level smoother: one sweep on 256 x 256 x nz (x, k, b read + x written = 16 B/point)\n")
    print("| nz | footprint MB | us per sweep | ps per point | effective GB/s |\n|---|---|---|---|---|")
    for nz in (32, 64, 96, 128, 192, 256):
        sp = mg.mg_create((256, 256, nz, 1.0 / 256), 1, w.bc, mg.MG_F32)
        kk = torch.rand((nz, 256, 256), device="cuda") + 0.5
        bb = torch.randn((nz, 256, 256), device="cuda")
        mg.mg_set_coefficient(sp, kk)
        xs = torch.zeros_like(bb)
        msp, _ = timed(lambda: mg.mg_smooth(sp, xs, bb, 40), 3)
        n = nz * 65536
        print("| %d | %.1f | %.2f | %.2f | %.0f |" % (nz, 16.0 * n / 1e6, msp / 40 * 1e3, msp / 40 * 1e9 / n, 16.0 * n / (msp / 40) * 1e-6))
        mg.mg_destroy(sp)
        del kk, bb, xs
    print("\n(footprints up to ~100 MB stay in the 126 MB L2, yet a point costs the same ~3 ps as at 268 MB, where the fields stream from"
          " HBM: the kernel is bound inside the SM -- issue slots and shared-memory pipe, profiles/r02_ncu_kernels.md -- not by HBM, so"
          " keeping an intermediate iterate in L2 cannot make a pass cheaper)")
    print("\n### Config 3 with the wave kernel: sweeps_per_pass stages of a level per launch (wave_kernel.cuh)\n")
    print("| sweeps_per_pass | us per V-cycle | V-cycles/s | us per sweep (mg_smooth, 24 sweeps) | launches per cycle |\n|---|---|---|---|---|")
    s = solver_for(w)
    mg.mg_set_coefficient_from_vof(s, f32(w.fields["alpha"]), w.rho_l, w.rho_g)
    for spp in (1, 2, 3, 4):
        mg.mg_set_params(s, nu_pre=2, nu_post=2, coarse_sweeps=50, sweeps_per_pass=spp, omega=w.omega, mixed_precision=1)
        x = torch.zeros_like(b)
        msc, _ = timed(lambda: mg.mg_vcycle(s, x, b), 100)
        l0 = mg.mg_launch_count(s); mg.mg_vcycle(s, x, b); lc = mg.mg_launch_count(s) - l0
        mss, _ = timed(lambda: mg.mg_smooth(s, x, b, 24), 3)
        print("| %d | %.1f | %.0f | %.1f | %d |" % (spp, msc * 1e3, 1e3 / msc, mss / 24 * 1e3, lc))
    mg.mg_destroy(s)

    # ---- config 4 ----
    w = configs.config4()
    print("\n## Config 4: 512x512x256 (3 fields = 0.8 GB), four bubbles, 7 levels, V(nu, nu) for nu = 1..4, 10 cycles each\n")
    s = solver_for(w)
    mg.mg_set_coefficient_from_vof(s, f32(w.fields["alpha"]), w.rho_l, w.rho_g)
    b = rhs_from_velocity(w)
    x = torch.zeros_like(b)
    print("| nu | sweeps_per_pass | us per cycle | V-cycles/s | GLUPS | residual over 10 cycles | mg_solve(1e-6, 10) |\n|---|---|---|---|---|---|---|")
    npts = [mg.mg_level_info(s, l)[0] for l in range(w.levels)]
    names = {mg.MG_OK: "MG_OK", mg.MG_NOT_CONVERGED: "MG_NOT_CONVERGED", mg.MG_STAGNATED: "MG_STAGNATED"}
    for nu in (1, 2, 3, 4):
        for spp in (1, 4):
            mg.mg_set_params(s, nu_pre=nu, nu_post=nu, coarse_sweeps=50, sweeps_per_pass=spp, omega=w.omega, mixed_precision=1)
            x.zero_()
            st, cyc, rel = mg.mg_solve(s, x, b, 0.0, 10)
            h = mg.mg_get_history(s)
            x.zero_()
            st2, cyc2, rel2 = mg.mg_solve(s, x, b, 1e-6, 10)
            msc, _ = timed(lambda: mg.mg_vcycle(s, x, b), 50)
            lups = sum(n * 2 * nu for n in npts[:-1]) + npts[-1] * 50
            print("| %d | %d | %.1f | %.0f | %.1f | %.2e -> %.2e | %s after %d cycles |"
                  % (nu, spp, msc * 1e3, 1e3 / msc, lups / msc * 1e-6, h[0], h[-1], names.get(st2, str(st2)), cyc2))
    print("\n(V(1,1) DIVERGES on this problem -- four 1000:1 bubbles, piecewise-constant transfers: mg_solve reports MG_STAGNATED;"
          " V(2,2) and up converge slowly, as on config 3.  sweeps_per_pass = 4 is the wave kernel, wave_kernel.cuh: on this grid"
          " level 0 has 256 tiles, more than fit the machine twice, so it keeps one stage per launch and the coarser levels carry"
          " up to 4; it is slower than one stage per launch, DESIGN.md 5.9)")
    mg.mg_destroy(s)
    del x, b

    # ---- config 5 ----
    w = configs.config5()
    print("\n## Config 5: full time step on 256^3 (momentum x2, pressure RHS, solve to 1e-6, projection, VoF)\n")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    # cycles_per_defect: 1 = an fp64 defect (residual check) after every cycle, the library's default; 0 = the solve loop picks the
    # cycles of every round from the contraction it observes (what bench.py uses)
    for cpd in (1, 0):
        s = solver_for(w, cycles_per_defect=cpd)
        C, u, v, ww = (f32(w.fields[q]) for q in ("alpha", "u", "v", "w"))
        p = torch.empty_like(C)
        cycs = []
        for it in range(12):
            if it == 2:
                torch.cuda.synchronize(); e0.record()
            st, cyc, rel = mg.flow_time_step(s, C, u, v, ww, p, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt, w.tol, 100)
            cycs.append(cyc)
        e1.record(); torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 10
        print("cycles_per_defect %d: 10 steps after 2 warm-up steps: %.2f ms per step = %.1f time-steps/s; cycles per solve %s (residual "
              "checks of the last solve after cycles %s); last status %d, relres %.2e\n"
              % (cpd, ms, 1e3 / ms, cycs[2:], mg.mg_get_history_cycles(s), st, rel))
        if cpd == 1:
            mg.mg_destroy(s)
    print("volume fraction after 12 steps: min %.4f max %.4f; max |q| %.4f" % (float(C.min()), float(C.max()),
          float(torch.maximum(torch.maximum(u.abs().max(), v.abs().max()), ww.abs().max()))))
    C, u, v, ww = (f32(w.fields[q]) for q in ("alpha", "u", "v", "w"))
    its = []
    for it in range(12):
        if it == 2:
            torch.cuda.synchronize(); e0.record()
        st, n_it, rel = mg.flow_time_step_pcg(s, C, u, v, ww, p, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt, w.tol, 100)
        its.append(n_it)
    e1.record(); torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / 10
    print("\nthe same 12 steps with V-cycle-preconditioned CG for the pressure (flow_time_step_pcg, not in the paper): %.2f ms per step = "
          "%.1f time-steps/s; iterations per solve %s; last status %d, relres %.2e" % (ms, 1e3 / ms, its[2:], st, rel))
    mg.mg_destroy(s)

    # ---- the paper's four-stage step ----
    print("\n### The paper's four-stage step (stage 1 hydrostatic + surface-tension pressure, 20 fixed cycles; free-slip walls; "
          "forcing terms of Eq. 18; stage 3 to 1e-6), flow_time_step_full, from rest under gravity\n")
    dt_full = 0.1 * w.h / 3.0          # Courant 0.1 at the free-fall speed sqrt(2 g H) ~ 3 m/s of a unit box
    for cpd in (1, 0):
        s_hs = solver_for(w, cycles_per_defect=cpd)
        s_nh = solver_for(w, cycles_per_defect=cpd)
        C = f32(w.fields["alpha"])
        u, v, ww = (torch.zeros_like(C) for _ in range(3))
        phs, pnh = torch.zeros_like(C), torch.zeros_like(C)
        cycs = []
        for it in range(7):
            if it == 2:
                torch.cuda.synchronize(); e0.record()
            st, cyc, rel = mg.flow_time_step_full(s_hs, s_nh, C, u, v, ww, phs, pnh, w.rho_l, w.rho_g, w.mu_l, w.mu_g, 9.81, 0.0728,
                                                  dt_full, w.tol, 100, 0.0, 20)
            cycs.append(cyc)
        e1.record(); torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / 5
        print("cycles_per_defect %d: 5 steps after 2 warm-up steps: %.2f ms per step = %.1f time-steps/s; stage-3 cycles per solve %s; last "
              "status %d, relres %.2e; max |q| %.4f m/s after 7 steps of %.2e s (g t = %.4f)\n"
              % (cpd, ms, 1e3 / ms, cycs[2:], st, rel, float(torch.maximum(torch.maximum(u.abs().max(), v.abs().max()), ww.abs().max())),
                 dt_full, 9.81 * 7 * dt_full))
        mg.mg_destroy(s_hs); mg.mg_destroy(s_nh)
        del phs, pnh

    collapsing_column(64)

    print("\n### The same step with the paper's own stage 3 (constant-coefficient Laplacian, density on the right, Eqs. 52-53; "
          "2 passes x 20 fixed cycles, P:429, P:498)\n")
    s = solver_for(w)
    init = [f32(w.fields[q]) for q in ("alpha", "u", "v", "w")]
    C, u, v, ww = (t.clone() for t in init)
    p = torch.empty_like(C)
    tot, umax = 0.0, []
    for it in range(7):                     # every step starts from the initial fields (see the note below)
        for dst, src in zip((C, u, v, ww), init):
            dst.copy_(src)
        e0.record()
        rel = mg.flow_time_step_paper(s, C, u, v, ww, p, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt, 20, 2)
        e1.record(); torch.cuda.synchronize()
        if it >= 2:
            tot += e0.elapsed_time(e1)
    umax = float(torch.maximum(torch.maximum(u.abs().max(), v.abs().max()), ww.abs().max()))
    ms = tot / 5
    print("5 single steps from the initial fields after 2 warm-up steps: %.2f ms per step = %.1f time-steps/s (40 V-cycles per step); "
          "relative residual of the last solve %.2e; max |q| after the step %.2f" % (ms, 1e3 / ms, rel, umax))
    print("\nNote: with this reading of Eqs. 52-54 the synthetic config-5 input is not stable over several steps (max |q| 1 -> 5 after one "
          "step, growing further): the correction divides by rho while the Laplacian is constant-coefficient, and the neglected "
          "dq . grad(rho) term is large at a sharp 1000:1 interface under a prescribed swirl.  The oracle shows the same numbers (parity "
          "is green); long-run fidelity of this variant is unverified, as SURVEY 8(c) C9 says of the VoF scheme.\n")
    x = torch.zeros_like(C); b = torch.randn_like(C)
    msc, _ = timed(lambda: mg.mg_vcycle(s, x, b), 200)
    print("\none constant-coefficient V-cycle (12 B per point update): %.1f us = %.0f V-cycles/s" % (msc * 1e3, 1e3 / msc))

    # Eq. 56: wall time per step and node = M_s + N_I N_nh H_s (no hydrostatic solve in this step: N_h = 0)
    print("\n### The paper's cost model, Eq. 56, fitted on this GPU (strategies i-j of Fig. 18, P:668: i corrections x j multigrid "
          "iterations)\n")
    print("| multigrid iteration | 1-10 ms | 2-10 ms | 1-20 ms | 2-20 ms | M_s s/node/step | H_s s/node/iteration | worst fit error |\n|---|---|---|---|---|---|---|---|")
    nn = float(C.numel())
    for label, nu, mp in (("V(2,2) + fp64 defect per iteration (the default here)", 2, 1), ("V(1,1), fp32 residual norm per iteration", 1, 0)):
        mg.mg_set_params(s, nu_pre=nu, nu_post=nu, coarse_sweeps=50, sweeps_per_pass=1, omega=w.omega, mixed_precision=mp)
        pts = []
        for i, j in ((1, 10), (2, 10), (1, 20), (2, 20)):
            tot = 0.0
            for it in range(4):
                for dst, src in zip((C, u, v, ww), init):
                    dst.copy_(src)
                e0.record()
                mg.flow_time_step_paper(s, C, u, v, ww, p, w.rho_l, w.rho_g, w.mu_l, w.mu_g, w.dt, j, i)
                e1.record(); torch.cuda.synchronize()
                if it >= 1:
                    tot += e0.elapsed_time(e1)
            pts.append((i * j, tot / 3))
        A = np.array([[1.0, q] for q, _ in pts]); y = np.array([t for _, t in pts])
        (a0, a1), *_ = np.linalg.lstsq(A, y, rcond=None)
        err = float(np.max(np.abs(A @ np.array([a0, a1]) - y) / y))
        print("| %s | %s | %.2e | %.2e | %.1f %% |" % (label, " | ".join("%.2f" % t for _, t in pts), a0 * 1e-3 / nn, a1 * 1e-3 / nn, 100 * err))
    print("\nThe paper's fit on an NVIDIA A10 (P:515): M_s = 1.2e-8, H_s = 1.1e-10 s per node; its multigrid iteration is a saw-tooth cycle "
          "whose sweep counts are not given (BASELINE.md), so H_s compares only in order of magnitude.")
    mg.mg_destroy(s)


if __name__ == "__main__":
    main()
