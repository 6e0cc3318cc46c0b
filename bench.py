#!/usr/bin/env python
"""bench.py -- Jacobian builds/s of the ghost/gluon DSE Newton-matrix hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

One "step" = one pass of the whole hot path (prep -> point kernel -> DMMA contraction -> assembly:
residual F and analytic Newton matrix J) over the workload's seeded synthetic inputs, through the
C ABI (include/dse.h).  Default workload: BASELINE.json configs[3] (N=64, N_r=1024, N_theta=128), the
configuration north_star quotes the "% of fp64 peak" metric on.  Prints ONE JSON line (rank 0).
N > 1: every rank builds its own replica of the workload (the path has no exchange step; DESIGN.md
"Multi-GPU": replicas / batch sharding only) -> weak scaling, value = all ranks' builds / max time.
--impl reference times the CPU oracle (oracle/, a deliberately plain serial program) on the same
workload; each step is a bounded sample (whole external points) of one build.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from workloads import CONFIGS, config_inputs   # noqa: E402

# fp64 FMA peak of one B200 derived from unit counts and clocks (B200_PROFILING.md: 148 SMs,
# clocks.max.sm 1965 MHz; 64 fp64 FMA lanes per SM = 16 per SM sub-partition): DESIGN.md "Roofline".
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def algorithmic_flops(w, n_batch):
    """12 N flops per quadrature point and system: 3N FMA for the two series at z with
    the shared T_j recurrence + 3N FMA for the three z-dependent Jacobian streams."""
    return 12.0 * w.n_cheb * w.points * n_batch


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML during the timed region."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag, self.max_mhz = index, [], set(), False, None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def sample(self):
        if self.nv is None:
            return
        nv = self.nv
        try:
            self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
            r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
            names = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20,
                     "hw_thermal_slowdown": 0x40, "hw_power_brake_slowdown": 0x80}
            for k, bit in names.items():
                if r & bit:
                    self.reasons.add(k)
        except Exception:
            pass

    def run(self):
        while not self.stop_flag:
            self.sample()
            time.sleep(0.01)

    def result(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def oracle_params(w):
    from oracle.oracle import make_params
    return make_params(w.n_cheb, w.n_r, w.n_theta, w.eps2, w.L2, w.x_G, w.x_Z, w.alpha_mu, w.n_colors, w.delta,
                       w.ir_exp_G, w.ir_exp_Z, w.uv_omega, getattr(w, "angular_rule", 0), getattr(w, "n_ir", 0), getattr(w, "radial_split", 0))


def time_oracle_points(w, c, n_points, start=0):
    """Times the oracle, as it stands, on `n_points` external points of one build (self-energies and
    all four derivative rows = everything a build computes for those points).  Returns seconds."""
    from oracle.oracle import Oracle
    orc = Oracle()
    p = oracle_params(w)
    tab = orc.tables(p)
    t0 = time.perf_counter()
    for e in range(start, start + n_points):
        orc.self_energy(p, c, tab["x_ext"][e % w.n_ext], tab["y"], tab["Wy"], tab["theta"], tab["Omega"], derivs=True)
    return time.perf_counter() - t0


def cpu_baseline(w, c, budget_s=12.0):
    """Oracle on a bounded sample: whole external points of one build, ~budget_s of CPU work."""
    t1 = time_oracle_points(w, c, 1)
    n = int(max(1, min(w.n_ext, budget_s / max(t1, 1e-6))))
    reps = int(max(1, min(50, budget_s / max(t1 * n, 1e-6)))) if n == w.n_ext else 1     # small builds: whole builds, repeated
    t = sum(time_oracle_points(w, c, n) for _ in range(reps)) / reps
    builds_per_s = (n / w.n_ext) / t
    return {"value": builds_per_s, "unit": "jacobian_builds/s", "cores": 1, "kind": "oracle",
            "sample": f"{reps} x {n} of {w.n_ext} external points of one {w.name} build ({n * w.n_r * w.n_theta} quadrature "
                      f"points, {t:.2f} s each, serial fp64 C, gcc -O2), scaled to a full build",
            "points_per_s": n * w.n_r * w.n_theta / t}


def oracle_converged_solve():
    """cpu_baseline leg, config 2 only: the oracle's own Newton loop on config 2' (same inputs, same relaxation rule)."""
    from oracle.oracle import Oracle
    from workloads import paper_scaling_workload, scaling_start_coefficients, PAPER_SCALING_BC
    ws = paper_scaling_workload()
    orc, p = Oracle(), oracle_params(ws)
    t0 = time.perf_counter()
    c, hist, status = orc.newton_solve(p, scaling_start_coefficients(ws), PAPER_SCALING_BC[0], PAPER_SCALING_BC[1],
                                       rho=1.0, step_cap=0.5, tol=1e-11, max_iter=30)
    dt = time.perf_counter() - t0
    al = []
    for xv in (91.2 ** 2, ws.eps2):
        g, z = orc.ln_dress(p, c, xv)
        al.append(float(np.exp(2 * g + z)))
    return {"iterations": len(hist), "status": status, "seconds_total": dt, "alpha_MZ2": al[0], "alpha_eps2": al[1]}


def run_reference(args, w, c):
    """--impl reference: the CPU oracle, as it stands, on the box's host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    t1 = time_oracle_points(w, c[0], 1)
    per_step_budget = 120.0 / max(1, args.steps + args.warmup)
    n = int(max(1, min(w.n_ext, per_step_budget / max(t1, 1e-6))))
    for i in range(args.warmup):
        time_oracle_points(w, c[0], n, start=i * n)
    t = 0.0
    for i in range(args.steps):
        t += time_oracle_points(w, c[0], n, start=i * n)
    ms = 1e3 * t / args.steps
    value = (n / w.n_ext) / (t / args.steps)
    sample = (f"each step = {n} of {w.n_ext} external points of one {w.name} build "
              f"({n * w.n_r * w.n_theta} quadrature points), scaled to full builds")
    line = {
        "impl": "reference", "metric": "fp64 Jacobian builds/s", "value": value, "unit": "jacobian_builds/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "n_cheb": w.n_cheb, "n_r": w.n_r, "n_theta": w.n_theta, "n_batch": 1,
                   "eps2": w.eps2, "L2": w.L2, "sample": sample},
        "cpu_baseline": {"value": value, "unit": "jacobian_builds/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "jacobian_builds/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
        "points_per_s": n * w.n_r * w.n_theta / (t / args.steps),
    }
    print(json.dumps(line), flush=True)


def measure(args, cfg_id, steps, warmup, geometry_cache, env, light=False):
    """One bench line (a dict) for BASELINE config `cfg_id`.  light: a per_config entry of the default run -- no CPU
    baseline, shorter side measurements."""
    import torch
    import torch.distributed as dist
    from paper_1206_1779_b200 import Dse, params_from_workload, DSE_FLAG_GEOMETRY_CACHE, DSE_FLAG_CONST_COEF
    from paper_1206_1779_b200.sharding import max_over_ranks

    rank, world, local, flush = env["rank"], env["world"], env["local"], env["flush"]
    w, c, bc = config_inputs(cfg_id)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    class _A:      # the knobs the body below reads
        pass
    a_ = _A(); a_.steps = steps; a_.warmup = warmup; a_.geometry_cache = geometry_cache; a_.config = cfg_id
    a_.const_coef = args.const_coef; a_.no_cpu_baseline = args.no_cpu_baseline or light
    args = a_

    nb = c.shape[0]
    flags = DSE_FLAG_GEOMETRY_CACHE if args.geometry_cache else 0
    if nb == 1 and w.n_cheb % 8 == 0 and w.n_theta >= 32 and args.const_coef:
        flags |= DSE_FLAG_CONST_COEF        # coefficients as constant-bank operands (explicit, one handle at a time)
    d = Dse(params_from_workload(w, n_batch=nb, flags=flags))
    n2 = 2 * w.n_cheb
    ct = torch.from_numpy(c).cuda()
    bt = torch.from_numpy(bc).cuda()
    J = torch.empty((nb, n2, n2), dtype=torch.float64, device="cuda")
    F = torch.empty((nb, n2), dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()

    newton = args.config == 2          # config 2: a step is one full Newton-Raphson step (build + LU + update)
    c_work = ct.clone()
    stats = torch.empty((nb, 4), dtype=torch.float64, device="cuda")

    def one_step():
        if newton:
            c_work.copy_(ct)            # every timed step solves from the same iterate (G = Z = 1)
            d.newton_step(c_work, bt, 1.0, stats)
        else:
            d.jacobian(ct, bt, J, F)

    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        one_step()
    barrier()

    # ---- timed region: K steps, each bracketed by its own event pair; L2 flushed between steps ----
    # (run twice: plain, then with per-kernel events; the clock sampler covers both)
    sampler = ClockSampler(local)
    sampler.sample()
    sampler.start()
    def timed_pass():
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        barrier()
        t0 = time.perf_counter()
        for k in range(args.steps):
            flush.zero_()
            ev[k][0].record(stream)
            one_step()
            ev[k][1].record(stream)
        barrier()
        return float(np.sum([a.elapsed_time(b) for a, b in ev])), time.perf_counter() - t0

    # pass 1: the K timed steps exactly as a user runs them -> value, ms_per_step
    l0 = d.launch_count()
    total_ms, t_wall = timed_pass()
    launches = d.launch_count() - l0
    # pass 2: the same K steps with a CUDA event pair around every point-kernel launch (dse_set_timing) -> roofline.
    # Kept apart from pass 1 because an event record between two kernels turns their programmatic (PDL) edge
    # into a full one; the instrumented pass reports its own ms_per_step beside the kernel time.
    d.set_timing(True)
    inst_total_ms, _ = timed_pass()
    kernel_ms, kernel_n = d.get_timing()
    d.set_timing(False)
    sampler.sample()
    sampler.stop_flag = True
    total_ms = max_over_ranks(total_ms, device="cuda")            # multi-GPU numbers: max over ranks
    ms_per_step = total_ms / args.steps
    value = world * nb * args.steps / (total_ms * 1e-3)

    # ---- end to end through the C ABI with host (pinned) buffers: H2D of c, bc and D2H of J, F each step ----
    c_h = torch.from_numpy(c).pin_memory(); bc_h = torch.from_numpy(bc).pin_memory()
    J_h = torch.empty((nb, n2, n2), dtype=torch.float64).pin_memory()
    F_h = torch.empty((nb, n2), dtype=torch.float64).pin_memory()
    e2e_steps = min(args.steps, 100 if light else 200)
    cn_h = torch.empty((nb, n2), dtype=torch.float64).pin_memory()          # config 2: the updated coefficients ...
    st_h = torch.empty((nb, 4), dtype=torch.float64).pin_memory()           # ... and the step's stats come back
    c_e2e = torch.empty_like(ct); bc_e2e = torch.empty_like(bt)

    def e2e_step():
        if newton:      # host c, bc -> device, one Newton step (build + LU + update), new c and stats -> host
            c_e2e.copy_(c_h, non_blocking=True); bc_e2e.copy_(bc_h, non_blocking=True)
            d.newton_step(c_e2e, bc_e2e, 1.0, stats)
            cn_h.copy_(c_e2e, non_blocking=True); st_h.copy_(stats, non_blocking=True)
            torch.cuda.current_stream().synchronize()
        else:           # host c, bc -> device, build, J and F -> host (dse_jacobian_host, synchronous)
            d.jacobian_host(c_h.numpy(), bc_h.numpy(), J_h.numpy(), F_h.numpy())

    for _ in range(3):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    t_e2e = max_over_ranks(t_e2e, device="cuda")
    e2e_value = world * nb * e2e_steps / t_e2e
    e2e_d2h = int(cn_h.numel() * 8 + st_h.numel() * 8) if newton else int(J_h.numel() * 8 + F_h.numel() * 8)

    # ---- every other config: the same build followed by the Newton update H9 (equilibrated LU, c <- c - Delta) ----
    with_update = None
    if not newton:
        n_up = min(args.steps, 100 if light else 200)
        for _ in range(3):
            c_work.copy_(ct)
            d.newton_step(c_work, bt, 1.0, stats)
        barrier()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_up)]
        for a, b in evs:
            flush.zero_()
            c_work.copy_(ct)
            a.record(stream)
            d.newton_step(c_work, bt, 1.0, stats)
            b.record(stream)
        barrier()
        ms_up = max_over_ranks(float(np.mean([a.elapsed_time(b) for a, b in evs])), device="cuda")
        with_update = {"value": world * nb / (ms_up * 1e-3), "unit": "newton_steps/s", "ms_per_step": ms_up, "steps": n_up,
                       "what": "build (H1-H8) + Newton update H9 (row-equilibrated LU with partial pivoting, solve, c <- c - Delta) "
                               "through dse_newton_step"}

    # ---- config 2 only: the whole iteration as ONE device-side graph (dse_newton_solve), fixed step count ----
    solve = None
    if newton:
        iters, reps = 8, (20 if light else 50)
        info_t = torch.empty((nb, 6), dtype=torch.float64, device="cuda")
        for _ in range(3):
            c_work.copy_(ct)
            d.newton_solve(c_work, bt, 1.0, 0.5, 0.0, iters, info_t)
        barrier()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(reps)]
        for a, b in evs:
            flush.zero_()
            c_work.copy_(ct)
            a.record(stream)
            d.newton_solve(c_work, bt, 1.0, 0.5, 0.0, iters, info_t)       # tol = 0: exactly `iters` steps
            b.record(stream)
        barrier()
        ms = float(np.mean([a.elapsed_time(b) for a, b in evs]))
        taken = float(info_t[:, 0].min().item())
        solve = {"steps_per_solve": taken, "ms_per_solve": ms, "ms_per_newton_step": ms / max(taken, 1.0),
                 "newton_steps_per_s": world * nb * taken / (ms * 1e-3),
                 "how": f"dse_newton_solve(rho=1, step_cap=0.5, tol=0, max_iter={iters}): CUDA graph with a WHILE node, "
                        "no host round trip between steps; mean of 50 solves, L2 flushed before each"}

        # config 2': the paper's own parameter set, which does converge (A17): iterations, total time, the
        # infrared exponents and the coupling, all read on the device (dse_newton_solve + dse_dressing)
        from workloads import paper_scaling_workload, scaling_start_coefficients, PAPER_SCALING_BC
        ws = paper_scaling_workload()
        d2 = Dse(params_from_workload(ws, flags=flags & ~DSE_FLAG_CONST_COEF))
        c0 = torch.from_numpy(scaling_start_coefficients(ws)[None, :]).cuda()
        bc2 = torch.tensor([PAPER_SCALING_BC], dtype=torch.float64, device="cuda")
        cw2 = c0.clone()
        info2 = torch.empty((1, 6), dtype=torch.float64, device="cuda")
        for _ in range(3):
            cw2.copy_(c0)
            d2.newton_solve(cw2, bc2, 1.0, 0.5, 1e-11, 30, info2)
        barrier()
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(20)]
        for a, b in evs:
            flush.zero_()
            cw2.copy_(c0)
            a.record(stream)
            d2.newton_solve(cw2, bc2, 1.0, 0.5, 1e-11, 30, info2)
            b.record(stream)
        barrier()
        hh = 1.02
        xs = torch.tensor([91.2 ** 2, ws.eps2, 3e-6 * hh, 3e-6 / hh], dtype=torch.float64, device="cuda")
        lnG, lnZ, al = (t.cpu().numpy()[0] for t in d2.dressing(cw2, xs))
        i2 = info2.cpu().numpy()[0]
        solve["converged_solve"] = {
            "workload": "config 2' = the paper's parameter set (L135, L364): N=36, 96+32 radial x 32 angular nodes, x_G=0, "
                        "1/G(0)=0, Z(L2)=0.256, start guess from eq.(16)-(19), step_cap=0.5, tol=1e-11",
            "iterations": int(i2[0]), "status": int(i2[5]), "last_delta_inf": float(i2[1]),
            "ms_total": float(np.mean([a.elapsed_time(b) for a, b in evs])),
            "alpha_MZ2": float(al[0]), "alpha_eps2": float(al[1]),
            "ir_slope_lnG": float((lnG[2] - lnG[3]) / (2 * np.log(hh))), "ir_slope_lnZ": float((lnZ[2] - lnZ[3]) / (2 * np.log(hh))),
            "paper": {"alpha_MZ2": 0.118, "alpha_0": 2.972, "kappa": 0.595353}}
        d2.close()

    info = d.kernel_info()
    line = None
    if rank == 0:
        flops = algorithmic_flops(w, nb)
        k_ms = kernel_ms / max(kernel_n, 1)
        achieved = flops / (k_ms * 1e-3) / 1e12
        traffic, traffic_source = None, None
        tpath = os.path.join(ROOT, "profiles", "point_kernel_traffic.txt")
        if os.path.exists(tpath) and args.geometry_cache:
            try:
                rec = json.load(open(tpath)).get(w.name)      # {"bytes": ..., "source": "..."}: an ncu capture, NOT this run
                if rec:
                    traffic, traffic_source = rec["bytes"], rec["source"]
            except Exception:
                pass
        one_kernel = info.get("kernels_per_build") == 1
        line = {
            "metric": "fp64 Newton steps/s (build + LU)" if newton else "fp64 Jacobian builds/s", "value": value,
            "unit": "newton_steps/s" if newton else "jacobian_builds/s", "n_gpus": world,
            "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n_cheb": w.n_cheb, "n_r": w.n_r, "n_theta": w.n_theta, "n_batch": nb,
                       "eps2": w.eps2, "L2": w.L2, "points_per_build": w.points * nb,
                       "geometry_cache": bool(args.geometry_cache), "const_coef": bool(flags & DSE_FLAG_CONST_COEF),
                       "l2": "flushed between steps (256 MiB memset outside the per-step event pairs)",
                       "parallelism": f"replicas x{world}" if world > 1 else "single GPU",
                       "point_kernel": info},
            "points_per_s": value * w.points, "paper_equiv_evals_per_s": value * w.paper_equiv_evals,
            "wall_s_timed_region": t_wall,
            "roofline": {"bound": "alu", "kernel": "point_kernel" + (" (the whole build: H1-H8 in one launch)" if one_kernel else ""),
                         "achieved": achieved, "peak": FP64_PEAK_TFLOPS,
                         "unit": "TFLOP/s", "frac": achieved / FP64_PEAK_TFLOPS, "traffic": traffic, "traffic_source": traffic_source,
                         "kernel_ms": k_ms, "kernel_share_of_step": k_ms / (inst_total_ms / args.steps),
                         "ms_per_step_instrumented": inst_total_ms / args.steps,
                         "peak_source": "derived: 148 SM x 64 fp64 FMA/clk x 2 x 1.965 GHz (MEASURED_PEAKS.json has no "
                                        "fp64 entry); measured sustained DFMA rate beside it: peak_measured_sustained",
                         "algorithmic_flops_per_launch": flops},
            "e2e": {"value": e2e_value, "unit": "newton_steps/s" if newton else "jacobian_builds/s",
                    "h2d_bytes_per_step": int(c.nbytes + bc.nbytes), "d2h_bytes_per_step": e2e_d2h, "steps": e2e_steps},
            "gpu_launches": int(launches),
            "clocks": sampler.result(),
        }
        if with_update is not None:
            line["with_newton_update"] = with_update
        if solve is not None:
            line["newton_solve"] = solve
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(w, c[0])
            if newton:
                line["cpu_baseline"]["converged_solve"] = oracle_converged_solve()
    d.close()
    return line


def sustained_fp64_probe(local, seconds=1.2):
    """the roofline denominator of an ALU-bound path, measured: >= 1 s of back-to-back DFMA launches (8
    independent chains per thread, 148 x 8 CTAs of 256 threads), SM clock sampled during the run."""
    import torch
    from paper_1206_1779_b200.binding import probe
    sink = torch.empty(148 * 8 * 256, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    probe("dfma", 148 * 8, 2000, sink)
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    sampler.start()
    iters, evs, t0 = 400000, [], time.perf_counter()          # ~54 ms per launch
    while time.perf_counter() - t0 < seconds or len(evs) < 4:
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        fl = probe("dfma", 148 * 8, iters, sink)
        b.record(stream)
        evs.append((a, b, fl))
        torch.cuda.synchronize()
    sampler.stop_flag = True
    tf = [fl / (a.elapsed_time(b) * 1e-3) / 1e12 for a, b, fl in evs]
    out = {"tflops_sustained": float(np.median(tf[len(tf) // 2:])), "tflops_first_launch": tf[0], "seconds": time.perf_counter() - t0,
           "launches": len(tf), "clocks": sampler.result()}
    # the fp64 tensor path (mma.sync.m8n8k4.f64), the denominator for the batched kernel (config 4)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    probe("dmma", 148 * 8, 2000, sink)
    a.record(stream)
    fl = probe("dmma", 148 * 8, 100000, sink)
    b.record(stream)
    torch.cuda.synchronize()
    out["dmma_tflops"] = fl / (a.elapsed_time(b) * 1e-3) / 1e12
    return out


def run_probes():
    """--probes: the fp64 micro-measurements DESIGN.md section 6 refers to (include/dse_diag.h), one JSON line each."""
    import torch
    from paper_1206_1779_b200.binding import probe, PROBE_KINDS
    torch.cuda.set_device(0)
    sink = torch.empty(148 * 8 * 256, dtype=torch.float64, device="cuda")
    s = torch.cuda.current_stream()
    for kind in PROBE_KINDS:
        for blocks in (148 * 8, 148 * 2):
            probe(kind, blocks, 2000, sink)
            torch.cuda.synchronize()
            res = []
            for _ in range(5):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(s)
                fl = probe(kind, blocks, 100000, sink)
                b.record(s)
                torch.cuda.synchronize()
                res.append(fl / (a.elapsed_time(b) * 1e-3) / 1e12)
            print(json.dumps({"probe": kind, "ctas": blocks, "warps_per_sm": blocks * 8 // 148,
                              "tflops_median": round(float(np.median(res)), 2), "tflops_min": round(min(res), 2),
                              "tflops_max": round(max(res), 2)}), flush=True)
    from paper_1206_1779_b200.binding import LATENCY_PROBE_KINDS
    for kind in LATENCY_PROBE_KINDS:              # one warp, dependent chain: cycles per iteration land in sink[0]
        res = []
        for _ in range(3):
            probe(kind, 1, 4096, sink)
            torch.cuda.synchronize()
            res.append(float(sink[0].item()))
        print(json.dumps({"probe": kind, "cycles_per_dependent_iteration": round(float(np.median(res)), 1)}), flush=True)


def run_phase_timeline():
    """--phase-timeline: the tables of DESIGN.md section 6 from the phase stamps of a library built with
    -DDSE_PHASE_TIMING (include/dse_diag.h: dse_diag_phase_stamps).  Config 1 and config 3 builds with the L2 flushed;
    the one-CTA LU at n = 32, 64, 128."""
    import torch
    from paper_1206_1779_b200 import Dse, params_from_workload, DSE_FLAG_GEOMETRY_CACHE, DSE_FLAG_CONST_COEF
    from paper_1206_1779_b200.binding import phase_stamps
    torch.cuda.set_device(0)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    for cfg in (1, 3):
        w, c, bc = config_inputs(cfg)
        d = Dse(params_from_workload(w, flags=DSE_FLAG_GEOMETRY_CACHE | DSE_FLAG_CONST_COEF))
        info = d.kernel_info()
        ct, bt = torch.from_numpy(c).cuda(), torch.from_numpy(bc).cuda()
        for _ in range(3):
            d.jacobian(ct, bt)
        flush.zero_()
        torch.cuda.synchronize()
        d.jacobian(ct, bt)
        torch.cuda.synchronize()
        a = phase_stamps(0).reshape(148, 16, 16).astype(np.float64)[:info["grid"], :info["block"] // 32, :]
        t0 = a[:, :, 0].min()
        print(f"## {w.name}: grid {info['grid']} x {info['block']} threads, us after the first CTA starts (min / mean / max over warps or owners)")

        def row(name, x):
            print("| %s | %.2f | %.2f | %.2f |" % (name, x.min() / 1e3, x.mean() / 1e3, x.max() / 1e3))
        print("| phase | min | mean | max |\n|---|---|---|---|")
        row("table requests issued", a[:, :, 1] - t0)
        row("H1 done, first barrier passed", a[:, :, 2] - t0)
        row("batches + segment ends (duration)", a[:, :, 3] - a[:, :, 2])
        row("... of which flush + H7 (duration)", a[:, :, 9])
        row("point phase ends", a[:, :, 3] - t0)
        row("arrival counters done", a[:, :, 5] - t0)
        for slot, name in ((6, "slot sums + derivative rows written (owners)"), (11, "subtraction rows seen (owners)"),
                           (13, "rows of J, F written (owners)"), (8, "counters cleared (finishing CTA)")):
            m = a[:, :, slot] > 0
            if m.any():
                row(name, (a[:, :, slot] - t0)[m])
        row("kernel exit", a[:, :, 7] - t0)
        d.close()
    d = Dse(params_from_workload(CONFIGS[0]))
    rng = np.random.default_rng(5)
    print("## lu_panel_kernel, clock64 cycles of system 0 (warm, back-to-back solves)")
    print("| n | columns per panel | load + equilibrate | elimination | back substitution | per panel: read record | apply to own columns | factorise + publish | hand-over to the next owner |\n|---|---|---|---|---|---|---|---|---|")
    for n in (32, 64, 128):
        A = torch.from_numpy(rng.normal(size=(1, n, n))).cuda()
        b = torch.from_numpy(rng.normal(size=(1, n))).cuda()
        for _ in range(5):
            d.lu_solve(A, b)
        torch.cuda.synchronize()
        s = phase_stamps(1)
        B = lambda P, k: s[256 + P * 8 + k]
        pb = 2 if n > 96 else 4                             # panel widths of csrc/dse_lu.cu
        r = np.array([(B(P, 1) - B(P, 0), B(P, 2) - B(P, 1), B(P, 3) - B(P, 2), B(P + 1, 0) - B(P, 3)) for P in range(1, n // pb - 2)])
        m = r.mean(axis=0)
        print("| %d | %d | %d | %d | %d | %.0f | %.0f | %.0f | %.0f |" % (n, pb, s[1] - s[0], s[2] - s[1], s[4] - s[3], *m))
    d.close()


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    env = {"rank": rank, "world": world, "local": local,
           "flush": torch.empty(256 << 20, dtype=torch.uint8, device="cuda")}      # > 126 MB L2
    line = measure(args, args.config, args.steps, args.warmup, args.geometry_cache, env)
    if rank == 0:
        peak = sustained_fp64_probe(local)
        r = line["roofline"]
        r["peak_measured_sustained"] = peak["tflops_sustained"]
        r["peak_measured"] = peak
        r["frac_of_measured"] = r["achieved"] / peak["tflops_sustained"]
        if line["config"]["n_batch"] >= 8:
            r["frac_of_measured_dmma"] = r["achieved"] / peak["dmma_tflops"]
    # one driver run covers all five configs north_star names (+ config 3 with the geometry computed in registers)
    if world == 1 and args.per_config and args.config == 3:
        per = {}
        keep = ("value", "unit", "ms_per_step", "e2e", "gpu_launches", "with_newton_update", "newton_solve", "points_per_s")
        for name, cid, geom in (("cfg0", 0, 1), ("cfg1", 1, 1), ("cfg2", 2, 1), ("cfg4", 4, 1), ("cfg3_on_the_fly", 3, 0)):
            l2 = measure(args, cid, args.per_config_steps, 5, geom, env, light=True)
            e = {k: l2[k] for k in keep if k in l2}
            e["workload"] = l2["config"]["workload"]; e["geometry_cache"] = bool(geom)
            e["kernel_ms"] = l2["roofline"]["kernel_ms"]; e["kernel_share_of_step"] = l2["roofline"]["kernel_share_of_step"]
            e["achieved_tflops"] = l2["roofline"]["achieved"]; e["frac"] = l2["roofline"]["frac"]
            e["frac_of_measured"] = l2["roofline"]["achieved"] / peak["tflops_sustained"]
            if cid == 4:
                e["frac_of_measured_dmma"] = l2["roofline"]["achieved"] / peak["dmma_tflops"]
            e["point_kernel"] = l2["config"]["point_kernel"]; e["steps"] = l2["steps"]
            per[name] = e
        line["per_config"] = per
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=3, choices=sorted(CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--geometry-cache", type=int, default=1,
                    help="1: coefficient-independent per-point factors are tabulated once in dse_create (default); "
                         "0: recomputed inside every build")
    ap.add_argument("--const-coef", type=int, default=1,
                    help="1: single-system builds ask for the constant-bank coefficient slot (DSE_FLAG_CONST_COEF)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--per-config", type=int, default=1,
                    help="1 (default run, config 3 only): add the key per_config with a short run of configs 0, 1, 2, 4 and of "
                         "config 3 without the geometry cache")
    ap.add_argument("--per-config-steps", type=int, default=300)
    ap.add_argument("--probes", action="store_true", help="print the fp64 throughput probes (include/dse_diag.h) and exit")
    ap.add_argument("--phase-timeline", action="store_true",
                    help="print the phase timelines of the one-kernel build and of the LU (needs a library built with -DDSE_PHASE_TIMING) and exit")
    args = ap.parse_args()
    if args.probes:
        run_probes()
        return
    if args.phase_timeline:
        run_phase_timeline()
        return
    if args.impl == "reference":
        w, c, bc = config_inputs(args.config)
        run_reference(args, w, c)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
