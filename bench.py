#!/usr/bin/env python
"""bench.py -- PM steps/s and particle-updates/s of the FastPM force-and-update step on B200.

Contract (see the task statement): `python bench.py --gpus N --steps K --warmup W` prints ONE JSON
line on rank 0.  A "step" is one PM step of the whole hot path (paint -> r2c -> transfer function ->
3x c2r -> readout -> kick -> drift) over all particles of the workload,
executed by libfpm's fpm_pm_step (the loop body of fpm_nbody).  The workload is BASELINE.json's
C4: 512^3 particles on a 512^3 mesh, 2LPT ICs at a = 0.1 (made by fpm_lpt_init from a seeded
Eisenstein-Hu Gaussian field), stepped along C4's 40-step schedule so the particle distribution
is the real, progressively clustered one.  Multi-GPU: replicas only -- each
rank runs an independent simulation (seed + rank), no collective on the data path.

`--impl reference` times the float64 CPU oracle (oracle/, test infrastructure) on the host cores
on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import fpm_inputs as fi  # noqa: E402

METRIC = "PM steps/sec at 512^3 (particle-updates/sec = value x 512^3)"
FALLBACK_HBM_GBS = 6650.0


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def algorithmic_bytes(n_p, ng):
    """Algorithmic HBM bytes per launch of each kernel."""
    n_g = ng ** 3
    n_k = ng * ng * (ng // 2 + 1)
    return {
        "paint": 12 * n_p + 4 * n_g,
        "fft_z_r2c": 4 * n_g + 8 * n_k,
        "fft_cols_y": 16 * n_k,
        "fft_cols_x": 16 * n_k,
        "fft_z_c2r": 8 * n_k + 4 * n_g,
        "fft_z_c2r3": 24 * n_k + 12 * n_g,      # fused path: 3 components, interleaved output (pad not credited)
        "apply_force_kernel": 32 * n_k,
        "fft_x_force": 24 * n_k,
        "fft_y_inv3": 40 * n_k,
        "readout_kick_drift": 48 * n_p + 12 * n_g,
        "readout": 24 * n_p + 12 * n_g,
        "kick": 36 * n_p,
        "drift": 36 * n_p,
    }


def ncu_traffic(config):
    """{kernel: dram__bytes_read.sum + dram__bytes_write.sum per launch} from profiles/ncu_traffic.csv
    (written from the `ncu --set full` capture named in its last column, e.g. profiles/r01_E_C4.md)."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    out, src = {}, {}
    if os.path.exists(path):
        with open(path) as f:
            next(f)
            for line in f:
                cfg, kernel, nbytes, capture = line.strip().split(",")
                if cfg == config:
                    out[kernel] = int(nbytes)
                    src[kernel] = capture
    return out, src


def step_bytes_unfused(n_p, ng):
    """SURVEY.md 8(d) unfused model: 96 n_p + 112 n_g bytes per PM step."""
    return 96 * n_p + 112 * ng ** 3


def step_bytes_fused_path(n_p, ng):
    """Compulsory bytes of the fused path as built: 60 n_p + 88 n_g = the sum of the seven
    kernels' algorithmic bytes + the 8 n_g of the interleaved force cell's pad (written and read, not credited
    per kernel)."""
    return 60 * n_p + 88 * ng ** 3


def step_bytes_useful(n_p, ng):
    """The fused path's bytes without the 4-byte pad of the 16-byte force cell (written once and read once per
    cell: 8 n_g of pure layout waste): 60 n_p + 80 n_g.  The headline step fraction credits only these."""
    return 60 * n_p + 80 * ng ** 3


def step_bytes_fused_bound(n_p, ng):
    """SURVEY.md 8(d) "fused lower bound": 60 n_p + 104 n_g."""
    return 60 * n_p + 104 * ng ** 3


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""
    QUERY = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap,power.draw")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.QUERY}",
                 "--format=csv,noheader,nounits", "-lms", "25"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.monotonic(), [c.strip() for c in line.split(",")]))

    def mark_begin(self):
        self.t_begin = time.monotonic()

    def mark_end(self):
        self.t_end = time.monotonic()

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        # samples taken while the timed region ran (nvidia-smi is started before the warm-up so that it is
        # already streaming); if the region was shorter than the sampling period, the nearest samples
        t0, t1 = getattr(self, "t_begin", None), getattr(self, "t_end", None)
        rows = [r for t, r in self.rows if t0 is None or (t0 <= t <= t1 + 0.05)]
        if len(rows) < 2 and t0 is not None:
            rows = [r for _, r in sorted(self.rows, key=lambda tr: abs(tr[0] - 0.5 * (t0 + t1)))[:3]]
        for r in rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0]))
                smax.append(float(r[1]))
                power.append(float(r[6]))
            except ValueError:
                continue
            for name, val in zip(names, r[2:6]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(smax) if smax else None,
                "reasons": sorted(reasons), "samples": len(sm),
                "power_w_max": max(power) if power else None}


def oracle_sample(cfg, n_side, n_steps, ng_side=None):
    """Times the float64 oracle on n_steps PM steps (paint, r2c, Eq. 3-5, 3 c2r, 3 readouts, kick, drift --
    each an oracle call, nothing tuned) of an n_side^3-particle slice of the workload with the workload's
    particle spacing and mesh resolution (n_side = np_side: the workload itself), from 1LPT ICs."""
    import oracle
    ng_side = n_side * cfg.resolution_factor if ng_side is None else ng_side
    box = cfg.box * n_side / cfg.np_side          # same particle spacing as the workload
    delta = fi.linear_field(n_side, box, cfg.seed).astype(np.float64)
    om = fi.COSMO["omega_m"]
    pos, mom = oracle.lpt_init(delta, ng_side, om, cfg.a0, 1)
    del delta
    stages = cfg.stages()
    mass = float(cfg.resolution_factor ** 3)
    times = []
    for j in range(n_steps):
        ai, af = stages[j], stages[j + 1]
        ah = (ai * af) ** 0.5
        t0 = time.perf_counter()
        f = oracle.force(pos, ng_side, scale=1.5 * om, mass=mass)
        mom = oracle.kick(mom, f, oracle.kick_factor(om, ai, ai, ah))
        pos = oracle.drift(pos, mom, oracle.drift_factor(om, ai, ah, af), ng_side)
        times.append(time.perf_counter() - t0)
    return times, oracle.num_threads()


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores, same metric, unit and workload.  One
    oracle PM step at 512^3 takes most of a minute, so the requested --steps / --warmup are CAPPED to what ends
    within a few minutes (default: 2 timed steps, no warm-up -- a CPU program has nothing to warm); the line
    says how many were really run, and `ms_per_step` is what was measured, not an extrapolation."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = fi.CONFIGS[args.config]
    n_side = cfg.np_side if args.ref_side is None else min(cfg.np_side, args.ref_side)
    cap = args.ref_max_steps
    steps, warmup = max(1, min(args.steps, cap)), min(args.warmup, max(0, cap - min(args.steps, cap)))
    times, cores = oracle_sample(cfg, n_side, steps + warmup)
    timed = times[warmup:]
    frac = (n_side / cfg.np_side) ** 3
    value = len(timed) / sum(timed) * frac        # steps/s of the workload (frac = 1: measured, not scaled)
    sample = (f"{len(timed)} PM steps (+{warmup} warm-up; requested --steps {args.steps} --warmup {args.warmup}, capped "
              f"to keep the run within minutes) of "
              + (f"the full workload {cfg.name}" if frac == 1.0 else
                 f"a {n_side}^3-particle slice of {cfg.name} (same particle spacing; steps/s scaled by {frac:g})")
              + ", float64 oracle, 1LPT ICs")
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "steps/s",
        "particle_updates_per_sec": value * cfg.n_particles, "n_gpus": args.gpus, "steps": len(timed),
        "warmup": warmup, "ms_per_step": 1e3 / value, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg), "sample": sample, "requested_steps": args.steps,
                   "requested_warmup": args.warmup, "ms_per_step_measured": [1e3 * t for t in timed]},
        "cpu_baseline": {"value": value, "unit": "steps/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)


def workload_name(cfg):
    return (f"{cfg.name}: {cfg.np_side}^3 particles on a {cfg.ng}^3 float32 mesh, box {cfg.box:g} Mpc/h, "
            f"{cfg.lpt_order}LPT ICs at a={cfg.a0}, {cfg.n_steps}-step FastPM schedule linear in a to a={cfg.a1}")


def side_measurements(args, ctx, cfg, pos, mom, factors, device):
    """Context numbers, N = 1 only, outside the timed region: (i) cuFFT (torch.fft, a library call) r2c +
    c2r on the same mesh size as the reference floor for the hand-written FFT passes -- never on the
    product path; (ii) one backward PM step (fpm_force_vjp at the current positions: recomputed force
    meshes, 3 adjoint paints, 3 r2c, transposed kernel, c2r, 2 gradient gathers -- C4's backward pass)."""
    import torch
    out = {}
    if args.no_side:
        return out
    ng, n_p = cfg.ng, cfg.n_particles

    def timed(fn, reps):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps

    try:
        x = torch.randn(ng, ng, ng, device=device)
        k = torch.fft.rfftn(x)
        ms_r2c = timed(lambda: torch.fft.rfftn(x), 5)
        ms_c2r = timed(lambda: torch.fft.irfftn(k, s=(ng, ng, ng)), 5)
        del x, k
        out["cufft_floor"] = {"r2c_ms": ms_r2c, "c2r_ms": ms_c2r, "one_r2c_three_c2r_ms": ms_r2c + 3 * ms_c2r,
                              "note": "torch.fft (cuFFT) on an ng^3 float32 mesh, timed alone as the reference "
                                      "floor for fft_z_r2c + fft_cols_y + fft_x_force + fft_y_inv3 + fft_z_c2r3; "
                                      "not on the product path"}
    except RuntimeError as e:      # noqa: BLE001  (cuFFT workspace may not fit beside a large config)
        out["cufft_floor"] = {"unavailable": str(e)[:120]}
    torch.cuda.empty_cache()
    gx = torch.zeros(3, n_p, device=device)
    v = mom.clone()
    ms_bwd = timed(lambda: ctx.force_vjp(pos, v, coef=factors[0], grad_pos=gx), 3)
    out["backward_step"] = {"ms": ms_bwd, "call": "fpm_force_vjp (one backward force evaluation of fpm_nbody_vjp)",
                            "steps_per_s": 1e3 / ms_bwd}
    del gx, v
    torch.cuda.empty_cache()
    # (iii) SURVEY.md 8(f) N1: one MAP-reconstruction iteration (loss + gradient through a 5-step 128^3 PM
    # forward model in a 400 Mpc/h box + Adam update), the configuration of PAPER.md:490-502.
    import paper_2010_11847_b200 as fpm
    n_r, box_r = 128, 400.0
    rctx = fpm.FPM(n_r, n_r, omega_m=fi.COSMO["omega_m"], box=box_r, device=device, force_path=fpm.FORCE_FUSED)
    stages = [0.1 + j * 0.9 / 5 for j in range(6)]
    truth = torch.from_numpy(fi.linear_field(n_r, box_r, 6)).to(device)
    p0, m0 = rctx.lpt_init(truth, stages[0], 2)
    rctx.nbody(p0, m0, stages)
    data = rctx.paint(p0) + torch.from_numpy(fi.noise_field(n_r, 1.0)).to(device)   # synthetic "observation"
    ipow = torch.from_numpy(fi.inverse_prior_power(n_r, box_r)).to(device)
    s = torch.zeros(n_r, n_r, n_r, device=device)
    am, av = torch.zeros_like(s), torch.zeros_like(s)
    state = {"t": 0, "loss": None}

    def iteration():
        state["t"] += 1
        loss, g = rctx.recon_loss_grad(s, data, 1.0, ipow, stages, 2)
        rctx.adam_step(s, g, am, av, 0.01, state["t"])
        state["loss"] = loss[0] + loss[1]

    iteration()
    first = state["loss"]
    ms_it = timed(iteration, 10)
    out["recon_iteration"] = {"ms": ms_it, "config": "5-step 128^3 PM forward model, 400 Mpc/h box, 2LPT ICs, loss + "
                              "gradient (fpm_recon_loss_grad) + Adam (fpm_adam_step)", "loss_first": first,
                              "loss_after_11_iterations": state["loss"],
                              "paper_context": "1.1 s/iteration on one V100, 4.6 s on 128 Haswell cores (PAPER.md:502)"}
    rctx.close()
    del truth, p0, m0, data, ipow, s, am, av
    torch.cuda.empty_cache()
    # (iv) SURVEY.md 8(f) N2: batched small simulations.  B independent C1 / C2 runs advance
    # in the same kernel launches and the whole run replays as one CUDA graph; compared with ONE simulation
    # run kernel by kernel (round 1's path) and with one simulation replayed as a graph.
    peak, _ = measured_peaks()
    out["batched_small_sims"] = {}
    for name, batch in (("C1", 64), ("C2", 16)):
        c = fi.CONFIGS[name]
        n_ev = c.n_steps + 1

        def run_rate(b, graph_mode, reps):
            bctx = fpm.FPM(c.ng, c.np_side, omega_m=fi.COSMO["omega_m"], box=c.box, device=device,
                           force_path=fpm.FORCE_FUSED, batch=b)
            bctx.set_graph_mode(graph_mode)
            fields = np.stack([fi.linear_field(c.np_side, c.box, c.seed + i) for i in range(b)])
            d = torch.from_numpy(fields if b > 1 else fields[0]).to(device)
            q0, r0 = bctx.lpt_init(d, c.a0, c.lpt_order)
            q, r = q0.clone(), r0.clone()
            for _ in range(2):                                # warm-up: FPM_GRAPH_AUTO captures a run the second
                q.copy_(q0)                                   # time the same argument set comes in
                r.copy_(r0)
                bctx.nbody(q, r, c.stages())
            torch.cuda.synchronize()
            total = 0.0
            for _ in range(reps):
                q.copy_(q0)
                r.copy_(r0)
                a, z = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record()
                bctx.nbody(q, r, c.stages())
                z.record()
                torch.cuda.synchronize()
                total += a.elapsed_time(z)
            bctx.close()
            return b * n_ev * reps * 1e3 / total, total / reps

        one_eager, _ = run_rate(1, fpm.GRAPH_OFF, 20)
        one_graph, _ = run_rate(1, fpm.GRAPH_ALWAYS, 20)
        many, ms_run = run_rate(batch, fpm.GRAPH_AUTO, 10)
        step_bytes = batch * step_bytes_fused_path(c.n_particles, c.ng)
        out["batched_small_sims"][f"{batch}x{name}"] = {
            "call": "fpm_nbody on a batch context (one CUDA graph launch per run)",
            "pm_steps_per_s_aggregate": many, "particle_updates_per_s": many * c.n_particles,
            "ms_per_run": ms_run, "force_evaluations_per_run": n_ev,
            "step_roofline_frac": step_bytes * n_ev / (ms_run * 1e-3) / 1e9 / peak,
            "one_sim_kernel_by_kernel_steps_per_s": one_eager, "one_sim_graph_steps_per_s": one_graph,
            "speedup_vs_one_sim_kernel_by_kernel": many / one_eager}
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="timed PM steps (default: the rest of the schedule)")
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C4", choices=sorted(fi.CONFIGS))
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-side", action="store_true", help="skip the cuFFT floor, whole-run, backward and N1/N2 timings")
    ap.add_argument("--ref-side", type=int, default=None, help="--impl reference: run a slice of this many particles per side")
    ap.add_argument("--ref-max-steps", type=int, default=2, help="--impl reference: cap on steps + warm-up really run")
    ap.add_argument("--force-path", default="fused", choices=["fused", "unfused"])
    args = ap.parse_args()
    cfg = fi.CONFIGS[args.config]
    n_sched = cfg.n_steps + 1          # PM steps (force evaluations) of the whole schedule
    if args.impl == "reference":
        args.steps = 20 if args.steps is None else args.steps
        run_reference(args)
        return
    args.warmup = max(args.warmup, 3)
    if args.steps is None:
        args.steps = n_sched - args.warmup
    if args.warmup + args.steps > n_sched or args.steps < 1:
        ap.error(f"--warmup {args.warmup} + --steps {args.steps} exceeds the {n_sched} PM steps of {cfg.name}'s schedule "
                 f"(the timed steps walk the real schedule; nothing is repeated)")

    from paper_2010_11847_b200 import replicas as rep
    if rep.needs_spawn(args.gpus):
        # `python bench.py --gpus N` outside torchrun: start the N replica ranks (one process per GPU)
        sys.exit(subprocess.call(rep.launch_command(args.gpus, os.path.abspath(__file__), sys.argv[1:])))

    import torch

    import paper_2010_11847_b200 as fpm   # raises if libfpm.so is missing: no fallback

    rank, local_rank, world = rep.env_world()
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    rep.init("nccl", device)

    n_p, ng = cfg.n_particles, cfg.ng
    ctx = fpm.FPM(ng, cfg.np_side, omega_m=fi.COSMO["omega_m"], box=cfg.box, device=device,
                  force_path=fpm.FORCE_FUSED if args.force_path == "fused" else fpm.FORCE_UNFUSED)

    # ---- inputs: seeded Gaussian field -> 2LPT particles, all resident in HBM -----------------
    delta = torch.from_numpy(fi.linear_field(cfg.np_side, cfg.box, rep.replica_seed(cfg.seed, rank))).to(device)
    pos, mom = ctx.lpt_init(delta, cfg.a0, cfg.lpt_order)
    stages = cfg.stages()
    factors = ctx.step_factors(stages)          # fpm_step_factors: the schedule arithmetic is behind the C-ABI

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    step_no = 0
    for _ in range(args.warmup):
        ctx.pm_step(pos, mom, *factors[step_no])
        step_no += 1
    torch.cuda.synchronize()
    rep.barrier()
    torch.cuda.synchronize()

    sampler.mark_begin()
    ctx.profile_reset()
    ctx.profile_enable(True)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    first_timed = step_no
    for _ in range(args.steps):
        ctx.pm_step(pos, mom, *factors[step_no])
        step_no += 1
    ev1.record()
    torch.cuda.synchronize()
    rep.barrier()
    torch.cuda.synchronize()
    sampler.mark_end()
    ms_total = ev0.elapsed_time(ev1)
    launches = ctx.launch_count()
    prof = ctx.profile_read()
    ctx.profile_enable(False)
    clocks = sampler.stop() if rank == 0 else None
    ms_total = rep.max_over_ranks(ms_total, device)
    ms_per_step = ms_total / args.steps
    value = rep.whole_job_rate(args.steps, ms_total, world)     # whole-job steps/s (replicas)

    # ---- end to end through the C-ABI with HOST buffers -----------------------------------------
    # (continues the schedule where it has steps left, else repeats its last full step: the state is the
    #  clustered end-of-run one either way, and this leg is dominated by the PCIe copies)
    e2e = None
    if args.e2e_steps > 0:
        def e2e_fac(i):
            return factors[min(i, n_sched - 2)]
        h_pos = torch.empty((3, n_p), dtype=torch.float32, pin_memory=True)
        h_mom = torch.empty((3, n_p), dtype=torch.float32, pin_memory=True)
        h_pos.copy_(pos)
        h_mom.copy_(mom)
        torch.cuda.synchronize()
        ctx.pm_step_host(h_pos, h_mom, pos, mom, *e2e_fac(step_no))   # warm-up
        step_no += 1
        rep.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.e2e_steps):
            ctx.pm_step_host(h_pos, h_mom, pos, mom, *e2e_fac(step_no))
            step_no += 1
        e1.record()
        torch.cuda.synchronize()
        e2e_ms = e0.elapsed_time(e1)
        e2e_ms = rep.max_over_ranks(e2e_ms, device)
        e2e = {"value": rep.whole_job_rate(args.e2e_steps, e2e_ms, world), "unit": "steps/s",
               "h2d_bytes_per_step": 24 * n_p, "d2h_bytes_per_step": 24 * n_p,
               "steps": args.e2e_steps,
               "call": "fpm_pm_step_host (pinned host pos+mom -> device, step, -> host)"}
        del h_pos, h_mom

    # ---- the whole run as ONE C call: fpm_nbody over every force evaluation of the schedule ------------
    whole_run = None
    if not args.no_side:
        pos2, mom2 = ctx.lpt_init(delta, cfg.a0, cfg.lpt_order)
        torch.cuda.synchronize()
        rep.barrier()
        w0, w1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        w0.record()
        ctx.nbody(pos2, mom2, stages)
        w1.record()
        torch.cuda.synchronize()
        ms_run = rep.max_over_ranks(w0.elapsed_time(w1), device)
        whole_run = {"call": "fpm_nbody (2LPT state -> a = 1), CUDA events around the one call",
                     "force_evaluations": n_sched, "ms": ms_run, "ms_per_step": ms_run / n_sched,
                     "steps_per_s": rep.whole_job_rate(n_sched, ms_run, world)}
        del pos2, mom2
    del delta

    extras = side_measurements(args, ctx, cfg, pos, mom, factors[min(step_no, n_sched - 2)], device) \
        if (rank == 0 and world == 1) else {}

    if rank != 0:
        rep.finalize()
        return

    # ---- per-kernel roofline from the live CUDA-event profile ------------------------------------
    peak, peak_src = measured_peaks()
    abytes = algorithmic_bytes(n_p, ng)
    kernels = {}
    for name, (ms, cnt) in prof.items():
        if cnt == 0:
            continue
        per = ms / cnt
        k = {"launches_per_step": cnt / args.steps, "ms_per_launch": per, "ms_per_step": ms / args.steps}
        if name in abytes:
            k["algorithmic_bytes"] = abytes[name]
            k["gbs"] = abytes[name] / per / 1e6
            k["frac"] = k["gbs"] / peak
        kernels[name] = k
    dominant = max(kernels, key=lambda n: kernels[n]["ms_per_step"])
    traffic_table, traffic_src = ncu_traffic(args.config)     # per-launch DRAM bytes from the committed ncu capture
    late_table, late_src = ncu_traffic(args.config + "-late")   # the same at the clustered end of the schedule
    traffic = traffic_table.get(dominant)
    for name, k in kernels.items():
        if name in traffic_table:
            k["ncu_dram_bytes"] = traffic_table[name]
    dk = kernels[dominant]
    roofline = {"bound": "hbm", "kernel": dominant, "achieved": dk.get("gbs"), "peak": peak,
                "unit": "GB/s", "frac": dk.get("frac"), "traffic": traffic, "peak_source": peak_src,
                "traffic_source": (f"profiles/ncu_traffic.csv, capture {traffic_src.get(dominant)} (an earlier ncu --set "
                                   f"full run of this command, not this run)") if traffic is not None else None,
                "traffic_late": late_table.get(dominant),
                "traffic_late_source": (f"profiles/ncu_traffic.csv, capture {late_src.get(dominant)}"
                                        if late_table.get(dominant) is not None else None),
                "share_of_step": dk["ms_per_step"] / ms_per_step}
    own, bound, unf = step_bytes_fused_path(n_p, ng), step_bytes_fused_bound(n_p, ng), step_bytes_unfused(n_p, ng)
    useful = step_bytes_useful(n_p, ng)
    fused = args.force_path == "fused"
    step_roofline = {"unit": "GB/s", "peak": peak,
                     "algorithmic_bytes_per_step": useful if fused else unf,
                     "achieved": (useful if fused else unf) / ms_per_step / 1e6,
                     "frac": (useful if fused else unf) / ms_per_step / 1e6 / peak,
                     "model": ("60 n_p + 80 n_g: the useful bytes of the fused path (DESIGN.md 6); the pad of the 16-byte "
                               "force cell is not credited" if fused else "96 n_p + 112 n_g (SURVEY.md 8(d), unfused)"),
                     "frac_as_built": own / ms_per_step / 1e6 / peak,
                     "as_built_bytes": own,
                     "as_built_model": "60 n_p + 88 n_g: useful bytes + 8 n_g of force-cell pad the path really moves",
                     "frac_vs_survey_fused_bound": bound / ms_per_step / 1e6 / peak,
                     "survey_fused_bound_bytes": bound,
                     "vs_unfused_model": {"bytes": unf, "frac": unf / ms_per_step / 1e6 / peak,
                                          "note": "bytes the fused path never moves; context only"}}

    # Scatter-add rate of paint (north_star: "atomic throughput for paint"): 8 deposits per particle,
    # from the live kernel time.  In the brick kernel a deposit inside the shared-memory window is one lane of an
    # ATOMS.ADD (8 n_p / 32 warp instructions), a particle outside it costs 8 global RED.ADD.F32, and the window is
    # flushed with RED.E.ADD.F32x4; the split between the two is in the ncu captures under profiles/, not measured here.
    paint_atomics = None
    if "paint" in kernels:
        pms = kernels["paint"]["ms_per_launch"]
        paint_atomics = {"scatter_adds_per_launch": 8 * n_p, "scatter_adds_per_s": 8 * n_p / pms * 1e3,
                         "shared_atoms_warp_instructions_per_launch": 8 * n_p // 32,
                         "shared_atoms_warp_instructions_per_s": 8 * n_p / 32 / pms * 1e3,
                         "ms_per_launch": pms,
                         "note": "counts are algorithmic (8 deposits per particle, all taken as in-window); the "
                                 "measured ATOMS / RED split per launch is in profiles/ (per-opcode tables)"}

    cpu_baseline = None
    if not args.no_cpu_baseline and world == 1:
        side = min(cfg.np_side, 256)
        times, cores = oracle_sample(cfg, side, 3)
        upd = side ** 3 * 2 / sum(times[1:])
        cpu_baseline = {"value": upd / n_p, "unit": "steps/s", "cores": cores, "kind": "oracle",
                        "particle_updates_per_sec": upd, "ms_per_sample_step": [1e3 * t for t in times[1:]],
                        "sample": f"2 PM steps (+1 warm-up) of a {side}^3-particle / {side * cfg.resolution_factor}^3-mesh "
                                  f"slice of {cfg.name} (same particle spacing), float64 oracle; steps/s scaled by "
                                  f"{side}^3/{cfg.np_side}^3 (`bench.py --impl reference` times the full-size step)"}

    out = {
        "metric": METRIC, "value": value, "unit": "steps/s",
        "particle_updates_per_sec": value * n_p,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_per_step,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": workload_name(cfg), "timed_schedule_steps": [first_timed, first_timed + args.steps - 1],
                   "schedule_pm_steps": n_sched,
                   "l2_policy": "inputs larger than L2 (3.2 GB particle state, 0.5 GB meshes vs 126 MB L2)",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "kernel_mode": "paper Eq. 4+5", "force_path": args.force_path,
                   "tile_movers": "tensor_maps" if ctx.tile_movers() == fpm.MOVERS_TENSOR_MAPS else "global"},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
        "roofline": roofline, "step_roofline": step_roofline, "kernels": kernels, "paint_atomics": paint_atomics,
        "whole_run": whole_run, "cpu_baseline": cpu_baseline,
    }
    out.update(extras)
    print(json.dumps(out), flush=True)
    rep.finalize()


if __name__ == "__main__":
    main()
