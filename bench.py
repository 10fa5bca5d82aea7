#!/usr/bin/env python
"""bench.py -- DOF-updates/s per Runge-Kutta stage of the fused DG Euler time step (fp64, B200).

One "step" = one LSERK45 time step = 5 passes of the whole hot path (flux, differentiation, traces,
Lax-Friedrichs flux, lift, 2/h scaling, stage update) over the whole mesh.  Default workload:
BASELINE.json config 3 (Taylor-Green vortex, 64^3 elements, p = 4, 32.8 M nodes), the configuration
the metric asks DOF-updates/s and HBM GB/s for; `--workload cfg5` runs the largest single-GPU case,
`--workload cfg4_p<k>` one point of the order sweep, and the default line also carries the whole
p = 1..7 sweep of config 4 ("p_sweep", skip with --no-sweep).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference]
    python -m torch.distributed.run --nproc-per-node N ... bench.py --gpus N ...   (N replicas)

Prints ONE JSON line (rank 0).  Timing: CUDA events on the stream the kernels are launched on,
after W >= 3 warm-up steps, barrier + synchronize on both sides, max over ranks.  The working set
(>= 2.6 GB per stage) is far larger than the 126 MB L2, so no flush is needed between iterations.

Besides the contract's keys the line carries: `sustained` (the same workload for >= 300 steps, i.e. under
the board's power cap), `cfg5` (the largest single-GPU case, 10 steps), `p_sweep` (config 4, p = 1..7),
`adaptive_dt` (dg_rk_step_cfl: CFL time step from the device-side max-wavespeed reduction every step),
`roofline` (HBM: 152 algorithmic bytes per DOF and stage against the measured copy bandwidth) and
`roofline_fp64` (algorithmic flops against the FP64 FMA rate measured by a microbenchmark in the same run).
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "DOF-updates/s per RK stage"
UNIT = "DOF-updates/s"
STAGES = 5
ALGO_BYTES_PER_DOF_STAGE = 152.0   # read Q,K + write Q,K = 4 x 40 B, stage 1 does not read K;
                                   # the kernel also skips the dead K store of stage 5 and moves 144
MOVED_BYTES_PER_DOF_STAGE = 144.0  # what this implementation has to move: `roofline.frac_moved` (frac credits 152)


def algo_flops_per_dof(p):
    """Algorithmic flops per DOF and stage: 178 + 30 N + 225 / N (volume 38 + 30 N from
    PAPER.md:135, traces 60, lift 60, 3 N^2 unique face nodes x 75, Runge-Kutta 20)."""
    N = p + 1
    return 178.0 + 30.0 * N + 225.0 / N
GAMMA = 1.4


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(workload):
    """Per-launch DRAM bytes of the stage kernel from the committed ncu --set full capture, or None."""
    path = os.path.join(ROOT, "profiles", "ncu_traffic.json")
    if os.path.exists(path):
        with open(path) as f:
            entry = json.load(f).get(workload)
        if entry:
            return entry
    return None


class ClockSampler:
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index):
        self.samples, self.power, self.reasons, self.max_mhz, self.power_limit = [], [], set(), None, None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.power_limit = pynvml.nvmlDeviceGetEnforcedPowerLimit(self.h) / 1000.0
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                 "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                 "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                 "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
                bits = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, v in names.items():
                    if bits & v:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.02)

    def __enter__(self):
        if self.nv:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thread:
            self._thread.join()

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}
        s = sorted(self.samples)
        pw = sorted(self.power)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s), "power_w": pw[len(pw) // 2] if pw else None, "power_limit_w": self.power_limit}


def physical_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ----------------------------------------------------------------------------------------------
# the oracle on the host cores: cpu_baseline leg and --impl reference
# ----------------------------------------------------------------------------------------------
def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_sample(workload, target_seconds=10.0, fixed_steps=None, build="omp", nodes=4.0e5):
    """Time the CPU oracle (as it stands: an unoptimised checker, NOT a tuned CPU DG code) on a bounded sample of
    the workload: the workload's own field formula and extent on a reduced periodic mesh of about `nodes` nodes
    (out of cache), so the sample is smooth and exactly periodic like the workload itself."""
    import numpy as np
    from oracle import Oracle
    from paper_2006_15698_b200 import inputs as I
    c = dict(I.CONFIGS[workload])
    p, ext = c["p"], c["extent"]
    ne = max(2, min(c["nx"], int(round((nodes / (p + 1) ** 3) ** (1.0 / 3.0)))))
    c.update(nx=ne, ny=ne, nz=ne)
    q = I.make_field(c)
    orc = Oracle(build)
    dt = I.cfl_dt(orc.max_wavespeed(q, p, GAMMA), p, ext, (ne, ne, ne), 0.1)
    dof = ne ** 3 * (p + 1) ** 3
    t0 = time.perf_counter()
    orc.rk_step(q, p, GAMMA, ext, dt, 1)
    t1 = time.perf_counter() - t0
    steps = fixed_steps if fixed_steps is not None else max(1, min(50, int(round(target_seconds / max(t1, 1e-6)))))
    t0 = time.perf_counter()
    out = orc.rk_step(q, p, GAMMA, ext, dt, steps)
    t = time.perf_counter() - t0
    return {"value": dof * STAGES * steps / t, "unit": UNIT, "cores": orc.threads, "kind": "oracle",
            "sample": f"{workload}'s field on a reduced periodic {ne}^3-element mesh (p={p}, {dof} nodes), {steps} LSERK45 "
                      f"steps, oracle/dg_oracle.c ({'OpenMP over elements' if 'omp' in build else 'single thread'}), {t:.1f} s; "
                      "the oracle is a plain checker, not a tuned CPU DG code",
            "seconds_per_step": t / steps, "dof": dof, "finite": bool(np.isfinite(out).all()), "cpu_model": cpu_model()}


def oracle_per_p():
    """SURVEY.md 8(d) "oracle timing": per p = 1..7 (config 4's field), single thread and OpenMP, bounded."""
    rows = []
    for p in range(1, 8):
        one = oracle_sample(f"cfg4_p{p}", fixed_steps=1, build="fp64", nodes=2.0e5)
        omp = oracle_sample(f"cfg4_p{p}", fixed_steps=2, build="omp", nodes=4.0e5)
        rows.append({"p": p, "single_thread": one["value"], "omp": omp["value"], "omp_threads": omp["cores"],
                     "dof_single": one["dof"], "dof_omp": omp["dof"]})
    return rows


def run_reference(args, rank):
    if rank != 0:
        return
    K, W = args.steps, args.warmup
    samp = oracle_sample(args.workload, fixed_steps=max(1, W))     # warm-up
    samp = oracle_sample(args.workload, fixed_steps=K)
    line = {"impl": "reference", "metric": METRIC, "value": samp["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": K, "warmup": W, "ms_per_step": 1e3 * samp["seconds_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{args.workload} (bounded sample: {samp['sample']})"},
            "cpu_baseline": {k: samp[k] for k in ("value", "unit", "cores", "kind", "sample", "finite", "cpu_model")},
            "e2e": {"value": samp["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------
# the CUDA path
# ----------------------------------------------------------------------------------------------
def time_workload(workload, K, W, device, dist, sampler_index=None, want_e2e=False, variant=None, lz=0):
    import torch
    from paper_2006_15698_b200 import DG
    from paper_2006_15698_b200 import inputs as I
    c = I.CONFIGS[workload]
    p, ext, n = c["p"], c["extent"], (c["nx"], c["ny"], c["nz"])
    q = I.make_field(workload, xp=torch, device=device)
    dg = DG(*n, p, GAMMA, ext, device=device, variant=variant, brick=(0, 0, lz) if lz else None)
    dg.set_state(q)
    dt = I.cfl_dt(dg.max_wavespeed(), p, ext, n, 0.1)
    dof = n[0] * n[1] * n[2] * (p + 1) ** 3
    stream = torch.cuda.current_stream(device)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(device)

    dg.rk_step(dt, W)
    barrier()
    l0 = dg.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(sampler_index) if sampler_index is not None else None
    if sampler:
        sampler.__enter__()
    e0.record(stream)
    dg.rk_step(dt, K)
    e1.record(stream)
    barrier()
    if sampler:
        sampler.__exit__()
    ms = e0.elapsed_time(e1)
    launches = dg.launch_count - l0
    finite = bool(torch.isfinite(dg.get_state(q)).all().item())
    out = {"workload": workload, "p": p, "elements": list(n), "dof": dof, "ms": ms, "launches": launches,
           "dt": dt, "finite": finite, "kernel": dg.kernel_info(),
           "clocks": sampler.summary() if sampler else None}

    if want_e2e:
        # second device-timed number: the max-wavespeed reduction (CFL time step) executed before every step
        # same protocol for both: CUDA events around blocks of 15 steps, fixed and adaptive alternating (3 blocks
        # each) after 30 more warm-up steps, so that both legs see the same clocks (the board is at its power cap)
        steps_a = 45
        dg.rk_step_cfl(0.1, 2)
        dg.rk_step(dt, 30)
        barrier()
        t_fixed = t_cfl = 0.0
        for _ in range(3):
            ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
            ev[0].record(stream)
            dg.rk_step(dt, 15)
            ev[1].record(stream)
            dg.rk_step_cfl(0.1, 15)       # dt formed on the device from the wavespeed the last stage reduced
            ev[2].record(stream)
            torch.cuda.synchronize(device)
            t_fixed += ev[0].elapsed_time(ev[1]) * 1e-3
            t_cfl += ev[1].elapsed_time(ev[2]) * 1e-3
        out["adaptive_dt"] = {"seconds": t_cfl, "steps": steps_a, "fixed_seconds": t_fixed}
        # end to end through the public API with HOST buffers: every step copies the state in from
        # pinned host memory, advances one LSERK45 step and copies the result back.
        steps = min(K, 10)
        host_in = torch.empty(q.shape, dtype=torch.float64, pin_memory=True)
        host_out = torch.empty(q.shape, dtype=torch.float64, pin_memory=True)
        dg.get_state(host_in)
        for _ in range(2):
            dg.set_state(host_in)
            dg.rk_step(dt, 1)
            dg.get_state(host_out)
        barrier()
        t0 = time.perf_counter()
        for _ in range(steps):
            dg.set_state(host_in)
            dg.rk_step(dt, 1)
            dg.get_state(host_out)            # synchronises
        torch.cuda.synchronize(device)
        t = time.perf_counter() - t0
        out["e2e"] = {"seconds": t, "steps": steps, "bytes_each_way": q.numel() * 8}
        del host_in, host_out
    dg.close()
    del q
    torch.cuda.empty_cache()
    return out


def per_kernel_breakdown(workload, steps, device):
    """the paper's Table II layout for this implementation: volume, surface and
    update-project kernels launched one by one (dg_split_*), each timed with CUDA events on the launching stream, next
    to the fused step on the same state.  Flop counts per DOF and evaluation: volume 38 + 30 N,
    surface 120 + 225 / N (traces, Lax-Friedrichs at 3 N^2 unique face nodes, lift: SURVEY.md 8(d)), update 20."""
    import torch
    from paper_2006_15698_b200 import DG
    from paper_2006_15698_b200 import inputs as I
    c = I.CONFIGS[workload]
    p, ext, n = c["p"], c["extent"], (c["nx"], c["ny"], c["nz"])
    N = p + 1
    q = I.make_field(workload, xp=torch, device=device)
    dg = DG(*n, p, GAMMA, ext, device=device)
    dg.set_state(q)
    dt = I.cfl_dt(dg.max_wavespeed(), p, ext, n, 0.1)
    dof = n[0] * n[1] * n[2] * N ** 3
    stream = torch.cuda.current_stream(device)
    dg.rk_step_split(dt, 2)
    torch.cuda.synchronize(device)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(steps * STAGES)]
    l0 = dg.launch_count
    for s in range(steps * STAGES):
        ev[s][0].record(stream)
        dg.split_volume()
        ev[s][1].record(stream)
        dg.split_surface()
        ev[s][2].record(stream)
        dg.split_update(dt, s % STAGES)
        ev[s][3].record(stream)
    torch.cuda.synchronize(device)
    launches = dg.launch_count - l0
    t = [sum(e[i].elapsed_time(e[i + 1]) for e in ev) * 1e-3 for i in range(3)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    dg.rk_step(dt, 2)
    e0.record(stream)
    dg.rk_step(dt, steps)
    e1.record(stream)
    torch.cuda.synchronize(device)
    fused = e0.elapsed_time(e1) * 1e-3
    finite = bool(torch.isfinite(dg.get_state(q)).all().item())
    dg.close()
    del q
    torch.cuda.empty_cache()
    evals = steps * STAGES
    flop = {"volume": 38.0 + 30.0 * N, "surface": 120.0 + 225.0 / N, "update_project": 20.0}
    rows = {}
    for name, sec in zip(("volume", "surface", "update_project"), t):
        rows[name] = {"seconds": sec, "dof_per_s": dof * evals / sec, "tflops": flop[name] * dof * evals / sec / 1e12,
                      "flop_per_dof": flop[name]}
    total = sum(t)
    return {"workload": f"{workload}: {list(n)} elements, p={p}, {dof} nodes", "steps": steps, "kernels": rows,
            "split_total_seconds": total, "split_dof_updates_per_s": dof * evals / total,
            "fused_seconds": fused, "fused_dof_updates_per_s": dof * evals / fused, "launches": launches, "finite": finite,
            "note": "update_project = K, Q update over the whole vectors + the face-trace kernel; the surface kernel evaluates "
                    "every face from both sides; flop rates use the algorithmic counts of PAPER.md:135 / SURVEY.md 8(d); "
                    "the paper's own per-V100 rates (Table II) are in BASELINE.md"}


VISC_BYTES_PER_DOF = 360.0   # viscous path, per evaluation: gradient + flux sweep (read Q 40, write Fv_x,y,z 120), divergence
                             # sweep (read Fv 120, read + write R 80); DESIGN.md 6.6


def navier_stokes_leg(workload, steps, device, mu=1e-3, prandtl=0.72):
    """LSERK45 steps of dQ/dt = L(Q) + div Fv (dg_rk_step_ns: per-kernel mode + the two viscous
    sweeps), timed with CUDA events on the launching stream; the viscous kernels on their own; the oracle's
    rk_step_ns on a reduced mesh of the same field beside it."""
    import torch
    from paper_2006_15698_b200 import DG
    from paper_2006_15698_b200 import inputs as I
    c = I.CONFIGS[workload]
    p, ext, n = c["p"], c["extent"], (c["nx"], c["ny"], c["nz"])
    N = p + 1
    q = I.make_field(workload, xp=torch, device=device)
    dg = DG(*n, p, GAMMA, ext, device=device, viscosity=(mu, prandtl))
    dg.set_state(q)
    dt = I.cfl_dt(dg.max_wavespeed(), p, ext, n, 0.1)
    dof = n[0] * n[1] * n[2] * N ** 3
    stream = torch.cuda.current_stream(device)
    dg.rk_step_ns(dt, 1)
    torch.cuda.synchronize(device)
    e = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
    l0 = dg.launch_count
    e[0].record(stream)
    dg.rk_step_ns(dt, steps)
    e[1].record(stream)
    l1 = dg.launch_count
    dg.split_volume().split_surface()
    e[2].record(stream)
    for _ in range(steps * STAGES):
        dg.split_viscous()
    e[3].record(stream)
    torch.cuda.synchronize(device)
    total, visc = e[0].elapsed_time(e[1]) * 1e-3, e[2].elapsed_time(e[3]) * 1e-3
    finite = bool(torch.isfinite(dg.get_state(q)).all().item())
    dg.close()
    del q
    torch.cuda.empty_cache()
    evals = steps * STAGES
    peak, _ = measured_peaks()
    out = {"workload": f"{workload}: {list(n)} periodic elements, p={p}, {dof} nodes, mu={mu}, Pr={prandtl}",
           "steps": steps, "value": dof * evals / total, "unit": UNIT, "seconds": total, "launches": l1 - l0,
           "viscous_kernels": {"seconds": visc, "dof_per_s": dof * evals / visc, "launches_per_evaluation": 2,
                               "roofline": {"bound": "hbm", "achieved": VISC_BYTES_PER_DOF * dof * evals / visc / 1e9,
                                            "peak": peak, "unit": "GB/s",
                                            "frac": VISC_BYTES_PER_DOF * dof * evals / visc / 1e9 / peak,
                                            "algorithmic_bytes_per_dof": VISC_BYTES_PER_DOF}},
           "finite": finite,
           "note": "not fused into the stage kernel: per-kernel mode (volume, surface, update-project) + two viscous sweeps per "
                   "stage (gradients and viscous flux; divergence); reading R20 (the paper prints no viscous equations)"}
    try:
        import numpy as np
        from oracle import Oracle
        orc = Oracle("omp")
        m = 12
        small = dict(c, nx=m, ny=m, nz=m, extent=tuple(ext[a] * m / n[a] for a in range(3)))
        qs = I.make_field(small)
        t0 = time.perf_counter()
        qo = orc.rk_step_ns(qs, p, GAMMA, small["extent"], mu, prandtl, dt, 1)
        sec = time.perf_counter() - t0
        out["cpu_baseline"] = {"value": m ** 3 * N ** 3 * STAGES / sec, "unit": UNIT, "cores": orc.threads, "kind": "oracle",
                               "sample": f"1 LSERK45 Navier-Stokes step of the same field on a periodic {m}^3-element box, "
                                         f"oracle_rk_step_ns (OpenMP), {sec:.1f} s", "finite": bool(np.isfinite(qo).all())}
    except Exception as ex:   # the oracle is a reported baseline only
        out["cpu_baseline"] = {"error": repr(ex)}
    return out


def decomposed_one_gpu_leg(workload, steps, device, procs=(2, 2, 2)):
    """SURVEY.md 8(f)-1 as far as one GPU goes: the workload's mesh cut into blocks, one context per block, ALL on this
    GPU and one stream (ordinary launches one after another; no kernel waits on another).  Times the export / import
    mode (six gather kernels per block and stage + device copies) and the push mode (the stage kernels store the faces
    into the neighbours' buffers; nothing else is launched) against the single-context run of the same mesh."""
    import torch
    from paper_2006_15698_b200 import DG
    from paper_2006_15698_b200 import decomposed as D
    from paper_2006_15698_b200 import inputs as I
    c = I.CONFIGS[workload]
    p, ext, n = c["p"], c["extent"], (c["nx"], c["ny"], c["nz"])
    dof = n[0] * n[1] * n[2] * (p + 1) ** 3
    stream = torch.cuda.current_stream(device)

    def timed(step):
        step(2)
        torch.cuda.synchronize(device)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        step(steps)
        e1.record(stream)
        torch.cuda.synchronize(device)
        return dof * STAGES * steps / (e0.elapsed_time(e1) * 1e-3)

    out = {"workload": f"{workload}: {list(n)} elements, p={p}, cut into {list(procs)} blocks on ONE GPU", "steps": steps, "unit": UNIT}
    single = DG(*n, p, GAMMA, ext, device=device)
    single.set_state(I.make_field(workload, xp=torch, device=device))
    dt = I.cfl_dt(single.max_wavespeed(), p, ext, n, 0.1)
    out["single_context"] = timed(lambda k: single.rk_step(dt, k))
    variant = single.kernel_info()["variant"]
    single.close()
    for mode in ("export_import", "push"):
        make = D.make_in_process_push if mode == "push" else D.make_in_process
        ranks = make(n, p, GAMMA, ext, procs, device=str(device), variant=variant)
        for r in ranks:
            r.dg.set_state(I.make_field(workload, box=r.box, xp=torch, device=device))
        if mode == "push":
            for r in ranks:
                for f, nb in r.dec.sends(r.rank):
                    r.dg.halo_export(f, ranks[nb].pairs[f ^ 1][0])
            step = lambda k: D.rk_step_in_process_push(ranks, dt, k)
        else:
            D.exchange_in_process(ranks)
            step = lambda k: D.rk_step_in_process(ranks, dt, k)
        l0 = sum(r.dg.launch_count for r in ranks)
        out[mode] = timed(step)
        out[mode + "_launches_per_stage"] = (sum(r.dg.launch_count for r in ranks) - l0) / ((steps + 2) * STAGES)
        for r in ranks:
            r.close()
        del ranks
        torch.cuda.empty_cache()
    out["note"] = ("blocks run one after another on the same GPU, so this measures what the decomposition costs (smaller launches, "
                   "duplicated shared faces, the exchange), not a speed-up; never run on more than one GPU")
    return out


def reduce_max(x, dist, device):
    """Max over ranks of a per-rank time (replicas: the slowest replica sets the whole-job rate)."""
    if dist is None:
        return x
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(dof_per_rank, steps, ms, world):
    """DOF-updates/s per RK stage of the whole job: every rank advances its own replica (weak scaling)."""
    return world * dof_per_rank * STAGES * steps / (ms * 1e-3)


def run_variant_sweep(args):
    """Tuning aid: one JSON line per compiled stage-kernel variant of the workload's degree (1 GPU)."""
    import torch
    from paper_2006_15698_b200 import inputs as I
    from paper_2006_15698_b200.binding import load_library
    device = torch.device("cuda:0")
    torch.cuda.set_device(device)
    peak, _ = measured_peaks()
    p = I.CONFIGS[args.workload]["p"]
    for v in range(load_library().dg_variant_count(p)):
        r = time_workload(args.workload, args.steps, max(3, args.warmup), device, None, variant=v, lz=args.lz)
        rate = r["dof"] * STAGES * args.steps / (r["ms"] * 1e-3)
        print(json.dumps({"workload": args.workload, "variant": v, "kernel": r["kernel"], "value": rate, "unit": UNIT,
                          "roofline_frac": rate * ALGO_BYTES_PER_DOF_STAGE / 1e9 / peak, "finite": r["finite"]}), flush=True)


def run_decomposed(args, rank, world, local_rank):
    """--decomposed: ONE mesh cut into `world` blocks, one rank per GPU, face traces exchanged over
    NCCL after every stage (paper_2006_15698_b200/decomposed.py).  Strong scaling: total work fixed.  Not the default
    (north_star / SURVEY.md 8(e): replicas only) and, this round, run on hardware with one GPU only (world = 1: no
    messages); the multi-rank data path is tested with several contexts in one process (tests/test_gpu_halo.py)."""
    import torch
    import torch.distributed as dist
    from paper_2006_15698_b200 import inputs as I
    from paper_2006_15698_b200.decomposed import DistributedDG
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    device = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(device)
    c = I.CONFIGS[args.workload]
    p, ext, n = c["p"], c["extent"], (c["nx"], c["ny"], c["nz"])
    procs = [1, 1, 1]
    w, a = world, 2
    while w > 1:                                  # factor the rank count over z, y, x in turn
        for f in (2, 3, 5, 7):
            if w % f == 0:
                procs[a] *= f
                w //= f
                a = (a - 1) % 3
                break
        else:
            procs[a] *= w
            w = 1
    local = None if world > 1 else (lambda r, s, v: None)
    dd = DistributedDG(n, p, GAMMA, ext, tuple(procs), rank, device=device, exchange=local,
                       reduce_max=None if world > 1 else (lambda x: x), push=bool(args.push) and world > 1)
    box = dd.box
    dd.set_state(I.make_field(args.workload, box=box, xp=torch, device=device))
    dt = I.cfl_dt(dd.max_wavespeed(), p, ext, n, 0.1)
    K, W = args.steps, max(3, args.warmup)
    dd.rk_step(dt, W)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize(device)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stream = torch.cuda.current_stream(device)
    e0.record(stream)
    dd.rk_step(dt, K)
    e1.record(stream)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize(device)
    ms = reduce_max(e0.elapsed_time(e1), dist if world > 1 else None, device)
    dof = n[0] * n[1] * n[2] * (p + 1) ** 3
    if rank == 0:
        peak, peak_src = measured_peaks()
        value = dof * STAGES * K / (ms * 1e-3)
        print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                          "ms_per_step": ms / K, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
                          "dtype": "f64", "data": "synthetic",
                          "config": {"workload": f"{args.workload}: {list(n)} elements, p={p}, ONE mesh in {procs} blocks, "
                                                 + ("face traces stored by the stage kernel straight into the neighbours' buffers (CUDA IPC / NVLink), "
                                                    "one barrier per stage" if (args.push and world > 1) else "face traces exchanged after every stage"),
                                     "parallelism": f"block decomposition {procs}"},
                          "gpu_launches": dd.dg.launch_count,
                          "roofline": {"bound": "hbm", "achieved": ALGO_BYTES_PER_DOF_STAGE * dof * STAGES * K / (ms * 1e-3) / 1e9 / world,
                                       "peak": peak, "unit": "GB/s per GPU", "frac": value * ALGO_BYTES_PER_DOF_STAGE / 1e9 / peak / world,
                                       "peak_source": peak_src, "traffic": None}}), flush=True)
    dd.close()
    if world > 1:
        dist.destroy_process_group()


def run_ours(args, rank, world, local_rank):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    dist = None
    if world > 1:
        import torch.distributed as td
        td.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
        dist = td
    device = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(device)
    K, W = args.steps, max(3, args.warmup)
    main = time_workload(args.workload, K, W, device, dist, physical_gpu_index(local_rank), want_e2e=True, lz=args.lz,
                         variant=args.variant)

    ms = reduce_max(main["ms"], dist, device)
    e2e_s = reduce_max(main["e2e"]["seconds"], dist, device)
    sweep, sustained, big, fp64, per_kernel, ns, dec1 = [], None, None, None, None, None, None
    # order: the short legs first (burst clocks, like the main leg), then the long ones that heat the board up
    if not args.no_sweep and world == 1:
        for p in range(1, 8):
            s = time_workload(f"cfg4_p{p}", 20, 3, device, None)
            rate = s["dof"] * STAGES * 20 / (s["ms"] * 1e-3)
            sweep.append({"p": p, "elements_per_side": s["elements"][0], "dof": s["dof"], "value": rate,
                          "ms_per_step": s["ms"] / 20, "brick": [s["kernel"][k] for k in ("bx", "by", "lz")],
                          "finite": s["finite"]})
    if world == 1 and not args.no_extras:
        from paper_2006_15698_b200.binding import fp64_peak
        fp64 = fp64_peak(device)
        per_kernel = per_kernel_breakdown("table2_p6", 10, device)
        ns = navier_stokes_leg("table2_p6", 4, device)
        dec1 = decomposed_one_gpu_leg(args.workload if args.workload != "cfg5" else "cfg3", 10, device)
        # the same workload for >= 300 steps: the board reaches its power cap after ~0.3 s and holds lower clocks
        sustained = time_workload(args.workload, max(300, K), W, device, None, physical_gpu_index(local_rank), lz=args.lz,
                                  variant=args.variant)
        if args.workload != "cfg5" and torch.cuda.mem_get_info(device)[1] >= 150 * 2 ** 30:
            big = time_workload("cfg5", 10, 3, device, None, physical_gpu_index(local_rank))
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    peak, peak_src = measured_peaks()
    dof = main["dof"]
    value = whole_job_rate(dof, K, ms, world)
    launch_s = ms * 1e-3 / main["launches"]                       # the step IS 5 stage-kernel launches
    achieved = ALGO_BYTES_PER_DOF_STAGE * dof / launch_s / 1e9

    def traffic_of(workload, n_dof):
        entry = ncu_traffic(workload)
        if not entry:
            return None, None
        return entry.get("dram_bytes_per_launch"), entry

    def frac_of(rate):
        return rate * ALGO_BYTES_PER_DOF_STAGE / 1e9 / peak

    for s in sweep:
        s["roofline_frac"] = frac_of(s["value"])
        t, _ = traffic_of(f"cfg4_p{s['p']}", s["dof"])
        s["traffic"] = t
        s["traffic_over_algorithmic"] = None if t is None else t / (ALGO_BYTES_PER_DOF_STAGE * s["dof"])
    e2e = main["e2e"]
    traffic, traffic_entry = traffic_of(args.workload, dof)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{args.workload}: {main['elements']} periodic elements, p={main['p']}, "
                               f"{dof} nodes ({5 * dof} unknowns), fixed dt, one step = one LSERK45 step (5 stages)",
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "l2": "working set per stage (Q+K, >= 2.6 GB) >> 126 MB L2; no flush needed",
                   "brick": main["kernel"]},
        "unknown_updates_per_s": 5 * value,
        "finite": main["finite"],
        "gpu_launches": main["launches"],
        "clocks": main["clocks"],
        "roofline": {"bound": "hbm", "kernel": "dg_stage_kernel", "achieved": achieved, "peak": peak, "unit": "GB/s",
                     "frac": achieved / peak, "peak_source": peak_src,
                     "algorithmic_bytes_per_launch": ALGO_BYTES_PER_DOF_STAGE * dof,
                     "avg_launch_ms": launch_s * 1e3, "frac_of_8TBs_nominal": achieved / 8000.0,
                     "traffic": traffic,
                     "traffic_unit": "DRAM bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum, ncu --set full)",
                     "traffic_static": True,
                     "traffic_source": None if traffic_entry is None else traffic_entry.get("source")},
        "e2e": {"value": whole_job_rate(dof, e2e["steps"], e2e_s * 1e3, world), "unit": UNIT,
                "h2d_bytes_per_step": e2e["bytes_each_way"], "d2h_bytes_per_step": e2e["bytes_each_way"],
                "steps": e2e["steps"], "api": "DG.set_state(pinned host) -> DG.rk_step(dt,1) -> DG.get_state(pinned host)"},
        "adaptive_dt": {"value": whole_job_rate(dof, main["adaptive_dt"]["steps"], main["adaptive_dt"]["seconds"] * 1e3, world),
                        "unit": UNIT, "steps": main["adaptive_dt"]["steps"],
                        "fixed_dt_same_protocol": whole_job_rate(dof, main["adaptive_dt"]["steps"],
                                                                 main["adaptive_dt"]["fixed_seconds"] * 1e3, world),
                        "ratio_to_fixed_dt": main["adaptive_dt"]["fixed_seconds"] / main["adaptive_dt"]["seconds"],
                        "what": "dg_rk_step_cfl: dt formed on the device by the CFL rule from the max wavespeed the last stage of "
                                "the previous step reduced (no host round trip per step); CUDA events, blocks of 15 steps "
                                "alternating with fixed-dt blocks on a warm board"},
        "p_sweep": sweep,
        "context": "paper: 1.13e9 DOF-updates/s per V100 (kernels only, derived from Table II, PAPER.md:264-269); "
                   "another machine, not a target",
    }
    # the driver's record keeps `roofline` (and cpu_baseline, e2e, config, clocks) and drops other top-level keys:
    # the p sweep, cfg5 and the sustained run are summarised INSIDE `roofline`
    moved = MOVED_BYTES_PER_DOF_STAGE / ALGO_BYTES_PER_DOF_STAGE
    rl = line["roofline"]
    rl["frac_moved"] = round(rl["frac"] * moved, 4)
    rl["frac_note"] = ("frac credits SURVEY.md 8(d)'s 152 B per DOF and stage (the figure the 60 % target is stated on); "
                       "frac_moved counts the 144 B this kernel must move (the dead K store of stage 5 is skipped)")
    if sweep:
        def r4(x):
            return None if x is None else round(x, 4)
        rl["per_p"] = [{"p": s["p"], "frac": r4(s["roofline_frac"]), "frac_moved": r4(s["roofline_frac"] * moved),
                        "value": float(f"{s['value']:.4g}"), "traffic_over_algorithmic": r4(s["traffic_over_algorithmic"])}
                       for s in sweep]
        rl["frac_min_over_p"] = r4(min(s["roofline_frac"] for s in sweep))
        rl["per_p_protocol"] = ("cfg4_p1..7, 20 steps after 3 warm-up steps each, CUDA events, run right after the main leg "
                                "and before the long legs (board warm from the main leg, not yet at the power cap)")
    if sustained is not None:
        s_rate = sustained["dof"] * STAGES * sustained["launches"] / 5 / (sustained["ms"] * 1e-3)
        line["sustained"] = {"value": s_rate, "unit": UNIT, "steps": sustained["launches"] // 5, "roofline_frac": frac_of(s_rate),
                             "clocks": sustained["clocks"],
                             "nj_per_dof_update": None if not sustained["clocks"] or not sustained["clocks"].get("power_w")
                             else 1e9 * sustained["clocks"]["power_w"] / s_rate}
        sc = sustained["clocks"] or {}
        rl["sustained"] = {"frac": round(frac_of(s_rate), 4), "value": float(f"{s_rate:.4g}"), "steps": sustained["launches"] // 5,
                           "sm_mhz": sc.get("sm_mhz"), "power_w": sc.get("power_w")}
    if big is not None:
        b_rate = big["dof"] * STAGES * 10 / (big["ms"] * 1e-3)
        t, _ = traffic_of("cfg5", big["dof"])
        line["cfg5"] = {"value": b_rate, "unit": UNIT, "steps": 10, "dof": big["dof"], "roofline_frac": frac_of(b_rate),
                        "brick": big["kernel"], "finite": big["finite"], "clocks": big["clocks"], "traffic": t}
        bc = big["clocks"] or {}
        rl["cfg5"] = {"frac": round(frac_of(b_rate), 4), "value": float(f"{b_rate:.4g}"), "dof": big["dof"],
                      "clocks": {k: bc.get(k) for k in ("sm_mhz", "sm_max_mhz", "power_w", "reasons")}}
    if per_kernel is not None:
        line["per_kernel"] = per_kernel
    if ns is not None:
        line["navier_stokes"] = ns
    if dec1 is not None:
        line["decomposed_one_gpu"] = dec1
    if fp64 is not None:
        flops = algo_flops_per_dof(main["p"]) * value
        line["roofline_fp64"] = {"bound": "fp64", "achieved": flops / 1e12, "peak": 2.0 * fp64 / 1e12, "unit": "TFLOP/s",
                                 "frac": flops / (2.0 * fp64),
                                 "peak_source": "measured in this run: dg_fp64_peak (8 independent DFMA chains per thread, "
                                                "8 blocks of 256 threads per SM), 2 flop per FMA",
                                 "algorithmic_flop_per_dof_stage": algo_flops_per_dof(main["p"]),
                                 "note": "flop count of SURVEY.md 8(d); executed FP64 instructions per DOF: profiles/"}
    if not args.no_cpu and world == 1:
        cb = oracle_sample(args.workload, target_seconds=10.0)
        line["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample", "finite", "cpu_model")}
        one = oracle_sample(args.workload, fixed_steps=1, build="fp64", nodes=2.0e5)
        line["cpu_baseline"]["single_thread"] = {"value": one["value"], "sample": one["sample"]}
        line["cpu_baseline"]["per_p"] = oracle_per_p()
    # a shorter line: nested floats to 6 significant digits (top-level scalars stay exact), and `roofline` moved to the
    # end, where a truncated tail of the line still shows it
    line["roofline"] = line.pop("roofline")
    print(json.dumps({k: _compact(v) if isinstance(v, (dict, list)) else v for k, v in line.items()}), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def _compact(x):
    if isinstance(x, float):
        return float(f"{x:.6g}") if x == x and abs(x) != float("inf") else x
    if isinstance(x, dict):
        return {k: _compact(v) for k, v in x.items()}
    if isinstance(x, (list, tuple)):
        return [_compact(v) for v in x]
    return x


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--no-sweep", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--decomposed", action="store_true",
                    help="one mesh cut into one block per GPU with halo exchange (strong scaling) instead of replicas")
    ap.add_argument("--push", action="store_true",
                    help="with --decomposed: push mode (dg_set_halo_push; the stage kernel stores the faces into the neighbours' buffers)")
    ap.add_argument("--no-extras", action="store_true", help="skip the sustained run, cfg5 and the FP64 microbenchmark")
    ap.add_argument("--variant", type=int, default=None, help="stage-kernel variant index (tuning; default: library's choice)")
    ap.add_argument("--lz", type=int, default=0, help="layers per chunk (tuning; 0 = library default)")
    ap.add_argument("--sweep-variants", action="store_true", help="time every compiled variant of --workload")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.sweep_variants:
        run_variant_sweep(args)
    elif args.impl == "reference":
        run_reference(args, rank)
    elif args.decomposed:
        run_decomposed(args, rank, world, local_rank)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
