#!/usr/bin/env python
"""bench.py -- throughput of the CHORUS-MHD hot path (SD-MHD residual + SSPRK(5,3) step) on B200.

  python bench.py --gpus N --steps K --warmup W [--workload config3] [--impl reference]

A "step" is one chorus_step(dt, 5): five residual evaluations (all SURVEY.md S8(a) rows A1-A9) fused with their
Runge-Kutta combinations, over one synthetic stratified shell.  metric = SD-MHD DOF-updates/s = solution points x 9
variables x RK stages / time (BASELINE.json).  One JSON line on stdout (rank 0).
With N > 1 every rank advances its own replica of the workload (weak scaling, no data-path collective: the
multi-GPU halo exchange of SURVEY.md S8(e) is a "next" row).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "SD-MHD DOF-updates/s (sol pts x 9 vars x RK stages)"
UNIT = "DOF-updates/s"
NSTAGES = 5
# Algorithmic work per solution point per RK stage at n = 6 (restated in DESIGN.md 7.3), keyed by
# "diffusion on": HBM bytes (whole stage, element kernel's share) and flop (whole stage, element kernel's share).
ALG_BYTES = {True: (660.0, 532.0), False: (548.0, 548.0)}
ALG_FLOPS = {True: (3550.0, 3360.0), False: (1370.0, 1370.0)}
# Other orders, full physics: n -> (flop, bytes) per point per stage, whole stage.
ALG_BY_ORDER = {4: (3008.0, 794.0), 5: (3267.0, 714.0), 6: (3550.0, 660.0), 7: (3840.0, 622.0), 8: (4141.0, 593.0), 9: (4447.0, 571.0)}


def alg_work(n, diff):
    """((stage_bytes, kernel_bytes), (stage_flops, kernel_flops)) per solution point per stage for order n.
    The element kernel's share of the stage is scaled from the n = 6 split (the rest is the viscous face kernel: face
    correction and next traces); without diffusion only the n = 6 figures exist and are scaled by the full-physics ratio."""
    if n == 6:
        return ALG_BYTES[diff], ALG_FLOPS[diff]
    f, b = ALG_BY_ORDER.get(n, ALG_BY_ORDER[6])
    if not diff:
        f, b = f * 1370.0 / 3550.0, b * 548.0 / 660.0
        return (b, b), (f, f)
    return (b, b * 532.0 / 660.0), (f, f * 3360.0 / 3550.0)
FP64_PEAK_TFLOPS = 37.2   # 148 SMs x 4 sub-partitions x 16 FMA/clk x 2 x 1.965 GHz (DMMA measured 37.0)


def cpu_sample_workload(w):
    """Bounded sample of the same workload for the CPU oracle: same order, physics, generator; fewer elements."""
    from paper_2502_17805_b200 import inputs as I
    return I.Workload(w.name + "-cpu-sample", w.order, 16, 6, w.N_rho, w.seed, w.diffusion, w.dipole, shell=w.shell)


def time_oracle(w, steps, warmup):
    """Oracle (as it stands) on the host cores: DOF-updates/s over `steps` SSPRK(5,3) steps of the sample."""
    from oracle import binding as ob
    from paper_2502_17805_b200 import inputs as I
    ws = cpu_sample_workload(w)
    mesh = ws.mesh()
    o = ob.Oracle(mesh, ws.order, I.Physics())
    Q = ws.state(o.geometry()["xsol"])
    o.set_state(Q)
    c_h = o.max_wavespeed()
    o.set_physics(ws.physics(c_h))
    _, xf = ob.nodes(ws.order)
    dt = ws.dt(c_h, xf[1] - xf[0])
    for _ in range(warmup):
        o.step(dt, NSTAGES)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step(dt, NSTAGES)
    t = time.perf_counter() - t0
    pts = mesh["n_elem"] * ws.order ** 3
    cores = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    return dict(value=pts * 9 * NSTAGES * steps / t, unit=UNIT, cores=cores, kind="oracle",
                sample=f"{steps} SSPRK(5,3) step(s) of the 6x{ws.n_z}x{ws.n_z}x{ws.n_r} = {mesh['n_elem']}-element shell, order {ws.order}, "
                       f"same physics and generator as {w.name}", seconds=t), t / steps


class ClockSampler:
    def __init__(self, index):
        self.rows, self._stop, self.index = [], threading.Event(), index
        self._t = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i", str(self.index)],
                                     capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([x.strip() for x in out.split(",")])
            except Exception:
                pass
            self._stop.wait(0.2)

    def __enter__(self):
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        if not self.rows:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(r[3 + i].lower().startswith("active") for r in self.rows if len(r) > 3 + i)]
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None, reasons=reasons,
                    samples=len(self.rows))


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def max_over_ranks(values, dist=None):
    """Element-wise max of a list of floats over all ranks (timing rule: multi-GPU numbers are the max over ranks).
    `dist` is an initialised torch.distributed module or None (single process); works on any backend."""
    if dist is None:
        return [float(v) for v in values]
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(v) for v in values], device=dev, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def job_value(units_per_rank_step, steps, world, ms_max):
    """Whole-job throughput: the units all ranks processed divided by the slowest rank's time."""
    return world * units_per_rank_step * steps / (ms_max * 1e-3)


def ncu_traffic(workload):
    """dram bytes per launch of the element kernel from the committed ncu --set full capture, if one exists."""
    p = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    if os.path.exists(p):
        try:
            return json.load(open(p)).get(workload)
        except Exception:
            return None
    return None


def run_reference(args, rank, world):
    """--impl reference: the oracle, as it stands, on the box's host cores (rank 0 only)."""
    if rank != 0:
        return
    from paper_2502_17805_b200 import inputs as I
    w = I.workload(args.workload)
    steps = max(1, min(args.steps, 10))
    cb, sec_per_step = time_oracle(w, steps, min(args.warmup, 3))
    line = dict(impl="reference", metric=METRIC, value=cb["value"], unit=UNIT, n_gpus=args.gpus, steps=steps, warmup=min(args.warmup, 3),
                ms_per_step=1e3 * sec_per_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", config=dict(workload=args.workload, sample=cb["sample"], order=w.order,
                                              parallelism="host cores (OpenMP over elements)"),
                cpu_baseline=dict(value=cb["value"], unit=UNIT, cores=cb["cores"], kind="oracle", sample=cb["sample"]),
                e2e=dict(value=cb["value"], unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config3")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", 0))
    world = int(os.environ.get("WORLD_SIZE", 1))
    local = int(os.environ.get("LOCAL_RANK", 0))
    if args.impl == "reference":
        return run_reference(args, rank, world)

    import torch
    import paper_2502_17805_b200 as P
    from paper_2502_17805_b200 import inputs as I
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the hot path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    warmup = max(args.warmup, 3)

    # ---- synthetic input (recipe in DESIGN.md "Inputs"): mesh -> library geometry -> seeded state at its solution points
    w = I.workload(args.workload)
    n = w.order
    mesh = w.mesh()
    g = P.Chorus(mesh, n, I.Physics())
    Q = w.state(g.xsol())
    del mesh
    pts = g.E * n ** 3
    host = torch.from_numpy(Q).pin_memory()
    del Q
    g.set_state(host.numpy())
    c_h = g.max_wavespeed()
    phys = w.physics(c_h)
    g.set_physics(phys)
    _, xf, _, _ = P.get_operators(n)
    dt = w.dt(c_h, xf[1] - xf[0])
    diff = w.diffusion > 0

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput
    for _ in range(warmup):
        g.step(dt, NSTAGES)
    g.profile(True)
    g.profile_read()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = g.launch_count()
    barrier()
    with ClockSampler(local) as clocks:
        ev0.record()
        for _ in range(args.steps):
            g.step(dt, NSTAGES)
        ev1.record()
        barrier()
    ms = ev0.elapsed_time(ev1)
    launches = g.launch_count() - l0
    prof = g.profile_read()
    g.profile(False)
    ws_after = g.max_wavespeed()          # also proves the state is still finite
    # ---- end to end through the C ABI with HOST buffers: H2D of the state, one step, D2H of the CFL wave speed
    e2e_ms, e2e_steps = None, 0
    if not args.no_e2e:
        e2e_steps = max(1, min(args.steps, 5))
        hnp = host.numpy()
        g.set_state(hnp); g.step(dt, NSTAGES); g.max_wavespeed()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            g.set_state(hnp)
            g.step(dt, NSTAGES)
            g.max_wavespeed()
        barrier()
        e2e_ms = 1e3 * (time.perf_counter() - t0)
    ms, e2e_max = max_over_ranks([ms, e2e_ms or 0.0], dist)
    e2e_ms = e2e_max if e2e_ms is not None else None
    peaks = None
    if rank == 0:   # sustained FP64 issue rates of this device (DFMA, DMMA), ~0.5 s each: the "alu" roofline's measured companion
        try:
            peaks = dict(dfma_tflops=P.fp64_peak(0, 0.5)[0], dmma_tflops=P.fp64_peak(1, 0.5)[0])
        except Exception as ex:   # measurement only
            peaks = dict(error=str(ex))
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    dof_per_step = pts * 9 * NSTAGES
    value = job_value(dof_per_step, args.steps, world, ms)
    hbm_peak, peak_src = measured_peaks()
    main_ms, main_cnt = prof["main"]
    main_avg_ms = main_ms / max(main_cnt, 1)
    (stage_bytes, kernel_bytes), (stage_flops, kernel_flops) = alg_work(n, diff)
    achieved = kernel_flops * pts / (main_avg_ms * 1e-3) / 1e12 if main_cnt else None        # TFLOP/s of the element kernel
    kernel_ms = {k: (v[0] / max(v[1], 1)) for k, v in prof.items()}
    stage_ms = ms / (args.steps * NSTAGES)
    t_hbm = stage_bytes * pts / (hbm_peak * 1e9) * 1e3
    t_alu = stage_flops * pts / (FP64_PEAK_TFLOPS * 1e12) * 1e3
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=warmup, ms_per_step=ms / args.steps,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=args.workload, mesh=f"6x{w.n_z}x{w.n_z}x{w.n_r} cubed-sphere shell", n_elem=g.E, order=n,
                            solution_points=pts, N_rho=w.N_rho, diffusion=w.diffusion, rk="SSPRK(5,3)",
                            parallelism="replicas" if world > 1 else "single GPU", l2="inputs larger than L2 (state %.0f MB)" % (pts * 72 / 1e6)),
                clocks=clocks.summary(), gpu_launches=launches,
                roofline=dict(bound="alu", kernel="stage_main_kernel" if 4 <= n <= 7 else "residual_kernel", achieved=achieved, peak=FP64_PEAK_TFLOPS, unit="TFLOP/s",
                              frac=(achieved / FP64_PEAK_TFLOPS) if achieved else None, traffic=ncu_traffic(args.workload),
                              peak_source="nominal FP64 pipe: 148 SMs x 4 x 16 FMA/clk x 2 x 1.965 GHz (DESIGN.md 7.3)",
                              measured_fp64=peaks, alg_flops_per_point=kernel_flops, alg_bytes_per_point=kernel_bytes,
                              kernel_hbm=dict(achieved_gbs=kernel_bytes * pts / (main_avg_ms * 1e-3) / 1e9 if main_cnt else None,
                                              peak_gbs=hbm_peak, peak_source=peak_src),
                              kernel_ms=kernel_ms, kernel_share_of_step={k: v[0] / ms for k, v in prof.items()},
                              stage=dict(ms=stage_ms, alg_bytes_per_point=stage_bytes, alg_flops_per_point=stage_flops,
                                         t_hbm_ms=t_hbm, t_alu_ms=t_alu, binding="alu" if t_alu >= t_hbm else "hbm",
                                         frac_of_binding=max(t_hbm, t_alu) / stage_ms,
                                         achieved_gbs=stage_bytes * pts / (stage_ms * 1e-3) / 1e9,
                                         achieved_fp64_tflops=stage_flops * pts / (stage_ms * 1e-3) / 1e12)),
                wavespeed_after=ws_after)
    if e2e_ms is not None:
        line["e2e"] = dict(value=world * dof_per_step * e2e_steps / (e2e_ms * 1e-3), unit=UNIT, h2d_bytes_per_step=pts * 72,
                           d2h_bytes_per_step=8, steps=e2e_steps, ms_per_step=e2e_ms / e2e_steps,
                           what="chorus_set_state(pinned host) + chorus_step(dt,5) + chorus_max_wavespeed")
    if world == 1 and not args.no_cpu_baseline:
        cb, _ = time_oracle(w, 3, 0)      # ~10-20 s of host work on the box's cores
        cb.pop("seconds", None)
        line["cpu_baseline"] = cb
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
