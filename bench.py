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
# Algorithmic work per solution point per RK stage: the MODEL of SURVEY.md S8(d) / Appendix A5 (restated in DESIGN.md 7.3 and
# BASELINE.md 3), not an operation tally of the kernels.  Full physics, whole stage: n -> (flop, bytes).
ALG_BY_ORDER = {4: (3008.0, 794.0), 5: (3267.0, 714.0), 6: (3550.0, 660.0), 7: (3840.0, 622.0), 8: (4141.0, 593.0), 9: (4447.0, 571.0)}
# The viscous face kernel's part of it, the same for every order per point up to the 6/n face points per point:
# 190 flop (108 for the next state's face traces, 54 n^3 FMA per element; 82 for the face correction, 7 components x 6 FMA)
# and 128 B x 6/n (own + neighbour face viscous fluxes, 14 words per face point, and |J|).
FACE_FLOPS, FACE_BYTES_N6 = 190.0, 128.0


def alg_work(n, diff):
    """((stage_bytes, kernel_bytes), (stage_flops, kernel_flops)) per solution point per stage for order n; "kernel" is the
    element kernel (the dominant one).  Diffusion off, Powell sources on (configs 0, 2): contraction FMA x 2 =
    2 [2 x 27 (n+1) + 3 (3 (n+1) + 9)] plus the pointwise work of the n = 6 model (434 flop) scaled with the flux points per
    point; bytes = the full-physics figure minus the face viscous traces (2 x 7 x 6/n words)."""
    f, b = ALG_BY_ORDER.get(n, ALG_BY_ORDER[6])
    if not diff:
        f = 2.0 * (54.0 * (n + 1) + 3.0 * (3.0 * (n + 1) + 9.0)) + 434.0 * ((n + 1) / n) / (7.0 / 6.0)
        b = b - 8.0 * 14.0 * 6.0 / n
        return (b, b), (f, f)
    return (b, b - FACE_BYTES_N6 * 6.0 / n), (f, f - FACE_FLOPS)


FP64_PEAK_TFLOPS = 37.2   # 148 SMs x 4 sub-partitions x 16 FMA/clk x 2 x 1.965 GHz (DMMA measured 37.0)


def cpu_sample_workload(w, n_r=8):
    """Bounded sample of the same workload for the CPU oracle: same order, physics, polytrope and generator on a
    6 x 16 x 16 x n_r shell (n_r = 8: 12,288 elements; the whole of config 3 needs 30 GB and minutes per step on the host)."""
    from paper_2502_17805_b200 import inputs as I
    return I.Workload(w.name + "-cpu-sample", w.order, 16, n_r, w.N_rho, w.seed, w.diffusion, w.dipole, shell=w.shell)


def omp_threads(n=None):
    """Thread count of the oracle's OpenMP runtime (set it when n is given)."""
    import ctypes
    try:
        gomp = ctypes.CDLL("libgomp.so.1")
        if n is not None:
            gomp.omp_set_num_threads(int(n))
        return int(gomp.omp_get_max_threads())
    except OSError:
        return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))


def time_oracle(w, steps, warmup, n_r=8, threads=None):
    """Oracle (as it stands) on the host cores: DOF-updates/s over `steps` SSPRK(5,3) steps of the sample, after `warmup`
    untimed steps (0: one untimed residual evaluation instead, which spins up the thread team and touches the arrays)."""
    from oracle import binding as ob
    from paper_2502_17805_b200 import inputs as I
    ws = cpu_sample_workload(w, n_r)
    mesh = ws.mesh()
    all_threads = omp_threads()
    cores = omp_threads(threads) if threads else all_threads
    try:
        o = ob.Oracle(mesh, ws.order, I.Physics())
        Q = ws.state(o.geometry()["xsol"])
        o.set_state(Q)
        c_h = o.max_wavespeed()
        o.set_physics(ws.physics(c_h))
        _, xf = ob.nodes(ws.order)
        dt = ws.dt(c_h, xf[1] - xf[0])
        if warmup == 0:
            o.residual()
        for _ in range(warmup):
            o.step(dt, NSTAGES)
        per_step = []
        for _ in range(steps):
            t0 = time.perf_counter()
            o.step(dt, NSTAGES)
            per_step.append(time.perf_counter() - t0)
    finally:
        if threads:
            omp_threads(all_threads)
    pts = mesh["n_elem"] * ws.order ** 3
    t_med = float(np.median(per_step))
    return dict(value=pts * 9 * NSTAGES / t_med, unit=UNIT, cores=cores, kind="oracle",
                sample=f"median of {steps} SSPRK(5,3) step(s) of the 6x{ws.n_z}x{ws.n_z}x{ws.n_r} = {mesh['n_elem']}-element shell, order "
                       f"{ws.order}, same physics, polytrope and generator as {w.name}", seconds=float(sum(per_step))), t_med


def workload_config(w, args, world, pts=None):
    """The `config` object of the JSON line: identical for both arms (the reference arm's sample is named in cpu_baseline)."""
    pts = w.n_elem * w.order ** 3 if pts is None else pts
    return dict(workload=args.workload, mesh=f"6x{w.n_z}x{w.n_z}x{w.n_r} cubed-sphere shell", n_elem=w.n_elem, order=w.order,
                solution_points=pts, N_rho=w.N_rho, diffusion=w.diffusion, rk="SSPRK(5,3)",
                parallelism=("single GPU" if world == 1 else f"{world} element partitions, halo all-to-all" if getattr(args, "parallel", "halo") == "halo"
                             else f"{world} replicas"), l2="inputs larger than L2 (state %.0f MB)" % (pts * 72 / 1e6))


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
    """--impl reference: the oracle, as it stands, on the box's host cores (rank 0 only).  Every one of the --steps K steps is
    one SSPRK(5,3) step of a bounded sample of the workload, sized so that K + W steps end within a few minutes."""
    if rank != 0:
        return
    from paper_2502_17805_b200 import inputs as I
    w = I.workload(args.workload)
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    n_r = 8 if steps + warmup <= 8 else 4 if steps + warmup <= 16 else 2 if steps + warmup <= 32 else 1
    cb, sec_per_step = time_oracle(w, steps, warmup, n_r=n_r)
    cb.pop("seconds", None)
    line = dict(impl="reference", metric=METRIC, value=cb["value"], unit=UNIT, n_gpus=args.gpus, steps=steps, warmup=warmup,
                ms_per_step=1e3 * sec_per_step, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64",
                data="synthetic", config=workload_config(w, args, world), cpu_baseline=cb,
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
    ap.add_argument("--parallel", default="halo", choices=["halo", "replicas"],
                    help="N > 1: 'halo' = ONE workload split into N element partitions with halo exchange (strong scaling); "
                         "'replicas' = every rank advances its own copy (weak scaling, no data-path collective)")
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
    halo = world > 1 and args.parallel == "halo"
    if halo:
        # one workload, `world` element partitions: this rank owns a contiguous block of elements plus ghost copies of its
        # off-rank face neighbours; face traces and viscous face fluxes of the partition boundary travel by NCCL all-to-all
        from paper_2502_17805_b200.partition import DistributedChorus
        job = DistributedChorus(mesh, n, I.Physics(), dist)
        g = job.g
        pts = mesh["n_elem"] * n ** 3                 # the whole job's solution points
    else:
        g = job = P.Chorus(mesh, n, I.Physics())
        pts = g.E * n ** 3
    Q = w.state(g.xsol())                             # the local elements' state (ghost slots are ignored by a partition)
    del mesh
    host = torch.from_numpy(Q).pin_memory()
    del Q
    g.set_state(host.numpy())
    c_h = job.max_wavespeed()
    phys = w.physics(c_h)
    job.set_physics(phys)
    _, xf, _, _ = P.get_operators(n)
    dt = w.dt(c_h, xf[1] - xf[0])
    diff = w.diffusion > 0

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput
    for _ in range(warmup):
        job.step(dt, NSTAGES)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = g.launch_count()
    barrier()
    with ClockSampler(local) as clocks:     # the headline loop: no per-launch events
        ev0.record()
        for _ in range(args.steps):
            job.step(dt, NSTAGES)
        ev1.record()
        barrier()
    ms = ev0.elapsed_time(ev1)
    launches = g.launch_count() - l0
    ws_after = job.max_wavespeed()        # also proves the state is still finite
    # ---- per-kernel device times: a separate pass with every launch bracketed by CUDA events on the library's stream
    g.profile(True)
    g.profile_read()
    prof_steps = max(1, min(args.steps, 4))
    for _ in range(prof_steps):
        job.step(dt, NSTAGES)
    prof = g.profile_read()
    g.profile(False)
    prof_ms = sum(v[0] for v in prof.values())
    # ---- end to end through the C ABI with HOST buffers: H2D of the state, one step, D2H of the CFL wave speed
    # Every step: H2D of the state from pinned memory, one step, D2H of the new state into pinned memory, the CFL wave speed.
    e2e_ms, e2e_nod2h_ms, e2e_pipe_ms, e2e_steps, pipe_steps = None, None, None, 0, 0
    if not args.no_e2e:
        e2e_steps = max(1, min(args.steps, 5))
        hnp = host.numpy()
        out = torch.empty_like(host).pin_memory().numpy()
        g.set_state(hnp); job.step(dt, NSTAGES); g.get_state(out); job.max_wavespeed()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            g.set_state(hnp)
            job.step(dt, NSTAGES)
            g.get_state(out)
            job.max_wavespeed()
        barrier()
        e2e_ms = 1e3 * (time.perf_counter() - t0)
        assert np.isfinite(out[:, ::max(1, out.shape[1] // 64)]).all()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):          # the same without the state coming back (round 1's figure), for comparison
            g.set_state(hnp)
            job.step(dt, NSTAGES)
            job.max_wavespeed()
        barrier()
        e2e_nod2h_ms = 1e3 * (time.perf_counter() - t0)
        if not halo:
            # the same jobs through chorus_step_host: copies on the library's copy streams beside the kernels (two staging slots)
            outs = [out, torch.empty_like(host).pin_memory().numpy()]
            wss = [torch.zeros(1, dtype=torch.float64).pin_memory().numpy() for _ in range(2)]
            for k in range(2):
                g.step_host(hnp, outs[k], dt, NSTAGES, wss[k])
            g.sync()
            barrier()
            pipe_steps = max(e2e_steps, min(args.steps, 20))      # the pipeline's fill and drain (one copy each way) are inside the timing
            t0 = time.perf_counter()
            for k in range(pipe_steps):
                g.step_host(hnp, outs[k & 1], dt, NSTAGES, wss[k & 1])
            g.sync()
            barrier()
            e2e_pipe_ms = 1e3 * (time.perf_counter() - t0)
            assert np.isfinite(outs[(pipe_steps - 1) & 1][:, ::max(1, out.shape[1] // 64)]).all() and np.isfinite(wss[(pipe_steps - 1) & 1][0])
    ms, e2e_max, e2e_nod2h_max, e2e_pipe_max = max_over_ranks([ms, e2e_ms or 0.0, e2e_nod2h_ms or 0.0, e2e_pipe_ms or 0.0], dist)
    if e2e_ms is not None:
        e2e_ms, e2e_nod2h_ms = e2e_max, e2e_nod2h_max
        if e2e_pipe_ms is not None:
            e2e_pipe_ms = e2e_pipe_max
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
    jobs = 1 if halo else world               # halo: the ranks share ONE workload; replicas: each rank advances its own
    value = job_value(dof_per_step, args.steps, jobs, ms)
    hbm_peak, peak_src = measured_peaks()
    main_ms, main_cnt = prof["main"]
    main_avg_ms = main_ms / max(main_cnt, 1)
    pts_local = (job.n_owned if halo else g.E) * n ** 3      # what this GPU's kernels process per stage (roofline figures are per GPU)
    (stage_bytes, kernel_bytes), (stage_flops, kernel_flops) = alg_work(n, diff)
    achieved = kernel_flops * pts_local / (main_avg_ms * 1e-3) / 1e12 if main_cnt else None        # TFLOP/s of the element kernel
    kernel_ms = {k: (v[0] / max(v[1], 1)) for k, v in prof.items()}
    stage_ms = ms / (args.steps * NSTAGES)
    t_hbm = stage_bytes * pts_local / (hbm_peak * 1e9) * 1e3
    t_alu = stage_flops * pts_local / (FP64_PEAK_TFLOPS * 1e12) * 1e3
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=args.steps, warmup=warmup, ms_per_step=ms / args.steps,
                higher_is_better=True, scaling="strong" if halo else "weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=workload_config(w, args, world, pts),
                clocks=clocks.summary(), gpu_launches=launches,
                roofline=dict(bound="alu", kernel="stage_main_kernel" if 4 <= n <= 8 else "residual_kernel", achieved=achieved, peak=FP64_PEAK_TFLOPS, unit="TFLOP/s",
                              frac=(achieved / FP64_PEAK_TFLOPS) if achieved else None, traffic=ncu_traffic(args.workload),
                              traffic_source="dram__bytes_read.sum + dram__bytes_write.sum of one launch, from the committed ncu --set full "
                                             "capture (profiles/roofline_traffic.md); not measured in this run",
                              alg_source="model of SURVEY.md S8(d) / Appendix A5 (BASELINE.md 3), not an operation tally",
                              peak_source="nominal FP64 pipe: 148 SMs x 4 x 16 FMA/clk x 2 x 1.965 GHz (DESIGN.md 7.3)",
                              measured_fp64=peaks, alg_flops_per_point=kernel_flops, alg_bytes_per_point=kernel_bytes,
                              kernel_hbm=dict(achieved_gbs=kernel_bytes * pts_local / (main_avg_ms * 1e-3) / 1e9 if main_cnt else None,
                                              peak_gbs=hbm_peak, peak_source=peak_src),
                              kernel_ms=kernel_ms, kernel_share_of_step={k: v[0] / prof_ms for k, v in prof.items()} if prof_ms else None,
                              kernel_timing=f"separate pass of {prof_steps} step(s) with per-launch CUDA events; the headline loop runs without them",
                              stage=dict(ms=stage_ms, alg_bytes_per_point=stage_bytes, alg_flops_per_point=stage_flops,
                                         t_hbm_ms=t_hbm, t_alu_ms=t_alu, binding="alu" if t_alu >= t_hbm else "hbm",
                                         frac_of_binding=max(t_hbm, t_alu) / stage_ms,
                                         achieved_gbs=stage_bytes * pts_local / (stage_ms * 1e-3) / 1e9,
                                         achieved_fp64_tflops=stage_flops * pts_local / (stage_ms * 1e-3) / 1e12)),
                wavespeed_after=ws_after)
    if e2e_ms is not None:
        line["e2e"] = dict(value=jobs * dof_per_step * e2e_steps / (e2e_ms * 1e-3), unit=UNIT, h2d_bytes_per_step=int(host.numel()) * 8,
                           d2h_bytes_per_step=int(host.numel()) * 8 + 8, steps=e2e_steps, ms_per_step=e2e_ms / e2e_steps,
                           what="chorus_set_state(pinned host) + chorus_step(dt,5) + chorus_get_state(pinned host) + chorus_max_wavespeed",
                           without_state_d2h=dict(value=jobs * dof_per_step * e2e_steps / (e2e_nod2h_ms * 1e-3),
                                                  ms_per_step=e2e_nod2h_ms / e2e_steps, d2h_bytes_per_step=8))
        if e2e_pipe_ms is not None:
            # headline e2e: the same jobs (same bytes each way, every step) issued through chorus_step_host, whose copies run on
            # the library's copy streams beside the kernels; the synchronous three-call sequence is kept beside it
            seq = {k: line["e2e"][k] for k in ("value", "ms_per_step", "what", "steps")}
            line["e2e"].update(value=jobs * dof_per_step * pipe_steps / (e2e_pipe_ms * 1e-3), ms_per_step=e2e_pipe_ms / pipe_steps, steps=pipe_steps,
                               what="chorus_step_host(pinned host in, pinned host out, dt, 5, wave speed) per step + one chorus_sync: "
                                    "H2D of the next job and D2H of the previous one overlap the kernels (DESIGN.md 7.7)",
                               sequential=seq)
    if world == 1 and not args.no_cpu_baseline:
        # the oracle on a 12,288-element sample of the same workload: one untimed residual, then one step on all cores
        # (~20-40 s of host work), and one step of a 1,536-element sample on one core
        cb, _ = time_oracle(w, 1, 0, n_r=8)
        cb.pop("seconds", None)
        one, _ = time_oracle(w, 1, 0, n_r=1, threads=1)
        cb["one_core"] = dict(value=one["value"], unit=UNIT, cores=one["cores"], sample=one["sample"])
        line["cpu_baseline"] = cb
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
