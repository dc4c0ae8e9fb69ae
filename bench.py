#!/usr/bin/env python
"""Benchmark of the hot path: SSP-RK3 steps of the matrix-free CG
Euler RHS + stage update on a synthetic limited-area tropical-cyclone workload.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg2|cfg2n7|cfg4nX|cfg5]
                    [--impl reference]

One "step" = one SSP-RK3 time step = 3 passes of the whole hot path (rows A2-A10 of SURVEY.md
8(a): volume RHS, DSS, sources + walls, RK stage update).  The metric is BASELINE.json's:
FP64 nodal RHS evaluations per second per RK stage, in GDOF/s with the paper's DOF = 5 x local
nodes, i.e. value = 5 * NL * 3 * K / t.  Prints ONE JSON line on rank 0.

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded
sample of the same workload; it is the slow reference arm, not a target.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "fp64_nodal_rhs_evals_per_s_per_rk_stage"
UNIT = "GDOF/s"


def parse_workload(name):
    """-> (config, N or None)"""
    name = name.lower()
    if name == "cfg2n7":
        return 2, 7
    if name in ("cfg4lit4", "cfg4lit7"):
        return 4, -int(name[-1])     # negative N: BASELINE.json's literal element counts (Q14)
    if name.startswith("cfg4n"):
        return 4, int(name[5:])
    if name == "table1":
        return 0, 5                  # the paper's Table-1 grid (80x80x24, N=5; inputs.paper_table1_workload)
    if name in ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5"):
        return int(name[3]), None
    raise SystemExit("unknown workload %r" % name)


def f_face(N):
    """Share of an element's nodes that lie on its faces."""
    return 1.0 - ((N - 1.0) / (N + 1.0)) ** 3


def b_alg_bytes(N, has_src):
    """Algorithmic bytes per local node per RK stage (fixed there):
    8 [5 qs + 5*2/3 q0 + 9 grad xi + 1 omega + 2 (rho0, theta0) + n_src + 5 q_out] + 2*8*5*f_face."""
    return volume_alg_bytes(N, has_src) + dss_alg_bytes(N)


def volume_alg_bytes(N, has_src):
    """The volume kernel's share of B_alg: everything except the DSS round trip."""
    n_src = 2 if has_src else 0
    return 8.0 * (5 + 5 * (2.0 / 3.0) + 9 + 1 + 2 + n_src + 5)


def dss_alg_bytes(N):
    """The DSS kernel's share of B_alg: face nodes of 5 fields read and written once."""
    return 2 * 8 * 5 * f_face(N)


def hd_lap_alg_bytes():
    """One application of omega div(tau grad .) to 4 fields: 4 in, 4 out (the second application also
    reads the 4 it accumulates into: counted as +2 on average), grad xi (9), tau (6), omega (1)."""
    return 8.0 * (4 + 4 + 2 + 9 + 6 + 1)


def f_alg_flops(N):
    """Algorithmic FP64 flop per local node per RK stage: 48 (N+1) for the 24
    contractions + 207 for chain rule, tendencies, DSS, sources and the stage update."""
    return 48.0 * (N + 1) + 207.0


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def captured_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload`, from the
    tracked ncu --set full summary profiles/traffic_r2.csv (columns: workload, kernel,
    dram_bytes_per_launch, capture; written from the captures named in its last column, commands in
    profiles/traffic_r2.md); None when no capture of this workload / kernel is tracked."""
    path = os.path.join(ROOT, "profiles", "traffic_r2.csv")
    try:
        with open(path) as f:
            for line in f:
                w, k, b, cap = [x.strip() for x in line.split(",")]
                if w == workload and k == kernel.split(" ")[0]:
                    return float(b), "profiles/traffic_r2.csv (%s)" % cap
    except Exception:
        pass
    return None, None


def set_omp_threads(n):
    """Thread count of the oracle's OpenMP runtime (libgomp, already loaded by the oracle)."""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                 "--format=csv,noheader,nounits", "-lms", "25"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0=None, t1=None):
        """Median SM clock and throttle reasons of the samples that arrived in [t0, t1] (wall
        clock of the timed region; all samples if none fell inside)."""
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 is None or (t0 <= t <= (t1 or t) + 0.03)]
        if not rows:
            rows = [r for (t, r) in self.rows if t0 is None or t >= t0] or [r for (_, r) in self.rows]
        for r in rows:
            parts = [p.strip() for p in r.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); smax = float(parts[1])
            except ValueError:
                continue
            for n, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": len(sm)}


def cpu_sample_workload(config, N):
    """Bounded sample of the workload for the oracle: same physics and element shapes, fewer
    element columns (about 1 M local nodes, i.e. seconds per RK3 step on a few cores)."""
    from paper_2504_08157_b200 import inputs
    if config in (1, 2):
        wl = inputs.make_workload(config, N=N)
        return wl, "whole workload %s (%d local nodes)" % (wl.name, wl.mesh.n_local)
    n = N or (7 if config == 5 else 4)
    nz = 24 if config == 5 else 20
    base = {3: 100, 4: inputs.CFG4_NXY.get(n, 113), 5: 160}[config]
    nxy = max(2, int(round((1.0e6 / (n + 1) ** 3 / nz) ** 0.5)))
    wl = inputs.make_workload(config, N=N, scale=min(1.0, nxy / base))
    return wl, "%s: %dx%dx%d elements (%d local nodes), same physics and element heights" % (
        wl.name, wl.mesh.nx, wl.mesh.ny, wl.mesh.nz, wl.mesh.n_local)


def time_oracle(wl, steps, warmup, threads=None):
    """Seconds for `steps` SSP-RK3 steps of the oracle (as it stands) and the threads it used."""
    from oracle import oracle as orc
    o = orc.Oracle.from_workload(wl)
    ncpu = os.cpu_count() or 1
    want = threads or int(os.environ.get("OMP_NUM_THREADS", ncpu))
    want = max(1, min(want, ncpu))
    if not set_omp_threads(want):
        want = int(os.environ.get("OMP_NUM_THREADS", ncpu))
    q = wl.q
    for _ in range(warmup):
        q = o.step_rk3(q, wl.dt, wl.heating)
    t0 = time.perf_counter()
    for _ in range(steps):
        q = o.step_rk3(q, wl.dt, wl.heating)
    t = time.perf_counter() - t0
    return t, want


def max_over_ranks(x, device, world):
    """MAX over ranks of one float (torch.distributed must be initialised when world > 1)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_gdof_per_s(n_local, steps, world, seconds):
    """Whole-job value: every rank (replica) advances n_local nodes x 5 DOF x 3 stages per step."""
    return 5.0 * n_local * 3 * steps * world / seconds / 1e9


def run_reference(args):
    """--impl reference: the CPU oracle on a bounded sample (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    config, N = parse_workload(args.workload)
    N = abs(N) if N else N
    wl, sample = cpu_sample_workload(config, N)
    steps = max(1, min(args.steps, 5))
    warm = max(0, min(args.warmup, 1))
    t, cores = time_oracle(wl, steps, warm)
    t1, _ = time_oracle(wl, max(1, min(steps, 2)), 0, threads=1)
    NL = wl.mesh.n_local
    value = 5.0 * NL * 3 * steps / t / 1e9
    value_1 = 5.0 * NL * 3 * max(1, min(steps, 2)) / t1 / 1e9
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": steps, "warmup": warm, "ms_per_step": 1e3 * t / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "sample_of": args.workload, "N": wl.mesh.N,
                   "local_nodes": NL, "integrator": "SSP-RK3", "dt": wl.dt},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": sample, "single_thread": {"value": value_1, "cores": 1}},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_gpu(args):
    import torch
    import torch.distributed as dist
    from paper_2504_08157_b200 import binding, inputs

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.gpus != world:
        # replicas only: the N ranks come from torchrun, bench.py spawns nothing itself
        raise SystemExit("bench.py --gpus %d needs %d ranks but WORLD_SIZE is %d: launch it as\n  python -m "
                         "torch.distributed.run --nnodes=1 --nproc-per-node %d --master-addr 127.0.0.1 "
                         "--master-port 29500 bench.py --gpus %d ..." % (args.gpus, args.gpus, world, args.gpus, args.gpus))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference "
                         "for the CPU oracle arm")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    config, N_arg = parse_workload(args.workload)
    literal = N_arg is not None and N_arg < 0
    N_arg = -N_arg if literal else N_arg
    wl = inputs.paper_table1_workload() if config == 0 else inputs.make_workload(config, N=N_arg, literal=literal)
    if args.integrator == "ark2":
        return run_gpu_ark2(args, wl, dev, rank, world)
    mesh = wl.mesh
    NL = mesh.n_local
    g = binding.Numa.from_workload(wl, device=str(dev))
    if args.hyperdiffusion:
        # tensor hyper-diffusion on (Eq. 14-16): coefficients that put dt * rho(H) near 1 on the
        # config-3 element shapes (measured with the oracle, tests/test_gpu_hyperdiffusion.py)
        g.hd_init((1.5e-5, 1.5e-5, 4.5e-5), wl.dt)
    q = g.state(wl.q)
    heat = None if wl.heating is None else g.state(wl.heating)
    g.scratch()
    stream = torch.cuda.current_stream()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    # heating fields of the refreshes that fall inside the timed steps, resident before timing
    seg = wl.heating_refresh_steps if (heat is not None and wl.heating_refresh_steps) else args.steps
    seg = max(1, min(seg, args.steps))
    n_seg = (args.steps + seg - 1) // seg
    heats = [heat] + [g.state(wl.heating_at(k)) for k in range(1, n_seg)] if heat is not None else [None]

    # ---- device-resident timing (per-kernel event timing OFF) --------------------------------
    g.step_rk3(q, wl.dt, heat, args.warmup)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)   # nvidia-smi needs a moment before its first sample; untimed
    l0 = g.launch_count
    ev0 = torch.cuda.Event(enable_timing=True); ev1 = torch.cuda.Event(enable_timing=True)
    barrier()
    wall0 = time.time()
    ev0.record(stream)
    done = 0
    while done < args.steps:     # one call per heating segment ("refreshed every 60 s": every 60 steps, Q12)
        n = min(seg, args.steps - done)
        g.step_rk3(q, wl.dt, heats[(done // seg) % len(heats)], n, graph=args.graph)
        done += n
    ev1.record(stream)
    barrier()
    wall1 = time.time()
    ms = ev0.elapsed_time(ev1)
    launches = g.launch_count - l0
    if rank == 0 and not any(wall0 <= t <= wall1 + 0.03 for (t, _) in sampler.rows):
        # very short timed region: keep the same load running until a sample has been taken
        n0 = len(sampler.rows)
        t_end = time.time() + 3.0
        while len(sampler.rows) == n0 and time.time() < t_end:
            g.step_rk3(q, wl.dt, heat, 5)
            torch.cuda.synchronize()
    clocks = sampler.stop(wall0, wall1) if rank == 0 else None
    finite = bool(torch.isfinite(q).all().item())
    ms = max_over_ranks(ms, dev, world)

    # ---- second pass: the per-kernel split (CUDA events around every launch) ----------------
    g.profile(True)
    g.step_rk3(q, wl.dt, heat, min(args.steps, 10))
    prof = g.profile_read()
    g.profile(False)
    prof_steps = min(args.steps, 10)

    # ---- FP64 ceiling of this device (DFMA micro-benchmark, numa_b200_measure.h) -------------
    fp64_peak = g.fp64_peak_tflops(5) if rank == 0 else None

    # ---- end to end through the C ABI with host buffers ---------------------------------
    qh = torch.from_numpy(wl.q.copy()).pin_memory()
    hh = None if wl.heating is None else torch.from_numpy(wl.heating.copy()).pin_memory()
    dq = torch.empty_like(q)
    dh = None if heat is None else torch.empty_like(heat)
    e2e_steps = max(1, min(args.steps, 10))
    g.step_rk3_host(qh, wl.dt, hh, 1, dq, dh)   # warm-up
    barrier()
    t0 = time.perf_counter()
    for k in range(e2e_steps):
        # every step: H2D state, 1 step, D2H state, sync; the heating is uploaded at its refreshes
        # only (first timed step here; every 60 steps in the workload), otherwise reused on the device
        g.step_rk3_host(qh, wl.dt, hh if k == 0 else None, 1, dq, dh)
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    t_e2e = max_over_ranks(t_e2e, dev, world)
    h2d = 5 * NL * 8 + (NL * 8 // e2e_steps if hh is not None else 0)   # average per step
    d2h = 5 * NL * 8

    # ---- optional: the RI-velocity diagnostic (numa_ri_*, Eq. 18-22) on the final state -----
    ri = None
    if args.ri and rank == 0:
        lev, n_lev = inputs.node_levels(mesh)
        r_max = 0.4 * min(mesh.extent[0], mesh.extent[1])
        g.ri_init(mesh.xyz, lev, n_lev, r_max, 50)
        g.ri_velocity(q)
        torch.cuda.synchronize()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(10):
            out_ri = g.ri_velocity(q)
        e1.record(stream)
        torch.cuda.synchronize()
        ri_ms = e0.elapsed_time(e1) / 10
        sc = out_ri[3].cpu().numpy()
        # per call: u, v, w, x, y, area + index per local node (centroid) and u, v, x, y + index per point
        ri_bytes = NL * (6 * 8 + 4) + mesh.n_global * (4 * 8 + 4)
        ri = {"ms_per_call": ri_ms, "u_ri": float(sc[0]), "max_horizontal_speed": float(sc[1]),
              "levels": n_lev, "strips": 50, "r_max": r_max, "alg_bytes": ri_bytes,
              "achieved_gbs": ri_bytes / (ri_ms * 1e-3) / 1e9}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    value = whole_job_gdof_per_s(NL, args.steps, world, ms * 1e-3)
    e2e_value = whole_job_gdof_per_s(NL, e2e_steps, world, t_e2e)

    # ---- roofline: the STAGE against max(t_HBM, t_FP64) ------------------------
    peak, peak_src = measured_peaks()
    has_src = wl.heating is not None
    N = mesh.N
    balg, falg = b_alg_bytes(N, has_src), f_alg_flops(N)
    if args.hyperdiffusion:
        # two Laplacian applications (12 + 36 contractions each on 4 fields) and one more 4-field DSS
        balg += 2 * hd_lap_alg_bytes() + dss_alg_bytes(N) * 4.0 / 5.0
        falg += 2 * (4 * 48 * 2.0 * (N + 1) + 4 * 60.0)
    stage_ms = ms / (3 * args.steps)
    hbm_achieved = balg * NL / (stage_ms * 1e-3) / 1e9             # GB/s, algorithmic
    fp64_achieved = falg * NL / (stage_ms * 1e-3) / 1e12           # TFLOP/s, algorithmic
    t_hbm = balg * NL / (peak * 1e9)
    t_fp64 = falg * NL / (fp64_peak * 1e12) if fp64_peak else 0.0
    bound = "hbm" if t_hbm >= t_fp64 else "fp64"
    kernels = {}
    for name, (kms, kn) in prof.items():
        kb = kernel_alg_bytes(name, N, has_src)
        per = kms / kn
        traffic, tsrc = captured_traffic(wl.name, name)
        kernels[name] = {"ms_per_launch": per, "launches_per_step": kn / prof_steps,
                         "share_of_step": kms / prof_steps / (ms / args.steps),
                         "alg_bytes_per_node": kb,
                         "achieved": kb * NL / (per * 1e-3) / 1e9 if kb else None,
                         "frac": kb * NL / (per * 1e-3) / 1e9 / peak if kb else None,
                         "traffic": traffic, "traffic_source": tsrc}
    stage_kernels = {k: v for k, v in kernels.items() if k.startswith("k_stage")}
    dom = max(stage_kernels.items(), key=lambda kv: kv[1]["share_of_step"])[0] if stage_kernels else None
    roofline = {
        "bound": bound,
        "achieved": hbm_achieved if bound == "hbm" else fp64_achieved * 1e3,
        "peak": peak if bound == "hbm" else fp64_peak * 1e3,
        "unit": "GB/s" if bound == "hbm" else "GFLOP/s",
        "frac": max(t_hbm, t_fp64) / (stage_ms * 1e-3),
        "traffic": kernels[dom]["traffic"] if dom else None,
        "traffic_source": kernels[dom]["traffic_source"] if dom else None,
        "what": "one RK stage = volume kernel + DSS kernel; frac = max(t_HBM, t_FP64) / t_stage with "
                "B_alg, F_alg of SURVEY.md 8(d) and the measured peaks",
        "stage_ms": stage_ms, "b_alg_bytes_per_node": balg, "f_alg_flops_per_node": falg,
        "peak_source": peak_src,
        "hbm": {"achieved_gbs": hbm_achieved, "peak_gbs": peak, "frac": hbm_achieved / peak},
        "fp64": {"achieved_tflops": fp64_achieved, "peak_tflops": fp64_peak,
                 "frac": fp64_achieved / fp64_peak if fp64_peak else None,
                 "peak_source": "DFMA micro-benchmark of this run (numa_measure_fp64_peak)"},
        "dominant_kernel": dom,
        "kernels": kernels,
    }

    # ---- CPU baseline: the oracle on a bounded sample, all cores and one core ------------------
    cpu = None
    if not args.no_cpu_baseline:
        swl, sample = cpu_sample_workload(config, N_arg)
        t_cpu, cores = time_oracle(swl, 5, 1)
        t_cpu1, _ = time_oracle(swl, 2, 0, threads=1)
        cpu = {"value": 5.0 * swl.mesh.n_local * 3 * 5 / t_cpu / 1e9, "unit": UNIT, "cores": cores,
               "kind": "oracle", "sample": sample + ", 5 RK3 steps after 1 warm-up",
               "single_thread": {"value": 5.0 * swl.mesh.n_local * 3 * 2 / t_cpu1 / 1e9, "cores": 1,
                                 "sample": "same sample, 2 RK3 steps"}}

    line = {
        "metric": METRIC, "value": value if finite else None, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wl.name, "N": mesh.N, "elements": [mesh.nx, mesh.ny, mesh.nz],
                   "local_nodes": NL, "integrator": "SSP-RK3 (3 RHS + 3 stage updates per step)",
                   "hyperdiffusion": bool(args.hyperdiffusion),
                   "dt": wl.dt, "multi_gpu": "replicas only" if world > 1 else "single",
                   "launch": "CUDA graph per step" if args.graph else "plain launches",
                   "l2": "inputs larger than L2" if 22 * NL * 8 > 4 * 126e6 else
                         "working set may be L2-resident (reported, not a roofline case)",
                   "heating_refreshes_in_timed_region": n_seg - 1 if heat is not None else None,
                   "finite": finite},
        "gnode_per_s": value / 5.0,
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d,
                "d2h_bytes_per_step": d2h, "steps": e2e_steps,
                "call": "numa_step_rk3_host (pinned host buffers)"},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "cpu_baseline": cpu,
    }
    if ri is not None:
        line["ri_diagnostic"] = ri
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    if not finite:
        raise SystemExit("bench.py: the state is not finite after the timed steps; no value reported")


def run_gpu_ark2(args, wl, dev, rank, world):
    """--integrator ark2: the paper's own integrator (IMEX ARK2 + matrix-free GMRES, Eq. 13) through
    numa_step_ark2.  Reported: ms per IMEX step (the quantity of the paper's Table 1), Krylov
    iterations per step, and nodal operator applications (S or L) per second."""
    import torch
    from paper_2504_08157_b200 import binding
    g = binding.Numa.from_workload(wl, device=str(dev))
    g.imex_init(args.krylov)
    q = g.state(wl.q)
    heat = None if wl.heating is None else g.state(wl.heating)
    dt = args.dt if args.dt else wl.dt
    warm = max(1, min(args.warmup, 2))
    g.step_ark2(q, dt, heat, warm, tol=args.tol, max_restarts=50)
    torch.cuda.synchronize()
    sampler = ClockSampler(dev.index or 0)
    if rank == 0:
        sampler.start(); time.sleep(0.3)
    ev0 = torch.cuda.Event(enable_timing=True); ev1 = torch.cuda.Event(enable_timing=True)
    stream = torch.cuda.current_stream()
    wall0 = time.time()
    ev0.record(stream)
    its, rel = g.step_ark2(q, dt, heat, args.steps, tol=args.tol, max_restarts=50)
    ev1.record(stream)
    torch.cuda.synchronize()
    wall1 = time.time()
    ms = max_over_ranks(ev0.elapsed_time(ev1), dev, world)
    clocks = sampler.stop(wall0, wall1) if rank == 0 else None
    finite = bool(torch.isfinite(q).all().item())
    if rank != 0:
        return
    # second pass: where the time of a step goes (CUDA events around every launch)
    g.profile(True)
    g.step_ark2(q, dt, heat, 1, tol=args.tol, max_restarts=50)
    prof = {k: {"ms_per_step": v[0], "launches_per_step": v[1]} for k, v in g.profile_read().items()}
    g.profile(False)
    NL = wl.mesh.n_local
    # operator applications per step: 3 S + 2 L for the stages, and per implicit stage one L per Krylov
    # iteration plus one per restart cycle (initial residual)
    evals = 5 * args.steps + its + 2 * args.steps
    line = {"metric": "imex_ark2_ms_per_step", "value": ms / args.steps if finite else None, "unit": "ms/step",
            "n_gpus": world, "steps": args.steps, "warmup": warm, "ms_per_step": ms / args.steps,
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "N": wl.mesh.N, "elements": [wl.mesh.nx, wl.mesh.ny, wl.mesh.nz],
                       "local_nodes": NL, "paper_dof": 5 * NL, "integrator": "IMEX ARK2 + GMRES(%d)" % args.krylov,
                       "dt": dt, "gmres_tol": args.tol, "finite": finite},
            "gmres_iterations_per_step": its / args.steps, "max_rel_residual": rel,
            "nodal_operator_evals_gdof_per_s": 5.0 * NL * evals / (ms * 1e-3) / 1e9,
            "clocks": clocks, "gpu_launches": int(g.launch_count), "kernels_of_one_step": prof,
            "context": "PAPER.md Table 1 (L399): 0.536 s per IMEX step on 4 A100 for 165,888,000 DOF (80x80x24, N=5, "
                       "dt=0.5 s); another machine, other inputs, an unknown GMRES tolerance: context, not a target"}
    print(json.dumps(line))


def kernel_alg_bytes(name, N, has_src):
    """Algorithmic bytes per local node per launch of one kernel, on SURVEY.md 8(d)'s terms (the
    stage kernels split B_alg between them; the four-call kernels count their own arrays)."""
    n_src = 2 if has_src else 0
    if name.startswith("k_rhs"):
        return 8.0 * (5 + 9 + 1 + 2 + 5)              # q, grad xi, omega, rho0/theta0 in; rhs out
    if name.startswith("k_dss") or name.startswith("k_stage_dss"):
        return dss_alg_bytes(N)                       # face nodes read + written
    if name.startswith("k_sources"):
        return 8.0 * (4 + n_src + 4 + 4)              # u,v,w,theta', heat, beta, rhs in/out (4 fields)
    if name.startswith("k_rk"):
        return 8.0 * (5 + 5 * (2.0 / 3.0) + 5 + 5)    # q0 (2/3 of stages), qs, rhs in; q out
    if name.startswith("k_stage_volume"):
        return volume_alg_bytes(N, has_src)
    if name.startswith("k_hd_lap"):
        return hd_lap_alg_bytes()
    if name.startswith("k_hd_dss"):
        return dss_alg_bytes(N) * 4.0 / 5.0
    return 0.0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="numa_b200", choices=["numa_b200", "reference"])
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ri", action="store_true", help="also time the RI-velocity diagnostic (NEXT-4) on the final state")
    ap.add_argument("--hyperdiffusion", action="store_true", help="switch the tensor hyper-diffusion on (NEXT-1)")
    ap.add_argument("--integrator", default="rk3", choices=["rk3", "ark2"],
                    help="ark2: IMEX ARK2 + GMRES through numa_step_ark2 (NEXT-3); prints its own line")
    ap.add_argument("--dt", type=float, default=0.0, help="time step for --integrator ark2 (default: the workload's)")
    ap.add_argument("--tol", type=float, default=1e-6, help="GMRES relative residual for --integrator ark2")
    ap.add_argument("--krylov", type=int, default=20, help="Krylov vectors per GMRES restart cycle")
    ap.add_argument("--graph", action="store_true",
                    help="launch every step as one CUDA graph (numa_step_rk3_graph; configs 1-2)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl != "reference":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
