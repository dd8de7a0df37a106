#!/usr/bin/env python
"""bench.py — MLUPS of the fused D3Q19 fp64 stream-collide step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
                    [--config i] [--scheme ab|aa] [--store f64|f32] [--block bx,by]

A "step" is one LBM time step over the whole grid.  How many launches that is depends on the grid (include/lbm.h,
lbm_step): D3Q19 / D3Q27 fp64 boxes without a solid mask take TWO time steps per launch (stream_collide_ab2), grids
small enough to be resident at once take all K steps in ONE launch of the persistent kernel, every other case is one
launch per step; `gpu_launches` and `roofline.steps_per_launch` say which it was.  The N=1
workload is BASELINE.json configs[3] (the headline roofline run: D3Q19 BGK fp64, 512^3 periodic
Taylor-Green vortex, tau 0.52); --config picks another one.  Prints ONE JSON line on stdout.
  value     MLUPS with the populations resident in HBM (CUDA events on the launch stream): the median of
            `repeats.n` timed segments of exactly --steps steps each
  e2e       MLUPS of the whole job through the host-buffer C-ABI calls: pinned-host rho,u -> device,
            equilibrium init, K steps, moments + diagnostics, rho,u -> pinned host
  roofline  algorithmic bytes (2*Q*8 B per cell update) / measured kernel time vs measured HBM peak (`frac`);
            beside it `floor_frac` = the bytes one launch cannot avoid moving (each population read once and written once
            per LAUNCH, whether the launch takes one step or two) / launch time / peak, and `dram_frac` = the DRAM bytes
            ncu counted for that launch (`traffic`) / launch time / peak: neither can exceed 1 by much, whatever `frac` says
  cpu_baseline  the oracle, as it stands, on this box's host cores, on a bounded sample
With --gpus N > 1 (torchrun) every rank runs an independent replica (the path does not shard in this
build); value = total cell updates of all ranks / max-over-ranks device time.
--impl reference times the CPU oracle (rank 0 only).
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "mlups_d3q19_fp64_fused_stream_collide"
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback, used only if MEASURED_PEAKS.json is absent


def log(*a):
    print(*a, file=sys.stderr, flush=True)


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons every 200 ms while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.lines, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "200", "-i", str(self.index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._pump, daemon=True)
        self.thread.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            parts = [p.strip() for p in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0]))
                smax.append(float(parts[1]))
                power.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(names, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------ helpers
def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, device copy)"
    except (OSError, KeyError, ValueError):
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md, MEASURED_PEAKS.json absent)"


def ncu_traffic(workload_name: str, scheme: str):
    """DRAM bytes per launch of the stream-collide kernel from the committed ncu --set full capture
    (profiles/traffic.csv: workload,scheme,kernel signature,dram_bytes_per_launch,capture file,notes) and where it comes
    from, or (None, None).  Capture and kernel signature are printed so that a row older than the kernel is visible."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        with open(p) as fh:
            for line in fh:
                parts = [x.strip() for x in line.split(",")]
                if len(parts) >= 5 and parts[0] == workload_name and parts[1] == scheme:
                    return float(parts[3]), {"capture": parts[4], "kernel": parts[2].replace(";", ",")}
    except (OSError, ValueError):
        pass
    return None, None


def lattice_name(Q):
    return "D2Q9" if Q == 9 else f"D3Q{Q}"


def l2_note(touched_bytes):
    """Timing rule: inputs larger than L2, or say that they are not (small configs are L2-resident by nature)."""
    gb = touched_bytes / 1e9
    if touched_bytes > 4 * 126e6:
        return f"inputs larger than L2: {gb:.2f} GB touched per step vs 126 MB L2"
    return f"NOT larger than L2: {gb:.3f} GB touched per step vs 126 MB L2 (no flush; not a roofline statement)"


def pick_sample(w, target_cells):
    """A reduced copy of workload w (same tau, fields recipe, walls, force, geometry) with at most target_cells
    cells: every length halved until it fits."""
    k = 1
    while (w.nx // k) * (w.ny // k) * (w.nz // k) > target_cells and min(w.nx, w.ny, w.nz) // k > 32:
        k *= 2
    return w.shrunk(k) if k > 1 else w


def oracle_mlups(ws, steps, warmup=1, budget_s=None):
    """Time the oracle as it stands on the sample workload ws.  With budget_s, `steps` is replaced by the
    number of steps that fills about budget_s seconds, estimated from the warm-up step(s)."""
    from oracle import Oracle, num_threads
    rho, u = ws.fields()
    o = Oracle(ws.nx, ws.ny, ws.nz, ws.Q, ws.tau, eq=ws.eq, face_kind=ws.face_kind, face_u=ws.face_u, force=ws.force,
               face_rho=ws.face_rho)
    if ws.has_geometry:
        o.set_geometry(ws.geo(), ws.wall_model)
    for face, prof in ws.face_profiles().items():
        o.set_face_velocity(face, prof)
    o.init_equilibrium(rho, u)
    t0 = time.perf_counter()
    o.step(warmup)
    if budget_s is not None:
        per_step = (time.perf_counter() - t0) / max(warmup, 1)
        steps = max(steps, min(2000, int(budget_s / max(per_step, 1e-6))))
    t0 = time.perf_counter()
    o.step(steps)
    dt = time.perf_counter() - t0
    o.close()
    return ws.N * steps / dt / 1e6, dt, num_threads(), steps


def cpu_info():
    model = "unknown"
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.lower().startswith("model name"):
                    model = line.split(":", 1)[1].strip()
                    break
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "cpu_model": model}


def oracle_mlups_subprocess(config_index, n, steps, threads):
    """The oracle on an n^3 reduced copy of config `config_index` with OMP_NUM_THREADS = threads, in a child process
    (the OpenMP runtime reads the variable once).  Returns MLUPS or None."""
    code = ("import sys, json; sys.path.insert(0, %r); import bench; from paper_2201_11330_b200 import inputs; "
            "w = inputs.config(%d); ws = w if w.nx == %d else w.scaled(%d); v, dt, cores, st = bench.oracle_mlups(ws, %d, 1); "
            "print(json.dumps({'v': v, 'dt': dt, 'cores': cores, 'steps': st}))" % (ROOT, config_index, n, n, steps))
    env = dict(os.environ, OMP_NUM_THREADS=str(threads))
    try:
        r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, env=env, timeout=300)
        return json.loads(r.stdout.strip().splitlines()[-1])
    except Exception as exc:  # noqa: BLE001 — a reported baseline, never fatal
        log(f"oracle subprocess failed: {exc}")
        return None


def cpu_baseline_block(w, budget_s=12.0):
    """S:§8(d) oracle-timing protocol, bounded to ~20 s: the oracle as it stands (never tuned for this) on the host
    cores of this box — all cores on a reduced copy of the timed workload, and all cores + ONE core on BJ config 2
    (128^3); nproc and the CPU model beside them."""
    ws = pick_sample(w, 256 ** 3)
    v, dt, cores, osteps = oracle_mlups(ws, 8, 2, budget_s=budget_s)
    out = {"value": v, "unit": "MLUPS", "cores": cores, "kind": "oracle",
           "sample": f"{ws.nx}x{ws.ny}x{ws.nz} reduced copy of {w.name} (same tau, fields recipe, walls, force, geometry), "
                     f"{osteps} oracle steps, {dt:.1f} s", **cpu_info()}
    a = oracle_mlups_subprocess(1, 128, 20, cores)
    one = oracle_mlups_subprocess(1, 128, 6, 1)
    out["cfg1_128"] = {"all_cores_mlups": a and a["v"], "all_cores": a and a["cores"], "one_core_mlups": one and one["v"],
                       "sample": "BASELINE.json configs[1] (D3Q19 128^3 Taylor-Green), 20 oracle steps on all cores, 6 on one core"}
    return out


# ------------------------------------------------------------------------------------------ reference arm
def run_reference(args, w):
    from paper_2201_11330_b200 import replicas
    rank, _, world = replicas.env_world()
    if rank != 0:
        return 0
    ws = pick_sample(w, 256 ** 3)
    t_all = time.perf_counter()
    value, dt, cores, _ = oracle_mlups(ws, args.steps, max(args.warmup, 1))
    sample = (f"{ws.nx}x{ws.ny}x{ws.nz} reduced copy of {w.name} (same tau, fields recipe, walls, force, geometry), "
              f"{args.steps} oracle steps, {dt:.1f} s")
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "MLUPS", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        # `grid` is the grid this arm actually timed (a bounded sample of the workload); `workload_grid` the workload's own
        "config": {"workload": w.name, "grid": [ws.nx, ws.ny, ws.nz], "workload_grid": [w.nx, w.ny, w.nz], "lattice": lattice_name(w.Q),
                   "tau": w.tau, "reference": "CPU oracle (oracle/lbm_oracle.cpp), host cores only"},
        "cpu_baseline": {"value": value, "unit": "MLUPS", "cores": cores, "kind": "oracle", "sample": sample, **cpu_info()},
        "e2e": {"value": value, "unit": "MLUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0, "wall_s": time.perf_counter() - t_all,
    }
    print(json.dumps(out), flush=True)
    return 0


# ------------------------------------------------------------------------------------------ GPU arm
def run_gpu(args, w):
    import numpy as np
    import torch

    from paper_2201_11330_b200 import lbm, replicas

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the CUDA library is the only implementation")
    lbm.load()
    rank, local_rank, world = replicas.init()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    scheme = {"ab": lbm.LBM_SCHEME_AB, "aa": lbm.LBM_SCHEME_AA}[args.scheme]
    store = {"f64": lbm.LBM_STORE_F64, "f32": lbm.LBM_STORE_F32}[args.store]
    stream = torch.cuda.Stream(device=dev)
    K, W = args.steps, max(args.warmup, 3)

    # synthetic inputs in pinned host memory (DESIGN.md input recipe)
    t0 = time.perf_counter()
    rho, u = w.fields()
    rho_h = torch.from_numpy(rho).pin_memory()
    u_h = torch.from_numpy(np.ascontiguousarray(u.reshape(-1))).pin_memory()
    rho_out = torch.empty(w.N, dtype=torch.float64).pin_memory()
    u_out = torch.empty(3 * w.N, dtype=torch.float64).pin_memory()
    del rho, u
    log(f"[rank {rank}] inputs {w.name} ready in {time.perf_counter() - t0:.1f} s")

    layout = lbm.LBM_LAYOUT_SOA if args.layout == "soa" else lbm.LBM_LAYOUT_ROWS
    s = lbm.Solver.from_workload(w, scheme=scheme, store=store, stream=stream, layout=layout)
    if args.block:
        s.set_block(*[int(v) for v in args.block.split(",")])
    s.set_two_step(args.two_step)
    with torch.cuda.stream(stream):
        # ---- device-resident measurement: R timed segments of EXACTLY K steps each, the median one is reported ----
        s.init_equilibrium_host(rho_h, u_h)
        d_init = s.diagnostics()
        ew0, ew1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ew0.record(stream)
        s.step(W)
        ew1.record(stream)
        torch.cuda.synchronize()
        est = replicas.max_over_ranks(ew0.elapsed_time(ew1) / 1e3 / W * K, dev)  # seconds per segment, from the warm-up
        R = args.repeats if args.repeats > 0 else max(1, min(5, int(60.0 / max(est, 1e-6))))
        sampler = ClockSampler(local_rank)
        if rank == 0:
            sampler.start()
        segs = []
        for _ in range(R):
            replicas.barrier()
            torch.cuda.synchronize()
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            l0 = s.launches
            ev0.record(stream)
            s.step(K)
            ev1.record(stream)
            torch.cuda.synchronize()
            replicas.barrier()
            segs.append((ev0.elapsed_time(ev1) / 1e3, s.launches - l0))
        clocks = sampler.stop() if rank == 0 else None
        d_end = s.diagnostics()
        # every rank reduces its segments in the same order: max over ranks per segment, then the median segment
        seg_max = [replicas.aggregate_throughput(w.N * K, t, dev)[1] for t, _ in segs]
        order = sorted(range(R), key=lambda i: seg_max[i])
        mid = order[(R - 1) // 2]
        secs, launches = segs[mid]
        secs_max = seg_max[mid]
        ups = world * w.N * K / secs_max
        steps_done = W + R * K

        # ---- end to end through the host-buffer C-ABI calls ----------------------------------------
        def e2e_run(nsteps):
            torch.cuda.synchronize()
            replicas.barrier()
            t0 = time.perf_counter()
            s.init_equilibrium_host(rho_h, u_h)
            s.step(nsteps)
            d = lbm.lbm_moments_host(s.h, rho_out, u_out, True)  # synchronises
            dt = time.perf_counter() - t0
            replicas.barrier()
            _, dt_max, e_ups = replicas.aggregate_throughput(w.N * nsteps, dt, dev)
            return d, dt_max, e_ups

        d_e2e, e2e_max, e2e_ups = e2e_run(K)
        e2e_cfg = None
        if K != w.steps and est / K * w.steps <= 30.0:  # also at the step count BASELINE.json gives the config
            _, t_cfg, ups_cfg = e2e_run(w.steps)
            e2e_cfg = {"steps": w.steps, "value": ups_cfg / 1e6, "seconds": t_cfg}
    s.close()

    if rank != 0:
        replicas.finalize()
        return 0

    # S:§8d algorithmic bytes per lattice update: every population read once and written once (+ the 4-byte
    # link mask of the geometry variant)
    bytes_per_cell = 2 * w.Q * (4 if args.store == "f32" else 8) + (4 if w.has_geometry else 0)
    ms_per_launch = secs / launches * 1e3
    # algorithmic bytes of the timed region / its duration (a launch covers K / launches time steps: 1 for the large
    # grids, all K for the small ones that run in the persistent kernel)
    achieved = bytes_per_cell * w.N * K / secs / 1e9
    peak, peak_src = measured_peak()
    # steps in pairs (stream_collide_ab2; an odd K ends with one single step) vs all K in one launch of the persistent kernel
    paired = K > 2 and 2 * launches in (K, K + 1)
    traffic, traffic_src = ncu_traffic(w.name, args.scheme + ("2" if paired else "") + ("" if args.store == "f64" else "_f32"))
    # What one launch cannot avoid moving through HBM: every stored population read once and written once per LAUNCH —
    # the same bytes for a one-step and for a two-step launch.  The persistent kernel keeps a small grid in the L2 over
    # all K steps, so it has no HBM floor.
    persistent = launches < K and not paired
    floor_bytes = None if persistent else float(bytes_per_cell * w.N)
    floor_frac = None if persistent else floor_bytes / (ms_per_launch * 1e-3) / 1e9 / peak
    dram_frac = None if (persistent or traffic is None) else traffic / (ms_per_launch * 1e-3) / 1e9 / peak
    out = {
        "metric": METRIC, "value": ups / 1e6, "unit": "MLUPS", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": secs_max / K * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "lattice": lattice_name(w.Q), "collision": "BGK", "tau": w.tau,
                   "equilibrium": "Eq. 5" if w.eq else "Eq. 2", "geometry": ("none" if not w.has_geometry else
                                                                              ("nodal" if w.wall_model else "halfway") + " walls, solid mask"),
                   "scheme": args.scheme, "storage": args.store, "layout": "f[z][y][a][x]" if args.layout == "rows" else "f[a][z][y][x]",
                   "parallelism": "1 GPU" if world == 1 else f"{world} independent replicas",
                   "l2": l2_note(bytes_per_cell * w.N)},
        "clocks": clocks,
        "e2e": {"value": e2e_ups / 1e6, "unit": "MLUPS", "h2d_bytes_per_step": 32 * w.N / K, "d2h_bytes_per_step": (32 * w.N + 64) / K,
                "what": "lbm_init_equilibrium_host(pinned rho,u: z-chunked copies overlapped with the init kernel) + lbm_step(K) + "
                        "lbm_moments_host(pinned rho,u,diagnostics: chunked likewise), host wall clock",
                "seconds": e2e_max, "at_config_steps": e2e_cfg},
        "gpu_launches": launches,
        "repeats": {"n": R, "reported": "median segment", "mlups": [world * w.N * K / t / 1e6 for t in seg_max]},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                     "traffic_source": traffic_src,
                     "frac_note": (("above 1: `achieved` counts the ALGORITHMIC bytes of one-step-per-pass streaming (2*Q*8 B per update, SURVEY.md 8d); "
                                    "this kernel takes two steps per pass and moves about half of them (see `traffic`)") if paired else
                                   ("above 1: the contract's denominator is a plain device copy (MEASURED_PEAKS.json), not a hardware limit; "
                                    "see frac_of_nominal_8TBs")) if achieved > peak else None,
                     "kernel": "stream_collide_" + args.scheme + ("2 (two steps per launch)" if paired else "_persistent" if launches < K else ""), "bytes_per_cell_update": bytes_per_cell, "ms_per_launch": ms_per_launch, "steps_per_launch": K / launches,
                     "peak_source": peak_src, "frac_of_nominal_8TBs": achieved / 8000.0,
                     "floor_bytes_per_launch": floor_bytes, "floor_frac": floor_frac, "dram_frac": dram_frac,
                     "bound_note": ("two steps per pass: the kernel runs at floor_frac of its own HBM floor (one read + one write of "
                                    "every population per launch); what holds it below 1 is latency / shared-memory staging, not DRAM "
                                    "bandwidth (profiles/README.md)") if paired else
                                   ("all steps in one launch on an L2-resident grid: no HBM floor, not a roofline statement" if persistent else None)},
        "checks": {"mass_drift_rel": abs(d_end[0] - d_init[0]) / d_init[0], "nonfinite_cells": d_end[7],
                   "kinetic_energy_ratio": d_end[4] / d_init[4] if d_init[4] else None, "e2e_mass": d_e2e[0]},
    }
    # ---- the oracle on this box's host cores, on a bounded sample (reported baseline, not the target) ----
    if world == 1 and not args.no_cpu_baseline:
        out["cpu_baseline"] = cpu_baseline_block(w)
    else:
        out["cpu_baseline"] = None
    print(json.dumps(out), flush=True)
    replicas.finalize()
    return 0


# ------------------------------------------------------------------------------------------ z-slab arm
def run_gpu_slabs(args, w):
    """--decomp zslab: ONE box cut into z-slabs.  Under torchrun: one slab per rank / GPU,
    halo planes filled by the neighbours' fused kernels over NVLink peer memory (strong scaling: the box is fixed).
    In a single process: --slabs R slabs on this GPU (measures what the slab path costs against the undivided box)."""
    import numpy as np
    import torch

    from paper_2201_11330_b200 import lbm, replicas, slabs

    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the CUDA library is the only implementation")
    lbm.load()
    rank, local_rank, world = replicas.init()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    store = {"f64": lbm.LBM_STORE_F64, "f32": lbm.LBM_STORE_F32}[args.store]
    K, W = args.steps, max(args.warmup, 3)
    if world > 1:
        stream = torch.cuda.Stream(device=dev)
        g = slabs.SlabSolver(w, rank, world, store=store, stream=stream)
        own_cells, nslabs = g.N_own, world
        sync = stream.synchronize
        with torch.cuda.stream(stream):
            g.init_equilibrium()
        diag = lambda: g.global_diagnostics(dev)
        rec = lambda ev: ev.record(stream)
    else:
        g = slabs.SlabGroup(w, args.slabs, store=store)
        own_cells, nslabs = w.N, args.slabs
        sync = g.synchronize
        g.init_equilibrium()
        diag = g.diagnostics
        rec = None
    sync()
    replicas.barrier()
    d_init = diag()
    g.step(W)
    sync()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    replicas.barrier()
    torch.cuda.synchronize()
    l0 = g.launches
    if rec is not None:
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        rec(ev0)
        g.step(K)
        rec(ev1)
        sync()
        secs = ev0.elapsed_time(ev1) / 1e3
    else:
        # several streams: an event pair on every slab's stream, the job time is first start -> last end
        evs = []
        for s in g.slabs:
            e0 = torch.cuda.Event(enable_timing=True)
            e0.record(s.torch_stream)
            evs.append([e0, None])
        g.step(K)
        for s, pair in zip(g.slabs, evs):
            pair[1] = torch.cuda.Event(enable_timing=True)
            pair[1].record(s.torch_stream)
        sync()
        first = evs[0][0]
        secs = max(first.elapsed_time(p[1]) for p in evs) / 1e3
    replicas.barrier()
    launches = g.launches - l0
    clocks = sampler.stop() if rank == 0 else None
    d_end = diag()
    units, secs_max, ups = replicas.aggregate_throughput(own_cells * K, secs, dev)
    g.close()
    if rank != 0:
        replicas.finalize()
        return 0
    bytes_per_cell = 2 * w.Q * (4 if args.store == "f32" else 8) + (4 if w.has_geometry else 0)
    peak, peak_src = measured_peak()
    achieved = bytes_per_cell * units / secs_max / 1e9 / world  # per GPU
    halo_dirs = sum(1 for ez in _EZ[w.Q] if ez == 1)
    out = {
        "metric": METRIC, "value": ups / 1e6, "unit": "MLUPS", "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": secs_max / K * 1e3, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "lattice": lattice_name(w.Q), "collision": "BGK", "tau": w.tau,
                   "scheme": "ab", "storage": args.store,
                   "parallelism": f"z-slabs: {nslabs} slab(s) on {world} GPU(s), fused halo push over peer memory",
                   "halo_bytes_per_step_per_cut": 2 * halo_dirs * w.nx * w.ny * (4 if args.store == "f32" else 8),
                   "l2": l2_note(bytes_per_cell * w.N)},
        "clocks": clocks, "e2e": None, "gpu_launches": launches,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                     "kernel": "stream_collide_ab<..., SLAB>", "bytes_per_cell_update": bytes_per_cell, "peak_source": peak_src,
                     "note": "per GPU: algorithmic bytes of all slabs / job time / GPUs"},
        "checks": {"mass_drift_rel": abs(d_end[0] - d_init[0]) / d_init[0], "nonfinite_cells": d_end[7]},
        "cpu_baseline": None,
    }
    print(json.dumps(out), flush=True)
    replicas.finalize()
    return 0


# e_z of every direction in the library's order (R4), only to count the populations that cross a z cut
_EZ = {9: [0] * 9,
       19: [0, -1, 0, 1, 0, -1, 0, 1, -1, 0, 1, -1, 0, 1, 0, -1, 0, 1, 0],
       27: [-1, 0, 1] * 9}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3,
                    help="index into BASELINE.json configs (default 3 = 512^3 headline); 5 / 8 = the paper's sphere case (periodic box / its own "
                         "boundaries), 6 / 7 = its 2-D channel-cylinder cases")
    ap.add_argument("--scheme", default="ab", choices=["ab", "aa"])
    ap.add_argument("--store", default="f64", choices=["f64", "f32"])
    ap.add_argument("--block", default="", help="bx,by block shape override")
    ap.add_argument("--layout", default="rows", choices=["rows", "soa"],
                    help="internal population layout: f[z][y][a][x] (default) or plain structure of arrays f[a][z][y][x]")
    ap.add_argument("--two-step", type=int, default=1, choices=[0, 1],
                    help="lbm_set_two_step: 0 one pass through HBM per step everywhere; 1 (default) fp64 A/B without a mask takes two steps per pass where the grid is large enough")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--repeats", type=int, default=0,
                    help="timed segments of --steps steps each, the median is reported (default: 5, fewer if 5 would exceed a minute)")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "zslab"],
                    help="--gpus N > 1: N independent replicas (default; BASELINE.json: no sharding) or ONE box cut into z-slabs")
    ap.add_argument("--slabs", type=int, default=2, help="--decomp zslab in a single process: slabs on this one GPU")
    args = ap.parse_args()
    from paper_2201_11330_b200 import inputs
    w = inputs.config(args.config)
    if args.impl == "reference":
        return run_reference(args, w)
    if args.decomp == "zslab":
        return run_gpu_slabs(args, w)
    return run_gpu(args, w)


if __name__ == "__main__":
    sys.exit(main())
