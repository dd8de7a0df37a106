#!/usr/bin/env python
"""bench.py — MLUPS of the fused D3Q19 fp64 stream-collide step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
                    [--config i] [--scheme ab|aa] [--store f64|f32] [--block bx,by]

A "step" is one LBM time step = one launch of the fused kernel over the whole grid.  The N=1
workload is BASELINE.json configs[3] (the headline roofline run: D3Q19 BGK fp64, 512^3 periodic
Taylor-Green vortex, tau 0.52); --config picks another one.  Prints ONE JSON line on stdout.
  value     MLUPS with the populations resident in HBM (CUDA events on the launch stream)
  e2e       MLUPS of the whole job through the host-buffer C-ABI calls: pinned-host rho,u -> device,
            equilibrium init, K steps, moments + diagnostics, rho,u -> pinned host
  roofline  algorithmic bytes (2*Q*8 B per cell update) / measured kernel time vs measured HBM peak
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
    (profiles/traffic.csv: workload,scheme,kernel,dram_bytes_per_launch,source), or None."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        with open(p) as fh:
            for line in fh:
                parts = [x.strip() for x in line.split(",")]
                if len(parts) >= 4 and parts[0] == workload_name and parts[1] == scheme:
                    return float(parts[3])
    except (OSError, ValueError):
        pass
    return None


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
        "config": {"workload": w.name, "grid": [w.nx, w.ny, w.nz], "lattice": lattice_name(w.Q), "tau": w.tau,
                   "reference": "CPU oracle (oracle/lbm_oracle.cpp), host cores only"},
        "cpu_baseline": {"value": value, "unit": "MLUPS", "cores": cores, "kind": "oracle", "sample": sample},
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
    with torch.cuda.stream(stream):
        # ---- device-resident measurement -------------------------------------------------------
        s.init_equilibrium_host(rho_h, u_h)
        d_init = s.diagnostics()
        s.step(W)
        torch.cuda.synchronize()
        sampler = ClockSampler(local_rank)
        if rank == 0:
            sampler.start()
        replicas.barrier()
        torch.cuda.synchronize()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = s.launches
        ev0.record(stream)
        s.step(K)
        ev1.record(stream)
        torch.cuda.synchronize()
        replicas.barrier()
        launches = s.launches - l0
        secs = ev0.elapsed_time(ev1) / 1e3
        clocks = sampler.stop() if rank == 0 else None
        d_end = s.diagnostics()
        units, secs_max, ups = replicas.aggregate_throughput(w.N * K, secs, dev)

        # ---- end to end through the host-buffer C-ABI calls ----------------------------------------
        torch.cuda.synchronize()
        replicas.barrier()
        t0 = time.perf_counter()
        s.init_equilibrium_host(rho_h, u_h)
        s.step(K)
        d_e2e = lbm.lbm_moments_host(s.h, rho_out, u_out, True)  # synchronises
        e2e_secs = time.perf_counter() - t0
        replicas.barrier()
        _, e2e_max, e2e_ups = replicas.aggregate_throughput(w.N * K, e2e_secs, dev)
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
    traffic = ncu_traffic(w.name, args.scheme + ("" if args.store == "f64" else "_f32"))
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
                "what": "lbm_init_equilibrium_host(pinned rho,u) + lbm_step(K) + lbm_moments_host(pinned rho,u,diagnostics), host wall clock",
                "seconds": e2e_max},
        "gpu_launches": launches,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
                     "kernel": "stream_collide_" + args.scheme + ("_persistent" if launches < K else ""), "bytes_per_cell_update": bytes_per_cell, "ms_per_launch": ms_per_launch, "steps_per_launch": K / launches,
                     "peak_source": peak_src, "frac_of_nominal_8TBs": achieved / 8000.0},
        "checks": {"mass_drift_rel": abs(d_end[0] - d_init[0]) / d_init[0], "nonfinite_cells": d_end[7],
                   "kinetic_energy_ratio": d_end[4] / d_init[4] if d_init[4] else None, "e2e_mass": d_e2e[0]},
    }
    # ---- the oracle on this box's host cores, on a bounded sample (reported baseline, not the target) ----
    if world == 1 and not args.no_cpu_baseline:
        ws = pick_sample(w, 256 ** 3)
        v, dt, cores, osteps = oracle_mlups(ws, 8, 2, budget_s=15.0)
        out["cpu_baseline"] = {"value": v, "unit": "MLUPS", "cores": cores, "kind": "oracle",
                               "sample": f"{ws.nx}x{ws.ny}x{ws.nz} reduced copy of {w.name} (same tau, fields recipe, walls, force, "
                                         f"geometry), {osteps} oracle steps, {dt:.1f} s"}
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
    ap.add_argument("--no-cpu-baseline", action="store_true")
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
