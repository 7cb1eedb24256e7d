#!/usr/bin/env python
"""bench.py -- throughput of the LBM-IMB-DEM hot path on B200 (BASELINE.json:metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3|C4|C2|C5] [--impl reference]

One "step" is one pass of the whole hot path over the workload (SURVEY.md 8(a) rows a1-a3, and a4
where the configuration has moving particles): lbmimb_map_particles -> lbmimb_step(1) ->
lbmimb_reduce_particle_forces [-> lbmimb_dem_step for C5].  Default workload: C3
(BASELINE.json:configs[2], D3Q19 fp64 256x1008x256, 24,600 spheres), the configuration the
north_star target (>= 70 % of HBM bandwidth for the fused D3Q19 step) is quoted on.

`value`   = lattice updates of all ranks / max-over-ranks device time, inputs resident in HBM.
`e2e`     = the same through the C-ABI with HOST buffers: every step uploads the particle state from
            pinned host memory (lbmimb_set_particles) and reads force/torque back to the host.
`roofline`= the fused collide-stream kernel alone: algorithmic bytes (2*Q*8 + 1 + 4 per node) / its
            launch duration measured with CUDA events on the launching stream inside the timed region.
`cpu_baseline` = the CPU oracle (tests' reference, never tuned) timed on a bounded sample.
N > 1: "replicas only": N independent replicas, one per GPU, no data-path collective.
`--impl reference` times the oracle itself (rank 0 only).
The default run (workload C3) also measures C4, BASELINE.json's "Throughput run" (configs[3]), after the C3
handle is destroyed (the two do not fit one GPU together), and reports it as `secondary` in the same line.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fp64 LBM-IMB MLUPS on 1 B200 and % of HBM roofline (bytes/update counted)"
UNIT = "MLUPS"


def profiled_traffic(workload, streaming):
    """dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the fused kernel, from the committed
    `ncu --set full` capture of this round (profiles/r2_traffic.csv names the capture, the kernel and the
    commit it was taken at; commands in profiles/README.md).  Not measured in this run: None where no capture
    exists for the combination."""
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "r2_traffic.csv"), newline="") as fh:
            for rec in csv.DictReader(fh):
                if rec["workload/streaming"] == "%s/%s" % (workload, streaming):
                    return int(rec["dram_bytes_per_launch"]), "profiles/r2_traffic.csv (%s, commit %s)" % (
                        rec["kernel"], rec["commit"])
    except Exception:
        pass
    return None, None


def measured_peak_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clocks and throttle reasons with nvidia-smi DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index = index
        self.rows = []
        self.proc = None
        self.t0 = self.t1 = None

    def mark_begin(self):
        self.t0 = time.time()

    def mark_end(self):
        self.t1 = time.time()

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            parts = [p.strip() for p in line.split(",")]
            if len(parts) >= 7:
                self.rows.append((time.time(), parts))

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        inside = [r for (t, r) in self.rows if self.t0 is None or (self.t0 <= t <= (self.t1 or t) + 0.1)]
        if not inside:          # region shorter than one sampling period: the sample nearest to it
            inside = [r for (t, r) in self.rows[-1:]]
        for r in inside:
            try:
                sm.append(float(r[0]))
                mx.append(float(r[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def get_workload(name):
    from paper_1011_2613_b200 import inputs
    return inputs.FULL[name]()


def oracle_sample(name, target_s=15.0, max_steps=50):
    """The oracle as it stands, timed on a bounded sample of the workload: a y-slab of the lattice with
    the same recipe and solid fraction.  Returns (mlups, cores, description, seconds)."""
    import oracle as orc
    from paper_1011_2613_b200 import inputs
    if name == "C3":
        w = inputs.c3(n=(256, 48, 256), P=1171, steps=1)
    elif name == "C4":
        w = inputs.c4(n=(8192, 512), grid=(540, 34), steps=1)
    elif name == "C2":
        w = inputs.c2(n=(1024, 1024), P=3500, steps=1)
    elif name == "C5":
        w = inputs.c5(n=(128, 128, 128), P=1024, steps=1)
    elif name == "P3D":
        w = inputs.p3d(n=(256, 96, 256), grid=(16, 6, 16), steps=1)      # the paper's pitch of 16
    elif name == "P2D":
        w = inputs.p2d(n=(2048, 1024), grid=(72, 36), steps=1)           # the paper's pitch of 28.44
    else:
        raise KeyError(name)
    f = orc.init(w.dim, w.n)
    pos, vel, om = w.pos.copy(), w.vel.copy(), w.omega.copy()

    def one_step(f, pos, vel, om):
        if w.dem:
            d = w.dem
            f, pos, vel, om, _ = orc.coupled_step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, pos, vel, om,
                                                  w.radius, w.mass, d["kn"], d["restitution"], d["g_particle"], d["dt"])
            return f, pos, vel, om
        eps, pid = orc.map_particles(w.dim, w.n, w.bc, w.subsamples, pos, w.radius)
        f, s = orc.step(w.dim, w.n, w.bc, w.tau, w.g_fluid, w.subsamples, f, eps_cnt=eps, pid=pid, pos=pos, vel=vel,
                        omega=om, want_s=True)
        orc.forces(w.dim, w.n, w.bc, s, pid, pos)
        return f, pos, vel, om

    f, pos, vel, om = one_step(f, pos, vel, om)          # warm-up (page faults, OpenMP pool)
    t0 = time.perf_counter()
    steps = 0
    while steps < max_steps and (steps < 2 or time.perf_counter() - t0 < target_s):
        f, pos, vel, om = one_step(f, pos, vel, om)
        steps += 1
    dt = time.perf_counter() - t0
    desc = "%s recipe on a %s slab (%d nodes, %d particles), %d whole-path steps" % (
        name, "x".join(str(v) for v in w.n), w.nodes, w.P, steps)
    return w.nodes * steps / dt / 1e6, orc.num_threads(), desc, dt


def run_reference(args):
    """--impl reference: the CPU oracle on the same config / metric (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    per_step = max(2.0, 60.0 / max(1, args.steps + args.warmup))
    vals = []
    desc = cores = None
    for it in range(args.warmup + args.steps):
        v, cores, desc, _ = oracle_sample(args.workload, target_s=min(per_step, 10.0), max_steps=4)
        if it >= args.warmup:
            vals.append(v)
    value = float(np.mean(vals))
    w = {"C3": (256, 1008, 256), "C4": (8192, 32768), "C2": (1024, 4096), "C5": (128, 512, 128),
         "P2D": (15360, 61440), "P3D": (512, 2016, 512)}[args.workload]
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": None, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "lattice": list(w), "note": "CPU oracle on a bounded sample"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def measure(args, name, lb, replicas, torch, rank, world, local, streaming, want_e2e, want_coupled, sampler_index):
    """Times one workload on this rank's GPU; returns the pieces of the JSON line (rank 0) or None."""
    w = get_workload(name)
    lat = lb.from_workload(w, device=local, map_mode=lb.MAP_TABLE if args.map_mode == "table" else lb.MAP_SAMPLING,
                           streaming=lb.STREAM_AA if streaming == "aa" else lb.STREAM_AB)
    dem = w.dem
    if args.neighbor_mode == "verlet":
        lat.set_neighbor_mode(lb.NEIGHBOR_VERLET, args.skin, args.every)
    Q = w.Q
    bytes_per_node = 2 * Q * 8 + 1 + 4        # distributions + eps count + particle id
    N = w.nodes

    def whole_step():
        lat.map_particles()
        lat.step(1)
        lat.reduce_particle_forces(to_host=False)
        if dem:
            lat.dem_step(dem["kn"], dem["restitution"], dem["g_particle"], dem["dt"])

    sampler = ClockSampler(sampler_index)
    if rank == 0:
        sampler.start()          # nvidia-smi needs a few hundred ms to deliver its first sample
    for _ in range(args.warmup):
        whole_step()
    lat.synchronize()

    # ---- timed region: device-resident inputs -------------------------------------------------
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(5)] for _ in range(args.steps)]
    replicas.barrier()
    torch.cuda.synchronize()
    sampler.mark_begin()
    launches0 = lat.launch_count()
    t_begin = lat.time()
    for k in range(args.steps):
        ev[k][0].record()
        lat.map_particles()
        ev[k][1].record()
        lat.step(1)
        ev[k][2].record()
        lat.reduce_particle_forces(to_host=False)
        ev[k][3].record()
        if dem:
            lat.dem_step(dem["kn"], dem["restitution"], dem["g_particle"], dem["dt"])
        ev[k][4].record()
    torch.cuda.synchronize()
    sampler.mark_end()
    replicas.barrier()
    launches = lat.launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    total_ms = ev[0][0].elapsed_time(ev[-1][4])
    seg = np.array([[e[i].elapsed_time(e[i + 1]) for i in range(4)] for e in ev])
    kern_ms = float(seg[:, 1].mean())
    units, ms_max = replicas.aggregate(float(N) * args.steps, total_ms)
    value = replicas.mlups(units, ms_max)

    # ---- end to end through host buffers ------------------------------------------------------
    e2e = None
    if want_e2e:
        P, D, nt = w.P, w.dim, (1 if w.dim == 2 else 3)
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
        hpos, hvel, hom, hrad, hmass = pin(w.pos), pin(w.vel), pin(w.omega), pin(w.radius), pin(w.mass)
        hF = torch.empty((D, P), dtype=torch.float64).pin_memory().numpy()
        hT = torch.empty((nt, P), dtype=torch.float64).pin_memory().numpy()
        h2d = (hpos.nbytes + hvel.nbytes + hom.nbytes + hrad.nbytes + hmass.nbytes)
        d2h = hF.nbytes + hT.nbytes

        def e2e_step():
            if dem:
                p_, v_, o_ = lat.get_particles()          # moving particles: the host owns the state
                hpos[...], hvel[...], hom[...] = p_, v_, o_
            lat.set_particles(hpos, hvel, hom, hrad, hmass)
            lat.map_particles()
            lat.step(1)
            lat.reduce_particle_forces(out=(hF, hT))
            if dem:
                lat.dem_step(dem["kn"], dem["restitution"], dem["g_particle"], dem["dt"])

        for _ in range(3):
            e2e_step()
        replicas.barrier()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(args.steps):
            e2e_step()
        b.record()
        torch.cuda.synchronize()
        replicas.barrier()
        e_units, e_ms = replicas.aggregate(float(N) * args.steps, a.elapsed_time(b))
        if dem:
            h2d, d2h = h2d, d2h + hpos.nbytes + hvel.nbytes + hom.nbytes
        e2e = {"value": replicas.mlups(e_units, e_ms), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
               "d2h_bytes_per_step": int(d2h), "ms_per_step": e_ms / args.steps}

    lat.synchronize()
    coupled = None
    if dem and want_coupled:      # the same K steps through ONE call: launches replayed from a CUDA graph
        dargs = (dem["kn"], dem["restitution"], dem["g_particle"], dem["dt"])
        lat.run_coupled(5, *dargs)
        replicas.barrier()
        torch.cuda.synchronize()
        l0 = lat.launch_count()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        lat.run_coupled(args.steps, *dargs)
        b.record()
        torch.cuda.synchronize()
        replicas.barrier()
        c_units, c_ms = replicas.aggregate(float(N) * args.steps, a.elapsed_time(b))
        coupled = {"value": replicas.mlups(c_units, c_ms), "unit": UNIT, "ms_per_step": c_ms / args.steps,
                   "call": "lbmimb_run_coupled(%d)" % args.steps,
                   "launches_per_step": (lat.launch_count() - l0) / float(args.steps)}
    diag = diag_ms = None
    if dem:                        # the Figs. 5/7 time-series sample: one device reduction per output step
        lat.map_particles()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        dd = lat.diagnostics()
        b.record()
        torch.cuda.synchronize()
        diag_ms = a.elapsed_time(b)
        diag = {"slip_y": float(dd["slip"][1]), "drag_y": float(dd["drag"][1]), "t": lat.time()}
    nl_info = lat.fetch_neighbor_list()[2] if (dem and args.neighbor_mode == "verlet") else None
    version = lb.version()
    lat.close()
    del lat
    torch.cuda.empty_cache()
    if rank != 0:
        return None

    peak, peak_src = measured_peak_gbs()
    achieved = bytes_per_node * N / (kern_ms * 1e-3) / 1e9
    traffic, traffic_src = profiled_traffic(name, streaming)
    roof = {"bound": "hbm", "kernel": ("collide_stream_aa_kernel<%d,IMB,forces,even|odd>" if streaming == "aa"
                                       else "collide_stream_kernel<%d,IMB,forces>") % w.dim, "achieved": achieved,
            "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
            "peak_source": peak_src, "bytes_per_node": bytes_per_node, "nodes_per_launch": N, "kernel_ms": kern_ms,
            "kernel_mlups": N / (kern_ms * 1e-3) / 1e6, "frac_of_nominal_8TBs": achieved / 8000.0,
            "kernel_share_of_step": kern_ms / (total_ms / args.steps),
            "whole_step_frac": bytes_per_node * N / (ms_max / args.steps * 1e-3) / 1e9 / peak}
    if streaming == "aa":      # the AA array is in its swapped layout after an odd number of steps
        odd = (t_begin + np.arange(args.steps)) % 2 == 1
        roof["kernel_ms_even_step"] = float(seg[~odd, 1].mean()) if (~odd).any() else None
        roof["kernel_ms_odd_step"] = float(seg[odd, 1].mean()) if odd.any() else None
    return {"value": value, "ms_per_step": ms_max / args.steps,
            "config": {"workload": name, "lattice": list(w.n), "Q": Q, "particles": w.P, "tau": w.tau,
                       "bc": list(w.bc), "map_mode": args.map_mode, "streaming": streaming,
                       "step": "map_particles + step(1) + reduce_particle_forces" +
                       (" + dem_step" if dem else ""),
                       "neighbor_mode": (args.neighbor_mode + (" skin=%g every=%d" % (args.skin, args.every)
                                                               if args.neighbor_mode == "verlet" else "")) if dem else None,
                       "parallelism": "replicas x%d" % world,
                       "env": {k: os.environ[k] for k in ("LBMIMB_NO_GRAPH",) if k in os.environ},
                       "l2": "inputs (%.1f GB of distributions) exceed the 126 MB L2; no flush needed" %
                       ((1 if streaming == "aa" else 2) * Q * N * 8 / 1e9)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roof,
            "breakdown_ms": {"map_particles": float(seg[:, 0].mean()), "step": kern_ms,
                             "reduce_particle_forces": float(seg[:, 2].mean()),
                             "dem_step": float(seg[:, 3].mean()) if dem else 0.0, "diagnostics_once": diag_ms},
            "diagnostics": diag, "neighbor_list": nl_info, "coupled_api": coupled, "version": version}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--workload", default="C3", choices=["C2", "C3", "C4", "C5", "P2D", "P3D"],
                    help="C2..C5 = BASELINE.json configs; P2D / P3D = the paper's own suspensions at full size "
                         "(PAPER.md:117, Table 2; coupled with DEM; P3D needs --streaming aa, the default for it)")
    ap.add_argument("--impl", default="lbmimb", choices=["lbmimb", "reference"])
    ap.add_argument("--map-mode", default="sampling", choices=["sampling", "table"],
                    help="a1 variant: sub-cell sampling (BASELINE.json configs) or the paper's table look-up")
    ap.add_argument("--streaming", default=None, choices=["ab", "aa"],
                    help="a2 variant: pull with two arrays (A-B) or in-place AA-pattern on one array")
    ap.add_argument("--neighbor-mode", default="cells", choices=["cells", "verlet"],
                    help="a4 variant (coupled workloads C5 / P2D / P3D): cell list rebuilt every step, or the paper's "
                         "neighbour lists (PAPER.md:69, DESIGN.md R19)")
    ap.add_argument("--skin", type=float, default=1.0, help="neighbour-list skin in lattice units")
    ap.add_argument("--every", type=int, default=100, help="neighbour lists are at most this many steps old")
    ap.add_argument("--coupled-api", action="store_true",
                    help="coupled workloads: also time lbmimb_run_coupled (the same loop replayed from a CUDA graph)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-secondary", action="store_true",
                    help="default workload only: skip the second measurement on C4 (BASELINE.json's 'Throughput run')")
    args = ap.parse_args()
    if args.streaming is None:      # 2 x 80.3 GB of distributions do not fit one B200: P3D runs in place
        args.streaming = "aa" if args.workload == "P3D" else "ab"
    if args.impl == "reference":
        return run_reference(args)
    if args.warmup < 3:
        args.warmup = 3

    import torch
    from paper_1011_2613_b200 import binding as lb, replicas
    rank, world, local = replicas.init_from_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the lbmimb path has no CPU fallback")
    torch.cuda.set_device(local)
    main_res = measure(args, args.workload, lb, replicas, torch, rank, world, local, args.streaming,
                       not args.no_e2e, args.coupled_api, local)
    second = None
    if args.workload == "C3" and args.streaming == "ab" and not args.no_secondary:
        second = measure(args, "C4", lb, replicas, torch, rank, world, local, "ab", False, False, local)
    if rank != 0:
        replicas.shutdown()
        return 0
    cpu = None
    if not args.no_cpu_baseline:
        v, cores, desc, secs = oracle_sample(args.workload)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "seconds": secs}
    line = {"metric": METRIC, "value": main_res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": main_res["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic"}
    for k in ("config", "clocks", "e2e", "gpu_launches", "roofline"):
        line[k] = main_res[k]
    line["cpu_baseline"] = cpu
    for k in ("breakdown_ms", "diagnostics", "neighbor_list", "coupled_api", "version"):
        line[k] = main_res[k]
    if second is not None:      # BASELINE.json configs[3], measured in the same invocation with its own clock sample
        line["secondary"] = {"workload": "C4", "metric": METRIC, "unit": UNIT, "value": second["value"],
                             "ms_per_step": second["ms_per_step"], "steps": args.steps, "warmup": args.warmup,
                             "roofline": second["roofline"], "breakdown_ms": second["breakdown_ms"],
                             "clocks": second["clocks"], "gpu_launches": second["gpu_launches"],
                             "config": second["config"]}
    print(json.dumps(line))
    replicas.shutdown()
    return 0


if __name__ == "__main__":
    sys.exit(main())
