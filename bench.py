#!/usr/bin/env python
"""bench.py -- GLUPS of the TSLB + Allen-Cahn step on one B200 (BASELINE.json metric).

A "step" is one tslb_step(1): every stage of SURVEY.md 8(a) over the whole 256^3 head-on
collision domain (BASELINE.json configs[3], synthetic, seeded).  `value` is timed with CUDA
events on the solver's stream with the state resident in HBM; `e2e` goes through the C ABI's
host-buffer calls (tslb_init_host -> tslb_step -> tslb_get_host) with the copies inside the
timed region.  Multi-GPU = independent replicas: weak scaling, no
data-path collective.  `--impl reference` times the CPU oracle on a bounded slab of the same
workload (it is a deliberately plain program: context, not a target).
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
sys.path.insert(0, ROOT)

METRIC = "GLUPS per B200 (fp32/fp64) and % of HBM roofline on 256^3 droplet domain"
STATE_SCALARS = 14                      # p*, u(3), Ahat(6), a(3), phi  -> 28 s bytes per update
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel on the 256^3
# workload, from the ncu --set full captures summarised in profiles/r1d_kernels_f64.txt and
# profiles/r1c_kernels_f32.txt
NCU_TRAFFIC = {("f64", "stream_collide"): 2.005029e9 + 2.102657e9,
               ("f32", "stream_collide"): 0.977743e9 + 1.031000e9}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--size", type=int, default=256, help="cube edge of the domain")
    ap.add_argument("--workload", default="collision", choices=["collision", "emulsion"],
                    help="collision = BASELINE.json configs[3] (the graded one); emulsion = "
                         "configs[4], the throughput sweep (use --size 384 for f64, 512 for f32)")
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"],
                    help="precision of the headline value (the other one is reported beside it)")
    ap.add_argument("--naive", action="store_true", help="time the validation kernels instead")
    ap.add_argument("--variant", type=int, default=0, help="tuning variant (flags bits 8-15)")
    ap.add_argument("--k1variant", type=int, default=0, help="Allen-Cahn tuning variant (bits 16-19)")
    ap.add_argument("--generic", action="store_true", help="force the wall-capable tiled kernel")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--only", default=None, choices=[None, "f64", "f32"],
                    help="measure a single precision only (used for ncu captures)")
    return ap.parse_args()


def peaks():
    """Roofline denominator: measured copy bandwidth (MEASURED_PEAKS.json), else the fallback of
    B200_PROFILING.md."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    except Exception:
        return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "100"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for nme, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm),
                "reasons": sorted(reasons)}


def make_workload(size, kind="collision"):
    from paper_2501_00846_b200 import inputs as I
    if kind == "emulsion":
        return I.emulsion_sweep(n=size)
    s = size / 256.0
    return I.head_on_collision(n=size, radius=24.0 * s, half_sep=40.0 * s)


def time_oracle(cfg, planes, steps, warmup=0):
    """Oracle (as it stands) on the central `planes`-thick z slab of the workload."""
    from oracle import tslb_ref as R
    nz, ny, nx = cfg["shape"]
    z0 = (nz - planes) // 2
    phi = np.ascontiguousarray(cfg["phi"][z0:z0 + planes])
    u = np.ascontiguousarray(cfg["u"][:, z0:z0 + planes])
    sim = R.RefSim(nx, ny, planes, R.make_params(**cfg["params"]))
    sim.init(phi, u)
    if warmup:
        sim.step(warmup)
    t = time.perf_counter()
    sim.step(steps)
    dt = time.perf_counter() - t
    sim.close()
    return nx * ny * planes * steps / dt / 1e9, dt


def omp_threads():
    v = os.environ.get("OMP_NUM_THREADS")
    try:
        return int(v) if v else len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count()


def run_reference(args):
    """--impl reference: the CPU oracle on a bounded slab, same metric / unit / config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = make_workload(args.size, args.workload)
    nz, ny, nx = cfg["shape"]
    rate, _ = time_oracle(cfg, 4, 1)                      # calibration: 4 planes, 1 step
    budget = 100.0                                         # seconds for warmup + steps
    planes = int(budget * rate * 1e9 / (nx * ny * max(1, args.steps + args.warmup)))
    planes = max(4, min(nz, planes))
    glups, dt = time_oracle(cfg, planes, args.steps, args.warmup)
    sample = f"central {nx}x{ny}x{planes} slab of the {nx}^3 input, {args.steps} steps"
    line = {"impl": "reference", "metric": METRIC, "value": glups, "unit": "GLUPS",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": cfg["name"], "sample": sample},
            "cpu_baseline": {"value": glups, "unit": "GLUPS", "cores": omp_threads(),
                             "kind": "oracle", "sample": sample},
            "e2e": {"value": glups, "unit": "GLUPS", "h2d_bytes_per_step": 0,
                    "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def measure(cfg, precision, args, device, flags, dist_barrier):
    """W warm-up steps, then exactly K steps between a barrier + synchronize on both sides.
    Returns whole-step ms, per-kernel ms, launches, clocks."""
    import torch
    from paper_2501_00846_b200 import binding as B
    nz, ny, nx = cfg["shape"]
    s = B.Solver(nx, ny, nz, cfg["params"], precision=precision, flags=flags, device=device)
    s.init(cfg["phi"], cfg["u"])
    s.step(args.warmup)
    torch.cuda.synchronize(device)
    dist_barrier()
    sampler = ClockSampler(torch.device(device).index or 0)
    sampler.start()
    l0 = s.launches
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize(device)
    e0.record(s.stream)
    kernel_ms = s.step_timed(args.steps)           # events around every kernel, same stream
    e1.record(s.stream)
    torch.cuda.synchronize(device)
    dist_barrier()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    launches = s.launches - l0
    # sanity of the timed run: finite fields, phi conserved (P7)
    g = s.get(("phi", "u"))
    ok = bool(torch.isfinite(g["phi"]).all()) and bool(torch.isfinite(g["u"]).all())
    drift = abs(float(g["phi"].double().sum()) / float(cfg["phi"].sum()) - 1.0)
    s.close()
    return dict(ms=ms, kernel_ms=kernel_ms, launches=launches, clocks=clocks, finite=ok,
                phi_drift=drift)


def measure_e2e(cfg, precision, args, device, flags):
    """Host buffers through the C ABI: tslb_init_host (H2D) -> tslb_step(K) -> tslb_get_host (D2H),
    all inside the timed region."""
    import torch
    from paper_2501_00846_b200 import binding as B
    nz, ny, nx = cfg["shape"]
    dt = torch.float64 if precision == "f64" else torch.float32
    phi = torch.from_numpy(cfg["phi"]).to(dt).pin_memory()
    u = torch.from_numpy(cfg["u"]).to(dt).pin_memory()
    out = {"rho": torch.empty_like(phi).pin_memory(), "p": torch.empty_like(phi).pin_memory(),
           "u": torch.empty_like(u).pin_memory(), "phi": torch.empty_like(phi).pin_memory()}
    s = B.Solver(nx, ny, nz, cfg["params"], precision=precision, flags=flags, device=device)
    s.init_host(phi, u)                            # warm-up of the copy path and the kernels
    s.step(3)
    s.get_host(out)
    torch.cuda.synchronize(device)
    t0 = time.perf_counter()
    s.init_host(phi, u)
    s.step(args.steps)
    s.get_host(out)                                # synchronises the stream
    t1 = time.perf_counter()
    s.close()
    es = 8 if precision == "f64" else 4
    n = nx * ny * nz
    return dict(value=n * args.steps / (t1 - t0) / 1e9, unit="GLUPS",
                h2d_bytes_per_step=4 * n * es / args.steps,
                d2h_bytes_per_step=6 * n * es / args.steps,
                note="host->device init + K steps + device->host read of rho,p,u,phi, wall clock")


class Ranks:
    """One process per GPU (torchrun env).  Replicas only: the data path has no collective; the
    only communication is the timing protocol (barrier, max of the device time over ranks)."""

    def __init__(self, backend):
        import torch
        import torch.distributed as dist
        self.torch, self.dist = torch, dist
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.rank = int(os.environ.get("RANK", "0"))
        self.local = int(os.environ.get("LOCAL_RANK", "0"))
        self.backend = backend
        self.device = f"cuda:{self.local}" if backend == "nccl" else "cpu"
        if self.world > 1:
            kw = {"device_id": torch.device(self.device)} if backend == "nccl" else {}
            dist.init_process_group(backend, **kw)

    def barrier(self):
        if self.world > 1:
            self.dist.barrier()

    def max(self, x):
        if self.world == 1:
            return x
        t = self.torch.tensor([x], dtype=self.torch.float64, device=self.device)
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX)
        return float(t.item())

    def close(self):
        if self.world > 1:
            self.dist.destroy_process_group()


def whole_job_glups(nodes, steps, ms_max, world):
    """Aggregate over all replicas: every rank advanced `nodes` nodes by `steps` steps in at most
    ms_max milliseconds (max over ranks)."""
    return world * nodes * steps / (ms_max * 1e-3) / 1e9


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    import torch
    ranks = Ranks("nccl")
    world, rank, device = ranks.world, ranks.rank, ranks.device
    torch.cuda.set_device(ranks.local)
    barrier, max_over_ranks = ranks.barrier, ranks.max

    flags = (1 if args.naive else 0) | (2 if args.generic else 0) | (args.variant << 8) | (args.k1variant << 16)
    cfg = make_workload(args.size, args.workload)
    n = int(np.prod(cfg["shape"]))
    peak, peak_kind = peaks()
    order = [args.only] if args.only else [args.precision, "f32" if args.precision == "f64" else "f64"]
    res = {}
    for prec in order:
        r = measure(cfg, prec, args, device, flags, barrier)
        r["ms"] = max_over_ranks(r["ms"])
        es = 8 if prec == "f64" else 4
        r["glups"] = whole_job_glups(n, args.steps, r["ms"], world)
        # dominant kernel and its roofline: algorithmic bytes of the
        # whole update, 28 s per node, charged to the dominant kernel's own duration only when
        # the step is a single kernel; for a split step each kernel is charged its own planes.
        dom = max(r["kernel_ms"], key=r["kernel_ms"].get)
        # scalars per update the dominant kernel must move: the periodic
        # stream-collide kernel reads 13 moments + phi^{n+1} and writes 13 moments + the flux Q (3);
        # the wall-capable / naive one writes no Q.
        periodic_fast = not (args.naive or args.generic) and not any(cfg["params"]["bc"])
        planes = {"stream_collide": 30 if periodic_fast else 27, "allen_cahn": 5, "normal": 4}[dom]
        k_ms = r["kernel_ms"][dom] / args.steps
        ach = planes * es * n / (k_ms * 1e-3) / 1e9
        step_ach = 2 * STATE_SCALARS * es * n / (r["ms"] / args.steps * 1e-3) / 1e9
        r["roofline"] = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak,
                         "unit": "GB/s", "frac": ach / peak,
                         "traffic": NCU_TRAFFIC.get((prec, dom)) if (periodic_fast and n == 256 ** 3) else None,
                         "peak_kind": peak_kind, "kernel_ms": k_ms,
                         "kernels_ms": {k: v / args.steps for k, v in r["kernel_ms"].items()},
                         "kernel_share_of_step": r["kernel_ms"][dom] / r["ms"],
                         "algorithmic_bytes_per_update": planes * es,
                         "step_achieved": step_ach, "step_frac": step_ach / peak,
                         "step_frac_of_8TBs": step_ach / 8000.0}
        res[prec] = r
    head = res[order[0]]
    e2e = None
    if not args.no_e2e:
        e2e = measure_e2e(cfg, order[0], args, device, flags)
        e2e["value"] = world * e2e["value"] if world > 1 else e2e["value"]
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        planes, osteps = min(64, cfg["shape"][0]), 8
        v, dt = time_oracle(cfg, planes, osteps)
        cpu = {"value": v, "unit": "GLUPS", "cores": omp_threads(), "kind": "oracle",
               "sample": f"central {cfg['shape'][2]}x{cfg['shape'][1]}x{planes} slab of the same "
                         f"input, {osteps} steps, {dt:.1f} s"}
    if rank == 0:
        line = {"metric": METRIC, "value": head["glups"], "unit": "GLUPS", "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": head["ms"] / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": order[0], "data": "synthetic",
                "config": {"workload": cfg["name"], "grid": list(cfg["shape"][::-1]),
                           "parallelism": f"replicas x{world}",
                           "l2": f"state {2 * STATE_SCALARS * (8 if order[0] == 'f64' else 4) * n / 1e9:.1f} GB ({order[0]}) >> 126 MB L2",
                           "path": "naive" if args.naive else ("tiled-generic" if args.generic else "tiled"),
                           "variant": args.variant},
                "clocks": head["clocks"], "gpu_launches": head["launches"],
                "roofline": head["roofline"], "finite": head["finite"],
                "phi_drift": head["phi_drift"]}
        if e2e:
            line["e2e"] = e2e
        if cpu:
            line["cpu_baseline"] = cpu
        for prec in order[1:]:
            o = res[prec]
            line[prec] = {"value": o["glups"], "unit": "GLUPS", "ms_per_step": o["ms"] / args.steps,
                          "roofline": o["roofline"], "clocks": o["clocks"],
                          "gpu_launches": o["launches"], "finite": o["finite"]}
        print(json.dumps(line), flush=True)
    ranks.close()


if __name__ == "__main__":
    main()
