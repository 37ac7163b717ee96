#!/usr/bin/env python
"""bench.py -- GLUPS of the TSLB + Allen-Cahn step on one B200 (BASELINE.json metric).

A "step" is one tslb_step(1): every stage of SURVEY.md 8(a) over the whole 256^3 head-on
collision domain (BASELINE.json configs[3], synthetic, seeded).  Protocol:
W warm-up steps, then R repeats of exactly K steps, each between two CUDA events on the solver's
stream with a barrier + synchronize on both sides (max over ranks per repeat); `value` comes
from the MEDIAN repeat, the minimum is reported beside it.  The state (3.8 GB in fp64) is far
larger than the 126 MB L2, so every step streams from HBM.  `e2e` goes through the C ABI's
host-buffer calls (tslb_init_host -> tslb_step -> tslb_get_host) with the copies inside the timed
region.  Multi-GPU = independent replicas: weak scaling, no data-path
collective.  `--impl reference` times the CPU oracle on a bounded slab of the same workload (a
deliberately plain program: context, not a target).

roofline.frac follows SURVEY.md 8(d): ALGORITHMIC bytes (14 scalars read + 14 written per update)
over the whole step's time, against the measured HBM copy rate; the per-kernel split is under
roofline.kernels.  roofline.alu_frac is the other side of the ridge: ~0.9 kflop per update
against the FMA throughput measured in this run (tslb_fma_peak).
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
FLOP_PER_UPDATE = 900.0                 # 0.8-1.0 kflop with every node quantity
                                        # computed once (a1 70, a2 150, a4 100, a5 300, a6-a9 250)
# flops actually EXECUTED per update (FMA = 2), from the instruction mix of the ncu captures in
# profiles/r2_kernels_*.txt (K2 + K1, ring-cell redundancy included): the 0.9 kflop above is
# SURVEY.md's estimate of the algorithm, this is what the kernels issue
FLOP_EXECUTED = {"f64": 603.0, "f32": 615.0}
# dram__bytes_read.sum + dram__bytes_write.sum per STEP (all kernels of one step) on the 256^3
# collision workload, copied from the ncu --set full captures named beside them (not measured by
# this run: ncu cannot run inside a timed bench)
NCU_TRAFFIC = {"f64": (1.979212e9 + 2.104534e9 + 0.562511e9 + 0.118631e9, "profiles/r2_kernels_f64.txt"),
               "f32": (0.977138e9 + 1.029165e9 + 0.285295e9 + 0.050446e9, "profiles/r2_kernels_f32.txt")}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--repeats", type=int, default=5, help="timed repeats of --steps steps")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--size", type=int, default=256, help="cube edge of the domain")
    ap.add_argument("--workload", default="collision",
                    choices=["collision", "emulsion", "bubble", "offaxis", "train"],
                    help="collision = BASELINE.json configs[3] (the graded one); emulsion = "
                         "configs[4] (--size 384 for f64, 512 for f32); bubble = configs[2] "
                         "(128x128x256, walls in z; --size scales it); offaxis = NEXT-2; train = NEXT-2's "
                         "droplet train falling onto a wall (128x128x768 at --size 256)")
    ap.add_argument("--precision", default="f64", choices=["f64", "f32"],
                    help="precision of the headline value (the other one is reported beside it)")
    ap.add_argument("--flags", type=int, default=0,
                    help="validation selector (include/tslb.h TSLB_FLAG_*), 0 = production")
    ap.add_argument("--bc", default=None,
                    help="override the boundary types, e.g. 1,1,1 = walls on x, y and z")
    ap.add_argument("--slab-overlap", default="auto", choices=["auto", "on", "off"],
                    help="--decomp slab: compute and send the face planes first and sweep the "
                         "interior while they travel (tslb_slab_step_faces / _interior); auto = "
                         "on when there is a transfer to hide (N > 1)")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (weak scaling; BASELINE.json's north star, "
                         "the default) or ONE lattice cut into z slabs with a halo exchange per "
                         "step (strong scaling; SURVEY.md NEXT-3, paper_2501_00846_b200/slab.py)")
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
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """SM clock, power and throttle reasons sampled IN PROCESS through NVML at ~200 Hz for the
    whole timed region (nvidia-smi -lms 100 in a child process missed 20 ms regions)."""
    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
               0x4: "sw_power_cap"}

    def __init__(self, index):
        self.index, self.rows, self.stop_flag, self.thread, self.h = index, [], False, None, None
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            phys = int(vis.split(",")[index]) if vis and vis.split(",")[index].isdigit() else index
            self.nv, self.h = pynvml, pynvml.nvmlDeviceGetHandleByIndex(phys)
        except Exception:
            self.nv = None

    def _loop(self):
        nv, h = self.nv, self.h
        while not self.stop_flag:
            try:
                sm = nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)
                try:
                    rs = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    rs = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                pw = nv.nvmlDeviceGetPowerUsage(h) / 1000.0
                self.rows.append((sm, rs, pw))
            except Exception:
                pass
            time.sleep(0.004)

    def start(self):
        if self.nv is None:
            return
        self.thread = threading.Thread(target=self._loop, daemon=True)
        self.thread.start()

    def stop(self):
        if self.nv is None or self.thread is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "samples": 0, "reasons": ["nvml unavailable"]}
        self.stop_flag = True
        self.thread.join(timeout=2)
        try:
            mx = float(self.nv.nvmlDeviceGetMaxClockInfo(self.h, self.nv.NVML_CLOCK_SM))
        except Exception:
            mx = None
        sm = [r[0] for r in self.rows]
        reasons = sorted({name for r in self.rows for bit, name in self.REASONS.items() if r[1] & bit})
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_min_mhz": float(min(sm)) if sm else None, "sm_max_mhz": mx,
                "power_w_max": max((r[2] for r in self.rows), default=None),
                "samples": len(sm), "reasons": reasons}


def make_workload(size, kind="collision"):
    from paper_2501_00846_b200 import inputs as I
    if kind == "emulsion":
        return I.emulsion_sweep(n=size)
    s = size / 256.0
    if kind == "bubble":                 # configs[2] is 128 x 128 x 256 = --size 256
        cfg = I.rising_bubble(nx=int(128 * s), ny=int(128 * s), nz=int(256 * s),
                              radius=16.0 * s, height=40.0 * s)
        # configs[2]'s parameters leave the scheme's stable range after ~500 steps at full size
        # (oracle and every CUDA path alike): each timed repeat restarts from t = 0
        cfg["reinit"] = True
        return cfg
    if kind == "offaxis":
        return I.off_axis_collision(n=size)
    if kind == "train":                  # PAPER.md:354-366; box 1 : 1 : 6, walls in z
        return I.droplet_train(nx=int(128 * s), ny=int(128 * s), nz=int(768 * s))
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


def oracle_one_core(cfg, planes, steps):
    """The same oracle on ONE core: a child process with OMP_NUM_THREADS=1 (the OpenMP runtime of
    this process already has its team)."""
    code = ("import sys, json; sys.path.insert(0, %r); import bench; "
            "cfg = bench.make_workload(%d, %r); v, dt = bench.time_oracle(cfg, %d, %d); "
            "print(json.dumps([v, dt]))" % (ROOT, cfg["_size"], cfg["_kind"], planes, steps))
    env = dict(os.environ, OMP_NUM_THREADS="1")
    try:
        out = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True,
                             timeout=600).stdout.strip().splitlines()[-1]
        v, dt = json.loads(out)
        return v, dt
    except Exception:
        return None, None


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
    sample = f"central {nx}x{ny}x{planes} slab of the {nx}x{ny}x{nz} input, {args.steps} steps"
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


def measure(cfg, precision, args, device, ranks):
    """W warm-up steps, then R repeats of exactly K steps between a barrier + synchronize on both
    sides; one more K-step pass with an event after every kernel gives the per-kernel split."""
    import torch
    from paper_2501_00846_b200 import binding as B
    nz, ny, nx = cfg["shape"]
    s = B.Solver(nx, ny, nz, cfg["params"], precision=precision, flags=args.flags, device=device)
    s.init(cfg["phi"], cfg["u"])
    d0 = s.diag()
    s.step(args.warmup)
    torch.cuda.synchronize(device)
    sampler = ClockSampler(torch.device(device).index or 0)
    sampler.start()
    l0 = s.launches
    reps = []
    for rep in range(max(1, args.repeats)):
        if cfg.get("reinit") and rep > 0:
            s.init(cfg["phi"], cfg["u"])
            s.step(args.warmup)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(device)
        ranks.barrier()
        e0.record(s.stream)
        s.step(args.steps)
        e1.record(s.stream)
        torch.cuda.synchronize(device)
        ranks.barrier()
        reps.append(ranks.max(e0.elapsed_time(e1)))
    launches = s.launches - l0
    if cfg.get("reinit"):                          # minus the init + warm-up launches in between
        launches -= (max(1, args.repeats) - 1) * (1 + 2 * args.warmup)
    launches //= max(1, args.repeats)
    clocks = sampler.stop()
    if cfg.get("reinit"):
        s.init(cfg["phi"], cfg["u"])
        s.step(args.warmup)
    kernel_ms = s.step_timed(args.steps)           # events around every kernel, same stream
    # sanity of the timed run through the on-device reductions (no field is read back):
    # finite fields, phi conserved (P7)
    d1 = s.diag()
    ok = all(np.isfinite(v) for v in d1.values())
    drift = abs(d1["sum_phi"] / d0["sum_phi"] - 1.0)
    s.close()
    fma = B.tslb_fma_peak(precision)
    return dict(ms=float(np.median(reps)), ms_min=float(min(reps)), reps=reps, kernel_ms=kernel_ms,
                launches=launches, clocks=clocks, finite=ok, phi_drift=drift, max_u=d1["max_u"],
                fma_tflops=fma)


def measure_slab(cfg, precision, args, device, ranks):
    """--decomp slab: this rank's z slab of the ONE global lattice; a step = tslb_step(1) on the
    slab + the halo exchange with both neighbours (torch.distributed P2P; a local copy at N = 1).
    Same protocol as measure(); the per-kernel split times the slab's own kernels only."""
    import torch
    from paper_2501_00846_b200 import binding as B, slab as S
    nz, ny, nx = cfg["shape"]
    sl = S.SlabSolver(nx, ny, nz, cfg["params"], ranks.rank, ranks.world, precision=precision,
                      device=device, flags=args.flags)
    sl.exchange = S.DistExchange(sl, ranks.rank, ranks.world, ranks.dist)
    sl.init(cfg["phi"], cfg["u"])
    sl.exchange()
    d0 = sl.solver.diag()
    overlap = args.slab_overlap == "on" or (args.slab_overlap == "auto" and ranks.world > 1)
    sl.step(args.warmup, overlap=overlap)
    torch.cuda.synchronize(device)
    sampler = ClockSampler(torch.device(device).index or 0)
    sampler.start()
    l0 = sl.solver.launches
    reps = []
    for _ in range(max(1, args.repeats)):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize(device)
        ranks.barrier()
        e0.record(sl.solver.stream)
        sl.step(args.steps, overlap=overlap)
        e1.record(sl.solver.stream)
        torch.cuda.synchronize(device)
        ranks.barrier()
        reps.append(ranks.max(e0.elapsed_time(e1)))
    launches = (sl.solver.launches - l0) // max(1, args.repeats)
    clocks = sampler.stop()
    kernel_ms = sl.solver.step_timed(args.steps)
    sl.exchange()
    d1 = sl.solver.diag()
    ok = all(np.isfinite(v) for v in d1.values())
    sl.close()
    return dict(ms=float(np.median(reps)), ms_min=float(min(reps)), reps=reps, kernel_ms=kernel_ms,
                launches=launches, clocks=clocks, finite=ok,
                phi_drift=abs(d1["sum_phi"] / d0["sum_phi"] - 1.0), max_u=d1["max_u"],
                fma_tflops=B.tslb_fma_peak(precision))


def measure_e2e(cfg, precision, args, device):
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
    s = B.Solver(nx, ny, nz, cfg["params"], precision=precision, flags=args.flags, device=device)
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


def roofline(r, prec, n, steps, peak, peak_kind, periodic_fast, full_size):
    """frac = algorithmic bytes (28 s per update) over the step time, against the
    measured copy rate.  Per kernel: its own duration and the scalars it really moves."""
    es = 8 if prec == "f64" else 4
    ms_step = r["ms"] / steps
    b_alg = 2 * STATE_SCALARS * es
    ach = b_alg * n / (ms_step * 1e-3) / 1e9
    dom = max(r["kernel_ms"], key=r["kernel_ms"].get)
    moved = ({"stream_collide": 30, "allen_cahn": 5} if periodic_fast
             else {"stream_collide": 27, "allen_cahn": 8, "normal": 4})
    tot_k = sum(r["kernel_ms"].values())
    kernels = {k: {"ms": v / steps, "share_of_step": v / tot_k,
                   "moved_scalars_per_update": moved.get(k),
                   "moved_gbs": moved[k] * es * n / (v / steps * 1e-3) / 1e9 if k in moved else None}
               for k, v in r["kernel_ms"].items()}
    traffic, src = NCU_TRAFFIC.get(prec, (None, None)) if (periodic_fast and full_size) else (None, None)
    alu_ach = FLOP_PER_UPDATE * n / (ms_step * 1e-3) / 1e12
    return {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s",
            "frac": ach / peak, "frac_min_repeat": b_alg * n / (r["ms_min"] / steps * 1e-3) / 1e9 / peak,
            "frac_of_8TBs": ach / 8000.0, "traffic": traffic, "traffic_source": src,
            "traffic_unit": "bytes per step (all kernels), ncu dram__bytes_read+write",
            "peak_kind": peak_kind, "algorithmic_bytes_per_update": b_alg,
            "kernels": kernels,
            "alu_frac": alu_ach / r["fma_tflops"], "alu_achieved_tflops": alu_ach,
            "alu_peak_tflops": r["fma_tflops"], "alu_flop_per_update": FLOP_PER_UPDATE,
            "alu_frac_executed": FLOP_EXECUTED[prec] * n / (ms_step * 1e-3) / 1e12 / r["fma_tflops"],
            "alu_flop_per_update_executed": FLOP_EXECUTED[prec],
            "alu_peak_kind": "measured in this run (tslb_fma_peak, dependent-chain-free FMA)"}


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    import torch
    ranks = Ranks("nccl")
    world, rank, device = ranks.world, ranks.rank, ranks.device
    torch.cuda.set_device(ranks.local)

    cfg = make_workload(args.size, args.workload)
    cfg["_size"], cfg["_kind"] = args.size, args.workload
    if args.bc:
        cfg["params"] = dict(cfg["params"], bc=tuple(int(v) for v in args.bc.split(",")))
        cfg["name"] += "_bc" + args.bc.replace(",", "")
    n = int(np.prod(cfg["shape"]))
    peak, peak_kind = peaks()
    order = [args.only] if args.only else [args.precision, "f32" if args.precision == "f64" else "f64"]
    bc = cfg["params"]["bc"]                       # lean pair: periodic x, y (walls in z allowed)
    periodic_fast = not (args.flags & 3) and not (bc[0] or bc[1])
    full = args.workload == "collision" and args.size == 256
    res = {}
    slab = args.decomp == "slab"
    for prec in order:
        if slab:            # one lattice over all ranks: strong scaling, per-GPU roofline
            r = measure_slab(cfg, prec, args, device, ranks)
            r["glups"] = whole_job_glups(n, args.steps, r["ms"], 1)
            r["roofline"] = roofline(r, prec, n // world, args.steps, peak, peak_kind, periodic_fast, False)
        else:
            r = measure(cfg, prec, args, device, ranks)
            r["glups"] = whole_job_glups(n, args.steps, r["ms"], world)
            r["roofline"] = roofline(r, prec, n, args.steps, peak, peak_kind, periodic_fast, full)
        if not args.no_e2e and not slab:
            r["e2e"] = measure_e2e(cfg, prec, args, device)
            r["e2e"]["value"] *= world
        res[prec] = r
    head = res[order[0]]
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        planes, osteps = min(64, cfg["shape"][0]), 8
        v, dt = time_oracle(cfg, planes, osteps)
        sample = (f"central {cfg['shape'][2]}x{cfg['shape'][1]}x{planes} slab of the same input, "
                  f"{osteps} steps, {dt:.1f} s")
        cpu = {"value": v, "unit": "GLUPS", "cores": omp_threads(), "kind": "oracle", "sample": sample}
        v1, dt1 = oracle_one_core(cfg, min(8, cfg["shape"][0]), 2)
        if v1 is not None:
            cpu["one_core"] = {"value": v1, "unit": "GLUPS", "cores": 1,
                               "sample": f"central slab of {min(8, cfg['shape'][0])} planes, 2 steps, {dt1:.1f} s"}
    if rank == 0:
        es0 = 8 if order[0] == "f64" else 4
        line = {"metric": METRIC, "value": head["glups"], "unit": "GLUPS", "n_gpus": world,
                "steps": args.steps, "warmup": args.warmup, "repeats": args.repeats,
                "ms_per_step": head["ms"] / args.steps,
                "ms_per_step_min": head["ms_min"] / args.steps,
                "higher_is_better": True,
                "scaling": "strong" if slab else "weak", "vs_baseline": None, "dtype": order[0],
                "data": "synthetic",
                "config": {"workload": cfg["name"], "grid": list(cfg["shape"][::-1]),
                           "parallelism": (f"z-slabs x{world}, halo exchange per step"
                                           + (", overlapped with the interior sweep"
                                              if args.slab_overlap == "on" or
                                              (args.slab_overlap == "auto" and world > 1) else "")
                                           if slab else f"replicas x{world}"),
                           "l2": f"state {2 * STATE_SCALARS * es0 * n / 1e9:.1f} GB ({order[0]}) >> 126 MB L2: "
                                 "inputs larger than L2, no flush needed",
                           "flags": args.flags,
                           "timing": f"median of {args.repeats} repeats of {args.steps} steps (CUDA events)"},
                "clocks": head["clocks"], "gpu_launches": head["launches"],
                "roofline": head["roofline"], "finite": head["finite"],
                "phi_drift": head["phi_drift"], "max_u": head["max_u"]}
        if "e2e" in head:
            line["e2e"] = head["e2e"]
        if cpu:
            line["cpu_baseline"] = cpu
        for prec in order[1:]:
            o = res[prec]
            line[prec] = {"value": o["glups"], "unit": "GLUPS", "ms_per_step": o["ms"] / args.steps,
                          "ms_per_step_min": o["ms_min"] / args.steps,
                          "roofline": o["roofline"], "clocks": o["clocks"],
                          "gpu_launches": o["launches"], "finite": o["finite"],
                          "phi_drift": o["phi_drift"]}
            if "e2e" in o:
                line[prec]["e2e"] = o["e2e"]
        print(json.dumps(line), flush=True)
    ranks.close()


if __name__ == "__main__":
    main()
