#!/usr/bin/env python
"""bench.py -- whole-job throughput of the Lagrangian-Eulerian coupling step (BASELINE.json metric:
Lagrangian points/s for the fused FE-force + spread + interp step, fp64) on synthetic LV-shell
input (config 3 of BASELINE.json / SURVEY.md §8(d)), plus the roofline of the dominant kernel and
the CPU oracle timed on the same box.

  python bench.py --gpus N --steps K --warmup W            # ours (CUDA path through the C ABI)
  python bench.py --impl reference --steps K --warmup W    # the CPU oracle as the reference arm

One "step" = one ib_coupling_step (SURVEY.md §8(a) a1-a9 incl. bin/sort and the zero-fill of f).
N > 1: one process per GPU (torchrun), independent replicas of the same problem ("replicas only",
DESIGN.md): no data-path collective, only the timing barrier / max-reduction.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "lagrangian_points_per_s_fused_coupling_step_fp64"
UNIT = "points/s"


# ----------------------------------------------------------------------------------------------
def make_workload(name):
    from paper_2503_22695_b200 import workloads as W
    if name == "C1":
        return W.config1()
    if name == "C2":
        return W.config2()
    if name == "C3":
        return W.config3()
    if name == "C3-s2":
        return W.config3(nsub=(2, 2, 2))
    if name == "C4":
        return W.config4()
    if name.startswith("C5"):                      # C5-L<level>-s<sub>
        parts = name.split("-")
        return W.config5(level=int(parts[1][1:]), sub=int(parts[2][1:]))
    raise SystemExit(f"unknown workload {name}")


def algorithmic_bytes(wl):
    """SURVEY.md §8(d) array-form accounting: 72 B/point (xp in, Gp in, Up out) + 48 B/cell
    (u,v,w in; fu,fv,fw out incl. zero-fill) + per element conn 32 + fibres 48 + per node
    X,x,B,Un 96.  Sort traffic is implementation overhead and is not counted."""
    return 72 * wl.n_points + 48 * wl.n_cells + 80 * wl.n_elems + 96 * wl.n_nodes


def dfma_slots(wl):
    """DESIGN.md flop model: ~600 DFMA slots per force point (weights 100 + interp 252 + spread
    252) + ~650 per Gauss point."""
    return 600 * wl.n_points + 650 * 8 * wl.n_elems


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML during the timed region."""

    def __init__(self, index, period=0.005):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=1.0)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def max_over_ranks(value, world, device=None):
    """Max of a per-rank scalar over all ranks (torch.distributed must be initialised when
    world > 1; works on nccl with a CUDA device and on gloo with device=None)."""
    if world <= 1:
        return float(value)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank_per_step, steps, t_rank_s, world, device=None):
    """Replicas only: every rank processes the same number of units; the job's time
    is the slowest rank's; value = units of all ranks / that time."""
    t = max_over_ranks(t_rank_s, world, device)
    return world * units_per_rank_per_step * steps / t, t


def kernel_source_sha():
    """sha256 over the sources of the dominant kernel: the stamp of an ncu capture (profiles/*_traffic.json)."""
    import hashlib
    h = hashlib.sha256()
    for f in ("ib_tiled.cu", "ib_common.cuh", "ib_point.cuh"):
        h.update(open(os.path.join(ROOT, "paper_2503_22695_b200", "csrc", f), "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic_bytes(workload_name, n_points=None):
    """(DRAM bytes per launch of the dominant kernel, source) from the newest committed ncu capture
    profiles/r*_traffic.json -- only if it was taken on THESE kernel sources (the file carries their
    sha256); otherwise (None, why): a stale capture is not a measurement of this build."""
    import glob
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_traffic.json")))
    if not files:
        return None, "no ncu capture committed"
    rec = json.load(open(files[-1]))
    if rec.get("kernel_source_sha256_16") != kernel_source_sha():
        return None, f"{os.path.basename(files[-1])} was captured on other kernel sources"
    key = workload_name if n_points is None else f"{workload_name}:{n_points}"
    v = rec.get("dram_bytes_per_launch", {}).get(key)
    if v is None:
        return None, f"{os.path.basename(files[-1])} has no capture of {key}"
    return int(v), f"ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum ({os.path.basename(files[-1])}, same kernel sources)"


# ----------------------------------------------------------------------------------------------
def cpu_sample(wl, frac):
    """Bounded sample of the workload for the oracle: the first `frac` of the elements (a
    contiguous band of the structured mesh), nodes re-indexed, same grid and velocity field."""
    ne = max(1, int(wl.n_elems * frac))
    conn = wl.conn[:ne]
    used = np.unique(conn)
    remap = -np.ones(wl.n_nodes, dtype=np.int64)
    remap[used] = np.arange(used.size)
    return dict(conn=remap[conn].astype(np.int32), X=np.ascontiguousarray(wl.X[:, used]),
                x=np.ascontiguousarray(wl.x[:, used]), fibers=np.ascontiguousarray(wl.fibers[:, :ne]),
                mat_id=np.ascontiguousarray(wl.mat_id[:ne]), nsub=np.ascontiguousarray(wl.nsub[:ne]),
                n_points=int(np.prod(wl.nsub[:ne].astype(np.int64), axis=1).sum()), n_elems=ne)


def time_oracle(wl, frac, reps=1, omp=False):
    import oracle
    s = cpu_sample(wl, frac)
    g = oracle.make_grid(wl.nx, wl.ny, wl.nz, wl.h, wl.origin)
    best = None
    for _ in range(reps):
        t0 = time.perf_counter()
        oracle.coupling_step(g, s["conn"], s["X"], s["fibers"], s["mat_id"], s["nsub"], wl.mats, s["x"],
                             wl.u, wl.v, wl.w, omp=omp)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return s, best


def run_reference(args):
    """The reference arm = the CPU oracle as it stands, on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = make_workload(args.workload)
    frac = args.cpu_frac
    for _ in range(args.warmup):
        time_oracle(wl, frac / 8)
    ts = []
    for _ in range(args.steps):
        s, dt = time_oracle(wl, frac)
        ts.append(dt)
    t = float(np.mean(ts))
    val = s["n_points"] / t
    sample = (f"first {s['n_elems']} of {wl.n_elems} elements ({s['n_points']} of {wl.n_points} force points) "
              f"of {wl.name}, full {wl.nx}x{wl.ny}x{wl.nz} grid, one oracle_coupling_step")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": wl.name, "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ----------------------------------------------------------------------------------------------
def relaunch(n):
    """`python bench.py --gpus N` without torchrun: start the N replica processes ourselves, one per GPU, the
    way the driver does (python -m torch.distributed.run, rendezvous on 127.0.0.1)."""
    import socket
    import subprocess
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={n}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_dry(args):
    """The launch and whole-job arithmetic of run_ours with no GPU: every rank 'processes' the workload's
    points in 1 + rank/10 seconds; rank 0 prints the line."""
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if world > 1:
        dist.init_process_group("gloo")
    units = 1000
    value, t = whole_job_value(units, args.steps, 1.0 + 0.1 * rank, world, None)
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                          "dry_run": True, "slowest_rank_s": t}))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2503_22695_b200 import build as ibbuild
    from paper_2503_22695_b200 import ibcouple

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if rank == 0:
        ibbuild.build()
    if world > 1:
        dist.barrier()
    ibcouple.lib()

    wl = make_workload(args.workload)
    ctx = ibcouple.Context.from_workload(wl, device=local)
    ctx.ib_set_variant(args.variant)
    dev = torch.device("cuda", local)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    x, u, v, w = t(wl.x), t(wl.u), t(wl.v), t(wl.w)
    fu, fv, fw = (torch.empty(wl.n_cells, dtype=torch.float64, device=dev) for _ in range(3))
    Un = torch.empty((3, wl.n_nodes), dtype=torch.float64, device=dev)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)       # 512 MiB > 126 MB L2
    # a stream of our own: the legacy default stream cannot be captured, and the library replays the
    # step as one CUDA graph from the third call on (include/ibcouple.h, ib_set_graph)
    stream = torch.cuda.Stream(device=dev)
    torch.cuda.synchronize()
    torch.cuda.set_stream(stream)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def step():
        ctx.ib_coupling_step(x, u, v, w, fu, fv, fw, Un, None, stream)

    for _ in range(max(args.warmup, 3)):
        flush.zero_()
        step()
    ctx.check()
    l0 = ctx.ib_launch_count()
    sampler = ClockSampler(local)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    sampler.start()
    t_wall0 = time.perf_counter()
    for i in range(args.steps):
        flush.zero_()                       # L2 flush between timed iterations (not timed)
        ev[i][0].record(stream)
        step()
        ev[i][1].record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    ms = [a.elapsed_time(b) for a, b in ev]
    launches = ctx.ib_launch_count() - l0
    ctx.check()
    # per-phase breakdown from a separate profiled pass (profiling serialises the phases that the
    # timed step overlaps on the context's side stream, so it is kept out of the timed region)
    ctx.ib_profile_enable(True)
    ctx.ib_profile_read()
    for _ in range(max(3, min(args.steps, 10))):
        flush.zero_()
        step()
    torch.cuda.synchronize()
    prof = ctx.ib_profile_read()
    ctx.ib_profile_enable(False)
    value, t_dev = whole_job_value(wl.n_points, args.steps, float(np.sum(ms)) * 1e-3, world, dev)
    # run-to-run deviation: the REDs of the spreading reorder the sums, so three
    # untimed runs on the same inputs are compared; B and the bin counts are order-free
    runs = []
    for _ in range(3):
        step()
        torch.cuda.synchronize()
        runs.append([a.clone() for a in (fu, fv, fw, Un)])
    dev_rr = {}
    for k, name in enumerate(("fu", "fv", "fw", "Un")):
        scale = float(runs[0][k].abs().max())
        d = max(float((runs[i][k] - runs[0][k]).abs().max()) for i in (1, 2))
        dev_rr[name] = d / scale if scale > 0 else 0.0
    del runs

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    hx, huvw = pin(wl.x), pin(np.stack([wl.u, wl.v, wl.w]))
    hf = torch.empty((3, wl.n_cells), dtype=torch.float64).pin_memory()
    hUn = torch.empty((3, wl.n_nodes), dtype=torch.float64).pin_memory()
    e2e_steps = max(2, min(args.steps, 10))
    for _ in range(2):
        ctx.ib_coupling_step_host3(hx, huvw, hf, hUn, None, stream)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ctx.ib_coupling_step_host3(hx, huvw, hf, hUn, None, stream)
    barrier()
    t_e2e = time.perf_counter() - t0
    e2e_val, _ = whole_job_value(wl.n_points, e2e_steps, t_e2e, world, dev)
    h2d = 8 * (3 * wl.n_nodes + 3 * wl.n_cells)
    d2h = 8 * (3 * wl.n_cells + 3 * wl.n_nodes)

    if rank == 0:
        peaks = {}
        pk = os.path.join(ROOT, "MEASURED_PEAKS.json")
        if os.path.exists(pk):
            peaks = json.load(open(pk))
        hbm_peak = float(peaks.get("hbm_gbs", 6650.0))
        hbm_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s"
        dom = "spread_interp"
        dom_ms = prof[dom][0] / max(prof[dom][1], 1)
        step_ms = 1e3 * t_dev / args.steps
        abytes = algorithmic_bytes(wl)
        dfma_peak, _ = ibcouple.probe_dfma(local)
        # dominant kernel: the points' 72 B and the 24 B/cell of u,v,w belong to it; the other 24 B/cell of the
        # SURVEY.md §8(d) figure (f out, incl. its zero-fill) are the zero phase's -- a memset on another
        # stream -- so that the fraction cannot exceed 1 on sparsely filled grids
        dom_bytes = 72 * wl.n_points + 24 * wl.n_cells
        traffic, traffic_src = ncu_traffic_bytes(wl.name, wl.n_points)
        # The dominant kernel is bound by the plain fp64 ALUs, not by HBM: the top-level
        # roofline is the ALU one -- algorithmic flops = 2 x 600 DFMA slots per force point (SURVEY.md
        # §8(d): weights 100 + interpolation 252 + spreading 252), peak derived from the unit count and
        # the clock (64 DFMA/clk/SM x SMs x max SM clock; ib_probe_dfma measures 92 % of it).  The HBM
        # roofline BASELINE.json's metric names is reported beside it under "hbm".
        dom_slots = 600 * wl.n_points
        sms = torch.cuda.get_device_properties(local).multi_processor_count
        sm_hz = 1e6 * float(clocks.get("sm_max_mhz") or 1965.0)
        alu_peak_tf = 2.0 * 64 * sms * sm_hz / 1e12
        dom_tf = 2.0 * dom_slots / (dom_ms * 1e-3) / 1e12
        roofline = {"bound": "alu", "kernel": "spread+interp (" + ("tiled" if args.variant else "per-point") + ")",
                    "achieved": dom_tf, "peak": alu_peak_tf, "unit": "TFLOP/s", "frac": dom_tf / alu_peak_tf,
                    "traffic": traffic, "traffic_source": traffic_src,
                    "peak_source": f"derived: 64 DFMA/clk/SM x {sms} SMs x {sm_hz / 1e6:.0f} MHz x 2 flop (fp64 vector pipe); "
                                   f"ib_probe_dfma measured {2 * dfma_peak / 1e12:.1f} TFLOP/s in this run",
                    "kernel_ms": dom_ms, "algorithmic_flops_per_launch": 2 * dom_slots,
                    "hbm": {"achieved": dom_bytes / (dom_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                            "frac": dom_bytes / (dom_ms * 1e-3) / 1e9 / hbm_peak, "peak_source": hbm_src,
                            "algorithmic_bytes_per_launch": dom_bytes},
                    "step": {"algorithmic_bytes": abytes, "achieved_GBps": abytes / (step_ms * 1e-3) / 1e9,
                             "frac_of_hbm_peak": abytes / (step_ms * 1e-3) / 1e9 / hbm_peak},
                    "alu": {"dfma_slots_per_step": dfma_slots(wl), "dfma_peak_per_s": dfma_peak,
                            "peak_source": "ib_probe_dfma (register-only DFMA loop, this run)",
                            "frac_of_dfma_peak": dfma_slots(wl) / (step_ms * 1e-3) / dfma_peak},
                    "phases_ms": {k: (prof[k][0] / max(prof[k][1], 1)) for k in prof}}
        s, dt = time_oracle(wl, args.cpu_frac)
        sample = (f"first {s['n_elems']} of {wl.n_elems} elements ({s['n_points']} force points) of {wl.name}, "
                  f"full grid, one oracle_coupling_step, {dt:.1f} s")
        # all-core leg (SURVEY.md §8(d) "Oracle timing (ii)"): the same source built with -fopenmp, 4x the sample
        cores = len(os.sched_getaffinity(0))
        s_all, dt_all = time_oracle(wl, min(1.0, 4 * args.cpu_frac), omp=True)
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": step_ms, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": wl.name, "grid": [wl.nx, wl.ny, wl.nz], "elements": wl.n_elems,
                           "nodes": wl.n_nodes, "force_points": wl.n_points, "law": "HO" if wl.mats[0]["law"] else "NH",
                           "variant": args.variant, "parallelism": f"replicas x{world}",
                           "l2": "512 MiB buffer rewritten between timed iterations (L2 flush, untimed)",
                           "elements_per_s": world * wl.n_elems * args.steps / t_dev,
                           "input_sha256": wl.sha256()},
                "clocks": clocks,
                "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "steps": e2e_steps, "api": "ib_coupling_step_host3 (pinned host buffers, u,v,w and fu,fv,fw as one [3][n_cells] array each; the step is pipelined in 8 z-slabs: H2D of u,v,w, fused spread + interpolate per slab, D2H of the finished f layers)"},
                "gpu_launches": int(launches),
                "wall_s_timed_region": t_wall,
                "run_to_run": {"runs": 3, "max_abs_dev_over_max_abs": dev_rr},
                "roofline": roofline,
                "cpu_baseline": {"value": s["n_points"] / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                 "sample": sample,
                                 "all_cores": {"value": s_all["n_points"] / dt_all, "unit": UNIT, "cores": cores,
                                               "kind": "oracle built with -fopenmp (spread: private grid per thread; interpolation over points; FE force serial)",
                                               "sample": f"first {s_all['n_elems']} elements ({s_all['n_points']} force points), {dt_all:.1f} s"}}}
        print(json.dumps(line))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C3")
    ap.add_argument("--variant", type=int, default=1)
    ap.add_argument("--cpu-frac", type=float, default=1.0 / 16, dest="cpu_frac")
    ap.add_argument("--dry-run", action="store_true", dest="dry_run",
                    help="launch and timing plumbing only, on CPU with gloo (tests/test_bench_replicas.py)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return relaunch(args.gpus)
    if args.dry_run:
        return run_dry(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
