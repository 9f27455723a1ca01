#!/usr/bin/env python
"""bench.py -- throughput of the BSL6D split-advection hot path on B200 (driver contract: one JSON line).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload C2]

One *step* = one pass of the whole hot path over the resident distribution function of
BASELINE.json configs[1] (C2: fp64 32^6, degree 7):
    six 1-D sweeps x1,x2,x3 (shift v_d*dt/dx_d) and v1,v2,v3 (shift E_d(x)*dt/dv_d), dt = 0.05      [a1-a4]
    the magnetic rotation as three velocity shears (B along x3, theta = 0.1: configs[3] on the same grid) [a5]
    the density moment rho(x)                                                                          [a6]
sequenced on one stream through the C ABI (a7's job).  `value` counts the 9 sweeps' point updates per second
(the density pass is inside the timed region but adds nothing to the numerator).

Timing: CUDA events on the launching stream, W >= 3 warm-up steps, barrier + synchronize on both sides, max over
ranks.  Inputs (8.6 GB per buffer) are far larger than the 126 MB L2, so no explicit flush is needed.
`--impl reference` times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
Multi-GPU: the path has no exchange step on one node (replicas only) -- every rank runs
an independent replica of the workload, `value` is the aggregate, scaling = weak.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time
from dataclasses import replace

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "fp64 1-D advection sweep Gpoint-updates/s (16 B/point/sweep), whole hot-path step"
UNIT = "Gpoint-updates/s"
ROT_DT = 0.1          # theta = |B| * dt = 0.1 (BASELINE.json configs[3])
ROT_B = (0.0, 0.0, 1.0)


def parse_args():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=10)
    p.add_argument("--warmup", type=int, default=3)
    p.add_argument("--impl", default="ours", choices=("ours", "reference"))
    p.add_argument("--workload", default="C2", help="C1..C5 (C2 = BASELINE configs[1] is the contract workload)")
    p.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end leg")
    p.add_argument("--no-cpu", action="store_true", help="skip the oracle cpu_baseline leg")
    p.add_argument("--no-fused", action="store_true", help="skip the fused-pass variant of the step")
    p.add_argument("--paper-benchmark", action="store_true",
                   help="instead of the contract step: the paper's own section-5 benchmark (37^6, random per-point "
                        "shifts, odd widths 3/5/7/9, every direction) through bsl6d_advect_pointwise")
    return p.parse_args()


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (driver-measured copy)"
    except Exception:
        return 6650.0, "fallback 6.65 TB/s (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------------------------
# clocks during the timed region
# ------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.proc = None
        self.tmp = None

    def start(self):
        try:
            self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        try:
            self.proc.terminate()
            self.proc.wait(timeout=5)
        except Exception:
            pass
        try:
            self.tmp.flush()
            self.tmp.seek(0)
            rows = [r.strip().split(",") for r in self.tmp.read().strip().splitlines() if r.strip()]
            self.tmp.close()
            os.unlink(self.tmp.name)
        except Exception:
            return out
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if r[3 + k].strip().lower().startswith("active"):
                    reasons.add(nm)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), power_w_max=float(max(pw)),
                       reasons=sorted(reasons), samples=len(sm))
        return out


# ------------------------------------------------------------------------------------------------------------
# the step, as a list of ops (shared description; the GPU leg and the oracle leg each execute it their own way)
# ------------------------------------------------------------------------------------------------------------
def step_ops(w):
    """[(name, kind, dim)]: the order of one step."""
    ops = [(nm, "advect", d) for d, nm in enumerate(("x1", "x2", "x3", "v1", "v2", "v3"))]
    ops.append(("rot", "rotate", -1))
    ops.append(("rho", "density", -1))
    return ops


N_SWEEPS = 9          # 6 advect + 3 shears


# ------------------------------------------------------------------------------------------------------------
# multi-rank host logic (replicas only: no data-path collective; covered by a world_size-2 gloo test on CPU)
# ------------------------------------------------------------------------------------------------------------
def max_over_ranks(x: float, device=None) -> float:
    """MAX of a per-rank scalar over the process group (identity without one)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(x)
    t = torch.tensor([float(x)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(npts: int, n_sweeps: int, steps: int, world: int, total_ms: float) -> float:
    """Gpoint-updates/s of the whole job: every rank advanced its own replica; time = max over ranks."""
    return world * n_sweeps * npts * steps / (total_ms * 1e-3) / 1e9


# ------------------------------------------------------------------------------------------------------------
# oracle leg (cpu_baseline and --impl reference): a BOUNDED sample of the same workload on the host cores
# ------------------------------------------------------------------------------------------------------------
class OracleSample:
    """For each op of the step, a crop of the workload's grid (same lo/dx/degree/fields): the swept dim and the
    three v dims keep their full extent, the other x dims are cropped so that a crop holds <= ~6.7e7 points
    (crops of equal shape share their buffers)."""

    def __init__(self, w, target_pts=1 << 26):
        import oracle
        self.oracle = oracle
        self.w = w
        self.cases = []
        shared = {}
        nv = int(np.prod(w.n[3:], dtype=np.int64))
        for name, kind, dim in step_ops(w):
            n = list(w.n)
            if kind == "advect" and dim < 3:
                rest = [d for d in range(3) if d != dim]
                budget = max(1, target_pts // (nv * w.n[dim]))
                c = max(1, int(round(budget ** 0.5)))
                for d in rest:
                    n[d] = min(w.n[d], c)
            else:
                budget = max(1, target_pts // nv)
                c = max(1, int(round(budget ** (1.0 / 3.0))))
                for d in range(3):
                    n[d] = min(w.n[d], c)
            sub = replace(w, n=tuple(n), name=f"{w.name}_crop_{name}")
            if tuple(n) not in shared:
                f = sub.make_f("cpu").numpy()
                shared[tuple(n)] = (f, np.empty_like(f))
            f, out = shared[tuple(n)]
            g = oracle.Grid(tuple(sub.n), tuple(sub.lo), tuple(sub.dx))
            E = sub.E()
            self.cases.append((name, kind, dim, sub, g, f, out, E))
        self.sweep_pts = sum((3 if k == "rotate" else 1) * c[3].npts for c in self.cases for k in [c[1]]
                             if k != "density")
        self.desc = "per op a crop of the %s grid: " % w.name + ", ".join(
            f"{c[0]}:{'x'.join(map(str, c[3].n))}" for c in self.cases)

    def run_once(self):
        o, w = self.oracle, self.w
        t0 = time.perf_counter()
        for name, kind, dim, sub, g, f, out, E in self.cases:
            if kind == "advect":
                o.advect(g, sub.degree, f, dim, None if dim < 3 else E[dim - 3], w.dt, out=out)
            elif kind == "rotate":
                o.rotate(g, sub.degree, f, ROT_B, ROT_DT, out=out)
            else:
                o.density(g, f)
        return time.perf_counter() - t0


def run_reference(args, w):
    """--impl reference: the oracle, as it stands, on the host cores.  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    oracle.build()
    samp = OracleSample(w)
    for _ in range(min(args.warmup, 1)):
        samp.run_once()
    t = 0.0
    for _ in range(args.steps):
        t += samp.run_once()
    val = samp.sweep_pts * args.steps / t / 1e9
    cores = oracle.num_threads()
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"{w.name} {'x'.join(map(str, w.n))} degree {w.degree}: six sweeps + rotation "
                               f"shears + density; oracle on a bounded sample", "sample": samp.desc},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": samp.desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------------------
# GPU leg
# ------------------------------------------------------------------------------------------------------------
def run_ours(args, w):
    import torch
    import torch.distributed as dist
    import paper_2303_05994_b200 as bsl

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    bsl.load_library()                                    # fail loudly if the extension is missing

    dev = torch.device("cuda", local)
    npts = w.npts
    nx = w.n[0] * w.n[1] * w.n[2]
    a = w.make_f(dev)                                     # seeded synthetic f (bsl6d_workloads), resident in HBM
    f0_host = None
    if not args.no_e2e:
        f0_host = torch.empty(w.n, dtype=torch.float64, pin_memory=True)
        f0_host.copy_(a)
    b = torch.empty_like(a)
    rho = torch.empty(w.n[:3], dtype=torch.float64, device=dev)
    E_host = [torch.from_numpy(e) for e in w.E()]
    E = [e.to(dev) for e in E_host]
    ctx = bsl.create(w.n, w.lo, w.dx, w.degree)
    ctx.set_fusion(0)                                     # the graded step: every sweep its own 16 B/point pass
    ops = step_ops(w)
    kernels = {nm: (ctx.kernel_name(d) if kind == "advect" else "") for nm, kind, d in ops}
    kernels["rot"] = f"{ctx.kernel_name(3)} + {ctx.kernel_name(4)} + {ctx.kernel_name(3)}"
    stream = torch.cuda.current_stream()

    def one_step(cur, oth, evs=None):
        for i, (name, kind, dim) in enumerate(ops):
            if evs is not None:
                evs[i].record(stream)
            if kind == "advect":
                ctx.advect(cur, oth, dim, None if dim < 3 else E[dim - 3], w.dt)
                cur, oth = oth, cur
            elif kind == "rotate":
                ctx.rotate(cur, oth, ROT_B, ROT_DT)
                cur, oth = oth, cur
            else:
                ctx.density(cur, rho)
        if evs is not None:
            evs[len(ops)].record(stream)
        return cur, oth

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cur, oth = a, b
    for _ in range(max(args.warmup, 0)):
        cur, oth = one_step(cur, oth)
    barrier()

    K = args.steps
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(len(ops) + 1)] for _ in range(K)]
    l0 = ctx.launch_count()
    clocks = ClockSampler(local)
    clocks.start()
    time.sleep(0.25)
    barrier()
    t_wall = time.perf_counter()
    for s in range(K):
        cur, oth = one_step(cur, oth, evs[s])
    barrier()
    t_wall = time.perf_counter() - t_wall
    # keep the sampler alive for a moment if the region was very short, so that it has samples under load
    clk = clocks.stop()
    launches = ctx.launch_count() - l0
    total_ms = evs[0][0].elapsed_time(evs[K - 1][len(ops)])
    per_op = {nm: float(np.mean([evs[s][i].elapsed_time(evs[s][i + 1]) for s in range(K)]))
              for i, (nm, _, _) in enumerate(ops)}
    assert torch.isfinite(rho).all()

    total_ms = max_over_ranks(total_ms, dev)
    value = whole_job_value(npts, N_SWEEPS, K, world, total_ms)
    step_bytes = (N_SWEEPS * 16 * npts + 8 * npts + 8 * nx)

    # ---- roofline of the dominant kernel: the strided sweep (x1,x2,x3,v1,v2 + the three shears = 8 launches/step)
    peak, peak_src = peaks()
    strided_ms = sum(per_op[nm] for nm in ("x1", "x2", "x3", "v1", "v2", "rot")) / 8.0
    achieved = 16.0 * npts / (strided_ms * 1e-3) / 1e9
    per_dim = {}
    for nm, kind, _ in ops:
        nl = 3 if kind == "rotate" else 1
        bytes_ = (8 * npts + 8 * nx) if kind == "density" else 16 * npts * nl
        gbs = bytes_ / (per_op[nm] * 1e-3) / 1e9
        per_dim[nm] = {"ms": per_op[nm], "GB/s": gbs, "frac_of_measured_peak": gbs / peak,
                       "frac_of_8TBs": gbs / 8000.0, "kernel": kernels.get(nm, "")}
        if kind != "density":
            per_dim[nm]["Gpoint-updates/s"] = nl * npts / (per_op[nm] * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.csv")         # copied from an `ncu --set full` capture (traffic.md)
    if os.path.exists(tpath):
        try:
            with open(tpath) as fh:
                for ln in fh.read().splitlines()[1:]:
                    c = ln.split(",")
                    if c[0] == w.name and c[1] == "sweep_strided_kernel":
                        traffic = float(c[2])
        except Exception:
            traffic = None
    roofline = {"bound": "hbm", "kernel": "sweep_strided_kernel (8 of 10 launches per step)", "achieved": achieved,
                "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": 16 * npts, "avg_launch_ms": strided_ms,
                "step_GB/s": step_bytes / (total_ms / K * 1e-3) / 1e9,
                "step_frac": step_bytes / (total_ms / K * 1e-3) / 1e9 / peak}

    # ---- the same step with the planner's fused passes: extra information, not `value` --------
    fused = None
    if not args.no_fused:
        ctx.set_fusion(1)
        six = [(d, None, 0, w.dt / w.dx[d]) for d in range(3)] + \
              [(3 + d, E[d], 0x7, w.dt / w.dx[3 + d]) for d in range(3)]

        def fused_step(cur, oth):
            ctx.advect_seq(cur, oth, six)
            ctx.rotate(oth, cur, ROT_B, ROT_DT)
            ctx.density(cur, rho)
            return cur, oth

        for _ in range(3):
            cur, oth = fused_step(cur, oth)
        barrier()
        lf0 = ctx.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(K):
            cur, oth = fused_step(cur, oth)
        e1.record(stream)
        barrier()
        fms = max_over_ranks(e0.elapsed_time(e1), dev)
        fused = {"value": whole_job_value(npts, N_SWEEPS, K, world, fms), "unit": UNIT, "ms_per_step": fms / K,
                 "launches_per_step": (ctx.launch_count() - lf0) // K, "speedup_vs_value": (total_ms / K) / (fms / K),
                 "note": "same nine sweeps + density, bit-identical results; consecutive sweeps over two dims share one "
                         "pass over f (bsl6d_advect_seq: x1 | x2+x3 | v1+v2 | v3; bsl6d_rotate: one pass), so bytes per "
                         "point-update drop below 16 and the per-sweep roofline does not apply"}
        # the full Strang step of BASELINE configs[4] on this grid (12 sweeps; x half, E, rotation, x half)
        def time_strang(mode):
            ctx.set_fusion(mode)
            l0_ = ctx.launch_count()
            for _ in range(2):
                ctx.strang_step(cur, oth, E, ROT_B, w.dt)
            barrier()
            per = (ctx.launch_count() - l0_) // 2
            s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s0.record(stream)
            for _ in range(K):
                ctx.strang_step(cur, oth, E, ROT_B, w.dt)
            s1.record(stream)
            barrier()
            return max_over_ranks(s0.elapsed_time(s1), dev) / K, per

        st_f, lp_f = time_strang(1)
        st_u, lp_u = time_strang(0)
        fused["strang_step"] = {"ms_fused": st_f, "launches_fused": lp_f, "ms_per_sweep_path": st_u,
                                "launches_per_sweep_path": lp_u,
                                "Gpoint-updates/s_fused": 12 * npts / (st_f * 1e-3) / 1e9,
                                "Gpoint-updates/s_per_sweep_path": 12 * npts / (st_u * 1e-3) / 1e9}
        ctx.set_fusion(0)

    # ---- e2e: the same step through bsl6d_run_host on HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        del a, b, cur, oth
        torch.cuda.empty_cache()
        hops = []
        for name, kind, dim in ops:
            if kind == "advect":
                hops.append({"kind": "advect", "dim": dim, "dt": w.dt,
                             "shift_source": None if dim < 3 else E_host[dim - 3]})
            elif kind == "rotate":
                hops.append({"kind": "rotate", "B": ROT_B, "dt": ROT_DT})
            else:
                hops.append({"kind": "density", "rho_host": torch.empty(w.n[:3], dtype=torch.float64,
                                                                           pin_memory=True)})
        ke = max(1, min(K, 5))
        ctx.run_host(f0_host, f0_host, hops)              # warm-up (allocates the context's device buffer)
        barrier()
        t0 = time.perf_counter()
        for _ in range(ke):
            ctx.run_host(f0_host, f0_host, hops)
        torch.cuda.synchronize()
        te = time.perf_counter() - t0
        te = max_over_ranks(te, dev)
        e2e = {"value": whole_job_value(npts, N_SWEEPS, ke, world, 1e3 * te), "unit": UNIT,
               "h2d_bytes_per_step": 8 * npts + 3 * 8 * nx, "d2h_bytes_per_step": 8 * npts + 8 * nx,
               "steps": ke, "ms_per_step": 1e3 * te / ke, "api": "bsl6d_run_host (pinned host buffers)"}
    ctx.destroy()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        import oracle
        oracle.build()
        samp = OracleSample(w)
        npass = 3
        tc = sum(samp.run_once() for _ in range(npass))
        cpu = {"value": npass * samp.sweep_pts / tc / 1e9, "passes": npass, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
               "sample": samp.desc, "seconds": tc}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{w.name} (BASELINE configs[1]) fp64 {'x'.join(map(str, w.n))}, degree "
                                   f"{w.degree}: sweeps x1,x2,x3,v1,v2,v3 (dt={w.dt}) + rotation shears v1,v2,v1 "
                                   f"(theta={ROT_DT}) + density, per replica",
                       "l2": (f"inputs ({8 * npts / 1e9:.1f} GB per buffer) larger than the 126 MB L2; no flush"
                              if 8 * npts > 2 * 126e6 else
                              f"inputs ({8 * npts / 1e6:.1f} MB per buffer) fit in the 126 MB L2: launch-latency-bound, "
                              "NOT an HBM measurement"),
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "wall_ms_per_step": 1e3 * t_wall / K},
            "clocks": clk, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
            "cpu_baseline": cpu, "fused_step": fused, "per_dim": per_dim,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_paper_benchmark(args):
    """one 1-D interpolation per direction on 37^6 points, random alpha/dx in [-1,1] per
    point, odd stencil widths.  Reports, per width and direction, the time and GB/s in the paper's convention
    (16 B/point: f read + f written, eq (8)) and with the alpha array counted (24 B/point)."""
    import torch
    import bsl6d_workloads as wl
    import paper_2303_05994_b200 as bsl
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device")
    torch.cuda.set_device(0)
    bsl.load_library()
    w = wl.P37
    f = w.make_f("cuda")
    alpha = wl.random_shifts(w.n, w.seed + 1, device="cuda")
    out = torch.empty_like(f)
    ctx = bsl.create(w.n, w.lo, w.dx, w.degree)
    stream = torch.cuda.current_stream()
    K = max(1, args.steps)
    res = {}
    clocks = ClockSampler(0)
    clocks.start()
    for q in (3, 5, 7, 9):
        row = {}
        for dim, nm in enumerate(("x1", "x2", "x3", "v1", "v2", "v3")):
            for _ in range(max(args.warmup, 1)):
                ctx.advect_pointwise(f, out, dim, alpha, q)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(K):
                ctx.advect_pointwise(f, out, dim, alpha, q)
            e1.record(stream)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / K
            row[nm] = {"ms": ms, "GB/s_16B_per_point": 16 * w.npts / ms / 1e6, "GB/s_24B_per_point": 24 * w.npts / ms / 1e6,
                       "Gpoint-updates/s": w.npts / ms / 1e6}
        res[f"q{q}"] = row
    clk = clocks.stop()
    ctx.destroy()
    peak, peak_src = peaks()
    allv = [v["GB/s_24B_per_point"] for r in res.values() for v in r.values()]
    line = {"metric": "paper section-5 benchmark: 1-D Lagrange interpolation per direction, 37^6 fp64 points, random "
                      "per-point shifts in [-1,1] cells, odd widths (GB/s; paper's convention 16 B/point)",
            "unit": "GB/s", "n_gpus": 1, "steps": K, "warmup": max(args.warmup, 1), "dtype": "f64", "data": "synthetic",
            "config": {"workload": "P37 37x37x37x37x37x37 (PAPER.md:194, 244), alpha array resident (24 B/point moved)"},
            "value": float(np.mean([v["GB/s_16B_per_point"] for r in res.values() for v in r.values()])),
            "mean_GB/s_24B": float(np.mean(allv)), "min_GB/s_24B": float(min(allv)), "max_GB/s_24B": float(max(allv)),
            "peak": peak, "peak_source": peak_src, "frac_of_peak_24B": float(np.mean(allv)) / peak,
            "paper_context": {"V100": "almost 500 GB/s", "Xeon Gold 6148 node": "around 100 GB/s", "cite": "PAPER.md:11"},
            "clocks": clk, "per_width": res}
    print(json.dumps(line), flush=True)


def main():
    args = parse_args()
    if args.paper_benchmark:
        run_paper_benchmark(args)
        return
    import bsl6d_workloads as wl
    w = wl.CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, w)
    else:
        run_ours(args, w)


if __name__ == "__main__":
    main()
