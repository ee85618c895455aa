#!/usr/bin/env python
"""bench.py — batched ADMM-MPC solves/s at B=4096, N=50, 100 fixed iterations (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 2]
                    [--method auto|srb|dense] [--B ..] [--N ..]

A "step" is one pinmpc_solve of the whole batch: assembly + factorisation + all ADMM iterations
 on synthetic inputs (gen/) that are resident in HBM when the timed region
starts.  Timing: CUDA events on the launching stream around every step, an L2 flush (256 MiB write)
between steps, max over ranks.  `e2e` repeats the measurement through the public API with HOST
(pinned) buffers: H2D copies of every input and D2H reads of x,u,residuals inside the timed region.
`--gpus N` (under torchrun) runs N independent replicas: the path does not shard across GPUs
(replicas only, no collective on the data path).
`--impl reference` times the fp64 CPU oracle (oracle/) on the host cores, a bounded sample per step.
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

METRIC = "batched ADMM-MPC solves/s at B=4096,N=50 (fixed iters); % of roofline"

# Algorithmic FLOPs of the formulation shipped (structured 6-D-input LQR): one stage of one ADMM
# iteration without the wrench projections, plus 95 per foot in stance (the exact projection of one 6-D wrench; a swing
# foot projects to 0 for free), counted from the workload's own contact flags
FLOP_PER_STAGE_ITER_BASE = {12: 740.0, 18: 960.0}
FLOP_PER_PROJECTION = 95.0
FLOP_PER_STAGE_ONCE = {12: 3900.0, 18: 4700.0}    # assembly + factorisation, once per solve
# dense-generic count of SURVEY.md 8(d), used when --method dense is timed
FLOP_DENSE_ITER = {12: 2700.0, 18: 3700.0}
FLOP_DENSE_ONCE = {12: 33000.0, 18: 60000.0}
FMA_LANES_PER_SM = 128
# DRAM bytes (read + write) of one launch of the dominant kernel from an `ncu --set full` capture: written by
# `bench.py --write-traffic <ncu raw csv>` together with a hash of the kernel sources it was measured on; reported only
# while that hash still matches the sources (else null)
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "r2_traffic.json")


def source_hash():
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2606_05687_b200", "csrc")
    # the sources the dominant kernel (k_iterate_tm) is compiled from
    for f in ("pinmpc_common.cuh", "pinmpc_srb_math.cuh", "pinmpc_tmem.cu"):
        h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def measured_traffic(workload):
    try:
        t = json.load(open(TRAFFIC_JSON))
    except (OSError, ValueError):
        return None
    return t.get("dram_bytes") if t.get("workload") == workload and t.get("source_hash") == source_hash() else None


def write_traffic(csv_path, workload):
    """Parse `ncu -i x.ncu-rep --page raw --csv` of the dominant kernel and record its DRAM traffic per launch."""
    import csv
    rows = list(csv.reader(open(csv_path)))
    hdr, units, vals = rows[0], rows[1], rows[2]
    col = {n: i for i, n in enumerate(hdr)}
    mult = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}

    def get(name):
        return float(vals[col[name]].replace(",", "")) * mult[units[col[name]]]
    out = {"workload": workload, "kernel": vals[col["Kernel Name"]], "source_hash": source_hash(),
           "dram_bytes": get("dram__bytes_read.sum") + get("dram__bytes_write.sum"),
           "dram_bytes_read": get("dram__bytes_read.sum"), "dram_bytes_write": get("dram__bytes_write.sum"),
           "gpu_time_ms": float(vals[col["gpu__time_duration.sum"]].replace(",", "")) * {"ns": 1e-6, "us": 1e-3, "ms": 1.0}[units[col["gpu__time_duration.sum"]]]}
    json.dump(out, open(TRAFFIC_JSON, "w"), indent=1)
    print(json.dumps(out))


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--method", default="auto", choices=["auto", "srb", "dense"])
    ap.add_argument("--B", type=int, default=None)
    ap.add_argument("--N", type=int, default=None)
    ap.add_argument("--envs-per-cta", type=int, default=0, help="tuning knob of the structured solver (0 = auto)")
    ap.add_argument("--sweep", action="store_true", help="BASELINE.json config 4: B x N table (one JSON line per point)")
    ap.add_argument("--split", action="store_true",
                    help="time the paper's own stage-local ADMM (pinmpc_split_solve) on the config instead (one JSON line)")
    ap.add_argument("--split-scaled", action="store_true", help="--split with the variable scaling Sx = Q^-1/2, su = 100 (DESIGN.md 7c)")
    ap.add_argument("--split-accel", action="store_true", help="--split with Nesterov acceleration and restart")
    ap.add_argument("--centroidal", action="store_true",
                    help="--split on the paper's own 9-state centroidal model (eq. (1)-(4)) with the state box of gen.centroidal_view, scaled")
    ap.add_argument("--converge", action="store_true",
                    help="iterations to tolerance x ms per iteration for the exact-dynamics path and the stage-local method (one JSON line per setting)")
    ap.add_argument("--split-sweep", action="store_true",
                    help="scalability table of the stage-local method like the paper's Fig. 3: envs x horizon up to N = 400")
    ap.add_argument("--chunks", type=int, default=0, help="horizon chunks of the equality step (0 = auto, 1 = sequential-pass kernel)")
    ap.add_argument("--write-traffic", default=None, metavar="NCU_RAW_CSV",
                    help="record the DRAM traffic of the dominant kernel from an ncu raw-page csv into profiles/r2_traffic.json and exit")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.th.join(timeout=2)
        sm, mx, reasons = [], None, set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def probe_fma(blocks, iters, d_out, stream):
    """Bench-only helper library (csrc/bench_probe.cu): enqueue `blocks` CTAs x 256 threads x 128*iters FMAs, return the FLOPs."""
    import ctypes
    lib = ctypes.CDLL(os.path.join(ROOT, "paper_2606_05687_b200", "libpinmpc_benchprobe.so"))
    lib.bench_probe_fma.restype = ctypes.c_double
    lib.bench_probe_fma.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
    return float(lib.bench_probe_fma(int(blocks), int(iters), ctypes.c_void_p(d_out.data_ptr()), ctypes.c_void_p(stream)))


def max_over_ranks(values, dist, device):
    """Replicas only: the one collective of a multi-GPU run is this MAX of the per-rank
    step times; `value` is then (envs of all ranks) / (the slowest rank's time)."""
    import torch
    if dist is None:
        return [float(v) for v in values]
    t = torch.tensor([float(v) for v in values], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def aggregate_value(envs_per_rank, world, ms):
    """Whole-job throughput of `world` replicas of `envs_per_rank` envs that all finished within `ms`."""
    return envs_per_rank * world / (ms * 1e-3)


def flop_per_stage_iter(w):
    """Algorithmic FLOPs of one stage of one ADMM iteration for this workload (projections counted per stance foot)."""
    feet = float(w.contact[..., :2].astype("float64").sum() / (w.B * w.N))
    return FLOP_PER_STAGE_ITER_BASE[w.nu] + FLOP_PER_PROJECTION * feet


def flops_per_solve(w, method):
    st = w.B * w.N
    if method == "dense":
        return st * (FLOP_DENSE_ONCE[w.nu] + w.iters * FLOP_DENSE_ITER[w.nu])
    return st * (FLOP_PER_STAGE_ONCE[w.nu] + w.iters * flop_per_stage_iter(w))


def time_oracle(w, n_envs, threads=0):
    import numpy as np
    import gen
    import oracle
    sub = gen.subset(w, np.arange(min(n_envs, w.B)))
    t0 = time.perf_counter()
    oracle.solve(sub, nthreads=threads)
    return sub.B, time.perf_counter() - t0


def run_reference(args):
    """The oracle, as it stands, on the host cores: each step solves a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import gen
    import oracle
    oracle.build()
    w = gen.make_config(args.config, B=args.B, N=args.N)
    n = min(w.B, 128)
    for _ in range(args.warmup):
        time_oracle(w, n)
    t = 0.0
    for _ in range(args.steps):
        t += time_oracle(w, n)[1]
    ms = 1e3 * t / args.steps
    val = n / (ms * 1e-3)
    sample = f"first {n} of {w.B} envs of {w.name} per step, all {w.iters} iterations, fp64"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": "solves/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "B": w.B, "N": w.N, "iters": w.iters, "nu": w.nu, "sample_envs_per_step": n},
        "cpu_baseline": {"value": val, "unit": "solves/s", "cores": oracle.max_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "solves/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def run_split(args):
    """The paper's own stage-local ADMM (eq. (18)-(22), pinmpc_split_solve) on the same workload: dynamics
    assembled on the device once (untimed), then factorisation + iters x (two stage-parallel kernels).  HBM-bound by
    construction in this first version: H_k, G_k, A_k, B_k are streamed every iteration."""
    import numpy as np
    import torch
    import gen
    from paper_2606_05687_b200 import Solver, SplitSolver, make_layout
    dev = torch.device("cuda", 0)
    stream = torch.cuda.current_stream(dev)
    w = gen.make_config(args.config, B=args.B, N=args.N)
    lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)
    s = Solver(w.nu, w.N, w.B, layout=lay, rho=w.rho, iters=w.iters, Qdiag=w.Qdiag, Rdiag=w.Rdiag, dt=w.dt, device=dev)
    s.set_workload(w)
    A, Bm, c = s.get_dynamics()
    d = lambda a, t=torch.float32: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev, t)
    x0, x_ref, u_ref, contact = d(w.x0), d(w.x_ref), d(w.u_ref), d(w.contact, torch.uint8)
    opts = {}
    Qd, nx = w.Qdiag, 13
    if args.centroidal:
        from paper_2606_05687_b200 import binding
        v = gen.centroidal_view(w)
        A, Bm, c = binding.assemble_centroidal(w.n_wrench, w.n_force, w.dt, d(w.mass), d(w.foot_r))
        x0, x_ref, Qd, nx = d(v["x0"]), d(v["x_ref"]), v["Qdiag"], 9
        opts.update(nx=9, x_lo=v["x_lo"], x_hi=v["x_hi"], scale_x=[1.0 / float(q) ** 0.5 for q in Qd], scale_u=100.0)
    if args.split_scaled and not args.centroidal:
        opts.update(scale_x=split_scale_x(w), scale_u=100.0)
    if args.split_accel:
        opts.update(accel=True)
    sp = SplitSolver(w.nu, w.N, w.B, lay, Qd, w.Rdiag, w.rho, w.iters, device=dev, **opts)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    run = lambda: sp.solve(A, Bm, c if (w.ext_wrench is not None or args.centroidal) else None, x0, None, x_ref, u_ref, contact)
    for _ in range(max(args.warmup, 3)):
        run()
    torch.cuda.synchronize(dev)
    ts = []
    for _ in range(args.steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream); run(); b.record(stream)
        torch.cuda.synchronize(dev)
        ts.append(a.elapsed_time(b))
    ms = float(np.mean(ts))
    n = nx + w.nu
    st = w.B * w.N
    # algorithmic bytes per stage-iteration: (21a) reads H_k (n^2), G_k (nu^2), B_k (nx nu), [A_{k+1} B_{k+1}] (nx n);
    # (21b,c) reads [A_k B_k]^T (nx n); lifted vectors: 6 read + xi, du written in (21a), 5 read + 5 written in (21b,c)
    per_stage_iter = 4 * (n * n + w.nu * w.nu + nx * w.nu + 2 * nx * n + 18 * n)
    gbs = per_stage_iter * st * w.iters / (ms * 1e-3) / 1e9
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except OSError:
        peaks = {"hbm_gbs": 6540.0}                            # fallback of the profiling guide
    print(json.dumps({"metric": "stage-local ADMM (paper eq. 22) solves/s", "value": w.B / (ms * 1e-3), "unit": "solves/s",
                      "ms_per_step": ms, "steps": args.steps, "n_gpus": 1, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": w.name, "B": w.B, "N": w.N, "iters": w.iters, "nu": w.nu, "method": "split",
                                 "scaled": bool(args.split_scaled or args.centroidal), "accel": bool(args.split_accel),
                                 "model": "centroidal 9-state (eq. 1-4), state box" if args.centroidal else "SRB 13-state"},
                      "stage_iters_per_s": st * w.iters / (ms * 1e-3), "gpu_launches": sp.launch_count(),
                      "roofline": {"bound": "hbm", "achieved": gbs, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                                   "frac": gbs / peaks["hbm_gbs"],
                                   # dram read + write of one k_split_a plus one k_split_b launch (one iteration),
                                   # ncu --set full, profiles/r1_split_ncu.md; measured at config 2 only
                                   "traffic": (1016841000 + 31662592 + 358631936 + 81859584) if (w.name == "c2_long_horizon" and not opts) else None,
                                   "traffic_unit": "bytes per iteration (both kernels)",
                                   "bytes_per_stage_iter": per_stage_iter, "scope": "whole solve (factorisation + all iterations)"},
                      "workspace_mb": sp.workspace_bytes / 1e6, "r_prim_max": float(sp.r_prim.max())}))


def split_scale_x(w):
    """Sx = Q^-1/2 (1 where Q = 0): the state scaling of the iterations-to-tolerance pin (tests/test_oracle_split.py)."""
    return [1.0 / float(q) ** 0.5 if q > 0 else 1.0 for q in w.Qdiag]


def run_converge(args):
    """Iterations to tolerance x time per iteration, both methods, full-size workload.
    Reference point: the exact-dynamics path run to convergence (rho = 1e-3, 20000 iterations); error of a run =
    max(|u - u*|_inf / (1 + |u*|_inf), |x - x*|_inf / (1 + |x*|_inf)) per env; a setting has reached eps when the median
    env has.  Iteration counts are scanned on a geometric grid (every run starts from zero), so "iters_to" is the
    first grid point at or below eps."""
    import numpy as np
    import torch
    import gen
    from paper_2606_05687_b200 import Solver, SplitSolver, make_layout
    dev = torch.device("cuda", 0)
    stream = torch.cuda.current_stream(dev)
    w = gen.make_config(args.config, B=args.B, N=args.N)
    lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)
    grid = [25, 50, 100, 200, 400, 800, 1600, 3200, 6400]

    def timed(fn):
        fn(); torch.cuda.synchronize(dev)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream); fn(); b.record(stream)
        torch.cuda.synchronize(dev)
        return a.elapsed_time(b)

    def exact(rho, iters):
        s = Solver(w.nu, w.N, w.B, layout=lay, rho=rho, iters=iters, Qdiag=w.Qdiag, Rdiag=w.Rdiag, dt=w.dt, device=dev)
        s.set_workload(w)
        ms = timed(s.solve)
        o = s.get()
        x, u = o["x"].clone(), o["u"].clone()
        s.close()
        return x, u, ms

    xs, us, _ = exact(1e-3, 20000)
    nx_ = 1 + xs.abs().amax(dim=(1, 2)); nu_ = 1 + us.abs().amax(dim=(1, 2))

    def err(x, u):
        e = torch.maximum((x - xs).abs().amax(dim=(1, 2)) / nx_, (u - us).abs().amax(dim=(1, 2)) / nu_)
        return float(e.median()), float(e.quantile(0.95))

    def report(name, runs):
        rec = {"converge": name, "workload": w.name, "B": w.B, "N": w.N, "grid": []}
        for it, (x, u, ms) in runs:
            med, p95 = err(x, u)
            rec["grid"].append({"iters": it, "ms": ms, "err_median": med, "err_p95": p95})
        for eps in (1e-2, 1e-3):
            hit = next((g for g in rec["grid"] if g["err_median"] <= eps), None)
            rec[f"iters_to_{eps:g}"] = hit["iters"] if hit else None
            rec[f"ms_to_{eps:g}"] = hit["ms"] if hit else None
        rec["ms_per_iter"] = rec["grid"][-1]["ms"] / rec["grid"][-1]["iters"]
        print(json.dumps(rec), flush=True)

    for rho in (1.0, 1e-1, 1e-2, 1e-3):
        runs = []
        for it in grid:
            runs.append((it, exact(rho, it)))
            if err(*runs[-1][1][:2])[0] <= 1e-3:
                break
        report(f"exact-dynamics ADMM (product path), rho = {rho:g}", runs)

    s = Solver(w.nu, w.N, w.B, layout=lay, rho=w.rho, iters=1, Qdiag=w.Qdiag, Rdiag=w.Rdiag, dt=w.dt, device=dev)
    s.set_workload(w)
    A, Bm, c = s.get_dynamics()
    d = lambda a, t=torch.float32: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev, t)
    x0, x_ref, u_ref, contact = d(w.x0), d(w.x_ref), d(w.u_ref), d(w.contact, torch.uint8)
    u_prev = u_ref[:, 0].contiguous()
    for name, opts in (("stage-local ADMM, unscaled, rho = 1", {}),
                       ("stage-local ADMM, Sx = Q^-1/2, su = 100, rho = 1", dict(scale_x=split_scale_x(w), scale_u=100.0)),
                       ("stage-local ADMM, scaled, accelerated with restart", dict(scale_x=split_scale_x(w), scale_u=100.0, accel=True))):
        runs = []
        for it in grid:
            sp = SplitSolver(w.nu, w.N, w.B, lay, w.Qdiag, w.Rdiag, 1.0, it, device=dev, **opts)
            fn = lambda: sp.solve(A, Bm, c if w.ext_wrench is not None else None, x0, u_prev, x_ref, u_ref, contact)
            ms = timed(fn)
            z = sp.z
            runs.append((it, (z[:, :, :13].clone(), z[:, :, 13:].clone(), ms)))
            del sp
            if err(*runs[-1][1][:2])[0] <= 1e-3:
                break
        report(name, runs)


def device_dynamics(w, lay, dev):
    """A_k, B_k, c_k of workload w assembled on the device by the library (pinmpc_get_dynamics).  The assembly is
    stage-local, so horizons beyond PINMPC_N_MAX are assembled as B * ceil(N / 200) shorter pseudo-envs and viewed back."""
    import numpy as np
    import torch
    from paper_2606_05687_b200 import Solver
    B, N = w.B, w.N
    parts = 1 if N <= 256 else -(-N // 200)
    while N % parts:
        parts += 1
    n1 = N // parts
    s = Solver(w.nu, n1, B * parts, layout=lay, rho=w.rho, iters=1, Qdiag=w.Qdiag, Rdiag=w.Rdiag, dt=w.dt, device=dev)
    rs = lambda a: None if a is None else np.ascontiguousarray(a.reshape((B * parts, n1) + a.shape[2:]))
    rep = lambda a: np.ascontiguousarray(np.repeat(a, parts, axis=0))
    s.set_problem(rep(w.x0), rs(w.x_ref), rs(w.u_ref), rs(w.contact), rs(w.foot_r), rs(w.yaw), rep(w.mass), rep(w.inertia),
                  rs(w.ext_wrench))
    A, Bm, c = s.get_dynamics()
    torch.cuda.synchronize(dev)
    s.close()
    return A.view(B, N, 13, 13), Bm.view(B, N, 13, w.nu), c.view(B, N, 13)


def run_split_sweep(args):
    """Scalability of the stage-local method over envs x horizon (Fig. 3: "even to N=400"; 200
    iterations is the paper's maximum iteration count for it).  One JSON line per point."""
    import numpy as np
    import torch
    import gen
    from paper_2606_05687_b200 import SplitSolver, make_layout
    dev = torch.device("cuda", 0)
    stream = torch.cuda.current_stream(dev)
    iters = 200
    for B in (256, 1024, 4096):
        for N in (10, 50, 100, 200, 400):
            w = gen.make_config(4, B=B, N=N, iters=iters)
            lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)
            A, Bm, _ = device_dynamics(w, lay, dev)
            d = lambda a, t=torch.float32: torch.from_numpy(np.ascontiguousarray(a)).to(dev, t)
            x0, x_ref, u_ref, contact = d(w.x0), d(w.x_ref), d(w.u_ref), d(w.contact, torch.uint8)
            sp = SplitSolver(w.nu, N, B, lay, w.Qdiag, w.Rdiag, w.rho, iters, device=dev)
            run = lambda: sp.solve(A, Bm, None, x0, None, x_ref, u_ref, contact)
            run(); torch.cuda.synchronize(dev)
            ts = []
            for _ in range(3):
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream); run(); b.record(stream)
                torch.cuda.synchronize(dev)
                ts.append(a.elapsed_time(b))
            ms = float(np.median(ts))
            print(json.dumps({"split_sweep": w.name, "B": B, "N": N, "iters": iters, "ms_per_solve": ms,
                              "solves_per_s": B / (ms * 1e-3), "stage_iters_per_s": B * N * iters / (ms * 1e-3),
                              "workspace_mb": sp.workspace_bytes / 1e6, "dynamics_mb": (A.numel() + Bm.numel()) * 4 / 1e6,
                              "r_prim_max": float(sp.r_prim.max())}), flush=True)
            del sp, A, Bm
            torch.cuda.empty_cache()


def run_sweep(args):
    """BASELINE.json config 4: B in {1024, 4096, 16384, 65536} x N in {10, 25, 50, 100}, 100 iterations, fp32:
    solves/s, achieved FP32 and HBM rates and the device-memory footprint of every point; then the long horizons
    N in {200, 400} of PAPER.md Fig. 3 (L277-279, "even to N = 400" L314) at B in {1024, 4096, 16384}."""
    import numpy as np
    import torch
    import gen
    from paper_2606_05687_b200 import METHOD_SRB, Solver, make_layout
    dev = torch.device("cuda", 0)
    stream = torch.cuda.current_stream(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    grid = [(B, N) for B in (1024, 4096, 16384, 65536) for N in (10, 25, 50, 100)]
    grid += [(B, N) for B in (1024, 4096, 16384) for N in (200, 400)]
    for B, N in grid:
        if True:
            w = gen.make_config(4, B=B, N=N)
            lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)
            s = Solver(w.nu, w.N, w.B, layout=lay, rho=w.rho, iters=w.iters, Qdiag=w.Qdiag, Rdiag=w.Rdiag, dt=w.dt,
                       method=METHOD_SRB, device=dev)
            s.set_workload(w)
            if args.chunks:
                s.set_horizon_chunks(args.chunks)
            for _ in range(3):
                s.solve()
            torch.cuda.synchronize(dev)
            ts = []
            for _ in range(max(args.steps // 4, 3)):
                flush.zero_()
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a.record(stream); s.solve(); b.record(stream)
                torch.cuda.synchronize(dev)
                ts.append(a.elapsed_time(b))
            ms = float(np.median(ts))
            inputs = sum(getattr(w, n).nbytes for n in gen.Workload.ARRAYS if getattr(w, n) is not None)
            io_bytes = inputs + w.B * w.N * (13 + 3 * w.nu) * 4 + w.B * 12
            G_used, C_used = s.launch_shape()
            print(json.dumps({"sweep": w.name, "B": B, "N": N, "iters": w.iters, "envs_per_cta": G_used, "horizon_chunks": C_used, "ms_per_solve": ms,
                              "solves_per_s": B / (ms * 1e-3), "stage_iters_per_s": B * N * w.iters / (ms * 1e-3),
                              "tflops": flops_per_solve(w, "srb") / (ms * 1e-3) / 1e12,
                              "hbm_gbs_algorithmic": io_bytes / (ms * 1e-3) / 1e9,
                              "footprint_mb": (s.workspace_bytes + inputs) / 2 ** 20}), flush=True)
            s.close()
            del s, w
            torch.cuda.empty_cache()


def main():
    args = parse()
    if args.write_traffic:
        import gen
        return write_traffic(args.write_traffic, gen.make_config(args.config, B=args.B, N=args.N).name)
    if args.impl == "reference":
        return run_reference(args)
    if args.split or args.centroidal:
        return run_split(args)
    if args.split_sweep:
        return run_split_sweep(args)
    if args.converge:
        return run_converge(args)
    if args.sweep:
        return run_sweep(args)

    import numpy as np
    import torch
    import gen
    from paper_2606_05687_b200 import METHOD_AUTO, METHOD_DENSE, METHOD_SRB, Solver, binding, make_layout

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    w = gen.make_config(args.config, B=args.B, N=args.N)
    method = {"auto": METHOD_AUTO, "srb": METHOD_SRB, "dense": METHOD_DENSE}[args.method]
    mname = "dense" if args.method == "dense" else "srb"
    lay = make_layout(w.n_wrench, w.n_force, w.mu, w.fz_max, w.mx_coef, w.my_coef, w.mz_coef, w.hand_fmax)
    s = Solver(w.nu, w.N, w.B, layout=lay, rho=w.rho, iters=w.iters, Qdiag=w.Qdiag, Rdiag=w.Rdiag, dt=w.dt,
               method=method, device=dev)
    s.set_workload(w)
    if args.envs_per_cta:
        s.set_tuning(args.envs_per_cta)
    if args.chunks:
        s.set_horizon_chunks(args.chunks)
    stream = torch.cuda.current_stream(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def timed(fn, steps):
        evs = []
        for _ in range(steps):
            flush.zero_()                                   # L2 flush, outside the per-step events
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream); fn(); b.record(stream)
            evs.append((a, b))
        torch.cuda.synchronize(dev)
        return [a.elapsed_time(b) for a, b in evs]

    # ---- device-resident timing ------------------------------------------------------------------
    for _ in range(max(args.warmup, 3)):
        s.solve()
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    kernel_ms = []
    profiled = mname == "srb"
    if profiled:
        s.set_profiling(True)

    def solve_profiled():
        s.solve()

    ms_steps = timed(solve_profiled, args.steps)
    if profiled:
        # events of the last solve only are kept by the handle; re-run K solves reading them one by one
        # (same kernels, same stream, device-resident inputs; outside the timed region above)
        for _ in range(args.steps):
            flush.zero_()
            s.solve()
            kernel_ms.append(s.kernel_ms())
        s.set_profiling(False)
    barrier()
    clocks = sampler.stop() if sampler else None
    launches = s.launch_count() * args.steps
    ms = float(np.mean(ms_steps))

    # ---- end to end through the public API with host buffers ----------------------------------------
    shape = s.launch_shape() if mname == "srb" else (None, None)     # (envs per CTA, horizon chunks) of the timed launches
    e2e = None
    if not args.no_e2e:
        names = [n for n in gen.Workload.ARRAYS if getattr(w, n) is not None]
        host = {n: torch.from_numpy(getattr(w, n)).pin_memory() for n in names}
        devbuf = {n: torch.empty_like(host[n], device=dev) for n in names}
        s.set_problem(**{n: devbuf.get(n) for n in gen.Workload.ARRAYS})
        for n in names:
            devbuf[n].copy_(host[n], non_blocking=True)
        s.solve()
        out_dev = s.get()
        out_host = {k: torch.empty_like(v, device="cpu").pin_memory() for k, v in out_dev.items()}
        h2d = sum(host[n].numel() * host[n].element_size() for n in names)
        d2h = sum(v.numel() * v.element_size() for v in out_host.values())

        def step_e2e():
            for n in names:
                devbuf[n].copy_(host[n], non_blocking=True)
            s.solve()
            binding.pinmpc_get(s.h, out_dev["x"], out_dev["u"], out_dev["r_prim"], out_dev["r_dual"],
                               out_dev["iters_done"], stream.cuda_stream)
            for k in out_host:
                out_host[k].copy_(out_dev[k], non_blocking=True)

        for _ in range(3):
            step_e2e()
        barrier()
        ms_e2e_serial = float(np.mean(timed(step_e2e, args.steps)))
        barrier()

        # The same through three streams: the copies of step i+1 / i-1 overlap the solve of step i (double-buffered
        # device inputs and outputs; every step still copies all its inputs from pinned host memory and reads all
        # its results back).  Timed as one region of K steps on the device, L2 flush inside, divided by K.
        s_c, s_in, s_out = torch.cuda.Stream(dev), torch.cuda.Stream(dev), torch.cuda.Stream(dev)
        dbuf = [devbuf, {n: torch.empty_like(host[n], device=dev) for n in names}]
        odev = [out_dev, {k: torch.empty_like(v) for k, v in out_dev.items()}]
        ohost = [out_host, {k: torch.empty_like(v, device="cpu").pin_memory() for k, v in out_dev.items()}]
        ev_in = [torch.cuda.Event() for _ in range(2)]
        ev_solved = [torch.cuda.Event() for _ in range(2)]
        ev_out = [torch.cuda.Event() for _ in range(2)]

        def run_pipelined(steps):
            for i in range(steps):
                j = i & 1
                s_in.wait_event(ev_solved[j])                  # solve i-2 no longer reads these inputs
                with torch.cuda.stream(s_in):
                    for n in names:
                        dbuf[j][n].copy_(host[n], non_blocking=True)
                    ev_in[j].record(s_in)
                s_c.wait_event(ev_in[j])
                s_c.wait_event(ev_out[j])                      # results of step i-2 have left the device buffers
                with torch.cuda.stream(s_c):
                    flush.zero_()
                    s.set_problem(**{n: dbuf[j].get(n) for n in gen.Workload.ARRAYS})
                    s.solve(stream=s_c)
                    binding.pinmpc_get(s.h, odev[j]["x"], odev[j]["u"], odev[j]["r_prim"], odev[j]["r_dual"],
                                       odev[j]["iters_done"], s_c.cuda_stream)
                    ev_solved[j].record(s_c)
                s_out.wait_event(ev_solved[j])
                with torch.cuda.stream(s_out):
                    for k in ohost[j]:
                        ohost[j][k].copy_(odev[j][k], non_blocking=True)
                    ev_out[j].record(s_out)

        torch.cuda.synchronize(dev)
        run_pipelined(4)
        torch.cuda.synchronize(dev)
        barrier()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record(s_c)
        run_pipelined(args.steps)
        s_c.wait_event(ev_out[0]); s_c.wait_event(ev_out[1])
        t1.record(s_c)
        torch.cuda.synchronize(dev)
        ms_e2e = t0.elapsed_time(t1) / args.steps
        # same inputs every step: both result buffers must hold exactly what the serial path returned
        for j in range(2):
            for k in ("x", "u", "r_prim", "r_dual"):
                if not torch.equal(ohost[j][k], ohost[0][k]) or not torch.equal(ohost[j][k], odev[0][k].cpu()):
                    raise SystemExit(f"pipelined end-to-end run returned a different {k}")
        barrier()
        s.set_problem(**{n: devbuf.get(n) for n in gen.Workload.ARRAYS})
        e2e = (ms_e2e, h2d, d2h, ms_e2e_serial)

    # ---- max over ranks ---------------------------------------------------------------------------
    if dist is not None:
        ms, e2e_ms = max_over_ranks([ms, e2e[0] if e2e else 0.0], dist, dev)
        e2e = (e2e_ms, e2e[1], e2e[2], e2e[3]) if e2e else None

    if rank == 0:
        total_solves = w.B * world
        value = aggregate_value(w.B, world, ms)
        fl = flops_per_solve(w, mname)
        if kernel_ms:
            # dominant kernel = the iteration kernel: its own algorithmic FLOPs over its own duration (CUDA events
            # recorded by pinmpc_solve on the launching stream around the kernel, averaged over K launches)
            k_ms = [float(np.mean([k[i] for k in kernel_ms])) for i in range(3)]
            fl = w.B * w.N * w.iters * flop_per_stage_iter(w)
            achieved = fl / (k_ms[2] * 1e-3) / 1e12
            G_used, C_used = shape
        else:
            k_ms = None
            achieved = fl / (ms * 1e-3) / 1e12                 # TFLOP/s of the whole step (dense variant)
        props = torch.cuda.get_device_properties(dev)
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except OSError:
            pass
        sm_max_mhz = (clocks or {}).get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
        peak = props.multi_processor_count * FMA_LANES_PER_SM * 2 * sm_max_mhz * 1e6 / 1e12
        # measured FMA-pipe peak on this device (register-resident loop), for context
        scratch = torch.zeros(1, device=dev)
        probe_fma(props.multi_processor_count * 8, 2000, scratch, stream.cuda_stream)
        torch.cuda.synchronize(dev)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        pf = probe_fma(props.multi_processor_count * 8, 20000, scratch, stream.cuda_stream)
        b.record(stream); torch.cuda.synchronize(dev)
        fma_meas = pf / (a.elapsed_time(b) * 1e-3) / 1e12

        io_bytes = sum(getattr(w, n).nbytes for n in gen.Workload.ARRAYS if getattr(w, n) is not None) + \
            w.B * w.N * (13 + 3 * w.nu) * 4 + w.B * 12
        line = {
            "metric": METRIC, "value": value, "unit": "solves/s", "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "B": w.B, "N": w.N, "iters": w.iters, "nu": w.nu, "rho": w.rho,
                       "method": mname, "horizon_chunks": shape[1], "l2": "flushed (256 MiB write) between timed steps; per-step CUDA events",
                       "multi_gpu": "replicas only (no collective on the data path)"},
            "stage_iters_per_s": total_solves * w.N * w.iters / (ms * 1e-3),
            "ms_min": float(np.min(ms_steps)), "ms_median": float(np.median(ms_steps)),
            "gpu_launches": launches,
            "clocks": clocks,
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                         "traffic": measured_traffic(w.name) if k_ms else None,
                         "kernel": (("k_iterate_tm (S3-S6, all iterations; chunked two-sweep equality step, gains in tensor memory)"
                                     if C_used > 1 else "k_iterate_srb (S3-S6, all iterations; sequential passes)")
                                    + f", {G_used} envs per CTA, {C_used} horizon chunks") if k_ms else "whole step",
                         "flop_per_stage_iter": flop_per_stage_iter(w) if k_ms else None,
                         "kernel_ms": {"assemble": k_ms[0], "factor": k_ms[1], "iterate": k_ms[2]} if k_ms else None,
                         "whole_step_tflops": flops_per_solve(w, mname) / (ms * 1e-3) / 1e12,
                         "peak_source": f"{props.multi_processor_count} SMs x {FMA_LANES_PER_SM} FP32 lanes x 2 x "
                                        f"{sm_max_mhz:.0f} MHz (guide unit counts, max SM clock)",
                         "peak_measured_fma_tflops": fma_meas,
                         "flops_per_launch": fl,
                         "hbm_algorithmic_bytes": io_bytes,
                         "hbm_gbs_achieved": io_bytes / (ms * 1e-3) / 1e9,
                         "hbm_peak_gbs": peaks.get("hbm_gbs")},
        }
        if e2e:
            line["e2e"] = {"value": total_solves / (e2e[0] * 1e-3), "unit": "solves/s", "ms_per_step": e2e[0],
                           "h2d_bytes_per_step": e2e[1], "d2h_bytes_per_step": e2e[2],
                           "how": "three streams, double-buffered: the host copies of neighbouring steps overlap the solve",
                           "ms_per_step_serial": e2e[3]}
        if not args.no_cpu_baseline and world == 1:
            import oracle
            oracle.build()
            n0, t0 = time_oracle(w, 32)
            n = int(min(w.B, max(32, 12.0 * n0 / max(t0, 1e-3))))        # about 12 s of CPU work
            n, t = time_oracle(w, n)
            reps = 1
            while t < 10.0 and reps < 64:                            # the whole batch is too quick: repeat it
                t += time_oracle(w, n)[1]
                reps += 1
            line["cpu_baseline"] = {"value": n * reps / t, "unit": "solves/s", "cores": oracle.max_threads(), "kind": "oracle",
                                    "sample": f"first {n} of {w.B} envs of {w.name} x {reps} repeats, all {w.iters} iterations, "
                                              f"fp64, {t:.1f} s"}
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
