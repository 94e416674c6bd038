#!/usr/bin/env python
"""bench.py -- grid-point CG updates/s of the omnidirectional pressure-integration hot path on B200.

A step = one omni_solve call (all rows a0-a8 of SURVEY.md section 8(a): constants, codes, source term, outer
boundary updates, CG inner loops under a CUDA graph, finalize) on one synthetic gradient field, with the outer and
inner iteration caps fixed (STEP_MAX_OUTER x STEP_MAX_CG) so that every step does the same, bounded work.
Unit of work: one grid point updated by one CG iteration.  See DESIGN.md section 8 for every figure printed here.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..4] [--dtype f32|f64] [--impl ours|reference]

N > 1 (torchrun): replicas only -- every rank solves its own copy of the workload, no data-path collective.
--impl reference times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

STEP_MAX_OUTER = 8
STEP_MAX_CG = 25
METRIC = "grid-point CG updates/s"
UNIT = "grid-point CG updates/s"
CPU_SAMPLE_EDGE = 320                   # 3D: edge of the corner crop the oracle is timed on (2D: the whole grid);
                                        # with the step's own caps that is ~10 s of work on 16 host threads
# roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel (K4) comes from an ncu
# --set full capture that cannot be taken inside a timed run; its per-launch bytes are kept in TRAFFIC_CSV together with
# the hash of the kernel sources they were captured from.  The figure is reported only while that hash matches the tree
# (a changed kernel must be re-captured); otherwise traffic is null and traffic_source says why.
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r2_ncu_traffic.csv")
CONV_MAX_CG = 16                        # Alg. 1 time-to-converged: the tuned inner cap of BASELINE.md 5a (same converged field)
ALL_CASES = [(0, "f64"), (1, "f32"), (1, "f64"), (2, "f64"), (3, "f32"), (3, "f64"), (4, "f32")]
L2_BYTES = 126e6


def csrc_hash():
    """sha1 over the kernel sources (csrc/*): identifies what an ncu capture in profiles/ was taken from."""
    import hashlib
    h = hashlib.sha1()
    d = os.path.join(ROOT, "paper_2311_16935_b200", "csrc")
    for name in sorted(os.listdir(d)):
        with open(os.path.join(d, name), "rb") as fh:
            h.update(name.encode() + b"\0" + fh.read())
    return h.hexdigest()[:16]


def k4_traffic(config, dtype, n_even, n_odd):
    """(average measured DRAM bytes per K4 launch over the step's mix of even / first-odd / odd CG iterations, source)."""
    import csv
    try:
        with open(TRAFFIC_CSV) as fh:
            rows = [r for r in csv.DictReader(fh) if int(r["config"]) == config and r["dtype"] == dtype and r["kernel"] == "K4"]
    except Exception:
        return None, "no ncu capture committed for this workload (profiles/r2_ncu_traffic.csv)"
    if not rows:
        return None, "no ncu capture committed for this workload (profiles/r2_ncu_traffic.csv)"
    t = {r["variant"]: float(r["dram_read_bytes"]) + float(r["dram_write_bytes"]) for r in rows}
    src = rows[0]["csrc_hash"]
    if src != csrc_hash():
        return None, f"stale: profiles/r2_ncu_traffic.csv was captured at csrc hash {src}, the tree is at {csrc_hash()}"
    if not all(k in t for k in ("even", "odd_first", "odd")):
        return None, "profiles/r2_ncu_traffic.csv lacks a K4 variant"
    avg = (n_even * t["even"] + (t["odd_first"] if n_odd else 0.0) + max(n_odd - 1, 0) * t["odd"]) / (n_even + n_odd)
    return avg, f"profiles/r2_ncu_traffic.csv (ncu --set full, csrc hash {src}), see profiles/r2_ncu_traffic.md"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--dtype", default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--converge", action="store_true",
                    help="instead of the fixed-cap step: time ONE solve to the config's tolerance (BASELINE.md table)")
    ap.add_argument("--max-cg", type=int, default=1000, help="--converge: CG cap per outer iteration")
    ap.add_argument("--max-outer", type=int, default=200000, help="--converge: outer iteration cap")
    ap.add_argument("--direct", action="store_true",
                    help="--converge: omni_solve_direct (CG on the fixed-point system L P = S) instead of Algorithm 1")
    ap.add_argument("--cascade", type=int, default=-1,
                    help="--converge: omni_solve_cascade with this many coarse levels (implies the direct solve)")
    ap.add_argument("--no-extras", action="store_true",
                    help="default run: skip the per_config and converged sections (profiling runs; always skipped for N > 1)")
    ap.add_argument("--certify", action="store_true",
                    help="--converge: let the oracle re-evaluate eps_R (Eq. 41) of the converged GPU field over all cells")
    ap.add_argument("--batch", type=int, default=1,
                    help="--converge on a 2D config: solve this many snapshots (same mask, different noise seeds) in one "
                         "omni_solve_batch2d call")
    return ap.parse_args()


def converge(args, cfg, dtype):
    """Time-to-converged P of one configuration (whole omni_solve call, CUDA events, inputs resident)."""
    import numpy as np
    import torch
    import paper_2311_16935_b200 as omni
    from workloads import make_config
    tdt = torch.float32 if dtype == "f32" else torch.float64
    tol = 1e-5 if dtype == "f32" else 1e-8
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if args.batch > 1:
        from workloads import CONFIGS, make_field
        c = CONFIGS[args.config]
        fs = [make_field(c["kind"], (c["n"], c["n"]), seed=1000 + b, noise=c["noise"]) for b in range(args.batch)]
        f = fs[0]
        gx = torch.from_numpy(np.stack([x["g"][0] for x in fs])).to(tdt).cuda()
        gy = torch.from_numpy(np.stack([x["g"][1] for x in fs])).to(tdt).cuda()
        m = None if f["mask"] is None else torch.from_numpy(f["mask"]).cuda()
        omni.solve_batch2d(gx, gy, m, f["d"], tol, 2, 2, direct=args.direct)
        torch.cuda.synchronize()
        e0.record()
        P, info = omni.solve_batch2d(gx, gy, m, f["d"], tol, args.max_outer, args.max_cg, direct=args.direct)
        e1.record()
        torch.cuda.synchronize()
        Pn = P[0].double().cpu().numpy()
        N = gx.numel()
    else:
        f = make_config(args.config, device="cuda")
        g = [torch.from_numpy(c).to(tdt).cuda() for c in f["g"]] + [None] * (3 - len(f["g"]))
        m = None if f["mask"] is None else torch.from_numpy(f["mask"]).cuda()
        fn = omni.solve_direct if args.direct else omni.solve
        if args.cascade >= 0:
            def fn(gx, gy, gz, m, d, tol, mo, mc):
                return omni.solve_cascade(gx, gy, gz, m, d, tol, mo, mc, levels=args.cascade)
        fn(g[0], g[1], g[2], m, f["d"], tol, 2, 2)                               # warm-up (module load, pool)
        torch.cuda.synchronize()
        e0.record()
        P, info = fn(g[0], g[1], g[2], m, f["d"], tol, args.max_outer, args.max_cg)
        e1.record()
        torch.cuda.synchronize()
        Pn = P.double().cpu().numpy()
        N = g[0].numel()
    sec = e0.elapsed_time(e1) * 1e-3
    valid = ~np.isnan(Pn)
    a, b = Pn[valid] - Pn[valid].mean(), f["P"][valid] - f["P"][valid].mean()
    cert = None
    if args.certify and args.batch == 1:
        cert = oracle_eps_R(f, g, Pn)
    print(json.dumps({"converge": True, "eps_R_oracle": cert, "workload": f"configs[{args.config}] {cfg['kind']} {cfg['n']} {dtype}", "tol": tol,
                      "max_cg": args.max_cg, "batch": args.batch, "direct": bool(args.direct or args.cascade >= 0), "cascade_levels": args.cascade, "outer_iters": info["outer_iters"], "cg_iters": info["cg_iters_total"],
                      "seconds": sec, "eps_R": info["eps_R_final"], "status": info["status"],
                      "updates_per_s": N * info["cg_iters_total"] / sec,
                      "rel_l2_vs_analytic_P": float(np.linalg.norm(a - b) / np.linalg.norm(b))}))


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)"
    except Exception:
        return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md recipe)."""
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.rows, self.stop, self.index = [], threading.Event(), index
        self.t = threading.Thread(target=self.run, daemon=True)

    def run(self):
        while not self.stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([c.strip() for c in out.strip().split(",")])
            except Exception:
                pass
            self.stop.wait(0.2)

    def __enter__(self):
        self.t.start()
        return self

    def __exit__(self, *a):
        self.stop.set()
        self.t.join(timeout=6)

    def summary(self):
        sm = sorted(int(r[0]) for r in self.rows if len(r) >= 6 and r[0].isdigit())
        reasons = set()
        for r in self.rows:
            if len(r) >= 6:
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[2:6]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
        mx = max((int(r[1]) for r in self.rows if len(r) >= 6 and r[1].isdigit()), default=None)
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


def max_over_ranks(values, world, device="cpu"):
    """Per-rank timings -> the maximum over ranks (the job finishes with its slowest replica)."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor(values, dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t]


def aggregate_value(units_per_step_per_rank, steps, world, seconds_max):
    """Whole-job throughput of N independent replicas (weak scaling): all ranks' units over the slowest rank's time."""
    return world * units_per_step_per_rank * steps / seconds_max


def cpu_sample(f, ndim):
    """Bounded sample of the workload for the oracle: the corner crop [0:e]^ndim of the same arrays."""
    import numpy as np
    e = min(CPU_SAMPLE_EDGE if ndim == 3 else 1024, f["g"][0].shape[0])
    sl = (slice(0, e),) * ndim
    g = [np.ascontiguousarray(c[sl]) for c in f["g"]]
    m = None if f["mask"] is None else np.ascontiguousarray(f["mask"][sl])
    return g, m, e


def run_oracle(f, dtype, steps, warmup):
    """CPU oracle, as it stands, on the bounded sample; returns (updates/s, cores, sample description)."""
    import numpy as np
    from oracle import omni_oracle as orc
    ndim = f["g"][0].ndim
    g, m, e = cpu_sample(f, ndim)
    if dtype == "f32":
        g = [c.astype(np.float32).astype(np.float64) for c in g]
    g = g + [None] * (3 - len(g))
    tol = 1e-5 if dtype == "f32" else 1e-8
    mo, mc = STEP_MAX_OUTER, STEP_MAX_CG
    for _ in range(warmup):
        orc.solve(g[0], g[1], g[2], m, *f["d"], tol=tol, max_outer=mo, max_cg=mc)
    t0 = time.perf_counter()
    units = 0
    for _ in range(steps):
        _, info = orc.solve(g[0], g[1], g[2], m, *f["d"], tol=tol, max_outer=mo, max_cg=mc)
        units += (g[0].size if m is None else int(m.sum())) * info["cg_iters_total"]
    dt = time.perf_counter() - t0
    desc = f"corner crop {e}^{ndim} of the same field, omni oracle solve max_outer={mo} max_cg={mc}, {steps} step(s)"
    return units / dt, orc.num_threads(), desc, dt / steps


def oracle_eps_R(f, g_dev, P_np):
    """SURVEY 8(c) parity protocol iii: eps_R (Eq. 41) of a GPU field re-evaluated by the ORACLE's per-cell operators over
    all cells, from the values the device consumed.  Reporting only (bench.py's cpu_baseline leg is where the bench may
    run the oracle); never inside a timed region."""
    import numpy as np
    from oracle import omni_oracle as orc
    g = [None if c is None else c.cpu().numpy().astype(np.float64) for c in g_dev]
    eps, _, _ = orc.eps_R_of_field(g[0], g[1], g[2], f["mask"], P_np, *f["d"])
    return eps


def _load_case(idx, dtype, dev):
    import torch
    from workloads import make_config
    f = make_config(idx, device=str(dev))
    tdt = torch.float32 if dtype == "f32" else torch.float64
    g = [torch.from_numpy(c).to(tdt).to(dev) for c in f["g"]] + [None] * (3 - len(f["g"]))
    m = None if f["mask"] is None else torch.from_numpy(f["mask"]).to(dev)
    return f, g, m


def _timed(fn, reps=1):
    """Best-of-reps CUDA-event time (s) of fn(), events on the current stream; returns (seconds, last result)."""
    import torch
    best, out = None, None
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        out = fn()
        e1.record()
        torch.cuda.synchronize()
        t = e0.elapsed_time(e1) * 1e-3
        best = t if best is None else min(best, t)
    return best, out


def per_config_entry(idx, dtype, dev, peak, cache=None):
    """CG inner loop of one config at full size (SURVEY 8(d) metric 1 and 3), two live measurements:
    * `cg_iteration_us`: whole-call CUDA-event time of two fixed-count solves that differ only in max_cg (one outer
      iteration, tol = 0), difference / iteration difference -- what one CG iteration costs in the loop driver the
      library picks by itself for this size, everything included;
    * `k3_us`, `k4_us`: CUDA events around every tile-kernel launch of the host-driven loop (loop mode 1)."""
    import paper_2311_16935_b200 as omni
    f, g, m = cache if cache is not None else _load_case(idx, dtype, dev)
    d = f["d"]
    N = g[0].numel()
    nvalid = N if m is None else int(m.sum().item())
    esz = 4 if dtype == "f32" else 8
    # enough iterations for ~20 ms of difference whatever the size
    m1 = 10
    m2 = m1 + int(min(2000, max(60, 3e9 / (N * esz))))
    omni.solve(g[0], g[1], g[2], m, d, 0.0, 1, m1, want_info=False)
    t1, _ = _timed(lambda: omni.solve(g[0], g[1], g[2], m, d, 0.0, 1, m1, want_info=False), 3)
    t2, _ = _timed(lambda: omni.solve(g[0], g[1], g[2], m, d, 0.0, 1, m2, want_info=False), 3)
    cg = (t2 - t1) / (m2 - m1)
    prev = omni.set_loop_mode(1)
    omni.profile_enable(1)
    omni.profile_read(reset=True)
    omni.solve(g[0], g[1], g[2], m, d, 0.0, 2, 25)
    prof = omni.profile_read(reset=True)
    omni.profile_enable(0)
    omni.set_loop_mode(prev)
    k3 = prof["K3"][0] / max(prof["K3"][1], 1) * 1e-3
    k4 = prof["K4"][0] / max(prof["K4"][1], 1) * 1e-3
    alg = 7.5 * esz * N                     # K3 3 passes, K4 3 / 6 by iteration parity
    resident = (5 * esz + 16) * N < L2_BYTES
    return {"workload": f"configs[{idx}] {f['kind']} {'x'.join(str(x) for x in f['shape'])} {dtype}", "cells": N,
            "valid_cells": nvalid, "cg_iteration_us": cg * 1e6, "updates_per_s_in_loop": nvalid / cg,
            "algorithmic_bytes_per_cg_iteration": alg, "algorithmic_GBps": alg / cg / 1e9,
            "frac_of_measured": alg / cg / 1e9 / peak, "frac_of_8TBps": alg / cg / 8e12,
            "memory": ("SM-resident loop (p in shared memory, DESIGN.md section 20): effective GB/s, not HBM" if N * esz <= 20e6
                       else "L2-resident: effective GB/s, not HBM") if resident else "HBM (state exceeds L2)",
            "k3_us": k3 * 1e6, "k4_us": k4 * 1e6, "tile_kernels_cg_iteration_us": (k3 + k4) * 1e6,
            "iterations_timed": [m1, m2]}


def converged_entries(idx, dtype, dev, cache=None, alg1=True):
    """Time to converged P (SURVEY 8(d) metric 2): whole call, CUDA events, inputs resident, eps_R <= tol -- by Alg. 1
    (the paper's iteration, max_cg = 16) and, separately named, by the fixed-point solves; each converged field has its
    eps_R re-evaluated by the oracle over all cells (parity protocol iii)."""
    import numpy as np
    import paper_2311_16935_b200 as omni
    f, g, m = cache if cache is not None else _load_case(idx, dtype, dev)
    d = f["d"]
    tol = 1e-5 if dtype == "f32" else 1e-8
    N = g[0].numel()
    nvalid = N if m is None else int(m.sum().item())
    import torch
    # fp32: also take the fp64 master pressure (omni_options::d_P64_out): the fp32 result is its rounding, whose own
    # residual is floored at 2^-24 |L||P| / ||S|| -- above tol on the large grids; the oracle certifies both
    P64 = torch.zeros_like(g[0], dtype=torch.float64) if dtype == "f32" else None

    def ex(method, mo, mc):
        return lambda: omni.solve_ex(g[0], g[1], g[2], m, d, tol, mo, mc, method=method, P64_out=P64)
    methods = []
    if alg1:
        methods.append((f"alg1 max_cg={CONV_MAX_CG}", ex("alg1", 400000, CONV_MAX_CG), True))
    methods.append(("direct (CG on L P = S)", ex("direct", 20, 30000), True))
    methods.append(("cascade levels=4", lambda: omni.solve_cascade(g[0], g[1], g[2], m, d, tol, 20, 30000, levels=4), False))
    methods.append(("pcg (multigrid-preconditioned CG on L P = S)", ex("pcg", 20, 300), True))
    out = []
    omni.solve(g[0], g[1], g[2], m, d, tol, 1, 2)          # pool / module warm-up
    for name, fn, has64 in methods:
        sec, (P, info) = _timed(fn)
        Pn = P.double().cpu().numpy()
        valid = ~np.isnan(Pn)
        a, b = Pn[valid] - Pn[valid].mean(), f["P"][valid] - f["P"][valid].mean()
        out.append({"workload": f"configs[{idx}] {f['kind']} {'x'.join(str(x) for x in f['shape'])} {dtype}", "method": name,
                    "tol": tol, "seconds": sec, "outer_iters": info["outer_iters"], "cg_iters": info["cg_iters_total"],
                    "status": info["status"], "eps_R_gpu": info["eps_R_final"],
                    "eps_R_oracle": oracle_eps_R(f, g, P.cpu().numpy()),
                    "eps_R_oracle_fp64_master": oracle_eps_R(f, g, P64.cpu().numpy()) if (P64 is not None and has64) else None,
                    "updates_per_s_whole_call": nvalid * info["cg_iters_total"] / sec,
                    "rel_l2_vs_analytic_P": float(np.linalg.norm(a - b) / np.linalg.norm(b))})
    return out


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    from workloads import CONFIGS, make_config
    cfg = CONFIGS[args.config]
    dtype = args.dtype or ("f32" if "f32" in cfg["dtypes"] else "f64")
    n = cfg["n"]
    ndim = 2 if cfg["kind"].endswith("2d") else 3
    workload = f"configs[{args.config}] {cfg['kind']} {n}^{ndim} {dtype} noise={cfg['noise']}"
    config = {"workload": workload, "step": f"omni_solve tol={'1e-5' if dtype == 'f32' else '1e-8'} "
              f"max_outer={STEP_MAX_OUTER} max_cg={STEP_MAX_CG} (fixed caps)", "parallelism": f"replicas x{world}",
              "units": "valid grid points x CG iterations",
              "l2": "inputs larger than L2 (no flush)" if n ** ndim * (4 if dtype == "f32" else 8) > 126e6
              else "CG state fits L2: numbers are L2-resident, flushed between steps by the solve's own setup passes"}

    if args.converge:
        if rank == 0:
            converge(args, cfg, dtype)
        return
    if args.impl == "reference":
        if rank != 0:
            return
        f = make_config(args.config)
        v, cores, desc, spstep = run_oracle(f, dtype, args.steps, args.warmup)
        print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
                          "steps": args.steps, "warmup": args.warmup, "ms_per_step": spstep * 1e3,
                          "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
                          "data": "synthetic", "config": config,
                          "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
                          "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))
        return

    import torch
    import paper_2311_16935_b200 as omni
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    f = make_config(args.config, device=f"cuda:{local_rank}")
    tdt = torch.float32 if dtype == "f32" else torch.float64
    g_host = [torch.from_numpy(c).to(tdt).pin_memory() for c in f["g"]]
    m_host = None if f["mask"] is None else torch.from_numpy(f["mask"]).pin_memory()
    g = [c.to(dev) for c in g_host] + [None] * (3 - len(g_host))
    m = None if m_host is None else m_host.to(dev)
    g_host = g_host + [None] * (3 - len(g_host))
    d = f["d"]
    tol = 1e-5 if dtype == "f32" else 1e-8
    N = g[0].numel()
    nvalid = N if m is None else int(m.sum().item())      # grid-point updates count VALID cells (masked cells do no work)
    esz = 4 if dtype == "f32" else 8
    P = torch.empty_like(g[0])

    def step(info=False):
        return omni.solve(g[0], g[1], g[2], m, d, tol, STEP_MAX_OUTER, STEP_MAX_CG, out=P, want_info=info)

    # warm-up (also gives the deterministic iteration and launch counts of one step)
    omni.launch_count(reset=True)
    _, info = step(info=True)
    launches_per_step = omni.launch_count(reset=True)
    for _ in range(max(args.warmup - 1, 0)):
        step()
    torch.cuda.synchronize()
    units_per_step = nvalid * info["cg_iters_total"]

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with ClockSampler(local_rank) as clk:
        barrier()
        e0.record()
        for _ in range(args.steps):
            step()
        e1.record()
        barrier()
        ms = e0.elapsed_time(e1)
        # end to end through the C ABI with HOST buffers (pinned): H2D of g/mask and D2H of P inside the timed region
        P_host = torch.empty_like(g_host[0]).pin_memory()
        omni.solve(g_host[0], g_host[1], g_host[2], m_host, d, tol, STEP_MAX_OUTER, STEP_MAX_CG, out=P_host)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            omni.solve(g_host[0], g_host[1], g_host[2], m_host, d, tol, STEP_MAX_OUTER, STEP_MAX_CG, out=P_host)
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
    clocks = clk.summary()

    ms, e2e_s = max_over_ranks([ms, e2e_s], world, dev)

    # per-kernel live timing of the same step (host-driven loop, CUDA events around each launch on the same stream)
    prev = omni.set_loop_mode(1)
    omni.profile_enable(1)
    omni.profile_read(reset=True)
    step(info=True)
    prof = omni.profile_read(reset=True)
    omni.profile_enable(0)
    omni.set_loop_mode(prev)
    peak, peak_src = measured_peak()
    k3_ms, k3_n = prof["K3"]
    k4_ms, k4_n = prof["K4"]
    k2_ms, k2_n = prof["K2"]
    t4 = k4_ms / max(k4_n, 1) * 1e-3
    t3 = k3_ms / max(k3_n, 1) * 1e-3
    # K3: R r,p W p.  K4 (lazy delta): even CG iterations R p,r W r (3 passes), odd ones
    # R p,p_old,r,delta W r,delta (6 passes; the first odd one does not read delta): the average over the step's launches
    n_even, n_odd = (STEP_MAX_CG + 1) // 2, STEP_MAX_CG // 2
    k4_passes = (3 * n_even + 6 * n_odd - (1 if n_odd else 0)) / STEP_MAX_CG
    alg4, alg3 = k4_passes * esz * N, 3 * esz * N
    ach = alg4 / t4 / 1e9 if t4 > 0 else 0.0
    traffic, traffic_src = k4_traffic(args.config, dtype, n_even, n_odd)
    roofline = {"bound": "hbm", "kernel": "K4 tma_kernel<OpT4> (operator recomputed + axpys + r.r)",
                "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak, "peak_source": peak_src,
                "traffic": traffic, "traffic_source": traffic_src,
                "algorithmic_bytes_per_launch": alg4, "k4_passes_avg": k4_passes, "us_per_launch": t4 * 1e6,
                "k3": {"achieved": alg3 / t3 / 1e9 if t3 > 0 else 0.0, "us_per_launch": t3 * 1e6,
                       "algorithmic_bytes_per_launch": alg3},
                "cg_iteration": {"us": (t3 + t4) * 1e6, "achieved": (alg3 + alg4) / (t3 + t4) / 1e9 if t3 + t4 > 0 else 0.0,
                                 "frac": (alg3 + alg4) / (t3 + t4) / 1e9 / peak if t3 + t4 > 0 else 0.0,
                                 "updates_per_s_in_loop": nvalid / (t3 + t4) if t3 + t4 > 0 else 0.0},
                "k2_us_per_launch": k2_ms / max(k2_n, 1) * 1e3,
                "share_of_step": {"K2": k2_ms, "K3": k3_ms, "K4": k4_ms}}

    if rank != 0:
        return
    out = {"metric": METRIC, "value": aggregate_value(units_per_step, args.steps, world, ms * 1e-3), "unit": UNIT,
           "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms / args.steps,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": dtype, "data": "synthetic",
           "config": config, "clocks": clocks, "gpu_launches": launches_per_step * args.steps,
           "e2e": {"value": aggregate_value(units_per_step, args.steps, world, e2e_s), "unit": UNIT,
                   "h2d_bytes_per_step": sum(c.numel() * c.element_size() for c in g_host if c is not None)
                   + (0 if m_host is None else m_host.numel()), "d2h_bytes_per_step": N * esz,
                   "ms_per_step": e2e_s / args.steps * 1e3},
           "step_info": {"outer_iters": info["outer_iters"], "cg_iters": info["cg_iters_total"],
                         "eps_R": info["eps_R_final"], "status": info["status"]},
           "roofline": roofline}
    if world == 1:
        if not args.no_extras:
            # the rest of BASELINE.json's metric, same run: the CG loop of the other 3D configs and the time to a
            # converged P of every config x dtype (sections per_config / converged)
            out["per_config"], out["converged"] = [], []
            for (ci, cd) in ALL_CASES:
                cache = (f, g, m) if (ci, cd) == (args.config, dtype) else _load_case(ci, cd, dev)
                if ci >= 1:
                    out["per_config"].append(per_config_entry(ci, cd, dev, peak, cache))
                out["converged"] += converged_entries(ci, cd, dev, cache)
                del cache
                torch.cuda.empty_cache()
        del g, P
        torch.cuda.empty_cache()
        v, cores, desc, _ = run_oracle(f, dtype, 1, 0)
        out["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
