#!/usr/bin/env python
"""bench.py -- headline measurement of the Monte Carlo DtN hot path on B200.

One "step" = one pass of the whole hot path over the
workload BASELINE.json's metric is quoted on (configs[1]): LBVH build of the
icosphere-L4 mesh, then the interior AND the exterior (killing term on) DtN
matrices, 2562 vertices x 4096 walks per operator.  Prints ONE JSON line (the
contract is in DESIGN.md "Measurement").

  python bench.py                       # N=1, this repo's CUDA path
  python bench.py --impl reference      # the CPU oracle, as it stands, on a bounded sample
  torchrun ... bench.py --gpus N        # N independent replicas
"""
from __future__ import annotations

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

METRIC = "walk_steps_per_s"
UNIT = "walk steps/s"


# ------------------------------------------------------------------------------
# workload = BASELINE.json configs[1]
# ------------------------------------------------------------------------------
def make_workload(level: int, walks_per_vertex: int, points_per_vertex: int, seed: int):
    from synth import icosphere, vertex_cell_samples
    v, f = icosphere(level)
    smp = vertex_cell_samples(v, f, points_per_vertex, seed=seed)
    W = walks_per_vertex // points_per_vertex
    return dict(v=v, f=f, smp=smp, W=W, name=f"icosphere_L{level}", V=len(v), F=len(f), n_s=len(smp["tri"]))


def config_dict(wl, args, extra=None):
    c = {"workload": f"configs[1]: {wl['name']} ({wl['V']} vertices, {wl['F']} faces), interior + exterior(killing on) "
                     f"DtN, hat basis, {args.walks_per_vertex} walks/vertex = {wl['n_s']} sample points x {wl['W']} walks "
                     f"per operator, eps={args.eps:g}, cap={args.cap:g} deg, Philox seed {args.seed}",
         "operators": ["interior", "exterior+killing"], "walks_per_operator": wl["n_s"] * wl["W"],
         "kill_walks": wl["n_s"] * wl["W"], "includes_bvh_build": True,
         "l2_policy": "256 MiB buffer written between timed steps (L2 flush); the 0.6 MB tree is re-read from HBM/L2 each step",
         "parallelism": "replicas" if args.gpus > 1 else "single"}
    if extra:
        c.update(extra)
    return c


# ------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md "clocks line")
# ------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None
        self.thread = None

    def start(self):
        if os.environ.get("MCS_BENCH_NO_CLOCKS"):
            return
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        def pump():
            for line in self.proc.stdout:
                self.rows.append(line.strip())
        self.thread = threading.Thread(target=pump, daemon=True)
        self.thread.start()

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, reasons, power = [], [], set(), []
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            p = [x.strip() for x in r.split(",")]
            if len(p) < 7:
                continue
            try:
                sm.append(float(p[0])); mx.append(float(p[1])); power.append(float(p[2]))
            except ValueError:
                continue
            for n, val in zip(names, p[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(n)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                "power_w_max": float(max(power)), "samples": len(sm)}


def read_traffic():
    """DRAM bytes of the walk-kernel launches of one step, from the committed ncu capture (profiles/)."""
    path = os.path.join(ROOT, "profiles", "walk_kernel_traffic.csv")
    if not os.path.exists(path):
        return None
    total = 0
    with open(path) as fh:
        for line in fh.read().splitlines()[1:]:
            p = line.split(",")
            if len(p) == 3:
                total += int(p[1]) + int(p[2])
    return total or None


def read_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------
# the CPU oracle on a bounded sample of the same workload (cpu_baseline / --impl reference)
# ------------------------------------------------------------------------------
def oracle_sample_run(wl, args, n_samples: int):
    """Runs interior + exterior(killing) through oracle/ on every (n_s // n_samples)-th sample point.
    Returns (walk steps, seconds, cores, description)."""
    from oracle import Oracle, OracleParams, mesh_geom
    smp = wl["smp"]
    stride = max(1, wl["n_s"] // n_samples)
    idx = np.arange(0, wl["n_s"], stride)[:n_samples]
    tri, bary, wgt = smp["tri"][idx], smp["bary"][idx], smp["weight"][idx]
    orc = Oracle(mesh_geom(wl["v"], wl["f"]))
    steps = 0
    t0 = time.perf_counter()
    for ext in (False, True):
        n_walks = len(idx) * wl["W"]
        p = OracleParams(seed=args.seed, walks_per_sample=wl["W"], eps=args.eps, cap_half_angle_deg=args.cap,
                         include_killing=ext, n_kill_walks=n_walks if ext else 0)
        res = orc.estimate_dtn(p, ext, tri, bary, wgt)
        st = res["records"]["steps"]
        steps += int(st[st > 0].sum())
    dt = time.perf_counter() - t0
    desc = (f"{len(idx)} of {wl['n_s']} sample points (every {stride}th) x {wl['W']} walks, interior + exterior "
            f"(+ {len(idx) * wl['W']} killing walks), brute-force fp64 closest point over {wl['F']} faces, then the dense "
            f"hat-basis accumulation")
    return steps, dt, orc.num_threads, desc


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = make_workload(args.level, args.walks_per_vertex, args.points_per_vertex, args.seed)
    for _ in range(args.warmup):
        oracle_sample_run(wl, args, max(1, args.ref_samples // 8))
    total_steps, total_t, cores, desc = 0, 0.0, 0, ""
    for _ in range(args.steps):
        s, dt, cores, desc = oracle_sample_run(wl, args, args.ref_samples)
        total_steps += s
        total_t += dt
    value = total_steps / total_t
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total_t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(wl, args, {"reference_sample": desc}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------
# multi-rank host logic (replicas only); covered on CPU with gloo
# ------------------------------------------------------------------------------
def replica_seed(seed: int, rank: int) -> int:
    """Rank r of an N-replica run uses Philox seed + r: independent walks, same workload."""
    return seed + rank


def max_over_ranks(x: float, device, world: int) -> float:
    """Device-timed durations are reduced with MAX over ranks (never wall clock)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, device, world: int) -> float:
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def whole_job_value(units_per_rank_step: float, world: int, seconds_per_step: float) -> float:
    """Weak scaling: every rank processes units_per_rank_step per step; the job's rate is the sum."""
    return world * units_per_rank_step / seconds_per_step


# ------------------------------------------------------------------------------
# this repo's CUDA path
# ------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_05581_b200 import api

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    api.lib()

    # replicas only: rank r runs the same workload with Philox seed + r
    seed = replica_seed(args.seed, rank)
    wl = make_workload(args.level, args.walks_per_vertex, args.points_per_vertex, args.seed)
    n_walks = wl["n_s"] * wl["W"]
    v_h = torch.as_tensor(wl["v"]).pin_memory()
    f_h = torch.as_tensor(wl["f"]).pin_memory()
    tri_h = torch.as_tensor(wl["smp"]["tri"]).pin_memory()
    bary_h = torch.as_tensor(wl["smp"]["bary"]).pin_memory()
    w_h = torch.as_tensor(wl["smp"]["weight"]).pin_memory()
    vd, fd = v_h.to(dev), f_h.to(dev)
    S = api.Samples(tri_h.to(dev), bary_h.to(dev), w_h.to(dev))
    P_int = api.Params(seed=seed, walks_per_sample=wl["W"], eps=args.eps, cap_half_angle_deg=args.cap)
    P_ext = api.Params(seed=seed, walks_per_sample=wl["W"], eps=args.eps, cap_half_angle_deg=args.cap,
                       include_killing=True, n_kill_walks=n_walks)
    bvh0 = api.build_bvh(vd, fd)
    ws_bytes = max(api.workspace_bytes(bvh0, S, P_int, False), api.workspace_bytes(bvh0, S, P_ext, True),
                   api.workspace_bytes_both(bvh0, S, P_int, P_ext))
    ws = torch.empty(ws_bytes, dtype=torch.uint8, device=dev)
    out_int = torch.empty((wl["V"], wl["V"]), dtype=torch.float32, device=dev)
    out_ext = torch.empty_like(out_int)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    # deterministic work counts of one step (counter build of the kernels; outside the timed region)
    _, st_i = api.estimate_dtn_interior(bvh0, S, P_int, want_stats=True, out=out_int, workspace=ws)
    _, st_e = api.estimate_dtn_exterior(bvh0, S, P_ext, want_stats=True, out=out_ext, workspace=ws)
    steps_per_step = st_i.n_steps + st_e.n_steps
    queries_per_step = st_i.n_queries + st_e.n_queries
    del bvh0

    phases = []

    def step(profile):
        bvh = api.build_bvh(vd, fd)
        if not args.serial:
            # one call for both operators: the two walk kernels overlap on two streams
            api.estimate_dtn_both(bvh, S, P_int, P_ext, out_interior=out_int, out_exterior=out_ext, workspace=ws)
            if profile:
                phases.append(("both", api.profile_last()))
            return
        api.estimate_dtn_interior(bvh, S, P_int, out=out_int, workspace=ws)
        if profile:
            phases.append(("interior", api.profile_last()))
        api.estimate_dtn_exterior(bvh, S, P_ext, out=out_ext, workspace=ws)
        if profile:
            phases.append(("exterior", api.profile_last()))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    clocks = ClockSampler(local)
    clocks.start()                 # before the warm-up: nvidia-smi's own start-up stays out of the timed region
    for _ in range(args.warmup):
        step(False)
        flush.fill_(1)
    api.profile_enable(True)
    stream = torch.cuda.current_stream(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    clocks.rows.clear()            # keep the samples taken during the timed region only
    launches0 = api.launch_count()
    e0.record(stream)
    for _ in range(args.steps):
        step(True)
        flush.fill_(1)
    e1.record(stream)
    barrier()
    launches = api.launch_count() - launches0
    clk = clocks.stop()
    api.profile_enable(False)
    ms = e0.elapsed_time(e1)
    ms = max_over_ranks(ms, dev, world)
    ms_per_step = ms / args.steps
    job_steps = sum_over_ranks(steps_per_step, dev, world)        # replicas differ by their Philox seed
    job_queries = sum_over_ranks(queries_per_step, dev, world)
    value = job_steps / (ms_per_step * 1e-3)

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    oi_h = torch.empty((wl["V"], wl["V"]), dtype=torch.float32, pin_memory=True)
    oe_h = torch.empty_like(oi_h).pin_memory()
    e2e_steps = max(1, min(args.steps, 10))
    # warm-up: the device idles while nvidia-smi is stopped and the host buffers are pinned, and the first ~0.3 s of
    # calls after that ran 6 % slower than the following ones (measured per call: 51.6, 51.6, 51.5, 48.4 ms)
    for _ in range(max(args.warmup, 8)):
        r = api.estimate_dtn_host(v_h, f_h, tri_h, bary_h, w_h, P_ext, out_interior=oi_h, out_exterior=oe_h, device=dev)
    barrier()
    t0 = time.perf_counter()
    e2e_each = []
    for _ in range(e2e_steps):
        # one call runs interior (killing flag ignored there) and exterior on one upload of the mesh
        tc = time.perf_counter()
        r = api.estimate_dtn_host(v_h, f_h, tri_h, bary_h, w_h, P_ext, out_interior=oi_h, out_exterior=oe_h, device=dev)
        e2e_each.append((time.perf_counter() - tc) * 1e3)      # the call blocks until the matrices are in host memory
        flush.fill_(1)
    barrier()
    e2e_t = (time.perf_counter() - t0) / e2e_steps
    e2e_t = max_over_ranks(e2e_t, dev, world)
    e2e_value = job_steps / e2e_t

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (the persistent walk kernel), DESIGN.md "Roofline"
    walk_ms = {"interior": [], "exterior": [], "both": []}
    prep_ms, acc_ms = [], []
    for name, ph in phases:
        walk_ms[name].append(ph.walk_ms)
        prep_ms.append(ph.prep_ms)
        acc_ms.append(ph.accumulate_ms)
    fp32_tflops = api.measure_fp32_tflops(dev)
    l2_gbs = api.measure_l2_gbs(dev)
    hbm_gbs, hbm_src = read_peaks()
    tree_bytes = 64 * (wl["F"] - 1) + 48 * wl["F"]
    level_gbs, level = (l2_gbs, "l2") if tree_bytes < 100e6 else (hbm_gbs, "hbm")
    roof = {}
    for name, st in (("interior", st_i), ("exterior", st_e)):
        t = float(np.mean(walk_ms[name])) * 1e-3 if args.serial else 0.0
        # walk kernel only: the tangent-ball traversals (A2) are counted separately
        nodes, tris = st.n_nodes_visited - st.n_prep_nodes, st.n_tris_tested - st.n_prep_tris
        queries = st.n_queries - st.n_prep_queries
        flops = 72.0 * nodes + 80.0 * tris          # 4-wide nodes: four 18-flop box tests per visit
        nbytes = 128.0 * nodes + 48.0 * tris
        t_alu, t_mem = flops / (fp32_tflops * 1e12), nbytes / (level_gbs * 1e9)
        roof[name] = dict(t=t, flops=flops, bytes=nbytes, t_alu=t_alu, t_mem=t_mem,
                          nodes_per_query=nodes / queries, tris_per_query=tris / queries)
    # overlapped launches: the denominator is the span from the interior kernel's start to the exterior kernel's
    # end (events on the two streams), which also holds whatever else ran in that span
    t_kernel = roof["interior"]["t"] + roof["exterior"]["t"] if args.serial else float(np.mean(walk_ms["both"])) * 1e-3
    nbytes = roof["interior"]["bytes"] + roof["exterior"]["bytes"]
    flops = roof["interior"]["flops"] + roof["exterior"]["flops"]
    t_mem = nbytes / (level_gbs * 1e9)
    t_alu = flops / (fp32_tflops * 1e12)
    mem_bound = t_mem >= t_alu
    roofline = {
        "kernel": "walk_kernel (interior launch + exterior launch of one step" + (")" if args.serial else ", overlapped on two streams: span of both)"),
        "bound": level if mem_bound else "alu",
        "achieved": (nbytes / t_kernel / 1e9) if mem_bound else (flops / t_kernel / 1e12),
        "peak": level_gbs if mem_bound else fp32_tflops,
        "unit": "GB/s" if mem_bound else "TFLOP/s",
        "frac": max(t_mem, t_alu) / t_kernel,
        "traffic": read_traffic(),
        "traffic_note": "dram bytes read+write of the two walk_kernel launches of one step (ncu --set full, profiles/walk_kernel_traffic.csv); algorithmic node+triangle bytes are served from L2",
        "peak_source": (f"{level} read bandwidth measured live by mcs_measure_l2_gbs (tree is {tree_bytes / 1e6:.2f} MB, "
                        f"{level}-resident); HBM {hbm_gbs:.0f} GB/s {hbm_src}; FP32 {fp32_tflops:.1f} TFLOP/s measured live"),
        "algorithmic": "bytes = 128 B x 4-wide nodes visited + 48 B x triangles tested; flops = 72 x nodes + 80 x triangles (DESIGN.md)",
        "alu_frac": t_alu / t_kernel, "mem_frac": t_mem / t_kernel,
        "kernel_ms_per_step": t_kernel * 1e3, "kernel_share_of_step": t_kernel * 1e3 / ms_per_step,
        "nodes_per_query": {k: roof[k]["nodes_per_query"] for k in roof},
        "tris_per_query": {k: roof[k]["tris_per_query"] for k in roof},
    }

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        s, dt, cores, desc = oracle_sample_run(wl, args, args.cpu_samples)
        cpu = {"value": s / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "seconds": dt}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": config_dict(wl, args),
            "queries_per_s": job_queries / (ms_per_step * 1e-3),
            "dtn_matrices_per_s": world * 2.0 / (ms_per_step * 1e-3),
            "walk_steps_per_step": steps_per_step, "queries_per_step": queries_per_step,
            "call": "mcs_build_bvh + " + ("mcs_estimate_dtn_interior + mcs_estimate_dtn_exterior" if args.serial else "mcs_estimate_dtn_both"),
            "phase_ms_per_step": {"prep": float(np.sum(prep_ms)) / args.steps, "walk": t_kernel * 1e3,
                                  "accumulate": float(np.sum(acc_ms)) / args.steps},
            "walk_end_ms": None if args.serial else {"interior": float(np.mean([ph.walk_interior_ms for _, ph in phases])),
                                                     "exterior": float(np.mean([ph.walk_exterior_ms for _, ph in phases]))},
            "clocks": clk,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": r["h2d_bytes"], "d2h_bytes_per_step": r["d2h_bytes"],
                    "ms_per_step": e2e_t * 1e3, "ms_per_call": e2e_each, "steps": e2e_steps, "call": "mcs_estimate_dtn_host (pinned host buffers)"},
            "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--level", type=int, default=4, help="icosphere subdivision level (configs[1]: 4)")
    ap.add_argument("--walks-per-vertex", type=int, default=4096)
    ap.add_argument("--points-per-vertex", type=int, default=16, help="G of DESIGN.md reading R1")
    ap.add_argument("--eps", type=float, default=1e-3)
    ap.add_argument("--cap", type=float, default=2.5)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--cpu-samples", type=int, default=768, help="sample points of the cpu_baseline leg (about 12 s on 16 cores)")
    ap.add_argument("--ref-samples", type=int, default=96, help="sample points per step of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--serial", action="store_true", help="two single-operator calls back to back instead of mcs_estimate_dtn_both")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
