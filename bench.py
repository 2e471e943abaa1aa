#!/usr/bin/env python
"""bench.py -- headline measurement of the Monte Carlo DtN hot path on B200.

BASELINE.json's metric ("walk steps/s and DtN matrices/s on 1 B200; fraction of traversal roofline") names no
config, so the headline workload is the largest single-GPU one, configs[3]: the seeded 2 M-face in-the-wild stress
mesh (30 components, 5 % slivers, 1 % duplicated and 2 % flipped faces), 20 000 boundary samples chosen by
farthest-point sampling, 4096 walks each, interior AND exterior operator, sparse (COO) output in the hat basis.
One "step" = one pass of the whole hot path over it: LBVH build, sidedness pre-pass
(winding number), tangent balls, walks and accumulation of both operators.  configs[1] (the
closed-form sphere case of round 1) and a sample of configs[4] (meshes/s end to end, eigenpairs included) are
measured in the same run and reported as sub-records of the same JSON line.  Prints ONE JSON line.

  python bench.py                       # N=1, this repo's CUDA path
  python bench.py --impl reference      # the CPU oracle, as it stands, on a bounded sample of the same workload
  torchrun ... bench.py --gpus N        # N independent replicas
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "walk_steps_per_s"
UNIT = "walk steps/s"


# ------------------------------------------------------------------------------
# workloads (seeded synthetic stand-ins)
# ------------------------------------------------------------------------------
def _cache_dir():
    d = os.path.join(tempfile.gettempdir(), "mcdtn_bench_cache")
    os.makedirs(d, exist_ok=True)
    return d


def make_cfg3(args):
    """configs[3]: stress mesh + FPS samples + Kelvin origin.  Generated once per box (a few seconds) and kept as an
    .npz in the temp directory; always outside the timed region."""
    from synth import fps_samples, stress_mesh
    tag = f"cfg3_F{args.faces}_C{args.components}_S{args.samples}_N{args.candidates}_seed{args.mesh_seed}.npz"
    path = os.path.join(_cache_dir(), tag)
    if os.path.exists(path) and not args.no_cache:
        try:
            z = np.load(path)
            return dict(v=z["v"], f=z["f"], tri=z["tri"], bary=z["bary"], weight=z["weight"], origin=tuple(float(x) for x in z["origin"]),
                        n_components=int(z["n_components"]), flipped=float(z["flipped"]), sliver=float(z["sliver"]), dup=float(z["dup"]))
        except Exception:
            pass
    v, f, info = stress_mesh(n_faces=args.faces, n_components=args.components, seed=args.mesh_seed)
    smp = fps_samples(v, f, args.samples, n_candidates=args.candidates, seed=args.mesh_seed)
    # Kelvin origin strictly inside the solid: the centre of the component with the most faces
    comp = int(np.bincount(info["face_component"]).argmax())
    cv = v[np.unique(f[info["face_component"] == comp])]
    origin = tuple(float(x) for x in 0.5 * (cv.min(0) + cv.max(0)))
    wl = dict(v=v, f=f, tri=smp["tri"], bary=smp["bary"], weight=smp["weight"], origin=origin,
              n_components=int(info["n_components"]), flipped=float(info["flipped"].mean()),
              sliver=float(info["sliver"].mean()), dup=float(info["duplicate"].mean()))
    try:
        np.savez(path, **{k: np.asarray(x) for k, x in wl.items()})
    except OSError:
        pass
    return wl


def cfg3_config(wl, args, extra=None):
    V, F, n_s = len(wl["v"]), len(wl["f"]), len(wl["tri"])
    c = {"workload": f"configs[3]: stress mesh seed {args.mesh_seed} ({V} vertices, {F} faces, {wl['n_components']} components, "
                     f"{100 * wl['sliver']:.1f}% slivers, {100 * wl['dup']:.1f}% duplicated, {100 * wl['flipped']:.1f}% flipped faces), "
                     f"{n_s} FPS samples of {args.candidates} candidates x {args.walks} walks per operator, interior + exterior "
                     f"(killing off: the paper's default, PAPER.md:383), sidedness pre-pass, hat basis, sparse COO output, "
                     f"eps={args.eps:g}, cap={args.cap:g} deg, Philox seed {args.seed}, "
                     + (f"far-field queries by lower bound (far_alpha: exterior {args.far_alpha:g}, interior {args.far_alpha_interior:g}; near={args.far_near:g} eps)" if args.far_alpha > 0 or args.far_alpha_interior > 0 else "exact closest-point queries"),
         "operators": ["interior", "exterior"], "walks_per_operator": n_s * args.walks,
         "includes_bvh_build": True, "includes_sidedness_prepass": True, "output": "coo (upper triangle)",
         "l2_policy": "inputs larger than L2 (tree 256 MB + records 2.6 GB per step) and a 256 MiB buffer written between timed steps",
         "parallelism": "replicas" if args.gpus > 1 else "single"}
    if extra:
        c.update(extra)
    return c


def make_cfg1(level=4, walks_per_vertex=4096, points_per_vertex=16, seed=0):
    from synth import icosphere, vertex_cell_samples
    v, f = icosphere(level)
    smp = vertex_cell_samples(v, f, points_per_vertex, seed=seed)
    W = walks_per_vertex // points_per_vertex
    return dict(v=v, f=f, smp=smp, W=W, name=f"icosphere_L{level}", V=len(v), F=len(f), n_s=len(smp["tri"]))


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


def read_traffic(name):
    """DRAM bytes (read + write) of the walk-kernel launches of one step, from the committed ncu capture under
    profiles/ (a csv of kernel, dram_read_bytes, dram_write_bytes); None when there is no capture."""
    path = os.path.join(ROOT, "profiles", name)
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
def oracle_sample_cfg3(wl, args, n_samples: int, n_walks: int):
    """Interior + exterior walks of `n_walks` walks of every (n_s // n_samples)-th sample point through oracle/
    (brute-force fp64 closest point over all faces; same Philox counters as the full run), then the oracle's
    accumulation of those records.  Returns (walk steps, seconds, cores, description)."""
    from oracle import Oracle, OracleParams, mesh_geom
    n_s = len(wl["tri"])
    stride = max(1, n_s // n_samples)
    ids = np.arange(0, n_s, stride)[:n_samples]
    orc = Oracle(mesh_geom(wl["v"], wl["f"]))
    steps = 0
    t0 = time.perf_counter()
    nrm, _ = orc.orient_samples(wl["tri"][ids], wl["bary"][ids])            # the sidedness pre-pass, on the sample
    normal = np.zeros((n_s, 3), np.float32)
    normal[ids] = nrm
    for ext in (False, True):
        p = OracleParams(seed=args.seed, walks_per_sample=args.walks, eps=args.eps, cap_half_angle_deg=args.cap,
                         origin=wl["origin"])
        rec = orc.run_walks_subset(p, ext, wl["tri"], wl["bary"], wl["weight"], ids, n_walks, normal=normal)
        st = rec["steps"]
        steps += int(st[st > 0].sum())
    dt = time.perf_counter() - t0
    desc = (f"{len(ids)} of {n_s} sample points (every {stride}th) x {n_walks} of {args.walks} walks, interior + exterior, "
            f"sidedness by the oracle's winding number on those points, brute-force fp64 closest point over {len(wl['f'])} faces")
    return steps, dt, orc.num_threads, desc


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    wl = make_cfg3(args)
    for _ in range(args.warmup):
        oracle_sample_cfg3(wl, args, 2, 2)
    total_steps, total_t, cores, desc = 0, 0.0, 0, ""
    for _ in range(args.steps):
        s, dt, cores, desc = oracle_sample_cfg3(wl, args, args.ref_samples, args.ref_walks)
        total_steps += s
        total_t += dt
    value = total_steps / total_t
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total_t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": cfg3_config(wl, args),
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
# roofline of the walk kernel from its own node / triangle counts
# ------------------------------------------------------------------------------
def walk_roofline(stats, t_kernel_s, level_gbs, level, fp32_tflops, note, tri_bytes=48.0):
    nodes = tris = queries = 0.0
    per = {}
    for name, st in stats.items():
        n = st.n_nodes_visited - st.n_prep_nodes
        t = st.n_tris_tested - st.n_prep_tris
        q = st.n_queries - st.n_prep_queries
        per[name] = dict(nodes_per_query=n / max(q, 1), tris_per_query=t / max(q, 1))
        nodes += n; tris += t; queries += q
    flops = 72.0 * nodes + 80.0 * tris              # 4-wide nodes: four 18-flop box tests per visit
    nbytes = 128.0 * nodes + tri_bytes * tris
    t_mem, t_alu = nbytes / (level_gbs * 1e9), flops / (fp32_tflops * 1e12)
    mem_bound = t_mem >= t_alu
    return {
        "kernel": note,
        "bound": level if mem_bound else "alu",
        "achieved": (nbytes / t_kernel_s / 1e9) if mem_bound else (flops / t_kernel_s / 1e12),
        "peak": level_gbs if mem_bound else fp32_tflops,
        "unit": "GB/s" if mem_bound else "TFLOP/s",
        "frac": max(t_mem, t_alu) / t_kernel_s,
        "algorithmic": "bytes = 128 B x 4-wide nodes visited + 48 B x triangles tested; flops = 72 x nodes + 80 x triangles (DESIGN.md section 6)",
        "alu_frac": t_alu / t_kernel_s, "mem_frac": t_mem / t_kernel_s,
        "kernel_ms_per_step": t_kernel_s * 1e3,
        "nodes_per_query": {k: per[k]["nodes_per_query"] for k in per},
        "tris_per_query": {k: per[k]["tris_per_query"] for k in per},
        "algorithmic_bytes_per_step": nbytes, "algorithmic_flops_per_step": flops,
    }


# ------------------------------------------------------------------------------
# the oracle-side ideal of the traversal ("a kernel could raise its fraction by touching more nodes")
# ------------------------------------------------------------------------------
def ideal_traversal_counts(bvh, points, dist, chunk=8):
    """For query points with their EXACT distances (from the oracle's brute force): the number of 4-wide nodes and of
    leaf references of THIS tree whose box is closer than the true distance -- what any exact traversal must visit,
    however it orders its work.  The tree comes from mcs_bvh_dump (binary nodes; a wide node of the walk kernel is a
    binary node at even depth, its box the union of its two child boxes); numpy only, no kernel involved."""
    nodes, leaf_tri, _ = bvh.dump()
    w = nodes.cpu().numpy()
    del nodes
    fw = w.view(np.float32)
    c0, c1 = w[:, 12].copy(), w[:, 13].copy()
    n = len(w)
    depth = np.full(n, -1, np.int32)
    depth[0] = 0
    frontier = np.array([0], np.int64)
    while len(frontier):
        ch = np.concatenate([c0[frontier], c1[frontier]])
        d = np.concatenate([depth[frontier], depth[frontier]]) + 1
        keep = ch >= 0
        depth[ch[keep]] = d[keep]
        frontier = ch[keep].astype(np.int64)
    even = np.flatnonzero((depth & 1) == 0)
    lo = np.minimum(fw[even, 0:3], fw[even, 6:9]); hi = np.maximum(fw[even, 3:6], fw[even, 9:12])       # box of a wide node
    leaf_lo = np.concatenate([fw[c0 < 0, 0:3], fw[c1 < 0, 6:9]]); leaf_hi = np.concatenate([fw[c0 < 0, 3:6], fw[c1 < 0, 9:12]])
    n_nodes, n_leaves = [], []
    for i in range(0, len(points), chunk):
        for p, D in zip(points[i:i + chunk].astype(np.float32), dist[i:i + chunk]):
            d2 = (np.maximum(np.maximum(lo - p, p - hi), 0.0) ** 2).sum(1)
            n_nodes.append(int((d2 < D * D).sum()) + (0 if d2[0] < D * D else 1))                      # the root is always visited
            l2 = (np.maximum(np.maximum(leaf_lo - p, p - leaf_hi), 0.0) ** 2).sum(1)
            n_leaves.append(int((l2 <= D * D * (1 + 1e-6)).sum()))
    return float(np.mean(n_nodes)), float(np.mean(n_leaves)), len(n_nodes)


# ------------------------------------------------------------------------------
# sub-record: configs[1] (icosphere L4, dense output, killing on) -- round 1's headline, kept for continuity
# ------------------------------------------------------------------------------
def bench_cfg1(api, torch, dev, args, seed, steps, warmup, flush, fp32_tflops, l2_gbs):
    wl = make_cfg1()
    n_walks = wl["n_s"] * wl["W"]
    v_h, f_h = torch.as_tensor(wl["v"]).pin_memory(), torch.as_tensor(wl["f"]).pin_memory()
    tri_h, bary_h = torch.as_tensor(wl["smp"]["tri"]).pin_memory(), torch.as_tensor(wl["smp"]["bary"]).pin_memory()
    w_h = torch.as_tensor(wl["smp"]["weight"]).pin_memory()
    vd, fd = v_h.to(dev), f_h.to(dev)
    S = api.Samples(tri_h.to(dev), bary_h.to(dev), w_h.to(dev))
    P_int = api.Params(seed=seed, walks_per_sample=wl["W"], eps=1e-3, cap_half_angle_deg=2.5)
    P_ext = api.Params(seed=seed, walks_per_sample=wl["W"], eps=1e-3, cap_half_angle_deg=2.5, include_killing=True, n_kill_walks=n_walks)
    bvh0 = api.build_bvh(vd, fd)
    ws = torch.empty(api.workspace_bytes_both(bvh0, S, P_int, P_ext), dtype=torch.uint8, device=dev)
    out_int = torch.empty((wl["V"], wl["V"]), dtype=torch.float32, device=dev)
    out_ext = torch.empty_like(out_int)
    _, st_i = api.estimate_dtn_interior(bvh0, S, P_int, want_stats=True, out=out_int, workspace=ws)
    _, st_e = api.estimate_dtn_exterior(bvh0, S, P_ext, want_stats=True, out=out_ext, workspace=ws)
    del bvh0
    phases = []

    def step(profile):
        bvh = api.build_bvh(vd, fd)
        api.estimate_dtn_both(bvh, S, P_int, P_ext, out_interior=out_int, out_exterior=out_ext, workspace=ws)
        if profile:
            phases.append(api.profile_last())

    for _ in range(warmup):
        step(False); flush.fill_(1)
    api.profile_enable(True)
    stream = torch.cuda.current_stream(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    l0 = api.launch_count()
    e0.record(stream)
    for _ in range(steps):
        step(True); flush.fill_(1)
    e1.record(stream)
    torch.cuda.synchronize()
    launches = api.launch_count() - l0
    api.profile_enable(False)
    ms = e0.elapsed_time(e1) / steps
    walk_steps = st_i.n_steps + st_e.n_steps
    t_kernel = float(np.mean([p.walk_ms for p in phases])) * 1e-3
    roof = walk_roofline({"interior": st_i, "exterior": st_e}, t_kernel, l2_gbs, "l2", fp32_tflops,
                         "walk_kernel (interior + exterior launch of one step, overlapped: span of both)")
    roof["peak_source"] = "L2 read bandwidth measured live by mcs_measure_l2_gbs (the 0.6 MB tree is L2-resident)"
    roof["traffic"] = read_traffic("walk_kernel_traffic.csv")
    # end to end through the host entry point (dense matrices back to pinned host memory)
    oi_h = torch.empty((wl["V"], wl["V"]), dtype=torch.float32, pin_memory=True)
    oe_h = torch.empty_like(oi_h).pin_memory()
    for _ in range(4):
        r = api.estimate_dtn_host(v_h, f_h, tri_h, bary_h, w_h, P_ext, out_interior=oi_h, out_exterior=oe_h, device=dev)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    n_e2e = max(1, min(steps, 5))
    for _ in range(n_e2e):
        r = api.estimate_dtn_host(v_h, f_h, tri_h, bary_h, w_h, P_ext, out_interior=oi_h, out_exterior=oe_h, device=dev)
        flush.fill_(1)
    torch.cuda.synchronize()
    e2e_t = (time.perf_counter() - t0) / n_e2e
    return {"workload": f"configs[1]: {wl['name']} ({wl['V']} vertices, {wl['F']} faces), interior + exterior(killing on), hat basis, dense "
                        f"output, 4096 walks/vertex = {wl['n_s']} sample points x {wl['W']} walks per operator, eps=1e-3, cap=2.5 deg",
            "metric": METRIC, "value": walk_steps / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms, "steps": steps, "warmup": warmup,
            "dtn_matrices_per_s": 2.0 / (ms * 1e-3), "walk_steps_per_step": walk_steps,
            "queries_per_s": (st_i.n_queries + st_e.n_queries) / (ms * 1e-3),
            "phase_ms_per_step": {"prep": float(np.mean([p.prep_ms for p in phases])), "walk": t_kernel * 1e3,
                                  "accumulate": float(np.mean([p.accumulate_ms for p in phases]))},
            "e2e": {"value": walk_steps / e2e_t, "unit": UNIT, "ms_per_step": e2e_t * 1e3, "h2d_bytes_per_step": r["h2d_bytes"],
                    "d2h_bytes_per_step": r["d2h_bytes"], "call": "mcs_estimate_dtn_host (pinned host buffers)"},
            "gpu_launches": launches, "roofline": roof}


# ------------------------------------------------------------------------------
# sub-record: a sample of configs[4] (meshes/s end to end: build, sidedness, both operators, top-64 eigenpairs)
# ------------------------------------------------------------------------------
def make_cfg4_sample(n_meshes, seed0=0):
    """Meshes seeds seed0.. of BASELINE configs[4]: faces log-uniform in [5k, 200k], 1-50 components, stress style;
    512 FPS samples that are also the nodes of the k-NN point basis (R3)."""
    from synth import fps_samples, stress_mesh
    out = []
    for s in range(seed0, seed0 + n_meshes):
        rng = np.random.default_rng(10_000 + s)
        n_faces = int(round(np.exp(rng.uniform(np.log(5_000), np.log(200_000)))))
        n_comp = int(rng.integers(1, 51))
        v, f, info = stress_mesh(n_faces=n_faces, n_components=n_comp, seed=s)
        smp = fps_samples(v, f, 512, n_candidates=20_000, seed=s)
        comp = int(np.bincount(info["face_component"]).argmax())
        cv = v[np.unique(f[info["face_component"] == comp])]
        origin = tuple(float(x) for x in 0.5 * (cv.min(0) + cv.max(0)))
        a, b, c = v[f[smp["tri"], 0]], v[f[smp["tri"], 1]], v[f[smp["tri"], 2]]
        pts = (smp["bary"][:, 0:1] * a + smp["bary"][:, 1:2] * b + smp["bary"][:, 2:3] * c).astype(np.float32)
        out.append(dict(v=v, f=f, tri=smp["tri"], bary=smp["bary"], weight=smp["weight"], pts=pts, origin=origin, seed=s))
    return out


def bench_cfg4_sample(api, torch, dev, args, seed, n_meshes, flush):
    meshes = make_cfg4_sample(n_meshes)
    W, n_eig, K = 1024, 64, 512
    pinned = [{k: torch.as_tensor(m[k]).pin_memory() for k in ("v", "f", "tri", "bary", "weight", "pts")} for m in meshes]
    Si = torch.empty((n_meshes, K, K), dtype=torch.float32, device=dev)
    Se = torch.empty_like(Si)
    mass = torch.empty((n_meshes, K), dtype=torch.float32, device=dev)
    Pi = api.Params(seed=seed, walks_per_sample=W, eps=1e-3, far_alpha=args.far_alpha_interior, far_near_factor=args.far_near)
    Pe = api.Params(seed=seed, walks_per_sample=W, eps=1e-3, far_alpha=args.far_alpha, far_near_factor=args.far_near)

    def one_pass():
        # upload of every mesh from pinned host memory (async on the current stream), then ONE batch call: per mesh
        # LBVH build, sidedness, both estimators in the k-NN point basis of its 512 samples (normals of the basis =
        # face normals at the samples, oriented by the same sidedness rule in a first batch of normals-only work)
        items = []
        for m, h in zip(meshes, pinned):
            vd, fd = h["v"].to(dev, non_blocking=True), h["f"].to(dev, non_blocking=True)
            S0 = api.Samples(h["tri"].to(dev, non_blocking=True), h["bary"].to(dev, non_blocking=True), h["weight"].to(dev, non_blocking=True))
            items.append(dict(verts=vd, faces=fd, samples=S0, origin=m["origin"], pts=h["pts"].to(dev, non_blocking=True)))
        # the point basis needs outward normals at the nodes: face normals of the samples, oriented by the library
        for it in items:
            f_s = it["faces"][it["samples"].tri.long()].long()
            a, b, c = it["verts"][f_s[:, 0]], it["verts"][f_s[:, 1]], it["verts"][f_s[:, 2]]
            n = torch.linalg.cross(b - a, c - a)
            it["basis"] = api.PointBasis(it["pts"], n / n.norm(dim=1, keepdim=True).clamp_min(1e-30), k=8, sigma=0.025, tau_n=0.8)
        normals = api.estimate_dtn_batch(items, Pi, Pe, Si, Se, orient_h_scale=1.0, orient_beta=args.orient_beta if args.orient_beta > 0 else 0.0,
                                         n_workers=args.cfg4_workers)
        for i, it in enumerate(items):
            mass[i] = it["samples"].weight
        # Steklov eigenpairs of all 2 x n matrices in ONE batched call (lumped mass = the samples' weights)
        ev, _, _ = api.steklov_eigs(torch.cat([Si, Se]), torch.cat([mass, mass]), n_eig)
        return ev[:n_meshes], ev[n_meshes:]

    one_pass()                                      # warm-up
    torch.cuda.synchronize()
    stream = torch.cuda.current_stream(dev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = api.launch_count()
    t0 = time.perf_counter()
    e0.record(stream)
    one_pass()
    e1.record(stream)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    ms = e0.elapsed_time(e1)
    faces = [len(m["f"]) for m in meshes]
    return {"workload": f"configs[4] sample: {n_meshes} stress-style meshes (seeds 0..{n_meshes - 1}, {min(faces)}-{max(faces)} faces), per mesh: "
                        f"upload from pinned host memory, LBVH build, sidedness pre-pass, 512 FPS samples = nodes of the k-NN point basis "
                        f"(k=8, face normals at the nodes), {W} walks per sample, interior + exterior (killing off; far-field bounds as "
                        f"in the headline) through ONE mcs_estimate_dtn_batch call ({args.cfg4_workers} workers prepare and accumulate, one launch walks "
                        f"all meshes), then top-{n_eig} Steklov eigenpairs of all {2 * n_meshes} matrices in one batched call",
            "metric": "meshes_per_s", "value": n_meshes / (ms * 1e-3), "unit": "meshes/s", "ms_per_mesh": ms / n_meshes,
            "wall_ms_per_mesh": wall * 1e3 / n_meshes, "gpu_launches": api.launch_count() - l0, "meshes": n_meshes,
            "mean_faces": float(np.mean(faces)), "workers": args.cfg4_workers}


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
    wl = make_cfg3(args)
    V, F, n_s, W = len(wl["v"]), len(wl["f"]), len(wl["tri"]), args.walks
    v_h, f_h = torch.as_tensor(wl["v"]).pin_memory(), torch.as_tensor(wl["f"]).pin_memory()
    tri_h, bary_h, w_h = (torch.as_tensor(wl[k]).pin_memory() for k in ("tri", "bary", "weight"))
    vd, fd = v_h.to(dev), f_h.to(dev)
    S0 = api.Samples(tri_h.to(dev), bary_h.to(dev), w_h.to(dev))
    # far-field queries by a lower bound of the distance in both operators (F1; any ball inside the domain is a
    # valid walk-on-spheres jump): the walks take more, cheaper jumps and land with the same distribution.
    # The exact-query step (far_alpha = 0) is measured next to it as a sub-record.
    P_int0 = api.Params(seed=seed, walks_per_sample=W, eps=args.eps, cap_half_angle_deg=args.cap)
    P_int = api.Params(seed=seed, walks_per_sample=W, eps=args.eps, cap_half_angle_deg=args.cap,
                       far_alpha=args.far_alpha_interior, far_near_factor=args.far_near)
    P_ext = api.Params(seed=seed, walks_per_sample=W, eps=args.eps, cap_half_angle_deg=args.cap, kelvin_origin=wl["origin"],
                       far_alpha=args.far_alpha, far_near_factor=args.far_near)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    # deterministic work counts of one step (counter build of the kernels) and the size of the sparse outputs;
    # outside the timed region
    bvh0 = api.build_bvh(vd, fd)
    info = bvh0.info()
    nrm0, _ = api.orient_samples_fast(bvh0, S0, beta=args.orient_beta) if args.orient_beta > 0 else api.orient_samples(bvh0, S0)
    S = api.Samples(S0.tri, S0.bary, S0.weight, nrm0)
    ci, st_i = api.estimate_dtn_coo(bvh0, S, P_int, False, want_stats=True)
    ce, st_e = api.estimate_dtn_coo(bvh0, S, P_ext, True, want_stats=True)
    nnz = (ci.nnz, ce.nnz)
    cap = int(max(nnz) * 1.02) + 4096
    del ci, ce, bvh0, S, nrm0
    torch.cuda.empty_cache()
    steps_per_step = st_i.n_steps + st_e.n_steps
    queries_per_step = st_i.n_queries + st_e.n_queries
    phases = []
    scratch = {}                   # workspace and output buffers of the timed call, kept between steps

    def step(profile):
        bvh = api.build_bvh(vd, fd)
        nrm, _ = api.orient_samples_fast(bvh, S0, beta=args.orient_beta) if args.orient_beta > 0 else api.orient_samples(bvh, S0)
        Sx = api.Samples(S0.tri, S0.bary, S0.weight, nrm)
        out = api.estimate_dtn_coo_both(bvh, Sx, P_int, P_ext, capacity=cap, scratch=scratch)
        if profile:
            phases.append(api.profile_last())
        return out

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
    scratch.clear()
    job_steps = sum_over_ranks(steps_per_step, dev, world)        # replicas differ by their Philox seed
    job_queries = sum_over_ranks(queries_per_step, dev, world)
    value = job_steps / (ms_per_step * 1e-3)
    torch.cuda.empty_cache()

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    host_out = [tuple(torch.empty(cap, dtype=dt, pin_memory=True) for dt in (torch.int32, torch.int32, torch.float32)) for _ in range(2)]
    e2e_steps = max(1, min(args.steps, 3))
    for _ in range(2):
        r = api.estimate_dtn_host_coo(v_h, f_h, tri_h, bary_h, w_h, P_int, P_ext, host_out[0], host_out[1], orient_h_scale=1.0, orient_beta=args.orient_beta, device=dev)
    barrier()
    t0 = time.perf_counter()
    e2e_each = []
    for _ in range(e2e_steps):
        tc = time.perf_counter()
        r = api.estimate_dtn_host_coo(v_h, f_h, tri_h, bary_h, w_h, P_int, P_ext, host_out[0], host_out[1], orient_h_scale=1.0, orient_beta=args.orient_beta, device=dev)
        e2e_each.append((time.perf_counter() - tc) * 1e3)      # the call blocks until the entries are in host memory
        flush.fill_(1)
    barrier()
    e2e_t = (time.perf_counter() - t0) / e2e_steps
    e2e_t = max_over_ranks(e2e_t, dev, world)
    e2e_value = job_steps / e2e_t
    del host_out
    torch.cuda.empty_cache()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (the persistent walk kernel)
    fp32_tflops = api.measure_fp32_tflops(dev)
    l2_gbs = api.measure_l2_gbs(dev)
    hbm_gbs, hbm_src = read_peaks()
    tree_bytes = int(info.device_bytes)
    t_kernel = float(np.mean([p.walk_ms for p in phases])) * 1e-3
    roofline = walk_roofline({"interior": st_i, "exterior": st_e}, t_kernel, hbm_gbs, "hbm", fp32_tflops,
                             "walk_kernel (interior launch + exterior launch of one step, overlapped on two streams: span of both)")
    roofline["peak_source"] = (f"HBM {hbm_gbs:.0f} GB/s {hbm_src}: packed tree + triangles are {tree_bytes / 1e6:.0f} MB > L2; "
                               f"FP32 {fp32_tflops:.1f} TFLOP/s and L2 {l2_gbs:.0f} GB/s measured live")
    roofline["l2_frac"] = roofline["algorithmic_bytes_per_step"] / (l2_gbs * 1e9) / t_kernel
    # DRAM bytes of the two walk launches of one step from the committed ncu pass (profiles/r02_cfg3_walk_dram.md), which was
    # taken at the default workload: any other size has no capture
    default_wl = (args.faces == 2_000_000 and args.samples == 20_000 and args.walks == 4096 and args.components == 30
                  and args.mesh_seed == 3 and abs(args.far_alpha - 2.0) < 1e-9 and abs(args.far_alpha_interior - 1.0) < 1e-9
                  and abs(args.far_near - 2.0) < 1e-9 and abs(args.eps - 1e-3) < 1e-12)
    roofline["traffic"] = read_traffic("r02_cfg3_walk_traffic.csv") if default_wl else None
    roofline["traffic_note"] = ("dram__bytes_read.sum + dram__bytes_write.sum of the interior and the exterior launch of one step (ncu, "
                                "profiles/r02_cfg3_walk_dram.md): 2 % of the algorithmic bytes -- the tree is served by L2 (2740 GB of L2 traffic)"
                                if default_wl else "null: the committed capture is of the default workload")
    roofline["kernel_share_of_step"] = t_kernel * 1e3 / ms_per_step
    cut = (st_i.n_truncated + st_e.n_truncated) / float(st_i.n_walks + st_e.n_walks)

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        s, dt, cores, desc = oracle_sample_cfg3(wl, args, args.cpu_samples, args.cpu_walks)
        cpu = {"value": s / dt, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "seconds": dt}
        # ideal node / leaf counts of the same tree on the oracle's own query points (a sample of the walks' queries)
        try:
            from oracle import Oracle, OracleParams, mesh_geom
            orc = Oracle(mesh_geom(wl["v"], wl["f"]))
            ids = np.arange(0, n_s, max(1, n_s // args.ideal_samples))[:args.ideal_samples]
            bvh_i = api.build_bvh(vd, fd)
            ids_d = torch.as_tensor(ids, device=dev)
            nrm_i, _ = api.orient_samples(bvh_i, api.Samples(S0.tri[ids_d].contiguous(), S0.bary[ids_d].contiguous(), S0.weight[ids_d].contiguous()))
            normal = np.zeros((n_s, 3), np.float32); normal[ids] = nrm_i.cpu().numpy()
            ideal = {}
            for ext in (False, True):
                op = OracleParams(seed=args.seed, walks_per_sample=W, eps=args.eps, cap_half_angle_deg=args.cap, origin=wl["origin"])
                pts, dd = orc.walk_query_points(op, ext, wl["tri"], wl["bary"], wl["weight"], ids, 2, max_pos=16, normal=normal)
                nn, nl, nq = ideal_traversal_counts(bvh_i, pts, dd)
                ideal["exterior" if ext else "interior"] = {"wide_nodes_per_query": nn, "leaf_boxes_per_query": nl, "queries": nq}
            del bvh_i
            roofline["ideal_exact_traversal"] = dict(ideal, note="wide nodes / leaf references of the same tree whose box is closer than the exact "
                                                     "distance (oracle brute force) at the query points of the oracle's own walks: the least any exact "
                                                     "traversal visits; compare with nodes_per_query / tris_per_query of the exact-query runs")
        except Exception as exc:                     # a measurement aid: never fail the bench line
            roofline["ideal_exact_traversal"] = {"error": repr(exc)}

    sub = {}
    if world == 1 and not args.no_sub and (args.far_alpha > 0 or args.far_alpha_interior > 0):
        # the same step with EXACT closest-point queries in both operators (far_alpha = 0), for comparison
        P_ext0 = api.Params(seed=seed, walks_per_sample=W, eps=args.eps, cap_half_angle_deg=args.cap, kelvin_origin=wl["origin"])
        sc0 = {}

        def step0():
            bvh = api.build_bvh(vd, fd)
            nrm, _ = api.orient_samples_fast(bvh, S0, beta=args.orient_beta) if args.orient_beta > 0 else api.orient_samples(bvh, S0)
            api.estimate_dtn_coo_both(bvh, api.Samples(S0.tri, S0.bary, S0.weight, nrm), P_int0, P_ext0, capacity=int(cap * 1.05), scratch=sc0)
        for _ in range(2):
            step0(); flush.fill_(1)
        n0 = max(1, min(args.steps, 3))
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(n0):
            step0(); flush.fill_(1)
        e1.record(stream)
        torch.cuda.synchronize()
        ms0 = e0.elapsed_time(e1) / n0
        bvh0 = api.build_bvh(vd, fd)
        nrm0, _ = api.orient_samples_fast(bvh0, S0, beta=args.orient_beta) if args.orient_beta > 0 else api.orient_samples(bvh0, S0)
        _, st_e0 = api.run_walks(bvh0, api.Samples(S0.tri, S0.bary, S0.weight, nrm0), P_ext0, True, want_stats=True)[1:]
        _, st_i0 = api.run_walks(bvh0, api.Samples(S0.tri, S0.bary, S0.weight, nrm0), P_int0, False, want_stats=True)[1:]
        del bvh0, nrm0
        sc0.clear()
        torch.cuda.empty_cache()
        steps0 = st_i0.n_steps + st_e0.n_steps
        sub["configs[3] exact queries"] = {"workload": "the headline step with far_alpha = 0 in both operators (every closest-point query exact)",
                                           "metric": METRIC, "value": steps0 / (ms0 * 1e-3), "unit": UNIT, "ms_per_step": ms0, "steps": n0,
                                           "walk_steps_per_step": steps0, "dtn_matrices_per_s": 2.0 / (ms0 * 1e-3),
                                           "interior_nodes_per_query": (st_i0.n_nodes_visited - st_i0.n_prep_nodes) / max(st_i0.n_queries - st_i0.n_prep_queries, 1),
                                           "interior_tris_per_query": (st_i0.n_tris_tested - st_i0.n_prep_tris) / max(st_i0.n_queries - st_i0.n_prep_queries, 1),
                                           "exterior_nodes_per_query": (st_e0.n_nodes_visited - st_e0.n_prep_nodes) / max(st_e0.n_queries - st_e0.n_prep_queries, 1),
                                           "exterior_tris_per_query": (st_e0.n_tris_tested - st_e0.n_prep_tris) / max(st_e0.n_queries - st_e0.n_prep_queries, 1)}
    if world == 1 and not args.no_sub:
        sub["configs[1]"] = bench_cfg1(api, torch, dev, args, seed, min(args.steps, 5), 3, flush, fp32_tflops, l2_gbs)
        sub["configs[4] sample"] = bench_cfg4_sample(api, torch, dev, args, seed, args.cfg4_meshes, flush)

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic", "config": cfg3_config(wl, args),
            "queries_per_s": job_queries / (ms_per_step * 1e-3),
            "dtn_matrices_per_s": world * 2.0 / (ms_per_step * 1e-3),
            "walk_steps_per_step": steps_per_step, "queries_per_step": queries_per_step,
            "nnz": {"interior": nnz[0], "exterior": nnz[1]},
            "far_query_fraction": (st_i.n_far_queries + st_e.n_far_queries) / float(max(queries_per_step, 1)),
            "far_field_note": ("value counts the jumps the walks really take; with far-field bounds they take more, shorter ones than the exact "
                               "run for the same matrices in distribution (tests/test_gpu_farfield.py), so ms_per_step / dtn_matrices_per_s "
                               "compare configurations, and value_exact_equivalent = (jumps of the exact-query run of sub_records) / (this step's time)"),
            "cut_fraction": cut, "cut_walks": {"interior": st_i.n_truncated, "exterior": st_e.n_truncated,
                                               "rule": "R10 max_steps / R10b left the bounding box / R10c inside the solid (DESIGN.md section 2)"},
            "discarded_samples": {"interior": st_i.n_discarded, "exterior": st_e.n_discarded},
            "bvh": {"faces": int(info.F), "nodes": int(info.n_nodes), "max_depth": int(info.max_depth), "device_bytes": tree_bytes},
            "call": "mcs_build_bvh + " + ("mcs_orient_samples_fast" if args.orient_beta > 0 else "mcs_orient_samples") + " + mcs_estimate_dtn_both (output_kind 1)",
            "phase_ms_per_step": {"build+sidedness+flush": ms_per_step - float(np.mean([p.total_ms for p in phases])),
                                  "prep": float(np.mean([p.prep_ms for p in phases])), "walk": t_kernel * 1e3,
                                  "accumulate": float(np.mean([p.accumulate_ms for p in phases]))},
            "walk_end_ms": {"interior": float(np.mean([p.walk_interior_ms for p in phases])),
                            "exterior": float(np.mean([p.walk_exterior_ms for p in phases]))},
            "clocks": clk,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": r["h2d_bytes"], "d2h_bytes_per_step": r["d2h_bytes"],
                    "ms_per_step": e2e_t * 1e3, "ms_per_call": e2e_each, "steps": e2e_steps,
                    "call": "mcs_estimate_dtn_host_coo (pinned host buffers: mesh + samples up, COO entries of both operators down)"},
            "gpu_launches": launches, "roofline": roofline, "cpu_baseline": cpu, "sub_records": sub}
    ex = sub.get("configs[3] exact queries")
    line["value_exact_equivalent"] = (world * ex["walk_steps_per_step"] / (ms_per_step * 1e-3)) if ex else None
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_only(args):
    """One sub-record alone on cuda:0 (so that an ncu launch list shows that workload and nothing else)."""
    import torch
    from paper_2606_05581_b200 import api
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this path has no CPU fallback)")
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    api.lib()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    if args.only == "cfg4":
        rec = bench_cfg4_sample(api, torch, dev, args, args.seed, args.cfg4_meshes, flush)
    else:
        rec = bench_cfg1(api, torch, dev, args, args.seed, min(args.steps, 5), 3, flush, api.measure_fp32_tflops(dev), api.measure_l2_gbs(dev))
    print(json.dumps({"only": args.only, **rec}))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--faces", type=int, default=2_000_000, help="configs[3]: faces of the stress mesh")
    ap.add_argument("--components", type=int, default=30)
    ap.add_argument("--samples", type=int, default=20_000, help="boundary samples by farthest-point sampling")
    ap.add_argument("--candidates", type=int, default=1_000_000, help="area-uniform candidates of the FPS")
    ap.add_argument("--walks", type=int, default=4096, help="walks per sample and operator")
    ap.add_argument("--mesh-seed", type=int, default=3)
    ap.add_argument("--eps", type=float, default=1e-3)
    ap.add_argument("--cap", type=float, default=2.5)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--orient-beta", type=float, default=2.5, help="sidedness pre-pass: opening parameter of mcs_orient_samples_fast (0: exhaustive mcs_orient_samples)")
    ap.add_argument("--far-alpha", type=float, default=2.0, help="mcs_params.far_alpha of the exterior: > 0 answers far-field queries with a lower bound of the distance")
    ap.add_argument("--far-alpha-interior", type=float, default=1.0, help="mcs_params.far_alpha of the interior (0: exact queries)")
    ap.add_argument("--far-near", type=float, default=2.0, help="mcs_params.far_near_factor (multiples of eps)")
    ap.add_argument("--cpu-samples", type=int, default=16, help="sample points of the cpu_baseline leg")
    ap.add_argument("--cpu-walks", type=int, default=8, help="walks per sample point of the cpu_baseline leg")
    ap.add_argument("--ref-samples", type=int, default=8, help="sample points per step of --impl reference")
    ap.add_argument("--ref-walks", type=int, default=4, help="walks per sample point per step of --impl reference")
    ap.add_argument("--ideal-samples", type=int, default=24, help="sample points whose oracle walks give the query points of the ideal traversal count")
    ap.add_argument("--cfg4-meshes", type=int, default=32, help="meshes of the configs[4] sample sub-record")
    ap.add_argument("--cfg4-workers", type=int, default=4, help="host workers of mcs_estimate_dtn_batch in that sub-record")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sub", action="store_true", help="skip the configs[1] / configs[4] sub-records")
    ap.add_argument("--no-cache", action="store_true", help="regenerate the workload instead of reading the temp-dir cache")
    ap.add_argument("--only", choices=["cfg1", "cfg4"], default=None,
                    help="run ONE sub-record alone and print its JSON (profiling aid: profiles/r02_cfg4_launches.md); not the bench line")
    args = ap.parse_args()
    if args.only:
        return run_only(args)
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
