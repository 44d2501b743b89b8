#!/usr/bin/env python
"""bench.py -- the Muon optimizer step of DMuon (arxiv/paper_2606_27153) on B200, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one pass of the whole hot path (momentum+Nesterov+cast+norm, 5 Newton-Schulz steps of grouped GEMMs per
shape bucket, the weight update applied in the last X-update epilogue) over one synthetic matrix set.  Default
workload: BASELINE.json configs[3], the Llama-3-8B-shaped set (224 matrices, 6.98 G elements, bf16 W/G/M resident in
HBM), the configuration the metric is quoted on.  `value` = dense-equivalent NS TFLOP/s of the whole step
(BASELINE.json: "counting the full dense FLOPs") = sum over matrices of 5 (4 m^2 n + 2 m^3) divided by the step time,
aggregated over ranks.  The timed loop runs with the library's per-launch profiling OFF; the per-kernel breakdown
(`kernels`, `launch_types`, `roofline`) comes from a second pass of the same K steps with CUDA events around every
launch.  The path does not shard (north_star: one GPU, no collectives): --gpus N runs N independent replicas
("replicas only"), timed as the max over ranks.
--impl reference times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
--sweep runs BASELINE.json configs[4] (NS-only shape sweep), one JSON line per shape.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Muon step NS throughput, dense-equivalent FLOPs (BASELINE: Muon step ms & NS TFLOP/s, % of B200 bf16 peak)"
UNIT = "TFLOP/s"
LR, MU, WD = 0.02, 0.95, 0.01
NS_STEPS = 5
WORKLOADS = {1: "config1: tiny NS batch 8 x (128x512)", 2: "config2: GPT-2-small-shaped, 72 matrices",
             3: "config3: Qwen-0.5B-style, 168 matrices", 4: "config4: Llama-3-8B-shaped, 224 matrices, 6.98 G elements"}
GEMM_X = ("ns_bx_update", "ns_bx_apply", "ns_bx_out", "ns_xb_update", "ns_xb_apply", "ns_xb_out")
PROGRAM = ("ns_program", "ns_program_out", "ns_program_apply")     # option program=1: a bucket's whole NS program, one launch
SMALL_FUSED = ("ns_small_fused", "ns_small_fused_out", "ns_small_fused_apply")     # the on-chip kernel: all steps, one launch


# ------------------------------------------------------------------------------------------------ accounting
def oriented(shape):
    r, c = shape
    return min(r, c), max(r, c)


def dense_flops(shapes, steps=NS_STEPS):
    """Metric FLOPs: 5 (4 m^2 n + 2 m^3) per matrix."""
    return sum(steps * (4 * m * m * n + 2 * m ** 3) for m, n in map(oriented, shapes))


def pad128(v):
    return -(-v // 128) * 128


def bucket_key(shape):
    """(m_pad, n_pad, kind) of the library's bucket for a stored shape: aligned matrices (rows, cols multiples of 128)
    are held as stored -- "wide" (rows <= cols) or "tall" -- the others oriented and padded ("generic")."""
    r, c = shape
    m, n = oriented(shape)
    aligned = r % 128 == 0 and c % 128 == 0
    return pad128(m), pad128(n), ("generic" if not aligned else ("wide" if r <= c else "tall"))


def launch_counts(shapes, plan):
    """Per matrix (m, n, products): how many launches of each product family the library's block schedule
    (dmuon_describe_plan) runs.  A block of length L: 1 Gram product (SYRK), L polynomial products, 3 (L - 1)
    Gram-space products (T = aG + BG, G' = aT + TB, R' = pB' + aR + B'R), 1 X update."""
    blocks, onchip = {}, {}
    for b in plan["buckets"]:
        blocks[(b["m"], b["n"], b.get("kind", "wide"))] = b["blocks"]
        blocks.setdefault((b["m"], b["n"]), b["blocks"])          # plans described without a kind
        onchip[(b["m"], b["n"], b.get("kind", "wide"))] = onchip[(b["m"], b["n"])] = bool(b.get("onchip", False))
    out = []
    for s in shapes:
        m, n = oriented(s)
        key = bucket_key(s)
        part = blocks.get(key) or blocks[key[:2]]
        out.append((m, n, {"syrk": len(part), "ns_sq_poly": sum(part), "ns_gram_mm": sum(3 * (L - 1) for L in part),
                           "xupd": len(part), "onchip": onchip.get(key, onchip.get(key[:2], False))}))
    return out


def executed_flops(shapes, plan):
    """FLOPs the kernels execute: every m x m result and X X^T is symmetric and only its upper-triangular 128-blocks
    are computed, a share (T+1)/(2T) of the dense product; X updates are dense.  The on-chip small-matrix kernel
    computes its 256 x 256 products in full."""
    tot = 0.0
    for m, n, cnt in launch_counts(shapes, plan):
        t = -(-m // 128)
        sym = 1.0 if cnt["onchip"] else (t + 1) / (2 * t)
        tot += sym * (cnt["syrk"] * 2 * m * m * n + (cnt["ns_sq_poly"] + cnt["ns_gram_mm"]) * 2 * m ** 3)
        tot += cnt["xupd"] * 2 * m * m * n
    return tot


def family_work(family, shapes, plan, x_share=1.0):
    """Algorithmic work per step of one kernel family over `shapes`: ("flop" | "byte", amount).
    For the symmetric products the algorithmic FLOPs are those of the upper-triangular 128-blocks, (T+1)/(2T) of the
    dense 2 m^2 n or 2 m^3 (the rest of the result is a mirror, not arithmetic); the X update is dense.  The X updates
    of a bucket run under two names (plain "_update", fused last "_apply" / "_out"): x_share = this name's share."""
    el = sum(r * c for r, c in shapes)
    if family == "momentum_nesterov_sumsq":
        return "byte", 8 * el                      # read G, M; write M', U          (a1 + a2)
    if family == "sumsq":
        return "byte", 2 * el
    if family == "normalize_cast":
        return "byte", 4 * el                      # read U; write X0
    if family == "apply_update":
        return "byte", 6 * el                      # read O, W; write W'             (a6, when not fused)
    if family == "store_ns_output":
        return "byte", 4 * el
    if family in PROGRAM:                          # every product of the bucket's schedule (symmetry-aware, as executed)
        return "flop", executed_flops(shapes, plan)
    if family in SMALL_FUSED:                      # every product of every step, dense, on the padded 256 x 256 matrix
        return "flop", sum((c["syrk"] + c["ns_sq_poly"] + c["xupd"]) * 2 * 256 ** 3 for m, n, c in launch_counts(shapes, plan) if c["onchip"])
    lc = [x for x in launch_counts(shapes, plan) if not x[2]["onchip"]]
    sym = lambda m: (-(-m // 128) + 1) / (2 * -(-m // 128))
    if family in ("ns_syrk_xxt", "ns_syrk_xtx"):
        return "flop", sum(c["syrk"] * sym(m) * 2 * m * m * n for m, n, c in lc)
    if family in ("ns_sq_poly", "ns_gram_mm"):
        return "flop", sum(c[family] * sym(m) * 2 * m ** 3 for m, n, c in lc)
    if family in GEMM_X:
        return "flop", x_share * sum(c["xupd"] * 2 * m * m * n for m, n, c in lc)
    return None, 0


def launch_type_key(name):
    """'family[R x C]' -> (m_pad, n_pad, tall?): GEMM launches are named by the bucket's stored shape."""
    R, C = (int(v) for v in name[name.index("[") + 1:-1].split("x"))
    return (min(R, C), max(R, C), R > C)


def shapes_of_launch_type(name, shapes):
    m_pad, n_pad, tall = launch_type_key(name)
    return [s for s in shapes if bucket_key(s)[:2] == (m_pad, n_pad) and (bucket_key(s)[2] == "tall") == tall]


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"hbm_gbs": p["hbm_gbs"], "tflops_burst": p["bf16_tflops"],
                "tflops_sustained": p.get("bf16_tflops_sustained", p["bf16_tflops"]), "source": "measured"}
    # fallback stated in /opt/skills/guides/B200_PROFILING.md
    return {"hbm_gbs": 6650.0, "tflops_burst": 1590.0, "tflops_sustained": 1400.0, "source": "fallback"}


def profile_breakdown(prof, steps, ms, shapes, plan, peaks):
    """(kernels per family, launch_types per family and bucket, dominant launch type) from the library's own CUDA events
    (recorded on the launching stream) over `steps` steps of `ms` each."""
    def entry(ms_tot, launches, kind, amount):
        per_step_ms = ms_tot / steps
        e = {"launches_per_step": launches / steps, "ms_per_step": per_step_ms, "share": per_step_ms / ms}
        if kind and per_step_ms > 0:
            if kind == "flop":
                ach = amount / (per_step_ms * 1e-3) / 1e12
                e.update({"bound": "tensor", "achieved": ach, "unit": "TFLOP/s", "frac": ach / peaks["tflops_sustained"],
                          "frac_of_burst": ach / peaks["tflops_burst"], "frac_of_nominal_2250": ach / 2250.0,
                          "work_per_step": amount})
            else:
                ach = amount / (per_step_ms * 1e-3) / 1e9
                e.update({"bound": "hbm", "achieved": ach, "unit": "GB/s", "frac": ach / peaks["hbm_gbs"], "work_per_step": amount})
        return e

    launch_types, kernels = {}, {}
    for name, rec in prof["kernels"].items():
        fam = name.split("[")[0]
        if "[" not in name:
            kernels[fam] = entry(rec["ms"], rec["launches"], *family_work(fam, shapes, plan))
            continue
        sub = shapes_of_launch_type(name, shapes)
        share = 1.0
        if fam in GEMM_X:           # plain and fused X updates of one bucket share its X updates, by launch count
            twins = [n for n in prof["kernels"] if n.split("[")[0] in GEMM_X and "[" in n and launch_type_key(n) == launch_type_key(name)]
            share = rec["launches"] / sum(prof["kernels"][n]["launches"] for n in twins)
        launch_types[name] = entry(rec["ms"], rec["launches"], *family_work(fam, sub, plan, share))
        m_pad, n_pad, tall = launch_type_key(name)
        chunks = [b["count"] for b in plan["buckets"] if (b["m"], b["n"]) == (m_pad, n_pad) and (b.get("kind") == "tall") == tall]
        launch_types[name]["matrices_per_launch"] = statistics.mean(chunks) if chunks else len(sub)
    agg = {}
    for name, e in launch_types.items():            # GEMM families: sum over buckets
        a = agg.setdefault(name.split("[")[0], {"ms": 0.0, "launches": 0.0, "work": 0.0})
        a["ms"] += e["ms_per_step"]
        a["launches"] += e["launches_per_step"]
        a["work"] += e.get("work_per_step", 0.0)
    for fam, a in agg.items():
        ach = a["work"] / (a["ms"] * 1e-3) / 1e12 if a["ms"] > 0 else 0.0
        kernels[fam] = {"launches_per_step": a["launches"], "ms_per_step": a["ms"], "share": a["ms"] / ms, "bound": "tensor",
                        "achieved": ach, "unit": "TFLOP/s", "frac": ach / peaks["tflops_sustained"]}
    dom = max(launch_types, key=lambda k: launch_types[k]["ms_per_step"], default=None)
    return kernels, launch_types, dom


# ------------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            f = tempfile.NamedTemporaryFile("w", suffix=".csv", delete=False)
            self.path = f.name
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=f, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if not self.proc:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        rows = []
        for line in open(self.path):
            parts = [p.strip() for p in line.split(",")]
            if len(parts) >= 9:
                try:
                    rows.append((float(parts[1]), float(parts[2]), float(parts[3]), parts[5], parts[6], parts[7], parts[8]))
                except ValueError:
                    pass
        os.unlink(self.path)
        if rows:
            pmax = max(r[2] for r in rows)
            load = [r for r in rows if r[2] >= 0.6 * pmax] or rows
            out["sm_mhz"] = statistics.median(r[0] for r in load)
            out["sm_max_mhz"] = rows[0][1]
            out["power_w_max"] = pmax
            out["samples"] = len(load)
            names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
            for k, name in enumerate(names):
                if any(r[3 + k].lower().startswith("active") for r in load):
                    out["reasons"].append(name)
        return out


# ------------------------------------------------------------------------------------------------ oracle arm
def _oracle_inputs(config: int, shapes, s):
    from paper_2606_27153_b200 import synth
    i = shapes.index(s)
    _, W, G, M = synth.muon_inputs(config, "cpu", False, indices=[i]) if config != 1 else (None, *([synth.ns_inputs("cpu")[1][:1]] * 3))
    return tuple(t[0].to(torch.float64).numpy() for t in (W, G, M))


def oracle_shape_seconds(config: int, s, shapes) -> tuple:
    """Seconds of one full oracle Muon step (NS_STEPS steps) of one matrix of shape s, and how they were obtained.
    Shapes whose full step fits ~3 s are timed whole.  Larger ones are timed at steps = 1 and steps = 0 and
    EXTRAPOLATED: t(0) + NS_STEPS * (t(1) - t(0)); the oracle's NS steps are the same plain loops at every step."""
    import oracle
    w, g, m = _oracle_inputs(config, shapes, s)
    if dense_flops([s]) / 4.5e10 <= 3.0:            # ~45 GFLOP/s plain loops on 16 cores
        t0 = time.perf_counter()
        oracle.muon_step(w, g, m, LR, MU, WD)
        return time.perf_counter() - t0, "whole"
    t0 = time.perf_counter()
    oracle.muon_step(w, g, m, LR, MU, WD, steps=0)
    t1 = time.perf_counter()
    oracle.muon_step(w, g, m, LR, MU, WD, steps=1)
    t2 = time.perf_counter()
    e0, e1 = t1 - t0, t2 - t1
    return e0 + NS_STEPS * (e1 - e0), "extrapolated from steps=0 and steps=1"


def oracle_sample(config: int, per_shape: dict = None):
    """Time the fp64 oracle, as it stands, on a bounded sample of the workload: one matrix of EVERY distinct shape (SURVEY
    8(d)), scaled by the shape counts.  With per_shape (seconds per shape from an earlier call) only the smallest shape
    is timed again and the others keep their seconds: the reference arm's repeated steps stay bounded.
    Returns (dense TFLOP/s of the whole config, description, cores, seconds spent, per_shape)."""
    import oracle
    from paper_2606_27153_b200 import synth
    shapes = synth.config_shapes(config)
    distinct = sorted(set(shapes), key=lambda s: dense_flops([s]))
    oracle.ns(torch.zeros(8, 8).double().numpy())          # build + load outside the timed region
    t_start = time.perf_counter()
    fresh = per_shape is None
    per_shape = {} if fresh else dict(per_shape)
    how = {}
    for s in (distinct if fresh else distinct[:1]):
        per_shape[s], how[s] = oracle_shape_seconds(config, s, shapes)
    spent = time.perf_counter() - t_start
    total = sum(per_shape[s] * shapes.count(s) for s in distinct)
    parts = ", ".join(f"{s[0]}x{s[1]} x{shapes.count(s)}: {per_shape[s]:.1f} s" + (f" ({how[s]})" if s in how else " (kept from the first step)")
                      for s in distinct)
    desc = (f"EXTRAPOLATED to {WORKLOADS[config].split(':')[0]}: one full Muon step ({NS_STEPS} NS steps, fp64, dense) of ONE matrix "
            f"of every distinct shape, times the shape counts [{parts}]")
    return dense_flops(shapes) / total / 1e12, desc, oracle.num_threads(), spent, per_shape


def run_reference(args):
    """--impl reference: the oracle on the host cores.  The first step times one matrix of every distinct shape; every
    later step re-times the smallest shape and keeps the others, so that K + W steps stay within a few minutes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    vals, secs, desc, cores, per_shape = [], [], "", 0, None
    for it in range(args.warmup + args.steps):
        v, desc, cores, s, per_shape = oracle_sample(args.config, per_shape)
        if it >= args.warmup:
            vals.append(v)
            secs.append(s)
    value = statistics.mean(vals)
    shapes = __import__("paper_2606_27153_b200.synth", fromlist=["config_shapes"]).config_shapes(args.config)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dense_flops(shapes) / (value * 1e12), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.config], "ns_steps": NS_STEPS, "coeffs": [3.4445, -4.7750, 2.0315], "lr": LR,
                   "mu": MU, "wd": WD, "note": "ms_per_step extrapolated from the sample by shape counts"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc,
                         "seconds_per_sample": statistics.mean(secs)},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------ our arm
def reduce_max(x: float, dist, device) -> float:
    """Max over ranks of a per-rank device time (the path does not shard: N replicas, the slowest one counts)."""
    if not dist:
        return x
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.item()


def whole_job_value(world: int, flops_per_replica: float, ms: float) -> float:
    """TFLOP/s of the whole job: every rank ran one replica of the step in `ms` (max over ranks)."""
    return world * flops_per_replica / (ms * 1e-3) / 1e12


def run_ours(args):
    import paper_2606_27153_b200 as dm
    from paper_2606_27153_b200 import synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a B200: the Muon step has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist_mod.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist = dist_mod

    def barrier():
        if dist:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x: float) -> float:
        return reduce_max(x, dist, "cuda")

    cfg = args.config
    shapes = synth.config_shapes(cfg)
    indices = None
    if args.layers > 0 and cfg != 1:          # profiling aid: the first L layers of the set (NOT a bench line)
        per_layer = {2: 6, 3: 7, 4: 7}[cfg]
        indices = list(range(min(len(shapes), per_layer * args.layers)))
        shapes = shapes[:len(indices)]
    peaks = load_peaks()
    dm.set_option("mode", "tc")
    dm.set_option("steps", NS_STEPS)
    dm.set_option("profile", 0)
    dm.set_option("keep_ns_output", 0)
    dm.set_option("fuse_epilogue", args.fuse)
    dm.set_option("program", args.program)
    if cfg == 1:
        _, W = synth.ns_inputs("cuda")
        G = M = None
    else:
        _, W, G, M = synth.muon_inputs(cfg, "cuda", False, indices=indices)
    stream = torch.cuda.current_stream()

    def step():
        if cfg == 1:
            dm.ns_batched(W, steps=NS_STEPS)
        else:
            dm.muon_step(W, G, M, LR, MU, WD)

    torch.cuda.synchronize()
    t_plan = time.perf_counter()
    step()                                    # first call: plan + workspace + autotune (reported, not timed)
    torch.cuda.synchronize()
    plan_s = time.perf_counter() - t_plan
    for _ in range(max(0, args.warmup - 1)):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    dm.profile_reset()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.nvtx.range_push("dmuon_timed")     # lets `ncu --nvtx --nvtx-include dmuon_timed/` profile timed launches only
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    torch.cuda.nvtx.range_pop()
    barrier()
    ms = max_over_ranks(e0.elapsed_time(e1)) / args.steps
    gpu_launches = dm.profile_read()["launches"]
    clocks = sampler.stop() if rank == 0 else {}

    plan_desc = dm.describe_plan(shapes, NS_STEPS)
    dflops, xflops = dense_flops(shapes), executed_flops(shapes, plan_desc)
    value = whole_job_value(world, dflops, ms)

    # ---- second pass of the same K steps with the library's events around every launch: per-kernel rooflines.  The
    #      library names GEMM launches family[rows x cols] per shape bucket; `kernels` aggregates per family,
    #      `launch_types` keeps the buckets apart, and `roofline` is the launch type that takes the most time.
    dm.set_option("profile", 1)
    step()
    dm.profile_reset()
    e0.record(stream)
    for _ in range(args.steps):
        step()
    e1.record(stream)
    torch.cuda.synchronize()
    ms_prof = e0.elapsed_time(e1) / args.steps
    prof = dm.profile_read()
    dm.set_option("profile", 0)
    kernels, launch_types, dom = profile_breakdown(prof, args.steps, ms_prof, shapes, plan_desc, peaks)
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    if dom and os.path.exists(tpath):
        for row in open(tpath).read().splitlines()[1:]:
            c, lt, nbytes = row.split(",")          # launch-type names hold no comma
            if c == f"config{cfg}" and lt == dom:
                traffic = int(nbytes)
    roofline = None
    if dom:
        k = launch_types[dom]
        roofline = {"kernel": dom, "bound": "tensor", "achieved": k["achieved"], "peak": peaks["tflops_sustained"],
                    "unit": "TFLOP/s", "frac": k["frac"], "traffic": traffic,
                    "launches_per_step": k["launches_per_step"], "matrices_per_launch": k["matrices_per_launch"],
                    "peak_kind": f"{peaks['source']} bf16 cuBLAS 8192^3, sustained (kernel timed inside a long step); "
                                 f"burst {peaks['tflops_burst']}, nominal 2250; cuBLAS fp16 on THIS kernel's shape and "
                                 f"operand bits: profiles/r2_energy_per_flop.md",
                    "flops_counted": "algorithmic FLOPs per launch: 2 m^2 n per matrix for an X update (dense, no "
                                     "symmetry); (T+1)/(2T) of 2 m^2 n or 2 m^3 per matrix for the symmetric products "
                                     "(upper-triangular 128-blocks; the mirror is not arithmetic)",
                    "traffic_unit": "bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum of one launch of this "
                                    "type in the full-size step; profiles/roofline_traffic.md)"}

    # ---- the HBM-bound kernels timed without the GEMM phase around them (steps = 0: momentum, norms, normalise, apply
    #      run back to back at the clocks a memory-bound phase gets); the in-step figures above inherit the ~1 GHz SM
    #      clock of the power-capped GEMM phase.  (With steps > 0 the apply pass does not exist: it is the last X
    #      update's epilogue.)
    hbm_alone = None
    if cfg != 1:
        dm.set_option("steps", 0)
        dm.set_option("profile", 1)
        for _ in range(2):
            step()
        torch.cuda.synchronize()
        dm.profile_reset()
        n_alone = 3
        for _ in range(n_alone):
            step()
        torch.cuda.synchronize()
        pa = dm.profile_read()["kernels"]
        dm.set_option("steps", NS_STEPS)
        dm.set_option("profile", 0)
        hbm_alone = {}
        for name in ("momentum_nesterov_sumsq", "normalize_cast", "apply_update"):
            if name in pa and pa[name]["ms"] > 0:
                gbs = family_work(name, shapes, plan_desc)[1] / (pa[name]["ms"] / n_alone * 1e-3) / 1e9
                hbm_alone[name] = {"ms": pa[name]["ms"] / n_alone, "achieved": gbs, "unit": "GB/s", "peak": peaks["hbm_gbs"],
                                   "frac": gbs / peaks["hbm_gbs"]}

    # ---- end to end through the C ABI with HOST buffers (copies inside the timed region)
    e2e = None
    if cfg != 1 and not args.no_e2e:
        try:
            pinned = True
            host = []
            for ts in (W, G, M):
                hs = []
                for t in ts:
                    try:
                        h = torch.empty(t.shape, dtype=t.dtype, pin_memory=pinned)
                    except RuntimeError:
                        pinned = False
                        h = torch.empty(t.shape, dtype=t.dtype)
                    h.copy_(t)
                    hs.append(h)
                host.append(hs)
            Wh, Gh, Mh = host
            del W, G, M
            torch.cuda.empty_cache()
            n_e2e = max(1, min(args.steps, 3))
            dm.muon_step_host(Wh, Gh, Mh, LR, MU, WD)         # warm-up: allocates the staging buffers
            barrier()
            e0.record(stream)
            for _ in range(n_e2e):
                dm.muon_step_host(Wh, Gh, Mh, LR, MU, WD)
            e1.record(stream)
            barrier()
            ms_e2e = max_over_ranks(e0.elapsed_time(e1)) / n_e2e
            elb = 2 * sum(r * c for r, c in shapes)
            e2e = {"value": world * dflops / (ms_e2e * 1e-3) / 1e12, "unit": UNIT, "ms_per_step": ms_e2e,
                   "h2d_bytes_per_step": 3 * elb, "d2h_bytes_per_step": 2 * elb, "steps": n_e2e,
                   "host_memory": "pinned" if pinned else "pageable", "api": "dmuon_muon_step_host"}
        except Exception as ex:  # an e2e failure must not hide the device-resident number
            e2e = {"value": None, "unit": UNIT, "error": str(ex)[:200]}

    cpu_baseline = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        v, desc, cores, secs, _ = oracle_sample(cfg)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "seconds": secs}

    if rank == 0:
        xt = xflops / (ms * 1e-3) / 1e12
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f16",
            "data": "synthetic",
            "config": {"workload": WORKLOADS[cfg] + (f" -- REDUCED to the first {args.layers} layers (profiling run, not a bench value)" if indices is not None else ""), "ns_steps": NS_STEPS, "coeffs": [3.4445, -4.7750, 2.0315], "lr": LR,
                       "mu": MU, "wd": WD, "schedule": plan_desc["buckets"], "workspace_bytes": plan_desc.get("workspace_bytes"),
                       "fused_epilogue": bool(args.fuse), "program_kernel": args.program, "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": "inputs (W, G, M + workspace, tens of GB) exceed the 126 MB L2; no flush needed",
                       "arithmetic": "bf16 in/out, fp16 operands on tcgen05 with fp32 TMEM accumulation, fp32 elementwise"},
            "muon_step_ms": ms, "ns_tflops_dense_equiv": value / world, "ns_tflops_executed": xt,
            "pct_of_bf16_peak": {"executed_of_measured_sustained": 100 * xt / peaks["tflops_sustained"],
                                 "executed_of_measured_burst": 100 * xt / peaks["tflops_burst"],
                                 "executed_of_nominal_2250": 100 * xt / 2250.0},
            "algorithmic_speed_vs_dense_at_peak": {
                "note": "dense-equivalent TFLOP/s (the metric's count) over a peak: NOT a hardware utilisation -- symmetry and "
                        "Gram blocks execute fewer FLOPs than the dense count",
                "vs_measured_sustained": value / world / peaks["tflops_sustained"],
                "vs_nominal_2250": value / world / 2250.0},
            "roofline": roofline, "kernels": kernels, "launch_types": launch_types, "profiled_pass_ms_per_step": ms_prof,
            "hbm_kernels_alone": hbm_alone, "cpu_baseline": cpu_baseline, "e2e": e2e,
            "gpu_launches": gpu_launches, "clocks": clocks, "plan_autotune_seconds": plan_s,
            "tune_seconds": plan_desc.get("tune_seconds"),
            "paper_context": "DMuon reports 6.85x-163x optimizer-step and 1.48x-3.01x end-to-end speedups on 8-256 A800 "
                             "(PAPER.md:5, :274) and ~2x on one GPU (:329): other hardware, context only",
            # last on purpose (a reader of the line's tail sees it): fraction of the measured HBM peak of the elementwise
            # passes as they run INSIDE the step, and of the tensor peak of the dominant launch type
            "in_step_frac": {k: round(v["frac"], 4) for k, v in kernels.items()
                             if v.get("frac") is not None and (v.get("bound") == "hbm" or k == "ns_program_apply")},
        }
        print(json.dumps(line))
    if dist:
        dist.destroy_process_group()


def run_sweep(args):
    """BASELINE.json configs[4]: the NS kernel alone (dmuon_ns_batched, 5 steps) over a shape sweep, one JSON line per
    shape with dense-equivalent and executed TFLOP/s and the roofline fraction of the executed rate.  Batches are the
    config's own (squares: 2^32 / n^2 matrices, i.e. 8 GiB of bf16 per shape); the library runs a bucket that needs
    more than its workspace cap ("chunk_mb", 12 GiB) as chunks of fewer matrices.  The MoE expert set is ONE call of
    128 matrices.  Not the bench line: a per-shape table for profiles/."""
    import paper_2606_27153_b200 as dm
    from paper_2606_27153_b200 import synth
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --sweep needs a B200")
    torch.cuda.set_device(0)
    peaks = load_peaks()
    dm.set_option("mode", "tc")
    dm.set_option("keep_ns_output", 0)
    points = [([s], b) for s, b in synth.sweep_shapes() if s not in ((2048, 1408), (1408, 2048))]
    points.append(([(2048, 1408), (1408, 2048)], 64))          # the MoE expert batch: 64 + 64 in one call
    for shape_list, batch in points:
        shapes, Xs, keep = [], [], []
        for r, c in shape_list:
            g = torch.Generator(device="cuda")
            g.manual_seed(5000 + r + c)
            big = torch.empty((batch, r, c), device="cuda", dtype=torch.bfloat16)
            per = max(1, (1 << 28) // (r * c))                  # fill 256 Mi elements at a time (fp32 staging)
            for b0 in range(0, batch, per):
                nb = min(per, batch - b0)
                big[b0:b0 + nb] = torch.randn((nb, r, c), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16)
            keep.append(big)
            Xs += [big[i] for i in range(batch)]
            shapes += [(r, c)] * batch
        Xs = dm.binding.marshal(Xs)            # pointer / shape arrays built once: for 65 536 matrices that is 60 ms of host time
        t0 = time.perf_counter()
        dm.ns_batched(Xs, steps=NS_STEPS)      # plan + autotune
        torch.cuda.synchronize()
        plan_s = time.perf_counter() - t0
        plan = dm.describe_plan(shapes, NS_STEPS)
        reps = 3
        for _ in range(2):
            dm.ns_batched(Xs, steps=NS_STEPS)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(reps):
            dm.ns_batched(Xs, steps=NS_STEPS)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        xt = executed_flops(shapes, plan) / ms / 1e9
        print(json.dumps({"sweep": True, "shapes": [list(s) for s in shape_list], "batch_per_shape": batch, "matrices": Xs.count, "ms": ms,
                          "tflops_dense_equiv": dense_flops(shapes) / ms / 1e9, "tflops_executed": xt,
                          "roofline_frac_executed_of_sustained": xt / peaks["tflops_sustained"],
                          "buckets": plan["buckets"], "workspace_bytes": plan["workspace_bytes"],
                          "plan_seconds": plan_s, "includes": "norm + normalise + 5 NS steps (bf16 store in the last epilogue)"}), flush=True)
        del Xs, keep, big
        dm.shutdown()
        torch.cuda.empty_cache()
    # PAPER.md:188 (Fig. 7): per-matrix NS time against the number of same-shape matrices advanced together
    for (r, c) in ((1024, 1024), (2048, 22016)):
        base = None
        for b in (1, 2, 4, 8, 16, 32):
            g = torch.Generator(device="cuda")
            g.manual_seed(5100 + b)
            big = torch.randn((b, r, c), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16)
            Xs = [big[i] for i in range(b)]
            for _ in range(3):
                dm.ns_batched(Xs, steps=NS_STEPS)
            reps = 20 if r == 1024 else 5
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(reps):
                dm.ns_batched(Xs, steps=NS_STEPS)
            e1.record()
            torch.cuda.synchronize()
            per = e0.elapsed_time(e1) / reps / b
            base = base or per
            print(json.dumps({"sweep": "batching", "shape": [r, c], "batch": b, "ms_per_matrix": per,
                              "speedup_vs_batch1": base / per}), flush=True)
            del Xs, big
            dm.shutdown()
            torch.cuda.empty_cache()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--layers", type=int, default=0, help="profiling aid: only the first L layers of the set (0 = all)")
    ap.add_argument("--sample-seconds", type=float, default=0.0, help="--impl reference: CPU seconds per step (0 = auto)")
    ap.add_argument("--fuse", type=int, default=1, choices=[0, 1], help="library option 'fuse_epilogue' (0: separate apply pass)")
    ap.add_argument("--program", default="auto", choices=["auto", "0", "1"],
                    help="library option 'program' (one launch per bucket's NS program: auto = small side >= 2048; 0: one launch per product)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="configs[4]: NS-only shape sweep, one JSON line per shape")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and not args.sweep:
        # `python bench.py --gpus N` without a launcher: start N ranks (one replica per GPU) the way the driver does
        import socket
        import subprocess
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr",
               "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))
    if args.sweep:
        run_sweep(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
