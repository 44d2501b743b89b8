#!/usr/bin/env python
"""bench.py -- the Muon optimizer step of DMuon (arxiv/paper_2606_27153) on B200, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one pass of the whole hot path (momentum+Nesterov+cast+norm, 5 Newton-Schulz steps of three grouped
GEMMs per shape bucket, apply) over one synthetic matrix set.  Default workload: BASELINE.json configs[3], the
Llama-3-8B-shaped set (224 matrices, 6.98 G elements, bf16 W/G/M resident in HBM), the configuration the metric
is quoted on.  `value` = dense-equivalent NS TFLOP/s of the whole step (BASELINE.json: "counting the full dense
FLOPs") = sum over matrices of 5 (4 m^2 n + 2 m^3) divided by the step time, aggregated over ranks.
The path does not shard (north_star: one GPU, no collectives): --gpus N runs N independent replicas ("replicas
only"), timed as the max over ranks.
--impl reference times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
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


# ------------------------------------------------------------------------------------------------ accounting
def oriented(shape):
    r, c = shape
    return min(r, c), max(r, c)


def dense_flops(shapes, steps=NS_STEPS):
    """Metric FLOPs: 5 (4 m^2 n + 2 m^3) per matrix."""
    return sum(steps * (4 * m * m * n + 2 * m ** 3) for m, n in map(oriented, shapes))


def pad128(v):
    return -(-v // 128) * 128


def launch_counts(shapes, plan):
    """Per matrix (m, n, products): how many launches of each product family the library's block schedule
    (dmuon_describe_plan) runs.  A block of length L: 1 SYRK, L polynomial products, 3 (L - 1) Gram-space products
    (T = aG + BG, G' = aT + TB, R' = pB' + aR + B'R), 1 X update."""
    blocks = {(b["m"], b["n"]): b["blocks"] for b in plan["buckets"]}
    out = []
    for m, n in map(oriented, shapes):
        part = blocks[(pad128(m), pad128(n))]
        out.append((m, n, {"ns_syrk_xxt": len(part), "ns_sq_poly": sum(part), "ns_gram_mm": sum(3 * (L - 1) for L in part),
                           "ns_bx_update": len(part)}))
    return out


def executed_flops(shapes, plan):
    """FLOPs the kernels execute: every m x m result and X X^T is symmetric and only its upper-triangular 128-blocks
    are computed, a share (T+1)/(2T) of the dense product; X updates are dense."""
    tot = 0.0
    for m, n, cnt in launch_counts(shapes, plan):
        t = -(-m // 128)
        sym = (t + 1) / (2 * t)
        tot += sym * (cnt["ns_syrk_xxt"] * 2 * m * m * n + (cnt["ns_sq_poly"] + cnt["ns_gram_mm"]) * 2 * m ** 3)
        tot += cnt["ns_bx_update"] * 2 * m * m * n
    return tot


def kernel_work(shapes, plan):
    """Algorithmic work per step of each kernel family: FLOPs or bytes.  For the symmetric
    products the algorithmic FLOPs are those of the upper-triangular 128-blocks, (T+1)/(2T) of the dense 2 m^2 n or
    2 m^3 (the rest of the result is a mirror, not arithmetic); the X update is dense."""
    el = sum(r * c for r, c in shapes)
    lc = launch_counts(shapes, plan)
    sym = lambda m: (-(-m // 128) + 1) / (2 * -(-m // 128))
    return {
        "ns_syrk_xxt": ("flop", sum(c["ns_syrk_xxt"] * sym(m) * 2 * m * m * n for m, n, c in lc)),
        "ns_sq_poly": ("flop", sum(c["ns_sq_poly"] * sym(m) * 2 * m ** 3 for m, n, c in lc)),
        "ns_gram_mm": ("flop", sum(c["ns_gram_mm"] * sym(m) * 2 * m ** 3 for m, n, c in lc)),
        "ns_bx_update": ("flop", sum(c["ns_bx_update"] * 2 * m * m * n for m, n, c in lc)),
        "momentum_nesterov_sumsq": ("byte", 8 * el),       # read G, M; write M', U          (a1 + a2)
        "normalize_orient_cast": ("byte", 4 * el),         # read U; write X0
        "apply_update": ("byte", 6 * el),                  # read O, W; write W'             (a6)
    }


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        p = json.load(open(path))
        return {"hbm_gbs": p["hbm_gbs"], "tflops_burst": p["bf16_tflops"],
                "tflops_sustained": p.get("bf16_tflops_sustained", p["bf16_tflops"]), "source": "measured"}
    # fallback stated in /opt/skills/guides/B200_PROFILING.md
    return {"hbm_gbs": 6650.0, "tflops_burst": 1590.0, "tflops_sustained": 1400.0, "source": "fallback"}


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
def oracle_sample(config: int, max_seconds: float = 30.0):
    """Time the fp64 oracle, as it stands, on a bounded sample of the workload: whole Muon steps of single matrices,
    smallest distinct shapes first, until ~max_seconds are used.  Returns (dense TFLOP/s, description, cores, seconds)."""
    import oracle
    from paper_2606_27153_b200 import synth
    shapes = synth.config_shapes(config)
    distinct = sorted(set(shapes), key=lambda s: dense_flops([s]))
    oracle.ns(torch.zeros(8, 8).double().numpy())          # build + load outside the timed region
    done, flops, secs = [], 0.0, 0.0
    for s in distinct:
        est = dense_flops([s]) / 7e10                       # ~70 GFLOP/s plain loops on 16 cores: skip what cannot fit the budget
        if done and secs + est > max_seconds:
            break
        i = shapes.index(s)
        _, W, G, M = synth.muon_inputs(config, "cpu", False, indices=[i]) if config != 1 else (None, *([synth.ns_inputs("cpu")[1][:1]] * 3))
        w, g, m = (t[0].to(torch.float64).numpy() for t in (W, G, M))
        t0 = time.perf_counter()
        oracle.muon_step(w, g, m, LR, MU, WD)
        secs += time.perf_counter() - t0
        flops += dense_flops([s])
        done.append(f"{s[0]}x{s[1]}")
        if secs > max_seconds:
            break
    desc = f"one full Muon step (5 NS steps, fp64, dense) of one matrix each of shape {', '.join(done)} from {WORKLOADS[config].split(':')[0]}"
    return flops / secs / 1e12, desc, oracle.num_threads(), secs


def run_reference(args):
    """--impl reference: the oracle on the host cores; each step is one bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    budget = args.sample_seconds if args.sample_seconds > 0 else max(5.0, 60.0 / max(1, args.steps + args.warmup))
    vals, secs, desc, cores = [], [], "", 0
    for it in range(args.warmup + args.steps):
        v, desc, cores, s = oracle_sample(args.config, budget)
        if it >= args.warmup:
            vals.append(v)
            secs.append(s)
    value = statistics.mean(vals)
    shapes = __import__("paper_2606_27153_b200.synth", fromlist=["config_shapes"]).config_shapes(args.config)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dense_flops(shapes) / (value * 1e12), "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": WORKLOADS[args.config], "note": "ms_per_step extrapolated from the sample by FLOPs"},
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
    dm.set_option("profile", 1)
    if args.variants:
        dm.set_option("variants", args.variants)
    dm.set_option("overlap", args.overlap)
    t_setup = time.perf_counter()
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

    step()                                    # first call: plan + workspace + autotune (reported, not timed)
    torch.cuda.synchronize()
    plan_s = time.perf_counter() - t_setup
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
    prof = dm.profile_read()
    clocks = sampler.stop() if rank == 0 else {}

    plan_desc = dm.describe_plan(shapes, NS_STEPS)
    dflops, xflops = dense_flops(shapes), executed_flops(shapes, plan_desc)
    value = whole_job_value(world, dflops, ms)

    # per-kernel rooflines from the library's own CUDA events (recorded on the launching stream, in the timed region).
    # The library names GEMM launches family[m x n] per shape bucket; `kernels` aggregates per family, `launch_types`
    # keeps the buckets apart, and `roofline` is the launch type that takes the most time.
    work = kernel_work(shapes, plan_desc)

    def entry(ms_tot, launches, kind, amount):
        per_step_ms = ms_tot / args.steps
        e = {"launches_per_step": launches / args.steps, "ms_per_step": per_step_ms, "share": per_step_ms / ms}
        if kind and per_step_ms > 0:
            if kind == "flop":
                ach = amount / (per_step_ms * 1e-3) / 1e12
                e.update({"bound": "tensor", "achieved": ach, "unit": "TFLOP/s", "frac": ach / peaks["tflops_sustained"],
                          "frac_of_burst": ach / peaks["tflops_burst"], "frac_of_nominal_2250": ach / 2250.0})
            else:
                ach = amount / (per_step_ms * 1e-3) / 1e9
                e.update({"bound": "hbm", "achieved": ach, "unit": "GB/s", "frac": ach / peaks["hbm_gbs"]})
        return e

    fam = {}
    for name, rec in prof["kernels"].items():
        f = fam.setdefault(name.split("[")[0], {"ms": 0.0, "launches": 0})
        f["ms"] += rec["ms"]
        f["launches"] += rec["launches"]
    kernels = {f: entry(v["ms"], v["launches"], *work.get(f, (None, 0))) for f, v in fam.items()}
    launch_types = {}
    for name, rec in prof["kernels"].items():
        if "[" not in name:
            continue
        f, dims = name[:-1].split("[")
        bm, bn = (int(v) for v in dims.split("x"))
        sub = [sh for sh in shapes if (pad128(min(sh)), pad128(max(sh))) == (bm, bn)]
        launch_types[name] = entry(rec["ms"], rec["launches"], *kernel_work(sub, plan_desc)[f])
        launch_types[name]["matrices_per_launch"] = len(sub)
    dom = max(launch_types, key=lambda k: launch_types[k]["ms_per_step"], default=None)
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
                    "peak_kind": f"{peaks['source']} bf16 cuBLAS, sustained (kernel timed inside a long step); "
                                 f"burst {peaks['tflops_burst']}, nominal 2250",
                    "flops_counted": "algorithmic FLOPs per launch: 2 m^2 n per matrix for an X update (dense, no "
                                     "symmetry); (T+1)/(2T) of 2 m^2 n or 2 m^3 per matrix for the symmetric products "
                                     "(upper-triangular 128-blocks; the mirror is not arithmetic)",
                    "traffic_unit": "bytes per launch (dram__bytes_read.sum + dram__bytes_write.sum, ncu --set full; "
                                    "profiles/roofline_traffic.csv)"}

    # ---- the HBM-bound kernels timed without the GEMM phase around them (steps = 0: momentum, norms, normalise,
    #      apply run back to back at the clocks a memory-bound phase gets); the in-step figures above inherit the
    #      ~1 GHz SM clock of the power-capped GEMM phase
    hbm_alone = None
    if cfg != 1:
        dm.set_option("steps", 0)
        dm.set_option("overlap", 0)           # one stream: the passes are timed one after the other
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
        dm.set_option("overlap", args.overlap)
        hbm_alone = {}
        for name in ("momentum_nesterov_sumsq", "normalize_orient_cast", "apply_update"):
            if name in pa and pa[name]["ms"] > 0:
                gbs = work[name][1] / (pa[name]["ms"] / n_alone * 1e-3) / 1e9
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
        v, desc, cores, secs = oracle_sample(cfg, 32.0)
        cpu_baseline = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc, "seconds": secs}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f16",
            "data": "synthetic",
            "config": {"workload": WORKLOADS[cfg] + (f" -- REDUCED to the first {args.layers} layers (profiling run, not a bench value)" if indices is not None else ""), "ns_steps": NS_STEPS, "coeffs": [3.4445, -4.7750, 2.0315], "lr": LR,
                       "mu": MU, "wd": WD, "schedule": plan_desc["buckets"],
                       "overlap": bool(args.overlap), "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2": "inputs (W, G, M + workspace, tens of GB) exceed the 126 MB L2; no flush needed",
                       "arithmetic": "bf16 in/out, fp16 operands on tcgen05 with fp32 TMEM accumulation, fp32 elementwise"},
            "muon_step_ms": ms, "ns_tflops_dense_equiv": value / world, "ns_tflops_executed": xflops / (ms * 1e-3) / 1e12,
            "pct_of_bf16_peak": {"dense_equiv_of_measured_sustained": 100 * value / world / peaks["tflops_sustained"],
                                 "dense_equiv_of_measured_burst": 100 * value / world / peaks["tflops_burst"],
                                 "dense_equiv_of_nominal_2250": 100 * value / world / 2250.0,
                                 "executed_of_measured_sustained": 100 * xflops / (ms * 1e-3) / 1e12 / peaks["tflops_sustained"]},
            "roofline": roofline, "kernels": kernels, "launch_types": launch_types, "hbm_kernels_alone": hbm_alone, "cpu_baseline": cpu_baseline, "e2e": e2e,
            "gpu_launches": prof["launches"], "clocks": clocks, "plan_autotune_seconds": plan_s,
            "paper_context": "DMuon reports 6.85x-163x optimizer-step and 1.48x-3.01x end-to-end speedups on 8-256 A800 "
                             "(PAPER.md:5, :274) and ~2x on one GPU (:329): other hardware, context only",
        }
        print(json.dumps(line))
    if dist:
        dist.destroy_process_group()


def run_sweep(args):
    """BASELINE.json configs[4]: the NS kernel alone (dmuon_ns_batched, 5 steps) over a shape sweep, one JSON line per
    shape with dense-equivalent and executed TFLOP/s.  Not the bench line: a per-shape table for profiles/."""
    import paper_2606_27153_b200 as dm
    from paper_2606_27153_b200 import synth
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --sweep needs a B200")
    torch.cuda.set_device(0)
    dm.set_option("mode", "tc")
    cap = 16384                      # bounds plan-building time (TMA descriptors per matrix); said in the output
    for (r, c), batch in synth.sweep_shapes():
        b = min(batch, cap)
        g = torch.Generator(device="cuda")
        g.manual_seed(5000 + r + c)
        big = torch.randn((b, r, c), generator=g, device="cuda", dtype=torch.float32).to(torch.bfloat16)
        Xs = [big[i] for i in range(b)]
        shapes = [(r, c)] * b
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
        print(json.dumps({"sweep": True, "shape": [r, c], "batch": b, "batch_in_config": batch, "ms": ms,
                          "tflops_dense_equiv": dense_flops(shapes) / ms / 1e9,
                          "tflops_executed": executed_flops(shapes, plan) / ms / 1e9,
                          "blocks": plan["buckets"][0]["blocks"], "variants": plan["buckets"][0]["variants"],
                          "plan_seconds": plan_s, "includes": "norm + normalise + 5 NS steps + bf16 store"}), flush=True)
        del Xs, big
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


def run_power_probe(args):
    """Sustained throughput of the grouped X-update and SYRK kernels (dmuon_ns_gemm, CTA-pair tiling, 8 matrices of
    4096 x 14336) against operand bit patterns: random fp16, low mantissa bits cleared, constant, zeros.  Shows how
    much of the 1 kW cap is operand toggling.  One JSON line per (pattern, kernel)."""
    import paper_2606_27153_b200 as dm
    from paper_2606_27153_b200.binding import OP_BX, OP_SYRK
    torch.cuda.set_device(0)
    m, n, cnt = 4096, 14336, 8

    def clear_low(x, bits):
        return (x.view(torch.int16) & ~((1 << bits) - 1)).view(torch.float16)

    for kind in ("random", "low3_cleared", "low6_cleared", "constant", "zeros", "random"):
        g = torch.Generator(device="cuda")
        g.manual_seed(1)
        B = [(torch.randn((m, m), generator=g, device="cuda") * 0.02).half() for _ in range(cnt)]
        X = [(torch.randn((m, n), generator=g, device="cuda") * 1e-2).half() for _ in range(cnt)]
        if kind == "zeros":
            B, X = [torch.zeros_like(t) for t in B], [torch.zeros_like(t) for t in X]
        elif kind == "constant":
            B, X = [torch.full_like(t, 0.01) for t in B], [torch.full_like(t, 0.01) for t in X]
        elif kind.startswith("low"):
            k = int(kind[3])
            B, X = [clear_low(t, k) for t in B], [clear_low(t, k) for t in X]
        C = [torch.empty((m, n), device="cuda", dtype=torch.float16) for _ in range(cnt)]
        A = [torch.empty((m, m), device="cuda", dtype=torch.float16) for _ in range(cnt)]
        for op, name, reps in ((OP_BX, "ns_bx_update_pair", 80), (OP_SYRK, "ns_syrk_xxt_pair", 150)):
            call = (lambda: dm.ns_gemm(OP_BX, B, X, C, 1.0, 3.4445, variant=5)) if op == OP_BX else \
                   (lambda: dm.ns_gemm(OP_SYRK, X, None, A, 1.0, 0.0, variant=4))
            for _ in range(3):
                call()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(reps):
                call()
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / reps
            flops = cnt * 2 * m * m * n * (1.0 if op == OP_BX else 136 * 4 / 1024)   # SYRK: 136 of 256 pair units
            print(json.dumps({"probe": "power", "operands": kind, "kernel": name, "ms": ms, "seconds_timed": ms * reps / 1e3,
                              "tflops_executed": flops / ms / 1e9}), flush=True)
        del B, X, C, A


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--layers", type=int, default=0, help="profiling aid: only the first L layers of the set (0 = all)")
    ap.add_argument("--sample-seconds", type=float, default=0.0, help="--impl reference: CPU seconds per step (0 = auto)")
    ap.add_argument("--overlap", type=int, default=0, choices=[0, 1], help="library option 'overlap' (side-stream schedule)")
    ap.add_argument("--variants", default="", help="tuning aid: force tile configurations 'syrk,sq,bx' (-1 = tuned)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--power-probe", action="store_true", help="kernel throughput vs operand bit patterns (power cap)")
    ap.add_argument("--sweep", action="store_true", help="configs[4]: NS-only shape sweep, one JSON line per shape")
    args = ap.parse_args()
    if args.sweep:
        run_sweep(args)
    elif args.power_probe:
        run_power_probe(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
