"""Host logic of bench.py that does not need a GPU: FLOP accounting against the block schedule, the N > 1
aggregation (world_size-2 gloo), and the reference arm's rank-0-only behaviour under torchrun."""
import json
import os
import subprocess
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import bench  # noqa: E402
from paper_2606_27153_b200 import synth  # noqa: E402


def test_dense_flops_match_survey_table():
    # cfg2 1.631, cfg3 7.192, cfg4 665.9 TFLOP dense; per matrix 4096x14336: 5497.6 GFLOP
    for cfg, want in ((2, 1.631), (3, 7.192), (4, 665.9)):
        assert abs(bench.dense_flops(synth.config_shapes(cfg)) / 1e12 - want) / want < 2e-3
    assert abs(bench.dense_flops([(14336, 4096)]) / 1e9 - 5497.6) < 1.0


def test_executed_flops_follow_the_block_schedule():
    m, n = 4096, 14336
    plain = {"buckets": [{"m": m, "n": n, "kind": "wide", "count": 1, "blocks": [1, 1, 1, 1, 1]},
                         {"m": m, "n": n, "kind": "tall", "count": 1, "blocks": [1, 1, 1, 1, 1]}]}
    blocks = {"buckets": [{"m": m, "n": n, "kind": "wide", "count": 1, "blocks": [3, 2]},
                          {"m": m, "n": n, "kind": "tall", "count": 1, "blocks": [3, 2]}]}
    sym = 33 / 64                                    # T = 32 blocks: (T + 1) / (2 T)
    want_plain = 5 * (sym * (2 * m * m * n + 2 * m ** 3) + 2 * m * m * n)
    want_blocks = 2 * sym * 2 * m * m * n + 14 * sym * 2 * m ** 3 + 2 * 2 * m * m * n
    assert bench.executed_flops([(m, n)], plain) == pytest.approx(want_plain)
    assert bench.executed_flops([(n, m)], blocks) == pytest.approx(want_blocks)     # tall: same oriented shape
    assert bench.family_work("ns_bx_update", [(m, n)], blocks) == ("flop", 2 * 2 * m * m * n)
    assert bench.family_work("ns_xb_apply", [(n, m)], blocks, 0.5) == ("flop", 2 * m * m * n)     # the fused one of two X updates
    assert bench.family_work("ns_gram_mm", [(m, n)], blocks)[1] == pytest.approx(9 * sym * 2 * m ** 3)
    assert bench.family_work("ns_sq_poly", [(n, m)], blocks)[1] == pytest.approx(5 * sym * 2 * m ** 3)
    assert bench.family_work("momentum_nesterov_sumsq", [(m, n)], blocks) == ("byte", 8 * m * n)
    assert bench.family_work("normalize_cast", [(m, n)], blocks) == ("byte", 4 * m * n)
    fams = ("ns_syrk_xxt", "ns_sq_poly", "ns_gram_mm", "ns_bx_update")
    assert sum(bench.family_work(f, [(m, n)], blocks)[1] for f in fams) == pytest.approx(want_blocks)


def test_profile_breakdown_maps_launch_types_to_buckets():
    """bench.profile_breakdown on a synthetic profile of config 4's buckets: tall buckets are named by the stored shape
    (rows x cols), chunks of one bucket accumulate under one name, plain and fused X updates share the bucket's work."""
    shapes = synth.config_shapes(4)
    plan = {"buckets": [{"m": 4096, "n": 14336, "kind": "tall", "count": 32, "blocks": [3, 2]},
                        {"m": 4096, "n": 14336, "kind": "tall", "count": 32, "blocks": [3, 2]},
                        {"m": 4096, "n": 14336, "kind": "wide", "count": 32, "blocks": [3, 2]},
                        {"m": 4096, "n": 4096, "kind": "wide", "count": 64, "blocks": [1] * 5},
                        {"m": 1024, "n": 4096, "kind": "wide", "count": 64, "blocks": [3, 2]}]}
    assert bench.bucket_key((14336, 4096)) == (4096, 14336, "tall") and bench.bucket_key((100, 260)) == (128, 384, "generic")
    assert len(bench.shapes_of_launch_type("ns_xb_update[14336x4096]", shapes)) == 64
    assert len(bench.shapes_of_launch_type("ns_bx_update[4096x14336]", shapes)) == 32
    assert len(bench.shapes_of_launch_type("ns_sq_poly[4096x4096]", shapes)) == 64
    prof = {"kernels": {"ns_xb_update[14336x4096]": {"launches": 2, "ms": 30.0}, "ns_xb_apply[14336x4096]": {"launches": 2, "ms": 31.0},
                        "ns_bx_update[4096x4096]": {"launches": 4, "ms": 32.0}, "ns_bx_apply[4096x4096]": {"launches": 1, "ms": 8.5},
                        "momentum_nesterov_sumsq": {"launches": 5, "ms": 10.0}}}
    peaks = {"hbm_gbs": 6500.0, "tflops_burst": 1600.0, "tflops_sustained": 1400.0}
    kernels, lt, dom = bench.profile_breakdown(prof, 1, 300.0, shapes, plan, peaks)
    one = 64 * 2 * 4096 * 4096 * 14336                # one X update of the 64 tall matrices
    assert lt["ns_xb_update[14336x4096]"]["work_per_step"] == pytest.approx(one)
    assert lt["ns_xb_apply[14336x4096]"]["work_per_step"] == pytest.approx(one)
    assert lt["ns_xb_update[14336x4096]"]["matrices_per_launch"] == 32
    assert lt["ns_bx_update[4096x4096]"]["work_per_step"] == pytest.approx(4 * 64 * 2 * 4096 ** 3)
    assert lt["ns_bx_apply[4096x4096]"]["achieved"] == pytest.approx(64 * 2 * 4096 ** 3 / 8.5e-3 / 1e12)
    assert dom == "ns_bx_update[4096x4096]"
    assert kernels["momentum_nesterov_sumsq"]["achieved"] == pytest.approx(8 * sum(r * c for r, c in shapes) / 10e-3 / 1e9)
    assert kernels["ns_xb_update"]["ms_per_step"] == 30.0


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.reduce_max(100.0 + 7.0 * rank, dist, "cpu")          # the slowest replica counts
    val = bench.whole_job_value(world, 1e12, ms)
    dist.barrier()
    dist.destroy_process_group()
    out.put((rank, ms, val))


def test_two_rank_aggregation_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 400
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for _, ms, val in res:
        assert ms == 107.0
        assert val == pytest.approx(2 * 1e12 / 0.107 / 1e12)
    assert bench.reduce_max(5.0, None, "cpu") == 5.0


def test_reference_arm_rank0_only_under_torchrun():
    """`bench.py --impl reference` under torchrun with 2 ranks: rank 0 prints one JSON line, rank 1 exits 0 silently."""
    port = 29900 + os.getpid() % 90
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--config", "1", "--sample-seconds", "0.5"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = lines[0]
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0


def test_gpus_flag_launches_the_ranks_itself():
    """`python bench.py --gpus 2` with no launcher (WORLD_SIZE unset) starts 2 ranks under torch.distributed.run."""
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    cmd = [sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "2", "--warmup", "1",
           "--config", "1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, cwd=ROOT, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1 and lines[0]["n_gpus"] == 2 and lines[0]["impl"] == "reference"


def test_cpu_baseline_covers_every_distinct_shape():
    """the oracle sample is one matrix of EVERY distinct shape scaled by the counts; a later step re-times
    only the smallest shape and keeps the rest."""
    import bench
    from paper_2606_27153_b200 import synth
    v, desc, cores, secs, per_shape = bench.oracle_sample(2)
    assert set(per_shape) == set(synth.config_shapes(2)) and all(t > 0 for t in per_shape.values())
    assert v > 0 and cores >= 1 and "EXTRAPOLATED" in desc and "768x768 x48" in desc and "3072x768 x12" in desc
    v2, desc2, _, secs2, per2 = bench.oracle_sample(2, per_shape)
    big = [s for s in per_shape if s != (768, 768)]
    assert all(per2[s] == per_shape[s] for s in big) and "kept from the first step" in desc2 and v2 > 0
