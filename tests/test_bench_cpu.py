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
    plain = {"buckets": [{"m": m, "n": n, "count": 1, "blocks": [1, 1, 1, 1, 1]}]}
    blocks = {"buckets": [{"m": m, "n": n, "count": 1, "blocks": [3, 2]}]}
    sym = 33 / 64                                    # T = 32 blocks: (T + 1) / (2 T)
    want_plain = 5 * (sym * (2 * m * m * n + 2 * m ** 3) + 2 * m * m * n)
    want_blocks = 2 * sym * 2 * m * m * n + 14 * sym * 2 * m ** 3 + 2 * 2 * m * m * n
    assert bench.executed_flops([(m, n)], plain) == pytest.approx(want_plain)
    assert bench.executed_flops([(n, m)], blocks) == pytest.approx(want_blocks)     # tall: same oriented shape
    w = bench.kernel_work([(m, n)], blocks)
    assert w["ns_bx_update"] == ("flop", 2 * 2 * m * m * n)
    assert w["ns_gram_mm"][1] == pytest.approx(9 * sym * 2 * m ** 3)
    assert w["ns_sq_poly"][1] == pytest.approx(5 * sym * 2 * m ** 3)
    assert w["momentum_nesterov_sumsq"] == ("byte", 8 * m * n)
    total = sum(v[1] for v in w.values() if v[0] == "flop")
    assert total == pytest.approx(want_blocks)


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
