"""GPU tests of the SURVEY 8(f) rows beyond the Muon step itself: the AdamW entry point for non-matrix parameters
 against the fp64 oracle, the measured cost model c_{s,b} + owner assignment, and the
autotuner's persistent cache ("subsequent invocations ... bypass the search entirely")."""
import os

import numpy as np
import pytest
import torch

import oracle
import paper_2606_27153_b200 as dm
from helpers import bf16_ulp, to64

pytestmark = pytest.mark.gpu


def test_adamw_matches_oracle():
    """Three AdamW steps over tensors of ragged sizes (vector path + scalar tails), compared step by step with the fp64
    oracle restarted from the GPU's state: moments to fp32 rounding, the bf16 parameter within one ulp of RNE(fp64)."""
    sizes = [(1000,), (3, 8192), (5,), (896,), (257, 33)]
    g = torch.Generator(device="cuda").manual_seed(9100)
    P = [(torch.randn(s, generator=g, device="cuda") * 0.5).to(torch.bfloat16) for s in sizes]
    M = [torch.randn(s, generator=g, device="cuda") * 1e-2 for s in sizes]
    V = [torch.rand(s, generator=g, device="cuda") * 1e-4 for s in sizes]
    lr, b1, b2, eps, wd = 3e-3, 0.9, 0.95, 1e-8, 0.1
    f32 = lambda v: float(np.float32(v))
    worst_share = 0.0
    for step in range(1, 4):
        G = [(torch.randn(s, generator=g, device="cuda") * (10.0 ** -step)).to(torch.bfloat16) for s in sizes]
        p0, m0, v0 = [to64(t) for t in P], [to64(t) for t in M], [to64(t) for t in V]
        G0 = [t.clone() for t in G]
        dm.adamw_step(P, G, M, V, lr, b1, b2, eps, wd, step)
        torch.cuda.synchronize()
        for i in range(len(sizes)):
            pn, mn, vn = oracle.adamw_step(p0[i], to64(G[i]), m0[i], v0[i], f32(lr), f32(b1), f32(b2), f32(eps), f32(wd), step)
            # fp32 arithmetic: a few 2^-24 of the TERMS of each moment update (the terms can cancel)
            g64 = to64(G[i])
            assert (np.abs(to64(M[i]) - mn) <= 3e-7 * (np.abs(b1 * m0[i]) + np.abs((1 - b1) * g64)) + 1e-37).all(), f"step {step} tensor {i}: exp_avg"
            assert (np.abs(to64(V[i]) - vn) <= 3e-7 * (np.abs(b2 * v0[i]) + np.abs((1 - b2) * g64 * g64)) + 1e-37).all(), f"step {step} tensor {i}: exp_avg_sq"
            want = oracle.round_bf16(pn)
            d = np.abs(to64(P[i]) - want)
            assert (d <= bf16_ulp(np.maximum(np.abs(want), np.abs(to64(P[i]))))).all(), f"step {step} tensor {i}: parameter off by more than 1 bf16 ulp"
            worst_share = max(worst_share, float((d != 0).mean()))
            assert torch.equal(G[i], G0[i]), "grads must never be written"
    assert worst_share < 0.02
    print(f"adamw: share of parameters differing from RNE(fp64) (all within 1 ulp): max {worst_share:.2e}")
    # zero gradient and zero moments: pure decay, no NaN from 0 / (0 + eps)
    p = torch.full((4096,), 0.5, dtype=torch.bfloat16, device="cuda")
    z = torch.zeros(4096, dtype=torch.bfloat16, device="cuda")
    m, v = torch.zeros(4096, device="cuda"), torch.zeros(4096, device="cuda")
    dm.adamw_step([p], [z], [m], [v], 0.1, 0.9, 0.999, 1e-8, 0.5, 1)
    torch.cuda.synchronize()
    assert torch.equal(p, torch.full_like(p, 0.5 * (1 - 0.05))) and m.abs().max().item() == 0 and v.abs().max().item() == 0


def test_measured_cost_model_and_assignment():
    """c_{s,b} measured through the whole Muon step for two shapes and batch sizes 1, 2, 4, then the
    owner assignment of 12 + 6 matrices on 4 ranks from those costs (Eq. 5)."""
    shapes = [(768, 768), (3072, 768)]
    batch_sizes = [[1, 2, 4], [1, 2]]
    costs = [[dm.measure_cost(s, b, reps=5) for b in bs] for s, bs in zip(shapes, batch_sizes)]
    for cs, bs in zip(costs, batch_sizes):
        assert all(c > 0 for c in cs)
        per = [c / b for c, b in zip(cs, bs)]
        assert per[-1] <= 1.15 * per[0], f"batching must not cost more per matrix: {per}"      # PAPER.md:188 Fig. 7
    counts = [12, 6]
    x, ms, exact = dm.assign_owners(counts, batch_sizes, costs, 4, mode=-1, threshold=64)
    total_best = sum(n * min(c / b for c, b in zip(cs, bs)) for n, cs, bs in zip(counts, costs, batch_sizes))
    assert total_best / 4 - 1e-9 <= ms <= 1.5 * total_best / 4
    for s in range(2):
        assert sum(b * sum(x[s][j]) for j, b in enumerate(batch_sizes[s])) == counts[s]
    print(f"c[s,b] (ms): {costs}; makespan on 4 ranks {ms:.3f} ms (exact={exact}), perfect split {total_best / 4:.3f} ms")


def test_tuning_cache_write_reload_same_plan(tmp_path):
    """Tune with a cache file, shut the library down, come back: the same tile configurations without any re-timing;
    an entry written by another build is ignored (the key carries the build id)."""
    path = str(tmp_path / "tune.txt")
    shapes = [(512, 1024)] * 4 + [(1024, 512)] * 3 + [(384, 384)] * 2
    dm.shutdown()
    dm.set_option("cache_path", path)
    dm.set_option("autotune", 1)
    dm.set_option("tune_ms", 3)
    try:
        first = dm.describe_plan(shapes, steps=5)
        assert first["tune_seconds"] > 0 and os.path.exists(path)
        lines = open(path).read().splitlines()
        assert len(lines) == 9 and all(l.startswith("v5 ") for l in lines)          # 3 bucket shapes x 3 products
        assert first["tune_cache_entries"] == 9
        dm.shutdown()                                                               # forgets plans AND the in-memory cache
        second = dm.describe_plan(shapes, steps=5)
        assert second["tune_seconds"] == 0, "cached choices must bypass the search (PAPER.md:184)"
        assert [b["variants"] for b in second["buckets"]] == [b["variants"] for b in first["buckets"]]
        # a cache written by another build: every line is ignored, the search runs again
        dm.shutdown()
        open(path, "w").write("\n".join(" ".join(["v5", "otherbuild"] + l.split()[2:]) for l in lines) + "\n")
        third = dm.describe_plan(shapes, steps=5)
        assert third["tune_seconds"] > 0
        # autotune off and no cache: the untuned default, no timing
        dm.shutdown()
        dm.set_option("cache_path", "")
        dm.set_option("autotune", 0)
        fourth = dm.describe_plan(shapes, steps=5)
        assert fourth["tune_seconds"] == 0 and all(b["variants"] == [4, 4, 4] for b in fourth["buckets"])
    finally:
        dm.shutdown()
        dm.set_option("autotune", 1)
        dm.set_option("tune_ms", 40)
        dm.set_option("cache_path", os.environ.get("DMUON_CACHE", os.path.expanduser("~/.cache/dmuon/tune.txt")))


def test_chunked_bucket_equals_unchunked():
    """A bucket over the workspace cap runs as chunks through one region: same bits as the unchunked run."""
    shapes = [(256, 512)] * 7 + [(512, 256)] * 5
    from paper_2606_27153_b200 import synth
    base = [synth.gradient(s, 9200 + i, "cuda") for i, s in enumerate(shapes)]
    dm.set_option("keep_ns_output", 0)
    res = []
    for mb in (12288, 1):                    # 1 MiB: a 256x512 matrix needs 0.5 + 5 x 0.125 = 1.1 MiB -> chunks of 1
        dm.set_option("chunk_mb", mb)
        Xs = [b.clone() for b in base]
        dm.ns_batched(Xs, steps=5)
        torch.cuda.synchronize()
        plan = dm.describe_plan(shapes, steps=5)
        res.append((Xs, plan))
    dm.set_option("chunk_mb", 12288)
    assert len(res[0][1]["buckets"]) == 2 and len(res[1][1]["buckets"]) == 12
    assert res[1][1]["workspace_bytes"] < res[0][1]["workspace_bytes"]
    assert all(torch.equal(a, b) for a, b in zip(res[0][0], res[1][0]))
