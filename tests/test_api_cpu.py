"""CPU-side checks: the C-ABI library loads and exports every symbol include/dmuon.h declares, argument
validation and options behave as the header says, and the host logic (shape sets, workspace sizing) is right.
No compute call needs a GPU here."""
import ctypes
import os
import re

import pytest
import torch

import paper_2606_27153_b200 as dm
from paper_2606_27153_b200 import binding, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "dmuon.h")).read()
    return sorted(set(re.findall(r"DMUON_API\s+[\w\s\*]+?\b(dmuon_\w+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    names = declared_symbols()
    assert len(names) >= 15
    assert sorted(binding.SYMBOLS) == names, "binding.SYMBOLS must list exactly what the header declares"
    L = ctypes.CDLL(binding.LIB_PATH)
    for n in names:
        assert hasattr(L, n), f"{n} not exported by libdmuon.so"
    assert "sm_100a" in dm.version()


def test_options_validation():
    dm.set_option("steps", 5)
    dm.set_option("coeffs", "3.4445,-4.7750,2.0315")
    dm.set_option("autotune", "1")
    dm.set_option("profile", "0")
    dm.set_option("coeffs_sched", "3.9,-6,2.8;3.4445,-4.775,2.0315")
    dm.set_option("coeffs_sched", "")
    dm.set_option("fuse_epilogue", "1")
    dm.set_option("keep_ns_output", "0")
    dm.set_option("chunk_mb", "12288")
    dm.set_option("tune_ms", "40")
    for v in ("0", "1", "auto"):
        dm.set_option("program", v)                 # one launch per bucket's NS program: never / always / from 2048 rows up
    dm.set_option("l2_group_mb", "64")
    dm.set_option("small_fused", "1")
    for key, val in (("program", "2"), ("program", "yes"), ("l2_group_mb", "0"), ("l2_group_mb", "x"), ("small_fused", "2")):
        with pytest.raises(dm.DmuonError) as ei:
            dm.set_option(key, val)
        assert ei.value.code == binding.ERR_INVALID_ARG
    for key, val in (("steps", "-1"), ("steps", "abc"), ("coeffs", "1,2"), ("mode", "bogus"), ("nope", "1"),
                     ("autotune", "maybe"), ("schedule", "gram"), ("coeffs_sched", "1,2;3"), ("coeffs_sched", "1,2,3/4,5,6"),
                     ("chunk_mb", "0"), ("tune_ms", "-1"), ("fuse_epilogue", "2"), ("overlap", "1")):
        with pytest.raises(dm.DmuonError) as ei:
            dm.set_option(key, val)
        assert ei.value.code == binding.ERR_INVALID_ARG
        assert binding.last_error() != ""
    dm.set_option("mode", "tc")


def test_invalid_arguments_rejected_before_any_device_work():
    L = binding.lib()
    shapes = (ctypes.c_int32 * 2)(128, 0)
    ptrs = (ctypes.c_void_p * 1)(0x1000)
    assert L.dmuon_ns_batched(ptrs, shapes, 1, 5, None, None) == binding.ERR_INVALID_ARG     # cols = 0
    shapes = (ctypes.c_int32 * 2)(128, 128)
    assert L.dmuon_ns_batched(ptrs, shapes, -1, 5, None, None) == binding.ERR_INVALID_ARG    # count < 0
    assert L.dmuon_ns_batched(ptrs, shapes, 1, -2, None, None) == binding.ERR_INVALID_ARG    # steps < 0
    assert L.dmuon_ns_batched(None, shapes, 1, 5, None, None) == binding.ERR_INVALID_ARG     # null array
    bad = (ctypes.c_void_p * 1)(0x1002)
    assert L.dmuon_ns_batched(bad, shapes, 1, 5, None, None) == binding.ERR_INVALID_ARG      # misaligned
    null = (ctypes.c_void_p * 1)(None)
    assert L.dmuon_muon_step(ptrs, null, ptrs, shapes, 1, 0.02, 0.95, 0.01, None) == binding.ERR_INVALID_ARG
    assert L.dmuon_ns_batched(ptrs, shapes, 0, 5, None, None) == binding.OK                   # count == 0: no-op
    assert L.dmuon_muon_step(None, None, None, None, 0, 0.02, 0.95, 0.01, None) == binding.OK
    assert L.dmuon_ns_gemm(7, ptrs, None, ptrs, 128, 128, 1, 1.0, 0.0, -1, None) == binding.ERR_INVALID_ARG
    assert L.dmuon_ns_gemm(0, ptrs, None, ptrs, 100, 128, 1, 1.0, 0.0, -1, None) == binding.ERR_INVALID_ARG
    assert L.dmuon_set_workspace(ctypes.c_void_p(0x1000), 0) == binding.ERR_INVALID_ARG
    assert L.dmuon_read_ns_output(0, None, None) == binding.ERR_INVALID_ARG
    assert L.dmuon_muon_step_master(ptrs, None, ptrs, ptrs, shapes, 1, 0.02, 0.95, 0.01, None) == binding.ERR_INVALID_ARG
    assert L.dmuon_muon_step_master(None, None, None, None, None, 0, 0.02, 0.95, 0.01, None) == binding.OK


@pytest.mark.skipif(torch.cuda.is_available(), reason="only meaningful on a box without a GPU")
def test_no_cpu_fallback():
    """Without an sm_100 device the product path must fail loudly, not compute somewhere else."""
    with pytest.raises(dm.DmuonError) as ei:
        dm.warmup([(128, 512)])
    assert ei.value.code == binding.ERR_UNSUPPORTED_DEVICE
    x = torch.zeros((128, 512), dtype=torch.bfloat16)
    with pytest.raises(ValueError):
        dm.ns_batched([x])            # host tensor handed to the device entry point


def test_workspace_bytes_formula():
    dm.set_option("mode", "tc")
    # one 4096 x 14336 matrix: two X buffers + five m x m buffers (G, B, B', T, R of the Gram blocks) in fp16
    want = 2 * 4096 * 14336 * 2 + 5 * 4096 * 4096 * 2
    assert dm.workspace_bytes([(4096, 14336)]) == want
    assert dm.workspace_bytes([(14336, 4096)]) == want                # tall: same oriented shape
    # square: plain iteration, two X buffers + A + B
    assert dm.workspace_bytes([(4096, 4096)]) == 4 * 4096 * 4096 * 2
    # ragged: padded to multiples of 128
    assert dm.workspace_bytes([(100, 260)]) == 2 * 128 * 384 * 2 + 2 * 128 * 128 * 2
    assert dm.workspace_bytes([]) == 0
    assert dm.workspace_bytes([(0, 5)]) == 0
    # buckets run one after the other through ONE region: the workspace is the largest bucket's, not the sum
    sq, wide = 4 * 4096 * 4096 * 2, want
    assert dm.workspace_bytes([(4096, 4096)] * 3 + [(4096, 14336)] * 2) == max(3 * sq, 2 * wide)
    # a bucket over the chunk cap runs as chunks of fewer matrices (64 tall matrices, 12 GiB cap -> 2 chunks of 32)
    assert dm.workspace_bytes([(14336, 4096)] * 64) == 32 * want == 12 << 30
    assert dm.workspace_bytes(synth.config_shapes(4)) == 12 << 30        # was 49 GB when every matrix owned its buffers
    dm.set_option("chunk_mb", 1024)
    assert dm.workspace_bytes([(14336, 4096)] * 64) == 2 * want          # 1 GiB cap: chunks of 2
    assert dm.workspace_bytes([(8192, 28672)]) == 2 * 8192 * 28672 * 2 + 5 * 8192 * 8192 * 2    # one matrix always fits
    dm.set_option("chunk_mb", 12288)
    # keep_ns_output: every matrix keeps its own buffers until the call returns (test hook)
    dm.set_option("keep_ns_output", 1)
    assert dm.workspace_bytes([(4096, 4096)] * 3 + [(4096, 14336)] * 2) == 3 * sq + 2 * wide
    dm.set_option("keep_ns_output", 0)
    dm.set_option("mode", "fp32_check")
    assert dm.workspace_bytes([(4096, 14336)]) == 2 * (2 * 4096 * 14336 * 2 + 2 * 4096 * 4096 * 2)
    dm.set_option("mode", "tc")


def test_block_schedule_host_logic():
    """Gram blocks (Eq. 4) only on wide buckets; a 3-block only first; lengths sum to the step count;
    blocks shrink when the recurrence's error gain prod a^2 exceeds 200."""
    dm.set_option("mode", "tc")
    dm.set_option("schedule", "auto")
    for shape in ((4096, 14336), (14336, 4096), (1024, 4096), (768, 3072), (896, 4864), (2048, 3072)):
        assert dm.block_schedule(shape, 5) == [3, 2]
        for k in range(0, 12):
            part = dm.block_schedule(shape, k)
            assert sum(part) == k and all(1 <= L <= 3 for L in part)
            assert all(L <= 2 for L in part[1:]), "a 3-block may only come first"
        assert dm.block_schedule(shape, 4) == [2, 2]
    for shape in ((4096, 4096), (896, 896), (128, 896), (128, 512), (1000, 1400), (1, 64), (37, 91)):
        assert dm.block_schedule(shape, 5) == [1] * 5              # square-ish or a single-block Gram matrix
    # large a: shorter blocks.  a = 4: a^4 = 256 > 200 forbids the 3-block; a = 15: a^2 = 225 forbids any block
    assert dm.block_schedule((1024, 4096), 5, (4.0, -5.0, 2.0)) == [2, 2, 1]
    assert dm.block_schedule((1024, 4096), 5, (15.0, -5.0, 2.0)) == [1] * 5
    sched = [(8.0, -20.0, 14.0), (4.0, -3.0, 0.5), (3.9, -2.9, 0.5), (3.3, -2.4, 0.4), (2.3, -1.7, 0.4)]
    assert dm.block_schedule((1024, 4096), 5, sched) == [2, 2, 1]  # 64 * 16 > 200 -> 2-block; then 3.9^2 -> 2-block
    dm.set_option("schedule", "x")
    assert dm.block_schedule((1024, 4096), 5) == [1] * 5
    dm.set_option("schedule", "auto")
    dm.set_option("mode", "fp32_check")
    assert dm.block_schedule((1024, 4096), 5) == [1] * 5           # the check mode is always the plain iteration
    dm.set_option("mode", "tc")
    L = binding.lib()
    out = (ctypes.c_int32 * 4)()
    assert L.dmuon_block_schedule(0, 5, 5, None, 0, out, 4) == binding.ERR_INVALID_ARG
    assert L.dmuon_block_schedule(8, 8, -1, None, 0, out, 4) == binding.ERR_INVALID_ARG
    assert L.dmuon_block_schedule(8, 8, 5, None, 1, out, 4) == binding.ERR_INVALID_ARG   # per-step without coeffs


def test_config_shape_sets_match_baseline():
    c2, c3, c4 = synth.config_shapes(2), synth.config_shapes(3), synth.config_shapes(4)
    assert (len(c2), len(c3), len(c4)) == (72, 168, 224)
    elems = lambda s: sum(r * c for r, c in s)
    assert abs(elems(c2) / 1e6 - 84.9) < 0.1
    assert abs(elems(c3) / 1e6 - 357.8) < 0.1
    assert abs(elems(c4) / 1e6 - 6979.3) < 0.1
    assert synth.config_shapes(1) == [(128, 512)] * 8
    sq = dict(synth.sweep_shapes())
    assert sq[(256, 256)] == 65536 and sq[(8192, 8192)] == 64


def test_synthetic_gradient_statistics():
    """configs[1] recipe: N(0, 1e-3^2) noise + rank-8 component carrying 10x the noise energy."""
    g = synth.gradient((768, 3072), 1234).to(torch.float64)
    energy = (g ** 2).sum().item()
    noise = 768 * 3072 * 1e-6
    assert 7.0 < energy / noise < 16.0
    sv = torch.linalg.svdvals(g)
    assert sv[7] / sv[8] > 3.0               # 8 spikes stand out of the bulk
    a = synth.gradient((64, 64), 5)
    b = synth.gradient((64, 64), 5)
    assert torch.equal(a, b)                 # seeded
    assert not torch.equal(a, synth.gradient((64, 64), 6))
    w = synth.weight((512, 512), 9).float()
    assert abs(w.std().item() - 0.02) < 2e-3


def _brute_force_assignment(counts, batch_sizes, costs, ranks):
    """Eq. 5 by exhaustive enumeration: every multiset of batches per shape, every placement."""
    import itertools
    jobs_per_shape = []
    for n, bs, cs in zip(counts, batch_sizes, costs):
        decomps = []

        def rec(rem, start, cur):
            if rem == 0:
                decomps.append(list(cur))
                return
            for j in range(start, len(bs)):
                if bs[j] <= rem:
                    cur.append(cs[j])
                    rec(rem - bs[j], j, cur)
                    cur.pop()
        rec(n, 0, [])
        jobs_per_shape.append(decomps)
    best = float("inf")
    for combo in itertools.product(*jobs_per_shape):
        jobs = [c for d in combo for c in d]
        for place in itertools.product(range(ranks), repeat=len(jobs)):
            load = [0.0] * ranks
            for c, r in zip(jobs, place):
                load[r] += c
            best = min(best, max(load))
    return best


def test_owner_assignment_against_brute_force():
    """dmuon_assign_owners: exact mode equals an exhaustive search of Eq. 5 on small instances; the
    greedy mode is feasible, never better than the optimum and within 4/3 of it (the LPT bound) on these."""
    import random
    rng = random.Random(5)
    for trial in range(25):
        S = rng.randint(1, 3)
        ranks = rng.randint(2, 3)
        counts = [rng.randint(1, 4) for _ in range(S)]
        batch_sizes, costs = [], []
        for s in range(S):
            bs = [1] + sorted(rng.sample([2, 3, 4], rng.randint(0, 2)))
            unit = rng.uniform(0.5, 4.0)
            cs = [unit * b * (1.0 if b == 1 else rng.uniform(0.55, 0.95)) for b in bs]   # batching amortises (Fig. 7)
            batch_sizes.append(bs)
            costs.append(cs)
        want = _brute_force_assignment(counts, batch_sizes, costs, ranks)
        for mode in (1, 0, -1):
            x, ms, exact = dm.assign_owners(counts, batch_sizes, costs, ranks, mode=mode, threshold=64)
            # feasibility: every matrix assigned exactly once; makespan as reported
            load = [0.0] * ranks
            for s in range(S):
                assert sum(batch_sizes[s][j] * sum(x[s][j]) for j in range(len(batch_sizes[s]))) == counts[s]
                for j in range(len(batch_sizes[s])):
                    assert all(v >= 0 for v in x[s][j])
                    for r in range(ranks):
                        load[r] += costs[s][j] * x[s][j][r]
            assert abs(max(load) - ms) < 1e-9
            if mode == 0:
                assert not exact and want - 1e-9 <= ms <= 4.0 / 3.0 * want + 1e-9
            else:
                assert exact and abs(ms - want) < 1e-9, (trial, counts, batch_sizes, costs, ranks, ms, want)


def test_owner_assignment_llama_like_and_threshold():
    """A config-4-like instance: 3 shape classes, 8 ranks.  Greedy lands within a few percent of the lower bound
    total/R; above the S_thr threshold mode -1 takes the greedy path."""
    counts = [64, 64, 96]                                   # q/o, k/v, gate/up/down
    batch_sizes = [[1, 2, 4, 8], [1, 4, 16], [1, 2, 4]]
    costs = [[1.30, 2.45, 4.75, 9.4], [0.10, 0.22, 0.70], [2.9, 5.6, 11.0]]
    x, ms, exact = dm.assign_owners(counts, batch_sizes, costs, 8, mode=-1, threshold=16)
    assert not exact                                        # 10 x 8 = 80 variables > 16
    total = 64 / 8 * 9.4 + 64 / 16 * 0.70 + 96 / 4 * 11.0   # cheapest batching of everything
    assert total / 8 - 1e-9 <= ms <= 1.05 * total / 8
    # rank0 ablation handle of PAPER.md:260: one rank owns everything -> makespan = total
    x1, ms1, _ = dm.assign_owners(counts, batch_sizes, costs, 1, mode=0)
    assert abs(ms1 - total) < 1e-9
    with pytest.raises(dm.DmuonError):
        dm.assign_owners([3], [[2]], [[1.0]], 2)            # 3 matrices cannot be cut into batches of 2


def test_adamw_and_cost_entry_points_validate_on_cpu():
    L = binding.lib()
    n = (ctypes.c_int64 * 1)(16)
    ptrs = (ctypes.c_void_p * 1)(0x1000)
    assert L.dmuon_adamw_step(ptrs, ptrs, ptrs, ptrs, n, 1, 1e-3, 0.9, 0.999, 1e-8, 0.01, 0, None) == binding.ERR_INVALID_ARG   # step < 1
    assert L.dmuon_adamw_step(ptrs, ptrs, ptrs, ptrs, n, 1, 1e-3, 1.0, 0.999, 1e-8, 0.01, 1, None) == binding.ERR_INVALID_ARG   # beta1 = 1
    assert L.dmuon_adamw_step(None, None, None, None, None, 0, 1e-3, 0.9, 0.999, 1e-8, 0.01, 1, None) == binding.OK            # count = 0
    bad = (ctypes.c_void_p * 1)(0x1004)
    assert L.dmuon_adamw_step(bad, ptrs, ptrs, ptrs, n, 1, 1e-3, 0.9, 0.999, 1e-8, 0.01, 1, None) == binding.ERR_INVALID_ARG    # misaligned
    out = ctypes.c_float(0)
    assert L.dmuon_measure_cost(0, 8, 1, 1, ctypes.byref(out), None) == binding.ERR_INVALID_ARG
