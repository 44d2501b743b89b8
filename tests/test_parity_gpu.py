"""Parity of the CUDA path (through the C ABI) against the PLAIN fp64 oracle on the same seeded bf16 inputs.

Bars (BASELINE.json north_star): relative Frobenius error of O = NS_5(.) <= 1e-2 on the tensor-core path
(16-bit operands, fp32 accumulation) and <= 1e-4 in the fp32-operand check mode.  M' is compared elementwise
with the fp64 oracle's (<= 1 bf16 ulp: fp32 vs fp64 arithmetic before the same rounding; the share of elements
that differ is printed), W' by the criterion of DESIGN.md ("error no worse than the output rounding plus 1 % of
the update").  Every comparison is against oracle.muon_step(..., momentum_fp32=False), the definition
north_star gives.  ADDITIONALLY M' is checked bit for bit against the oracle's binary32-momentum mode (reading
N16, steps = 0 so no NS work is repeated): that check is extra, it replaces none of the fp64 ones.
"""
import functools

import numpy as np
import pytest
import torch

import oracle
import paper_2606_27153_b200 as dm
from paper_2606_27153_b200 import synth
from helpers import LR, LR_F, MU, MU_F, TOL_CHECK, TOL_TC, WD, WD_F, bf16_ulp, rel_fro, to64

pytestmark = pytest.mark.gpu


@pytest.fixture(autouse=True)
def _reset_options():
    dm.set_option("mode", "tc")
    dm.set_option("steps", 5)
    dm.set_option("coeffs", "3.4445,-4.7750,2.0315")
    dm.set_option("schedule", "auto")
    dm.set_option("overlap", 0)
    yield
    dm.set_option("mode", "tc")
    dm.set_option("steps", 5)
    dm.set_option("schedule", "auto")
    dm.set_option("overlap", 0)


@functools.lru_cache(maxsize=None)
def oracle_muon(config: int, index: int, random_momentum: bool):
    """Oracle Muon step for matrix `index` of a config (inputs regenerated on the GPU with the same seed and read back)."""
    _, W, G, M = synth.muon_inputs(config, "cuda", random_momentum, indices=[index])
    return oracle_both(to64(W[0]), to64(G[0]), to64(M[0]))


def oracle_both(w, g, m):
    """The plain fp64 oracle step, plus (key "M_n16") the stored M' of the binary32-momentum mode (N16)."""
    orc = oracle.muon_step(w, g, m, LR_F, MU_F, WD_F)
    orc["M_n16"] = oracle.muon_step(w, g, m, LR_F, MU_F, WD_F, steps=0, momentum_fp32=True)["M_new"]
    return orc


STATS = {"m_mismatch": []}     # share of M' elements that differ from RNE(fp64 M') (printed by the callers)


def check_muon_matrix(idx, shape, W0, Wg, Mg, Og, orc, tol):
    """Wg, Mg: GPU results (bf16 tensors); Og: unrounded GPU O (fp32); W0: W before the step (float64)."""
    e_o = rel_fro(to64(Og), orc["O"])
    assert e_o <= tol, f"matrix {idx} {shape}: O rel err {e_o:.3e} > {tol}"
    # M' against the fp64 oracle: a quantised value, so fp32 (kernel) and fp64 (oracle) arithmetic before the same
    # RNE rounding may land on neighbouring bf16 values where the exact value sits on a tie: <= 1 bf16 ulp elementwise
    mg, m_orc = to64(Mg), oracle.round_bf16(orc["M_new"])
    dm_ = np.abs(mg - m_orc)
    assert (dm_ <= bf16_ulp(np.maximum(np.abs(mg), np.abs(m_orc)))).all(), f"matrix {idx}: M' off by more than 1 bf16 ulp"
    STATS["m_mismatch"].append(float((dm_ != 0).mean()))
    # additional check (reading N16): formed in binary32 with one fused rounding on both sides -> identical bits
    if "M_n16" in orc:
        m16 = oracle.round_bf16(orc["M_n16"])
        assert np.array_equal(mg, m16), f"matrix {idx}: M' differs from the binary32 mode ({(mg != m16).mean():.2e} of elements)"
    # W': no worse than the output rounding plus 1 % of the update (2 % slack on the rounding term: the two
    # roundings are different random draws of the same distribution)
    w_orc = orc["W_new"]
    r = np.linalg.norm(oracle.round_bf16(w_orc) - w_orc)
    upd = np.linalg.norm(w_orc - W0)
    err = np.linalg.norm(to64(Wg) - w_orc)
    assert err <= 1.02 * r + tol * upd, f"matrix {idx}: W' err {err:.3e} > {1.02 * r + tol * upd:.3e}"
    return e_o


# ------------------------------------------------------------------------------------------------ configs[0]

@pytest.mark.parametrize("mode,tol", [("tc", TOL_TC), ("fp32_check", TOL_CHECK)])
def test_config1_ns_batched(mode, tol):
    dm.set_option("mode", mode)
    shapes, Xs = synth.ns_inputs("cuda")
    X64 = [to64(x) for x in Xs]
    dm.ns_batched(Xs, steps=5)
    torch.cuda.synchronize()
    worst = 0.0
    for i, (x64, xg) in enumerate(zip(X64, Xs)):
        o = oracle.ns(x64)
        og = dm.binding.read_ns_output(i, shapes[i])
        e = rel_fro(to64(og), o)
        worst = max(worst, e)
        assert e <= tol, f"matrix {i}: O rel err {e:.3e}"
        # the in-place bf16 result is the RNE of the unrounded one
        assert torch.equal(xg, og.to(torch.bfloat16))
        assert rel_fro(to64(xg), o) <= max(tol, 3e-3)          # bf16 output rounding floor ~1.7e-3
    print(f"config1 {mode}: worst rel err {worst:.3e}")


# ------------------------------------------------------------------------------------------------ configs[1]

def _run_muon_config(config, random_momentum, mode, check_indices, tol):
    dm.set_option("mode", mode)
    shapes, W, G, M = synth.muon_inputs(config, "cuda", random_momentum)
    W0 = {i: to64(W[i]) for i in check_indices}
    G0 = [g.clone() for g in G]
    dm.muon_step(W, G, M, LR, MU, WD)
    torch.cuda.synchronize()
    worst = 0.0
    for i in check_indices:
        og = dm.binding.read_ns_output(i, shapes[i])
        orc = oracle_muon(config, i, random_momentum)
        worst = max(worst, check_muon_matrix(i, shapes[i], W0[i], W[i], M[i], og, orc, tol))
    for g, g0 in zip(G, G0):
        assert torch.equal(g, g0), "grads must never be written"
    mm = STATS["m_mismatch"][-len(check_indices):]
    print(f"config{config} {mode} momentum={random_momentum}: worst O rel err vs fp64 oracle {worst:.3e} over {len(check_indices)} matrices; "
          f"M' elements differing from RNE(fp64 M') (all within 1 ulp): mean {np.mean(mm):.2e}, max {np.max(mm):.2e}")


def test_config2_muon_step_all_matrices():
    _run_muon_config(2, False, "tc", list(range(72)), TOL_TC)


def test_config2_muon_step_check_mode_first_layer():
    _run_muon_config(2, False, "fp32_check", list(range(6)), TOL_CHECK)


def test_config2_with_momentum_state():
    _run_muon_config(2, True, "tc", [0, 4, 5, 66, 70, 71], TOL_TC)


def test_config2_plain_iteration_schedule():
    """schedule=x: the wide buckets (3072x768, 768x3072) take the plain X iteration instead of Gram blocks."""
    dm.set_option("schedule", "x")
    _run_muon_config(2, True, "tc", [0, 4, 5, 70, 71], TOL_TC)


def test_config2_schedule_reported():
    plan = dm.describe_plan(synth.config_shapes(2), steps=5)
    blocks = {(b["m"], b["n"]): b["blocks"] for b in plan["buckets"]}
    assert blocks == {(768, 768): [1, 1, 1, 1, 1], (768, 3072): [3, 2]}
    assert sum(b["count"] for b in plan["buckets"]) == 72


@pytest.mark.parametrize("steps", [1, 2, 3, 4, 5, 6, 7])
def test_gram_blocks_every_step_count(steps):
    """Wide matrices (Gram-block buckets, incl. a tall and a ragged one) against the oracle for every block
    partition: [1], [2], [3], [2,2], [3,2], [3,2,1], [3,2,2] (Eq. 4 PAPER.md:172 is an exact reformulation of Eq. 2)."""
    shapes = [(256, 1024), (1024, 256), (384, 640), (257, 1000), (512, 1536)]
    Xs = [synth.gradient(s, 7300 + i, "cuda") if i % 2 == 0 else synth.iid_normal(s, 7300 + i, "cuda")
          for i, s in enumerate(shapes)]
    assert all(sum(dm.block_schedule(s, steps)) == steps for s in shapes)
    assert dm.block_schedule(shapes[0], steps) != [1] * steps or steps == 1
    X64 = [to64(x) for x in Xs]
    dm.ns_batched(Xs, steps=steps)
    torch.cuda.synchronize()
    for i, s in enumerate(shapes):
        e = rel_fro(to64(dm.binding.read_ns_output(i, s)), oracle.ns(X64[i], steps=steps))
        assert e <= TOL_TC, f"steps={steps} {s}: rel err {e:.3e}"


def test_gram_blocks_per_step_coefficients():
    """dmuon_ns_batched_sched on a Gram-block bucket: P_i = a_i I + B_i with a different triple per step."""
    sched = [[3.9, -6.0, 2.8], [3.6, -5.2, 2.3], [3.4445, -4.775, 2.0315], [3.0, -3.6, 1.3], [2.4, -2.2, 0.6]]
    shapes = [(256, 1024), (640, 384)]
    assert dm.block_schedule(shapes[0], 5, sched) == [3, 2]
    Xs = [synth.gradient(s, 7400 + i, "cuda") for i, s in enumerate(shapes)]
    X64 = [to64(x) for x in Xs]
    dm.ns_batched_sched(Xs, sched)
    torch.cuda.synchronize()
    for i, s in enumerate(shapes):
        e = rel_fro(to64(dm.binding.read_ns_output(i, s)), oracle.ns(X64[i], steps=5, coeffs=np.array(sched)))
        assert e <= TOL_TC, f"{s}: rel err {e:.3e}"


# ------------------------------------------------------------------------------------------------ configs[2]

def test_config3_full_launch_sampled_layers():
    """All 168 matrices go through the GPU in the configuration bench.py would time; the oracle checks one full
    layer (7 matrices, every distinct shape incl. the tall 4864x896 and the 128-row k/v) plus the last matrix."""
    _run_muon_config(3, True, "tc", [0, 1, 2, 3, 4, 5, 6, 167], TOL_TC)


# ------------------------------------------------------------------------------------------------ configs[3]

@pytest.mark.slow
def test_config4_full_size_sampled():
    """Llama-3-8B-shaped set at full size (42 GB resident), in the launch configuration bench.py times.  The plain
    fp64 oracle runs a whole Muon step of one matrix of EVERY distinct shape: k (1024x4096, layers 0 and 31),
    q (4096x4096), gate (14336x4096, tall) and down (4096x14336) -- the three shapes that carry 99 % of the FLOPs
    (>= one matrix per distinct shape).  O, M' and W' are compared as on the small configs."""
    import time
    dm.set_option("mode", "tc")
    shapes, W, G, M = synth.muon_inputs(4, "cuda", False)
    idx = [1, 218, 0, 4, 6]
    pre = {i: (to64(W[i]), to64(G[i]), to64(M[i])) for i in idx}
    dm.muon_step(W, G, M, LR, MU, WD)
    torch.cuda.synchronize()
    got = {i: (W[i].clone(), M[i].clone(), dm.binding.read_ns_output(i, shapes[i]).cpu()) for i in idx}
    plan = dm.describe_plan(shapes, steps=5)
    del W, G, M
    torch.cuda.empty_cache()
    for i in idx:
        w0, g0, m0 = pre.pop(i)
        t0 = time.perf_counter()
        orc = oracle_both(w0, g0, m0)
        secs = time.perf_counter() - t0
        wg, mg, og = got.pop(i)
        e = check_muon_matrix(i, shapes[i], w0, wg, mg, og, orc, TOL_TC)
        print(f"config4 matrix {i} {shapes[i]}: O rel err vs fp64 oracle {e:.3e}; M' mismatch share {STATS['m_mismatch'][-1]:.2e} "
              f"(oracle {secs:.0f} s on {oracle.num_threads()} threads)")
        del orc, w0, g0, m0
    print("config4 plan:", plan["buckets"])


# ------------------------------------------------------------------------------------------------ edge cases

RAGGED = [(100, 260), (130, 70), (1, 64), (64, 1), (200, 200), (37, 91), (8, 8), (257, 129), (128, 128), (3, 1000)]


@pytest.mark.parametrize("mode,tol", [("tc", TOL_TC), ("fp32_check", TOL_CHECK)])
def test_ragged_and_degenerate_shapes(mode, tol):
    dm.set_option("mode", mode)
    Xs = [synth.iid_normal(s, 7000 + i, "cuda", std=0.3) for i, s in enumerate(RAGGED)]
    X64 = [to64(x) for x in Xs]
    dm.ns_batched(Xs, steps=5)
    torch.cuda.synchronize()
    for i, s in enumerate(RAGGED):
        og = dm.binding.read_ns_output(i, s)
        e = rel_fro(to64(og), oracle.ns(X64[i]))
        assert e <= tol, f"{s}: rel err {e:.3e}"


def test_zero_matrix_steps0_count0_and_schedule():
    z = torch.zeros((128, 256), dtype=torch.bfloat16, device="cuda")
    x = synth.iid_normal((96, 160), 7100, "cuda")
    x64 = to64(x)
    dm.ns_batched([z, x.clone()], steps=5)
    torch.cuda.synchronize()
    assert torch.count_nonzero(z).item() == 0                       # reading N14: zero in, zero out, no NaN
    # steps = 0: normalisation only
    y = x.clone()
    dm.ns_batched([y], steps=0)
    torch.cuda.synchronize()
    assert rel_fro(to64(dm.binding.read_ns_output(0, (96, 160))), oracle.ns(x64, steps=0)) < 1e-3
    # count = 0
    dm.ns_batched([], steps=5)
    dm.muon_step([], [], [], LR, MU, WD)
    # per-step schedule (NEXT-1 entry) == oracle with the same schedule
    sched = [[3.0, -3.5, 1.2], [2.5, -2.0, 0.6], [1.5, -0.5, 0.0]]
    y = x.clone()
    dm.ns_batched_sched([y], sched)
    torch.cuda.synchronize()
    assert rel_fro(to64(dm.binding.read_ns_output(0, (96, 160))), oracle.ns(x64, steps=3, coeffs=np.array(sched))) <= TOL_TC


def test_zero_gradient_muon_step():
    w = synth.weight((256, 128), 7200, "cuda")
    w0 = to64(w)
    g = torch.zeros_like(w)
    m = torch.zeros_like(w)
    dm.muon_step([w], [g], [m], LR, MU, WD)
    torch.cuda.synchronize()
    want = oracle.round_bf16(w0 - LR_F * WD_F * w0)
    assert np.abs(to64(w) - want).max() <= bf16_ulp(want).max()
    assert torch.count_nonzero(m).item() == 0


def test_master_weights_step():
    """dmuon_muon_step_master: the update lands in the fp32 master; the bf16 parameter is its rounding.
    Covers the flat, the transposing and the generic (ragged) apply paths.  With a master the UPDATE itself is
    checked to the NS tolerance, which bf16 weights cannot show (their rounding swamps a 1-5 ulp update)."""
    shapes = [(768, 768), (3072, 768), (768, 3072), (100, 260), (130, 70)]
    G = [synth.gradient(s, 7500 + i, "cuda") for i, s in enumerate(shapes)]
    M = [synth.gradient(s, 7600 + i, "cuda") for i, s in enumerate(shapes)]
    W32 = []
    for i, s in enumerate(shapes):
        g = torch.Generator(device="cuda")
        g.manual_seed(7700 + i)
        W32.append((torch.randn(s, generator=g, device="cuda", dtype=torch.float32) * 0.02).contiguous())   # not bf16-representable
    W = [torch.full(s, float("nan"), dtype=torch.bfloat16, device="cuda") for s in shapes]   # must be overwritten, never read
    W0 = [to64(w) for w in W32]
    M0 = [to64(m) for m in M]
    dm.muon_step_master(W, W32, G, M, LR, MU, WD)
    torch.cuda.synchronize()
    for i, s in enumerate(shapes):
        orc = oracle_both(W0[i], to64(G[i]), M0[i])
        assert torch.equal(W[i], W32[i].to(torch.bfloat16)), f"{s}: bf16 parameter is not the rounding of the master"
        assert np.array_equal(to64(M[i]), oracle.round_bf16(orc["M_n16"])), f"{s}: M' differs from the binary32 mode"
        m_orc = oracle.round_bf16(orc["M_new"])
        assert (np.abs(to64(M[i]) - m_orc) <= bf16_ulp(m_orc)).all(), f"{s}: M' off the fp64 oracle by more than 1 bf16 ulp"
        upd_orc = orc["W_new"] - W0[i]
        upd_gpu = to64(W32[i]) - W0[i]
        e = np.linalg.norm(upd_gpu - upd_orc) / np.linalg.norm(upd_orc)
        # fp32 rounding of a weight of size 0.02 is ~1e-9, the update per element ~1e-4..1e-3: negligible next to TOL_TC
        assert e <= TOL_TC + 1e-4, f"{s}: relative error of the applied update {e:.3e}"
    with pytest.raises(dm.DmuonError):                                  # misaligned master
        buf = torch.zeros(128 * 128 + 4, dtype=torch.float32, device="cuda")
        dm.binding._check(dm.binding.lib().dmuon_muon_step_master(
            dm.binding._ptr_array([W[0][:128, :128].contiguous()]), dm.binding._ptr_array([buf[1:1 + 128 * 128]]),
            dm.binding._ptr_array([G[0][:128, :128].contiguous()]), dm.binding._ptr_array([M[0][:128, :128].contiguous()]),
            dm.binding._shape_array([(128, 128)])[0], 1, 0.02, 0.95, 0.01, None))
    # a following plain step on the same shapes must not touch the masters (the binding is per call)
    keep = [w.clone() for w in W32]
    dm.muon_step(W, G, M, LR, MU, WD)
    torch.cuda.synchronize()
    assert all(torch.equal(a, b) for a, b in zip(keep, W32))


@pytest.mark.parametrize("overlap", [0, 1])
def test_step_is_cuda_graph_capturable(overlap):
    """After the first call for a shape set (plan, autotune, pointer binding) a step only enqueues kernels on the
    caller's stream, so it can be captured into a CUDA graph; the replay equals the eager step bit for bit."""
    dm.set_option("overlap", overlap)                      # 1: the library's side stream forks and joins inside the capture
    shapes, W, G, M = synth.muon_inputs(2, "cuda", True, indices=list(range(12)))
    W0, M0 = [w.clone() for w in W], [m.clone() for m in M]
    dm.muon_step(W, G, M, LR, MU, WD)                      # eager: builds the plan, binds these pointers
    torch.cuda.synchronize()
    W1, M1 = [w.clone() for w in W], [m.clone() for m in M]
    for w, w0, m, m0 in zip(W, W0, M, M0):
        w.copy_(w0)
        m.copy_(m0)
    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            dm.muon_step(W, G, M, LR, MU, WD)
    for w, w0, m, m0 in zip(W, W0, M, M0):               # capture does not execute: restore, then replay
        w.copy_(w0)
        m.copy_(m0)
    graph.replay()
    torch.cuda.synchronize()
    assert all(torch.equal(a, b) for a, b in zip(W, W1)) and all(torch.equal(a, b) for a, b in zip(M, M1))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(10):
        graph.replay()
    e1.record()
    torch.cuda.synchronize()
    t_graph = e0.elapsed_time(e1) / 10
    e0.record()
    for _ in range(10):
        dm.muon_step(W, G, M, LR, MU, WD)
    e1.record()
    torch.cuda.synchronize()
    print(f"2 layers of config 2: graph replay {t_graph:.3f} ms/step, eager {e0.elapsed_time(e1) / 10:.3f} ms/step")


def test_overlap_off_equals_overlap_on():
    """The side-stream schedule changes only when kernels run, never what they compute."""
    res = []
    for ov in (1, 0):
        dm.set_option("overlap", ov)
        shapes, W, G, M = synth.muon_inputs(3, "cuda", True, indices=list(range(14)))
        for _ in range(2):
            dm.muon_step(W, G, M, LR, MU, WD)
        torch.cuda.synchronize()
        res.append((W, M))
    assert all(torch.equal(a, b) for a, b in zip(res[0][0], res[1][0]))
    assert all(torch.equal(a, b) for a, b in zip(res[0][1], res[1][1]))


def test_two_steps_state_carried():
    """Two consecutive steps; the oracle restarts each step from the GPU's bf16 state (DESIGN.md parity rules)."""
    shapes, W, G, M = synth.muon_inputs(2, "cuda", False, indices=[0, 4, 5])
    for step in range(2):
        W0 = [to64(w) for w in W]
        M0 = [to64(m) for m in M]
        dm.muon_step(W, G, M, LR, MU, WD)
        torch.cuda.synchronize()
        for i in range(3):
            orc = oracle_both(W0[i], to64(G[i]), M0[i])
            og = dm.binding.read_ns_output(i, shapes[i])
            check_muon_matrix(i, shapes[i], W0[i], W[i], M[i], og, orc, TOL_TC)


def test_deterministic_and_host_entry_and_caller_workspace():
    shapes, W, G, M = synth.muon_inputs(2, "cuda", True, indices=[0, 4, 5, 6])
    Wa, Ma = [w.clone() for w in W], [m.clone() for m in M]
    Wb, Mb = [w.clone() for w in W], [m.clone() for m in M]
    dm.muon_step(Wa, G, Ma, LR, MU, WD)
    dm.muon_step(Wb, G, Mb, LR, MU, WD)
    torch.cuda.synchronize()
    for a, b in zip(Wa + Ma, Wb + Mb):
        assert torch.equal(a, b), "two runs on the same inputs must agree bitwise"
    # host entry point: same bits as the device entry point
    Wh = [w.cpu().pin_memory() for w in W]
    Gh = [g.cpu().pin_memory() for g in G]
    Mh = [m.cpu().pin_memory() for m in M]
    dm.muon_step_host(Wh, Gh, Mh, LR, MU, WD)
    torch.cuda.synchronize()
    for a, h in zip(Wa + Ma, Wh + Mh):
        assert torch.equal(a.cpu(), h)
    # caller-owned workspace
    need = dm.workspace_bytes(shapes)
    assert need > 0
    ws = torch.empty(need, dtype=torch.uint8, device="cuda")
    dm.set_workspace(ws)
    Wc, Mc = [w.clone() for w in W], [m.clone() for m in M]
    dm.muon_step(Wc, G, Mc, LR, MU, WD)
    torch.cuda.synchronize()
    for a, c in zip(Wa + Ma, Wc + Mc):
        assert torch.equal(a, c)
    dm.set_workspace(None)
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    dm.set_workspace(small)
    with pytest.raises(dm.DmuonError) as ei:
        dm.muon_step([w.clone() for w in W], G, [m.clone() for m in M], LR, MU, WD)
    assert ei.value.code == dm.binding.ERR_OOM
    dm.set_workspace(None)


def test_profile_counts_launches():
    dm.set_option("profile", 1)
    dm.profile_reset()
    shapes, W, G, M = synth.muon_inputs(2, "cuda", False, indices=[0, 4, 5])
    dm.muon_step(W, G, M, LR, MU, WD)
    prof = dm.profile_read()
    dm.set_option("profile", 0)
    k = {}
    for name, rec in prof["kernels"].items():          # GEMM launches are named family[m x n] per shape bucket
        f = k.setdefault(name.split("[")[0], {"launches": 0, "ms": 0.0})
        f["launches"] += rec["launches"]
        f["ms"] += rec["ms"]
    assert prof["kernels"]["ns_bx_update[768x3072]"]["launches"] == 2 and prof["kernels"]["ns_bx_update[768x768]"]["launches"] == 5
    # bucket 768x768: 5 plain steps x (SYRK, polynomial, X update); bucket 768x3072: blocks [3, 2] = 2 SYRK, 5 polynomial
    # products, 3 (3 - 1) + 3 (2 - 1) = 9 Gram-space products, 2 X updates; + momentum, norms, normalise, apply
    assert k["ns_syrk_xxt"]["launches"] == 7 and k["ns_sq_poly"]["launches"] == 10 and k["ns_bx_update"]["launches"] == 7
    assert k["ns_gram_mm"]["launches"] == 9
    # normalise and apply: one flat launch (768x768, 768x3072) + one transposing launch (3072x768) each
    assert k["momentum_nesterov_sumsq"]["launches"] == 1 and k["apply_update"]["launches"] == 2
    assert k["normalize_orient_cast"]["launches"] == 2
    assert prof["launches"] == 39
    assert all(v["ms"] > 0 for v in k.values())


def test_misaligned_pointer_rejected():
    buf = torch.zeros(128 * 128 + 8, dtype=torch.bfloat16, device="cuda")
    x = buf[1:1 + 128 * 128].view(128, 128)        # 2-byte offset: not 16-byte aligned
    with pytest.raises(dm.DmuonError) as ei:
        dm.ns_batched([x], steps=5)
    assert ei.value.code == dm.binding.ERR_INVALID_ARG
