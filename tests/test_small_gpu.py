"""The on-chip small-matrix kernel (csrc/ns_small_sm100.cu: all NS steps of a 256 x 256 padded matrix in one launch,
X / G / B resident in the shared memory of a CTA pair) against the PLAIN fp64 oracle, and against the grouped
per-product path of the same library (option small_fused=0) as a cross-check of every matrix of a batch.

Bars as in test_parity_gpu.py: O <= 1e-2 relative Frobenius error (16-bit operands, fp32 accumulation), M' <= 1 bf16
ulp, W' no worse than the output rounding plus 1 % of the update.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2606_27153_b200 as dm
from paper_2606_27153_b200 import synth
from helpers import LR, LR_F, MU, MU_F, TOL_TC, WD, WD_F, bf16_ulp, rel_fro, to64, w_bound

pytestmark = pytest.mark.gpu

SEED = 77000


@pytest.fixture(autouse=True)
def _reset_options():
    def base():
        dm.set_option("mode", "tc")
        dm.set_option("steps", 5)
        dm.set_option("coeffs", "3.4445,-4.7750,2.0315")
        dm.set_option("coeffs_sched", "")
        dm.set_option("schedule", "auto")
        dm.set_option("fuse_epilogue", 1)
        dm.set_option("small_fused", 1)
    base()
    dm.set_option("keep_ns_output", 1)
    yield
    base()
    dm.set_option("keep_ns_output", 0)


def _onchip(shapes, steps=5):
    return [b["onchip"] for b in dm.describe_plan(shapes, steps)["buckets"]]


def test_plan_reports_onchip_buckets():
    assert _onchip([(256, 256)] * 3) == [True]
    assert _onchip([(200, 250), (250, 200), (129, 256)]) == [True]          # generic shapes padded to 256 x 256
    assert _onchip([(256, 512)]) == [False] and _onchip([(128, 256)]) == [False] and _onchip([(512, 256)]) == [False]
    assert _onchip([(256, 256)], steps=17) == [False]                       # more steps than the kernel's table holds
    dm.set_option("small_fused", 0)
    assert _onchip([(256, 256)] * 3) == [False]


@pytest.mark.parametrize("count", [1, 3, 200])
def test_ns_batched_256_against_oracle(count):
    """More matrices than CTA pairs (200 > 74): every worker loops, X tiles of the next matrix land in the buffers the
    previous one used.  Oracle on a sample, the grouped path (small_fused=0) on every matrix."""
    shapes = [(256, 256)] * count
    Xs = [synth.iid_scaled(s, SEED + i, "cuda") for i, s in enumerate(shapes)]
    X64 = [to64(x) for x in Xs]
    assert _onchip(shapes) == [True]
    dm.ns_batched(Xs, steps=5)
    torch.cuda.synchronize()
    O = [to64(dm.binding.read_ns_output(i, s)) for i, s in enumerate(shapes)]
    sample = sorted({0, count // 2, count - 1, min(count - 1, 74), min(count - 1, 147), min(count - 1, 148)})
    worst = 0.0
    for i in sample:
        o = oracle.ns(X64[i])
        e = rel_fro(O[i], o)
        worst = max(worst, e)
        assert e <= TOL_TC, f"matrix {i}: O rel err {e:.3e}"
        # the bf16 output the caller receives is the rounding of the unrounded O
        assert rel_fro(to64(Xs[i]), o) <= TOL_TC + 2.0 ** -8
    # the grouped per-product path on the same inputs: two 16-bit routes to the same result
    dm.set_option("small_fused", 0)
    Ys = [synth.iid_scaled(s, SEED + i, "cuda") for i, s in enumerate(shapes)]
    dm.ns_batched(Ys, steps=5)
    torch.cuda.synchronize()
    for i, s in enumerate(shapes):
        e = rel_fro(O[i], to64(dm.binding.read_ns_output(i, s)))
        assert e <= 6e-3, f"matrix {i}: on-chip vs grouped {e:.3e}"
    print(f"on-chip 256 x 256 x {count}: worst O rel err vs oracle {worst:.2e}")


@pytest.mark.parametrize("steps", [1, 2, 3, 4, 6, 7])
def test_step_counts(steps):
    shapes = [(256, 256)] * 5
    Xs = [synth.iid_normal(s, SEED + 100 + i, "cuda") for i, s in enumerate(shapes)]
    X64 = [to64(x) for x in Xs]
    dm.ns_batched(Xs, steps=steps)
    torch.cuda.synchronize()
    for i in (0, 4):
        e = rel_fro(to64(dm.binding.read_ns_output(i, shapes[i])), oracle.ns(X64[i], steps=steps))
        assert e <= TOL_TC, f"steps {steps} matrix {i}: {e:.3e}"


def test_per_step_schedule():
    sched = [(4.0848, -6.8946, 2.9270), (3.9505, -6.3029, 2.6377), (3.7418, -5.5913, 2.3037), (2.8769, -3.1427, 1.2046),
             (2.8366, -3.0525, 1.2012)]
    shapes = [(256, 256)] * 4
    Xs = [synth.iid_normal(s, SEED + 200 + i, "cuda") for i, s in enumerate(shapes)]
    X64 = [to64(x) for x in Xs]
    dm.ns_batched_sched(Xs, sched)
    torch.cuda.synchronize()
    for i in range(4):
        e = rel_fro(to64(dm.binding.read_ns_output(i, shapes[i])), oracle.ns(X64[i], steps=5, coeffs=sched))
        assert e <= TOL_TC, f"matrix {i}: {e:.3e}"


def test_ragged_shapes_padded_to_256():
    """Generic shapes (not multiples of 128) are padded to 256 x 256 by the elementwise kernels (tall ones transposed) and
    run on chip; the result is stored back by the unfused pass."""
    shapes = [(200, 250), (250, 200), (129, 256), (256, 129), (255, 255), (131, 140)]
    Xs = [synth.iid_normal(s, SEED + 300 + i, "cuda") for i, s in enumerate(shapes)]
    X64 = [to64(x) for x in Xs]
    assert _onchip(shapes) == [True]
    dm.ns_batched(Xs, steps=5)
    torch.cuda.synchronize()
    for i, s in enumerate(shapes):
        o = oracle.ns(X64[i])
        e = rel_fro(to64(dm.binding.read_ns_output(i, s)), o)
        assert e <= TOL_TC, f"matrix {i} {s}: {e:.3e}"
        assert rel_fro(to64(Xs[i]), o) <= TOL_TC + 2.0 ** -8


def test_mixed_with_other_buckets():
    """A shape set with an on-chip bucket between grouped ones: buckets share one workspace region, one after another."""
    shapes = [(256, 256), (512, 512), (256, 256), (128, 512), (256, 256), (256, 1024)]
    Xs = [synth.iid_normal(s, SEED + 400 + i, "cuda") for i, s in enumerate(shapes)]
    X64 = [to64(x) for x in Xs]
    dm.set_option("keep_ns_output", 0)          # the layout the bench runs: buckets reuse one region
    dm.ns_batched(Xs, steps=5)
    torch.cuda.synchronize()
    for i, s in enumerate(shapes):
        e = rel_fro(to64(Xs[i]), oracle.ns(X64[i]))
        assert e <= TOL_TC + 2.0 ** -8, f"matrix {i} {s}: {e:.3e}"


def _muon_inputs(shapes, seed):
    W = [synth.weight(s, seed + 3 * i, "cuda") for i, s in enumerate(shapes)]
    G = [synth.gradient(s, seed + 3 * i + 1, "cuda") for i, s in enumerate(shapes)]
    M = [synth.gradient(s, seed + 3 * i + 2, "cuda") for i, s in enumerate(shapes)]
    return W, G, M


@pytest.mark.parametrize("keep", [1, 0])
def test_muon_step_fused_update(keep):
    """Full Muon step on 256 x 256 weights: momentum, norm, on-chip NS, W' written by the last X update's epilogue.
    keep = 0 is the configuration the bench runs (no O stored): W' and M' must be the same bits."""
    shapes = [(256, 256)] * 90 + [(250, 256), (256, 250)]
    W, G, M = _muon_inputs(shapes, SEED + 500)
    W0, G0, M0 = [to64(t) for t in W], [to64(t) for t in G], [to64(t) for t in M]
    dm.set_option("keep_ns_output", keep)
    dm.muon_step(W, G, M, LR, MU, WD)
    torch.cuda.synchronize()
    for i in (0, 45, 89, 90, 91):
        orc = oracle.muon_step(W0[i], G0[i], M0[i], LR_F, MU_F, WD_F)
        if keep:
            e = rel_fro(to64(dm.binding.read_ns_output(i, shapes[i])), orc["O"])
            assert e <= TOL_TC, f"matrix {i}: O {e:.3e}"
        m_orc = oracle.round_bf16(orc["M_new"])
        assert (np.abs(to64(M[i]) - m_orc) <= bf16_ulp(np.maximum(np.abs(to64(M[i])), np.abs(m_orc)))).all()
        w_orc = orc["W_new"]
        err, bound = w_bound(to64(W[i]), w_orc, W0[i], TOL_TC, oracle.round_bf16)
        assert err <= bound, f"matrix {i}: W' err {err:.3e} > {bound:.3e}"
    if keep:
        test_muon_step_fused_update.kept = ([w.clone() for w in W], [m.clone() for m in M])
    elif hasattr(test_muon_step_fused_update, "kept"):
        Wk, Mk = test_muon_step_fused_update.kept
        assert all(torch.equal(a, b) for a, b in zip(W, Wk)) and all(torch.equal(a, b) for a, b in zip(M, Mk))


def test_master_weights_on_chip():
    shapes = [(256, 256)] * 4
    W, G, M = _muon_inputs(shapes, SEED + 600)
    masters = [w.to(torch.float32) + 1e-4 * torch.randn_like(w, dtype=torch.float32) for w in W]
    P0 = [to64(p) for p in masters]
    G0, M0 = [to64(t) for t in G], [to64(t) for t in M]
    dm.muon_step_master(W, masters, G, M, LR, MU, WD)
    torch.cuda.synchronize()
    for i in range(4):
        orc = oracle.muon_step(P0[i], G0[i], M0[i], LR_F, MU_F, WD_F)
        assert torch.equal(W[i], masters[i].to(torch.bfloat16)), "bf16 parameter = RNE of the new master"
        upd, upd_orc = to64(masters[i]) - P0[i], orc["W_new"] - P0[i]
        assert np.linalg.norm(upd - upd_orc) <= (TOL_TC + 1e-4) * np.linalg.norm(upd_orc)


def test_deterministic_and_graph_capturable():
    shapes = [(256, 256)] * 80
    X1 = [synth.iid_normal(s, SEED + 700 + i, "cuda") for i, s in enumerate(shapes)]
    X2 = [x.clone() for x in X1]
    X3 = [x.clone() for x in X1]
    dm.set_option("keep_ns_output", 0)
    dm.ns_batched(X1, steps=5)
    dm.ns_batched(X2, steps=5)
    torch.cuda.synchronize()
    assert all(torch.equal(a, b) for a, b in zip(X1, X2))
    keep = [x.clone() for x in X3]
    dm.ns_batched(keep, steps=5)                 # eager: the plan exists and these tensors are bound before the capture
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(graph, stream=side):
            dm.ns_batched(keep, steps=5)
    for a, b in zip(keep, X3):                   # capture does not execute: restore the inputs, then replay
        a.copy_(b)
    graph.replay()
    torch.cuda.synchronize()
    assert all(torch.equal(a, b) for a, b in zip(keep, X1))
