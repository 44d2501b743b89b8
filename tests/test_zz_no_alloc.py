"""dmuon_adamw_step_noalloc: the AdamW step for callers that cannot allocate device memory.

Some users of this library run it where a cudaMalloc from inside a library call is not an option: the training
framework's own allocator already holds the GPU's memory (a raw cudaMalloc then fails while the framework could still
hand out tensors), collectives are in flight on another stream (cudaMalloc / cudaFree synchronise the whole device), or
the loop simply cannot take that synchronisation.  dmuon_adamw_step allocates its per-call work table with cudaMalloc;
dmuon_adamw_step_noalloc keeps that table in a fixed 192 KiB array inside the library image instead and is limited to
DMUON_ADAMW_NOALLOC_MAX_TENSORS tensors per call.  Every call on a device shares that array, so the test below makes
two calls in a row with different tensor lists and checks each against dmuon_adamw_step on copies of the same inputs.

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests of the Muon step."""
import ctypes

import pytest
import torch

import paper_2606_27153_b200 as dm
from paper_2606_27153_b200 import binding

HYPER = dict(lr=3e-3, beta1=0.9, beta2=0.95, eps=1e-8, wd=0.1)


def _state(sizes, seed):
    g = torch.Generator(device="cuda").manual_seed(seed)
    P = [(torch.randn(s, generator=g, device="cuda") * 0.5).to(torch.bfloat16) for s in sizes]
    G = [(torch.randn(s, generator=g, device="cuda") * 1e-2).to(torch.bfloat16) for s in sizes]
    M = [torch.randn(s, generator=g, device="cuda") * 1e-2 for s in sizes]
    V = [torch.rand(s, generator=g, device="cuda") * 1e-4 for s in sizes]
    return P, G, M, V


def _clone(lists):
    return tuple([t.clone() for t in ts] for ts in lists)


@pytest.mark.gpu
def test_noalloc_adamw_equals_allocating_path_on_two_calls_in_a_row():
    """Call 1: seven tensors of ragged sizes (vector path and scalar tails), step 1.  Call 2, straight after on the same
    stream with no synchronisation in between: a different, shorter list (other tensors, other sizes) -- its table
    overwrites call 1's in the shared array.  Call 3: the first list again, step 2, so a table that was overwritten in
    between is rebuilt.  Every call must leave parameters and both moments bitwise equal to dmuon_adamw_step on copies
    of the same inputs (the two entry points run the same kernel, so the suite's AdamW tolerance -- 1 bf16 ulp on p,
    3e-7 relative on the moments -- is met with room to spare) and must never write the gradients.  Device memory in
    use must not grow across the calls that follow the first (the first one may load the kernel image)."""
    A = _state([(1000,), (3, 8192), (5,), (896,), (257, 33), (8192,), (2, 3, 7)], 9300)
    B = _state([(4864,), (129, 65), (7,)], 9301)

    ref_a, ref_b = _clone(A), _clone(B)                  # the existing, allocating path
    dm.adamw_step(*ref_a, step=1, **HYPER)
    dm.adamw_step(*ref_b, step=2, **HYPER)
    dm.adamw_step(*ref_a, step=2, **HYPER)

    new_a, new_b = _clone(A), _clone(B)
    torch.cuda.synchronize()
    dm.adamw_step_noalloc(*new_a, step=1, **HYPER)       # the first call on a device also looks up the array's address
    free_before = torch.cuda.mem_get_info()[0]
    dm.adamw_step_noalloc(*new_b, step=2, **HYPER)
    dm.adamw_step_noalloc(*new_a, step=2, **HYPER)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before, "device memory in use grew across no-alloc calls"

    for tag, new, ref, src in (("first list", new_a, ref_a, A), ("second list", new_b, ref_b, B)):
        for i in range(len(src[0])):
            assert torch.equal(new[1][i], src[1][i]), f"{tag} tensor {i}: the gradient was written"
            for name, k in (("parameter", 0), ("exp_avg", 2), ("exp_avg_sq", 3)):
                assert torch.equal(new[k][i], ref[k][i]), f"{tag} tensor {i}: {name} differs from dmuon_adamw_step"
            assert torch.isfinite(new[0][i].float()).all()
            assert not torch.equal(new[2][i], src[2][i]), f"{tag} tensor {i}: the step did not run"


def test_noalloc_adamw_rejects_lists_beyond_the_static_table():
    """More tensors than the built-in table holds: a clear DMUON_ERR_INVALID_ARG before anything touches the GPU (so
    this runs on the CPU box too); the limit in the binding is the header's."""
    L = binding.lib()
    n = binding.ADAMW_NOALLOC_MAX_TENSORS + 1
    import os
    import re
    header = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "dmuon.h")).read()
    assert int(re.search(r"#define\s+DMUON_ADAMW_NOALLOC_MAX_TENSORS\s+(\d+)", header).group(1)) == binding.ADAMW_NOALLOC_MAX_TENSORS
    ptrs = (ctypes.c_void_p * n)(*([0x10000] * n))
    numel = (ctypes.c_int64 * n)(*([8] * n))
    rc = L.dmuon_adamw_step_noalloc(ptrs, ptrs, ptrs, ptrs, numel, n, 1e-3, 0.9, 0.999, 1e-8, 0.01, 1, None)
    assert rc == binding.ERR_INVALID_ARG
    msg = binding.last_error()
    assert "dmuon_adamw_step_noalloc" in msg and str(binding.ADAMW_NOALLOC_MAX_TENSORS) in msg
    # the other argument checks of dmuon_adamw_step hold here as well
    one = (ctypes.c_void_p * 1)(0x10000)
    cnt = (ctypes.c_int64 * 1)(8)
    assert L.dmuon_adamw_step_noalloc(one, one, one, one, cnt, 1, 1e-3, 0.9, 0.999, 1e-8, 0.01, 0, None) == binding.ERR_INVALID_ARG   # step < 1
    bad = (ctypes.c_void_p * 1)(0x10008)
    assert L.dmuon_adamw_step_noalloc(bad, one, one, one, cnt, 1, 1e-3, 0.9, 0.999, 1e-8, 0.01, 1, None) == binding.ERR_INVALID_ARG   # misaligned
    assert L.dmuon_adamw_step_noalloc(None, None, None, None, None, 0, 1e-3, 0.9, 0.999, 1e-8, 0.01, 1, None) == binding.OK            # count = 0
