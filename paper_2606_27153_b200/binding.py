"""Thin ctypes binding over libdmuon.so (include/dmuon.h).  Argument marshalling only: every step of the path
runs in the library's CUDA kernels.  There is no fallback: if the library is missing, loading raises."""
from __future__ import annotations

import ctypes
import json
import os
from typing import Iterable, List, Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("DMUON_LIB") or os.path.join(_HERE, "libdmuon.so")      # DMUON_LIB: another build of the same library (A/B measurements)

OK = 0
ERR_INVALID_ARG = -1
ERR_UNSUPPORTED_DEVICE = -2
ERR_OOM = -3
ERR_CUDA = -4
ERR_INTERNAL = -5

OP_SYRK, OP_SQ, OP_BX, OP_SYRK_T, OP_XB = 0, 1, 2, 4, 5

#: every symbol include/dmuon.h declares
SYMBOLS = ("dmuon_ns_batched", "dmuon_ns_batched_sched", "dmuon_muon_step", "dmuon_muon_step_host", "dmuon_warmup",
           "dmuon_workspace_bytes", "dmuon_set_workspace", "dmuon_set_option", "dmuon_last_error",
           "dmuon_profile_read", "dmuon_profile_reset", "dmuon_ns_gemm", "dmuon_ns_gemm_variants", "dmuon_read_ns_output", "dmuon_shutdown",
           "dmuon_version", "dmuon_describe_plan", "dmuon_ns_sym_mm", "dmuon_block_schedule", "dmuon_muon_step_master",
           "dmuon_adamw_step", "dmuon_adamw_step_noalloc", "dmuon_measure_cost", "dmuon_assign_owners")


class DmuonError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"libdmuon error {code}: {message}")
        self.code = code


_lib = None


def lib() -> ctypes.CDLL:
    """Load libdmuon.so (built by paper_2606_27153_b200.build).  Fails loudly if it is not there."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2606_27153_b200.build` "
                              "(there is no CPU or PyTorch fallback for the Muon step)")
        L = ctypes.CDLL(LIB_PATH)
        vp, i32, f32 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_float
        pp = ctypes.POINTER(ctypes.c_void_p)
        pi = ctypes.POINTER(ctypes.c_int32)
        pf = ctypes.POINTER(ctypes.c_float)
        L.dmuon_ns_batched.argtypes = [pp, pi, i32, i32, pf, vp]
        L.dmuon_ns_batched_sched.argtypes = [pp, pi, i32, i32, pf, vp]
        L.dmuon_muon_step.argtypes = [pp, pp, pp, pi, i32, f32, f32, f32, vp]
        L.dmuon_muon_step_master.argtypes = [pp, pp, pp, pp, pi, i32, f32, f32, f32, vp]
        L.dmuon_muon_step_host.argtypes = [pp, pp, pp, pi, i32, f32, f32, f32, vp]
        L.dmuon_warmup.argtypes = [pi, i32, vp]
        L.dmuon_workspace_bytes.argtypes = [pi, i32]
        L.dmuon_workspace_bytes.restype = ctypes.c_size_t
        L.dmuon_set_workspace.argtypes = [vp, ctypes.c_size_t]
        L.dmuon_set_option.argtypes = [ctypes.c_char_p, ctypes.c_char_p]
        L.dmuon_last_error.restype = ctypes.c_char_p
        L.dmuon_profile_read.argtypes = [ctypes.c_char_p, ctypes.c_size_t]
        L.dmuon_ns_gemm.argtypes = [i32, pp, pp, pp, i32, i32, i32, f32, f32, i32, vp]
        L.dmuon_ns_gemm_variants.argtypes = [i32]
        L.dmuon_ns_sym_mm.argtypes = [pp, pp, pp, pp, pp, i32, i32, f32, f32, f32, i32, vp]
        L.dmuon_block_schedule.argtypes = [i32, i32, i32, pf, i32, pi, i32]
        L.dmuon_describe_plan.argtypes = [pi, i32, i32, ctypes.c_char_p, ctypes.c_size_t, vp]
        L.dmuon_read_ns_output.argtypes = [i32, vp, vp]
        pl = ctypes.POINTER(ctypes.c_int64)
        pd = ctypes.POINTER(ctypes.c_double)
        L.dmuon_adamw_step.argtypes = [pp, pp, pp, pp, pl, i32, f32, f32, f32, f32, f32, i32, vp]
        L.dmuon_adamw_step_noalloc.argtypes = L.dmuon_adamw_step.argtypes
        L.dmuon_measure_cost.argtypes = [i32, i32, i32, i32, pf, vp]
        L.dmuon_assign_owners.argtypes = [pi, pi, pi, pd, i32, i32, i32, i32, pi, pd]
        L.dmuon_shutdown.restype = None
        L.dmuon_version.restype = ctypes.c_char_p
        for name in SYMBOLS:
            fn = getattr(L, name)
            if fn.restype is ctypes.c_int and name not in ("dmuon_shutdown",):
                fn.restype = ctypes.c_int
        _lib = L
    return _lib


def _check(rc: int) -> None:
    if rc != OK:
        raise DmuonError(rc, lib().dmuon_last_error().decode())


def _stream(stream) -> ctypes.c_void_p:
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
    elif isinstance(stream, torch.cuda.Stream):
        stream = stream.cuda_stream
    return ctypes.c_void_p(int(stream))


def _ptr_array(tensors: Sequence[torch.Tensor]):
    return (ctypes.c_void_p * len(tensors))(*[t.data_ptr() for t in tensors])


def _shape_array(shapes: Iterable[Sequence[int]]):
    flat: List[int] = []
    for s in shapes:
        flat += [int(s[0]), int(s[1])]
    return (ctypes.c_int32 * len(flat))(*flat), len(flat) // 2


def _check_mats(tensors: Sequence[torch.Tensor], device_type: str, what: str) -> None:
    for i, t in enumerate(tensors):
        if t.dim() != 2 or t.dtype != torch.bfloat16 or not t.is_contiguous() or t.device.type != device_type:
            raise ValueError(f"{what}[{i}] must be a contiguous 2-D bfloat16 {device_type} tensor")


class Marshalled:
    """The C arguments of a tensor list (pointer array, shape array, count), built once by marshal() and reusable for any
    number of calls: for tens of thousands of small matrices building them costs more host time than the GPU call
    itself.  Holds the tensors, so the pointers stay valid as long as this object lives."""

    def __init__(self, tensors: Sequence[torch.Tensor], device_type: str = "cuda", what: str = "tensors"):
        self.tensors = list(tensors)
        _check_mats(self.tensors, device_type, what)
        self.ptrs = _ptr_array(self.tensors)
        self.shapes, self.count = _shape_array([t.shape for t in self.tensors])


def marshal(tensors: Sequence[torch.Tensor]) -> Marshalled:
    return tensors if isinstance(tensors, Marshalled) else Marshalled(tensors)


# ---------------------------------------------------------------- entry points (names follow include/dmuon.h)

def version() -> str:
    return lib().dmuon_version().decode()


def last_error() -> str:
    return lib().dmuon_last_error().decode()


def set_option(key: str, value) -> None:
    _check(lib().dmuon_set_option(key.encode(), str(value).encode()))


def ns_batched(tensors: Sequence[torch.Tensor], steps: int = 5, coeffs: Optional[Sequence[float]] = None, stream=None) -> None:
    """dmuon_ns_batched: each tensor is overwritten by NS_steps(X / (||X||_F + 1e-7)).  `tensors`: a list of tensors or
    the Marshalled form of one (marshal())."""
    a = marshal(tensors)
    co = (ctypes.c_float * 3)(*coeffs) if coeffs is not None else None
    _check(lib().dmuon_ns_batched(a.ptrs, a.shapes, a.count, int(steps), co, _stream(stream)))


def ns_batched_sched(tensors: Sequence[torch.Tensor], coeffs: Sequence[Sequence[float]], stream=None) -> None:
    """dmuon_ns_batched_sched: one (a, b, c) per step."""
    a = marshal(tensors)
    flat = [float(v) for row in coeffs for v in row]
    co = (ctypes.c_float * len(flat))(*flat)
    _check(lib().dmuon_ns_batched_sched(a.ptrs, a.shapes, a.count, len(coeffs), co, _stream(stream)))


def muon_step(params: Sequence[torch.Tensor], grads: Sequence[torch.Tensor], momenta: Sequence[torch.Tensor],
              lr: float, mu: float, wd: float, stream=None) -> None:
    """dmuon_muon_step: params and momenta updated in place; grads read only."""
    if not (len(params) == len(grads) == len(momenta)):
        raise ValueError("params, grads, momenta must have one length")
    for name, ts in (("params", params), ("grads", grads), ("momenta", momenta)):
        _check_mats(ts, "cuda", name)
    for p, g, m in zip(params, grads, momenta):
        if p.shape != g.shape or p.shape != m.shape:
            raise ValueError("param / grad / momentum shapes differ")
    shp, n = _shape_array([t.shape for t in params])
    _check(lib().dmuon_muon_step(_ptr_array(params), _ptr_array(grads), _ptr_array(momenta), shp, n, float(lr),
                                 float(mu), float(wd), _stream(stream)))


def muon_step_master(params: Sequence[torch.Tensor], masters: Sequence[torch.Tensor], grads: Sequence[torch.Tensor],
                     momenta: Sequence[torch.Tensor], lr: float, mu: float, wd: float, stream=None) -> None:
    """dmuon_muon_step_master: fp32 masters and momenta updated in place, params overwritten with bf16(master)."""
    if not (len(params) == len(masters) == len(grads) == len(momenta)):
        raise ValueError("params, masters, grads, momenta must have one length")
    for name, ts in (("params", params), ("grads", grads), ("momenta", momenta)):
        _check_mats(ts, "cuda", name)
    for i, (p, w) in enumerate(zip(params, masters)):
        if w.dtype != torch.float32 or not w.is_contiguous() or w.device.type != "cuda" or w.shape != p.shape:
            raise ValueError(f"masters[{i}] must be a contiguous float32 cuda tensor of the parameter's shape")
    shp, n = _shape_array([t.shape for t in params])
    _check(lib().dmuon_muon_step_master(_ptr_array(params), _ptr_array(masters), _ptr_array(grads), _ptr_array(momenta),
                                        shp, n, float(lr), float(mu), float(wd), _stream(stream)))


def muon_step_host(params: Sequence[torch.Tensor], grads: Sequence[torch.Tensor], momenta: Sequence[torch.Tensor],
                   lr: float, mu: float, wd: float, stream=None) -> None:
    """dmuon_muon_step_host: the same step for HOST tensors (pinned for asynchronous copies)."""
    for name, ts in (("params", params), ("grads", grads), ("momenta", momenta)):
        _check_mats(ts, "cpu", name)
    shp, n = _shape_array([t.shape for t in params])
    _check(lib().dmuon_muon_step_host(_ptr_array(params), _ptr_array(grads), _ptr_array(momenta), shp, n, float(lr),
                                      float(mu), float(wd), _stream(stream)))


def warmup(shapes: Sequence[Sequence[int]], stream=None) -> None:
    shp, n = _shape_array(shapes)
    _check(lib().dmuon_warmup(shp, n, _stream(stream)))


def workspace_bytes(shapes: Sequence[Sequence[int]]) -> int:
    shp, n = _shape_array(shapes)
    return int(lib().dmuon_workspace_bytes(shp, n))


def set_workspace(buf: Optional[torch.Tensor]) -> None:
    if buf is None:
        _check(lib().dmuon_set_workspace(None, 0))
    else:
        _check(lib().dmuon_set_workspace(ctypes.c_void_p(buf.data_ptr()), buf.numel() * buf.element_size()))


def profile_reset() -> None:
    _check(lib().dmuon_profile_reset())


def profile_read() -> dict:
    buf = ctypes.create_string_buffer(1 << 16)
    rc = lib().dmuon_profile_read(buf, len(buf))
    if rc < 0:
        _check(rc)
    return json.loads(buf.value.decode())


def ns_gemm(op: int, in0: Sequence[torch.Tensor], in1: Optional[Sequence[torch.Tensor]], out: Sequence[torch.Tensor],
            alpha: float, beta: float, variant: int = -1, stream=None) -> None:
    """dmuon_ns_gemm: one grouped launch of an NS product on fp16 matrices (dims multiples of 128)."""
    for ts in (in0, in1 or [], out):
        for t in ts:
            if t.dtype != torch.float16 or not t.is_contiguous() or t.device.type != "cuda" or t.dim() != 2:
                raise ValueError("ns_gemm takes contiguous 2-D float16 cuda tensors")
    if op == OP_SYRK_T:                      # in0 = Y [n x m]
        m, n = in0[0].shape[1], in0[0].shape[0]
    elif op == OP_XB:                        # in0 = B [m x m], in1 = Y [n x m]
        m, n = in0[0].shape[0], out[0].shape[0]
    else:
        m = in0[0].shape[0]
        n = in0[0].shape[1] if op == OP_SYRK else (out[0].shape[1] if op == OP_BX else m)
    _check(lib().dmuon_ns_gemm(op, _ptr_array(in0), _ptr_array(in1) if in1 else None, _ptr_array(out), m, n, len(in0),
                               float(alpha), float(beta), int(variant), _stream(stream)))


def ns_sym_mm(a: Sequence[torch.Tensor], b: Sequence[torch.Tensor], d: Optional[Sequence[torch.Tensor]],
              d2: Optional[Sequence[torch.Tensor]], out: Sequence[torch.Tensor], alpha: float, beta: float = 0.0,
              beta2: float = 0.0, variant: int = -1, stream=None) -> None:
    """dmuon_ns_sym_mm: out = alpha a b^T + beta d + beta2 d2 on fp16 m x m matrices (symmetric result)."""
    for ts in (a, b, d or [], d2 or [], out):
        for t in ts:
            if t.dtype != torch.float16 or not t.is_contiguous() or t.device.type != "cuda" or t.dim() != 2:
                raise ValueError("ns_sym_mm takes contiguous 2-D float16 cuda tensors")
    _check(lib().dmuon_ns_sym_mm(_ptr_array(a), _ptr_array(b), _ptr_array(d) if d else None,
                                 _ptr_array(d2) if d2 else None, _ptr_array(out), a[0].shape[0], len(a), float(alpha),
                                 float(beta), float(beta2), int(variant), _stream(stream)))


def block_schedule(shape: Sequence[int], steps: int = 5, coeffs: Optional[Sequence] = None) -> List[int]:
    """dmuon_block_schedule (host only): block lengths for one matrix; coeffs = (a, b, c) or one triple per step."""
    per_step, co = 0, None
    if coeffs is not None:
        per_step = int(len(coeffs) > 0 and hasattr(coeffs[0], "__len__"))
        flat = [float(v) for row in coeffs for v in row] if per_step else [float(v) for v in coeffs]
        co = (ctypes.c_float * len(flat))(*flat)
    out = (ctypes.c_int32 * 64)()
    rc = lib().dmuon_block_schedule(int(shape[0]), int(shape[1]), int(steps), co, per_step, out, 64)
    if rc < 0:
        _check(rc)
    return [int(out[i]) for i in range(rc)]


def describe_plan(shapes: Sequence[Sequence[int]], steps: int = 5, stream=None) -> dict:
    """dmuon_describe_plan: buckets, block schedule and tile variants the library uses for this shape set."""
    shp, n = _shape_array(shapes)
    buf = ctypes.create_string_buffer(1 << 16)
    rc = lib().dmuon_describe_plan(shp, n, int(steps), buf, len(buf), _stream(stream))
    if rc < 0:
        _check(rc)
    return json.loads(buf.value.decode())


def read_ns_output(index: int, shape: Sequence[int], stream=None) -> torch.Tensor:
    """dmuon_read_ns_output: the unrounded NS result of matrix `index` of the last call, as an fp32 cuda tensor."""
    out = torch.empty(tuple(shape), dtype=torch.float32, device="cuda")
    _check(lib().dmuon_read_ns_output(int(index), ctypes.c_void_p(out.data_ptr()), _stream(stream)))
    return out


def adamw_step(params: Sequence[torch.Tensor], grads: Sequence[torch.Tensor], exp_avg: Sequence[torch.Tensor],
               exp_avg_sq: Sequence[torch.Tensor], lr: float, beta1: float, beta2: float, eps: float, wd: float, step: int,
               stream=None) -> None:
    """dmuon_adamw_step: decoupled AdamW over non-matrix parameters (bf16 p, g; fp32 moments), any shapes."""
    n = len(params)
    if not (len(grads) == len(exp_avg) == len(exp_avg_sq) == n):
        raise ValueError("params, grads, exp_avg, exp_avg_sq must have one length")
    for i in range(n):
        p, g, m, v = params[i], grads[i], exp_avg[i], exp_avg_sq[i]
        if p.dtype != torch.bfloat16 or g.dtype != torch.bfloat16 or m.dtype != torch.float32 or v.dtype != torch.float32:
            raise ValueError(f"tensor {i}: params/grads must be bfloat16, moments float32")
        if not (p.is_contiguous() and g.is_contiguous() and m.is_contiguous() and v.is_contiguous()):
            raise ValueError(f"tensor {i}: tensors must be contiguous")
        if not (p.numel() == g.numel() == m.numel() == v.numel()) or any(t.device.type != "cuda" for t in (p, g, m, v)):
            raise ValueError(f"tensor {i}: sizes differ or not on cuda")
    numel = (ctypes.c_int64 * n)(*[p.numel() for p in params])
    _check(lib().dmuon_adamw_step(_ptr_array(params), _ptr_array(grads), _ptr_array(exp_avg), _ptr_array(exp_avg_sq),
                                  numel, n, float(lr), float(beta1), float(beta2), float(eps), float(wd), int(step),
                                  _stream(stream)))


ADAMW_NOALLOC_MAX_TENSORS = 4096      # DMUON_ADAMW_NOALLOC_MAX_TENSORS


def adamw_step_noalloc(params: Sequence[torch.Tensor], grads: Sequence[torch.Tensor], exp_avg: Sequence[torch.Tensor],
                       exp_avg_sq: Sequence[torch.Tensor], lr: float, beta1: float, beta2: float, eps: float, wd: float,
                       step: int, stream=None) -> None:
    """dmuon_adamw_step_noalloc: adamw_step for processes where the library must not call cudaMalloc (a framework pool
    owns the GPU's memory, collectives are in flight, or the loop cannot take the device-wide synchronisation).  Same
    results; at most ADAMW_NOALLOC_MAX_TENSORS tensors per call; the per-call table sits in a fixed 192 KiB array inside
    the library that every call on the device shares, so keep these calls on one stream.  The first call on a device
    does a one-time address lookup: make it at start-up."""
    n = len(params)
    if not (len(grads) == len(exp_avg) == len(exp_avg_sq) == n):
        raise ValueError("params, grads, exp_avg, exp_avg_sq must have one length")
    for i in range(n):
        p, g, m, v = params[i], grads[i], exp_avg[i], exp_avg_sq[i]
        if p.dtype != torch.bfloat16 or g.dtype != torch.bfloat16 or m.dtype != torch.float32 or v.dtype != torch.float32:
            raise ValueError(f"tensor {i}: params/grads must be bfloat16, moments float32")
        if not (p.is_contiguous() and g.is_contiguous() and m.is_contiguous() and v.is_contiguous()):
            raise ValueError(f"tensor {i}: tensors must be contiguous")
        if not (p.numel() == g.numel() == m.numel() == v.numel()) or any(t.device.type != "cuda" for t in (p, g, m, v)):
            raise ValueError(f"tensor {i}: sizes differ or not on cuda")
    numel = (ctypes.c_int64 * n)(*[p.numel() for p in params])
    _check(lib().dmuon_adamw_step_noalloc(_ptr_array(params), _ptr_array(grads), _ptr_array(exp_avg),
                                          _ptr_array(exp_avg_sq), numel, n, float(lr), float(beta1), float(beta2),
                                          float(eps), float(wd), int(step), _stream(stream)))


def measure_cost(shape: Sequence[int], batch: int, reps: int = 3, stream=None) -> float:
    """dmuon_measure_cost: c_{s,b} (ms) of one batch of `batch` matrices of `shape` through the whole Muon step."""
    out = ctypes.c_float(0.0)
    _check(lib().dmuon_measure_cost(int(shape[0]), int(shape[1]), int(batch), int(reps), ctypes.byref(out), _stream(stream)))
    return float(out.value)


def assign_owners(counts: Sequence[int], batch_sizes: Sequence[Sequence[int]], costs: Sequence[Sequence[float]],
                  num_ranks: int, mode: int = -1, threshold: int = 64):
    """dmuon_assign_owners (host only).  batch_sizes[s], costs[s]: candidate batch sizes of shape s and their measured
    costs.  Returns (x, makespan, exact) with x[s][j][r] = batches of batch_sizes[s][j] given to rank r."""
    S = len(counts)
    nb = [len(b) for b in batch_sizes]
    flat_b = [int(v) for b in batch_sizes for v in b]
    flat_c = [float(v) for c in costs for v in c]
    if len(flat_b) != len(flat_c):
        raise ValueError("batch_sizes and costs must have one shape")
    K = len(flat_b)
    x = (ctypes.c_int32 * max(1, K * num_ranks))()
    ms = ctypes.c_double(0.0)
    rc = lib().dmuon_assign_owners((ctypes.c_int32 * max(1, S))(*[int(c) for c in counts]), (ctypes.c_int32 * max(1, S))(*nb),
                                   (ctypes.c_int32 * max(1, K))(*flat_b), (ctypes.c_double * max(1, K))(*flat_c), S,
                                   int(num_ranks), int(mode), int(threshold), x, ctypes.byref(ms))
    if rc < 0:
        _check(rc)
    out, k = [], 0
    for s in range(S):
        rows = []
        for _ in range(nb[s]):
            rows.append([int(x[k * num_ranks + r]) for r in range(num_ranks)])
            k += 1
        out.append(rows)
    return out, float(ms.value), bool(rc == 1)


def ns_gemm_variants(op: int) -> int:
    return int(lib().dmuon_ns_gemm_variants(op))


def shutdown() -> None:
    lib().dmuon_shutdown()
