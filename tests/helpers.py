"""Shared helpers for the parity tests (no method arithmetic here, apart from binary32_momentum, which documents the
kernel's own precision and is never used as the expected value of a parity check)."""
import numpy as np
import torch

# tolerances of BASELINE.json north_star: relative Frobenius error against the fp64 oracle on the same inputs
TOL_TC = 1e-2       # 16-bit operands, fp32 accumulation (tensor-core path)
TOL_CHECK = 1e-4    # fp32-operand check mode

LR, MU, WD = 0.02, 0.95, 0.01      # BASELINE.json configs[1]
MU_F = float(np.float32(MU))       # the values the C ABI receives (floats)
LR_F = float(np.float32(LR))
WD_F = float(np.float32(WD))


def to64(t: torch.Tensor) -> np.ndarray:
    """Exact bf16/fp16/fp32 tensor -> float64 numpy (host)."""
    return t.detach().to("cpu").to(torch.float64).numpy()


def rel_fro(a: np.ndarray, b: np.ndarray) -> float:
    """||a - b||_F / ||b||_F  (b = oracle)."""
    den = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / (den if den > 0 else 1.0))


def binary32_momentum(M: np.ndarray, G: np.ndarray, mu: float):
    """What the tensor-core path's a1 kernel is documented to form (N16): M' = fma(mu, M, G) and
    U = fma(mu, M', G) in binary32, one rounding each.  mu*M + G is exact in float64 for a 24-bit mu and bf16 M, G of
    comparable scale, so rounding it once to float32 is the fused result.  A statement about the KERNEL's precision kept
    beside the tests; the oracle holds only the paper's real-arithmetic definition and knows nothing of this."""
    mn = (mu * M + G).astype(np.float32)
    u = (mu * mn.astype(np.float64) + G).astype(np.float32)
    return mn.astype(np.float64), u.astype(np.float64)


def bf16_ulp(x: np.ndarray) -> np.ndarray:
    """Spacing of bf16 at |x| (normal range)."""
    ax = np.maximum(np.abs(x), 2.0 ** -126)
    return 2.0 ** (np.floor(np.log2(ax)) - 7)


W_USED = []      # (err - r) / (tol * upd) per checked matrix: the share of the update allowance a W' check used


def w_bound(w_gpu: np.ndarray, w_orc: np.ndarray, w_before: np.ndarray, tol: float, round_bf16) -> tuple:
    """(err, bound) of the stored parameter against the oracle's unrounded W' (DESIGN.md section 5 derives it):
    err = ||W'_gpu - w_orc||, bound = (1 + s) r + tol ||w_orc - W||, r = ||RNE_bf16(w_orc) - w_orc|| the rounding the
    oracle's own result takes when stored.  s = min(0.02, 4 / sqrt(N)): the GPU rounds ITS unrounded value, another
    draw of the same rounding-error distribution, whose norm differs from r by a relative 0.63 / sqrt(N) (one sigma)."""
    r = np.linalg.norm(round_bf16(w_orc) - w_orc)
    upd = np.linalg.norm(w_orc - w_before)
    err = np.linalg.norm(w_gpu - w_orc)
    s = min(0.02, 4.0 / np.sqrt(w_orc.size))
    if upd > 0:
        W_USED.append(float((err - r) / (tol * upd)))
    return err, (1.0 + s) * r + tol * upd
