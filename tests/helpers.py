"""Shared helpers for the parity tests (no method arithmetic here)."""
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


def bf16_ulp(x: np.ndarray) -> np.ndarray:
    """Spacing of bf16 at |x| (normal range)."""
    ax = np.maximum(np.abs(x), 2.0 ** -126)
    return 2.0 ** (np.floor(np.log2(ax)) - 7)
