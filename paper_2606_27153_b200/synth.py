"""Seeded synthetic inputs shaped like BASELINE.json's configs (recipe: DESIGN.md "Input recipe").

This module holds NONE of the method's arithmetic: it only draws random matrices.  It is the one
module both the tests' oracle side and the CUDA side use, so that the two see the same bits: the
tensors it returns are bf16, and the oracle is always fed the exact bf16 values read back from them.

The paper's own workloads (Wall-OSS-0.5 / Pi0 / Wall-WM / Qwen2.5-7B training runs) are not
available; these LLM-shaped matrix sets stand in for them and use only public architecture dimensions.
"""
from __future__ import annotations

import math
from typing import List, Tuple

import torch

Shape = Tuple[int, int]

SIGMA_G = 1e-3      # noise std of a gradient (configs[1])
LOW_RANK = 8        # rank of the ill-conditioning component
LOW_RANK_ENERGY = 10.0  # its energy relative to the noise
SIGMA_W = 0.02      # weight std


def config_shapes(config: int) -> List[Shape]:
    """(rows, cols) of every 2-D weight, in layer order (BASELINE.json configs[config-1])."""
    if config == 1:
        return [(128, 512)] * 8
    if config == 2:      # GPT-2-small-shaped, 12 layers, d = 768
        layer = [(768, 768)] * 4 + [(3072, 768), (768, 3072)]
        return layer * 12
    if config == 3:      # Qwen-0.5B-style, 24 layers, d = 896, GQA
        layer = [(896, 896), (128, 896), (128, 896), (896, 896), (4864, 896), (4864, 896), (896, 4864)]
        return layer * 24
    if config == 4:      # Llama-3-8B-shaped, 32 layers
        layer = [(4096, 4096), (1024, 4096), (1024, 4096), (4096, 4096), (14336, 4096), (14336, 4096),
                 (4096, 14336)]
        return layer * 32
    raise ValueError("config must be 1..4 (config 5 is a sweep: see sweep_shapes)")


def sweep_shapes() -> List[Tuple[Shape, int]]:
    """configs[4]: ((rows, cols), batch) per sweep point; batch = 2^32 / n^2 for the squares (reading N13)."""
    out = [((n, n), (1 << 32) // (n * n)) for n in (256, 512, 1024, 2048, 4096, 8192)]
    out += [((2048, 2048 * r), 16) for r in (1, 2, 4, 8)]
    out += [((2048, 1408), 64), ((1408, 2048), 64)]
    return out


def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def iid_scaled(shape: Shape, seed: int, device="cpu", log10_lo=-3.0, log10_hi=1.0) -> torch.Tensor:
    """configs[0]: Z * 10^u, Z iid N(0,1), u ~ U(log10_lo, log10_hi) per matrix; bf16."""
    g = _gen(seed, device)
    u = torch.rand((), generator=g, device=device).item() * (log10_hi - log10_lo) + log10_lo
    z = torch.randn(shape, generator=g, device=device, dtype=torch.float32)
    return (z * (10.0 ** u)).to(torch.bfloat16)


def iid_normal(shape: Shape, seed: int, device="cpu", std: float = 1.0) -> torch.Tensor:
    g = _gen(seed, device)
    return (torch.randn(shape, generator=g, device=device, dtype=torch.float32) * std).to(torch.bfloat16)


def gradient(shape: Shape, seed: int, device="cpu") -> torch.Tensor:
    """configs[1]: N(0, 1e-3^2) noise plus a rank-8 component of 10x the noise energy; bf16."""
    r, c = shape
    g = _gen(seed, device)
    z = torch.randn((r, c), generator=g, device=device, dtype=torch.float32)
    p = torch.randn((r, LOW_RANK), generator=g, device=device, dtype=torch.float32)
    q = torch.randn((c, LOW_RANK), generator=g, device=device, dtype=torch.float32)
    alpha = SIGMA_G * math.sqrt(LOW_RANK_ENERGY / LOW_RANK)
    return (SIGMA_G * z + alpha * (p @ q.t())).to(torch.bfloat16)


def weight(shape: Shape, seed: int, device="cpu") -> torch.Tensor:
    return iid_normal(shape, seed, device, SIGMA_W)


def seed_for(config: int, index: int, stream: int = 0) -> int:
    """seed = 1000*config + matrix index; `stream` separates G (0), W (1), M (2) of one matrix."""
    return 1000 * config + index + 1_000_000 * stream


def muon_inputs(config: int, device="cpu", random_momentum: bool = False, indices=None):
    """(shapes, W, G, M) lists for a Muon-step config (2, 3 or 4).  M = 0 as in configs[1] unless
    random_momentum (then M ~ the gradient recipe with another seed)."""
    shapes = config_shapes(config)
    idx = range(len(shapes)) if indices is None else indices
    S, W, G, M = [], [], [], []
    for i in idx:
        s = shapes[i]
        S.append(s)
        G.append(gradient(s, seed_for(config, i, 0), device))
        W.append(weight(s, seed_for(config, i, 1), device))
        if random_momentum:
            M.append(gradient(s, seed_for(config, i, 2), device))
        else:
            M.append(torch.zeros(s, dtype=torch.bfloat16, device=device))
    return S, W, G, M


def ns_inputs(device="cpu"):
    """configs[0]: the tiny NS batch, 8 x (128 x 512)."""
    shapes = config_shapes(1)
    return shapes, [iid_scaled(s, seed_for(1, i), device) for i, s in enumerate(shapes)]


# ---------------------------------------------------------------- hostile spectra (Gram-block error study)
def with_spectrum(shape: Shape, sigmas: torch.Tensor, seed: int, device="cpu") -> torch.Tensor:
    """A matrix with prescribed singular values: Q1 diag(sigmas) Q2^T with Haar-like orthonormal factors (QR of
    Gaussians), rounded to bf16.  len(sigmas) = min(shape)."""
    r, c = shape
    m = min(r, c)
    g = _gen(seed, device)
    q1, _ = torch.linalg.qr(torch.randn((r, m), generator=g, device=device, dtype=torch.float64))
    q2, _ = torch.linalg.qr(torch.randn((c, m), generator=g, device=device, dtype=torch.float64))
    return ((q1 * sigmas.to(device=device, dtype=torch.float64)) @ q2.t()).to(torch.float32).to(torch.bfloat16)


def hostile_inputs(shape: Shape, seed: int, device="cpu"):
    """(name, matrix) pairs that stress 16-bit Newton-Schulz and the Gram-space recurrence in particular: spectra with a
    huge dynamic range, clusters at both ends, low rank plus rounding noise, extreme overall scales."""
    r, c = shape
    m = min(r, c)
    out = []
    gen = _gen(seed, device)
    z = torch.randn((r, c), generator=gen, device=device, dtype=torch.float32)
    p = torch.randn((r, LOW_RANK), generator=gen, device=device, dtype=torch.float32)
    q = torch.randn((c, LOW_RANK), generator=gen, device=device, dtype=torch.float32)
    out.append(("rank8_energy_1000x", (SIGMA_G * z + SIGMA_G * math.sqrt(1000.0 / LOW_RANK) * (p @ q.t())).to(torch.bfloat16)))
    out.append(("geometric_decay_1_to_1e-6", with_spectrum(shape, torch.logspace(0, -6, m, dtype=torch.float64), seed + 1, device)))
    half = torch.cat([torch.ones(m // 2, dtype=torch.float64), torch.full((m - m // 2,), 1e-4, dtype=torch.float64)])
    out.append(("half_converged_half_tiny", with_spectrum(shape, half, seed + 2, device)))
    out.append(("exact_rank8_plus_bf16_noise", (p @ q.t()).to(torch.bfloat16)))
    out.append(("iid_scale_1e-3", (z * 1e-3).to(torch.bfloat16)))
    out.append(("iid_scale_1e1", (z * 1e1).to(torch.bfloat16)))
    two = torch.cat([torch.full((m // 16,), 1.0, dtype=torch.float64), torch.full((m - m // 16,), 0.02, dtype=torch.float64)])
    out.append(("spikes_over_flat_bulk", with_spectrum(shape, two, seed + 3, device)))
    return out
