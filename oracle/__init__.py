"""fp64 CPU oracle for the DMuon Muon step -- TEST INFRASTRUCTURE, not the product.

Only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` / ``--impl reference`` legs
of ``bench.py`` may import this package.  ``paper_2606_27153_b200`` never does.

The arithmetic lives in ``dmuon_oracle.c`` (plain fp64 C, written from PAPER.md Eq. 1, Eq. 2 and
the Gram form of section 3.3); this module only builds it with gcc, loads it with ctypes and
marshals numpy float64 arrays.  See the header of the C file for what is pinned and what is not.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "dmuon_oracle.c")
_LIB = os.path.join(_HERE, "libdmuon_oracle.so")

#: the standard quintic (BASELINE.json north_star; "standard (a, b, c)-quintic")
DEFAULT_COEFFS = (3.4445, -4.7750, 2.0315)
DEFAULT_EPS = 1e-7

_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle (x86-64-v3 so the binary runs on any recent host, not just this one)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O3", "-march=x86-64-v3", "-fopenmp", "-fPIC", "-shared", "-fvisibility=hidden",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_round_bf16.restype = ctypes.c_double
        lib.oracle_round_bf16.argtypes = [ctypes.c_double]
        lib.oracle_round_bf16_array.restype = None
        lib.oracle_round_bf16_array.argtypes = [dp, dp, ctypes.c_longlong]
        lib.oracle_fro_norm.restype = ctypes.c_double
        lib.oracle_fro_norm.argtypes = [dp, ctypes.c_longlong]
        lib.oracle_ns.restype = ctypes.c_int
        lib.oracle_ns.argtypes = [dp, ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, ctypes.c_int,
                                  ctypes.c_int, ctypes.c_double, dp]
        lib.oracle_muon_step.restype = ctypes.c_int
        lib.oracle_muon_step.argtypes = [dp, dp, dp, ctypes.c_int, ctypes.c_int, ctypes.c_double,
                                         ctypes.c_double, ctypes.c_double, ctypes.c_int, dp, ctypes.c_int,
                                         ctypes.c_double, ctypes.c_int, dp, dp, dp, dp]
        lib.oracle_adamw_step.restype = ctypes.c_int
        lib.oracle_adamw_step.argtypes = [dp, dp, dp, dp, ctypes.c_longlong, ctypes.c_double, ctypes.c_double,
                                          ctypes.c_double, ctypes.c_double, ctypes.c_double, ctypes.c_int, dp, dp, dp]
        _lib = lib
    return _lib


def _ptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if a is not None else None


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def round_bf16(x):
    """Elementwise fp64 -> nearest bf16 value (ties to even), returned as float64."""
    x = np.ascontiguousarray(x, dtype=np.float64)
    out = np.empty_like(x)
    _load().oracle_round_bf16_array(_ptr(x), _ptr(out), x.size)
    return out


def _coeff_array(coeffs, steps):
    c = np.ascontiguousarray(np.asarray(coeffs, dtype=np.float64))
    if c.shape == (3,):
        return c, 0
    if c.shape == (steps, 3):
        return c.reshape(-1).copy(), 1
    raise ValueError("coeffs must have shape (3,) or (steps, 3)")


def ns(X, steps: int = 5, coeffs=DEFAULT_COEFFS, eps: float = DEFAULT_EPS, normalize: bool = True,
       return_A1: bool = False):
    """NS_steps(X) (Eq. 2 in the Gram form of :170).  X: 2-D float64; returns a new array."""
    X = np.array(X, dtype=np.float64, order="C", copy=True)
    if X.ndim != 2:
        raise ValueError("X must be 2-D")
    r, c = X.shape
    co, per = _coeff_array(coeffs, steps)
    A1 = np.zeros((min(r, c), min(r, c))) if return_A1 else None
    rc = _load().oracle_ns(_ptr(X), r, c, int(steps), _ptr(co), per, int(bool(normalize)), float(eps), _ptr(A1))
    if rc != 0:
        raise RuntimeError("oracle_ns failed")
    return (X, A1) if return_A1 else X


def muon_step(W, G, M, lr: float, mu: float, wd: float, steps: int = 5, coeffs=DEFAULT_COEFFS,
              eps: float = DEFAULT_EPS, u_cast: bool = True):
    """One Muon step (Eq. 1, Alg. 1 l.12-15).  Returns dict with M_new, U, O, W_new (float64,
    unrounded except U when u_cast).  M' and U are formed in float64 (PAPER.md:49-51 defines them in real arithmetic)."""
    W = np.ascontiguousarray(W, dtype=np.float64)
    G = np.ascontiguousarray(G, dtype=np.float64)
    M = np.ascontiguousarray(M, dtype=np.float64)
    if W.ndim != 2 or W.shape != G.shape or W.shape != M.shape:
        raise ValueError("W, G, M must be 2-D with one shape")
    r, c = W.shape
    co, per = _coeff_array(coeffs, steps)
    Mo, U, O, Wo = (np.empty((r, c)) for _ in range(4))
    rc = _load().oracle_muon_step(_ptr(W), _ptr(G), _ptr(M), r, c, float(lr), float(mu), float(wd), int(steps),
                                  _ptr(co), per, float(eps), int(bool(u_cast)), _ptr(Mo), _ptr(U),
                                  _ptr(O), _ptr(Wo))
    if rc != 0:
        raise RuntimeError("oracle_muon_step failed")
    return {"M_new": Mo, "U": U, "O": O, "W_new": Wo}


def adamw_step(p, g, m, v, lr: float, beta1: float, beta2: float, eps: float, wd: float, step: int):
    """One decoupled-AdamW step (reading N17 of DESIGN.md) in float64.  Returns (p_new, m_new, v_new),
    unrounded; the caller rounds p_new with round_bf16 to get the stored parameter."""
    arrs = [np.ascontiguousarray(a, dtype=np.float64).reshape(-1) for a in (p, g, m, v)]
    n = arrs[0].size
    if any(a.size != n for a in arrs):
        raise ValueError("p, g, m, v must have one size")
    po, mo, vo = (np.empty(n) for _ in range(3))
    rc = _load().oracle_adamw_step(_ptr(arrs[0]), _ptr(arrs[1]), _ptr(arrs[2]), _ptr(arrs[3]), n, float(lr), float(beta1),
                                   float(beta2), float(eps), float(wd), int(step), _ptr(po), _ptr(mo), _ptr(vo))
    if rc != 0:
        raise RuntimeError("oracle_adamw_step failed")
    shape = np.shape(p)
    return po.reshape(shape), mo.reshape(shape), vo.reshape(shape)
