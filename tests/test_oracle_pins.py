"""Pins for oracle/ (CPU only).  Each test checks the oracle against something that is NOT the oracle:
a closed form, an SVD from LAPACK, a brute-force long-double evaluation of PAPER.md Eq. 2, an invariant.
A plausible mistake in the oracle (dropped term, wrong sign or index, transposed operand, wrong
normalisation) fails at least one of them."""
import os

import numpy as np
import pytest
import torch

import oracle

A_, B_, C_ = oracle.DEFAULT_COEFFS
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def p(s, a=A_, b=B_, c=C_):
    return a * s + b * s ** 3 + c * s ** 5


def pk(s, k=5):
    for _ in range(k):
        s = p(s)
    return s


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def svd_closed_form(X, k=5, eps=0.0):
    """NS_k(X) from an SVD: NS acts on each singular value as p."""
    U, S, Vt = np.linalg.svd(X, full_matrices=False)
    s = S / (np.linalg.norm(X) + eps)
    return (U * pk(s, k)) @ Vt


def read_blocks(path):
    blocks, name = {}, None
    for line in open(path):
        line = line.strip()
        if not line:
            continue
        if line.startswith("#"):
            name = line[1:].strip().split()[0]
            blocks[name] = []
        else:
            blocks[name].append([float(t) for t in line.split()])
    return {k: np.array(v) for k, v in blocks.items() if v}


# ---------------------------------------------------------------- scalar closed form

def test_golden_quintic_table():
    tab = np.loadtxt(os.path.join(GOLD, "quintic_p5.txt"))
    for s, want in tab:
        assert abs(pk(s) - want) < 5e-10, (s, pk(s), want)      # the fixture itself is the polynomial
    # and the oracle reproduces it on 1 x 1 ... no: on diagonal inputs (next test).  p(1) = a + b + c:
    assert abs(p(1.0) - 0.7010) < 1e-12


def test_diagonal_input_follows_scalar_map():
    X = np.array([[3.0, 0, 0], [0, 4.0, 0]])
    Y = oracle.ns(X, eps=0.0)
    want = np.array([[pk(0.6), 0, 0], [0, pk(0.8), 0]])
    assert np.abs(Y - want).max() < 1e-14
    assert abs(Y[0, 0] - 0.722876168617) < 1e-11 and abs(Y[1, 1] - 1.119203929916) < 1e-11
    # one step at a time (catches a wrong step count / coefficient order)
    for k in range(1, 6):
        Yk = oracle.ns(X, steps=k, eps=0.0)
        assert abs(Yk[0, 0] - pk(0.6, k)) < 1e-14 and abs(Yk[1, 1] - pk(0.8, k)) < 1e-14
    # wider diagonal with many sigmas incl. the golden ones
    s = np.array([0.6, 0.5, 0.3, 0.1, 0.02, 0.005])
    X = np.zeros((6, 9)); X[np.arange(6), np.arange(6)] = s
    Y = oracle.ns(X, eps=0.0)
    sn = s / np.linalg.norm(s)
    assert np.abs(np.diag(Y[:, :6]) - pk(sn)).max() < 1e-13
    assert np.abs(Y - np.diag(np.diag(Y[:, :6])) @ np.eye(6, 9)).max() == 0.0


def test_orthogonal_times_diagonal():
    th, ph = 0.3, 1.1
    U = np.array([[np.cos(th), -np.sin(th)], [np.sin(th), np.cos(th)]])
    V = np.array([[np.cos(ph), -np.sin(ph), 0], [np.sin(ph), np.cos(ph), 0], [0, 0, 1.0]])
    X = U @ np.array([[3.0, 0, 0], [0, 4.0, 0]]) @ V.T
    want = U @ np.diag([pk(0.6), pk(0.8)]) @ V.T[:2, :]
    assert np.abs(oracle.ns(X, eps=0.0) - want).max() < 1e-14


@pytest.mark.parametrize("shape", [(4, 6), (6, 4), (5, 5), (1, 7), (7, 1), (96, 200), (130, 70)])
def test_singular_vectors_invariant_vs_svd(shape):
    rng = np.random.default_rng(11 + shape[0])
    Z = rng.standard_normal(shape)
    Y = oracle.ns(Z, eps=0.0)
    assert Y.shape == Z.shape
    assert rel(Y, svd_closed_form(Z)) < 1e-11
    U, S, Vt = np.linalg.svd(Z, full_matrices=False)
    D = U.T @ Y @ Vt.T
    assert np.abs(D - np.diag(np.diag(D))).max() < 1e-11          # same singular vectors
    assert np.abs(np.diag(D) - pk(S / np.linalg.norm(S))).max() < 1e-11


def test_band_of_the_quintic():
    # critical points of p and the invariant band [p(min), p(max)]
    lo, hi = p(1.0501360791), p(0.5545287909)
    assert abs(lo - 0.6818314622) < 1e-9 and abs(hi - 1.2023686052) < 1e-9
    rng = np.random.default_rng(5)
    Z = rng.standard_normal((40, 64))
    sv_in = np.linalg.svd(Z, compute_uv=False) / np.linalg.norm(Z)
    assert sv_in.min() > 1.51e-3
    sv = np.linalg.svd(oracle.ns(Z), compute_uv=False)
    assert sv.max() <= hi + 1e-12 and sv.min() >= lo - 1e-12
    # below the threshold the map is ~ a^5 * sigma
    X = np.zeros((2, 3)); X[0, 0] = 1.0; X[1, 1] = 1e-6
    Y = oracle.ns(X, eps=0.0)
    assert abs(Y[1, 1] / 1e-6 - A_ ** 5) / A_ ** 5 < 1e-6


def test_gram_matrix_exactly_symmetric_and_correct():
    rng = np.random.default_rng(3)
    Z = rng.standard_normal((37, 91))
    _, A1 = oracle.ns(Z, steps=1, normalize=False, return_A1=True)
    assert np.array_equal(A1, A1.T)                                # bitwise
    assert rel(A1, Z @ Z.T) < 1e-14


def test_transpose_equivariance_exact():
    rng = np.random.default_rng(7)
    Z = rng.standard_normal((5, 3))
    assert np.array_equal(oracle.ns(Z.T.copy()), oracle.ns(Z).T)
    Z = rng.standard_normal((20, 33))
    assert np.array_equal(oracle.ns(Z.T.copy()), oracle.ns(Z).T)


@pytest.mark.parametrize("shape", [(3, 5), (8, 8), (6, 2)])
def test_eq2_literal_long_double(shape):
    """PAPER.md:55 Eq. 2 evaluated literally, X' = aX + b X X^T X + c (X X^T)^2 X, with long-double loops."""
    rng = np.random.default_rng(21)
    Z = rng.standard_normal(shape)
    X = (Z / np.linalg.norm(Z)).astype(np.longdouble)
    a, b, c = (np.longdouble(v) for v in (A_, B_, C_))

    def mm(P, Q):
        out = np.zeros((P.shape[0], Q.shape[1]), dtype=np.longdouble)
        for i in range(P.shape[0]):
            for j in range(Q.shape[1]):
                acc = np.longdouble(0)
                for k in range(P.shape[1]):
                    acc += P[i, k] * Q[k, j]
                out[i, j] = acc
        return out

    for _ in range(5):
        XXt = mm(X, X.T)
        X = a * X + b * mm(XXt, X) + c * mm(mm(XXt, XXt), X)      # no transposition: Eq. 2 as printed
    Y = oracle.ns(Z, eps=0.0)
    assert rel(Y, X.astype(np.float64)) < 1e-12


def test_eq4_gram_recurrence():
    """PAPER.md:172 Eq. 4: G_{i+1} = P_i G_i P_i with P_i = aI + bG_i + cG_i^2."""
    rng = np.random.default_rng(9)
    X = rng.standard_normal((6, 10)); X /= np.linalg.norm(X)
    for _ in range(4):
        Xn, G = oracle.ns(X, steps=1, normalize=False, return_A1=True)
        _, Gn = oracle.ns(Xn, steps=1, normalize=False, return_A1=True)
        P = A_ * np.eye(6) + B_ * G + C_ * G @ G
        assert rel(Gn, P @ G @ P) < 1e-12
        assert rel(Xn, P @ X) < 1e-13
        X = Xn


def test_classical_cubic_converges_to_polar_factor():
    """(a,b,c) = (1.5,-0.5,0) is the textbook Newton-Schulz polar iteration: exact U V^T in the limit."""
    rng = np.random.default_rng(13)
    Z = rng.standard_normal((6, 9))
    U, S, Vt = np.linalg.svd(Z, full_matrices=False)
    Z = (U * np.linspace(0.5, 1.0, 6)) @ Vt                           # well conditioned -> fast convergence
    Y = oracle.ns(Z, steps=40, coeffs=(1.5, -0.5, 0.0), eps=0.0)
    assert rel(Y, U @ Vt) < 1e-12


def test_per_step_schedule_is_composition():
    rng = np.random.default_rng(17)
    Z = rng.standard_normal((7, 12))
    sched = np.array([[3.0, -3.5, 1.2], [2.5, -2.0, 0.6], [1.5, -0.5, 0.0]])
    Y = oracle.ns(Z, steps=3, coeffs=sched, eps=0.0)
    X = Z / np.linalg.norm(Z)
    for a, b, c in sched:
        G = X @ X.T
        X = a * X + b * G @ X + c * G @ G @ X
    assert rel(Y, X) < 1e-13


def test_normalisation_and_eps():
    rng = np.random.default_rng(19)
    Z = rng.standard_normal((4, 9))
    # scale invariance up to eps: NS(1000 Z) == NS(Z) when eps = 0
    assert rel(oracle.ns(1000 * Z, eps=0.0), oracle.ns(Z, eps=0.0)) < 1e-13
    # eps is ADDED TO THE NORM (reading N2): X0 = Z / (||Z|| + eps)
    eps = 0.5
    want = svd_closed_form(Z, eps=eps)
    assert rel(oracle.ns(Z, eps=eps), want) < 1e-12
    # zero input -> zero output, no NaN (reading N14)
    assert np.array_equal(oracle.ns(np.zeros((3, 5))), np.zeros((3, 5)))
    # normalize=False really skips it
    X = Z / np.linalg.norm(Z)
    assert np.array_equal(oracle.ns(X, normalize=False), oracle.ns(X, normalize=False))
    assert rel(oracle.ns(X, normalize=False), svd_closed_form(Z)) < 1e-12


# ---------------------------------------------------------------- bf16 rounding

def test_round_bf16_matches_torch_rne():
    rng = np.random.default_rng(23)
    x = np.concatenate([rng.standard_normal(5000) * 10.0 ** rng.uniform(-30, 30, 5000),
                        [0.0, -0.0, 1.0, 1.00390625, 1.001953125, 1.005859375, 3.3895313892515355e38,
                         3.39e38, 1e-40, 9.2e-41, 4.5e-41, -2.5]]).astype(np.float32)
    got = oracle.round_bf16(x.astype(np.float64))
    want = torch.from_numpy(x).to(torch.bfloat16).to(torch.float64).numpy()
    assert np.array_equal(got, want)
    # ties to even: 1 + 2^-8 is halfway between 1 and 1 + 2^-7 -> 1 ; 1 + 3*2^-8 -> 1 + 2^-6
    assert oracle.round_bf16([1.00390625])[0] == 1.0
    assert oracle.round_bf16([1.01171875])[0] == 1.015625


# ---------------------------------------------------------------- Muon step

def test_muon_step_2x3_golden_and_svd_closed_form():
    b = read_blocks(os.path.join(GOLD, "muon_step_2x3.txt"))
    W, G, M = b["W"], b["G"], b["M"]
    lr, mu, wd = 0.02, 0.95, 0.01
    out = oracle.muon_step(W, G, M, lr, mu, wd, u_cast=False)
    assert np.abs(out["M_new"] - b["M_new"]).max() < 1e-15
    assert np.abs(out["O"] - b["O"]).max() < 5e-12
    assert np.abs(out["W_new"] - b["W_new"]).max() < 5e-12
    # independent derivation: Nesterov by hand + SVD closed form + Eq. 1
    Mn = mu * M + G
    U = G + mu * Mn
    O = svd_closed_form(U, eps=1e-7)
    assert rel(out["O"], O) < 1e-12
    assert rel(out["W_new"], W - lr * (1.0 * O + wd * W)) < 1e-13
    # tall (3 x 2): scale sqrt(rows/cols) = sqrt(1.5)  (reading N4), O = transpose of the wide O
    outT = oracle.muon_step(W.T.copy(), G.T.copy(), M.T.copy(), lr, mu, wd, u_cast=False)
    assert np.abs(outT["W_new"] - b["W_new_transposed_problem"]).max() < 5e-12
    assert rel(outT["O"], O.T) < 1e-12
    assert rel(outT["W_new"], W.T - lr * (np.sqrt(1.5) * O.T + wd * W.T)) < 1e-13


def test_muon_step_u_cast_and_degenerate():
    rng = np.random.default_rng(29)
    r, c = 12, 20
    bf = lambda a: torch.from_numpy(a.astype(np.float32)).to(torch.bfloat16).to(torch.float64).numpy()
    W, G, M = bf(rng.standard_normal((r, c)) * 0.02), bf(rng.standard_normal((r, c)) * 1e-3), bf(
        rng.standard_normal((r, c)) * 1e-3)
    mu = float(np.float32(0.95))
    out = oracle.muon_step(W, G, M, 0.02, mu, 0.01, u_cast=True)
    U_unr = G + mu * (mu * M + G)
    assert np.array_equal(out["U"], oracle.round_bf16(U_unr))        # reading N15: the cast is applied to U
    assert np.array_equal(out["M_new"], mu * M + G)                    # and M' is NOT rounded before U is formed
    assert rel(out["O"], svd_closed_form(out["U"], eps=1e-7)) < 1e-11
    # zero gradient and momentum: O = 0, W' = W (1 - lr wd)   (reading N14)
    z = np.zeros((r, c))
    out0 = oracle.muon_step(W, z, z, 0.02, mu, 0.01)
    assert np.array_equal(out0["O"], z)
    assert np.abs(out0["W_new"] - W * (1 - 0.02 * 0.01)).max() < 1e-17
    # wd = 0, lr = 1: W' = W - scale*O exactly Eq. 1
    out1 = oracle.muon_step(W, G, M, 1.0, mu, 0.0)
    assert np.abs(out1["W_new"] - (W - out1["O"])).max() < 1e-16


def test_muon_step_momentum_is_the_real_arithmetic_definition():
    """M' = mu M + G and U = G + mu M' in real arithmetic.  The oracle forms them in float64, where both
    are EXACT for bf16 inputs and a 24-bit mu (8-bit x 24-bit products, same-scale sums: under 53 bits), so the oracle's
    values must equal exact rational arithmetic; a binary32 evaluation (what a GPU kernel would do) must NOT be what it
    returns (it differs in a visible share of the bf16 quantisation decisions, N16)."""
    from fractions import Fraction
    rng = np.random.default_rng(31)
    r, c = 16, 24
    bf = lambda a: torch.from_numpy(a.astype(np.float32)).to(torch.bfloat16).to(torch.float64).numpy()
    W, G, M = bf(rng.standard_normal((r, c)) * 0.02), bf(rng.standard_normal((r, c))), bf(rng.standard_normal((r, c)))
    mu = float(np.float32(0.95))
    out = oracle.muon_step(W, G, M, 0.02, mu, 0.01, u_cast=False)
    for i in range(r):
        for j in range(c):
            mn = Fraction(mu) * Fraction(M[i, j]) + Fraction(G[i, j])
            assert Fraction(out["M_new"][i, j]) == mn
            u = Fraction(G[i, j]) + Fraction(mu) * mn
            assert abs(Fraction(out["U"][i, j]) - u) <= abs(u) * Fraction(1, 2 ** 52)
    m32 = (mu * M + G).astype(np.float32).astype(np.float64)
    assert (out["M_new"] != m32).mean() > 0.5          # the oracle is not a binary32 evaluation


def test_oracle_on_config1_matrix_against_svd():
    """A matrix of configs[0] (128 x 512, bf16 bits): oracle == SVD closed form."""
    from paper_2606_27153_b200 import synth
    shapes, Xs = synth.ns_inputs("cpu")
    X = Xs[3].to(torch.float64).numpy()
    assert rel(oracle.ns(X), svd_closed_form(X, eps=1e-7)) < 1e-10


# ---------------------------------------------------------------- AdamW (non-matrix parameters)

def test_adamw_against_torch_optim_float64():
    """oracle.adamw_step against torch.optim.AdamW (CPU, float64) over 6 steps with changing gradients: moments, bias
    correction, eps placement and the decoupled decay (reading N17: the host stack's convention)."""
    g = torch.Generator().manual_seed(11)
    p0 = torch.randn(257, generator=g, dtype=torch.float64) * 0.3
    lr, b1, b2, eps, wd = 3e-3, 0.9, 0.95, 1e-8, 0.1
    pt = torch.nn.Parameter(p0.clone())
    opt = torch.optim.AdamW([pt], lr=lr, betas=(b1, b2), eps=eps, weight_decay=wd)
    p, m, v = p0.numpy().copy(), np.zeros(257), np.zeros(257)
    for step in range(1, 7):
        grad = torch.randn(257, generator=g, dtype=torch.float64) * (0.1 * step)
        pt.grad = grad.clone()
        opt.step()
        p, m, v = oracle.adamw_step(p, grad.numpy(), m, v, lr, b1, b2, eps, wd, step)
        st = opt.state[pt]
        assert np.abs(p - pt.detach().numpy()).max() < 1e-14
        assert np.abs(m - st["exp_avg"].numpy()).max() < 1e-15 and np.abs(v - st["exp_avg_sq"].numpy()).max() < 1e-15


def test_adamw_first_step_closed_form():
    """Step 1 from zero moments: mhat = g, vhat = g^2, so p1 = p0 (1 - lr wd) - lr g / (|g| + eps)."""
    p0 = np.array([0.5, -0.25, 1.0, 0.0, 2.0])
    g = np.array([0.1, -3.0, 1e-4, 7.0, 0.0])
    lr, b1, b2, eps, wd = 1e-2, 0.9, 0.999, 1e-8, 0.05
    p1, m1, v1 = oracle.adamw_step(p0, g, np.zeros(5), np.zeros(5), lr, b1, b2, eps, wd, 1)
    want = p0 * (1 - lr * wd) - lr * g / (np.abs(g) + eps)
    assert np.abs(p1 - want).max() < 1e-12       # sqrt(vhat) = |g| up to an ulp of the division by (1 - beta2)
    assert np.allclose(m1, (1 - b1) * g, rtol=0, atol=1e-17) and np.allclose(v1, (1 - b2) * g * g, rtol=1e-15, atol=0)
    # zero gradient: pure decay
    assert p1[4] == 2.0 * (1 - lr * wd)
    # wd = 0 and a huge eps: p moves by ~ -lr mhat / eps
    p2, _, _ = oracle.adamw_step(p0, g, np.zeros(5), np.zeros(5), lr, b1, b2, 1e6, 0.0, 1)
    assert np.abs((p2 - p0) + lr * g / (np.abs(g) + 1e6)).max() < 2.3e-16      # one ulp of the subtraction p2 - p0
