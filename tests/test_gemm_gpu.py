"""The three tcgen05 NS products (dmuon_ns_gemm) against a plain fp32 matmul of the same fp16 inputs.
This checks the kernel family (TMA/UMMA descriptors, triangular scheduling, mirrored stores, epilogues) in
isolation; parity of the whole path against the fp64 oracle is in test_parity_gpu.py."""
import pytest
import torch

import paper_2606_27153_b200 as dm
from paper_2606_27153_b200.binding import OP_BX, OP_SQ, OP_SYRK, OP_SYRK_T, OP_XB

pytestmark = pytest.mark.gpu


def _rand(shape, seed, scale):
    g = torch.Generator(device="cuda")
    g.manual_seed(seed)
    return (torch.randn(shape, generator=g, device="cuda", dtype=torch.float32) * scale).to(torch.float16)


def _rel(a, b):
    return (torch.linalg.norm(a.double() - b.double()) / torch.linalg.norm(b.double())).item()


SHAPES = [(128, 128, 1), (128, 512, 3), (256, 256, 2), (384, 640, 2), (768, 3072, 2), (896, 896, 3), (1024, 4096, 1),
          (2048, 1408 + 128, 2)]


@pytest.mark.parametrize("m,k,count", SHAPES)
@pytest.mark.parametrize("variant", [0, 1, 4, 6])   # single CTA N=256 / N=128, CTA pair 256 x 256, pair with 8 epilogue warps
def test_syrk(m, k, count, variant):
    X = [_rand((m, k), 10 + i, k ** -0.5) for i in range(count)]
    C = [torch.full((m, m), float("nan"), device="cuda", dtype=torch.float16) for _ in range(count)]
    dm.ns_gemm(OP_SYRK, X, None, C, alpha=0.75, beta=0.0, variant=variant)
    torch.cuda.synchronize()
    for x, c in zip(X, C):
        ref = 0.75 * (x.float() @ x.float().t())
        assert torch.isfinite(c).all()
        assert _rel(c, ref) < 1e-3
        assert torch.equal(c, c.t())          # mirrored store: bitwise symmetric


@pytest.mark.parametrize("m,count", [(128, 1), (256, 3), (384, 2), (896, 2), (1024, 2), (4096, 1)])
@pytest.mark.parametrize("variant", [0, 1, 4, 6])
def test_sq(m, count, variant):
    A = []
    for i in range(count):
        x = _rand((m, 2 * m), 20 + i, (2 * m) ** -0.5)
        a = (x.float() @ x.float().t()).to(torch.float16)
        A.append(torch.triu(a) + torch.triu(a, 1).t())      # exactly symmetric fp16
    C = [torch.full((m, m), float("nan"), device="cuda", dtype=torch.float16) for _ in range(count)]
    dm.ns_gemm(OP_SQ, A, None, C, alpha=2.0315, beta=-4.775, variant=variant)
    torch.cuda.synchronize()
    for a, c in zip(A, C):
        ref = 2.0315 * (a.float() @ a.float()) - 4.775 * a.float()
        assert torch.isfinite(c).all()
        assert _rel(c, ref) < 1e-3
        assert torch.equal(c, c.t())


def _commuting_pair(m, seed):
    """Two exactly symmetric fp16 matrices that are polynomials of one Gram matrix (so their product is symmetric up
    to the fp16 rounding of the factors), as in a Gram block: G and B = b G + c G G."""
    x = _rand((m, 2 * m), seed, (2 * m) ** -0.5).double()
    g = x @ x.t()
    b = -4.775 * g + 2.0315 * (g @ g)
    sym16 = lambda t: (torch.triu(t) + torch.triu(t, 1).t()).to(torch.float16)
    return sym16(g), sym16(b)


@pytest.mark.parametrize("m,count", [(128, 2), (256, 3), (384, 2), (896, 2), (1024, 1), (2048, 1)])
@pytest.mark.parametrize("variant", [0, 1, 4, 6])
def test_sym_mm(m, count, variant):
    """dmuon_ns_sym_mm: the Gram-block products T = a G + B G (one addend) and R' = p B' + a R + B' R (two addends)."""
    pairs = [_commuting_pair(m, 50 + i) for i in range(count)]
    G = [p[0] for p in pairs]
    B = [p[1] for p in pairs]
    nan = lambda: [torch.full((m, m), float("nan"), device="cuda", dtype=torch.float16) for _ in range(count)]
    T, R, S = nan(), nan(), nan()
    dm.ns_sym_mm(B, G, G, None, T, alpha=1.0, beta=3.4445, variant=variant)
    dm.ns_sym_mm(B, G, B, G, R, alpha=0.5, beta=3.4445, beta2=-1.25, variant=variant)
    dm.ns_sym_mm(B, G, None, None, S, alpha=2.0, variant=variant)
    torch.cuda.synchronize()
    for g, b, t, r, s_ in zip(G, B, T, R, S):
        bg = b.double() @ g.double()
        for got, ref in ((t, 3.4445 * g.double() + bg), (r, 0.5 * bg + 3.4445 * b.double() - 1.25 * g.double()),
                         (s_, 2.0 * bg)):
            assert torch.isfinite(got).all()
            # the reference product is symmetric only up to the rounding of the factors; compare on the upper triangle
            assert _rel(torch.triu(got), torch.triu(ref)) < 2e-3
            # off-diagonal 128-blocks are mirrored (bitwise symmetric); diagonal blocks are computed in full
            blk = torch.arange(m, device="cuda") // 128
            off = blk[:, None] != blk[None, :]
            assert torch.equal(got[off], got.t()[off])
            assert _rel(got, got.t()) < 2e-3


@pytest.mark.parametrize("m,n,count", SHAPES)
@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4, 5, 6, 7])
def test_bx(m, n, count, variant):
    B = [_rand((m, m), 30 + i, m ** -0.5) for i in range(count)]       # not symmetric on purpose: catches a transposed operand
    X = [_rand((m, n), 40 + i, 1.0) for i in range(count)]
    C = [torch.full((m, n), float("nan"), device="cuda", dtype=torch.float16) for _ in range(count)]
    dm.ns_gemm(OP_BX, B, X, C, alpha=1.0, beta=3.4445, variant=variant)
    torch.cuda.synchronize()
    for b, x, c in zip(B, X, C):
        ref = b.float() @ x.float() + 3.4445 * x.float()
        assert torch.isfinite(c).all()
        assert _rel(c, ref) < 1e-3


@pytest.mark.parametrize("variant", [0, 4, 6])
def test_many_problems_more_units_than_sms(variant):
    """Persistent loop + double-buffered TMEM across many work units per CTA (or CTA pair)."""
    m, k, count = 256, 384, 200
    X = [_rand((m, k), 100 + i, k ** -0.5) for i in range(count)]
    C = [torch.empty((m, m), device="cuda", dtype=torch.float16) for _ in range(count)]
    dm.ns_gemm(OP_SYRK, X, None, C, alpha=1.0, beta=0.0, variant=variant)
    torch.cuda.synchronize()
    for i in (0, 1, 57, 148, 199):
        assert _rel(C[i], X[i].float() @ X[i].float().t()) < 1e-3


@pytest.mark.parametrize("m,k,count", SHAPES)
@pytest.mark.parametrize("variant", [0, 1, 4, 6])
def test_syrk_t(m, k, count, variant):
    """G = Y^T Y for a tall matrix held as stored (Y is k x m): both operands MN-major."""
    Y = [_rand((k, m), 60 + i, k ** -0.5) for i in range(count)]
    C = [torch.full((m, m), float("nan"), device="cuda", dtype=torch.float16) for _ in range(count)]
    dm.ns_gemm(OP_SYRK_T, Y, None, C, alpha=0.75, beta=0.0, variant=variant)
    torch.cuda.synchronize()
    for y, c in zip(Y, C):
        ref = 0.75 * (y.float().t() @ y.float())
        assert torch.isfinite(c).all()
        assert _rel(c, ref) < 1e-3
        assert torch.equal(c, c.t())


@pytest.mark.parametrize("m,n,count", SHAPES)
@pytest.mark.parametrize("variant", [0, 1, 2, 3, 4, 5, 6, 7])
def test_xb(m, n, count, variant):
    """Y' = Y B + beta Y for a tall matrix held as stored (Y is n x m, B symmetric m x m)."""
    B = []
    for i in range(count):
        b = _rand((m, m), 70 + i, m ** -0.5)
        B.append((torch.triu(b) + torch.triu(b, 1).t()).contiguous())     # exactly symmetric fp16
    Y = [_rand((n, m), 80 + i, 1.0) for i in range(count)]
    C = [torch.full((n, m), float("nan"), device="cuda", dtype=torch.float16) for _ in range(count)]
    dm.ns_gemm(OP_XB, B, Y, C, alpha=1.0, beta=3.4445, variant=variant)
    torch.cuda.synchronize()
    for b, y, c in zip(B, Y, C):
        ref = y.float() @ b.float() + 3.4445 * y.float()
        assert torch.isfinite(c).all()
        assert _rel(c, ref) < 1e-3


@pytest.mark.parametrize("variant", [0, 4, 6])
def test_sq_small_m_many_problems(variant):
    """64 problems of m = 1024 (config 4's k/v bucket): short contractions, where the epilogue sets the pace.  Also the
    target of the small-m ncu capture in profiles/."""
    m, count = 1024, 64
    A = []
    for i in range(count):
        x = _rand((m, 256), 200 + i, 256 ** -0.5)
        a = (x.float() @ x.float().t()).to(torch.float16)
        A.append(torch.triu(a) + torch.triu(a, 1).t())
    C = [torch.empty((m, m), device="cuda", dtype=torch.float16) for _ in range(count)]
    for _ in range(3):
        dm.ns_gemm(OP_SQ, A, None, C, alpha=2.0315, beta=-4.775, variant=variant)
    torch.cuda.synchronize()
    for i in (0, 31, 63):
        ref = 2.0315 * (A[i].float() @ A[i].float()) - 4.775 * A[i].float()
        assert _rel(C[i], ref) < 1e-3 and torch.equal(C[i], C[i].t())


def test_variant_table():
    assert dm.binding.ns_gemm_variants(OP_BX) == 8
    x = _rand((128, 128), 1, 1.0)
    c = torch.empty_like(x)
    for bad in (2, 3, 5, 7, 8):        # symmetric ops have one ordering; 8 is out of range
        with pytest.raises(dm.DmuonError):
            dm.ns_gemm(OP_SYRK, [x], None, [c], alpha=1.0, beta=0.0, variant=bad)
