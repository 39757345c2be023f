"""-m gpu: the GEMM's two ways to form a complex product (context option "complex_product"):
    "4m"  four real DMMAs per block pair and k-step  (Re = ArBr - AiBi, Im = ArBi + AiBr)
    "3m"  three                                       (P1 = ArBr, P2 = AiBi, P3 = (Ar+Ai)(Br+Bi); Re = P1 - P2, Im = P3 - P1 - P2)
    "auto" 3m where both operands are TMA-fed and K >= 32 (csrc/plan.cpp).
Both against the nested-loop oracle within north_star's 1e-11 * snorm, element by element, over the shapes that exercise the
3M kernel's own geometry (48 x 48 tiles, 16-deep k-tiles with tails of 1 ... 3 k-steps, warps of up to 3 x 3 blocks, M-major
atoms issued by all four warps, stream-K
fragments, gathered operands, K tails); what 3M gives up (bit-exact products with exactly representable operands) is
asserted as well, with its bound."""
import numpy as np
import pytest

import oracle
import paper_2409_06759_b200 as pkg
from gpu_util import TOL, rc, parity_error, split_expr, sampled_contraction_parity
from paper_2409_06759_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    c = pkg.Context(0)
    yield c
    c.set_option("complex_product", "auto")
    c.destroy()


def _run(ctx, expr, ext, alpha, seed, mode, extra=None):
    rng = np.random.default_rng(seed)
    dl, ll, rl = split_expr(expr)
    D, L, R = (rc(rng, *[ext[x] for x in labs]) for labs in (dl, ll, rl))
    opts = dict(extra or {}, complex_product=mode)
    for k, v in opts.items():
        ctx.set_option(k, v)
    try:
        dD, dL, dR = ctx.tensor_from_numpy(D), ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R)
        ctx.contract(expr, dD, dL, dR, alpha)
        got = ctx.tensor_download(dD)
        plan = ctx.plan_describe(expr, dD, dL, dR)
    finally:
        for k in opts:
            ctx.set_option(k, "dynamic" if k == "gemm_deal" else "auto")
    ref, sn = oracle.contract(expr, D, L, R, alpha)
    for t in (dD, dL, dR):
        t.destroy()
    return parity_error(got, ref, sn), plan, got


GEOMETRY = [   # (expr, extents): all four TMA layout pairs, ragged tiles, one-block tiles, K tails of 1..7 and of <= 4
    ("C(m,n)=A(m,k)*B(k,n)", dict(m=150, n=97, k=333)),        # M-major A (atoms issued by four warps), K-major B
    ("C(m,n)+=A(k,m)*B(k,n)", dict(m=49, n=48, k=131)),        # K-major both; 49 rows = a 48-row tile and a 1-row tile
    ("C(m,n)=A(m,k)*B(n,k)", dict(m=100, n=52, k=260)),        # M-major both
    ("C(m,n)+=A(k,m)*B(n,k)", dict(m=7, n=300, k=129)),        # K-major A, M-major B, one block of rows
    ("C(m,n)=A(m,k)*B(k,n)", dict(m=2, n=3, k=1000)),          # six outputs in one block (N = 1 would take the GEMV route)
    ("C(m,n)=A(m,k)*B(k,n)", dict(m=96, n=96, k=4)),           # one k-step
    ("C(m,n)=A(m,k)*B(k,n)", dict(m=96, n=96, k=13)),          # one 16-deep k-tile, 4 k-steps, the last with one valid k
    ("C(m,n)=A(k,m)*B(n,k)", dict(m=50, n=96, k=16 * 5 + 9)),  # tail k-tile of 3 k-steps, K-major A / M-major B
    ("C(m,n)=A(k,m)*B(k,n)", dict(m=96, n=50, k=16 * 3 + 5)),  # tail k-tile of 2 k-steps
    ("C(m,n)=A(m,k)*B(n,k)", dict(m=70, n=70, k=16 * 2 + 1)),  # tail k-tile of 1 k-step, both M-major
    ("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", dict(a=13, b=13, c=13, d=13, i=5, j=5)),
    ("X(a,b,i,j)=T(a,c,i,k)*I(k,b,c,j)", dict(a=11, b=11, c=11, i=6, j=6, k=6)),      # ring term: transposed or gathered operands
]


@pytest.mark.parametrize("expr,ext", GEOMETRY)
@pytest.mark.parametrize("mode", ["3m", "4m"])
@pytest.mark.parametrize("alpha", [1.0, -0.5, 0.75 - 1.25j])
def test_parity_under_both_products(ctx, expr, ext, mode, alpha):
    err, plan, _ = _run(ctx, expr, ext, alpha, len(expr) + sum(ext.values()), mode)
    assert plan["complex_product"] == mode and err <= TOL, (plan, err)


@pytest.mark.parametrize("extra", [{"operand_loads": "gather"}, {"operand_loads": "permute"}, {"splitk": "7"},
                                   {"epilogue": "twopass"}, {"gemm_deal": "static"}])
def test_3m_with_every_feed_schedule_and_epilogue(ctx, extra):
    """gathered operands into 48-row stages, every tile cut along K (the fix-up sums COMBINED fragments), the two-pass epilogue"""
    for expr, ext in (("X(a,b,i,j)+=T(a,c,i,k)*I(k,b,c,j)", dict(a=14, b=9, c=10, i=5, j=7, k=6)),
                      ("C(m,n)=A(m,k)*B(k,n)", dict(m=130, n=61, k=700))):
        err, plan, _ = _run(ctx, expr, ext, 0.5 - 0.25j, 5, "3m", extra)
        assert plan["complex_product"] == "3m" and err <= TOL, (plan, err)


def test_auto_takes_3m_where_it_was_measured_faster_and_4m_elsewhere(ctx):
    def plan_of(expr, shapes, **opts):
        ts = [ctx.tensor_create(s, zero=False) for s in shapes]
        for k, v in opts.items():
            ctx.set_option(k, v)
        try:
            return ctx.plan_describe(expr, *ts)
        finally:
            for k in opts:
                ctx.set_option(k, "auto")
            for t in ts:
                t.destroy()
    mm = "C(m,n)=A(m,k)*B(k,n)"
    assert plan_of(mm, [(200, 200), (200, 32), (32, 200)])["complex_product"] == "3m"             # K = 32, TMA-fed
    assert plan_of(mm, [(200, 200), (200, 31), (31, 200)])["complex_product"] == "4m"             # short K
    assert plan_of("C(m,n)=A(m,k)*B(n,k)", [(200, 200), (200, 500), (200, 500)])["complex_product"] == "3m"   # any layout pair
    ring = "X(a,b,i,j)=T(a,c,i,k)*I(k,b,c,j)"
    shapes = [(40, 40, 10, 10), (40, 40, 10, 10), (10, 40, 40, 10)]
    assert plan_of(ring, shapes, operand_loads="gather")["complex_product"] == "4m"               # a gathered operand
    assert plan_of(ring, shapes, operand_loads="permute")["complex_product"] == "3m"              # K = 400, both transposed
    assert plan_of(ring, shapes, operand_loads="gather", complex_product="3m")["complex_product"] == "3m"
    assert plan_of("Y(a)=A(a,k)*x(k)", [(300,), (300, 500), (500,)])["complex_product"] == "fma"  # GEMV route: no DMMA at all
    with pytest.raises(pkg.TcbError):
        ctx.set_option("complex_product", "2m")


def test_what_3m_gives_up_and_what_it_keeps(ctx):
    """A delta tensor: 4M returns alpha * T bit for bit (sums of exact zeros); 3M forms Im = (Tr + Ti) * 1 - Tr * 1 - 0, one
    rounding of Tr + Ti away from Ti: |error| <= 2^-52 (|Tr| + |Ti|) per element, far inside 1e-11 * snorm, but not zero.
    Kept by both: real operands give an exactly real result, structural zeros stay exact zeros, the call is deterministic."""
    v, o = 9, 4
    V = np.zeros((v, v, v, v), dtype=np.complex128, order="F")
    for a in range(v):
        for b in range(v):
            V[a, b, a, b] = 1.0
    T = rc(np.random.default_rng(9), v, v, o, o)
    expr = "R(a,b,i,j)=V(a,b,c,d)*T(c,d,i,j)"
    out = {}
    for mode in ("4m", "3m"):
        ctx.set_option("complex_product", mode)
        dR, dV, dT = ctx.tensor_create((v, v, o, o)), ctx.tensor_from_numpy(V), ctx.tensor_from_numpy(T)
        ctx.contract(expr, dR, dV, dT, 2.0)
        out[mode] = ctx.tensor_download(dR)
        ctx.contract(expr, dR, dV, dT, 2.0)
        assert np.array_equal(ctx.tensor_download(dR), out[mode])                 # the same bits twice
        # real operands: exactly real result under both
        dTr = ctx.tensor_from_numpy(np.asfortranarray(T.real + 0j))
        ctx.contract(expr, dR, dV, dTr, 2.0)
        got = ctx.tensor_download(dR)
        assert np.array_equal(got.imag, np.zeros_like(got.imag)) and np.array_equal(got.real, 2.0 * T.real)
        for t in (dR, dV, dT, dTr):
            t.destroy()
    ctx.set_option("complex_product", "auto")
    assert np.array_equal(out["4m"], 2.0 * T)
    assert np.array_equal(out["3m"].real, 2.0 * T.real)
    bound = 2.0 * 2.0 ** -52 * (np.abs(T.real) + np.abs(T.imag))
    assert np.all(np.abs(out["3m"].imag - 2.0 * T.imag) <= bound) and not np.array_equal(out["3m"].imag, 2.0 * T.imag)


def test_3m_error_stays_at_rounding_level_on_a_long_contraction(ctx):
    """K = 40 000 (the headline's K): normalised error of both products against the long-double oracle on sampled outputs;
    3M within a small factor of 4M, both four orders of magnitude inside the tolerance."""
    ext = dict(m=512, n=96, k=40000)
    errs = {}
    for mode in ("4m", "3m"):
        ctx.set_option("complex_product", mode)
        errs[mode], n = sampled_contraction_parity(ctx, "C(m,n)=A(m,k)*B(k,n)", ext, 1.0, synth.SEED0 + 70,
                                                   np.random.default_rng(1), nsub=16)
        assert n == 256
    ctx.set_option("complex_product", "auto")
    assert errs["4m"] <= 1e-14 and errs["3m"] <= 1e-14 and errs["3m"] <= 8 * errs["4m"] + 1e-16, errs
