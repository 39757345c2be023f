"""-m gpu: S1-S5 through the C ABI (tcb_contract) against the nested-loop oracle, element by element.
Tolerance: BASELINE.json north_star, max normalised error 1e-11 (gpu_util.TOL); snorm == 0 -> exact."""
import numpy as np
import pytest

import oracle
import paper_2409_06759_b200 as pkg
from paper_2409_06759_b200 import synth
from gpu_util import TOL, rc, parity_error, split_expr

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    c = pkg.Context(0)
    yield c
    c.destroy()


def run_case(ctx, expr, ext, alpha=1.0, seed=0, options=None):
    rng = np.random.default_rng(seed)
    dl, ll, rl = split_expr(expr)
    D = rc(rng, *[ext[x] for x in dl])
    L = rc(rng, *[ext[x] for x in ll])
    R = rc(rng, *[ext[x] for x in rl])
    for k, v in (options or {}).items():
        ctx.set_option(k, v)
    try:
        dD, dL, dR = ctx.tensor_from_numpy(D), ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R)
        ctx.contract(expr, dD, dL, dR, alpha)
        got = ctx.tensor_download(dD)
        plan = ctx.plan_describe(expr, dD, dL, dR)
    finally:
        for k in (options or {}):
            ctx.set_option(k, "auto")
    ref, sn = oracle.contract(expr, D, L, R, alpha)
    err = parity_error(got, ref, sn)
    assert err <= TOL, (expr, ext, err, plan)
    for t in (dD, dL, dR):
        t.destroy()
    return plan, err


def test_config1_ladder_and_transpose(ctx):
    """BASELINE.json configs[0]: o=8, v=24 pp ladder into a zero R, plus the (a,b,i,j)->(i,j,a,b) transpose."""
    o, v = 8, 24
    V, T = synth.config_ladder(o, v, 1)
    dV, dT = ctx.tensor_from_numpy(V), ctx.tensor_from_numpy(T)
    dR = ctx.tensor_create((v, v, o, o))
    expr = "R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)"
    ctx.contract(expr, dR, dV, dT, 0.5)
    R = ctx.tensor_download(dR)
    ref, sn = oracle.contract(expr, np.zeros((v, v, o, o)), V, T, 0.5)
    assert parity_error(R, ref, sn) <= TOL
    plan = ctx.plan_describe(expr, dR, dV, dT)
    assert (plan["M"], plan["N"], plan["K"]) == (576, 64, 576)
    assert not plan["permute_A"] and not plan["permute_B"]          # canonical order: pure ZGEMM
    # antisymmetry carried through exactly in (i,j)?  not guaranteed bitwise; within tolerance:
    assert np.max(np.abs(R + R.transpose(1, 0, 2, 3))) <= 1e-11 * np.max(sn)
    dTt = ctx.tensor_create((o, o, v, v))
    ctx.permute("Tt(i,j,a,b)=T(a,b,i,j)", dTt, dT)
    assert ctx.tensor_download(dTt).tobytes() == oracle.permute("Tt(i,j,a,b)=T(a,b,i,j)", T, (o, o, v, v)).tobytes()


CASES = [
    # plain matrices, all four layout variants, several tiles + ragged tails in M, N and K
    ("C(m,n)+=A(m,k)*B(k,n)", dict(m=150, n=97, k=45)),
    ("C(m,n)+=A(k,m)*B(k,n)", dict(m=131, n=70, k=53)),
    ("C(m,n)+=A(m,k)*B(n,k)", dict(m=67, n=129, k=31)),
    ("C(m,n)=A(k,m)*B(n,k)", dict(m=65, n=66, k=9)),
    ("C(n,m)+=A(m,k)*B(k,n)", dict(m=70, n=75, k=20)),
    # CC shapes (reduced o, v): ladders, ring, Fock, skinny, rank-6
    ("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", dict(a=13, b=13, c=13, d=13, i=5, j=5)),
    ("R(a,b,i,j)+=T(a,b,k,l)*I(k,l,i,j)", dict(a=13, b=13, k=5, l=5, i=5, j=5)),
    ("I(k,l,i,j)+=W(k,l,c,d)*T(c,d,i,j)", dict(c=13, d=13, k=5, l=5, i=5, j=5)),
    ("X(a,b,i,j)=T(a,c,i,k)*I(k,b,c,j)", dict(a=11, b=11, c=11, i=4, j=4, k=4)),
    ("I(k,b,c,j)+=W(k,l,c,d)*T(b,d,j,l)", dict(b=11, c=11, d=11, j=4, k=4, l=4)),
    ("X(a,b,i,j)=T(a,c,i,j)*f(b,c)", dict(a=17, b=17, c=17, i=6, j=6)),
    ("X(a,b,i,j)=T(a,b,i,k)*f(k,j)", dict(a=17, b=17, i=6, j=6, k=6)),
    ("R(b,a,i,j)+=T(a,c,i,j)*f(b,c)", dict(a=17, b=17, c=17, i=6, j=6)),
    ("R(a,b,j,i)+=T(a,b,i,k)*f(k,j)", dict(a=17, b=17, i=6, j=6, k=6)),
    ("I(l,i)=W(k,l,c,d)*T(d,c,i,k)", dict(c=19, d=19, i=5, k=5, l=5)),
    ("I(a,d)=W(k,l,c,d)*T(a,c,l,k)", dict(a=19, c=19, d=19, k=5, l=5)),
    ("X(a,b,c,i,j,k)=W(b,c,d,k)*T(a,d,i,j)", dict(a=9, b=9, c=9, d=9, i=3, j=3, k=3)),
    ("X(a,b,c,i,j,k)+=T(a,b,i,l)*W(l,c,j,k)", dict(a=7, b=7, c=7, i=3, j=3, k=3, l=3)),
    # K = 1 (outer product), N = 1 (R fully contracted), extent-1 indices, rank 2..6 mixes
    ("t(a,b,i,j)=T(a,i)*S(b,j)", dict(a=33, b=34, i=7, j=5)),
    ("R(a,i)+=T(a,e,i,m)*F(m,e)", dict(a=37, e=21, i=6, m=5)),
    ("R(a,i)+=F(m,e)*T(a,e,i,m)", dict(a=37, e=21, i=6, m=5)),
    ("R(a,x,i)+=T(a,e,y,i)*F(e,x,y)", dict(a=70, e=40, i=9, x=1, y=1)),
    ("R(i,a)+=T(e,a)*F(i,e)", dict(a=70, e=3, i=2)),
    ("Z(p,q,r,s,t,u)+=A(p,x,r,y,t)*B(u,y,s,x,q)", dict(p=5, q=4, r=3, s=6, t=2, u=7, x=5, y=3)),
]


@pytest.mark.parametrize("expr,ext", CASES)
def test_contraction_parity(ctx, expr, ext):
    run_case(ctx, expr, ext, alpha=0.5, seed=1)


def test_complex_alpha_and_assign(ctx):
    run_case(ctx, "C(m,n)+=A(m,k)*B(k,n)", dict(m=80, n=33, k=29), alpha=0.3 - 1.7j, seed=2)
    run_case(ctx, "C(m,n)=A(m,k)*B(k,n)", dict(m=80, n=33, k=29), alpha=-2j, seed=3)


def test_assign_ignores_nan_in_D(ctx):
    """'=' must not read D: a NaN-filled D comes out clean."""
    rng = np.random.default_rng(4)
    L, R = rc(rng, 40, 30), rc(rng, 30, 20)
    dD = ctx.tensor_create((40, 20))
    ctx.tensor_fill(dD, complex(np.nan, np.nan))
    ctx.contract("D(m,n)=L(m,k)*R(k,n)", dD, ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R), 1.0)
    got = ctx.tensor_download(dD)
    ref, sn = oracle.contract("D(m,n)=L(m,k)*R(k,n)", np.zeros((40, 20)), L, R, 1.0)
    assert parity_error(got, ref, sn) <= TOL


@pytest.mark.parametrize("splits", ["2", "5", "auto"])
def test_split_k(ctx, splits):
    plan, _ = run_case(ctx, "I(l,i)=W(k,l,c,d)*T(d,c,i,k)", dict(c=40, d=40, i=6, k=6, l=6), seed=5,
                       options={"splitk": splits})
    if splits != "auto":
        assert plan["splits"] == int(splits)
    plan, _ = run_case(ctx, "C(m,n)+=A(m,k)*B(k,n)", dict(m=70, n=20, k=4000), seed=6, options={"splitk": splits})


def test_split_k_is_run_to_run_deterministic(ctx):
    rng = np.random.default_rng(7)
    L, R = rc(rng, 50, 3000), rc(rng, 3000, 40)
    dL, dR = ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R)
    outs = []
    for _ in range(3):
        dD = ctx.tensor_create((50, 40))
        ctx.contract("D(m,n)=L(m,k)*R(k,n)", dD, dL, dR, 1.0)
        outs.append(ctx.tensor_download(dD).tobytes())
    assert outs[0] == outs[1] == outs[2]


def test_forced_operand_permutation_matches(ctx):
    run_case(ctx, "R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", dict(a=13, b=13, c=13, d=13, i=5, j=5), seed=8,
             options={"permute_operands": "always"})


def test_delta_tensor_returns_input_exactly(ctx):
    """V(a,b,c,d) = delta_ac delta_bd  =>  R = alpha * T bit for bit (sums of exact zeros)."""
    v, o = 9, 4
    V = np.zeros((v, v, v, v), dtype=np.complex128, order="F")
    for a in range(v):
        for b in range(v):
            V[a, b, a, b] = 1.0
    T = rc(np.random.default_rng(9), v, v, o, o)
    dR = ctx.tensor_create((v, v, o, o))
    ctx.set_option("complex_product", "4m")       # the property of four real products (3M: tests/test_gpu_complex_product.py)
    try:
        ctx.contract("R(a,b,i,j)=V(a,b,c,d)*T(c,d,i,j)", dR, ctx.tensor_from_numpy(V), ctx.tensor_from_numpy(T), 2.0)
    finally:
        ctx.set_option("complex_product", "auto")
    assert np.array_equal(ctx.tensor_download(dR), 2.0 * T)


def test_power_of_two_alpha_scales_exactly(ctx):
    rng = np.random.default_rng(10)
    L, R = rc(rng, 70, 50), rc(rng, 50, 66)
    dL, dR = ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R)
    d1, d2 = ctx.tensor_create((70, 66)), ctx.tensor_create((70, 66))
    ctx.contract("D(m,n)=L(m,k)*R(k,n)", d1, dL, dR, 1.0)
    ctx.contract("D(m,n)=L(m,k)*R(k,n)", d2, dL, dR, 4.0)
    assert np.array_equal(4.0 * ctx.tensor_download(d1), ctx.tensor_download(d2))


def test_errors_leave_D_untouched(ctx):
    rng = np.random.default_rng(11)
    D, L, R = rc(rng, 4, 5), rc(rng, 4, 6), rc(rng, 6, 5)
    dD, dL, dR = ctx.tensor_from_numpy(D), ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R)
    for expr, code in [("D(m,n)+=L(m,k)*R(k,n", pkg.TCB_EINVAL_EXPR), ("D(m,n)+=L(m,k)*R(n,k)", pkg.TCB_ESHAPE),
                       ("D(m,n)+=L(m,n)*R(k,n)", pkg.TCB_ESHAPE), ("D(m,m)+=L(m,k)*R(k,n)", pkg.TCB_EUNSUPPORTED),
                       ("D(m,n,q)+=L(m,k)*R(k,n)", pkg.TCB_ESHAPE)]:
        with pytest.raises(pkg.TcbError) as ei:
            ctx.contract(expr, dD, dL, dR, 1.0)
        assert ei.value.code == code, (expr, ei.value.code)
    with pytest.raises(pkg.TcbError) as ei:
        ctx.contract("D(m,n)+=L(m,k)*R(k,n)", dD, dD, dR, 1.0)
    assert ei.value.code in (pkg.TCB_EALIAS, pkg.TCB_ESHAPE)
    assert np.array_equal(ctx.tensor_download(dD), D)


def _random_contraction(rng):
    """a random valid binary contraction: ranks 1..6 (a rank-0 D has its own test), every label twice, random index orders"""
    labels = list("abcdefghijkl")
    for _ in range(1000):
        nfl, nfr, nc = int(rng.integers(0, 4)), int(rng.integers(0, 4)), int(rng.integers(0, 4))
        if nfl + nc == 0 or nfr + nc == 0 or nfl + nfr == 0 or nfl + nc > 6 or nfr + nc > 6 or nfl + nfr > 6:
            continue
        labs = labels[:nfl + nfr + nc]
        fl, fr, cc = labs[:nfl], labs[nfl:nfl + nfr], labs[nfl + nfr:]
        ext = {x: int(rng.choice([1, 2, 3, 5, 7, 9, 16, 23])) for x in labs}
        if np.prod([ext[x] for x in fl + cc]) > 60000 or np.prod([ext[x] for x in fr + cc]) > 60000:
            continue
        d, l, r = list(fl + fr), list(fl + cc), list(fr + cc)
        rng.shuffle(d); rng.shuffle(l); rng.shuffle(r)
        op = "+=" if rng.integers(2) else "="
        return f"D({','.join(d)}){op}L({','.join(l)})*R({','.join(r)})", ext
    raise RuntimeError("no contraction drawn")


@pytest.mark.parametrize("loads", ["auto", "gather", "permute"])
def test_random_contractions_under_every_operand_feed(ctx, loads):
    """80 random index patterns (ranks 1..6, extents 1..23, '=' and '+=', complex alpha) per planner setting: whatever the
    cost model or the forced option picks -- TMA in place, gathered, transposed first, GEMV, outer product -- the result is the
    oracle's within 1e-11 of each element's own snorm"""
    rng = np.random.default_rng({"auto": 101, "gather": 102, "permute": 103}[loads])
    routes = {}
    for case in range(80):
        expr, ext = _random_contraction(rng)
        alpha = complex(rng.choice([1.0, -1.0, 0.5, 0.3 - 0.7j]))
        plan, _ = run_case(ctx, expr, ext, alpha=alpha, seed=case, options={"operand_loads": loads})
        key = (plan["route"], plan["feed_A"], plan["feed_B"])
        routes[key] = routes.get(key, 0) + 1
    assert len(routes) >= 4, routes               # the draw exercises several routes and feeds
