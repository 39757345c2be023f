"""-m gpu: the round-2 paths against the oracle -- permutation-free operand loads, the two-pass epilogue
option, the stream-K fix-up under both deals, the outer-product route, lanes (8(f)-4) eager and captured, and the capture
contract."""
import numpy as np
import pytest

import oracle
import paper_2409_06759_b200 as pkg
from paper_2409_06759_b200 import binding
from gpu_util import TOL, rc, parity_error, split_expr

pytestmark = pytest.mark.gpu


@pytest.fixture()
def ctx():
    c = pkg.Context(0)
    yield c
    c.destroy()


def run(ctx, expr, ext, alpha=0.5 - 0.25j, seed=0):
    rng = np.random.default_rng(seed)
    dl, ll, rl = split_expr(expr)
    D, L, R = (rc(rng, *[ext[x] for x in labs]) for labs in (dl, ll, rl))
    dD, dL, dR = ctx.tensor_from_numpy(D), ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R)
    plan = ctx.plan_describe(expr, dD, dL, dR)
    ctx.contract(expr, dD, dL, dR, alpha)
    got = ctx.tensor_download(dD)
    ref, sn = oracle.contract(expr, D, L, R, alpha)
    for t in (dD, dL, dR):
        t.destroy()
    return parity_error(got, ref, sn), plan, got


GATHER_CASES = [
    # ring term: neither operand matrix-shaped; A's unit-stride index free (lanes along m), B's contracted (lanes along k)
    ("X(a,b,i,j)=T(a,c,i,k)*I(k,b,c,j)", dict(a=13, b=11, c=9, i=5, j=6, k=7)),
    ("X(a,b,i,j)+=T(a,c,i,k)*I(k,b,c,j)", dict(a=70, b=33, c=17, i=3, j=4, k=5)),
    # interleaved free / contracted indices on both sides, D in another order
    ("D(j,a,i,b)+=L(a,c,i,d)*R(d,b,c,j)", dict(a=9, b=10, c=11, d=5, i=6, j=7)),
    # unit-stride index contracted but not first in the common order: no contiguous direction (16-byte gathers)
    ("D(a,b)+=L(c,a,d)*R(d,b,c)", dict(a=37, b=29, c=19, d=23)),
    # rank 6 x rank 4 (the T3 term with W in a non-matrix order)
    ("X(a,b,c,i,j,k)=W(b,d,c,k)*T(a,d,i,j)", dict(a=6, b=5, c=7, d=9, i=3, j=4, k=2)),
    # skinny, long K, operand gathered: stream-K chunks over gathered k-tiles, summed by the fix-up kernel
    ("F(m,i)+=V(m,n,e,f)*T(e,f,i,n)", dict(m=6, i=5, n=7, e=31, f=29)),
    ("F(a,e)+=T(a,f,m,n)*V(m,n,e,f)", dict(a=20, e=18, f=41, m=6, n=5)),
    # extent-1 indices and a K tail of 1
    ("D(a,x,b)+=L(a,c,y,b2)*R(c,x,b,y,b2)", dict(a=8, x=1, b=9, c=3, y=1, b2=3)),
]


@pytest.mark.parametrize("loads", ["auto", "gather", "permute"])
@pytest.mark.parametrize("expr,ext", GATHER_CASES)
def test_gathered_operand_loads_match_the_oracle(ctx, expr, ext, loads):
    ctx.set_option("operand_loads", loads)
    err, plan, _ = run(ctx, expr, ext, seed=sum(ext.values()))
    assert err <= TOL, (expr, loads, err, plan)
    if loads == "gather":
        assert not plan["permute_A"] and not plan["permute_B"]
    if loads == "permute":
        assert plan["feed_A"] != "gather" and plan["feed_B"] != "gather"


def test_gather_and_permute_plans_agree_to_rounding_and_gather_is_run_to_run_identical(ctx):
    expr, ext = "X(a,b,i,j)+=T(a,c,i,k)*I(k,b,c,j)", dict(a=40, b=37, c=40, i=9, j=8, k=9)
    outs = {}
    for loads in ("gather", "gather", "permute"):
        ctx.set_option("operand_loads", loads)
        err, plan, got = run(ctx, expr, ext, seed=2)
        assert err <= TOL
        outs.setdefault(loads, []).append(got)
    assert outs["gather"][0].tobytes() == outs["gather"][1].tobytes()


@pytest.mark.parametrize("expr,ext", [
    ("X(b,i,a,j)+=T(a,c,i,k)*I(k,b,c,j)", dict(a=13, b=11, c=9, i=5, j=6, k=7)),
    ("C(m,n)=A(m,k)*B(k,n)", dict(m=130, n=70, k=60)),
    ("R(j,i,b,a)+=V(a,b,c,d)*T(c,d,i,j)", dict(a=7, b=8, c=9, d=6, i=3, j=4)),
])
def test_twopass_epilogue_option(ctx, expr, ext):
    """"epilogue" = "twopass": GEMM into a plain workspace matrix, then the permute-accumulate pass"""
    ctx.set_option("epilogue", "twopass")
    err, plan, _ = run(ctx, expr, ext, alpha=0.3 - 0.7j, seed=7)
    assert plan["epilogue"] == "twopass" and err <= TOL


@pytest.mark.parametrize("k", [2000, 9000])
def test_stream_k_fixup_is_deterministic_under_both_deals(ctx, k):
    """every tile is cut along K (29 / 34 chunks per tile); zgemm_fixup_kernel (32 CTAs per tile, one fragment entry each)
    sums a tile's chunks in k order: the dynamic and the static deal give the same bits, run to run."""
    m, n = 150, 150
    rng = np.random.default_rng(5)
    D, L, R = rc(rng, m, n), rc(rng, m, k), rc(rng, k, n)
    dL, dR = ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R)
    outs, launches = [], []
    for deal in ("dynamic", "static", "dynamic"):
        ctx.set_option("gemm_deal", deal)
        dD = ctx.tensor_from_numpy(D)
        l0 = ctx.launch_count()
        ctx.contract("C(m,n)+=A(m,k)*B(k,n)", dD, dL, dR, 0.5)
        launches.append(ctx.launch_count() - l0)
        outs.append(ctx.tensor_download(dD))
        dD.destroy()
    assert outs[0].tobytes() == outs[1].tobytes() == outs[2].tobytes()
    assert launches == [2, 2, 2]
    ref, sn = oracle.contract("C(m,n)+=A(m,k)*B(k,n)", D, L, R, 0.5)
    assert parity_error(outs[0], ref, sn) <= TOL


def _two_branch_list(ctx, T, A, B, X1, X2, R):
    """two independent contractions on two lanes, joined into a third"""
    ctx.lane_wait(1, 0)
    ctx.contract("X(a,b)=T(a,c)*A(c,b)", X1, T, A, 1.0)
    ctx.lane_set(1)
    ctx.contract("X(a,b)=T(a,c)*B(c,b)", X2, T, B, 1.0)
    ctx.lane_set(0)
    ctx.lane_wait(0, 1)
    ctx.contract("R(a,b)+=X(a,c)*Y(c,b)", R, X1, X2, 0.5)


def test_lanes_eager_and_captured_as_parallel_graph_branches(ctx):
    n = 300
    rng = np.random.default_rng(8)
    hT, hA, hB, hR = rc(rng, n, n), rc(rng, n, n), rc(rng, n, n), rc(rng, n, n)
    T, A, B = ctx.tensor_from_numpy(hT), ctx.tensor_from_numpy(hA), ctx.tensor_from_numpy(hB)
    X1, X2 = ctx.tensor_create((n, n)), ctx.tensor_create((n, n))
    R = ctx.tensor_from_numpy(hR)
    assert ctx.lane_count() >= 2
    _two_branch_list(ctx, T, A, B, X1, X2, R)
    eager = ctx.tensor_download(R)
    x1, s1 = oracle.contract("X(a,b)=T(a,c)*A(c,b)", np.zeros((n, n)), hT, hA, 1.0)
    x2, s2 = oracle.contract("X(a,b)=T(a,c)*B(c,b)", np.zeros((n, n)), hT, hB, 1.0)
    ref, sn = oracle.contract("R(a,b)+=X(a,c)*Y(c,b)", hR, x1, x2, 0.5)
    assert np.max(np.abs(eager - ref) / sn) <= 1e-10          # three chained roundings: looser than one call's TOL
    # the same list, captured: lanes become parallel branches (more edges than a chain has), replay is bit-identical
    ctx.tensor_upload(R, hR)
    ctx.capture_begin()
    _two_branch_list(ctx, T, A, B, X1, X2, R)
    g = ctx.capture_end()
    info = ctx.graph_info(g)
    assert info["launches"] >= 3 and info["nodes"] >= 3
    assert info["depth"] < info["nodes"], info               # a chain has depth = nodes: two of the three run side by side
    ctx.graph_launch(g)
    assert ctx.tensor_download(R).tobytes() == eager.tobytes()
    ctx.graph_destroy(g)


def test_capturing_a_cold_call_list_is_refused_and_the_context_survives(ctx):
    """an uncached plan / workspace growth / sync / upload inside a capture must not kill the context"""
    rng = np.random.default_rng(3)
    hA, hB = rc(rng, 40, 50), rc(rng, 50, 30)
    A, B, C = ctx.tensor_from_numpy(hA), ctx.tensor_from_numpy(hB), ctx.tensor_create((40, 30))
    ctx.capture_begin()
    with pytest.raises(pkg.TcbError) as ei:
        ctx.contract("C(m,n)=A(m,k)*B(k,n)", C, A, B, 1.0)          # never planned before: refused, nothing enqueued
    assert ei.value.code == binding.TCB_EUNSUPPORTED
    with pytest.raises(pkg.TcbError) as ei:
        ctx.sync()
    assert ei.value.code == binding.TCB_EUNSUPPORTED
    with pytest.raises(pkg.TcbError) as ei:
        ctx.capture_end()
    assert ei.value.code == binding.TCB_EUNSUPPORTED
    # call by call the same list works, and a warm capture too
    ctx.contract("C(m,n)=A(m,k)*B(k,n)", C, A, B, 1.0)
    ref, sn = oracle.contract("C(m,n)=A(m,k)*B(k,n)", np.zeros((40, 30)), hA, hB, 1.0)
    assert parity_error(ctx.tensor_download(C), ref, sn) <= TOL
    ctx.capture_begin()
    ctx.contract("C(m,n)=A(m,k)*B(k,n)", C, A, B, 1.0)
    g = ctx.capture_end()
    ctx.tensor_fill(C, 0.0)
    ctx.graph_launch(g)
    assert parity_error(ctx.tensor_download(C), ref, sn) <= TOL
    ctx.graph_destroy(g)


def test_graph_launch_is_refused_after_the_workspace_moved(ctx):
    """a captured graph carries workspace addresses; after a later call grew the workspace the graph is stale"""
    rng = np.random.default_rng(4)
    e = "X(a,b,i,j)=T(a,c,i,k)*I(k,b,c,j)"
    ctx.set_option("operand_loads", "permute")                # permuted operands live in the workspace
    ext = dict(a=9, b=8, c=7, i=3, j=4, k=5)
    shp = lambda s, x: tuple(x[c] for c in s)
    T, I, X = (ctx.tensor_from_numpy(rc(rng, *shp(s, ext))) for s in ("acik", "kbcj", "abij"))
    ctx.contract(e, X, T, I, 1.0)
    ctx.capture_begin()
    ctx.contract(e, X, T, I, 1.0)
    g = ctx.capture_end()
    ctx.graph_launch(g)
    big = dict(a=40, b=40, c=40, i=9, j=9, k=9)
    T2, I2, X2 = (ctx.tensor_from_numpy(rc(rng, *shp(s, big))) for s in ("acik", "kbcj", "abij"))
    ctx.contract(e, X2, T2, I2, 1.0)                          # grows the workspace
    with pytest.raises(pkg.TcbError) as ei:
        ctx.graph_launch(g)
    assert ei.value.code == binding.TCB_EINVAL
    ctx.sync()
    ctx.graph_destroy(g)


@pytest.mark.parametrize("expr,ext", [
    ("tt(a,b,i,j)=T1(a,i)*T2(b,j)", dict(a=37, b=29, i=5, j=7)),           # the CCSD outer product
    ("tt(a,b,i,j)+=T1(a,i)*T2(b,j)", dict(a=300, b=3, i=2, j=41)),
    ("D(j,a)+=L(a)*R(j)", dict(a=1000, j=33)),
    ("D(b,a,x)=R(b,x)*L(a)", dict(a=17, b=9, x=1)),                        # D's unit-stride index in the second operand
])
def test_outer_product_route(ctx, expr, ext):
    """K = 1 (nothing contracted): the store-stream kernel of gemv.cu instead of a GEMM with K padded to 4"""
    err, plan, _ = run(ctx, expr, ext, alpha=0.75 - 0.5j, seed=len(expr))
    assert plan["route"] == "outer" and plan["K"] == 1 and err <= TOL


def test_lane_api_argument_errors_leave_the_context_usable(ctx):
    for bad in (-1, ctx.lane_count()):
        with pytest.raises(pkg.TcbError) as ei:
            ctx.lane_set(bad)
        assert ei.value.code == binding.TCB_EINVAL
        with pytest.raises(pkg.TcbError) as ei:
            ctx.lane_wait(0, bad)
        assert ei.value.code == binding.TCB_EINVAL
    ctx.lane_wait(1, 1)                                        # a lane waiting on itself is a no-op
    ctx.lane_set(1)
    with pytest.raises(pkg.TcbError) as ei:
        ctx.capture_begin()                                    # a capture starts on lane 0
    assert ei.value.code == binding.TCB_EINVAL
    t = ctx.tensor_create((4, 4))                              # created, filled and destroyed on lane 1
    ctx.tensor_fill(t, 2.0 - 1.0j)
    assert np.all(ctx.tensor_download(t) == 2.0 - 1.0j)
    t.destroy()
    ctx.lane_set(0)
    ctx.sync()
