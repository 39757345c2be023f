"""-m gpu: the edges of the schedule (ragged 8-wide blocks, K tails, tiles cut along K, the dynamic deal) and the
full-size launch configuration that bench.py times, against the oracle.  Tolerance: gpu_util.TOL (north_star)."""
import numpy as np
import pytest

import oracle
import paper_2409_06759_b200 as pkg
from paper_2409_06759_b200 import synth
from gpu_util import TOL, rc, parity_error

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    c = pkg.Context(0)
    yield c
    c.destroy()


def gemm(ctx, m, n, k, expr="C(m,n)+=A(m,k)*B(k,n)", alpha=0.5 - 0.25j, seed=0, shapes=None):
    rng = np.random.default_rng(seed)
    sd, sl, sr = shapes or ((m, n), (m, k), (k, n))
    D, L, R = rc(rng, *sd), rc(rng, *sl), rc(rng, *sr)
    dD, dL, dR = ctx.tensor_from_numpy(D), ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R)
    ctx.contract(expr, dD, dL, dR, alpha)
    got = ctx.tensor_download(dD)
    for t in (dD, dL, dR):
        t.destroy()
    return got, (D, L, R)


@pytest.mark.parametrize("m,n,k", [(1, 1, 1), (7, 5, 3), (8, 8, 4), (9, 17, 5), (67, 45, 13), (130, 70, 60),
                                   (64, 64, 8), (65, 129, 9), (200, 24, 1), (24, 200, 4), (513, 77, 61)])
@pytest.mark.parametrize("expr", ["C(m,n)+=A(m,k)*B(k,n)", "C(m,n)=A(k,m)*B(n,k)"])
def test_ragged_blocks_and_k_tails(ctx, m, n, k, expr):
    shapes = ((m, n), (m, k), (k, n)) if "A(m,k)" in expr else ((m, n), (k, m), (n, k))
    alpha = 0.5 - 0.25j
    got, (D, L, R) = gemm(ctx, m, n, k, expr=expr, alpha=alpha, seed=m * 1000 + n, shapes=shapes)
    ref, sn = oracle.contract(expr, D, L, R, alpha)
    assert parity_error(got, ref, sn) <= TOL


@pytest.mark.parametrize("alpha", [1.0, -1.0, 0.5, 2.0 + 0.0j, 0.3 - 0.7j])
@pytest.mark.parametrize("op", ["+=", "="])
def test_epilogue_alpha_modes(ctx, alpha, op):
    """alpha = 1 (no multiply), real alpha (one FMA per component), complex alpha -- each with and without the read of D"""
    expr = f"C(m,n){op}A(m,k)*B(k,n)"
    got, (D, L, R) = gemm(ctx, 70, 90, 33, expr=expr, alpha=alpha, seed=11)
    ref, sn = oracle.contract(expr, D, L, R, alpha)
    assert parity_error(got, ref, sn) <= TOL


def test_dynamic_and_static_deal_agree_bit_for_bit_and_run_to_run(ctx):
    """Tiles cut along K are fixed k-ranges summed in k order: who computes them does not matter."""
    m, n, k = 150, 150, 9000                      # 9 tiles x 1125 k-tiles: everything is stream-K
    rng = np.random.default_rng(5)
    D, L, R = rc(rng, m, n), rc(rng, m, k), rc(rng, k, n)
    dL, dR = ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R)
    outs = []
    for deal in ("dynamic", "dynamic", "static", "dynamic"):
        ctx.set_option("gemm_deal", deal)
        dD = ctx.tensor_from_numpy(D)
        ctx.contract("C(m,n)+=A(m,k)*B(k,n)", dD, dL, dR, 0.5)
        outs.append(ctx.tensor_download(dD))
        dD.destroy()
    ctx.set_option("gemm_deal", "dynamic")
    assert all(o.tobytes() == outs[0].tobytes() for o in outs)
    ref, sn = oracle.contract("C(m,n)+=A(m,k)*B(k,n)", D, L, R, 0.5)
    assert parity_error(outs[0], ref, sn) <= TOL


def test_many_waves_plus_remainder(ctx):
    """more tiles than resident CTAs (296): whole-tile waves plus a stream-K remainder, ragged in M and N"""
    m, n, k = 1500, 1300, 40                      # 24 x 21 = 504 tiles
    got, (D, L, R) = gemm(ctx, m, n, k, seed=3)
    ref, sn = oracle.contract("C(m,n)+=A(m,k)*B(k,n)", D, L, R, 0.5 - 0.25j)
    assert parity_error(got, ref, sn) <= TOL


@pytest.mark.parametrize("shape,perm", [((2, 300, 70), (2, 1, 0)), ((3, 5, 400, 3), (3, 2, 1, 0)),
                                        ((1, 64, 1, 65, 1, 3), (5, 3, 1, 0, 2, 4)), ((70000, 3), (1, 0)),
                                        ((6, 6, 6, 28, 28, 4), (3, 0, 4, 1, 5, 2))])
def test_permute_short_rows_and_unit_extents(ctx, shape, perm):
    """rows of 2-6 elements (32-96 byte bulk copies), extent-1 indices, a very long thin matrix: bit-exact"""
    lab = "abcdef"[:len(shape)]
    L = np.asfortranarray((np.arange(np.prod(shape), dtype=np.float64) * (1 - 0.5j)).reshape(shape, order="F"))
    e = "D(" + ",".join(lab[p] for p in perm) + ")=L(" + ",".join(lab) + ")"
    dL = ctx.tensor_from_numpy(L)
    dD = ctx.tensor_create(tuple(shape[p] for p in perm))
    ctx.permute(e, dD, dL)
    got = ctx.tensor_download(dD)
    ref = oracle.permute(e, L, tuple(shape[p] for p in perm))
    assert got.tobytes() == ref.tobytes()
    dL.destroy(); dD.destroy()


def test_fullsize_ccd_pp_ladder_sampled_columns(ctx):
    """BASELINE.json configs[1] sizes (o=20, v=80), the launch bench.py times: R(a,b,i,j) += 1/2 vvvv(a,b,c,d) T(c,d,i,j),
    6400 x 400 x 6400.  Inputs come from the device twin of the seeded generator (bit-identical to synth.py:
    test_gpu_permute/test_synth) and are downloaded; the oracle evaluates 6 sampled (i,j) columns (38 400 outputs,
    every M tile, ragged and full N tiles) with long-double accumulators."""
    o, v = 20, 80
    V, T, R0 = ctx.tensor_create((v, v, v, v)), ctx.tensor_create((v, v, o, o)), ctx.tensor_create((v, v, o, o))
    ctx.synth_normal(V, synth.SEED0 + 2, 1, antisym=((0, 1), (2, 3)), sigma=0.1)
    ctx.synth_normal(T, synth.SEED0 + 2, 2, antisym=((0, 1), (2, 3)))
    ctx.synth_normal(R0, synth.SEED0 + 2, 3)
    hV, hT, hR0 = ctx.tensor_download(V), ctx.tensor_download(T), ctx.tensor_download(R0)
    expr = "R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)"
    ctx.contract(expr, R0, V, T, 0.5)
    got = ctx.tensor_download(R0)
    plan = ctx.plan_describe(expr, R0, V, T)
    assert (plan["M"], plan["N"], plan["K"]) == (6400, 400, 6400)
    worst = 0.0
    for (i, j) in [(0, 0), (3, 0), (19, 19), (7, 12), (12, 7), (5, 16)]:
        Tc = np.asfortranarray(hT[:, :, i:i + 1, j:j + 1])
        Rc = np.asfortranarray(hR0[:, :, i:i + 1, j:j + 1])
        ref, sn = oracle.contract(expr, Rc, hV, Tc, 0.5)
        worst = max(worst, parity_error(np.asfortranarray(got[:, :, i:i + 1, j:j + 1]), ref, sn))
    assert worst <= TOL
    for t in (V, T, R0):
        t.destroy()


@pytest.mark.parametrize("o,v", [(3, 5), (4, 9)])
def test_every_ccsd_contraction_in_every_emitted_output_order(ctx, o, v):
    """BASELINE.json configs[4] (first half) at oracle-sized extents: all 32 binary contractions of the CCSD list, each in
    every output index order its permutation operators unroll into (rank 2-4, K = 1 and N = 1 included)."""
    from paper_2409_06759_b200 import ccsd_contractions as cl
    rng = np.random.default_rng(o * 100 + v)
    worst = 0.0
    for e, sign, sd, sl, sr in cl.all_calls(o, v):
        D, L, R = rc(rng, *sd), rc(rng, *sl), rc(rng, *sr)
        dD, dL, dR = ctx.tensor_from_numpy(D), ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R)
        ctx.contract(e, dD, dL, dR, 0.5 * sign)
        got = ctx.tensor_download(dD)
        ref, sn = oracle.contract(e, D, L, R, 0.5 * sign)
        err = parity_error(got, ref, sn)
        assert err <= TOL, (e, err)
        worst = max(worst, err)
        for t in (dD, dL, dR):
            t.destroy()
    assert worst <= TOL


@pytest.mark.parametrize("expr,ext", [
    ("D(a,e)+=L(m,a,f,e)*R(f,m)", dict(a=13, e=11, m=5, f=7)),            # k-fast: L's unit-stride index is contracted
    ("D(a,i)=L(a,e,i,m)*R(m,e)", dict(a=40, i=9, e=17, m=6)),             # m-fast: L's unit-stride index is free
    ("D(i)+=R(k,j)*L(j,i,k)", dict(i=3, j=300, k=301)),                   # few rows, long K: K cut, operands swapped
    ("D(a,b)+=L(a,k,b)*R(k)", dict(a=700, b=3, k=2500)),                  # m-fast with the K cut
])
def test_gemv_route_reads_the_operand_in_place(ctx, expr, ext):
    """N = 1 (one operand contracted away): no permutation, tables of row / column offsets, deterministic K split"""
    from gpu_util import split_expr
    rng = np.random.default_rng(sum(ext.values()))
    dl, ll, rl = split_expr(expr)
    D, L, R = rc(rng, *[ext[x] for x in dl]), rc(rng, *[ext[x] for x in ll]), rc(rng, *[ext[x] for x in rl])
    dD, dL, dR = ctx.tensor_from_numpy(D), ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R)
    plan = ctx.plan_describe(expr, dD, dL, dR)
    assert plan["route"] == "gemv" and not plan["permute_A"] and not plan["permute_B"]
    alpha = 0.75 - 0.5j
    ctx.contract(expr, dD, dL, dR, alpha)
    got = ctx.tensor_download(dD)
    ref, sn = oracle.contract(expr, D, L, R, alpha)
    assert parity_error(got, ref, sn) <= TOL
    dD2 = ctx.tensor_from_numpy(D)
    ctx.contract(expr, dD2, dL, dR, alpha)
    assert ctx.tensor_download(dD2).tobytes() == got.tobytes()           # run-to-run identical
