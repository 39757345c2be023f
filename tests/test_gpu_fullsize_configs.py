"""-m gpu: every workload bench.py times, checked at the size and in the launch configuration it is timed in
(north_star: "every config matches the oracle within tolerance ... permutations must be bit-exact"; the paper's own method,
PAPER.md:266: brute-force nested loops against the optimised code).  The oracle cannot run these sizes whole, so it runs on
sampled outputs: operands are generated on the device by the seeded generator and REGENERATED on the host by
its index-keyed twin (synth.py) for the sampled rows and columns -- nothing the oracle reads comes from the device.
Transpositions are checked in closed form over the WHOLE output (re = linear input index, im = -index - 0.5)."""
import itertools

import numpy as np
import pytest

import oracle
import paper_2409_06759_b200 as pkg
from paper_2409_06759_b200 import synth
from gpu_util import TOL, rc, parity_error, sampled_contraction_parity, sample_indices, download_at, slab

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    c = pkg.Context(0)
    yield c
    c.destroy()


def test_claim_ahead_schedule_full_parity(ctx):
    """zgemm's claim-one-tile-ahead mode (>= 8 x 296 whole tiles): 3200 x 3200 x 8 = 2500 tiles, every element checked"""
    m = n = 3200
    k = 8
    rng = np.random.default_rng(17)
    D, L, R = rc(rng, m, n), rc(rng, m, k), rc(rng, k, n)
    dD, dL, dR = ctx.tensor_from_numpy(D), ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(R)
    p = ctx.plan_describe("C(m,n)+=A(m,k)*B(k,n)", dD, dL, dR)
    assert (p["M"] + 63) // 64 * ((p["N"] + 63) // 64) >= 8 * 296 and p["splits"] == 1
    ctx.contract("C(m,n)+=A(m,k)*B(k,n)", dD, dL, dR, 0.5 - 0.25j)
    got = ctx.tensor_download(dD)
    ref, sn = oracle.contract("C(m,n)+=A(m,k)*B(k,n)", D, L, R, 0.5 - 0.25j)
    assert parity_error(got, ref, sn) <= TOL
    for t in (dD, dL, dR):
        t.destroy()


def test_configs2_ladder_fullsize_sampled(ctx):
    """BASELINE.json configs[2]: R(a,b,i,j) += 1/2 V(a,b,c,d) T(c,d,i,j), o=40, v=200 (40000 x 1600 x 40000, V 25.6 GB,
    15 625 tiles: claim-ahead mode + stream-K remainder), in the canonical order and with T given as T(i,j,c,d) and V as
    V(c,d,a,b); 3 sample sets of 8^4 = 4096 outputs each per variant, long-double oracle over K = 40 000."""
    o, v = 40, 200
    seed = synth.SEED0 + 3
    rng = np.random.default_rng(3)
    ext = dict(a=v, b=v, c=v, d=v, i=o, j=o)
    anti = ((0, 1), (2, 3))
    V = ctx.tensor_create((v, v, v, v))
    ctx.synth_normal(V, seed, 1, antisym=anti)
    R = ctx.tensor_create((v, v, o, o))
    for expr, t_shape in (("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", (v, v, o, o)),
                          ("R(a,b,i,j)+=V(a,b,c,d)*T(i,j,c,d)", (o, o, v, v)),
                          ("R(a,b,i,j)+=V(c,d,a,b)*T(c,d,i,j)", (v, v, o, o))):
        T = ctx.tensor_create(t_shape)
        ctx.synth_normal(T, seed, 2, antisym=anti)
        p = ctx.plan_describe(expr, R, V, T)
        assert (p["M"], p["N"], p["K"]) == (40000, 1600, 40000) and not p["permute_A"] and not p["permute_B"]
        err, n = sampled_contraction_parity(ctx, expr, ext, 0.5, seed, rng, nsub=8, antisym_l=anti, antisym_r=anti,
                                            sets=3, operands=(V, T, R))
        assert n >= 3 * 4096 and err <= TOL, (expr, err)
        T.destroy()
    V.destroy(); R.destroy()


def test_configs3_t3_contraction_fullsize_sampled(ctx):
    """BASELINE.json configs[3], first stage: X(a,b,c,i,j,k) = sum_d W(b,c,d,k) T2(a,d,i,j), o=12, v=60
    (8640 x 43200 x 60, 91 125 tiles, X 5.97 GB); 4 sample sets of 4^6 = 4096 outputs"""
    o, v = 12, 60
    ext = dict(a=v, b=v, c=v, d=v, i=o, j=o, k=o)
    rng = np.random.default_rng(4)
    err, n = sampled_contraction_parity(ctx, "X(a,b,c,i,j,k)=W(b,c,d,k)*T(a,d,i,j)", ext, 1.0, synth.SEED0 + 4, rng,
                                        nsub=4, antisym_l=((0, 1),), antisym_r=((0, 1), (2, 3)), sets=4)
    assert n == 4 * 4096 and err <= TOL


def test_configs3_nine_term_antisymmetriser_fullsize_sampled_bit_exact(ctx):
    """BASELINE.json configs[3], second stage: R3 += P(a/bc) P(k/ij) X on 60^3 x 12^3 (the orbit kernel with 1000 cubes per
    slab, 1728 slabs, 64-bit slab offsets).  A set S_v^3 x S_o^3 of index values is closed under the nine permutations,
    so the oracle's permute-sum on that sub-tensor IS the full result there: bit-exact, 4 sets of 4^6 = 4096 outputs."""
    o, v = 12, 60
    seed = synth.SEED0 + 4
    X, R3 = ctx.tensor_create((v, v, v, o, o, o)), ctx.tensor_create((v, v, v, o, o, o))
    ctx.synth_normal(X, seed, 4)
    ctx.synth_normal(R3, seed, 3)
    ctx.antisymmetrize("P(a/bc)P(k/ij):R(a,b,c,i,j,k)+=X(a,b,c,i,j,k)", R3, X, 1.0)
    rng = np.random.default_rng(9)
    lab = "abcijk"
    perms, coefs = [], []
    for (sv, pv) in ((1, "abc"), (-1, "bac"), (-1, "cba")):                 # P(a/bc) = 1 - (a<->b) - (a<->c)
        for (so, po) in ((1, "ijk"), (-1, "kji"), (-1, "ikj")):             # P(k/ij) = 1 - (k<->i) - (k<->j)
            perms.append([lab.index(x) for x in pv + po])
            coefs.append(sv * so)
    for s in range(4):
        Sv, So = sample_indices(rng, v, 4, edges=(s == 0)), sample_indices(rng, o, 4, edges=(s == 0))
        sub = [Sv, Sv, Sv, So, So, So]
        hX = synth.tensor(seed, 4, [v, v, v, o, o, o], sub=sub)
        hR = synth.tensor(seed, 3, [v, v, v, o, o, o], sub=sub)
        ref = oracle.permsum(hR, hX, perms, coefs, 1.0)
        got = download_at(ctx, R3, sub)
        assert got.tobytes() == ref.tobytes(), f"sample set {s}"
    X.destroy(); R3.destroy()


def _check_transpose_whole_output(ctx, shape, perm, chunk_elems=1 << 25):
    """D(perm) = L with L[idx] = (lin(idx), -lin(idx) - 0.5): every output element checked in closed form, the output
    downloaded in slabs of its last index"""
    lab = "abcdef"[:len(shape)]
    oshape = tuple(shape[p] for p in perm)
    L, D = ctx.tensor_create(shape, zero=False), ctx.tensor_create(oshape, zero=False)
    ctx.synth_index_linear(L)
    e = "D(" + ",".join(lab[p] for p in perm) + ")=L(" + ",".join(lab) + ")"
    ctx.permute(e, D, L)
    istride = np.cumprod([1] + list(shape[:-1])).astype(np.float64)
    # expected linear input index of the output slab [.., q]: sum over output dims of idx * istride[perm[dim]]
    lead = np.zeros(oshape[:-1], dtype=np.float64, order="F")
    for d in range(len(oshape) - 1):
        view = [1] * (len(oshape) - 1)
        view[d] = oshape[d]
        lead = lead + (np.arange(oshape[d], dtype=np.float64) * istride[perm[d]]).reshape(view)
    lead = np.asfortranarray(lead)
    for q in range(oshape[-1]):
        view = slab(ctx, D, q)
        got = ctx.tensor_download(view)
        view.destroy()
        lin = lead + q * istride[perm[-1]]
        assert np.array_equal(got.real, lin) and np.array_equal(got.imag, -lin - 0.5), (shape, perm, q)
    L.destroy(); D.destroy()


@pytest.mark.parametrize("shape,perm", [
    ((200, 200, 40, 40), (2, 3, 0, 1)),          # 1.02 GB, T(a,b,i,j) -> (i,j,a,b)
    ((200, 200, 40, 40), (1, 0, 3, 2)),
    ((60, 60, 60, 12, 12, 12), (3, 4, 5, 0, 1, 2)),   # 5.97 GB, the (i,j,k,a,b,c) half swap
    ((60, 60, 60, 12, 12, 12), (1, 0, 2, 3, 4, 5)),   # a single transposition of P(a/bc)
    ((150, 150, 150, 150), (3, 2, 1, 0)),        # 8.1 GB, full reversal
    ((150, 150, 150, 150), (0, 2, 1, 3)),
])
def test_configs4_transpositions_whole_output_closed_form(ctx, shape, perm):
    _check_transpose_whole_output(ctx, shape, perm)


def test_transposition_with_64bit_tile_offsets(ctx):
    """permute_kernel<.., long long>: a tile-local offset of 2^31 elements and more (a 2-D transpose whose long dim has
    2^26 + 8 elements and whose tile spans 33 of the other): 35 GB in, 35 GB out, sampled slabs checked in closed form"""
    n0, n1 = (1 << 26) + 8, 33
    L, D = ctx.tensor_create((n0, n1), zero=False), ctx.tensor_create((n1, n0), zero=False)
    ctx.synth_index_linear(L)
    ctx.permute("D(b,a)=L(a,b)", D, L)
    rng = np.random.default_rng(1)
    rows = sorted(set(rng.integers(0, n0, size=48).tolist()) | {0, 1, n0 - 1, n0 // 2})
    for a in rows:                                  # D[:, a] = L[a, :]: linear input index a + n0 * b
        view = slab(ctx, D, a)
        got = ctx.tensor_download(view)
        view.destroy()
        lin = a + n0 * np.arange(n1, dtype=np.float64)
        assert np.array_equal(got.real, lin) and np.array_equal(got.imag, -lin - 0.5), a
    L.destroy(); D.destroy()


def test_configs4_ccsd_contraction_list_fullsize_sampled(ctx):
    """BASELINE.json configs[4], first half: every binary contraction of the CCSD list at o=30, v=150 whose tensors hold
    100 MB or more, in every emitted output order, on sampled outputs (per free label 6 index values, every contracted
    index value: 36 ... 1296 outputs per call, K up to 675 000 with the long-double oracle)."""
    from paper_2409_06759_b200 import ccsd_contractions as cl
    from gpu_util import split_expr
    o, v = 30, 150
    rng = np.random.default_rng(5)
    seen, worst = 0, 0.0
    for e, sign, sd, sl, sr in cl.all_calls(o, v):
        if 16 * (np.prod(sd) + np.prod(sl) + np.prod(sr)) < 100e6:
            continue
        dl, ll, rl = split_expr(e)
        ext = {}
        for labs, shp in ((dl, sd), (ll, sl), (rl, sr)):
            ext.update(dict(zip(labs, shp)))
        err, n = sampled_contraction_parity(ctx, e, ext, 0.5 * sign, synth.SEED0 + 5, rng, nsub=6)
        assert err <= TOL, (e, err)
        worst = max(worst, err)
        seen += 1
    assert seen >= 20 and worst <= TOL


PACKED_CCSDT_CALLS = [  # the contractions of ccd.ccsdt_residual_packed that hold >= 100 MB at o=16, v=100, on their packed extents
    ("X(a,i,x,y)=W(m,a,i,e)*T(x,y,e,m)", 1.0),        # ring term: 1600 x 594000 x 1600, T and X 15.2 GB, operand permuted
    ("X(x,c,t)=W(x,z)*T(z,c,t)", 2.0),                # vvvv term on a<b, d<e, i<j<k: 4950 x 56000 x 4950
    ("X(x,c,t)+=T(x,e,t)*F(c,e)", 1.0),               # K = 100 accumulation into 4.4 GB
    ("X(t,y,k)=T(t,z,k)*W(z,y)", 2.0),                # oooo term on a<b<c, l<m: 2587200 x 120 x 120
    ("X(t,y,k)+=T(t,y,m)*F(m,k)", 1.0),               # K = 16
    ("X(a,i,x,y)+=W(x,i,d)*T(d,a,y)", 1.0),           # 12000 x 79200 x 100 accumulation into 15.2 GB
    ("X(a,i,x,y)+=W(l,a,y)*T(x,l,i)", 1.0),           # K = 16
    ("W(x,i,d)+=T(x,z,e,i)*g(z,d,e)", -0.25),         # 79200 x 100 x 12000, T3 view gathered
    ("W(l,a,y)+=g(l,m,z)*T(z,y,a,m)", -0.25),         # 16 x 12000 x 79200
    ("X(x,i,j)=T(x,z,d,j)*W(z,i,d)", 2.0),            # doubles <- T3: 79200 x 16 x 12000
    ("X(a,b,y)=W(l,a,z)*T(z,y,b,l)", 2.0),            # doubles <- T3: 100 x 12000 x 79200
    ("R(x,y)=T(x,y,d,l)*f(l,d)", 1.0),                # GEMV over a 15.2 GB view
    ("R(a,i)+=T(x,y,a,i)*W(y,x)", 1.0),               # GEMV, K = 594000
]


def test_packed_ccsdt_contractions_at_the_timed_size_sampled(ctx):
    """bench.py times ccd.ccsdt_residual_packed at o=16, v=100 (dense T3: 65.5 GB per tensor).  Every contraction of that
    program that touches a packed view of T3 or a packed accumulator, with the packed extents it has there (pairs 4950 / 120,
    triples 161700 / 560), on sampled outputs: per free label 5 index values, every contracted index value, long-double
    oracle on host-regenerated operands."""
    from gpu_util import split_expr
    o, v = 16, 100
    nv2, nv3, no2, no3 = v * (v - 1) // 2, v * (v - 1) * (v - 2) // 6, o * (o - 1) // 2, o * (o - 1) * (o - 2) // 6
    # extents by the role a label plays in the driver's expressions
    sizes = {"X(a,i,x,y)=W(m,a,i,e)*T(x,y,e,m)": dict(a=v, i=o, x=nv2, y=no2, m=o, e=v),
             "X(x,c,t)=W(x,z)*T(z,c,t)": dict(x=nv2, z=nv2, c=v, t=no3),
             "X(x,c,t)+=T(x,e,t)*F(c,e)": dict(x=nv2, c=v, e=v, t=no3),
             "X(t,y,k)=T(t,z,k)*W(z,y)": dict(t=nv3, y=no2, z=no2, k=o),
             "X(t,y,k)+=T(t,y,m)*F(m,k)": dict(t=nv3, y=no2, m=o, k=o),
             "X(a,i,x,y)+=W(x,i,d)*T(d,a,y)": dict(a=v, i=o, x=nv2, y=no2, d=v),
             "X(a,i,x,y)+=W(l,a,y)*T(x,l,i)": dict(a=v, i=o, x=nv2, y=no2, l=o),
             "W(x,i,d)+=T(x,z,e,i)*g(z,d,e)": dict(x=nv2, i=o, d=v, z=no2, e=v),
             "W(l,a,y)+=g(l,m,z)*T(z,y,a,m)": dict(l=o, a=v, y=no2, m=o, z=nv2),
             "X(x,i,j)=T(x,z,d,j)*W(z,i,d)": dict(x=nv2, i=o, j=o, z=no2, d=v),
             "X(a,b,y)=W(l,a,z)*T(z,y,b,l)": dict(a=v, b=v, y=no2, l=o, z=nv2),
             "R(x,y)=T(x,y,d,l)*f(l,d)": dict(x=nv2, y=no2, d=v, l=o),
             "R(a,i)+=T(x,y,a,i)*W(y,x)": dict(a=v, i=o, x=nv2, y=no2)}
    rng = np.random.default_rng(16)
    worst = 0.0
    for k, (e, alpha) in enumerate(PACKED_CCSDT_CALLS):
        err, n = sampled_contraction_parity(ctx, e, sizes[e], alpha, synth.SEED0 + 40 + k, rng, nsub=5, sigma=0.5)
        assert err <= TOL and n >= 25, (e, err, n)
        worst = max(worst, err)
    assert worst <= TOL


def test_packed_ccsd_ladder_contractions_at_the_timed_size_sampled(ctx):
    """bench.py times ccd.ccsd_residual(packed={}) at o=30, v=150: its two contractions on packed indices (pairs 11175 / 435)
    on sampled outputs, as above."""
    o, v = 30, 150
    nv2, no2 = v * (v - 1) // 2, o * (o - 1) // 2
    rng = np.random.default_rng(30)
    for k, (e, alpha, ext) in enumerate([("R(x,y)=W(x,z)*t(z,y)", 1.0, dict(x=nv2, y=no2, z=nv2)),
                                         ("X(a,b,z)=V(a,m,z)*T1(b,m)", 1.0, dict(a=v, b=v, z=nv2, m=o))]):
        err, n = sampled_contraction_parity(ctx, e, ext, alpha, synth.SEED0 + 60 + k, rng, nsub=8, sigma=0.5)
        assert err <= TOL and n >= 64, (e, err, n)
