"""-m gpu: index-permutation-symmetric packed storage against oracle/sym.py -- tcb_pack is bit-exact,
tcb_unpack with unit alpha is bit-exact, and the packed pp ladder matches the DENSE oracle contraction, also at the
configs[2] size (o=40, v=200) on sampled outputs."""
import numpy as np
import pytest

import oracle
from oracle import sym
import paper_2409_06759_b200 as pkg
from paper_2409_06759_b200 import binding, ccd, synth
from gpu_util import TOL, rc, parity_error, sample_indices, download_at, slab

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    c = pkg.Context(0)
    yield c
    c.destroy()


PACK_CASES = [
    ("Tp(a<b,i<j)=T(a,b,i,j)", (7, 7, 5, 5)),
    ("Tp(i<j,a<b)=T(a,b,i,j)", (7, 7, 5, 5)),              # groups in another order
    ("Wp(a<b,i<j)=W(a,i,b,j)", (6, 4, 6, 4)),              # group members not adjacent in the dense tensor
    ("Tq(a<b,i,j)=T(a,b,i,j)", (9, 9, 3, 4)),              # a group beside plain indices
    ("Tq(i,a<b,j)=T(a,b,i,j)", (9, 9, 3, 4)),
    ("T3(a<b<c,i<j<k)=T(a,b,c,i,j,k)", (7, 7, 7, 4, 4, 4)),  # triples (T3 amplitudes: 36x less memory)
    ("T3(i<j<k,c,a<b)=T(a,b,c,i,j,k)", (5, 5, 6, 4, 4, 4)),
    ("Vp(x<y)=V(x,y)", (300, 300)),
]


@pytest.mark.parametrize("spec,shape", PACK_CASES)
def test_pack_is_bit_exact(ctx, spec, shape):
    rng = np.random.default_rng(len(spec))
    L = rc(rng, *shape)
    ref = sym.pack(spec, L)
    dL, dD = ctx.tensor_from_numpy(L), ctx.tensor_create(ref.shape, zero=False)
    ctx.pack(spec, dD, dL)
    assert ctx.tensor_download(dD).tobytes() == ref.tobytes()
    dL.destroy(); dD.destroy()


@pytest.mark.parametrize("spec,shape", PACK_CASES)
@pytest.mark.parametrize("op,alpha", [("=", 1.0), ("+=", 1.0), ("+=", -1.0), ("=", 0.5 - 2.0j)])
def test_unpack_matches_the_oracle(ctx, spec, shape, op, alpha):
    lhs, rhs = spec.split("=")
    uspec = rhs + op + lhs                                    # 'T(a,b,i,j)+=Tp(a<b,i<j)'
    labs = rhs[rhs.index("(") + 1:-1].split(",")
    rng = np.random.default_rng(len(spec) + 1)
    pshape = sym.pack(spec, np.zeros(shape)).shape
    Lp, D0 = rc(rng, *pshape), rc(rng, *shape)
    ref = sym.unpack(uspec, Lp, D=D0, alpha=alpha)
    dLp, dD = ctx.tensor_from_numpy(Lp), ctx.tensor_from_numpy(D0)
    ctx.unpack(uspec, dD, dLp, alpha)
    got = ctx.tensor_download(dD)
    if alpha in (1.0, -1.0):
        assert np.array_equal(got, ref)                      # +-1: one exact negation, one rounded addition -- same bits
    else:
        assert np.max(np.abs(got - ref)) <= 1e-15 * (np.abs(D0).max() + 3 * np.abs(Lp).max())
    dLp.destroy(); dD.destroy()


def test_round_trip_of_an_antisymmetric_tensor_is_bit_exact(ctx):
    T = synth.tensor(synth.SEED0, 2, [24, 24, 8, 8], antisym=((0, 1), (2, 3)))
    dT = ctx.tensor_from_numpy(T)
    dP = ctx.tensor_create((ctx.packed_extent(24, 2), ctx.packed_extent(8, 2)), zero=False)
    dU = ctx.tensor_create(T.shape, zero=False)
    ctx.pack("Tp(a<b,i<j)=T(a,b,i,j)", dP, dT)
    ctx.unpack("T(a,b,i,j)=Tp(a<b,i<j)", dU, dP, 1.0)
    assert np.array_equal(ctx.tensor_download(dU), T)
    for t in (dT, dP, dU):
        t.destroy()


def test_bad_specs_are_rejected_and_leave_the_context_usable(ctx):
    T, P = ctx.tensor_create((5, 5, 3, 3)), ctx.tensor_create((10, 4))
    for spec, D, L, code in [("Tp(a<b,i<j)=T(a,b,i,j)", P, T, binding.TCB_ESHAPE),              # packed extent of (i<j) must be 3
                             ("Tp(a,b,i,j)=T(a,b,i,j)", T, T, binding.TCB_EINVAL_EXPR),          # no group
                             ("Tp(a<i,b<j)=T(a,b,i,j)", P, T, binding.TCB_ESHAPE),               # unequal extents in a group
                             ("Tp(a<b,i<j)+=T(a,b,i,j)", P, T, binding.TCB_EINVAL_EXPR),
                             ("Tp(a<b,i<j=T(a,b,i,j)", P, T, binding.TCB_EINVAL_EXPR)]:
        with pytest.raises(pkg.TcbError) as ei:
            ctx.pack(spec, D, L)
        assert ei.value.code == code, spec
    assert ctx.packed_extent(200, 2) == 19900 and ctx.packed_extent(60, 3) == 34220 and ctx.packed_extent(5, 4) == -1
    ctx.tensor_fill(T, 1.0)
    ctx.sync()


def test_packed_pp_ladder_matches_the_dense_oracle(ctx):
    o, v = 6, 14
    V, T = synth.config_ladder(o, v, 1)
    R0 = synth.tensor(synth.SEED0 + 1, 3, [v, v, o, o], antisym=((0, 1), (2, 3)))
    dV, dT, dR = ctx.tensor_from_numpy(V), ctx.tensor_from_numpy(T), ctx.tensor_from_numpy(R0)
    Vp = ccd.pp_ladder_packed(ctx, dR, dV, dT)
    got = ctx.tensor_download(dR)
    ref, sn = oracle.contract("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", R0, V, T, 0.5)
    assert parity_error(got, ref, sn) <= TOL
    assert np.array_equal(got, -got.transpose(1, 0, 2, 3)) and np.array_equal(got, -got.transpose(0, 1, 3, 2))
    for t in (dV, dT, dR, Vp):
        t.destroy()


def test_packed_pp_ladder_fullsize_sampled_and_faster_than_dense(ctx):
    """configs[2] on packed storage: Vp 19900 x 19900 (6.3 GB instead of 25.6 GB), GEMM 19900 x 780 x 19900 = 1/8 of the dense
    flops; sampled outputs against the DENSE long-double oracle (K = 40 000 terms each), operands regenerated on the host"""
    o, v = 40, 200
    seed, anti = synth.SEED0 + 3, ((0, 1), (2, 3))
    V, T, R = ctx.tensor_create((v, v, v, v), zero=False), ctx.tensor_create((v, v, o, o), zero=False), ctx.tensor_create((v, v, o, o))
    ctx.synth_normal(V, seed, 1, antisym=anti)
    ctx.synth_normal(T, seed, 2, antisym=anti)
    nv = ctx.packed_extent(v, 2)
    Vp = ctx.tensor_create((nv, nv), zero=False)
    ctx.pack("Vp(a<b,c<d)=V(a,b,c,d)", Vp, V)
    ccd.pp_ladder_packed(ctx, R, V, T, Vp=Vp)
    rng = np.random.default_rng(6)
    worst = 0.0
    for s in range(2):
        pa, pb = sample_indices(rng, v, 8, edges=(s == 0)), sample_indices(rng, v, 8, edges=(s == 0))
        pi, pj = sample_indices(rng, o, 8, edges=(s == 0)), sample_indices(rng, o, 8, edges=(s == 0))
        full = np.arange(v)
        hV = synth.tensor(seed, 1, [v] * 4, antisym=anti, sub=[pa, pb, full, full])
        hT = synth.tensor(seed, 2, [v, v, o, o], antisym=anti, sub=[full, full, pi, pj])
        ref, sn = oracle.contract("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", np.zeros((8, 8, 8, 8)), hV, hT, 0.5)
        got = download_at(ctx, R, [pa, pb, pi, pj])
        worst = max(worst, parity_error(got, ref, sn))
    assert worst <= TOL
    # timing: packed (pack T + GEMM + unpack; V packed once) against the dense call on the same device
    def timed(fn, reps=3):
        fn(); ctx.sync()
        ts = []
        for _ in range(reps):
            ctx.timer_start(); fn(); ts.append(ctx.timer_stop())
        return min(ts)
    t_dense = timed(lambda: ctx.contract("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", R, V, T, 0.5))
    t_packed = timed(lambda: ccd.pp_ladder_packed(ctx, R, V, T, Vp=Vp))
    assert t_dense / t_packed >= 5.0, (t_dense, t_packed)
    for t in (V, T, R, Vp):
        t.destroy()


# ---- packed views of packed tensors (tcb_unpack with groups on D) and tcb_antisym_pack ----------------------------------------
VIEW_CASES = [("Tq(d<e,c,i<j<k)=T(d<e<c,i<j<k)", dict(d=7, e=7, c=7, i=5, j=5, k=5)),
              ("To(a<b<c,l<m,k)=T(a<b<c,l<m<k)", dict(a=7, b=7, c=7, l=5, m=5, k=5)),
              ("Tr(b<c,j<k,e,m)=T(b<c<e,j<k<m)", dict(b=6, c=6, e=6, j=5, k=5, m=5)),
              ("Tr(j<k,e,b<c,m)=T(e<b<c,m<j<k)", dict(b=6, c=6, e=6, j=5, k=5, m=5)),
              ("Ts(a<c,b,i)=T(a<b<c,i)", dict(a=9, b=9, c=9, i=3)),
              ("D(a<b,c)=L(a,b<c)", dict(a=8, b=8, c=8)),                            # regrouping: zeros at b == c
              ("D(x<y,p)=L(p,y,x)", dict(x=11, y=11, p=4)),                          # dense L: a pack with a transposition
              # index 0 of D >= 128: the tiled kernel; 2080 pairs = one full tile of 2048 + a ragged one
              ("Tq(d<e,c,q)=T(d<e<c,q)", dict(d=65, e=65, c=65, q=3)),
              ("Tr(b<c,j<k,e,m)=T(b<c<e,j<k<m)", dict(b=17, c=17, e=17, j=5, k=5, m=5)),
              ("D(p,x<y)=L(y,x,p)", dict(x=9, y=9, p=130)),                          # a plain index first
              ("To(a<b<c,l<m,k)=T(a<b<c,l<m<k)", dict(a=12, b=12, c=12, l=5, m=5, k=5))]


def _shape(groups, ext):
    return tuple(sym.packed_extent(ext[g[0]], len(g)) for g in groups)


@pytest.mark.parametrize("spec,ext", VIEW_CASES)
@pytest.mark.parametrize("op,alpha", [("=", 1.0), ("+=", -1.0), ("+=", 0.75 + 0.5j)])
def test_packed_views_match_the_oracle(ctx, spec, ext, op, alpha):
    dg, lg, _ = sym.parse_both(spec)
    rng = np.random.default_rng(len(spec) + len(op))
    L, D0 = rc(rng, *_shape(lg, ext)), rc(rng, *_shape(dg, ext))
    uspec = spec.replace("=", op, 1)
    ref = sym.unpack(uspec, L, D=D0, alpha=alpha)
    dL, dD = ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(D0)
    ctx.unpack(uspec, dD, dL, alpha)
    got = ctx.tensor_download(dD)
    if alpha in (1.0, -1.0):
        assert np.array_equal(got, ref)
    else:
        assert np.max(np.abs(got - ref)) <= 1e-15 * (np.abs(D0).max() + 3 * np.abs(L).max())
    dL.destroy(); dD.destroy()


MERGE_CASES = [("R(a<b<c,i<j<k)=X(a,i,b<c,j<k)", dict(a=7, b=7, c=7, i=5, j=5, k=5), 9),
               ("R(a<b<c,i<j<k)=X(b<c,a,i<j<k)", dict(a=7, b=7, c=7, i=5, j=5, k=5), 3),
               ("R(a<b<c,i<j<k)=X(a<b<c,j<k,i)", dict(a=7, b=7, c=7, i=5, j=5, k=5), 3),
               ("R(a<b<c,i<j<k)=X(a,b,c,i,j,k)", dict(a=5, b=5, c=5, i=4, j=4, k=4), 36),
               ("R(i<j,a<b)=X(a,i,b,j)", dict(a=9, b=9, i=6, j=6), 4),
               ("R(a<b<c,q)=X(c,q,a<b)", dict(a=10, b=10, c=10, q=3), 3),
               ("R(a<b<c,i<j<k)=X(a<b<c,i<j<k)", dict(a=6, b=6, c=6, i=5, j=5, k=5), 1),
               # index 0 of D >= 128: the tiled kernel
               ("R(a<b<c,i<j<k)=X(a,i,b<c,j<k)", dict(a=12, b=12, c=12, i=5, j=5, k=5), 9),
               ("R(a<b<c,i<j<k)=X(a<b,i,c,j<k)", dict(a=12, b=12, c=12, i=5, j=5, k=5), 9),
               ("R(a<b<c,q)=X(b<c,a,q)", dict(a=13, b=13, c=13, q=4), 3),
               ("R(a<b,i<j)=X(a,i,b,j)", dict(a=18, b=18, i=4, j=4), 4),
               ("R(a<b<c,i<j<k)=X(a,b,c,i,j,k)", dict(a=11, b=11, c=11, i=4, j=4, k=4), 36)]


@pytest.mark.parametrize("spec,ext,nterms", MERGE_CASES)
@pytest.mark.parametrize("op,alpha", [("=", 1.0), ("+=", 4.0), ("+=", 0.5 - 1.5j)])
def test_antisym_pack_matches_the_oracle_within_the_north_star_tolerance(ctx, spec, ext, nterms, op, alpha):
    """the shuffle sum under snorm = |alpha| * (sum over the shuffles of |L|) + |D_in|, element by element"""
    dg, lg, _ = sym.parse_both(spec)
    rng = np.random.default_rng(nterms + len(spec))
    L, D0 = rc(rng, *_shape(lg, ext)), rc(rng, *_shape(dg, ext))
    uspec = spec.replace("=", op, 1)
    ref = sym.antisym_pack(uspec, L, D=D0, alpha=alpha)
    # |terms| summed: the same call on |L| with every sign made + is not available, so bound it by nterms * max over reads
    snorm = abs(alpha) * nterms * np.abs(L).max() + (np.abs(D0) if op == "+=" else 0.0)
    dL, dD = ctx.tensor_from_numpy(L), ctx.tensor_from_numpy(D0)
    ctx.antisym_pack(uspec, dD, dL, alpha)
    got = ctx.tensor_download(dD)
    assert np.max(np.abs(got - ref) / snorm) <= TOL
    if nterms == 1 and alpha == 1.0 and op == "=":
        assert np.array_equal(got, L)
    dL.destroy(); dD.destroy()


def test_antisym_pack_and_view_errors(ctx):
    P3, P2, Dn = ctx.tensor_create((20, 4)), ctx.tensor_create((6, 15)), ctx.tensor_create((6, 6, 6))
    for fn, spec, D, L, code in [(ctx.antisym_pack, "R(a<b,c)=X(a,b<c)", ctx.tensor_create((15, 6)), P2, binding.TCB_EINVAL_EXPR),
                                 (ctx.antisym_pack, "R(a<b<c,q)=X(a,b<c)", P3, P2, binding.TCB_EINVAL_EXPR),   # q on one side
                                 (ctx.antisym_pack, "R(a<b<c,q)=X(q,a,b<c)", P3, P2, binding.TCB_ESHAPE),      # rank of X
                                 (ctx.unpack, "D(a<b,c)=L(a,b<c)", ctx.tensor_create((14, 6)), P2, binding.TCB_ESHAPE),
                                 (ctx.unpack, "D(a<b,c)=L(a,b<d)", ctx.tensor_create((15, 6)), P2, binding.TCB_EINVAL_EXPR),
                                 (ctx.antisym_pack, "R(a<b<c)=X(a,b,c)", Dn, Dn, binding.TCB_ESHAPE)]:
        with pytest.raises(pkg.TcbError) as ei:
            fn(spec, D, L, 1.0)
        assert ei.value.code == code, spec
    R = ctx.tensor_create((20,))
    ctx.antisym_pack("R(a<b<c)=X(a,b,c)", R, Dn, 1.0)           # the context still works
    ctx.sync()


@pytest.mark.parametrize("o,v", [(12, 60), (16, 100)])
def test_packed_t3_views_and_antisymmetriser_at_the_ccsdt_size(ctx, o, v):
    """o = 12, v = 60 (the CCSDT bench size): T3p(a<b<c,i<j<k) is 120 MB instead of 6 GB; o = 16, v = 100: 1.45 GB instead of
    65.5 GB, the view and X of 15.2 GB each (byte offsets beyond 2^33).  Sampled elements of the view Tr and of the 9-term
    packed antisymmetriser against the oracle's rule evaluated one by one on host copies."""
    nv2, nv3, no2, no3 = (ctx.packed_extent(v, 2), ctx.packed_extent(v, 3), ctx.packed_extent(o, 2), ctx.packed_extent(o, 3))
    Tp = ctx.tensor_create((nv3, no3), zero=False)
    ctx.synth_normal(Tp, synth.SEED0, 41)
    hTp = ctx.tensor_download(Tp)
    tv3 = {t: p for p, t in enumerate(sym.tuples(v, 3))}
    to3 = {t: p for p, t in enumerate(sym.tuples(o, 3))}
    pv2, po2 = sym.tuples(v, 2), sym.tuples(o, 2)

    def t3(abc, ijk):
        (sa, sga), (si, sgi) = sym._sort_sign(abc), sym._sort_sign(ijk)
        return 0.0 if sga * sgi == 0 else sga * sgi * hTp[tv3[sa], to3[si]]
    rng = np.random.default_rng(5)
    Tr = ctx.tensor_create((nv2, no2, v, o), zero=False)
    ctx.unpack("Tr(b<c,j<k,e,m)=T(b<c<e,j<k<m)", Tr, Tp, 1.0)
    for m in (0, 5, o - 1):
        view = slab(ctx, Tr, m)
        hs = ctx.tensor_download(view)
        view.destroy()
        for _ in range(100):
            x, y, e = (int(rng.integers(n)) for n in (nv2, no2, v))
            assert hs[x, y, e] == t3(pv2[x] + (e,), po2[y] + (m,))
    Tr.destroy()
    # the 9-term antisymmetriser of Xr(a,i,b<c,j<k) on packed storage
    Xr = ctx.tensor_create((v, o, nv2, no2), zero=False)
    ctx.synth_normal(Xr, synth.SEED0, 42)
    R = ctx.tensor_create((nv3, no3), zero=False)
    ctx.antisym_pack("R(a<b<c,i<j<k)=X(a,i,b<c,j<k)", R, Xr, 4.0)
    hX, hR = ctx.tensor_download(Xr), ctx.tensor_download(R)
    pv2i, po2i = {t: p for p, t in enumerate(pv2)}, {t: p for p, t in enumerate(po2)}
    lv3, lo3 = sym.tuples(v, 3), sym.tuples(o, 3)
    for _ in range(200):
        p, q = int(rng.integers(nv3)), int(rng.integers(no3))
        (a, b, c), (i, j, k) = lv3[p], lo3[q]
        ref, sn = 0.0, 0.0
        for (s, rest, sg) in ((a, (b, c), 1), (b, (a, c), -1), (c, (a, b), 1)):
            for (u, orest, sg2) in ((i, (j, k), 1), (j, (i, k), -1), (k, (i, j), 1)):
                w = hX[s, u, pv2i[rest], po2i[orest]]
                ref, sn = ref + sg * sg2 * w, sn + abs(w)
        assert abs(hR[p, q] - 4.0 * ref) <= TOL * 4.0 * sn
    for t in (Tp, Xr, R):
        t.destroy()


def test_packed_storage_calls_in_a_capture_cold_refused_warm_replayed():
    """the first use of an (extent, group size) builds a tuple table (tcb_pack: an offset table): refused inside a capture
    like a first plan; after one eager pass the same list is captured and the replay is bit-identical"""
    c = pkg.Context(0)
    rng = np.random.default_rng(8)
    n, m = 13, 6                                             # extents no other test of this module uses first
    Tp = rc(rng, sym.packed_extent(n, 3), m)
    X = rc(rng, n, m, sym.packed_extent(n, 2))
    dTp, dX = c.tensor_from_numpy(Tp), c.tensor_from_numpy(X)
    dV, dR = c.tensor_create((sym.packed_extent(n, 2), n, m)), c.tensor_create((sym.packed_extent(n, 3), m))
    calls = [lambda: c.unpack("V(a<b,c,q)=T(a<b<c,q)", dV, dTp, 1.0),
             lambda: c.antisym_pack("R(a<b<c,q)=X(a,q,b<c)", dR, dX, 2.0)]
    c.capture_begin()
    for f in calls:
        with pytest.raises(pkg.TcbError) as ei:
            f()
        assert ei.value.code == binding.TCB_EUNSUPPORTED
    with pytest.raises(pkg.TcbError):
        c.capture_end()
    for f in calls:
        f()
    want_v, want_r = c.tensor_download(dV), c.tensor_download(dR)
    assert np.array_equal(want_v, sym.unpack("V(a<b,c,q)=T(a<b<c,q)", Tp))
    c.capture_begin()
    for f in calls:
        f()
    g = c.capture_end()
    c.tensor_fill(dV, 0.0)
    c.tensor_fill(dR, 0.0)
    c.graph_launch(g)
    assert np.array_equal(c.tensor_download(dV), want_v) and np.array_equal(c.tensor_download(dR), want_r)
    c.graph_destroy(g)
    c.destroy()
