"""-m gpu: index-permutation-symmetric packed storage against oracle/sym.py -- tcb_pack is bit-exact,
tcb_unpack with unit alpha is bit-exact, and the packed pp ladder matches the DENSE oracle contraction, also at the
configs[2] size (o=40, v=200) on sampled outputs."""
import numpy as np
import pytest

import oracle
from oracle import sym
import paper_2409_06759_b200 as pkg
from paper_2409_06759_b200 import binding, ccd, synth
from gpu_util import TOL, rc, parity_error, sample_indices, download_at

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
