"""-m gpu: S3 (transposition, bit-exact), S6 (permute-sum), S7 (add / scale / fill) through the C ABI vs the oracle."""
import itertools

import numpy as np
import pytest

import oracle
from oracle import cc
import paper_2409_06759_b200 as pkg
from paper_2409_06759_b200 import synth
from gpu_util import rc

pytestmark = pytest.mark.gpu
LABELS = "abcdef"


@pytest.fixture(scope="module")
def ctx():
    c = pkg.Context(0)
    yield c
    c.destroy()


def pexpr(perm):
    r = len(perm)
    return "D(" + ",".join(LABELS[p] for p in perm) + ")=L(" + ",".join(LABELS[:r]) + ")"


def check_permutation(ctx, shape, perm, L=None):
    L = synth.index_linear_tensor(shape) if L is None else L
    dL = ctx.tensor_from_numpy(L)
    oshape = tuple(shape[p] for p in perm)
    dD = ctx.tensor_create(oshape)
    ctx.permute(pexpr(perm), dD, dL)
    got = ctx.tensor_download(dD)
    ref = oracle.permute(pexpr(perm), L, oshape)
    assert got.tobytes() == ref.tobytes(), (shape, perm)
    dL.destroy()
    dD.destroy()


@pytest.mark.parametrize("shape", [(33, 7, 13, 2), (5, 40, 3, 37), (1, 64, 65, 3), (70, 2, 2, 33)])
def test_all_24_rank4_permutations(ctx, shape):
    for perm in itertools.permutations(range(4)):
        check_permutation(ctx, shape, perm)


def test_sampled_rank6_permutations(ctx):
    rng = np.random.default_rng(5)
    all6 = list(itertools.permutations(range(6)))
    must = [(0, 1, 2, 3, 4, 5), (5, 4, 3, 2, 1, 0), (3, 4, 5, 0, 1, 2), (1, 0, 2, 3, 4, 5), (2, 1, 0, 3, 4, 5),
            (0, 2, 1, 3, 4, 5), (0, 1, 2, 4, 3, 5), (0, 1, 2, 5, 4, 3), (0, 1, 2, 3, 5, 4)]
    sample = must + [all6[i] for i in rng.choice(len(all6), 39, replace=False)]
    for shape in [(7, 5, 6, 3, 4, 2), (13, 1, 9, 2, 7, 3)]:
        for perm in sample:
            check_permutation(ctx, shape, perm)


@pytest.mark.parametrize("shape,perm", [((300, 5), (1, 0)), ((5, 300), (1, 0)), ((1000, 3, 2), (2, 0, 1)),
                                        ((2, 3, 1000), (2, 1, 0)), ((129, 130), (1, 0)), ((6, 5, 4, 3, 2), (4, 3, 2, 1, 0)),
                                        ((1, 1, 1), (2, 1, 0)), ((77,), (0,))])
def test_rank_1_2_3_5_and_ragged(ctx, shape, perm):
    check_permutation(ctx, shape, perm)


def test_special_values_are_moved_bit_exactly(ctx):
    """-0.0, NaN payloads, infinities, denormals survive (the kernel must not do arithmetic on a copy)."""
    shape = (9, 8, 5, 4)
    n = int(np.prod(shape))
    bits = np.random.default_rng(6).integers(0, 2 ** 63, size=2 * n, dtype=np.uint64)
    bits[:8] = [0x8000000000000000, 0x7FF8000000000123, 0xFFF0000000000000, 0x7FF0000000000000, 1, 0x000FFFFFFFFFFFFF,
                0x7FF4000000000001, 0]
    L = bits.view(np.float64).view(np.complex128).reshape(shape, order="F")
    for perm in [(3, 2, 1, 0), (1, 0, 3, 2), (2, 3, 0, 1)]:
        check_permutation(ctx, shape, perm, L)


def test_inverse_permutation_roundtrip(ctx):
    shape = (33, 6, 17, 5)
    L = rc(np.random.default_rng(7), *shape)
    dL = ctx.tensor_from_numpy(L)
    dM = ctx.tensor_create((6, 5, 33, 17))
    ctx.permute("M(b,d,a,c)=L(a,b,c,d)", dM, dL)
    dB = ctx.tensor_create(shape)
    ctx.permute("B(a,b,c,d)=M(b,d,a,c)", dB, dM)
    assert ctx.tensor_download(dB).tobytes() == L.tobytes()


def test_add_scale_fill(ctx):
    rng = np.random.default_rng(8)
    D, L = rc(rng, 30, 9, 31, 4), rc(rng, 9, 30, 4, 31)
    dD, dL = ctx.tensor_from_numpy(D), ctx.tensor_from_numpy(L)
    a = 0.7 - 0.2j
    ctx.add("D(a,b,i,j)+=L(b,a,j,i)", dD, dL, a)
    ref = oracle.add("D(a,b,i,j)+=L(b,a,j,i)", D, L, a)
    got = ctx.tensor_download(dD)
    assert np.max(np.abs(got - ref)) <= 4e-16 * np.max(np.abs(ref))
    ctx.add("D(a,b,i,j)=L(b,a,j,i)", dD, dL, 1.0)
    assert ctx.tensor_download(dD).tobytes() == oracle.permute("D(a,b,i,j)=L(b,a,j,i)", L, D.shape).tobytes()
    # same order: axpy
    E = rc(rng, 30, 9, 31, 4)
    dE = ctx.tensor_from_numpy(E)
    ctx.add("D(a,b,i,j)+=E(a,b,i,j)", dD, dE, -2.0)
    ref = oracle.add("D(a,b,i,j)+=E(a,b,i,j)", oracle.permute("D(a,b,i,j)=L(b,a,j,i)", L, D.shape), E, -2.0)
    assert np.array_equal(ctx.tensor_download(dD), ref)           # power-of-two alpha: exact
    ctx.scale(dD, 1.5j)
    assert np.max(np.abs(ctx.tensor_download(dD) - oracle.scale(ref, 1.5j))) <= 4e-16 * np.max(np.abs(ref))
    ctx.tensor_fill(dD, 3 - 4j)
    assert np.all(ctx.tensor_download(dD) == 3 - 4j)


def test_permsum_matches_oracle_bit_for_bit_with_unit_coefficients(ctx):
    """Same term order, separately rounded products and sums on both sides -> identical bits for c_t = +-1."""
    rng = np.random.default_rng(9)
    D, X = rc(rng, 11, 11, 5, 5), rc(rng, 11, 11, 5, 5)
    perms = [[0, 1, 2, 3], [1, 0, 2, 3], [0, 1, 3, 2], [1, 0, 3, 2]]
    coefs = [1, -1, -1, 1]
    dD, dX = ctx.tensor_from_numpy(D), ctx.tensor_from_numpy(X)
    ctx.permsum(dD, dX, perms, coefs, 1.0)
    assert ctx.tensor_download(dD).tobytes() == oracle.permsum(D, X, perms, coefs, 1.0).tobytes()
    # general complex coefficients and beta: tolerance of SURVEY 8(c) O3
    coefs = [0.5, -0.25j, 1 + 1j, -3]
    dD2 = ctx.tensor_from_numpy(D)
    ctx.permsum(dD2, dX, perms, coefs, 0.5 - 1j)
    ref = oracle.permsum(D, X, perms, coefs, 0.5 - 1j)
    assert np.max(np.abs(ctx.tensor_download(dD2) - ref)) <= 1e-14 * (np.abs(D).max() * 1.2 + 6 * np.abs(X).max())
    # beta = 0 does not read D
    dN = ctx.tensor_create(D.shape)
    ctx.tensor_fill(dN, complex(np.nan, np.nan))
    ctx.permsum(dN, dX, perms, [1, -1, -1, 1], 0.0)
    assert ctx.tensor_download(dN).tobytes() == oracle.permsum(np.zeros(D.shape), X, perms, [1, -1, -1, 1], 0.0).tobytes()


def test_antisymmetrize_9_term_rank6_and_36_equals_4x9(ctx):
    v, o = 7, 4
    W, T2 = synth.config_t3(o, v)
    R3 = synth.config_t3_r3(o, v)
    X, _ = cc.t3_term_unfactorised(W, T2)
    X = np.asfortranarray(X)
    dX, dR = ctx.tensor_from_numpy(X), ctx.tensor_from_numpy(R3)
    ctx.antisymmetrize("P(a/bc)P(k/ij):R(a,b,c,i,j,k)+=X(a,b,c,i,j,k)", dR, dX, 1.0)
    perms, coefs = cc.p9_terms()
    ref = oracle.permsum(R3, X, perms, coefs, 1.0)
    got = ctx.tensor_download(dR)
    assert np.max(np.abs(got - ref)) <= 1e-14 * (np.abs(R3).max() + 9 * np.abs(X).max())
    # 36-term full antisymmetriser of this X = 4 x the 9-term one (SURVEY 8(c) reading #3)
    p36, c36 = cc.full_antisymmetriser_terms()
    d36, d9 = ctx.tensor_create(X.shape), ctx.tensor_create(X.shape)
    ctx.permsum(d36, dX, p36, c36, 0.0)
    ctx.permsum(d9, dX, perms, coefs, 0.0)
    a36, a9 = ctx.tensor_download(d36), ctx.tensor_download(d9)
    assert np.max(np.abs(a36 - 4 * a9)) <= 1e-13 * np.abs(a36).max()


def test_device_generator_matches_host_generator(ctx):
    """csrc/synth.cu is the device twin of synth.py (bit-identical), so full-size inputs can be made on the GPU."""
    o, v = 5, 9
    V, T = synth.config_ladder(o, v, 3)
    dV, dT = ctx.tensor_create((v, v, v, v)), ctx.tensor_create((v, v, o, o))
    ctx.synth_normal(dV, synth.SEED0 + 3, 1, antisym=((0, 1), (2, 3)))
    ctx.synth_normal(dT, synth.SEED0 + 3, 2, antisym=((0, 1), (2, 3)))
    assert ctx.tensor_download(dV).tobytes() == V.tobytes()
    assert ctx.tensor_download(dT).tobytes() == T.tobytes()
    dI = ctx.tensor_create((7, 3, 5))
    ctx.synth_index_linear(dI)
    assert ctx.tensor_download(dI).tobytes() == synth.index_linear_tensor((7, 3, 5)).tobytes()


@pytest.mark.parametrize("shape,spec,nterms", [
    ((12, 12, 12, 6, 6, 6), "P(a/bc)P(k/ij):R(a,b,c,i,j,k)+=X(a,b,c,i,j,k)", 9),     # orbit kernel, 9 terms, 3 outer classes
    ((12, 12, 12, 6, 6, 6), "P(a/bc):R(a,b,c,i,j,k)+=X(a,b,c,i,j,k)", 3),            # orbit kernel, 3 terms inside a slab
    ((14, 14, 14, 3, 3, 3), "P(a/bc)P(k/ij):R(a,b,c,i,j,k)+=X(a,b,c,i,j,k)", 9),     # orbit kernel, ragged cubes (14 = 2*6 + 2)
    ((14, 14, 14, 3, 3, 3), "P(a/bc)P(k/ij):R(a,b,c,i,j,k)=X(a,b,c,i,j,k)", 9),      # ... beta = 0
    ((42, 42, 42), "P(a/bc):R(a,b,c)+=X(a,b,c)", 3),                                 # orbit kernel, no outer index
    ((18, 18, 18, 13), "P(c/ab):R(a,b,c,i)+=X(a,b,c,i)", 3),                         # orbit kernel, one outer index
    ((12, 12, 12, 6, 6, 6), "P(ab)P(k/ij):R(a,b,c,i,j,k)+=X(a,b,c,i,j,k)", 6),       # c stays put: cube kernel
    ((12, 12, 12, 6, 6, 6), "P(k/ij):R(a,b,c,i,j,k)=X(a,b,c,i,j,k)", 3),             # one unit-stride index, beta = 0
    ((64, 64, 8, 8), "P(ij)P(ab):R(a,b,i,j)+=X(a,b,i,j)", 4),                        # cube 8 x 4, all 32 lanes
    ((30, 30, 18, 18), "P(ab):R(a,b,i,j)+=X(a,b,i,j)", 2),                           # cube 6 x 5, two idle lanes
    ((66, 66, 8, 8), "P(ij)P(ab):R(a,b,i,j)+=X(a,b,i,j)", 4),                        # 66 = 2*3*11: cube 6 x 3 < 24 lanes -> generic
])
def test_permsum_cube_path_is_bit_identical_to_the_oracle(ctx, shape, spec, nterms):
    """Term sets that permute three leading indices among themselves take permsum_orbit_kernel (TMA-staged orbit cubes),
    other tensors of >= 2^18 elements permsum_cube_kernel (warp = micro-cube, running offsets); same term order and
    rounding as the oracle -> identical bits for unit coefficients, 1e-14 for a complex alpha."""
    rng = np.random.default_rng(len(shape) * 1000 + nterms)
    D, X = rc(rng, *shape), rc(rng, *shape)
    dX = ctx.tensor_from_numpy(X)
    # the spec's own expansion, replayed for the oracle through tcb_permsum's (perms, coefs) form
    import re
    ops = re.findall(r"P\(([^)]*)\)", spec.split(":")[0])
    labels = re.findall(r"\(([^()]*)\)", spec.split(":")[1])[0].split(",")
    terms = [(list(labels), 1.0)]
    for op in ops:
        pivot, others = (op.split("/")[0], list(op.split("/")[1])) if "/" in op else (op[0], [op[1]])
        nxt = []
        for lab, sg in terms:
            nxt.append((lab, sg))
            for o_ in others:
                nxt.append(([o_ if t == pivot else pivot if t == o_ else t for t in lab], -sg))
        terms = nxt
    assert len(terms) == nterms
    perms = [[labels.index(t) for t in lab] for lab, _ in terms]
    coefs = [sg for _, sg in terms]
    beta = 1.0 if "+=" in spec else 0.0
    dD = ctx.tensor_from_numpy(D)
    ctx.antisymmetrize(spec, dD, dX, 1.0)
    assert ctx.tensor_download(dD).tobytes() == oracle.permsum(D, X, perms, coefs, beta).tobytes()
    dD2 = ctx.tensor_from_numpy(D)
    alpha = 0.5 - 0.25j
    ctx.antisymmetrize(spec, dD2, dX, alpha)
    ref = oracle.permsum(D, X, perms, [alpha * c for c in coefs], beta)
    assert np.max(np.abs(ctx.tensor_download(dD2) - ref)) <= 1e-14 * (np.abs(D).max() + nterms * np.abs(X).max())
    # the gather kernels give the same bits (the option is read per call)
    import os
    os.environ["TCB_PERMSUM_NO_ORBIT"] = "1"
    try:
        dD3 = ctx.tensor_from_numpy(D)
        ctx.antisymmetrize(spec, dD3, dX, alpha)
        assert ctx.tensor_download(dD3).tobytes() == ctx.tensor_download(dD2).tobytes()
    finally:
        del os.environ["TCB_PERMSUM_NO_ORBIT"]
    # ... and so does the orbit kernel where it is not the default (fewer than 4 terms); a no-op for other term sets
    os.environ["TCB_PERMSUM_ORBIT"] = "1"
    try:
        dD4 = ctx.tensor_from_numpy(D)
        ctx.antisymmetrize(spec, dD4, dX, 1.0)
        assert ctx.tensor_download(dD4).tobytes() == ctx.tensor_download(dD).tobytes()
    finally:
        del os.environ["TCB_PERMSUM_ORBIT"]
    for t in (dD, dD2, dD3, dD4, dX):
        t.destroy()
