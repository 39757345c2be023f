"""Pins for oracle.permute / add / permsum / scale: closed forms and group identities
(PAPER.md:87 transposition, 194/230/284 permutation operators)."""
import itertools

import numpy as np
import pytest

import oracle
from oracle import cc

LAB = "abcdef"


def lin_tensor(shape):
    n = int(np.prod(shape))
    x = np.arange(n, dtype=np.float64) + 1j * (-np.arange(n, dtype=np.float64) - 0.5)
    return x.reshape(shape, order="F")


def pexpr(perm):
    r = len(perm)
    return f"D({','.join(LAB[p] for p in perm)})=L({','.join(LAB[:r])})"


@pytest.mark.parametrize("shape", [(3, 5), (2, 3, 4), (7, 2, 3, 5), (2, 3, 1, 4, 2), (2, 3, 2, 3, 2, 3)])
def test_closed_form_linear_index(shape):
    """L[idx] = linear index  =>  D[j] must equal the closed-form source offset, no second implementation."""
    r = len(shape)
    L = lin_tensor(shape)
    sL = np.cumprod((1,) + shape[:-1])
    perms = list(itertools.permutations(range(r)))
    if len(perms) > 24:
        rng = np.random.default_rng(1)
        perms = [perms[i] for i in rng.choice(len(perms), 24, replace=False)] + [tuple(reversed(range(r)))]
    for perm in perms:
        shD = tuple(shape[p] for p in perm)
        D = oracle.permute(pexpr(perm), L, shD)
        for j in itertools.product(*[range(e) for e in shD]):
            src = sum(j[k] * sL[perm[k]] for k in range(r))
            assert D[j].real == src and D[j].imag == -src - 0.5


def test_inverse_and_composition():
    rng = np.random.default_rng(2)
    shape = (3, 4, 2, 5)
    L = np.asfortranarray(rng.standard_normal(shape) + 1j * rng.standard_normal(shape))
    for p in itertools.permutations(range(4)):
        shD = tuple(shape[k] for k in p)
        D = oracle.permute(pexpr(p), L, shD)
        assert np.array_equal(D, L.transpose(p))                        # numpy transpose as library routine
        inv = tuple(np.argsort(p))
        back = oracle.permute(pexpr(inv), D, shape)
        assert back.tobytes() == L.tobytes()
        q = tuple(rng.permutation(4))
        DQ = oracle.permute(pexpr(q), D, tuple(shD[k] for k in q))
        comp = tuple(p[k] for k in q)
        assert np.array_equal(DQ, oracle.permute(pexpr(comp), L, tuple(shape[k] for k in comp)))


def test_bit_exact_special_values():
    """NaN payloads, -0.0, infinities and denormals are moved as bytes."""
    bits = np.array([0x7FF8000000000123, 0x8000000000000000, 0xFFF0000000000000, 0x0000000000000001,
                     0x7FF0000000000001, 0x3FF0000000000000] * 2, dtype=np.uint64)
    flat = bits.view(np.complex128)                      # 6 complex numbers
    L = flat.reshape((2, 3), order="F")
    D = oracle.permute("D(j,i)=L(i,j)", L, (3, 2))
    for i in range(2):
        for j in range(3):
            assert D[j, i].tobytes() == L[i, j].tobytes()


def test_add_and_scale():
    rng = np.random.default_rng(3)
    D0 = np.asfortranarray(rng.standard_normal((3, 4)) + 1j * rng.standard_normal((3, 4)))
    L = np.asfortranarray(rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3)))
    a = 0.5 - 2j
    assert np.allclose(oracle.add("D(i,j)+=L(j,i)", D0, L, a), D0 + a * L.T, rtol=1e-15, atol=0)
    assert np.array_equal(oracle.add("D(i,j)+=L(i,j)", D0, D0, 1.0), 2 * D0)
    assert np.allclose(oracle.scale(D0, a), a * D0, rtol=1e-15)
    assert np.array_equal(oracle.scale(D0, 2.0), 2 * D0)


def test_permsum_identities():
    rng = np.random.default_rng(4)
    v, o = 3, 3
    X = np.asfortranarray(rng.standard_normal((v, v, o, o)) + 1j * rng.standard_normal((v, v, o, o)))
    z = np.zeros_like(X)
    # explicit numpy form
    for (perms, coefs), ref in [(cc.P_AB, X - X.transpose(1, 0, 2, 3)),
                                (cc.P_IJ, X - X.transpose(0, 1, 3, 2)),
                                (cc.P_IJ_AB, X - X.transpose(1, 0, 2, 3) - X.transpose(0, 1, 3, 2) + X.transpose(1, 0, 3, 2))]:
        got = oracle.permsum(z, X, perms, coefs, 0.0)
        assert np.allclose(got, ref, rtol=1e-15, atol=1e-15)
    # P(ab) of a symmetric tensor is exactly zero
    S = X + X.transpose(1, 0, 2, 3)
    assert not np.any(oracle.permsum(z, S, *cc.P_AB, 0.0))
    # beta and accumulate
    D0 = np.asfortranarray(rng.standard_normal(X.shape) + 0j)
    got = oracle.permsum(D0, X, *cc.P_AB, 2.0)
    assert np.allclose(got, 2 * D0 + X - X.transpose(1, 0, 2, 3), rtol=1e-14)
    # beta = 0 does not read D (NaN does not propagate)
    nan = np.full(X.shape, np.nan + 0j)
    assert np.all(np.isfinite(oracle.permsum(nan, X, *cc.P_AB, 0.0)))


def test_three_cycle_convention():
    """D(a,b,c) = X(b,c,a): position 0 of X takes D index 1, etc. (non-involutive, fixes the convention)."""
    X = lin_tensor((2, 3, 4))                        # X(p,q,r)
    D = oracle.permsum(np.zeros((4, 2, 3)), X, [[1, 2, 0]], [1.0], 0.0)
    for a, b, c in itertools.product(range(4), range(2), range(3)):
        assert D[a, b, c] == X[b, c, a]


def test_full_antisymmetriser_idempotent_and_36_equals_4x9():
    rng = np.random.default_rng(5)
    v = o = 3
    X = np.asfortranarray(rng.standard_normal((v, v, v, o, o, o)) + 1j * rng.standard_normal((v, v, v, o, o, o)))
    p36, c36 = cc.full_antisymmetriser_terms()
    assert len(c36) == 36
    z = np.zeros_like(X)
    AX = oracle.permsum(z, X, p36, c36, 0.0)
    AAX = oracle.permsum(z, AX, p36, c36, 0.0)
    assert np.abs(AAX - 36 * AX).max() <= 1e-13 * np.abs(AAX).max()           # A(AX) = 3!3! AX
    # for X already antisymmetric in (b,c) and (i,j) -- as W(b,c,d,k) T(a,d,i,j) is -- 36-term = 4 x 9-term
    Y = X - X.transpose(0, 2, 1, 3, 4, 5)
    Y = Y - Y.transpose(0, 1, 2, 4, 3, 5)
    p9, c9 = cc.p9_terms()
    assert len(c9) == 9
    A36, A9 = oracle.permsum(z, Y, p36, c36, 0.0), oracle.permsum(z, Y, p9, c9, 0.0)
    assert np.abs(A36 - 4 * A9).max() <= 1e-13 * np.abs(A36).max()
