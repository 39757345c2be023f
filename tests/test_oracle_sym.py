"""Pins of oracle/sym.py (index-permutation-symmetric packed storage; reading 16).  None of them
calls the function under test to make its own expectation: enumeration orders are printed literally, packed positions are
re-derived by running counters in nested loops, signs by determinants of permutation matrices, and the packed contraction is
tied to the DENSE oracle contraction (itself pinned in tests/test_oracle_contract.py)."""
import itertools

import numpy as np
import pytest

import oracle
from oracle import sym


def antisym4(rng, n, m):
    """T(a,b,i,j) antisymmetric in (a,b) and (i,j), exactly"""
    g = rng.standard_normal((n, n, m, m)) + 1j * rng.standard_normal((n, n, m, m))
    t = g - g.transpose(1, 0, 2, 3)
    return np.asfortranarray(t - t.transpose(0, 1, 3, 2))


def test_enumeration_orders_are_the_documented_ones():
    assert sym.tuples(4, 2) == [(0, 1), (0, 2), (1, 2), (0, 3), (1, 3), (2, 3)]
    assert sym.tuples(5, 3) == [(0, 1, 2), (0, 1, 3), (0, 2, 3), (1, 2, 3), (0, 1, 4), (0, 2, 4), (1, 2, 4), (0, 3, 4),
                                (1, 3, 4), (2, 3, 4)]
    for n in range(2, 9):
        assert sym.packed_extent(n, 2) == n * (n - 1) // 2 and sym.packed_extent(n, 3) == n * (n - 1) * (n - 2) // 6
        # closed forms of the position, checked by a running counter in plain nested loops
        p = 0
        for b in range(n):
            for a in range(b):
                assert sym.tuples(n, 2)[p] == (a, b) and p == b * (b - 1) // 2 + a
                p += 1
        p = 0
        for c in range(n):
            for b in range(c):
                for a in range(b):
                    assert sym.tuples(n, 3)[p] == (a, b, c) and p == c * (c - 1) * (c - 2) // 6 + b * (b - 1) // 2 + a
                    p += 1


def test_pack_picks_the_stored_elements_by_running_counter():
    rng = np.random.default_rng(0)
    n, m = 5, 4
    T = antisym4(rng, n, m)
    P = sym.pack("Tp(a<b,i<j)=T(a,b,i,j)", T)
    assert P.shape == (10, 6)
    q = 0
    for j in range(m):
        for i in range(j):
            p = 0
            for b in range(n):
                for a in range(b):
                    assert P[p, q] == T[a, b, i, j]
                    p += 1
            q += 1
    # groups may sit anywhere in the dense tensor and in any order in the packed one
    P2 = sym.pack("Tp(i<j,a<b)=T(a,b,i,j)", T)
    assert np.array_equal(P2, P.T)
    W = np.asfortranarray(T.transpose(0, 2, 1, 3))               # W(a,i,b,j)
    assert np.array_equal(sym.pack("Wp(a<b,i<j)=W(a,i,b,j)", W), P)
    # a group beside plain indices
    assert np.array_equal(sym.pack("Tq(a<b,i,j)=T(a,b,i,j)", T)[:, 1, 3], P[:, sym.tuples(m, 2).index((1, 3))])


def test_round_trips_are_bit_exact():
    rng = np.random.default_rng(1)
    n, m = 6, 5
    T = antisym4(rng, n, m)
    P = sym.pack("Tp(a<b,i<j)=T(a,b,i,j)", T)
    U = sym.unpack("T(a,b,i,j)=Tp(a<b,i<j)", P, extents=dict(a=n, b=n, i=m, j=m))
    assert U.tobytes() == T.tobytes() or np.array_equal(U, T)     # -0.0 vs 0.0 on the diagonals compare equal
    assert np.array_equal(U, T)
    assert np.array_equal(sym.pack("Tp(a<b,i<j)=T(a,b,i,j)", U), P)
    # any packed tensor unpacks to an exactly antisymmetric one
    Q = np.asfortranarray(rng.standard_normal((15, 10)) + 1j * rng.standard_normal((15, 10)))
    D = sym.unpack("T(a,b,i,j)=Tp(a<b,i<j)", Q, extents=dict(a=6, b=6, i=5, j=5))
    assert np.array_equal(D, -D.transpose(1, 0, 2, 3)) and np.array_equal(D, -D.transpose(0, 1, 3, 2))
    assert not np.any(D[np.arange(6), np.arange(6)]) and not np.any(D[:, :, np.arange(5), np.arange(5)])


def test_unpack_signs_are_permutation_determinants():
    """triples: D[a,b,c] = det(P) * Lp[sorted], the determinant of the permutation matrix that sorts (a,b,c)"""
    rng = np.random.default_rng(2)
    n = 5
    Lp = rng.standard_normal(10) + 1j * rng.standard_normal(10)
    D = sym.unpack("D(a,b,c)=Lp(a<b<c)", Lp, extents=dict(a=n, b=n, c=n))
    tl = sym.tuples(n, 3)
    for idx in itertools.product(range(n), repeat=3):
        if len(set(idx)) < 3:
            assert D[idx] == 0
            continue
        order = np.argsort(idx)
        M = np.zeros((3, 3))
        M[np.arange(3), order] = 1.0
        assert D[idx] == round(np.linalg.det(M)) * Lp[tl.index(tuple(sorted(idx)))]
    # accumulate form with a complex alpha
    D0 = rng.standard_normal((n, n, n)) + 0j
    D1 = sym.unpack("D(a,b,c)+=Lp(a<b<c)", Lp, D=D0, alpha=0.5 - 2j)
    assert np.allclose(D1, D0 + (0.5 - 2j) * D, rtol=0, atol=1e-15)


def test_packed_ladder_equals_the_dense_oracle_contraction_without_the_factor_one_half():
    """R(a,b,i,j) += 1/2 sum_cd V(a,b,c,d) T(c,d,i,j) on antisymmetric operands is, on packed operands,
    Rp(ab,ij) += sum_{c<d} Vp(ab,cd) Tp(cd,ij): 1/8 of the multiply-adds and no factor 1/2 (the c<d sum visits each unordered
    pair once).  Both sides through the pinned dense oracle contraction."""
    rng = np.random.default_rng(3)
    v, o = 6, 4
    V, T = antisym4(rng, v, v), antisym4(rng, v, o)
    R0 = antisym4(rng, v, o)
    dense, sn = oracle.contract("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", R0, V, T, 0.5)
    Vp, Tp = sym.pack("Vp(a<b,c<d)=V(a,b,c,d)", V), sym.pack("Tp(c<d,i<j)=T(c,d,i,j)", T)
    Rp, _ = oracle.contract("Rp(x,y)=Vp(x,z)*Tp(z,y)", np.zeros((15, 6)), Vp, Tp, 1.0)
    packed = sym.unpack("R(a,b,i,j)+=Rp(a<b,i<j)", Rp, D=R0, alpha=1.0)
    assert np.max(np.abs(packed - dense) / np.where(sn > 0, sn, 1.0)) <= 1e-14
    assert np.array_equal(packed[sn == 0], dense[sn == 0])


def test_bad_specs_are_rejected():
    T = np.zeros((3, 3, 2, 2))
    with pytest.raises(ValueError):
        sym.pack("Tp(a,b,i,j)=T(a,b,i,j)", T)                    # no group at all
    with pytest.raises(ValueError):
        sym.pack("Tp(a<b,i<j)+=T(a,b,i,j)", T)                   # pack does not accumulate
    with pytest.raises(AssertionError):
        sym.pack("Tp(a<i,b,j)=T(a,b,i,j)", T)                    # unequal extents inside a group
