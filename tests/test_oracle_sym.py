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


# ---- packed views of packed tensors, and the permutation operators on packed storage ------------------------------------------
def _exactly_antisymmetric_t3(rng, v, o):
    """(packed, dense) of a T(a,b,c,i,j,k) that is antisymmetric bit for bit: the dense one is written from the packed one
    with the sign of the permutation determinant (no function of oracle/sym.py involved)"""
    tv = [t for t in itertools.combinations(range(v), 3)]
    tv.sort(key=lambda t: t[::-1])
    to = [t for t in itertools.combinations(range(o), 3)]
    to.sort(key=lambda t: t[::-1])
    P = rng.standard_normal((len(tv), len(to))) + 1j * rng.standard_normal((len(tv), len(to)))
    T = np.zeros((v, v, v, o, o, o), dtype=np.complex128, order="F")
    for p, abc in enumerate(tv):
        for q, ijk in enumerate(to):
            for pv in itertools.permutations(range(3)):
                sv = round(np.linalg.det(np.eye(3)[list(pv)]))
                for po in itertools.permutations(range(3)):
                    so = round(np.linalg.det(np.eye(3)[list(po)]))
                    T[abc[pv[0]], abc[pv[1]], abc[pv[2]], ijk[po[0]], ijk[po[1]], ijk[po[2]]] = sv * so * P[p, q]
    return np.asfortranarray(P), T


VIEWS = [("Tq(d<e,c,i<j<k)=T(d<e<c,i<j<k)", "Tq(d<e,c,i<j<k)=T(d,e,c,i,j,k)"),
         ("To(a<b<c,l<m,k)=T(a<b<c,l<m<k)", "To(a<b<c,l<m,k)=T(a,b,c,l,m,k)"),
         ("Tr(b<c,j<k,e,m)=T(b<c<e,j<k<m)", "Tr(b<c,j<k,e,m)=T(b,c,e,j,k,m)"),
         ("Tr(j<k,e,b<c,m)=T(e<b<c,m<j<k)", "Tr(j<k,e,b<c,m)=T(e,b,c,m,j,k)"),     # the single label first in L's group
         ("Ts(a<c,b,i<j<k)=T(a<b<c,i<j<k)", "Ts(a<c,b,i<j<k)=T(a,b,c,i,j,k)")]     # the outer two labels of a triple


@pytest.mark.parametrize("view,from_dense", VIEWS)
def test_a_packed_view_is_the_pack_of_the_dense_tensor(view, from_dense):
    """groups on both sides of `unpack`: the view of the packed tensor equals `pack` (pinned above by running counters)
    applied to the dense antisymmetric tensor -- bit for bit, signs included"""
    rng = np.random.default_rng(len(view))
    P, T = _exactly_antisymmetric_t3(rng, 5, 4)
    got = sym.unpack(view, P)
    ref = sym.pack(from_dense, T)
    assert got.shape == ref.shape and np.array_equal(got, ref)
    base = rng.standard_normal(ref.shape) + 0j
    acc = sym.unpack(view.replace("=", "+=", 1), P, D=base, alpha=2.0)
    assert np.array_equal(acc, base + 2.0 * ref)
    assert np.count_nonzero(got) > got.size // 4         # zeros only where a label of the view repeats inside a group of L


def test_a_view_that_repeats_a_value_inside_a_group_of_l_reads_zero():
    """D(a<b, c) = L(a, b<c) at c == b: L's group (b,c) has two equal labels -> 0; at c < b the sign flips"""
    rng = np.random.default_rng(3)
    n = 5
    L = rng.standard_normal((n, sym.packed_extent(n, 2))) + 0j
    D = sym.unpack("D(a<b,c)=L(a,b<c)", L)
    pairs = sym.tuples(n, 2)
    pos = {t: p for p, t in enumerate(pairs)}
    for p, (a, b) in enumerate(pairs):
        for c in range(n):
            want = 0.0 if b == c else (L[a, pos[(b, c)]] if b < c else -L[a, pos[(c, b)]])
            assert D[p, c] == want


def _dense_operator(spec_ops, labels, X):
    """P(x/yz)-style operators on a DENSE tensor through oracle.permsum (pinned in tests/test_oracle_permute.py); the
    expansion of the operator string into signed permutations is written out here by hand-rolled transpositions"""
    terms = [(list(labels), 1)]
    for op in spec_ops:                                  # e.g. ("a", "bc"): 1 - (a b) - (a c)
        x, rest = op
        nxt = []
        for lab, sg in terms:
            nxt.append((lab, sg))
            for y in rest:
                sw = [y if q == x else x if q == y else q for q in lab]
                nxt.append((sw, -sg))
        terms = nxt
    perms = [[list(labels).index(q) for q in lab] for lab, _ in terms]
    return oracle.permsum(np.zeros_like(X), X, perms, [float(s) for _, s in terms], 0.0)


MERGES = [("R(a<b<c,i<j<k)=X(a,i,b<c,j<k)", "X(a,b,c,i,j,k)=P(a,i,b<c,j<k)", [("a", "bc"), ("i", "jk")], 9),
          ("R(a<b<c,i<j<k)=X(b<c,a,i<j<k)", "X(a,b,c,i,j,k)=P(b<c,a,i<j<k)", [("a", "bc")], 3),
          ("R(a<b<c,i<j<k)=X(a<b<c,j<k,i)", "X(a,b,c,i,j,k)=P(a<b<c,j<k,i)", [("i", "jk")], 3),
          ("R(a<b<c,i<j<k)=X(a<b,c,i<j,k)", "X(a,b,c,i,j,k)=P(a<b,c,i<j,k)", [("c", "ab"), ("k", "ij")], 9),
          ("R(a<b,i<j)=X(a,i,b,j)", "X(a,b,i,j)=P(a,i,b,j)", [("a", "b"), ("i", "j")], 4)]


@pytest.mark.parametrize("spec,expand,ops,nterms", MERGES)
def test_antisym_pack_is_the_permutation_operator_on_the_dense_expansion(spec, expand, ops, nterms):
    """antisym_pack == pack( P(..)P(..) [ dense expansion of L ] ): the operator applied by oracle.permsum to the tensor
    `unpack` (pinned above) writes out; and the number of shuffles is the paper's term count for the operator"""
    rng = np.random.default_rng(nterms + len(spec))
    v, o = 5, 4
    labels = expand[expand.index("(") + 1:expand.index(")")].split(",")
    ext = {x: (v if x in "abc" else o) for x in labels}
    groups = sym.parse_both(spec)[1]
    shape = [sym.packed_extent(ext[g[0]], len(g)) for g in groups]
    L = rng.standard_normal(shape) + 1j * rng.standard_normal(shape)
    if "<" in expand:
        Xd = sym.unpack(expand, L, extents=ext)
    else:                                                 # L is dense already: only its index order differs
        Xd = np.asfortranarray(np.transpose(L, [[g[0] for g in groups].index(x) for x in labels]))
    Rd = _dense_operator(ops, labels, Xd)
    dgroups = sym.parse_both(spec)[0]
    ref = sym.pack("P(" + ",".join("<".join(g) for g in dgroups) + ")=R(" + ",".join(labels) + ")", Rd)
    got = sym.antisym_pack(spec, L)
    assert got.shape == ref.shape and np.abs(got - ref).max() <= 1e-14 * np.abs(ref).max()
    count = 1
    for g in dgroups:
        count *= len(sym.shuffles(g, [set(b) for b in groups]))
    assert count == nterms
    base = rng.standard_normal(ref.shape) + 0j
    acc = sym.antisym_pack(spec.replace("=", "+=", 1), L, D=base, alpha=0.5 - 1.5j)
    assert np.abs(acc - (base + (0.5 - 1.5j) * ref)).max() <= 1e-14 * np.abs(ref).max()


def test_antisym_pack_of_a_dense_tensor_is_the_36_term_antisymmetriser_and_of_a_packed_one_the_identity():
    from oracle import cc
    rng = np.random.default_rng(12)
    v, o = 4, 4
    X = rng.standard_normal((v, v, v, o, o, o)) + 1j * rng.standard_normal((v, v, v, o, o, o))
    got = sym.antisym_pack("R(a<b<c,i<j<k)=X(a,b,c,i,j,k)", X)
    ref = sym.pack("P(a<b<c,i<j<k)=A(a,b,c,i,j,k)", cc.antisymmetrise_abc_ijk(X))
    assert np.abs(got - ref).max() <= 1e-14 * np.abs(ref).max()
    assert len(sym.shuffles(["a", "b", "c"], [{"a"}, {"b"}, {"c"}])) == 6
    same = sym.antisym_pack("R(a<b<c,i<j<k)=P(a<b<c,i<j<k)", got)        # one shuffle per group: a copy
    assert np.array_equal(same, got)
    with pytest.raises(ValueError):
        sym.antisym_pack("R(a<b,c)=X(a,b<c)", np.zeros((4, 6)))           # L's group straddles two groups of D
    with pytest.raises(ValueError):
        sym.unpack("D(a<b,c)=L(a,b<d)", np.zeros((4, 6)))                 # labels differ
