"""Pins for oracle.contract (order A, C nested loops) -- none of them re-types its formula in C or
re-calls it: brute-force python loops, an independent numpy implementation with the loops the other way
round (order B), numpy.einsum / matmul as library special cases, and exact algebraic invariants.
Passages: PAPER.md:87-91 (what a contraction is), 230 (scalar factor), 262 (binary), 266 (brute force)."""
import itertools

import numpy as np
import pytest

import oracle


def rc(rng, *s):
    return np.asfortranarray(rng.standard_normal(s) + 1j * rng.standard_normal(s))


def brute(dl, ll, rl, ext, D, L, R, alpha, acc):
    """Pure python: one dict of label -> value, loops over every label."""
    labels = list(dict.fromkeys(dl + ll + rl))
    con = [x for x in labels if x not in dl]
    out = np.array(D, dtype=np.complex128, copy=True)
    for d in itertools.product(*[range(ext[x]) for x in dl]):
        env = dict(zip(dl, d))
        s = 0j
        for c in itertools.product(*[range(ext[x]) for x in con]):
            env.update(zip(con, c))
            s += L[tuple(env[x] for x in ll)] * R[tuple(env[x] for x in rl)]
        out[d] = (out[d] if acc else 0) + alpha * s
    return out


CASES = [
    ("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", dict(a=3, b=2, c=3, d=2, i=2, j=3)),
    ("X(a,b,i,j)=T(a,c,i,k)*I2(k,b,c,j)", dict(a=3, b=2, c=2, i=2, j=3, k=2)),
    ("I3(l,i)=W(k,l,c,d)*T(d,c,i,k)", dict(l=2, i=3, k=2, c=3, d=2)),
    ("tt(a,b,i,j)=T1(a,i)*T1b(b,j)", dict(a=3, b=2, i=2, j=2)),                 # K = 1 (outer product)
    ("R1(a,i)+=T2(a,e,i,m)*Fme(m,e)", dict(a=3, i=2, e=2, m=3)),                # N = 1
    ("X(a,b,c,i,j,k)=W(b,c,d,k)*T(a,d,i,j)", dict(a=2, b=3, c=2, d=3, i=2, j=1, k=2)),   # rank 6, extent 1
    ("D(p1,h1)+=L(p1,p2)*R(p2,h1)", dict(p1=5, p2=7, h1=3)),                    # multi-character labels
    ("D(i,a)=L(k,a)*R(i,k)", dict(i=2, a=5, k=7)),
    ("D(a,b,c,d,e)+=L(e,x,c,a)*R(d,x,b)", dict(a=2, b=3, c=2, d=2, e=3, x=2)),
    ("D(a,b,c,d,e,f)+=L(f,d,b)*R(a,c,e)", dict(a=2, b=2, c=2, d=2, e=2, f=2)),
    ("D(a,b)+=L(u,v,w,x,a,y)*R(y,x,b,w,v,u)", dict(a=2, b=2, u=2, v=3, w=2, x=2, y=3)),
]


def split(expr):
    import re
    parts = re.findall(r"\(([^()]*)\)", expr)
    return [[x.strip() for x in p.split(",")] for p in parts], "+=" in expr


@pytest.mark.parametrize("expr,ext", CASES)
def test_brute_force_and_order_b_and_einsum(expr, ext):
    rng = np.random.default_rng(abs(hash(expr)) % 2**31)
    (dl, ll, rl), acc = split(expr)
    D0, L, R = (rc(rng, *[ext[x] for x in t]) for t in (dl, ll, rl))
    alpha = 0.75 - 0.5j
    got, sn = oracle.contract(expr, D0, L, R, alpha)
    ref = brute(dl, ll, rl, ext, D0, L, R, alpha, acc)
    assert np.all(np.abs(got - ref) <= 1e-14 * sn)
    gotb = oracle.contract_order_b(expr, D0, L, R, alpha)
    assert np.all(np.abs(got - gotb) <= 1e-13 * sn)                 # order A vs order B
    letters = {x: chr(97 + n) for n, x in enumerate(dict.fromkeys(dl + ll + rl))}
    sub = "".join(letters[x] for x in ll) + "," + "".join(letters[x] for x in rl) + "->" + "".join(letters[x] for x in dl)
    ein = (D0 if acc else 0) + alpha * np.einsum(sub, L, R)
    assert np.all(np.abs(got - ein) <= 1e-14 * sn)
    # double-accumulator variant (the timed baseline) agrees too
    gotd, _ = oracle.contract(expr, D0, L, R, alpha, long_double=False)
    assert np.all(np.abs(got - gotd) <= 1e-14 * sn)


def test_random_index_patterns():
    """Seeded random contractions, ranks 2..6 per tensor where possible, extents from {1,2,3,5}."""
    rng = np.random.default_rng(12345)
    n_done = 0
    while n_done < 40:
        nfl, nfr, nc = rng.integers(0, 4), rng.integers(0, 4), rng.integers(0, 4)
        if nfl + nc < 1 or nfr + nc < 1 or nfl + nfr < 1 or nfl + nfr > 6:
            continue
        labs = [f"x{n}" for n in range(nfl + nfr + nc)]
        fl, fr, cc = labs[:nfl], labs[nfl:nfl + nfr], labs[nfl + nfr:]
        ext = {x: int(rng.choice([1, 2, 3, 5])) for x in labs}
        dl = list(rng.permutation(fl + fr))
        ll = list(rng.permutation(fl + cc))
        rl = list(rng.permutation(fr + cc))
        op = "+=" if rng.integers(2) else "="
        expr = f"D({','.join(dl)}){op}L({','.join(ll)})*R({','.join(rl)})"
        D0, L, R = (rc(rng, *[ext[x] for x in t]) for t in (dl, ll, rl))
        got, sn = oracle.contract(expr, D0, L, R, 1.5 + 0.5j)
        ref = brute(dl, ll, rl, ext, D0, L, R, 1.5 + 0.5j, op == "+=")
        assert np.all(np.abs(got - ref) <= 1e-14 * sn), expr
        n_done += 1


def test_plain_gemm_special_case_is_matmul():
    rng = np.random.default_rng(5)
    A, B = rc(rng, 13, 7), rc(rng, 7, 11)
    got, sn = oracle.contract("C(m,n)=A(m,k)*B(k,n)", np.zeros((13, 11)), A, B, 1.0)
    assert np.all(np.abs(got - A @ B) <= 1e-14 * sn)
    # the ladder is a plain GEMM on the (a,b) x (c,d) x (i,j) matricisation (column-major reshape)
    V, T = rc(rng, 3, 4, 3, 4), rc(rng, 3, 4, 2, 5)
    got, sn = oracle.contract("R(a,b,i,j)=V(a,b,c,d)*T(c,d,i,j)", np.zeros((3, 4, 2, 5)), V, T, 1.0)
    mm = V.reshape(12, 12, order="F") @ T.reshape(12, 10, order="F")
    assert np.all(np.abs(got.reshape(12, 10, order="F") - mm) <= 1e-14 * sn.reshape(12, 10, order="F"))


def test_delta_tensor_returns_input_exactly():
    """V(a,b,c,d) = delta_ac delta_bd  =>  R = alpha*T bit for bit (sums of exact zeros)."""
    rng = np.random.default_rng(6)
    v, o = 4, 3
    V = np.zeros((v, v, v, v), dtype=np.complex128)
    for a in range(v):
        for b in range(v):
            V[a, b, a, b] = 1.0
    T = rc(rng, v, v, o, o)
    got, _ = oracle.contract("R(a,b,i,j)=V(a,b,c,d)*T(c,d,i,j)", np.zeros((v, v, o, o)), V, T, 2.0)
    assert np.array_equal(got, 2.0 * T)


def test_power_of_two_scaling_is_exact_and_linear():
    rng = np.random.default_rng(7)
    V, T = rc(rng, 3, 3, 3, 3), rc(rng, 3, 3, 2, 2)
    z = np.zeros((3, 3, 2, 2))
    e = "R(a,b,i,j)=V(a,b,c,d)*T(c,d,i,j)"
    r1, _ = oracle.contract(e, z, V, T, 0.5, long_double=False)
    r2, _ = oracle.contract(e, z, V, T, 1.0, long_double=False)
    assert np.array_equal(2.0 * r1, r2)
    r3, _ = oracle.contract(e, z, 4.0 * V, T, 0.25, long_double=False)
    assert np.array_equal(r3, r2)


def test_antisymmetry_is_carried_through():
    rng = np.random.default_rng(8)
    v, o = 4, 3
    V = rc(rng, v, v, v, v); V = V - V.transpose(1, 0, 2, 3)
    T = rc(rng, v, v, o, o); T = T - T.transpose(0, 1, 3, 2)
    R, sn = oracle.contract("R(a,b,i,j)=V(a,b,c,d)*T(c,d,i,j)", np.zeros((v, v, o, o)), V, T, 0.5)
    assert np.all(np.abs(R + R.transpose(1, 0, 2, 3)) <= 1e-15 * sn)
    assert np.all(np.abs(R + R.transpose(0, 1, 3, 2)) <= 1e-15 * sn)
    assert np.all(R[np.arange(v), np.arange(v)] == 0)      # a = b: snorm-style exact zeros? (V row is exactly 0)


def test_snorm_closed_form_and_assign_vs_accumulate():
    L = np.full((2, 5), 1 + 1j); R = np.full((5, 3), 2 - 0j); D0 = np.full((2, 3), 3 + 4j)
    got, sn = oracle.contract("D(m,n)+=L(m,k)*R(k,n)", D0, L, R, 2j)
    assert np.allclose(sn, 2 * 5 * np.sqrt(2) * 2 + 5)
    assert np.allclose(got, D0 + 2j * 5 * (1 + 1j) * 2)
    got2, sn2 = oracle.contract("D(m,n)=L(m,k)*R(k,n)", D0, L, R, 2j)
    assert np.allclose(got2, 2j * 5 * (1 + 1j) * 2) and np.allclose(sn2, 2 * 5 * np.sqrt(2) * 2)


@pytest.mark.parametrize("expr", [
    "D(a,b)+=L(a,k)*R(k,c)",        # c only in R, b only in D
    "D(a,b)+=L(a,b)*R(a,b)",        # Hadamard / batch
    "D(a,a)+=L(a,k)*R(k,a)",        # repeated label
    "D(a,b)+=L(a,k,k)*R(b)",        # trace
    "D(a,b)+L(a,k)*R(k,b)",         # no operator
    "D(a,b)+=L(a,k)*R(k,b",         # unbalanced
])
def test_invalid_expressions_are_rejected(expr):
    z = np.zeros((2, 2)); z3 = np.zeros((2, 2, 2))
    with pytest.raises(oracle.OracleError):
        oracle.contract(expr, z, z3 if "k,k" in expr else z, z if "R(b)" not in expr else np.zeros(2), 1.0)


def test_extent_mismatch_rejected():
    with pytest.raises(oracle.OracleError):
        oracle.contract("D(a,b)+=L(a,k)*R(k,b)", np.zeros((2, 2)), np.zeros((2, 3)), np.zeros((4, 2)), 1.0)
