"""oracle.sym -- index-permutation-symmetric (antisymmetric) packed storage, CPU oracle.  TEST INFRASTRUCTURE ONLY.

What it follows: the paper names "index-permutation symmetry" of tensors as the feature its production code does not exploit
yet (PAPER.md:202 feature list, 264 "work in progress", 440 and 452 outlook: the main stated limitation).  The paper gives
no storage scheme, so this is a reading (reading 16), the plainest one:

  * a GROUP  a<b  (or a<b<c) of labels of equal extent n, in which the tensor is antisymmetric, is stored as ONE packed index
    that runs over the strictly increasing tuples only: n(n-1)/2 pairs, n(n-1)(n-2)/6 triples;
  * tuples are enumerated with the FIRST label fastest (the library's column-major convention):
        pairs   (0,1) (0,2) (1,2) (0,3) (1,3) (2,3) ...          p = b(b-1)/2 + a
        triples (0,1,2) (0,1,3) (0,2,3) (1,2,3) (0,1,4) ...      p = c(c-1)(c-2)/6 + b(b-1)/2 + a
  * pack   : Dp[.., p(a<b), ..] = L[.., a, .., b, ..]     (a copy of the stored elements: bit-exact)
  * unpack : D[.., a, .., b, ..] (+)= alpha * sign * Lp[.., p(sorted a,b), ..];  sign = parity of the sorting permutation,
             0 when two labels of a group coincide.  With alpha = 1 and '=' an exactly antisymmetric tensor is reproduced
             bit for bit (negation is exact).

Everything here is explicit Python loops over index tuples (tiny sizes) or numpy `take` on index lists built by those
loops; no closed-form index arithmetic is shared with the CUDA side.
"""
import itertools
import re

import numpy as np


def tuples(n, k):
    """strictly increasing k-tuples of range(n), FIRST element fastest: built by explicit enumeration + sort key"""
    tl = [t for t in itertools.combinations(range(n), k)]
    tl.sort(key=lambda t: tuple(reversed(t)))          # last element slowest ... first element fastest
    return tl


def packed_extent(n, k):
    return len(tuples(n, k))


def _parse_side(text):
    m = re.fullmatch(r"\s*\w+\s*\(([^()]*)\)\s*", text)
    if not m:
        raise ValueError(f"cannot parse {text!r}")
    items = [x.strip() for x in m.group(1).split(",")] if m.group(1).strip() else []
    return [[y.strip() for y in it.split("<")] for it in items]


def parse(spec):
    """'Vp(a<b,c<d)=V(a,b,c,d)' -> (packed items, dense labels, accumulate, packed_on_left)"""
    m = re.fullmatch(r"(.*?)(\+=|=)(.*)", spec)
    if not m:
        raise ValueError(f"cannot parse {spec!r}")
    lhs, rhs = _parse_side(m.group(1)), _parse_side(m.group(3))
    acc = m.group(2) == "+="
    lhs_packed = any(len(it) > 1 for it in lhs)
    rhs_packed = any(len(it) > 1 for it in rhs)
    if lhs_packed == rhs_packed:
        raise ValueError("exactly one side must carry a<b groups")
    return lhs, rhs, acc, lhs_packed


def _sort_sign(vals):
    """(sorted tuple, sign of the sorting permutation), sign 0 when two values coincide -- by bubble sort, counting swaps"""
    v = list(vals)
    if len(set(v)) < len(v):
        return tuple(sorted(v)), 0
    sign = 1
    for i in range(len(v)):
        for j in range(len(v) - 1 - i):
            if v[j] > v[j + 1]:
                v[j], v[j + 1] = v[j + 1], v[j]
                sign = -sign
    return tuple(v), sign


def pack(spec, L):
    """spec 'Vp(a<b,c<d)=V(a,b,c,d)': returns the packed tensor (Fortran order)."""
    items, dense, acc, lhs_packed = parse(spec)
    if not lhs_packed or acc:
        raise ValueError("pack: 'P(a<b,..)=D(a,b,..)'")
    labs = [d[0] for d in dense]
    L = np.asarray(L, dtype=np.complex128)
    ext = dict(zip(labs, L.shape))
    lists = []
    for it in items:
        n = ext[it[0]]
        assert all(ext[x] == n for x in it), "labels of a group need equal extents"
        lists.append(tuples(n, len(it)))
    out = np.zeros([len(t) for t in lists], dtype=np.complex128, order="F")
    for pidx in itertools.product(*[range(len(t)) for t in lists]):
        val = {}
        for it, t, p in zip(items, lists, pidx):
            for lab, x in zip(it, t[p]):
                val[lab] = x
        out[pidx] = L[tuple(val[x] for x in labs)]
    return out


def unpack(spec, Lp, D=None, alpha=1.0, extents=None):
    """spec 'R(a,b,i,j)+=Rp(a<b,i<j)': returns D (+)= alpha * sign * Lp[packed position]; D=None starts from zeros of
    `extents` (dict label -> extent, or taken from the packed extents when unambiguous)."""
    dense, items, acc, lhs_packed = parse(spec)
    if lhs_packed:
        raise ValueError("unpack: 'D(a,b,..)(+)=P(a<b,..)'")
    labs = [d[0] for d in dense]
    Lp = np.asarray(Lp, dtype=np.complex128)
    if D is not None:
        D = np.array(D, dtype=np.complex128, order="F")
        ext = dict(zip(labs, D.shape))
    else:
        ext = dict(extents)
        D = np.zeros([ext[x] for x in labs], dtype=np.complex128, order="F")
    where = []
    for it, pe in zip(items, Lp.shape):
        tl = tuples(ext[it[0]], len(it))
        assert len(tl) == pe, "packed extent does not match the dense extents"
        where.append({t: p for p, t in enumerate(tl)})
    a = complex(alpha)
    for idx in itertools.product(*[range(ext[x]) for x in labs]):
        val = dict(zip(labs, idx))
        sign, pidx = 1, []
        for it, w in zip(items, where):
            srt, sg = _sort_sign([val[x] for x in it])
            sign *= sg
            pidx.append(w.get(srt, 0))
        term = 0.0 if sign == 0 else a * Lp[tuple(pidx)] * sign
        D[idx] = (D[idx] if acc else 0.0) + term
    return D
