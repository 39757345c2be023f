"""Helpers shared by the -m gpu parity tests (the CUDA path through the C ABI vs the CPU oracle)."""
import numpy as np

TOL = 1e-11     # BASELINE.json north_star: max |gpu - oracle| / snorm, snorm = |alpha| sum|L||R| + |D_in|


def rc(rng, *shape):
    """complex N(0,1)+iN(0,1), Fortran order"""
    return np.asfortranarray(rng.standard_normal(shape) + 1j * rng.standard_normal(shape))


def parity_error(got, ref, snorm):
    """max normalised error; where snorm == 0 the values must agree exactly"""
    zero = snorm == 0
    assert np.array_equal(got[zero], ref[zero]), "elements with zero normaliser must be exact"
    if zero.all():
        return 0.0
    return float(np.max(np.abs(got - ref)[~zero] / snorm[~zero]))


def split_expr(expr):
    """'D(a,b)+=L(a,c)*R(c,b)' -> (['a','b'], ['a','c'], ['c','b'])"""
    import re
    groups = re.findall(r"\(([^()]*)\)", expr)
    return [[s.strip() for s in g.split(",")] if g.strip() else [] for g in groups]
