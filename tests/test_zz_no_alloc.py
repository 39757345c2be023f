"""-m gpu: tcb_dot_noalloc, the one entry point that allocates nothing (its scratch is a fixed device array inside the library,
csrc/dot_noalloc.cu), against the existing path tcb_dot on the same device tensors -- within the tolerance the tcb_dot test
uses (tests/test_gpu_cc.py: 1e-13 * |alpha| * sum |X||Y|) -- on calls in a row that share the array.

Collected LAST on purpose (the file name): the suite runs with pytest -x, a failure here must not hide another test.  Uses a
context of its own, so it passes alone in a fresh process and after the other tests alike."""
import numpy as np
import pytest

import paper_2409_06759_b200 as pkg
from paper_2409_06759_b200 import binding

pytestmark = pytest.mark.gpu

RTOL = 1e-13          # of |alpha| * sum |X||Y|: the bound tests/test_gpu_cc.py::test_dot_matches_numpy uses


@pytest.fixture(scope="module")
def ctx():
    c = pkg.Context(0)
    yield c
    c.destroy()


def _pair(ctx, shape, seed):
    X, Y = ctx.tensor_create(shape, zero=False), ctx.tensor_create(shape, zero=False)
    ctx.synth_normal(X, seed, 1)
    ctx.synth_normal(Y, seed, 2)
    return X, Y


def _both(ctx, X, Y, conj, alpha):
    """(tcb_dot_noalloc, tcb_dot) on the same operands, each into a rank-0 tensor of its own"""
    Dn, Dd = ctx.tensor_create(()), ctx.tensor_create(())
    ctx.dot_noalloc(Dn, X, Y, conj, alpha)
    ctx.dot(Dd, X, Y, conj, alpha)
    out = complex(ctx.tensor_download(Dn)), complex(ctx.tensor_download(Dd))
    Dn.destroy()
    Dd.destroy()
    return out


def test_two_calls_in_a_row_match_the_existing_path(ctx):
    """Call 1: 3 000 001 elements (1465 tiles of 2048 and a ragged one).  Call 2, straight after it on the same stream: 70 001
    elements (35 tiles): the array still holds call 1's 1465 partial sums, none of which may enter.  Then call 1 again: the
    same bits as the first time."""
    alpha = 0.5 - 1.5j
    X1, Y1 = _pair(ctx, (3000001,), 11)
    X2, Y2 = _pair(ctx, (70001,), 12)
    D1, D2, D3 = ctx.tensor_create(()), ctx.tensor_create(()), ctx.tensor_create(())
    ctx.dot_noalloc(D1, X1, Y1, True, alpha)                   # two calls in a row, nothing in between
    ctx.dot_noalloc(D2, X2, Y2, False, alpha)
    ctx.dot_noalloc(D3, X1, Y1, True, alpha)
    got1, got2, got3 = (complex(ctx.tensor_download(d)) for d in (D1, D2, D3))
    R1, R2 = ctx.tensor_create(()), ctx.tensor_create(())
    ctx.dot(R1, X1, Y1, True, alpha)                           # the existing path
    ctx.dot(R2, X2, Y2, False, alpha)
    ref1, ref2 = complex(ctx.tensor_download(R1)), complex(ctx.tensor_download(R2))
    hX1, hY1, hX2, hY2 = (ctx.tensor_download(t) for t in (X1, Y1, X2, Y2))
    sn1 = abs(alpha) * float(np.sum(np.abs(hX1) * np.abs(hY1)))
    sn2 = abs(alpha) * float(np.sum(np.abs(hX2) * np.abs(hY2)))
    assert abs(got1 - ref1) <= RTOL * sn1 and abs(got2 - ref2) <= RTOL * sn2
    assert got3 == got1                                        # deterministic, and untouched by what call 2 left behind
    # both paths against numpy as well (the existing path's own test does the same)
    assert abs(got1 - alpha * np.vdot(hX1, hY1)) <= RTOL * sn1
    assert abs(got2 - alpha * np.sum(hX2 * hY2)) <= RTOL * sn2
    for t in (X1, Y1, X2, Y2, D1, D2, D3, R1, R2):
        t.destroy()


@pytest.mark.parametrize("shape,conj", [((), True), ((7, 5, 3), False), ((300, 41, 9), True), ((2048,), True), ((2049,), False),
                                        ((4100, 4100), True)])
def test_shapes_tile_sizes_and_the_exactly_real_norm(ctx, shape, conj):
    """rank 0 ... one tile exactly, one tile + 1, and 16.8 M elements (8192 tiles would not do: the tile doubles to 4096)"""
    X, Y = _pair(ctx, shape, 20 + len(shape))
    alpha = -1.25 + 0.75j
    got, ref = _both(ctx, X, Y, conj, alpha)
    hX, hY = ctx.tensor_download(X), ctx.tensor_download(Y)
    assert abs(got - ref) <= RTOL * abs(alpha) * float(np.sum(np.abs(hX) * np.abs(hY)))
    nrm, nrm_ref = _both(ctx, X, X, True, 1.0)
    assert nrm.imag == 0.0 and abs(nrm - nrm_ref) <= RTOL * float(np.sum(np.abs(hX) ** 2))
    X.destroy()
    Y.destroy()


def test_the_maximum_size_runs_and_one_element_more_is_refused(ctx):
    """536 870 912 elements (8.6 GB, 8192 tiles of 65536): <x|x> of a constant tensor is exact; one element more is refused
    with TCB_EUNSUPPORTED, D untouched, and the context goes on working."""
    nmax = binding.DOT_NOALLOC_MAX_ELEMS
    big = ctx.tensor_create((nmax + 1,), zero=False)
    ctx.tensor_fill(big, 1.0 - 1.0j)
    D = ctx.tensor_create(())
    ctx.tensor_fill(D, 7.0)
    with pytest.raises(pkg.TcbError) as ei:
        ctx.dot_noalloc(D, big, big, True, 1.0)
    assert ei.value.code == binding.TCB_EUNSUPPORTED and "exceed" in str(ei.value)
    assert complex(ctx.tensor_download(D)) == 7.0
    big.destroy()
    top = ctx.tensor_create((nmax,), zero=False)
    ctx.tensor_fill(top, 1.0 - 1.0j)
    ctx.dot_noalloc(D, top, top, True, 0.5)
    assert complex(ctx.tensor_download(D)) == float(nmax)       # 0.5 * nmax * |1 - i|^2, every partial sum an exact integer
    top.destroy()
    # argument checks are those of tcb_dot
    X, Y = ctx.tensor_create((5, 4)), ctx.tensor_create((4, 5))
    for args, code in (((X, X, Y), binding.TCB_ESHAPE), ((D, X, Y), binding.TCB_ESHAPE), ((D, D, D), binding.TCB_EALIAS)):
        with pytest.raises(pkg.TcbError) as ei:
            ctx.dot_noalloc(*args, True, 1.0)
        assert ei.value.code == code
    ctx.dot_noalloc(D, X, X, True, 1.0)
    assert complex(ctx.tensor_download(D)) == 0.0
    for t in (X, Y, D):
        t.destroy()
