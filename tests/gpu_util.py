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


# ---- full-size parity: the oracle on sampled outputs, inputs regenerated on the host -------------------------------------
def slab(ctx, t, last_index):
    """Borrowed view of t[..., last_index] (contiguous in the column-major layout): a tensor of rank - 1."""
    n = int(np.prod(t.extents[:-1], dtype=np.int64))
    return ctx.tensor_wrap(t.extents[:-1], ctx.tensor_device_ptr(t) + 16 * n * int(last_index))


def download_at(ctx, t, subs):
    """t[np.ix_(*subs)] without downloading all of t: one slab per sampled value of the last index."""
    out = np.empty([len(s) for s in subs], dtype=np.complex128, order="F")
    if t.nbytes <= (1 << 28) or len(t.extents) < 2:
        return np.asfortranarray(ctx.tensor_download(t)[np.ix_(*subs)])
    for q, last in enumerate(subs[-1]):
        view = slab(ctx, t, last)
        out[..., q] = download_at(ctx, view, subs[:-1])
        view.destroy()
    return out


def sample_indices(rng, extent, n, edges=True):
    """n sorted distinct indices of range(extent); with edges the first and the last index are among them"""
    n = min(n, extent)
    pick = set(rng.choice(extent, size=n, replace=False).tolist())
    if edges and n >= 2:
        pick = set(list(pick)[:n - 2]) | {0, extent - 1}
        while len(pick) < n:
            pick.add(int(rng.integers(extent)))
    return np.array(sorted(pick), dtype=np.int64)


def sampled_contraction_parity(ctx, expr, ext, alpha, seed, rng, nsub=8, antisym_l=(), antisym_r=(), sets=1,
                               sigma=1.0, operands=None):
    """Full-size parity of one tcb_contract call on sampled outputs (the oracle cannot run these sizes whole).

    The operands are generated ON THE DEVICE by the seeded generator (tensor ids 1, 2, 3 = L, R, D); the oracle's inputs
    are the host twin's values (paper_2409_06759_b200/synth.py, index-keyed and bit-identical: tests/test_gpu_permute.py)
    for the sampled rows and columns only: per free label `nsub` sampled index values, every value of every contracted
    label.  Nothing the oracle reads comes from the device.  Returns (max normalised error, outputs checked)."""
    import oracle
    from paper_2409_06759_b200 import synth
    dl, ll, rl = split_expr(expr)
    shp = lambda labs: [ext[x] for x in labs]
    if operands is None:
        L, R, D = ctx.tensor_create(shp(ll)), ctx.tensor_create(shp(rl)), ctx.tensor_create(shp(dl))
        ctx.synth_normal(L, seed, 1, antisym=antisym_l, sigma=sigma)
        ctx.synth_normal(R, seed, 2, antisym=antisym_r, sigma=sigma)
        ctx.synth_normal(D, seed, 3, sigma=sigma)
    else:
        L, R, D = operands
        ctx.synth_normal(D, seed, 3, sigma=sigma)          # D back to its seeded start
    ctx.contract(expr, D, L, R, alpha)
    worst, checked = 0.0, 0
    for s in range(sets):
        pick = {x: (sample_indices(rng, ext[x], nsub, edges=(s == 0)) if x in dl else np.arange(ext[x])) for x in ext}
        hL = synth.tensor(seed, 1, shp(ll), antisym=antisym_l, sigma=sigma, sub=[pick[x] for x in ll])
        hR = synth.tensor(seed, 2, shp(rl), antisym=antisym_r, sigma=sigma, sub=[pick[x] for x in rl])
        hD = synth.tensor(seed, 3, shp(dl), sigma=sigma, sub=[pick[x] for x in dl])
        ref, sn = oracle.contract(expr, hD, hL, hR, alpha)
        got = download_at(ctx, D, [pick[x] for x in dl])
        worst = max(worst, parity_error(got, ref, sn))
        checked += got.size
    if operands is None:
        for t in (L, R, D):
            t.destroy()
    return worst, checked
