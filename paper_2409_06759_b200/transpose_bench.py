"""Standalone transposition benchmark of BASELINE.json configs[4]: every one of the 24 rank-4 permutations and a seeded
sample of 48 rank-6 permutations of complex128 tensors from 64 MB to 8 GB, each one tcb_permute call timed with CUDA
events on the context's stream.  GB/s = 2 * 16 bytes per element / time (read once, write once).

    python -m paper_2409_06759_b200.transpose_bench                      # the whole sweep, one JSON line per shape
    python -m paper_2409_06759_b200.transpose_bench --shape 200,200,40,40 --perm 1,0,2,3 --reps 2     # one case (profiling)

The rank-6 sample (seed 5) always holds the identity, the full reversal, the (i,j,k,a,b,c) half swap and the 6 single
transpositions used by P(a/bc) and P(k/ij); the rest are drawn with random.Random(5)."""
import argparse
import itertools
import json
import random
import sys

RANK4_SHAPES = [(100, 100, 20, 20), (150, 150, 30, 30), (200, 200, 40, 40), (150, 150, 150, 150)]
RANK6_SHAPES = [(28, 28, 28, 6, 6, 6), (40, 40, 40, 8, 8, 8), (60, 60, 60, 12, 12, 12)]


def rank6_sample(n=48, seed=5):
    fixed = [tuple(range(6)), tuple(reversed(range(6))), (3, 4, 5, 0, 1, 2)]
    for a, b in [(0, 1), (0, 2), (1, 2), (3, 4), (3, 5), (4, 5)]:
        p = list(range(6))
        p[a], p[b] = p[b], p[a]
        fixed.append(tuple(p))
    rng = random.Random(seed)
    out = list(fixed)
    while len(out) < n:
        p = tuple(rng.sample(range(6), 6))
        if p not in out:
            out.append(p)
    return out


def expression(perm):
    lab = "abcdef"[:len(perm)]
    return "D(" + ",".join(lab[p] for p in perm) + ")=L(" + ",".join(lab) + ")"


ROTATE_BELOW_BYTES = 512e6      # source + destination under 4x the 126 MB L2: rotate over distinct buffer pairs


def time_permutation(ctx, Ls, shape, perm, reps=3, warm=1):
    """ms per call.  Ls: the source tensors; with more than one, a timed repetition runs the permutation once on every
    (source, destination) pair back to back -- together larger than 4x L2, so every call reads from HBM, and the
    CUDA-event granularity (4 us on this box) is spread over all of them."""
    Ds = [ctx.tensor_create(tuple(shape[p] for p in perm)) for _ in Ls]
    e = expression(perm)
    for _ in range(warm):
        for D, L in zip(Ds, Ls):
            ctx.permute(e, D, L)
    ctx.sync()
    ts = []
    for _ in range(reps):
        ctx.timer_start()
        for D, L in zip(Ds, Ls):
            ctx.permute(e, D, L)
        ts.append(ctx.timer_stop() / len(Ls))
    for D in Ds:
        D.destroy()
    return min(ts)


def rotation(shape):
    n = 1
    for e in shape:
        n *= e
    return 1 if 32.0 * n >= ROTATE_BELOW_BYTES else int(-(-ROTATE_BELOW_BYTES // (32.0 * n)))


def sweep_shape(ctx, shape, perms, reps=3):
    n = 1
    for e in shape:
        n *= e
    Ls = [ctx.tensor_create(shape) for _ in range(rotation(shape))]
    for L in Ls:
        ctx.synth_index_linear(L)
    gbs = [32.0 * n / time_permutation(ctx, Ls, shape, p, reps) * 1e-6 for p in perms]
    for L in Ls:
        L.destroy()
    ctx.sync()
    return gbs


def summary(shape, gbs, hbm_gbs):
    s = sorted(gbs)
    return {"shape": list(shape), "megabytes": 16e-6 * __import__("math").prod(shape), "permutations": len(s),
            "l2": "larger than L2" if rotation(shape) == 1 else f"rotating over {rotation(shape)} buffer pairs per timed repetition",
            "gbs_min": s[0], "gbs_median": s[len(s) // 2], "gbs_max": s[-1],
            "frac_hbm_measured_median": s[len(s) // 2] / hbm_gbs,
            "share_at_or_above_75pct": sum(g >= 0.75 * hbm_gbs for g in s) / len(s)}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--shape", default=None, help="comma-separated extents; default: the whole configs[4] sweep")
    ap.add_argument("--perm", default=None, help="comma-separated permutation, e.g. 1,0,2,3 (needs --shape)")
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--hbm-gbs", type=float, default=6546.6, help="measured copy bandwidth (MEASURED_PEAKS.json)")
    ap.add_argument("--max-gb", type=float, default=9.0, help="skip shapes above this size")
    args = ap.parse_args()
    from . import Context
    ctx = Context(0)
    if args.shape:
        shape = tuple(int(x) for x in args.shape.split(","))
        if args.perm:
            perms = [tuple(int(x) for x in args.perm.split(","))]
        else:
            perms = list(itertools.permutations(range(4))) if len(shape) == 4 else rank6_sample()
        gbs = sweep_shape(ctx, shape, perms, args.reps)
        print(json.dumps({"shape": list(shape), "perms": [list(p) for p in perms], "gbs": gbs}), flush=True)
    else:
        for shape in RANK4_SHAPES + RANK6_SHAPES:
            n = 1
            for e in shape:
                n *= e
            if 16e-9 * n > args.max_gb:
                continue
            perms = list(itertools.permutations(range(4))) if len(shape) == 4 else rank6_sample()
            print(json.dumps(summary(shape, sweep_shape(ctx, shape, perms, args.reps), args.hbm_gbs)), flush=True)
    ctx.destroy()


if __name__ == "__main__":
    sys.exit(main())
