"""Per-call timing table of one CCSDT residual evaluation on seeded synthetic integrals and amplitudes:
every library call of the driver program is timed on its own with CUDA events on the context's stream (a synchronise in
front of each), after the whole program has run four times un-instrumented (wall clock of those passes printed first).

    python -m paper_2409_06759_b200.ccsdt_profile 12 60            # packed storage (ccd.ccsdt_residual_packed) and, at
                                                                   # o=12 v=60 only, the dense program beside it
    python -m paper_2409_06759_b200.ccsdt_profile 16 100 --top 30  # a size whose dense T3 does not fit one GPU

Inputs: h, g = <pq||rs> over n = o + v spinors (normal, antisymmetrised), T1, T2 (antisymmetric), T3p(a<b<c,i<j<k): the
counter-based generator of synth.py / tcb_synth_normal, seed 3.  TF = the planner's flop count (8 M N K) / time."""
import argparse
import time

import numpy as np


class _Timed:
    """forwards to a Context; times contract / pack / unpack / antisym_pack / antisymmetrize / add one by one"""

    def __init__(self, ctx):
        self.ctx, self.rows = ctx, []

    def __getattr__(self, name):
        return getattr(self.ctx, name)

    def _t(self, what, fn, *args):
        self.ctx.sync()
        self.ctx.timer_start()
        fn(*args)
        self.rows.append([self.ctx.timer_stop(), what, None])

    def contract(self, e, D, L, R, alpha=1.0):
        p = self.ctx.plan_describe(e, D, L, R)
        self._t(f"{e:44s} {p['M']}x{p['N']}x{p['K']} {p['route']} {p['feed_A'][0]}{p['feed_B'][0]}", self.ctx.contract, e, D, L, R, alpha)
        self.rows[-1][2] = p["flops"]

    def pack(self, s, D, L):
        self._t("pack " + s, self.ctx.pack, s, D, L)

    def unpack(self, s, D, L, a=1.0):
        self._t("unpack " + s, self.ctx.unpack, s, D, L, a)

    def antisym_pack(self, s, D, L, a=1.0):
        self._t("antisym_pack " + s, self.ctx.antisym_pack, s, D, L, a)

    def antisymmetrize(self, s, D, X, a=1.0):
        self._t("antisymmetrize " + s, self.ctx.antisymmetrize, s, D, X, a)

    def add(self, s, D, L, a=1.0):
        self._t("add " + s, self.ctx.add, s, D, L, a)


def table(rows, top):
    for ms, what, flops in sorted(rows, key=lambda r: -r[0])[:top]:
        print(f"{ms:9.3f} ms  {what}" + (f"  {flops / ms * 1e-9:.1f} TF" if flops else ""))
    fl = sum(r[2] for r in rows if r[2])
    tot = sum(r[0] for r in rows)
    print(f"sum of the {len(rows)} timed calls: {tot:.2f} ms, {fl:.4g} flop executed, {fl / tot * 1e-9:.1f} TFLOP/s")


def main():
    import paper_2409_06759_b200 as pkg
    from paper_2409_06759_b200 import ccd
    ap = argparse.ArgumentParser()
    ap.add_argument("o", type=int, nargs="?", default=12)
    ap.add_argument("v", type=int, nargs="?", default=60)
    ap.add_argument("--top", type=int, default=24)
    a = ap.parse_args()
    o, v = a.o, a.v
    n = o + v
    ctx = pkg.Context(0)
    hh, gg = ctx.tensor_create((n, n)), ctx.tensor_create((n, n, n, n))
    ctx.synth_normal(hh, 3, 1, sigma=0.05)
    ctx.synth_normal(gg, 3, 2, antisym=((0, 1), (2, 3)), sigma=0.02)
    T1, T2 = ctx.tensor_create((v, o)), ctx.tensor_create((v, v, o, o))
    ctx.synth_normal(T1, 3, 3, sigma=0.05)
    ctx.synth_normal(T2, 3, 4, antisym=((0, 1), (2, 3)), sigma=0.05)
    T3p = ctx.tensor_create((ctx.packed_extent(v, 3), ctx.packed_extent(o, 3)))
    ctx.synth_normal(T3p, 3, 5, sigma=0.01)
    print(f"o={o} v={v}: T3p {T3p.nbytes / 1e6:.0f} MB packed, {16e-9 * v ** 3 * o ** 3:.2f} GB dense")
    Rs = None
    for rep in range(4):
        ctx.sync()
        t0 = time.perf_counter()
        Rs = ccd.ccsdt_residual_packed(ctx, o, hh, gg, T1, T2, T3p, *(Rs or ()))
        ctx.sync()
        print(f"ccsdt_residual_packed pass {rep}: {(time.perf_counter() - t0) * 1e3:.2f} ms wall")
    tm = _Timed(ctx)
    ccd.ccsdt_residual_packed(tm, o, hh, gg, T1, T2, T3p, *Rs)
    table(tm.rows, a.top)
    if (o, v) == (12, 60):
        T3 = ctx.tensor_create((v, v, v, o, o, o), zero=False)
        ctx.unpack("T(a,b,c,i,j,k)=P(a<b<c,i<j<k)", T3, T3p, 1.0)
        Ds = None
        for rep in range(3):
            ctx.sync()
            t0 = time.perf_counter()
            Ds = ccd.ccsdt_residual(ctx, o, hh, gg, T1, T2, T3, *(Ds or ()))
            ctx.sync()
            print(f"ccsdt_residual (dense) pass {rep}: {(time.perf_counter() - t0) * 1e3:.2f} ms wall")
        for name, x, y in (("R1", Rs[0], Ds[0]), ("R2", Rs[1], Ds[1])):
            x, y = ctx.tensor_download(x), ctx.tensor_download(y)
            print(f"{name}: max |packed - dense| / max |dense| = {float(np.abs(x - y).max() / np.abs(y).max()):.2e}")
        D3p = ctx.tensor_create(Rs[2].extents, zero=False)
        ctx.pack("P(a<b<c,i<j<k)=R(a,b,c,i,j,k)", D3p, Ds[2])
        x, y = ctx.tensor_download(Rs[2]), ctx.tensor_download(D3p)
        print(f"R3: max |R3p - pack(dense R3)| / max = {float(np.abs(x - y).max() / np.abs(y).max()):.2e}")
        tm = _Timed(ctx)
        ccd.ccsdt_residual(tm, o, hh, gg, T1, T2, T3, *Ds)
        table(tm.rows, 8)


if __name__ == "__main__":
    main()
