"""BASELINE.json configs[4], first half: every binary contraction of a spin-orbital CCSD residual, in every output
index order a generator that unrolls its permutation operators would emit (binary
contractions only; unrolled permutations).  tenpi's own OpMin-factorised list is not available (there is
no tenpi output in /root/reference); this is the stand-in derived from the verified CCSD equations (reading 9):
Stanton-type intermediates, t_i^a stored T1(a,i), t_ij^ab stored T2(a,b,i,j), integral blocks in bra-ket order.

    python -m paper_2409_06759_b200.ccsd_contractions [--o 30 --v 150]      # the timed sweep, one JSON line per call

Index letters: i j k l m n = occupied (extent o), a b c d e f = virtual (extent v).  `P` lists the permutation
operators of the term: "ij" = P(ij), "ab" = P(ab); each operator doubles the emitted output orders (with sign)."""
import argparse
import json
import sys

OCC = "ijklmn"

# (expression, permutation operators)
CONTRACTIONS = [
    ("tt(a,b,i,j)=T1(a,i)*T1(b,j)", ""),                       # K = 1 outer product
    ("Fae(a,e)+=T1(a,m)*fov(m,e)", ""),
    ("Fae(a,e)+=ovvv(m,a,f,e)*T1(f,m)", ""),                   # N = 1
    ("Fae(a,e)+=tau(a,f,m,n)*oovv(m,n,e,f)", ""),
    ("Fmi(m,i)+=fov(m,e)*T1(e,i)", ""),
    ("Fmi(m,i)+=ooov(m,n,i,e)*T1(e,n)", ""),                   # N = 1
    ("Fmi(m,i)+=oovv(m,n,e,f)*tau(e,f,i,n)", ""),
    ("Fme(m,e)+=oovv(m,n,e,f)*T1(f,n)", ""),                   # N = 1
    ("Wmnij(m,n,i,j)+=ooov(m,n,i,e)*T1(e,j)", "ij"),
    ("Wmnij(m,n,i,j)+=oovv(m,n,e,f)*tau(e,f,i,j)", ""),
    ("Wabef(a,b,e,f)+=vovv(a,m,e,f)*T1(b,m)", "ab"),
    ("Wabef(a,b,e,f)+=tau(a,b,m,n)*oovv(m,n,e,f)", ""),
    ("Wmbej(m,b,e,j)+=ovvv(m,b,e,f)*T1(f,j)", ""),
    ("Wmbej(m,b,e,j)+=oovo(m,n,e,j)*T1(b,n)", ""),
    ("Wmbej(m,b,e,j)+=oovv(m,n,e,f)*Q(f,b,j,n)", ""),
    ("R1(a,i)+=Fae(a,e)*T1(e,i)", ""),
    ("R1(a,i)+=T1(a,m)*Fmi(m,i)", ""),
    ("R1(a,i)+=T2(a,e,i,m)*Fme(m,e)", ""),                     # N = 1
    ("R1(a,i)+=ovov(n,a,i,f)*T1(f,n)", ""),                    # N = 1
    ("R1(a,i)+=ovvv(m,a,e,f)*T2(e,f,i,m)", ""),
    ("R1(a,i)+=T2(a,e,m,n)*oovo(n,m,e,i)", ""),
    ("G(b,e)+=T1(b,m)*Fme(m,e)", ""),
    ("R2(a,b,i,j)+=T2(a,e,i,j)*G(b,e)", "ab"),
    ("Gm(m,j)+=Fme(m,e)*T1(e,j)", ""),
    ("R2(a,b,i,j)+=T2(a,b,i,m)*Gm(m,j)", "ij"),
    ("R2(a,b,i,j)+=tau(a,b,m,n)*Wmnij(m,n,i,j)", ""),
    ("R2(a,b,i,j)+=Wabef(a,b,e,f)*tau(e,f,i,j)", ""),
    ("R2(a,b,i,j)+=T2(a,e,i,m)*Wmbej(m,b,e,j)", "ij,ab"),
    ("Z(m,b,i,j)+=ovvo(m,b,e,j)*T1(e,i)", ""),
    ("R2(a,b,i,j)+=T1(a,m)*Z(m,b,i,j)", "ij,ab"),
    ("R2(a,b,i,j)+=vvvo(a,b,e,j)*T1(e,i)", "ij"),
    ("R2(a,b,i,j)+=T1(a,m)*ovoo(m,b,i,j)", "ab"),
]


def split(expr):
    """'D(a,b)+=L(a,c)*R(c,b)' -> (['a','b'], op, ['a','c'], ['c','b'])"""
    import re
    m = re.fullmatch(r"\s*\w+\(([^)]*)\)\s*(\+?=)\s*\w+\(([^)]*)\)\s*\*\s*\w+\(([^)]*)\)\s*", expr)
    lab = lambda g: [x.strip() for x in g.split(",") if x.strip()]
    return lab(m.group(1)), m.group(2), lab(m.group(3)), lab(m.group(4))


def extent(label, o, v):
    return o if label[0] in OCC else v


def shapes(expr, o, v):
    d, _, l, r = split(expr)
    return tuple(extent(x, o, v) for x in d), tuple(extent(x, o, v) for x in l), tuple(extent(x, o, v) for x in r)


def output_orders(expr, ops):
    """Unroll the permutation operators on the OUTPUT: returns [(expression with permuted D labels, sign)].
    P(xy) F = F - F(x<->y): the generator emits the same contraction once more with x and y exchanged in D and -alpha."""
    d, op, l, r = split(expr)
    variants = [(list(d), 1.0)]
    for pair in [p for p in ops.split(",") if p]:
        x, y = pair[0], pair[1]
        more = []
        for labels, sign in variants:
            sw = [y if t == x else x if t == y else t for t in labels]
            more.append((sw, -sign))
        variants += more
    name = expr[:expr.index("(")]
    rhs = expr[expr.index(op) + len(op):]
    return [(f"{name}({','.join(labels)}){op}{rhs}", sign) for labels, sign in variants]


def all_calls(o, v):
    """every (expression, alpha sign, shapes) the sweep issues"""
    out = []
    for expr, ops in CONTRACTIONS:
        sd, sl, sr = shapes(expr, o, v)
        for e, sign in output_orders(expr, ops):
            d, _, _, _ = split(e)
            out.append((e, sign, tuple(extent(x, o, v) for x in d), sl, sr))
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--o", type=int, default=30)
    ap.add_argument("--v", type=int, default=150)
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--peak-tflops", type=float, default=148 * 128 * 1.965e-3)
    ap.add_argument("--hbm-gbs", type=float, default=6546.6)
    args = ap.parse_args()
    from . import Context
    ctx = Context(0)
    cache = {}

    def tensor(shape, tid):
        key = (shape, tid)
        if key not in cache:
            t = ctx.tensor_create(shape)
            ctx.synth_normal(t, 20240911, tid)
            cache[key] = t
        return cache[key]

    total_ms, total_flops = 0.0, 0.0
    for e, sign, sd, sl, sr in all_calls(args.o, args.v):
        D, L, R = tensor(sd, 1), tensor(sl, 2), tensor(sr, 3)
        plan = ctx.plan_describe(e, D, L, R)
        ctx.contract(e, D, L, R, 0.5 * sign)
        ctx.sync()
        ts = []
        for _ in range(args.reps):
            ctx.timer_start()
            ctx.contract(e, D, L, R, 0.5 * sign)
            ts.append(ctx.timer_stop())
        ms = min(ts)
        bound_ms = max(plan["flops"] / (args.peak_tflops * 1e9), plan["bytes"] / (args.hbm_gbs * 1e6))
        total_ms += ms
        total_flops += plan["flops"]
        print(json.dumps({"expr": e, "M": plan["M"], "N": plan["N"], "K": plan["K"], "ms": ms,
                          "tflops": plan["flops"] / ms * 1e-9, "gbs": plan["bytes"] / ms * 1e-6,
                          "bound": "tensor" if plan["flops"] / (args.peak_tflops * 1e9) >= plan["bytes"] / (args.hbm_gbs * 1e6) else "hbm",
                          "frac_of_bound": bound_ms / ms, "permute_A": plan["permute_A"], "permute_B": plan["permute_B"]}),
              flush=True)
    print(json.dumps({"total_ms": total_ms, "total_tflops": total_flops / total_ms * 1e-9, "o": args.o, "v": args.v}),
          flush=True)
    ctx.destroy()


if __name__ == "__main__":
    sys.exit(main())
