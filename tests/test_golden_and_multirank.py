"""-m "not gpu": (1) the oracle's CCD equations against the paper's printed diagram count (tests/golden/, PAPER.md
Table I); (2) the only cross-rank step of bench.py -- max over ranks of the device time, whole-job throughput --
on two gloo ranks (the path does not shard: DESIGN.md "Multi-GPU: replicas only")."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLDEN = os.path.join(ROOT, "tests", "golden", "paper_table1_diagram_counts.txt")


def read_counts():
    out = {}
    for line in open(GOLDEN):
        line = line.strip()
        if line and not line.startswith("#"):
            k, v = line.split()
            out[k] = int(v)
    return out


def test_paper_table1_fixture_is_the_papers():
    c = read_counts()
    assert c == {"CCD": 11, "CCSD": 48, "CCSDT": 102, "CCSDTQ": 183, "CCSDTQP": 289}


def test_oracle_ccd_term_count_matches_paper_table1():
    """CCD has 11 diagrams = 10 doubles-amplitude terms + 1 energy term.  A dropped or duplicated term in
    oracle/cc.py changes the count (and the Fock-space pin in test_oracle_cc.py catches a wrong one)."""
    from oracle import cc
    from paper_2409_06759_b200 import synth
    o, v = 2, 3
    n = o + v
    rng = np.random.default_rng(1)
    f = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    f = f + f.conj().T
    g = synth.tensor(7, 1, [n] * 4, antisym=((0, 1), (2, 3)), sigma=0.1, hermitian=True)
    t = synth.tensor(7, 2, [v, v, o, o], antisym=((0, 1), (2, 3)))
    _, _, n_amp, n_en = cc.ccd_residual_unfactorised(o, f, g, t)
    assert n_amp + n_en == read_counts()["CCD"]
    assert (n_amp, n_en) == (10, 1)


def _rank_main(rank, world, port, q):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r "measured" (10 + r) ms for the step and (30 - r) ms end to end
    ms, e2e = bench.max_over_ranks([10.0 + rank, 30.0 - rank], dist, "cpu")
    dist.barrier()
    dist.destroy_process_group()
    q.put((rank, ms, e2e))


def test_two_rank_replicas_take_the_slowest_rank_time():
    import torch.multiprocessing as mp
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got == [(0, 11.0, 30.0), (1, 11.0, 30.0)]
    sys.path.insert(0, ROOT)
    import bench
    # whole-job value: both replicas' flops over the slowest rank's time
    assert bench.job_throughput(2, 1e9, 11.0) == pytest.approx(2 * 1e9 / 11e-3 * 1e-9)
    assert bench.max_over_ranks([1.0, 2.0], None, "cpu") == [1.0, 2.0]


def test_transpose_benchmark_sample_holds_the_required_permutations():
    """BASELINE.json configs[4]: 48 sampled rank-6 permutations; the sample is seeded and always contains the identity,
    the reversal, the half swap and the six transpositions of P(a/bc), P(k/ij)."""
    from paper_2409_06759_b200 import transpose_bench as tb
    s = tb.rank6_sample()
    assert len(s) == 48 and len(set(s)) == 48 and s == tb.rank6_sample()
    assert all(sorted(p) == list(range(6)) for p in s)
    for need in [(0, 1, 2, 3, 4, 5), (5, 4, 3, 2, 1, 0), (3, 4, 5, 0, 1, 2), (1, 0, 2, 3, 4, 5), (2, 1, 0, 3, 4, 5),
                 (0, 1, 2, 5, 4, 3), (0, 1, 2, 3, 5, 4)]:
        assert need in s
    assert tb.expression((1, 0, 2, 3)) == "D(b,a,c,d)=L(a,b,c,d)"


def test_ccsd_contraction_list_is_well_formed():
    """configs[4]: every expression of the CCSD stand-in list is a valid binary contraction for the host planner (labels
    twice overall, extents by index type), and the permutation operators unroll into the signed output orders."""
    from paper_2409_06759_b200 import ccsd_contractions as cl, binding
    o, v = 3, 5
    calls = cl.all_calls(o, v)
    assert len(calls) == sum(2 ** len([p for p in ops.split(",") if p]) for _, ops in cl.CONTRACTIONS)
    for e, sign, sd, sl, sr in calls:
        plan = binding.plan_describe_host(e, sd, sl, sr)
        d, _, l, r = cl.split(e)
        assert plan["M"] * plan["N"] == int(np.prod(sd)) and sign in (1.0, -1.0)
    orders = cl.output_orders("R2(a,b,i,j)+=T2(a,e,i,m)*Wmbej(m,b,e,j)", "ij,ab")
    assert [(x[:12], s) for x, s in orders] == [("R2(a,b,i,j)+", 1.0), ("R2(a,b,j,i)+", -1.0), ("R2(b,a,i,j)+", -1.0),
                                                ("R2(b,a,j,i)+", 1.0)]
    kinds = {(p["K"] == 1, p["N"] == 1) for p in (binding.plan_describe_host(e, sd, sl, sr) for e, _, sd, sl, sr in calls)}
    assert (True, False) in kinds and (False, True) in kinds          # the list holds an outer product and N = 1 cases


def test_e2e_rank_groups_fit_the_host():
    """bench.py e2e: N replicas each pin 30.7 GB; on a 196 GB host eight of them do not fit at once"""
    import bench
    per = 27_648_000_000 + 1_024_000_000 + 2 * 1_024_000_000
    assert bench.e2e_ranks_at_once(1, 196 << 30, per) == 1
    assert bench.e2e_ranks_at_once(4, 196 << 30, per) == 4
    assert bench.e2e_ranks_at_once(8, 196 << 30, per) == 4
    assert bench.e2e_ranks_at_once(8, 2048 << 30, per) == 8
    assert bench.e2e_ranks_at_once(8, 16 << 30, per) == 1
