#!/usr/bin/env python
"""bench.py -- one JSON line for the driver (contract in DESIGN.md "Measurement").

A step = one pass of the whole hot path (S1-S7) over one batch of synthetic input: the full spin-orbital CCD
residual of BASELINE.json configs[1] (o=20, v=80, complex128) issued call by call through the C ABI, i.e. 11
contractions (S1-S5, four of them with operand permutations S3), 6 fused permute-sums (S6) and 3 adds (S7).
metric = complex-FP64 contraction throughput, GFLOP/s with 8 real flop per complex multiply-add.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-extras]

N > 1 (torchrun): the path does not shard (replicas only) -- every rank runs an
independent replica on its own GPU, no data-path collective; value = all ranks' flops / max-over-ranks time.
--impl reference: the CPU oracle (oracle/, as it stands) on the host cores, on a bounded sample of the same
workload.  Inputs are seeded and synthetic (paper_2409_06759_b200/synth.py recipe), generated on the device.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "complex-FP64 contraction GFLOP/s (CCD residual, 8 flop per complex MAC)"
O, V = 20, 80                                   # BASELINE.json configs[1]
WORKLOAD = f"configs[1]: full spin-orbital CCD residual, complex128, o={O}, v={V}"
# nominal FP64 tensor peak derived from unit counts: 148 SMs x 4 sub-partitions x one DMMA.8x8x4
# (512 flop) per 16 cycles x 1.965 GHz; the register-resident DMMA loop (tcb_measure_fp64_tensor_peak) reaches 37.0.
FP64_TENSOR_PEAK_TFLOPS = 148 * 128 * 1.965e9 * 1e-12
# DRAM traffic of the 11 zgemm_dmma_kernel launches of one step, from the ncu --set full capture committed as
# profiles/r1b_zgemm_ncu_full.md (2.751 GB read + 0.277 GB written); bench.py itself never runs under a profiler
ZGEMM_DRAM_BYTES_PER_STEP = 3.028e9
ZGEMM_LAUNCHES_PER_STEP = 11


EVENT_EVERY = 5          # per-launch event pairs on every 5th timed step (see run_ours)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip the configs[2..4] context measurements")
    ap.add_argument("--no-graph", action="store_true", help="issue every timed step call by call (no CUDA graph replay)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md recipe)
# ---------------------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), [x.strip() for x in line.split(",")]))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        rows = [r for t, r in self.rows if t0 <= t <= t1 + 0.1 and len(r) >= 7] or [r for _, r in self.rows if len(r) >= 7]
        if not rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm = sorted(float(r[0]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(rows[0][1]), "reasons": reasons,
                "samples": len(rows), "power_w_max": max(float(r[2]) for r in rows)}


# ---------------------------------------------------------------------------------------------------------
# workload: configs[1] on the device (same recipe and seeds as synth.config_ccd, generated by csrc/synth.cu)
# ---------------------------------------------------------------------------------------------------------
def make_ccd_inputs(ctx, o, v, config_no=2, sigma=0.1, want_energies=False):
    import numpy as np
    from paper_2409_06759_b200 import synth
    seed, n = synth.SEED0 + config_no, o + v
    eo, ev = synth.orbital_energies(seed, o, v)
    rng = {"o": (0, o), "v": (o, v)}
    B = {}
    for name in ("vvoo", "oovv", "oooo", "vvvv", "ovvo"):
        t = ctx.tensor_create([rng[c][1] for c in name])
        ctx.synth_normal(t, seed, 1, antisym=((0, 1), (2, 3)), sigma=sigma, hermitian=True,
                         label_offset=[rng[c][0] for c in name], label_extents=[n] * 4)
        B[name] = t
    B["foo"] = ctx.tensor_from_numpy(np.diag(eo).astype(np.complex128))
    B["fvv"] = ctx.tensor_from_numpy(np.diag(ev).astype(np.complex128))
    T = ctx.tensor_create((v, v, o, o))
    ctx.synth_mp2_amplitudes(T, B["vvoo"], eo, ev)
    if want_energies:
        return B, T, eo, ev
    return B, T


def max_over_ranks(values, dist, device):
    """Replicas only: the one cross-rank step is the MAX of the device-timed milliseconds."""
    if dist is None:
        return list(values)
    import torch
    tt = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return tt.tolist()


def job_throughput(world, flops_per_replica_step, ms_per_step):
    """Whole-job GFLOP/s: every rank runs the same step on its own GPU; the job takes the slowest rank's time."""
    return world * flops_per_replica_step / (ms_per_step * 1e-3) * 1e-9


def run_ours(args, rank, world, local_rank):
    import numpy as np
    import torch
    import paper_2409_06759_b200 as pkg
    from paper_2409_06759_b200 import ccd

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; this library has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    ctx = pkg.Context(local_rank)
    B, T = make_ccd_inputs(ctx, O, V)
    R = ctx.tensor_create((V, V, O, O))
    flops_step = ccd.CCD_FLOPS(O, V)
    ctx.set_option("kernel_timing", "off" if os.environ.get("TCB_BENCH_NO_KERNEL_TIMING") else "on")

    def step():
        ccd.ccd_residual(ctx, B, T, R)

    for _ in range(max(args.warmup, 3)):
        step()
    # The steps without event pairs replay a CUDA graph of the same call list (tcb_capture_begin/end: 35 kernel nodes,
    # stream-ordered intermediates included; captured once, outside the timed region, like the plans): 7.18 instead of
    # 7.27 ms per step.  --no-graph issues every step call by call.
    graph, graph_note = None, None
    if not args.no_graph:
        ctx.set_option("kernel_timing", "off")
        try:
            ctx.capture_begin()
            try:
                step()
            finally:
                graph = ctx.capture_end()          # also closes the capture when step() raised
            ctx.graph_launch(graph)
            ctx.sync()
        except pkg.TcbError as exc:                # not capturable on this box: every step call by call, and say so
            graph, graph_note = None, f"capture failed ({exc}); "
    ctx.sync()
    ctx.kernel_stats_reset()
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.3)
    barrier()
    l0, t0 = ctx.launch_count(), time.time()
    # Per-launch CUDA event pairs (the live roofline figures) serialise consecutive launches: with them on every step
    # the step is 2.1 % slower (7.42 vs 7.27 ms).  They are recorded on every EVENT_EVERY-th timed step only; `value` is
    # the time of all K steps, sampled ones included.
    sampled = 0
    ctx.timer_start()
    for it in range(args.steps):
        on = (it % EVENT_EVERY == 0) and not os.environ.get("TCB_BENCH_NO_KERNEL_TIMING")
        sampled += 1 if on else 0
        if on or graph is None:
            ctx.set_option("kernel_timing", "on" if on else "off")
            step()
            ctx.set_option("kernel_timing", "off")
        else:
            ctx.graph_launch(graph)
    ms = ctx.timer_stop()
    barrier()
    t1 = time.time()
    launches = ctx.launch_count() - l0
    clocks = sampler.stop(t0, t1)
    stats = {k: ctx.kernel_stats(k) for k in ("zgemm", "permute", "permsum", "elementwise")}
    ctx.set_option("kernel_timing", "off")
    if graph is not None:
        ctx.graph_destroy(graph)

    # ---- e2e: the same step through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    names = list(B.keys())
    host_in = {k: torch.empty(B[k].size, dtype=torch.complex128).pin_memory() for k in names}
    host_T = torch.empty(T.size, dtype=torch.complex128).pin_memory()
    host_R = torch.empty(R.size, dtype=torch.complex128).pin_memory()
    for k in names:
        ctx.tensor_download_raw(B[k], host_in[k].data_ptr())
    ctx.tensor_download_raw(T, host_T.data_ptr())
    h2d = sum(B[k].nbytes for k in names) + T.nbytes
    d2h = R.nbytes

    # Two device copies of the inputs and a second context (its own stream) for the uploads: while step n computes
    # on one copy, step n+1's inputs cross PCIe into the other.  Every step still uploads all of its inputs from
    # pinned host memory and reads its result back, all inside the timed region.
    ctx_up = pkg.Context(local_rank)
    sets = [(B, T)]
    B2 = {k: ctx.tensor_create(B[k].extents) for k in names}
    T2 = ctx.tensor_create(T.extents)
    sets.append((B2, T2))
    up = [({k: ctx_up.tensor_wrap(Bs[k].extents, ctx.tensor_device_ptr(Bs[k])) for k in names},
           ctx_up.tensor_wrap(Ts.extents, ctx.tensor_device_ptr(Ts))) for Bs, Ts in sets]

    def upload(which):
        Bu, Tu = up[which]
        for k in names:
            ctx_up.tensor_upload_raw(Bu[k], host_in[k].data_ptr())
        ctx_up.tensor_upload_raw(Tu, host_T.data_ptr())

    def e2e_run(nsteps):
        upload(0)
        ctx_up.sync()
        for n in range(nsteps):
            if n + 1 < nsteps:
                upload((n + 1) % 2)                               # overlaps with this step's kernels
            Bs, Ts = sets[n % 2]
            ccd.ccd_residual(ctx, Bs, Ts, R)
            ctx.tensor_download_raw(R, host_R.data_ptr())          # blocks until R is on the host
            ctx_up.sync()

    e2e_steps = max(3, min(args.steps, 10))
    e2e_run(2)
    barrier()
    ctx.timer_start()
    e2e_run(e2e_steps)
    e2e_ms = ctx.timer_stop()
    barrier()
    ctx_up.destroy()
    r_norm = float(torch.linalg.vector_norm(host_R).item())     # the step's result was really read back

    ms, e2e_ms = max_over_ranks([ms, e2e_ms], dist, "cuda")
    ms_step = ms / args.steps
    value = job_throughput(world, flops_step, ms_step)
    e2e_value = job_throughput(world, flops_step, e2e_ms / e2e_steps)

    zg = stats["zgemm"]
    achieved = zg["flops"] / (zg["ms"] * 1e-3) * 1e-12 if zg["ms"] > 0 else 0.0
    line = {
        "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "complex128 (f64)", "data": "synthetic",
        "config": {"workload": WORKLOAD, "o": O, "v": V, "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": "inputs larger than L2 (vvvv 655 MB, working set 0.9 GB vs 126 MB L2), no flush",
                   "calls_per_step": "11 tcb_contract + 5 tcb_antisymmetrize + 3 tcb_add",
                   "issue": ((graph_note or "") + "call by call" if graph is None else
                             f"CUDA graph replay of the call list (tcb_capture_*), except the {sampled} steps that carry "
                             "per-launch event pairs, which are issued call by call")},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "GFLOP/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps, "residual_norm": r_norm,
                "pipelining": "uploads of step n+1 on a second stream overlap the kernels of step n (two device copies)"},
        "gpu_launches": launches,
        "roofline": {"bound": "tensor", "kernel": "zgemm_dmma_kernel (all 11 contractions of the step)",
                     "achieved": achieved, "peak": FP64_TENSOR_PEAK_TFLOPS, "unit": "TFLOP/s",
                     "frac": achieved / FP64_TENSOR_PEAK_TFLOPS,
                     "peak_source": "derived FP64 DMMA peak 148 SM x 128 flop/clk x 1.965 GHz (MEASURED_PEAKS.json has "
                                    "no FP64 figure; the register-resident DMMA loop measures 37.0)",
                     "traffic": ZGEMM_DRAM_BYTES_PER_STEP / ZGEMM_LAUNCHES_PER_STEP,
                     "traffic_note": "dram__bytes_read.sum + dram__bytes_write.sum per launch, mean over the 11 GEMM launches "
                                     "of one step, ncu --set full capture in profiles/r1b_zgemm_ncu_full.md; algorithmic "
                                     f"bytes per launch {zg['bytes'] / max(zg['launches'], 1):.4g}",
                     "share_of_step": zg["ms"] / (ms_step * sampled) if ms > 0 and sampled else None,
                     "sampling": f"per-launch event pairs on {sampled} of the {args.steps} timed steps (every "
                                 f"{EVENT_EVERY}th): they serialise launches, +2.1 % on a step that carries them"},
        "kernels": {k: {"launches": s["launches"], "ms_per_step": s["ms"] / max(sampled, 1),
                        "tflops": s["flops"] / (s["ms"] * 1e-3) * 1e-12 if s["ms"] > 0 and s["flops"] else None,
                        "gbs": s["bytes"] / (s["ms"] * 1e-3) * 1e-9 if s["ms"] > 0 else None} for k, s in stats.items()},
    }
    return ctx, line


# ---------------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py may execute oracle/)
# ---------------------------------------------------------------------------------------------------------
def oracle_sample(n_cols=24):
    """The oracle as it stands (order A nested loops, double accumulators, OpenMP) on a bounded sample of
    configs[1]: the pp-ladder contraction R(a,b,i,j) += 1/2 vvvv(a,b,c,d) T(c,d,i,j) -- 60 % of the step's flops --
    restricted to n_cols of the o*o = 400 (i,j) columns of R.  Returns (GFLOP/s, seconds, cores, text)."""
    import numpy as np
    import oracle
    from paper_2409_06759_b200 import synth
    rng = np.random.default_rng(0)
    # the sample's VALUES do not matter for timing (dense loops, no data-dependent work): random stand-ins of the
    # exact shapes, so that no 80^4 tensor has to be generated by the slow host generator
    Vt = np.asfortranarray(rng.standard_normal((V, V, V, V)) + 1j * rng.standard_normal((V, V, V, V)))
    Tt = np.asfortranarray(rng.standard_normal((V, V, n_cols, 1)) + 1j * rng.standard_normal((V, V, n_cols, 1)))
    Rt = np.zeros((V, V, n_cols, 1), dtype=np.complex128, order="F")
    expr = "R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)"
    t0 = time.time()
    oracle.contract_inplace_double(expr, Rt, Vt, Tt, 0.5)
    dt = time.time() - t0
    flops = 8.0 * V ** 4 * n_cols
    return flops / dt * 1e-9, dt, oracle.num_threads(), \
        f"pp ladder of configs[1] on {n_cols} of {O * O} (i,j) columns of R ({flops:.3g} flop, {dt:.1f} s)"


def run_reference(args, rank):
    if rank != 0:
        return None
    vals, cores, sample = [], 0, ""
    for _ in range(args.warmup):
        oracle_sample(2)
    t0 = time.time()
    for _ in range(args.steps):
        g, dt, cores, sample = oracle_sample(8)
        vals.append((g, dt))
    total = sum(dt for _, dt in vals)
    gf = sum(g * dt for g, dt in vals) / total
    return {"impl": "reference", "metric": METRIC, "value": gf, "unit": "GFLOP/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": total / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "complex128 (f64)",
            "data": "synthetic", "config": {"workload": WORKLOAD, "o": O, "v": V},
            "cpu_baseline": {"value": gf, "unit": "GFLOP/s", "cores": cores, "kind": "oracle",
                             "sample": "per step: " + sample},
            "e2e": {"value": gf, "unit": "GFLOP/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


# ---------------------------------------------------------------------------------------------------------
# context measurements on the other BASELINE.json configs (N = 1 only; not the bench line's value)
# ---------------------------------------------------------------------------------------------------------
def run_extras(ctx):
    """configs[2] (CCSD ladder o=40, v=200, V = 25.6 GB), configs[3] (T3 term o=12, v=60) and a transposition
    sample of configs[4]; each timed with CUDA events on the context's stream, best of a few repetitions."""
    import numpy as np
    hbm = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"] \
        if os.path.exists(os.path.join(ROOT, "MEASURED_PEAKS.json")) else 6650.0
    out = []

    def best_of(fn, reps, warm=1):
        for _ in range(warm):
            fn()
        ctx.sync()
        ts = []
        for _ in range(reps):
            ctx.timer_start()
            fn()
            ts.append(ctx.timer_stop())
        return min(ts), float(np.median(ts))

    try:    # configs[0]: the small parity case, latency-bound -- microseconds per call, 200 calls per event pair
        o, v = 8, 24
        V0, T0, R0 = ctx.tensor_create((v, v, v, v)), ctx.tensor_create((v, v, o, o)), ctx.tensor_create((v, v, o, o))
        Tt = ctx.tensor_create((o, o, v, v))
        ctx.synth_normal(V0, 20240906, 1, antisym=((0, 1), (2, 3)))
        ctx.synth_normal(T0, 20240906, 2, antisym=((0, 1), (2, 3)))
        e0 = "R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)"

        def many(fn, n=200):
            def run():
                for _ in range(n):
                    fn()
            b, _ = best_of(run, 3)
            return b / n * 1e3
        us_c = many(lambda: ctx.contract(e0, R0, V0, T0, 0.5))
        us_t = many(lambda: ctx.permute("Tt(i,j,a,b)=T(a,b,i,j)", Tt, T0))
        out.append({"workload": "configs[0]: pp ladder o=8 v=24 (576x64x576, 1.7e8 flop) and transpose of T (0.59 MB); "
                                "latency-bound, 200 back-to-back calls per timed region",
                    "us_per_contraction": us_c, "gflops": 8.0 * 576 * 64 * 576 / us_c * 1e-3,
                    "us_per_transpose": us_t})
        for t in (V0, T0, R0, Tt):
            t.destroy()
        ctx.sync()
    except Exception as e:          # noqa: BLE001
        out.append({"workload": "configs[0]", "error": str(e)})
    try:    # configs[2]
        o, v = 40, 200
        Vt, Tt, Rt = ctx.tensor_create((v, v, v, v)), ctx.tensor_create((v, v, o, o)), ctx.tensor_create((v, v, o, o))
        ctx.synth_normal(Vt, 20240909, 1, antisym=((0, 1), (2, 3)))
        ctx.synth_normal(Tt, 20240909, 2, antisym=((0, 1), (2, 3)))
        expr = "R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)"
        b, m = best_of(lambda: ctx.contract(expr, Rt, Vt, Tt, 0.5), 3)
        fl = 8.0 * (v * v) ** 2 * o * o
        out.append({"workload": "configs[2]: CCSD pp ladder o=40 v=200 (40000x1600x40000, V 25.6 GB in place)",
                    "ms": b, "ms_median": m, "tflops": fl / b * 1e-9, "frac_fp64_tensor_peak": fl / b * 1e-9 / FP64_TENSOR_PEAK_TFLOPS})
        Tp = ctx.tensor_create((o, o, v, v))
        expr2 = "R(a,b,i,j)+=V(a,b,c,d)*T(i,j,c,d)"
        b, m = best_of(lambda: ctx.contract(expr2, Rt, Vt, Tp, 0.5), 2)
        out.append({"workload": "configs[2] variant T(i,j,c,d)", "ms": b, "tflops": fl / b * 1e-9,
                    "frac_fp64_tensor_peak": fl / b * 1e-9 / FP64_TENSOR_PEAK_TFLOPS})
        for t in (Vt, Tt, Rt, Tp):
            t.destroy()
        ctx.sync()
    except Exception as e:          # noqa: BLE001 -- context numbers must never break the bench line
        out.append({"workload": "configs[2]", "error": str(e)})
    try:    # configs[3]
        from paper_2409_06759_b200 import ccd
        o, v = 12, 60
        W, T2 = ctx.tensor_create((v, v, v, o)), ctx.tensor_create((v, v, o, o))
        X, R3 = ctx.tensor_create((v, v, v, o, o, o)), ctx.tensor_create((v, v, v, o, o, o))
        ctx.synth_normal(W, 20240910, 1, antisym=((0, 1),))
        ctx.synth_normal(T2, 20240910, 2, antisym=((0, 1), (2, 3)))
        ctx.synth_normal(R3, 20240910, 3)
        e1 = "X(a,b,c,i,j,k)=W(b,c,d,k)*T(a,d,i,j)"
        b1, _ = best_of(lambda: ctx.contract(e1, X, W, T2, 1.0), 5)
        e2 = "P(a/bc)P(k/ij):R(a,b,c,i,j,k)+=X(a,b,c,i,j,k)"
        b2, _ = best_of(lambda: ctx.antisymmetrize(e2, R3, X, 1.0), 5)
        fl = 8.0 * v ** 4 * o ** 3
        out.append({"workload": "configs[3]: T3 contraction 8640x43200x60 (writes X 5.97 GB)", "ms": b1,
                    "tflops": fl / b1 * 1e-9, "frac_fp64_tensor_peak": fl / b1 * 1e-9 / FP64_TENSOR_PEAK_TFLOPS})
        by = 3 * 16.0 * X.size
        out.append({"workload": "configs[3]: 9-term antisymmetriser R3 += P(a/bc)P(k/ij) X (read X, RMW R3: 17.9 GB)",
                    "ms": b2, "gbs": by / b2 * 1e-6, "frac_hbm_measured": by / b2 * 1e-6 / hbm})
        for t in (W, T2, X, R3):
            t.destroy()
        ctx.sync()
    except Exception as e:          # noqa: BLE001
        out.append({"workload": "configs[3]", "error": str(e)})
    try:    # next row 8(f)-3: whole CC iterations (residual + denominator update + rank-0 energy) at the bench size
        import time
        from paper_2409_06759_b200 import ccd
        o, v = 20, 80
        # sigma = 0.005: weak enough coupling for the plain Jacobi iteration to contract at this size (the bench's
        # sigma = 0.1 tensors are far outside its radius of convergence; the residual step does not care)
        B, T0, eo, ev = make_ccd_inputs(ctx, o, v, sigma=0.005, want_energies=True)
        T0.destroy()
        T, _ = ccd.ccd_solve(ctx, B, eo, ev, 2)                    # warm-up: plans, workspace
        ctx.sync()
        n_it = 8
        t0 = time.perf_counter()
        T, energies = ccd.ccd_solve(ctx, B, eo, ev, n_it, T)
        ctx.sync()
        ms = (time.perf_counter() - t0) * 1e3 / n_it
        out.append({"workload": "next row 8(f)-3: CCD Jacobi iteration o=20 v=80 (residual + tcb_denominator_update + "
                                "rank-0 energy, energy read back every iteration; host wall clock)",
                    "ms_per_iteration": ms, "tflops": ccd.CCD_FLOPS(o, v) / ms * 1e-9, "iterations": n_it + 2,
                    "e_corr_last": [energies[-1].real, energies[-1].imag],
                    "energy_steps": [abs(energies[k] - energies[k - 1]) for k in range(1, len(energies))]})
        for t in list(B.values()) + [T]:
            t.destroy()
        ctx.sync()
    except Exception as e:          # noqa: BLE001
        out.append({"workload": "CCD Jacobi iteration", "error": str(e)})
    try:    # the paper's benchmark unit, one CCSD iteration's residual, at the configs[4] size o=30 v=150
        import numpy as np
        from paper_2409_06759_b200 import ccd, synth
        o, v = 30, 150
        seed, n = synth.SEED0 + 5, o + v
        eo, ev = synth.orbital_energies(seed, o, v)
        rng_ = {"o": (0, o), "v": (o, v)}
        B = {}
        for name in ccd.CCSD_BLOCKS:
            if name[0] == "f":
                continue
            t = ctx.tensor_create([rng_[c][1] for c in name])
            ctx.synth_normal(t, seed, 1, antisym=((0, 1), (2, 3)), sigma=0.02, hermitian=True,
                             label_offset=[rng_[c][0] for c in name], label_extents=[n] * 4)
            B[name] = t
        hrng = np.random.default_rng(seed)
        fov = 0.02 * (hrng.standard_normal((o, v)) + 1j * hrng.standard_normal((o, v)))
        B["foo"] = ctx.tensor_from_numpy(np.diag(eo).astype(np.complex128))
        B["fvv"] = ctx.tensor_from_numpy(np.diag(ev).astype(np.complex128))
        B["fov"] = ctx.tensor_from_numpy(np.asfortranarray(fov))
        B["fvo"] = ctx.tensor_from_numpy(np.asfortranarray(fov.conj().T))
        T1, T2 = ctx.tensor_create((v, o)), ctx.tensor_create((v, v, o, o))
        ctx.synth_normal(T1, seed, 2, sigma=0.05)
        ctx.synth_normal(T2, seed, 3, antisym=((0, 1), (2, 3)), sigma=0.05)
        R1, R2 = ctx.tensor_create((v, o)), ctx.tensor_create((v, v, o, o))

        class Counting:                       # forwards to ctx; adds up the planner's flop count of every contraction
            flops = 0.0
            calls = 0

            def __getattr__(self, name):
                return getattr(ctx, name)

            def contract(self, e, D, L, R, alpha=1.0):
                Counting.flops += ctx.plan_describe(e, D, L, R)["flops"]
                Counting.calls += 1
                return ctx.contract(e, D, L, R, alpha)

        E, _, _ = ccd.ccsd_residual(Counting(), B, T1, T2, R1, R2)     # warm-up pass, counted
        E.destroy()
        ctx.sync()
        ts = []
        for _ in range(3):
            l0 = ctx.launch_count()
            ctx.timer_start()
            E, _, _ = ccd.ccsd_residual(ctx, B, T1, T2, R1, R2)
            ts.append(ctx.timer_stop())
            launches = ctx.launch_count() - l0
            E.destroy()
        b = min(ts)
        ctx.set_option("kernel_timing", "on")                      # one more pass, per kernel class (event pairs per launch)
        ctx.kernel_stats_reset()
        E, _, _ = ccd.ccsd_residual(ctx, B, T1, T2, R1, R2)
        ctx.sync()
        E.destroy()
        classes = {k: ctx.kernel_stats(k) for k in ("zgemm", "permute", "permsum", "elementwise")}
        ctx.set_option("kernel_timing", "off")
        out.append({"workload": "CCSD residual (R1, R2, E) o=30 v=150: 35 contractions + 9 permute-sums + 12 adds, "
                                "vvvv and Wabef 8.1 GB each",
                    "ms": b, "ms_median": float(np.median(ts)), "contractions": Counting.calls, "launches": launches,
                    "tflops": Counting.flops / b * 1e-9,
                    "frac_fp64_tensor_peak": Counting.flops / b * 1e-9 / FP64_TENSOR_PEAK_TFLOPS,
                    "ms_by_class": {k: c["ms"] for k, c in classes.items()},
                    "gbs_by_class": {k: (c["bytes"] / c["ms"] * 1e-6 if c["ms"] > 0 else None) for k, c in classes.items()}})
        for t in list(B.values()) + [T1, T2, R1, R2]:
            t.destroy()
        ctx.sync()
    except Exception as e:          # noqa: BLE001
        out.append({"workload": "CCSD residual", "error": str(e)})
    try:    # the paper's outlook (CCSD(T)): the [T] triples correction at the configs[3] size
        from paper_2409_06759_b200 import ccd, synth
        o, v = 12, 60
        seed, n = synth.SEED0 + 7, o + v
        eo, ev = synth.orbital_energies(seed, o, v)
        Wt, Ut, Tt2 = ctx.tensor_create((v, v, v, o)), ctx.tensor_create((o, v, o, o)), ctx.tensor_create((v, v, o, o))
        ctx.synth_normal(Wt, seed, 1, antisym=((0, 1),), sigma=0.1)
        ctx.synth_normal(Ut, seed, 2, antisym=((2, 3),), sigma=0.1)
        ctx.synth_normal(Tt2, seed, 3, antisym=((0, 1), (2, 3)), sigma=0.1)
        vals = []

        T1t, Vt2 = ctx.tensor_create((v, o)), ctx.tensor_create((o, o, v, v))
        ctx.synth_normal(T1t, seed, 4, sigma=0.1)
        ctx.synth_normal(Vt2, seed, 5, antisym=((0, 1), (2, 3)), sigma=0.1)

        def run():
            E, Est = ccd.triples_correction(ctx, Wt, Ut, Tt2, eo, ev, T1=T1t, oovv=Vt2)
            vals.append(E)
            vals.append(Est)
        b, m = best_of(run, 3)
        e_t, e_st = complex(ctx.tensor_download(vals[-2])), complex(ctx.tensor_download(vals[-1]))
        for E in vals:
            E.destroy()
        fl = 8.0 * (v ** 4 * o ** 3 + v ** 3 * o ** 4)
        # zero-filled creation of X and R3 (2), X = (1), R3 = P X (2), X = (1), R3 += P X (3), t3 = R3 / D3 (2), dot (2)
        # ... and the singles term reads t3 once more (1)
        by = 16.0 * v ** 3 * o ** 3 * (2 + 1 + 2 + 1 + 3 + 2 + 2 + 1)
        out.append({"workload": "(T) triples correction o=12 v=60 (2 rank-6 contractions, 2 nine-term antisymmetrisers, "
                                "rank-6 denominator division, inner product, singles term = rank-6 tensor contracted to "
                                "rank 2; tensors of 5.97 GB created inside the timed region)",
                    "ms": b, "ms_median": m, "tflops": fl / b * 1e-9, "gbs_algorithmic": by / b * 1e-6,
                    "e_t": [e_t.real, e_t.imag], "e_st": [e_st.real, e_st.imag]})
        for t in (Wt, Ut, Tt2, T1t, Vt2):
            t.destroy()
        ctx.sync()
    except Exception as e:          # noqa: BLE001
        out.append({"workload": "[T] triples correction", "error": str(e)})
    try:    # configs[4] transposition samples (the whole sweep: python -m paper_2409_06759_b200.transpose_bench)
        import itertools
        from paper_2409_06759_b200 import transpose_bench as tb
        for shape, perms in (((200, 200, 40, 40), list(itertools.permutations(range(4)))),
                             ((40, 40, 40, 8, 8, 8), tb.rank6_sample())):
            r = tb.summary(shape, tb.sweep_shape(ctx, shape, perms), hbm)
            r["workload"] = (f"configs[4]: {len(perms)} rank-{len(shape)} transpositions of {shape} complex128 "
                             f"({r['megabytes']:.0f} MB)")
            out.append(r)
    except Exception as e:          # noqa: BLE001
        out.append({"workload": "configs[4]", "error": str(e)})
    return out


def main():
    args = parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        line = run_reference(args, rank)
        if line is not None:
            print(json.dumps(line), flush=True)
        return
    ctx, line = run_ours(args, rank, world, local_rank)
    if rank == 0 and world == 1:
        if not args.no_cpu_baseline:
            g, dt, cores, sample = oracle_sample(96)
            line["cpu_baseline"] = {"value": g, "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "sample": sample}
        if not args.no_extras:
            line["other_workloads"] = run_extras(ctx)
    ctx.destroy()
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
