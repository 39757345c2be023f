#!/usr/bin/env python
"""bench.py -- one JSON line for the driver (contract in DESIGN.md "Measurement").

A step = BASELINE.json configs[2], the largest single-GPU configuration: the CCSD particle-particle ladder
    R(a,b,i,j) += 1/2 sum_cd V(a,b,c,d) T(c,d,i,j),   complex128, o=40, v=200   (40000 x 1600 x 40000; V = 25.6 GB)
issued as ONE tcb_contract call through the C ABI ("timed as a single contraction including operand permutations": the
planner finds none to do -- V and T are read in place by TMA).  metric = complex-FP64 contraction throughput, GFLOP/s with
8 real flop per complex multiply-add; the GB/s half of BASELINE.json's metric (transposition) is `roofline_hbm`.

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

METRIC = "complex-FP64 contraction GFLOP/s (CCSD pp ladder, 8 flop per complex MAC)"
O, V = 40, 200                                  # BASELINE.json configs[2]
EXPR = "R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)"
FLOPS_STEP = 8.0 * (V * V) ** 2 * (O * O)
WORKLOAD = (f"configs[2]: CCSD pp ladder R(a,b,i,j) += 1/2 V(a,b,c,d) T(c,d,i,j), complex128, o={O}, v={V} "
            f"({V * V} x {O * O} x {V * V}, V 25.6 GB read in place)")
# nominal FP64 tensor peak derived from unit counts: SMs x 4 sub-partitions x one DMMA.8x8x4 (512 flop) per 16
# cycles x max SM clock = 148 x 128 x 1.965 GHz.  bench.py also MEASURES the register-resident DMMA loop in the same process
# (tcb_measure_fp64_tensor_peak) and prints it beside this figure.
FP64_TENSOR_PEAK_TFLOPS = 148 * 128 * 1.965e9 * 1e-12
# DRAM traffic per launch of the dominant kernels, from the committed ncu --set full captures (bench.py never runs under a
# profiler): profiles/r2_dram_traffic.json.txt, written from the .ncu-rep files named inside it
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "r2_dram_traffic.json.txt")


def committed_traffic(key):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of kernel `key` from the committed profile, or None"""
    try:
        with open(TRAFFIC_FILE) as f:
            return json.load(f)[key]
    except Exception:          # noqa: BLE001 -- no capture committed for this kernel
        return None


def hbm_peak():
    """(GB/s, source): the driver-measured copy bandwidth, else the profiling guide's fallback"""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (driver-measured copy bandwidth)"
        except Exception:      # noqa: BLE001
            pass
    return 6650.0, "fallback: B200_PROFILING.md measured copy bandwidth (MEASURED_PEAKS.json absent)"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-extras", action="store_true", help="skip the configs[2..4] context measurements")
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
                                          "--format=csv,noheader,nounits", "-lms", "10"],
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


def e2e_ranks_at_once(world, host_ram_bytes, pinned_bytes_per_rank):
    """How many replicas measure their end-to-end step at the same time: all of them when 60 % of the host's memory holds
    every rank's pinned buffers, otherwise as many as fit (at least one); the others wait their turn."""
    return max(1, min(world, int(0.6 * host_ram_bytes // pinned_bytes_per_rank)))


def job_throughput(world, flops_per_replica_step, ms_per_step):
    """Whole-job GFLOP/s: every rank runs the same step on its own GPU; the job takes the slowest rank's time."""
    return world * flops_per_replica_step / (ms_per_step * 1e-3) * 1e-9


def run_ours(args, rank, world, local_rank):
    import numpy as np
    import torch
    import paper_2409_06759_b200 as pkg
    from paper_2409_06759_b200 import synth

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
    seed, anti = synth.SEED0 + 3, ((0, 1), (2, 3))
    Vt, Tt, Rt = ctx.tensor_create((V, V, V, V), zero=False), ctx.tensor_create((V, V, O, O), zero=False), \
        ctx.tensor_create((V, V, O, O))
    ctx.synth_normal(Vt, seed, 1, antisym=anti)
    ctx.synth_normal(Tt, seed, 2, antisym=anti)
    plan = ctx.plan_describe(EXPR, Rt, Vt, Tt)

    def step():
        ctx.contract(EXPR, Rt, Vt, Tt, 0.5)

    warmup = max(args.warmup, 3)
    for _ in range(warmup):
        step()
    ctx.sync()
    # the roofline denominator, measured in this process: register-resident DMMA.8x8x4 loop on every SM for 0.2 s
    peak_sampler = ClockSampler(local_rank)
    peak_sampler.start()
    time.sleep(0.05)
    tp0 = time.time()
    peak_live = ctx.measure_fp64_tensor_peak(200.0)
    ctx.sync()
    peak_clocks = peak_sampler.stop(tp0, time.time())

    # one kernel launch per step, so the per-launch event pairs (tcb_kernel_stats) serialise nothing: they stay on
    ctx.set_option("kernel_timing", "on")
    ctx.kernel_stats_reset()
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.2)
    barrier()
    l0, t0 = ctx.launch_count(), time.time()
    ctx.timer_start()
    for _ in range(args.steps):
        step()
    ms = ctx.timer_stop()
    barrier()
    t1 = time.time()
    launches = ctx.launch_count() - l0
    clocks = sampler.stop(t0, t1)
    zg = ctx.kernel_stats("zgemm")
    ctx.set_option("kernel_timing", "off")

    # ---- the GB/s half of the metric: the dominant permutation kernel on a configs[4] transposition, same process ------
    hbm, hbm_src = hbm_peak()
    ctx.set_option("kernel_timing", "on")
    tshape = (200, 200, 40, 40)
    Lp, Dp = ctx.tensor_create(tshape, zero=False), ctx.tensor_create((40, 40, 200, 200), zero=False)
    ctx.synth_index_linear(Lp)
    for _ in range(3):
        ctx.permute("D(i,j,a,b)=L(a,b,i,j)", Dp, Lp)
    ctx.kernel_stats_reset()
    for _ in range(20):
        ctx.permute("D(i,j,a,b)=L(a,b,i,j)", Dp, Lp)
    pm = ctx.kernel_stats("permute")
    ctx.set_option("kernel_timing", "off")
    Lp.destroy(); Dp.destroy()
    pm_gbs = pm["bytes"] / (pm["ms"] * 1e-3) * 1e-9 if pm["ms"] > 0 else 0.0

    # ---- e2e: the same step through the C ABI with HOST buffers (pinned), copies inside the timed region ---------------
    # Every step uploads V (25.6 GB), T and R from pinned host memory and reads R back.  Two device copies of V and T and a
    # second context (its own stream) for the uploads: while step n computes on one copy, step n+1's operands cross PCIe
    # into the other.
    h2d, d2h = Vt.nbytes + Tt.nbytes + Rt.nbytes, Rt.nbytes
    e2e_steps = max(3, min(args.steps, 20))
    # N replicas on one host each pin 27.6 GB: when the host cannot hold all of them at once the ranks take turns in groups
    # (PCIe links are per GPU; what the turns leave out is contention for host memory bandwidth -- said in the JSON line)
    host_ram = os.sysconf("SC_PAGE_SIZE") * os.sysconf("SC_PHYS_PAGES")
    group = e2e_ranks_at_once(world, host_ram, h2d + d2h + 2 * Rt.nbytes)

    def e2e_measure():
        host_V = torch.empty(Vt.size, dtype=torch.complex128).pin_memory()
        host_T = torch.empty(Tt.size, dtype=torch.complex128).pin_memory()
        host_R = torch.empty(Rt.size, dtype=torch.complex128).pin_memory()
        host_Rin = torch.zeros(Rt.size, dtype=torch.complex128).pin_memory()
        ctx.tensor_download_raw(Vt, host_V.data_ptr())
        ctx.tensor_download_raw(Tt, host_T.data_ptr())
        ctx_up = pkg.Context(local_rank)
        V2, T2 = ctx.tensor_create(Vt.extents, zero=False), ctx.tensor_create(Tt.extents, zero=False)
        sets = [(Vt, Tt), (V2, T2)]
        up = [(ctx_up.tensor_wrap(a.extents, ctx.tensor_device_ptr(a)), ctx_up.tensor_wrap(b.extents, ctx.tensor_device_ptr(b)))
              for a, b in sets]

        def upload(which):
            ctx_up.tensor_upload_raw(up[which][0], host_V.data_ptr())
            ctx_up.tensor_upload_raw(up[which][1], host_T.data_ptr())

        def e2e_run(nsteps):
            upload(0)
            ctx_up.sync()
            for n in range(nsteps):
                Vs, Ts = sets[n % 2]
                ctx.tensor_upload_raw(Rt, host_Rin.data_ptr())         # R_in travels too ('+=' reads it)
                ctx.contract(EXPR, Rt, Vs, Ts, 0.5)
                # the next step's operands are queued on the host->device copy engine AFTER this step's R_in (the engine
                # serves its queue in order: queued before it, the 26.6 GB would hold the kernel back by 0.5 s) and cross
                # PCIe while the kernel runs
                if n + 1 < nsteps:
                    upload((n + 1) % 2)
                ctx.tensor_download_raw(Rt, host_R.data_ptr())         # blocks until R is on the host
                ctx_up.sync()

        e2e_run(2)
        ctx.sync()
        ctx.timer_start()
        e2e_run(e2e_steps)
        t_ms = ctx.timer_stop()
        ctx_up.destroy()
        norm = float(torch.linalg.vector_norm(host_R).item())     # the step's result was really read back
        V2.destroy(); T2.destroy()
        return t_ms, norm

    e2e_ms, r_norm = 0.0, 0.0
    for g0 in range(0, world, group):
        barrier()
        if g0 <= rank < g0 + group:
            e2e_ms, r_norm = e2e_measure()
        barrier()

    ms, e2e_ms = max_over_ranks([ms, e2e_ms], dist, "cuda")
    ms_step = ms / args.steps
    value = job_throughput(world, FLOPS_STEP, ms_step)
    e2e_value = job_throughput(world, FLOPS_STEP, e2e_ms / e2e_steps)

    achieved = zg["flops"] / (zg["ms"] * 1e-3) * 1e-12 if zg["ms"] > 0 else 0.0
    alg_bytes = zg["bytes"] / max(zg["launches"], 1)
    line = {
        "metric": METRIC, "value": value, "unit": "GFLOP/s", "n_gpus": world, "steps": args.steps,
        "warmup": warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "complex128 (f64)", "data": "synthetic",
        "config": {"workload": WORKLOAD, "o": O, "v": V, "parallelism": "replicas only" if world > 1 else "1 gpu",
                   "l2": "inputs larger than L2 (V 25.6 GB, T and R 1.02 GB each vs 126 MB L2), no flush",
                   "calls_per_step": "1 tcb_contract (2 launches: GEMM + stream-K fix-up)",
                   "plan": {k: plan[k] for k in ("M", "N", "K", "feed_A", "feed_B", "A_layout", "B_layout", "splits", "epilogue",
                                                "complex_product")}},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": "GFLOP/s", "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": e2e_ms / e2e_steps, "steps": e2e_steps, "residual_norm": r_norm,
                "pipelining": "V and T of step n+1 cross PCIe on a second stream while step n computes (two device copies)",
                "ranks_at_once": group},
        "gpu_launches": launches,
        "roofline": {"bound": "tensor", "kernel": "zgemm_dmma_kernel + zgemm_fixup_kernel (GEMM with the fused permute-accumulate "
                                                  "epilogue; the fix-up sums the remainder tiles cut along K)",
                     "achieved": achieved, "peak": FP64_TENSOR_PEAK_TFLOPS, "unit": "TFLOP/s",
                     "frac": achieved / FP64_TENSOR_PEAK_TFLOPS,
                     # SURVEY 8(d) counts 8 real flop per complex multiply-add ("achieved", "frac").  With complex_product = 3m
                     # the kernel ISSUES three real DMMA products per complex product instead of four (6 flop per complex
                     # multiply-add on the tensor pipe): frac may exceed 1 against the real-arithmetic peak; frac_issued
                     # is what the pipe does.
                     "complex_product": plan.get("complex_product"),
                     "frac_note": "achieved and frac count SURVEY 8(d)'s 8 real flop per complex multiply-add; with complex_product = 3m "
                                  "the kernel forms a complex product from 3 real tensor-core products instead of 4 (6 flop issued per "
                                  "complex multiply-add), so frac > 1 is the algorithmic gain over the real-arithmetic peak and "
                                  "frac_issued (= 0.75 frac) is what the tensor pipe executes; ncu: profiles/r2_gemm_3m.md",
                     "issued_tensor_flops_per_launch": zg["flops"] / max(zg["launches"], 1) * (0.75 if plan.get("complex_product") == "3m" else 1.0),
                     "frac_issued": achieved / FP64_TENSOR_PEAK_TFLOPS * (0.75 if plan.get("complex_product") == "3m" else 1.0),
                     "peak_source": "derived FP64 DMMA peak 148 SM x 128 flop/clk x 1.965 GHz (MEASURED_PEAKS.json has no FP64 "
                                    "figure); peak_measured_live is the register-resident DMMA loop run in this process",
                     "peak_measured_live": peak_live, "peak_measured_clocks": peak_clocks,
                     "frac_of_measured_live": achieved / peak_live if peak_live else None,
                     "algorithmic_flops_per_launch": zg["flops"] / max(zg["launches"], 1),
                     "algorithmic_bytes_per_launch": alg_bytes,
                     "avg_launch_ms": zg["ms"] / max(zg["launches"], 1), "launches_timed": zg["launches"],
                     "traffic": committed_traffic("zgemm_configs2"),
                     "traffic_note": "dram__bytes_read.sum + dram__bytes_write.sum of this launch, read from the committed "
                                     "ncu --set full summary profiles/r2_dram_traffic.json.txt (null: no capture committed)",
                     "share_of_step": zg["ms"] / ms if ms > 0 else None},
        "roofline_hbm": {"bound": "hbm", "kernel": "permute_kernel: configs[4] transposition D(i,j,a,b) = L(a,b,i,j) of a "
                                                   "(200,200,40,40) complex128 tensor (1.02 GB), 20 launches",
                         "achieved": pm_gbs, "peak": hbm, "unit": "GB/s", "frac": pm_gbs / hbm, "peak_source": hbm_src,
                         "algorithmic_bytes_per_launch": pm["bytes"] / max(pm["launches"], 1),
                         "avg_launch_ms": pm["ms"] / max(pm["launches"], 1),
                         "traffic": committed_traffic("permute_1gb")},
    }
    return ctx, (Vt, Tt, Rt), line


# ---------------------------------------------------------------------------------------------------------
# CPU oracle legs (the only places bench.py may execute oracle/)
# ---------------------------------------------------------------------------------------------------------
def oracle_sample(n_rows=80, t_cache={}):
    """The oracle as it stands (order A nested loops, double accumulators, OpenMP) on a bounded sample of configs[2]:
    the same contraction restricted to n_rows of the v*v = 40 000 (a,b) rows of R (all 1 600 columns, all of K).
    Returns (GFLOP/s, seconds, cores, text)."""
    import numpy as np
    import oracle
    rng = np.random.default_rng(0)
    # the sample's VALUES do not matter for timing (dense loops, no data-dependent work): random stand-ins of the exact
    # shapes, so that no 200^4 tensor has to be generated by the slow host generator
    if "T" not in t_cache:
        Tt = np.empty((V, V, O, O), dtype=np.complex128, order="F")
        Tt.real = rng.standard_normal(Tt.shape)
        Tt.imag = rng.standard_normal(Tt.shape)
        t_cache["T"] = Tt
    Tt = t_cache["T"]
    Vs = np.asfortranarray(rng.standard_normal((1, n_rows, V, V)) + 1j * rng.standard_normal((1, n_rows, V, V)))
    Rs = np.zeros((1, n_rows, O, O), dtype=np.complex128, order="F")
    t0 = time.time()
    oracle.contract_inplace_double(EXPR, Rs, Vs, Tt, 0.5)
    dt = time.time() - t0
    flops = 8.0 * n_rows * (O * O) * (V * V)
    return flops / dt * 1e-9, dt, oracle.num_threads(), \
        f"configs[2] ladder on {n_rows} of the {V * V} (a,b) rows of R ({flops:.3g} flop, {dt:.1f} s)"


def oracle_check(ctx, tensors, n=8):
    """cpu_baseline leg, part two: the oracle (long-double accumulators) on n^4 sampled outputs of the step the GPU just
    ran -- its operands regenerated on the host by the index-keyed twin of the device generator, nothing read back from
    the device but R -- gives the line's max_norm_err (north_star: <= 1e-11)."""
    import numpy as np
    import oracle
    from paper_2409_06759_b200 import synth
    Vt, Tt, Rt = tensors
    seed, anti = synth.SEED0 + 3, ((0, 1), (2, 3))
    rng = np.random.default_rng(11)
    pa, pb = np.sort(rng.choice(V, n, replace=False)), np.sort(rng.choice(V, n, replace=False))
    pi, pj = np.sort(rng.choice(O, n, replace=False)), np.sort(rng.choice(O, n, replace=False))
    full = np.arange(V)
    hV = synth.tensor(seed, 1, [V] * 4, antisym=anti, sub=[pa, pb, full, full])
    hT = synth.tensor(seed, 2, [V, V, O, O], antisym=anti, sub=[full, full, pi, pj])
    ctx.tensor_fill(Rt, 0.0)
    ctx.contract(EXPR, Rt, Vt, Tt, 0.5)
    got = ctx.tensor_download(Rt)[np.ix_(pa, pb, pi, pj)]
    ref, sn = oracle.contract(EXPR, np.zeros((n, n, n, n)), hV, hT, 0.5)
    nz = sn > 0
    err = float(np.max(np.abs(got - ref)[nz] / sn[nz]))
    exact = bool(np.array_equal(got[~nz], ref[~nz]))
    return {"max_norm_err": err, "outputs_checked": int(got.size), "zero_norm_outputs_exact": exact,
            "tolerance": 1e-11}


def run_reference(args, rank):
    if rank != 0:
        return None
    vals, cores, sample = [], 0, ""
    for _ in range(args.warmup):
        oracle_sample(8)
    for _ in range(args.steps):
        g, dt, cores, sample = oracle_sample(80)
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
    try:    # configs[1]: the whole CCD residual (every S row: contractions, gathered operands, permute-sums, adds), lanes + graph
        from paper_2409_06759_b200 import ccd
        o, v = 20, 80
        B, T = make_ccd_inputs(ctx, o, v)
        R = ctx.tensor_create((v, v, o, o))
        for _ in range(3):
            ccd.ccd_residual(ctx, B, T, R)
        ctx.sync()
        l0 = ctx.launch_count()
        ctx.capture_begin()
        ccd.ccd_residual(ctx, B, T, R)
        g = ctx.capture_end()
        per_step = ctx.launch_count() - l0
        info = ctx.graph_info(g)
        b_graph, m_graph = best_of(lambda: [ctx.graph_launch(g) for _ in range(10)], 5)
        b_eager, _ = best_of(lambda: [ccd.ccd_residual(ctx, B, T, R) for _ in range(10)], 3)
        b_chain, _ = best_of(lambda: [ccd.ccd_residual(ctx, B, T, R, lanes=False) for _ in range(10)], 3)
        ctx.graph_destroy(g)
        ctx.set_option("kernel_timing", "on")
        ctx.kernel_stats_reset()
        ccd.ccd_residual(ctx, B, T, R, lanes=False)
        classes = {k: ctx.kernel_stats(k) for k in ("zgemm", "permute", "permsum", "elementwise")}
        ctx.set_option("kernel_timing", "off")
        fl = ccd.CCD_FLOPS(o, v)
        out.append({"workload": "configs[1]: full spin-orbital CCD residual o=20 v=80 (11 contractions, 5 permute-sums, 3 adds)",
                    "ms_graph_replay": b_graph / 10, "ms_graph_replay_median": m_graph / 10, "ms_call_by_call_lanes": b_eager / 10,
                    "ms_call_by_call_one_lane": b_chain / 10, "tflops": fl / (b_graph / 10) * 1e-9,
                    "frac_fp64_tensor_peak": fl / (b_graph / 10) * 1e-9 / FP64_TENSOR_PEAK_TFLOPS,
                    "launches_per_step": per_step, "graph": info,
                    "one_lane_ms_by_class": {k: c["ms"] for k, c in classes.items()},
                    "one_lane_launches_by_class": {k: c["launches"] for k, c in classes.items()},
                    "one_lane_gbs_by_class": {k: (c["bytes"] / c["ms"] * 1e-6 if c["ms"] > 0 else None) for k, c in classes.items()}})
        cache = {}
        for _ in range(3):
            ccd.ccd_residual(ctx, B, T, R, packed=cache)
        ctx.sync()
        ctx.capture_begin()
        ccd.ccd_residual(ctx, B, T, R, packed=cache)
        g = ctx.capture_end()
        bp_graph, _ = best_of(lambda: [ctx.graph_launch(g) for _ in range(10)], 5)
        bp_eager, _ = best_of(lambda: [ccd.ccd_residual(ctx, B, T, R, packed=cache) for _ in range(10)], 3)
        ctx.graph_destroy(g)
        out.append({"workload": "next row 8(f)-2: the configs[1] CCD residual with the pp ladder on packed storage (<ab||cd> packed "
                                "once: 160 MB instead of 655 MB; ladder at 1/8 of the flops)",
                    "ms_graph_replay": bp_graph / 10, "ms_call_by_call_lanes": bp_eager / 10,
                    "dense_program_ms_graph_replay": b_graph / 10, "speedup_over_dense_program": b_graph / bp_graph})
        for t in list(B.values()) + list(cache.values()) + [T, R]:
            t.destroy()
        ctx.sync()
    except Exception as e:          # noqa: BLE001
        out.append({"workload": "configs[1]", "error": str(e)})
    try:    # configs[2] variants: "including operand permutations" -- T given as T(i,j,c,d), V as V(c,d,a,b), and TTGT forced
        o, v = 40, 200
        Vt, Rt = ctx.tensor_create((v, v, v, v), zero=False), ctx.tensor_create((v, v, o, o))
        ctx.synth_normal(Vt, 20240909, 1, antisym=((0, 1), (2, 3)))
        fl = 8.0 * (v * v) ** 2 * o * o
        for expr, tshape, opt in (("R(a,b,i,j)+=V(a,b,c,d)*T(i,j,c,d)", (o, o, v, v), None),
                                  ("R(a,b,i,j)+=V(c,d,a,b)*T(c,d,i,j)", (v, v, o, o), None),
                                  ("R(a,b,i,j)+=V(a,b,c,d)*T(c,i,d,j)", (v, o, v, o), None),
                                  ("R(a,b,i,j)+=V(a,b,c,d)*T(c,i,d,j)", (v, o, v, o), "permute")):
            Tp = ctx.tensor_create(tshape, zero=False)
            ctx.synth_normal(Tp, 20240909, 2)
            ctx.set_option("operand_loads", opt or "auto")
            plan = ctx.plan_describe(expr, Rt, Vt, Tp)
            b, m = best_of(lambda: ctx.contract(expr, Rt, Vt, Tp, 0.5), 3)
            ctx.set_option("operand_loads", "auto")
            out.append({"workload": f"configs[2] variant {expr}" + (f" [operand_loads={opt}]" if opt else ""), "ms": b,
                        "ms_median": m, "tflops": fl / b * 1e-9, "frac_fp64_tensor_peak": fl / b * 1e-9 / FP64_TENSOR_PEAK_TFLOPS,
                        "feed_A": plan["feed_A"], "feed_B": plan["feed_B"]})
            Tp.destroy()
        Vt.destroy(); Rt.destroy()
        ctx.sync()
    except Exception as e:          # noqa: BLE001 -- context numbers must never break the bench line
        out.append({"workload": "configs[2] variants", "error": str(e)})
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
        out.append({"workload": "CCSD residual (R1, R2, E) o=30 v=150: 34 contractions + 9 permute-sums + 12 adds, "
                                "vvvv and Wabef 8.1 GB each",
                    "ms": b, "ms_median": float(np.median(ts)), "contractions": Counting.calls, "launches": launches,
                    "tflops": Counting.flops / b * 1e-9,
                    "frac_fp64_tensor_peak": Counting.flops / b * 1e-9 / FP64_TENSOR_PEAK_TFLOPS,
                    "ms_by_class": {k: c["ms"] for k, c in classes.items()},
                    "gbs_by_class": {k: (c["bytes"] / c["ms"] * 1e-6 if c["ms"] > 0 else None) for k, c in classes.items()}})
        dense_ms = b
        # the same residual with the pp ladder on packed storage (8(f)-2): W_abef only as Wp(a<b, e<f); the packed integral
        # blocks are built by the warm-up pass and kept, as over the iterations of a solve
        cache = {}
        Counting.flops, Counting.calls = 0.0, 0
        E, _, _ = ccd.ccsd_residual(Counting(), B, T1, T2, R1, R2, cache)
        E.destroy()
        ctx.sync()
        ts = []
        for _ in range(3):
            l0 = ctx.launch_count()
            ctx.timer_start()
            E, _, _ = ccd.ccsd_residual(ctx, B, T1, T2, R1, R2, cache)
            ts.append(ctx.timer_stop())
            launches = ctx.launch_count() - l0
            E.destroy()
        bp = min(ts)
        out.append({"workload": "next row 8(f)-2: the same CCSD residual o=30 v=150 with the pp ladder on packed storage "
                                "(Wp(a<b,e<f) 2.0 GB instead of 8.1 GB; ladder at 1/8, its T1 term at 1/2 of the flops; "
                                "P(ab) = tcb_antisym_pack)",
                    "ms": bp, "ms_median": float(np.median(ts)), "contractions": Counting.calls, "launches": launches,
                    "tflops_executed": Counting.flops / bp * 1e-9,
                    "frac_fp64_tensor_peak": Counting.flops / bp * 1e-9 / FP64_TENSOR_PEAK_TFLOPS,
                    "dense_program_ms": dense_ms, "speedup_over_dense_program": dense_ms / bp})
        for t in list(B.values()) + list(cache.values()) + [T1, T2, R1, R2]:
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
        vals = []

        def run_packed():
            E, Est = ccd.triples_correction_packed(ctx, Wt, Ut, Tt2, eo, ev, T1=T1t, oovv=Vt2)
            vals.append(E)
            vals.append(Est)
        bp, mp = best_of(run_packed, 3)
        p_t, p_st = complex(ctx.tensor_download(vals[-2])), complex(ctx.tensor_download(vals[-1]))
        for E in vals:
            E.destroy()
        out.append({"workload": "(T) triples correction o=12 v=60 on packed storage (8(f)-2): R3p, t3p(a<b<c,i<j<k) of 120 MB, "
                                "two contractions at 1/4 of the dense flops, two tcb_antisym_pack, packed denominators",
                    "ms": bp, "ms_median": mp, "dense_program_ms": b, "speedup_over_dense_program": b / bp,
                    "e_t": [p_t.real, p_t.imag], "e_st": [p_st.real, p_st.imag],
                    "rel_diff_e_t_vs_dense": abs(p_t - e_t) / abs(e_t), "rel_diff_e_st_vs_dense": abs(p_st - e_st) / abs(e_st)})
        for t in (Wt, Ut, Tt2, T1t, Vt2):
            t.destroy()
        ctx.sync()
    except Exception as e:          # noqa: BLE001
        out.append({"workload": "[T] triples correction", "error": str(e)})
    try:    # next row 8(f)-3: one CCSDT residual evaluation (R1, R2, R3) at the configs[3] size o=12 v=60 (T3, X, R3 of 5.97 GB)
        from paper_2409_06759_b200 import ccd
        o, v = 12, 60
        n = o + v
        hh, gg = ctx.tensor_create((n, n), zero=False), ctx.tensor_create((n, n, n, n), zero=False)
        ctx.synth_normal(hh, 20240913, 1, sigma=0.05)
        ctx.synth_normal(gg, 20240913, 2, antisym=((0, 1), (2, 3)), sigma=0.02)
        T1, T2, T3 = ctx.tensor_create((v, o), zero=False), ctx.tensor_create((v, v, o, o), zero=False), \
            ctx.tensor_create((v, v, v, o, o, o), zero=False)
        ctx.synth_normal(T1, 20240913, 3, sigma=0.05)
        ctx.synth_normal(T2, 20240913, 4, antisym=((0, 1), (2, 3)), sigma=0.05)
        ctx.synth_normal(T3, 20240913, 5, sigma=0.01)

        class CountingT:                      # forwards to ctx; adds up the planner's flop count of every contraction
            flops = 0.0
            calls = 0

            def __getattr__(self, name):
                return getattr(ctx, name)

            def contract(self, e, D, L, R, alpha=1.0):
                CountingT.flops += ctx.plan_describe(e, D, L, R)["flops"]
                CountingT.calls += 1
                return ctx.contract(e, D, L, R, alpha)

        Rs = ccd.ccsdt_residual(CountingT(), o, hh, gg, T1, T2, T3)          # warm-up pass, counted
        ctx.sync()
        ts = []
        for _ in range(3):
            l0 = ctx.launch_count()
            ctx.timer_start()
            ccd.ccsdt_residual(ctx, o, hh, gg, T1, T2, T3, *Rs)
            ts.append(ctx.timer_stop())
            launches = ctx.launch_count() - l0
        b = min(ts)
        out.append({"workload": "next row 8(f)-3: CCSDT residual (R1, R2, R3) o=12 v=60: T1 dressing of the integrals, CCD "
                                "program on the dressed blocks, 7 rank-6 contractions into one X, one 36-term antisymmetrisation; "
                                "T3, X, R3 of 5.97 GB each",
                    "ms": b, "ms_median": float(np.median(ts)), "contractions": CountingT.calls, "launches": launches,
                    "tflops": CountingT.flops / b * 1e-9,
                    "frac_fp64_tensor_peak": CountingT.flops / b * 1e-9 / FP64_TENSOR_PEAK_TFLOPS})
        dense_ms = b
        for t in (hh, gg, T1, T2, T3) + tuple(Rs):
            t.destroy()
        ctx.sync()
        # the same residual on packed storage (8(f)-2 applied to 8(f)-3): T3, R3 only as (a<b<c, i<j<k); then a size whose
        # dense T3 (65.5 GB per tensor, four of them live) does not fit one GPU at all
        for (o, v) in ((12, 60), (16, 100)):
            n = o + v
            hh, gg = ctx.tensor_create((n, n), zero=False), ctx.tensor_create((n, n, n, n), zero=False)
            ctx.synth_normal(hh, 20240913, 1, sigma=0.05)
            ctx.synth_normal(gg, 20240913, 2, antisym=((0, 1), (2, 3)), sigma=0.02)
            T1, T2 = ctx.tensor_create((v, o), zero=False), ctx.tensor_create((v, v, o, o), zero=False)
            T3p = ctx.tensor_create((ctx.packed_extent(v, 3), ctx.packed_extent(o, 3)), zero=False)
            ctx.synth_normal(T1, 20240913, 3, sigma=0.05)
            ctx.synth_normal(T2, 20240913, 4, antisym=((0, 1), (2, 3)), sigma=0.05)
            ctx.synth_normal(T3p, 20240913, 5, sigma=0.01)
            CountingT.flops, CountingT.calls = 0.0, 0
            Rs = ccd.ccsdt_residual_packed(CountingT(), o, hh, gg, T1, T2, T3p)
            ctx.sync()
            ts = []
            for _ in range(3):
                l0 = ctx.launch_count()
                ctx.timer_start()
                ccd.ccsdt_residual_packed(ctx, o, hh, gg, T1, T2, T3p, *Rs)
                ts.append(ctx.timer_stop())
                launches = ctx.launch_count() - l0
            b = min(ts)
            row = {"workload": f"next rows 8(f)-2 + 8(f)-3: CCSDT residual on packed storage o={o} v={v}: T3 and R3 only as "
                               f"(a<b<c, i<j<k) tensors of {T3p.nbytes / 1e6:.0f} MB (dense: {16e-9 * v ** 3 * o ** 3:.1f} GB each), "
                               "three packed views of T3, three packed accumulators, tcb_antisym_pack",
                   "ms": b, "ms_median": float(np.median(ts)), "contractions": CountingT.calls, "launches": launches,
                   "tflops_executed": CountingT.flops / b * 1e-9,
                   "frac_fp64_tensor_peak": CountingT.flops / b * 1e-9 / FP64_TENSOR_PEAK_TFLOPS}
            if (o, v) == (12, 60):
                row["dense_program_ms"] = dense_ms
                row["speedup_over_dense_program"] = dense_ms / b
            out.append(row)
            for t in (hh, gg, T1, T2, T3p) + tuple(Rs):
                t.destroy()
            ctx.sync()
    except Exception as e:          # noqa: BLE001
        out.append({"workload": "CCSDT residual", "error": str(e)})
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
    ctx, tensors, line = run_ours(args, rank, world, local_rank)
    if rank == 0 and world == 1:
        if not args.no_cpu_baseline:
            g, dt, cores, sample = oracle_sample(400)
            line["cpu_baseline"] = {"value": g, "unit": "GFLOP/s", "cores": cores, "kind": "oracle", "sample": sample}
            line["cpu_baseline"].update(oracle_check(ctx, tensors))
    for t in tensors:
        t.destroy()
    if rank == 0 and world == 1 and not args.no_extras:
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
