#!/usr/bin/env python
"""bench.py -- measurement harness.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl bkr|reference] [--workload cfg3|cfg4|cfg5|cfg2]
                    [--no-solve] [--sweep] [--microbench] [--ablation]

A "step" is one blockCGrQ iteration (Algorithm 1 l.8-l.12 of arXiv:1710.09745: 2 multi-rhs Dslash, 2 Gram
reductions, the block updates of P, X, Q and the one-CTA small-matrix kernels) on the workload's block of N rhs,
enqueued through the C ABI (bkr_bench_iterations).  Prints ONE JSON line.

  value      effective GB/s of the iteration = ALGORITHMIC bytes of one fused iteration (links twice + 14 block
             passes) / device time per step, inputs resident in HBM;
  e2e        the same metric through bkr_solve_block_host: host buffers in, K iterations, true-residual check,
             host buffer out, all copies inside the timed region;
  roofline   the dominant kernel (multi-rhs Dslash), timed alone with CUDA events on the launching stream;
  kernels    Dslash / Gram / block-update GB/s and roofline fractions at the workload's N;
  solve      block-CG time-to-solution and iterations against N sequential CGs and one batched CG;
  cpu_baseline  the oracle (as it stands) on the host cores, on a bounded sample.

Multi-GPU: the path does not shard: "replicas only" -- every rank runs the same step on its
own GPU with no data-path collective, value = sum over ranks / max time.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

WORKLOADS = {
    # name: (BASELINE.json config, dims, link kind, mass, N)
    "cfg2": ("configs[1]: 16^4, N=8, m=0.05", (16, 16, 16, 16), "perturbed", 0.05, 8),
    "cfg3": ("configs[2]: 32^3x64, N=16, m=0.01", (32, 32, 32, 64), "perturbed", 0.01, 16),
    "cfg4": ("configs[3]: 48^3x96, N=32, m=0.005", (48, 48, 48, 96), "perturbed", 0.005, 32),
    "cfg5": ("configs[4]: 32^4 kernel sweep, N=16", (32, 32, 32, 32), "random", 0.05, 16),
}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# ---------------------------------------------------------------- algorithmic bytes / flops

def volume(dims):
    v = 1
    for d in dims:
        v *= d
    return v


def bytes_dslash(dims, N, w, xpay=False):
    return w * volume(dims) * (144 + 6 * N + (3 * N if xpay else 0))


def flops_dslash(dims, N, xpay=False):
    return (1158 if xpay else 1146) * (volume(dims) // 2) * N


def block_bytes(dims, N, w):
    return 2 * w * 3 * (volume(dims) // 2) * N


def bytes_iteration(dims, N, w):
    """fused-iteration traffic: links twice + 14 block passes."""
    return 2 * 144 * w * volume(dims) + 14 * block_bytes(dims, N, w)


def flops_iteration(dims, N):
    L = 3 * (volume(dims) // 2)
    return 2304 * (volume(dims) // 2) * N + 36 * L * N * N


# ---------------------------------------------------------------- clocks sampler

class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index
        self.t0 = self.t1 = None

    def mark_begin(self):
        self.t0 = time.time()

    def mark_end(self):
        self.t1 = time.time()

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([time.time()] + [c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, mx, reasons, power = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        # samples taken between mark_begin() and mark_end() (the timed steps and the per-kernel timing loops: the GPU
        # is busy throughout); a sample is stamped when its line arrives
        inside = [r for r in self.rows if self.t0 is None or (self.t0 <= r[0] <= (self.t1 or 1e30))]
        for r in inside:
            try:
                sm.append(float(r[1]))
                mx = float(r[2])
                power.append(float(r[3]))
            except (ValueError, IndexError):
                continue
            for n, v in zip(names, r[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "sm_mhz_min": sm[0] if sm else None, "samples": len(sm), "power_w_max": max(power) if power else None,
                "window": "timed steps + per-kernel timing loops"}


# ---------------------------------------------------------------- timing helpers

def time_loop(torch, fn, reps, warmup):
    """average ms per call of fn over `reps` calls, CUDA events on the current (= the library's) stream."""
    for _ in range(warmup):
        fn()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(reps):
        fn()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1) / reps


SM_COUNT, SM_MAX_MHZ = 148, 1965.0


def kernel_source_hash():
    """sha256 over the CUDA sources of the library: the key a stored ncu capture is valid for."""
    import glob
    import hashlib
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_1710_09745_b200", "csrc", "*.cu*"))):
        h.update(os.path.basename(f).encode())
        h.update(open(f, "rb").read())
    return h.hexdigest()


def ncu_traffic(workload, N, dtype):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel from the committed `ncu --set full`
    capture (profiles/r2_traffic.json).  The capture names the sha256 of the kernel sources it was taken from; if the
    sources have changed since, the number is stale and None is returned instead (never a pasted literal)."""
    path = os.path.join(ROOT, "profiles", "r2_traffic.json")
    if not os.path.exists(path):
        return None, None
    d = json.load(open(path))
    for e in d.get("captures", []):
        if e["workload"] == workload and e["N"] == N and e["dtype"] == dtype:
            info = {"commit": e.get("commit"), "source_sha256": e.get("source_sha256"), "kernel": e.get("kernel")}
            if e.get("source_sha256") == kernel_source_hash():
                return e["dram_bytes_read"] + e["dram_bytes_write"], info
            info["stale"] = True
            return None, info
    return None, None


# FMA-pipe peaks (GFLOP/s).  Default: DESIGN.md section 6.4's derivation from the guide's unit counts (148 SMs x 64 FP64 /
# 128 FP32 lanes x 2 flop x 1.965 GHz); run_bkr() replaces them by the register-only microbenchmark of bkr_microbench
# measured on this box and says so in the JSON line.
ALU_PEAK = {True: SM_COUNT * 64 * 2 * SM_MAX_MHZ * 1e-3, False: SM_COUNT * 128 * 2 * SM_MAX_MHZ * 1e-3, "source": "derived (unit counts x 1.965 GHz)"}

MICROBENCH_KINDS = [(0, "fp64_fma_tflops", 1e-9), (1, "fp32_fma_tflops", 1e-9), (2, "fp64_mma_m8n8k4_tflops", 1e-9),
                    (6, "stencil_fma_pattern_rhs_major_tflops", 1e-9), (7, "stencil_fma_pattern_link_major_tflops", 1e-9),
                    (3, "l2_to_sm_ldg_tbps", 1e-9), (4, "l2_to_sm_tma_tbps", 1e-9), (5, "smem_read_tbps", 1e-9)]


def run_microbench(ctx, reps=5):
    """on-chip peaks measured on this box (bkr_microbench): units / ms * 1e-9 = TFLOP/s or TB/s"""
    out = {}
    for kind, name, scale in MICROBENCH_KINDS:
        ms, units = ctx.microbench(kind, reps)
        out[name] = units / ms * scale
    return out


# on-chip probes of csrc/probes.cu (kind, name, what the number is): cycles of one SM and work per SM -> per-cycle rates
PROBE_KINDS = [(10, "lds128_conflict_free_B_per_clk_sm", "bytes"), (11, "lds128_broadcast8_B_per_clk_sm", "bytes"),
               (12, "lds128_with_tma_fills_B_per_clk_sm", "bytes+aux"), (13, "lds128_with_ldg_stream_B_per_clk_sm", "bytes+aux"),
               (14, "dfma_2_register_reads_per_clk_sm", "dfma"), (15, "dfma_3_register_reads_per_clk_sm", "dfma"),
               (16, "dfma_with_4_lds128_per_64_per_clk_sm", "dfma"), (17, "dfma_with_8_lds128_per_64_per_clk_sm", "dfma"),
               (18, "dry_stencil_T4_8warps_dfma_per_clk_sm", "dfma"), (19, "dry_stencil_T8_4warps_dfma_per_clk_sm", "dfma"),
               (20, "dry_stencil_T8_8warps_dfma_per_clk_sm", "dfma"),
               (21, "tma_9KB_issue_interval_clk_one_lane", "interval"), (22, "tma_9KB_round_trip_clk_idle_l2", "interval"),
               (23, "mma_sync_tf32_m16n8k8_flop_per_clk_sm", "flop"),
               (24, "latency_dfma_dependent_clk", "interval"), (25, "latency_fp64_reciprocal_plus_add_clk", "interval"),
               (26, "latency_fp64_rsqrt_plus_add_clk", "interval"), (27, "latency_shfl64_plus_add_clk", "interval"),
               (28, "latency_sts_lds_round_trip_clk", "interval"), (29, "latency_syncthreads_1024_clk", "interval")]


def run_probes(ctx):
    """the probes behind the stencil design (profiles/r2_onchip_probes.md), as per-cycle, per-SM rates"""
    out = {}
    for kind, name, what in PROBE_KINDS:
        cyc, units, aux = ctx.probe(kind)
        if what == "interval":
            out[name] = cyc / units
        else:
            out[name] = units / cyc
            if what.endswith("+aux"):
                out[name.replace("lds128_", "other_stream_")] = aux / cyc
    return out


def alu_peak_gflops(fp64):
    return ALU_PEAK[bool(fp64)]


def roofline_entry(ms, by, fl, hbm, fp64_math):
    """GB/s, GFLOPS, fraction of the HBM roofline, and fraction of max(bytes / BW, flops / ALU peak) with the binding
    term named."""
    t_hbm = by / hbm * 1e-6      # ms
    t_alu = fl / alu_peak_gflops(fp64_math) * 1e-6
    return {"ms": ms, "GBps": by / ms * 1e-6, "GFLOPS": fl / ms * 1e-6, "frac_hbm": t_hbm / ms,
            "frac_roofline": max(t_hbm, t_alu) / ms, "binding": "hbm" if t_hbm >= t_alu else "alu"}


def kernel_numbers(torch, ctx, binding, dims, N, prec, reps, warmup, hbm):
    """Dslash / Gram / block-update timings at one (N, precision): dict of GB/s, GFLOPS, fraction of HBM peak."""
    w = 8 if prec == binding.F64 else 4
    L = ctx.L
    nb = 3  # rotate over several buffers so that small blocks are not served from L2 alone
    blk = [ctx.empty_native(N, prec).normal_() for _ in range(nb + 1)]
    a = torch.randn(N, N, dtype=torch.complex128, device=ctx.device) * 0.1
    K = torch.empty(N, N, dtype=torch.complex128, device=ctx.device)
    out = {}
    i = [0]

    def rot():
        i[0] = (i[0] + 1) % nb
        return blk[i[0]], blk[(i[0] + 1) % nb]

    def f_dslash():
        s, d = rot()
        ctx.dslash(i[0] & 1, N, s, d, prec)
    ms = time_loop(torch, f_dslash, reps, warmup)
    by, fl = bytes_dslash(dims, N, w), flops_dslash(dims, N)
    out["dslash"] = roofline_entry(ms, by, fl, hbm, prec == binding.F64)
    out["dslash"]["variant"] = {0: "dslash_kernel (register tiling + link ring)",
                                1: "dslash_win_kernel (shared-memory window, cluster-multicast links)"}.get(ctx.dslash_variant(), "?")

    def f_dslash_xpay():
        s, d = rot()
        ctx.dslash_xpay(i[0] & 1, N, 4e-4, blk[nb], s, d, prec)
    ms = time_loop(torch, f_dslash_xpay, reps, warmup)
    by, fl = bytes_dslash(dims, N, w, xpay=True), flops_dslash(dims, N, xpay=True)
    out["dslash_xpay"] = roofline_entry(ms, by, fl, hbm, prec == binding.F64)

    def f_gram2():
        s, d = rot()
        ctx.gram(N, s, d, hermitian=False, prec=prec, out=K)
    ms = time_loop(torch, f_gram2, reps, warmup)
    by, fl = 2 * block_bytes(dims, N, w), 8 * L * N * N
    out["gram_xy"] = roofline_entry(ms, by, fl, hbm, True)

    def f_gram2h():
        s, d = rot()
        ctx.gram(N, s, d, hermitian=True, prec=prec, out=K)
    ms = time_loop(torch, f_gram2h, reps, warmup)
    by, fl = 2 * block_bytes(dims, N, w), 4 * L * N * (N + 1)
    out["gram_xy_herm"] = roofline_entry(ms, by, fl, hbm, True)

    def f_gram1():
        s, _ = rot()
        ctx.gram(N, s, s, hermitian=True, prec=prec, out=K)
    ms = time_loop(torch, f_gram1, reps, warmup)
    by, fl = block_bytes(dims, N, w), 4 * L * N * (N + 1)
    out["gram_xx"] = roofline_entry(ms, by, fl, hbm, True)

    def f_axpy():
        s, d = rot()
        ctx.block_axpy(N, a, s, d, prec)
    ms = time_loop(torch, f_axpy, reps, warmup)
    by, fl = 3 * block_bytes(dims, N, w), 8 * L * N * N
    out["block_axpy"] = roofline_entry(ms, by, fl, hbm, True)

    # the two fused kernels of the iteration: 6 and 3 block passes
    tri_u = torch.triu(a).contiguous()
    tri_l = torch.tril(a).contiguous()
    X64 = blk[nb] if prec == binding.F64 else ctx.empty_native(N, binding.F64).normal_()

    def f_pqx():
        s, d = rot()
        ctx.block_qpx_update(N, tri_u, tri_l, a, s, d, blk[(i[0] + 2) % nb], X64, prec)
    ms = time_loop(torch, f_pqx, reps, warmup)
    by = 4 * block_bytes(dims, N, w) + 2 * block_bytes(dims, N, 8)  # Q', P in, Q, P out (storage precision); X in and out (fp64)
    out["pqx_update"] = roofline_entry(ms, by, 16 * L * N * N, hbm, True)  # ~ half of 3 x 8 L N^2 for the triangular pair

    def f_ug():
        s, d = rot()
        ctx.block_axpy_gram(N, a, s, d, prec, out=K)
    ms = time_loop(torch, f_ug, reps, warmup)
    out["update_gram"] = roofline_entry(ms, 3 * block_bytes(dims, N, w), 8 * L * N * N + 4 * L * N * (N + 1), hbm, True)
    return out


# ---------------------------------------------------------------- CPU baseline (the oracle, as it stands)

_ORACLE_INPUTS = {}


def _omp_set_threads(n):
    """thread count of the oracle's OpenMP loops (same libgomp instance as liboracle.so)"""
    import ctypes
    try:
        ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))
        return True
    except OSError:
        return False


def oracle_sample(dims_full, N, kind, seed=5, max_sites_rhs=None, threads=None):
    """One blockCGrQ iteration's operations (1 x M, 2 x Gram, 4 x block update) with the oracle, as it stands, on the host
    cores.  Default: the FULL lattice of the workload when that is at most configs[2]'s size (32^3 x 64 x 16 rhs: a few
    seconds on 16 cores); larger workloads and the 1-thread figure use the same N and link generator on a lattice halved
    along its longest directions until it is bounded (stated in the returned description).
    returns (seconds, algorithmic bytes of the sample, sample description, threads)."""
    import numpy as np
    import oracle
    from paper_1710_09745_b200 import synth
    dims = list(dims_full)
    cap = max_sites_rhs if max_sites_rhs else 32 ** 3 * 64 * 16
    while volume(dims) * N > cap:
        k = max(range(4), key=lambda mu: dims[mu])
        dims[k] //= 2
    dims = tuple(dims)
    key = (dims, N, kind, seed)
    if key not in _ORACLE_INPUTS:  # inputs are generated once per process, outside every timed step
        fat, lng = synth.make_links(dims, kind, seed)
        _ORACLE_INPUTS.clear()
        _ORACLE_INPUTS[key] = (fat.numpy(), lng.numpy(), synth.make_sources(dims, N, seed + 1).numpy(),
                               synth.make_sources(dims, N, seed + 2).numpy())
    fat, lng, P, Q = _ORACLE_INPUTS[key]
    Q = Q.copy()
    a = (np.eye(N) * 0.5).astype(np.complex128)
    oracle.lib()
    ncpu = int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    used = ncpu
    if threads is not None and _omp_set_threads(threads):
        used = threads
    t0 = time.perf_counter()
    AP = oracle.apply_M(dims, fat, lng, 0.05, P)
    oracle.gram(P, AP)
    oracle.gram(Q, Q)
    for _ in range(4):
        oracle.block_axpy(a, P, Q)
    dt = time.perf_counter() - t0
    if threads is not None:
        _omp_set_threads(ncpu)
    full = tuple(dims) == tuple(dims_full)
    desc = "one blockCGrQ iteration's operations (1 x M, 2 x Gram, 4 x block update), N=%d, on %s %s lattice" % (
        N, "the full" if full else "a reduced", "x".join(str(d) for d in dims))
    return dt, bytes_iteration(dims, N, 8), desc, used


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/unit/config, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    name, dims, kind, mass, N = WORKLOADS[args.workload]
    times = []
    for i in range(args.warmup + args.steps):
        dt, by, desc, threads = oracle_sample(dims, N, kind)
        if i >= args.warmup:
            times.append(dt)
        if sum(times) > 120:  # bounded: the whole run ends within a few minutes whatever --steps says
            break
    ms = 1e3 * sum(times) / len(times)
    val = by / ms * 1e-6
    line = {
        "impl": "reference", "metric": "blockcg_iteration_effective_GBps", "value": val, "unit": "GB/s",
        "n_gpus": args.gpus, "steps": len(times), "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "dims": list(dims), "N": N, "mass": mass, "links": kind},
        "cpu_baseline": {"value": val, "unit": "GB/s", "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---------------------------------------------------------------- multi-GPU aggregation ("replicas only")

def max_over_ranks(dist, value, device):
    """MAX all-reduce of a host scalar (the timing of the slowest replica); identity without a process group."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replicas_value(world, bytes_per_step_per_rank, ms_step_max):
    """whole-job throughput of `world` independent replicas (no data-path collective): every
    rank moves the same algorithmic bytes per step; the job takes as long as its slowest rank."""
    return world * bytes_per_step_per_rank / ms_step_max * 1e-6


# ---------------------------------------------------------------- the CUDA path

def run_bkr(args):
    import torch
    from paper_1710_09745_b200 import binding, synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    hbm, peak_src = peaks()
    name, dims, kind, mass, N = WORKLOADS[args.workload]
    if args.N:
        N = args.N
    prec = binding.F32 if args.prec == "f32" else binding.F64
    w = 8 if prec == binding.F64 else 4
    dev = "cuda:%d" % local

    # inputs: seeded synthetic links and sources drawn on the device (synth.py), resident in HBM
    fat, lng = synth.make_links(dims, kind, seed=1000 + rank, device=dev)
    B = synth.make_sources(dims, N, seed=2000 + rank, device=dev)
    ctx = binding.Context(dims, device=local)
    ctx.load_links(fat, lng, also_f32=True)
    ctx.set_f32_math(args.f32_math)
    for kv in args.tune:
        ctx.set_option(binding.OPT_TUNE + int(kv.split("=")[0]), int(kv.split("=")[1]))
    del fat, lng
    torch.cuda.empty_cache()
    # on-chip peaks measured on this box: the "alu" roofline denominators
    micro = run_microbench(ctx)
    ALU_PEAK[True], ALU_PEAK[False] = micro["fp64_fma_tflops"] * 1e3, micro["fp32_fma_tflops"] * 1e3
    ALU_PEAK["source"] = "measured (bkr_microbench register-only FMA, this run)"
    sampler = ClockSampler(local)
    sampler.start()  # nvidia-smi takes a while to start: launched before the warm-up, windowed to the timed region

    # ---- timed region: K iterations after W warm-up iterations, device-resident
    launches_w = ctx.bench_iterations(mass, B, args.warmup, prec)
    torch.cuda.synchronize()
    sampler.mark_begin()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if dist:
        dist.barrier()
    torch.cuda.synchronize()
    e0.record()
    launches = ctx.bench_iterations(mass, B, args.steps, prec)
    e1.record()
    torch.cuda.synchronize()
    if dist:
        dist.barrier()
    ms_total = max_over_ranks(dist, e0.elapsed_time(e1), dev)
    ms_step = ms_total / args.steps
    # every timed iteration must have done its full work: the loop kernels become no-ops once the device-side `done`
    # flag is set (convergence or a Cholesky breakdown), which would time empty launches
    state = ctx.solver_state()
    if state["done"] or state["breakdown"] or state["iters"] != args.warmup + args.steps:
        raise RuntimeError("timed iterations did not all run: %r (expected %d iterations)" % (state, args.warmup + args.steps))
    by_iter = bytes_iteration(dims, N, w)
    value = replicas_value(world, by_iter, ms_step)

    # ---- the dominant kernel alone (multi-rhs Dslash), and the multi-BLAS kernels, at this N
    kern = kernel_numbers(torch, ctx, binding, dims, N, prec, reps=max(50, args.steps), warmup=3, hbm=hbm)
    sampler.mark_end()
    clocks = sampler.stop()

    # ---- end to end through the host-buffer entry point (copies inside the timed region)
    e2e = None
    if rank == 0 or dist:
        Bh = B.cpu().pin_memory()
        Xh = torch.zeros_like(Bh).pin_memory()
        ctx.solve_block_host(mass, Bh, Xh, tol=1e-10, maxiter=2, inner_prec=prec)  # warm-up (allocations)
        Xh.zero_()
        torch.cuda.synchronize()
        if dist:
            dist.barrier()
        t0 = time.perf_counter()
        rr, st = ctx.solve_block_host(mass, Bh, Xh, tol=1e-10, maxiter=args.steps, inner_prec=prec)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        dt = max_over_ranks(dist, dt, dev)
        k = max(1, st["iters"])
        e2e = {"value": world * k * by_iter / dt * 1e-9, "unit": "GB/s",
               "h2d_bytes_per_step": 2 * Bh.numel() * 16 / k, "d2h_bytes_per_step": Xh.numel() * 16 / k,
               "iterations": k, "seconds": dt,
               "note": "bkr_solve_block_host: H2D of B and X0, init QR, %d iterations, fp64 true-residual check, D2H of X" % k}
        del Bh, Xh

    # ---- time to solution: block CG vs N x CG (rank 0, N = 1 GPU runs only)
    solve = None
    if rank == 0 and world == 1 and not args.no_solve:
        solve = solve_comparison(torch, ctx, binding, mass, B, args)

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return 0

    cpu = None
    if world == 1 and not args.no_cpu:
        dt, sby, desc, threads = oracle_sample(dims, N, kind)
        cpu = {"value": sby / dt * 1e-9, "unit": "GB/s", "cores": threads, "kind": "oracle", "sample": desc,
               "seconds": dt}
        dt1, sby1, desc1, th1 = oracle_sample(dims, N, kind, max_sites_rhs=16 ** 3 * 32 * 16, threads=1)
        cpu["one_thread"] = {"value": sby1 / dt1 * 1e-9, "unit": "GB/s", "cores": th1, "sample": desc1, "seconds": dt1}

    ablation = None
    if rank == 0 and world == 1 and args.ablation:
        ablation = run_ablation(torch, ctx, binding, mass, B, prec)

    d = kern["dslash"]
    traffic, traffic_info = ncu_traffic(args.workload, N, "f64" if prec == binding.F64 else "f32")
    line = {
        "metric": "blockcg_iteration_effective_GBps", "value": value, "unit": "GB/s", "n_gpus": world,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64" if prec == binding.F64 else "f32", "data": "synthetic",
        "config": {"workload": name, "dims": list(dims), "N": N, "mass": mass, "links": kind,
                   "step": "one blockCGrQ iteration (Alg. 1 l.8-12): 2 Dslash, Gram P^H MP, fused Q+P+X update, fused Q' update + Gram, 2 small-matrix kernels",
                   "l2": "inputs larger than L2 (links %.2f GB + blocks %.2f GB each)" % (
                       144 * w * volume(dims) * 1e-9, block_bytes(dims, N, w) * 1e-9),
                   "f32_math": {0: "fp64 tensor products", 1: "split-TF32", 2: "split-TF32 updates", 3: "split-TF32 reductions"}[args.f32_math],
                   "parallelism": "replicas only" if world > 1 else "1 GPU"},
        "frac_hbm_iteration": value / world / hbm,
        "GFLOPS_iteration": world * flops_iteration(dims, N) / ms_step * 1e-6,
        "roofline": {"bound": "hbm", "kernel": "%s: multi-rhs Dslash, one parity, N=%d" % (d.get("variant", "dslash"), N),
                     "achieved": d["GBps"], "peak": hbm, "unit": "GB/s", "frac": d["GBps"] / hbm,
                     "traffic": traffic, "traffic_capture": traffic_info,
                     "frac_roofline": d["frac_roofline"], "binding": d["binding"],
                     "peak_source": peak_src, "ms_per_launch": d["ms"],
                     "algorithmic_bytes_per_launch": bytes_dslash(dims, N, w), "GFLOPS": d["GFLOPS"]},
        "kernels": kern,
        "alu_peak": {"fp64_gflops": ALU_PEAK[True], "fp32_gflops": ALU_PEAK[False], "source": ALU_PEAK["source"]},
        "microbench": micro,
        "iterations_completed": state["iters"],
        "e2e": e2e,
        "gpu_launches": launches,
        "clocks": clocks,
        "cpu_baseline": cpu,
        "solve": solve,
        "ablation": ablation,
    }
    print(json.dumps(line))
    if dist:
        dist.destroy_process_group()
    return 0


def run_ablation(torch, ctx, binding, mass, B, prec, iters=100):
    """The comparison of the paper's Fig. 4: time for 100 blockCGrQ iterations with (i) nothing
    blocked -- single-vector caxpys / dot products and one stencil call per rhs, (ii) block BLAS only, (iii) block BLAS +
    block Dslash (unfused kernels), (iv) the shipped iteration (fused updates, deferred X).  Same arithmetic in every arm
    (tests/test_gpu_multiblas_instances.py::test_ablation_switches...)."""
    arms = [("no_block", binding.ABL_VECTOR_BLAS | binding.ABL_VECTOR_DSLASH | binding.ABL_UNFUSED_UPDATES | binding.ABL_UNFUSED_GRAM),
            ("block_blas", binding.ABL_VECTOR_DSLASH | binding.ABL_UNFUSED_UPDATES | binding.ABL_UNFUSED_GRAM),
            ("block_blas_block_dslash", binding.ABL_UNFUSED_UPDATES | binding.ABL_UNFUSED_GRAM),
            ("fused (shipped)", 0)]
    out = {"iterations": iters, "N": int(B.shape[0])}
    try:
        for name, mask in arms:
            ctx.set_option(binding.OPT_ABLATION, mask)
            ctx.solve_block(mass, B, tol=1e-10, maxiter=0, inner_prec=prec)  # re-initialises the solver state
            ctx.bench_iterations(mass, B, 2, prec)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            n = ctx.bench_iterations(mass, B, iters, prec)
            e1.record()
            torch.cuda.synchronize()
            st = ctx.solver_state()
            out[name] = {"seconds": e0.elapsed_time(e1) * 1e-3, "launches": n, "completed": st["iters"], "done": st["done"]}
    finally:
        ctx.set_option(binding.OPT_ABLATION, 0)
        ctx.solve_block(mass, B, tol=1e-10, maxiter=0, inner_prec=prec)
    out["paper_context"] = "paper Fig. 4 (GP100, fp64): with block BLAS + block Dslash the time per rhs is about half that of 1-rhs CG"
    return out


def solve_comparison(torch, ctx, binding, mass, B, args):
    """block CG vs N sequential CGs vs one batched CG, tol 1e-10 (north_star).  Sequential CG is measured on
    `--cg-rhs` right-hand sides and scaled to N (stated in the output)."""
    N = int(B.shape[0])
    out = {"tol": 1e-10, "N": N}
    X, rr, st = ctx.solve_block(mass, B, tol=1e-10, maxiter=args.maxiter)
    out["block_cg"] = {"seconds": st["seconds"], "iters": st["iters"], "status": st["status"], "restarts": st["restarts"],
                       "true_relres_max": max(rr)}
    X, rr, st = ctx.solve_block(mass, B, tol=1e-10, maxiter=args.maxiter, inner_prec=binding.F32, delta=0.1)
    out["block_cg_mixed"] = {"seconds": st["seconds"], "iters": st["iters"], "status": st["status"],
                             "reliable_updates": st["reliable_updates"], "true_relres_max": max(rr)}
    n_seq = min(N, args.cg_rhs)
    X, its, rr, st = ctx.solve_cg(mass, B[:n_seq].contiguous(), tol=1e-10, maxiter=args.maxiter, batched=False)
    out["cg_sequential"] = {"seconds": st["seconds"] * N / n_seq, "measured_rhs": n_seq, "scaled_to": N,
                            "iters_mean": sum(its) / len(its), "status": st["status"], "true_relres_max": max(rr)}
    X, its, rr, st = ctx.solve_cg(mass, B, tol=1e-10, maxiter=args.maxiter, batched=True)
    out["cg_batched"] = {"seconds": st["seconds"], "iters_max": max(its), "status": st["status"], "true_relres_max": max(rr)}
    out["speedup_vs_sequential_cg"] = out["cg_sequential"]["seconds"] / out["block_cg"]["seconds"]
    out["speedup_vs_batched_cg"] = out["cg_batched"]["seconds"] / out["block_cg"]["seconds"]
    out["paper_context"] = "paper: 5x over sequential CG on SaturnV (PAPER.md:27, 370-378), other hardware and real ensembles"
    return out


def run_sweep(args):
    """BASELINE.json configs[4]: 32^4, random SU(3), N in {1,2,4,8,16,24,32}, fp64 and fp32: one JSON line per point."""
    import torch
    from paper_1710_09745_b200 import binding, synth
    hbm, _ = peaks()
    name, dims, kind, mass, _ = WORKLOADS["cfg5"]
    fat, lng = synth.make_links(dims, kind, seed=1000, device="cuda")
    ctx = binding.Context(dims)
    ctx.load_links(fat, lng, also_f32=True)
    del fat, lng
    # third pass: fp32 blocks with the split-TF32 multi-BLAS (BKR_TUNE_F32_MATH = 1; not the default).
    # Its "frac_roofline" still divides by the FP64 FMA peak: read frac_hbm there.
    for prec, pname, math in ((binding.F64, "f64", binding.F32_MATH_FP64), (binding.F32, "f32", binding.F32_MATH_FP64),
                              (binding.F32, "f32_tf32", binding.F32_MATH_TF32)):
        ctx.set_f32_math(math)
        for N in ((1, 2, 4, 8, 16, 24, 32) if pname != "f32_tf32" else (8, 16, 24, 32)):
            k = kernel_numbers(torch, ctx, binding, dims, N, prec, reps=args.steps, warmup=3, hbm=hbm)
            if pname == "f32_tf32":
                for kn in ("dslash", "dslash_xpay"):
                    k.pop(kn, None)
            row = {"sweep": name, "dtype": pname, "N": N}
            for kn, v in k.items():
                row[kn] = {a: (round(b, 4) if isinstance(b, float) else b) for a, b in v.items()}
            print(json.dumps(row), flush=True)
    return 0


def run_many(args):
    """The paper's model workload on synthetic links: `--many-rhs` Gaussian sources solved in blocks of N
    with bkr_solve_many (sloppy sweep to 5e-6, fine sweep to 2e-9), for each N of the paper's list that divides the count,
    fp64 and fp32-inner, next to sequential CG to 2e-9 (measured on --cg-rhs sources and scaled).  One JSON line."""
    import torch
    from paper_1710_09745_b200 import binding, synth
    name, dims, kind, mass, _ = WORKLOADS[args.workload]
    fat, lng = synth.make_links(dims, kind, seed=1000, device="cuda")
    ctx = binding.Context(dims)
    ctx.load_links(fat, lng, also_f32=True)
    ctx.set_f32_math(args.f32_math)
    del fat, lng
    nrhs = args.many_rhs
    B = synth.make_sources(dims, nrhs, seed=2000, device="cuda")
    out = {"many_rhs": nrhs, "workload": name, "tol_sloppy": 5e-6, "tol_fine": 2e-9, "blocks": {}}
    for N in (8, 16, 24, 32, 48, 64):
        if nrhs % N:
            continue
        for pname, kw in (("f64", {}), ("f32_inner", dict(inner_prec=binding.F32, delta=0.1))):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            X, rr, st = ctx.solve_many(mass, B, N, tol_sloppy=5e-6, tol_fine=2e-9, maxiter=args.maxiter, **kw)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            out["blocks"]["N=%d %s" % (N, pname)] = {
                "seconds": dt, "solver_seconds": sum(s[0]["seconds"] + s[1]["seconds"] for s in st),
                "iters_sloppy": sum(s[0]["iters"] for s in st), "iters_fine": sum(s[1]["iters"] for s in st),
                "status": [max(abs(s[0]["status"]), abs(s[1]["status"])) for s in st], "true_relres_max": max(rr),
                "reliable_updates": sum(s[0]["reliable_updates"] + s[1]["reliable_updates"] for s in st)}
            del X
            print("# N=%d %s: %.2f s" % (N, pname, dt), file=sys.stderr, flush=True)
    ncg = max(1, min(args.cg_rhs, nrhs))
    X, its, rr, st = ctx.solve_cg(mass, B[:ncg].contiguous(), tol=2e-9, maxiter=args.maxiter)
    out["cg_sequential"] = {"seconds": st["seconds"] * nrhs / ncg, "measured_rhs": ncg, "scaled_to": nrhs,
                            "iters_mean": float(sum(its)) / len(its), "true_relres_max": max(rr)}
    best = min(v["seconds"] for v in out["blocks"].values())
    out["speedup_best_block_vs_sequential_cg"] = out["cg_sequential"]["seconds"] / best
    out["paper_context"] = "paper Figs. 5-7: time to solution for 192 rhs falls monotonically with the block size; 5x at scale (other hardware, real ensembles)"
    print(json.dumps(out))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="bkr", choices=["bkr", "reference"])
    ap.add_argument("--workload", default="cfg3", choices=sorted(WORKLOADS))
    ap.add_argument("--N", type=int, default=0)
    ap.add_argument("--prec", default="f64", choices=["f64", "f32"])
    ap.add_argument("--many-rhs", type=int, default=0, help="run the many-rhs workload of PAPER.md:322-324 with this many sources (e.g. 192)")
    ap.add_argument("--no-solve", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--sweep", action="store_true")
    ap.add_argument("--microbench", action="store_true", help="print the on-chip microbenchmark numbers only")
    ap.add_argument("--ablation", action="store_true", help="add the Fig. 4-style ablation (100 iterations per arm)")
    ap.add_argument("--f32-math", type=int, default=0, choices=[0, 1, 2, 3],
                    help="tensor path of the multi-BLAS on fp32 blocks (bkr.h BKR_TUNE_F32_MATH): 0 FP64 DMMA (default), 1 split-TF32, "
                         "2 / 3 TF32 updates / reductions only; affects --prec f32 and the fp32-inner solver")
    ap.add_argument("--tune", action="append", default=[], metavar="K=V",
                    help="launch-policy knob BKR_TUNE_K = V (bkr.h), e.g. --tune 5=32 --tune 6=32; repeatable")
    ap.add_argument("--maxiter", type=int, default=20000)
    ap.add_argument("--cg-rhs", type=int, default=2, help="sequential CG is measured on this many rhs and scaled to N")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "bkr" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    if args.many_rhs:
        return run_many(args)
    if args.microbench:
        from paper_1710_09745_b200 import binding
        c8 = binding.Context((8, 8, 8, 8))
        print(json.dumps({"microbench": run_microbench(c8, reps=10), "unit": "TFLOP/s or TB/s", "probes": run_probes(c8),
                          "probes_unit": "per SM clock and SM (64 = FP64 peak, 128 B = shared-memory port) or clocks"}))
        return 0
    return run_bkr(args)


if __name__ == "__main__":
    sys.exit(main())
