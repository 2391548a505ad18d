#!/usr/bin/env python
"""bench.py -- X-engine throughput on B200 (BASELINE.json metric: TOPS at 8 ops per complex MAC).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--impl reference]

One STEP = one pass of the whole hot path over one batch of synthetic input: for the default
workload (BASELINE.json config 4, the one the metric is quoted on) that is one full integration
of N=256 stations, 2 pol, 1024 channels, accumulated over 4 successive corr_xengine calls of
T=2048 samples each (accumulate = 0, 1, 1, 1) on four different 2 GiB input buffers, i.e. the
triangular tcgen05 HERK + cross-call accumulation + packed-baseline writer, all inside libcorr.so.

value    device-resident inputs, CUDA events on the launching stream, max over ranks.
e2e      the same metric through corr_xengine_host (HOST pinned buffers; H2D of every call's
         input and D2H of the integrated visibilities inside the timed region).
roofline dominant kernel (the only kernel of a call) against the tensor peak for its dtype:
         MEASURED_PEAKS.json bf16 x nominal ratio (int8 2x, fp16 1x) -- see DESIGN.md.
cpu_baseline / --impl reference: the CPU oracle (oracle/) as it stands, on the host cores, on a
         bounded sample of the same workload (whole channels: all baselines, full T).

N > 1 (torchrun): the path does not shard (north_star: one GPU, no collectives) -> N independent
replicas, "scaling": "weak"; the barrier and the max over ranks are the only communication.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "xengine_tops_8ops_per_cmac"
UNIT = "TOPS"
NOMINAL_RATIO = {"ci8": 2.0, "cf16": 1.0}     # dense tensor peak relative to bf16 (guide: 4.5 / 2.25 / 2.25 PF)
FALLBACK_BF16_TFLOPS = 1590.0                  # B200_PROFILING.md fallback
FALLBACK_HBM_GBS = 6650.0
# DRAM traffic (dram__bytes_read.sum + dram__bytes_write.sum) of ONE xengine_direct_kernel launch from
# the committed `ncu --set full` capture of this workload (profiles/), or None where not captured.
NCU_TRAFFIC_BYTES = {
    # profiles/r1c_final_ncu_pair_feed.md (dram__bytes_read.sum + dram__bytes_write.sum of one launch)
    "cfg4": (3.198e9 + 3 * 4.275e9) / 4,          # accumulate = 0 once, accumulate = 1 three times per step
    "cfg3": 4.651e9,
    "cfg5_n64": 1.200e9,
    "cfg5_n32": 1.139e9,
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg4")
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "single", "pair", "quad", "simt"],
                    help="force a kernel variant (default: the library's own choice)")
    ap.add_argument("--piece", default="xengine", choices=["xengine", "corner_turn", "fengine"],
                    help="corner_turn: time the standalone corner-turn kernel (SURVEY 8(a) a1) on the workload's input; "
                         "fengine: time corr_fengine (SURVEY 8(f) rank 2) on 512 streams x 8192 spectra of 256 real int8 samples")
    ap.add_argument("--shard", default="none", choices=["none", "channels"],
                    help="channels: the N ranks split the workload's channels (strong scaling, SURVEY 8(f) rank 3); "
                         "default: N independent replicas (north_star: the path does not shard)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-gemm-peak", action="store_true",
                    help="skip the cuBLAS int8 / fp16 GEMM measured beside the kernel (context for the tensor peak)")
    ap.add_argument("--e2e-steps", type=int, default=0, help="steps of the host-buffer leg (default min(K, 5))")
    return ap.parse_args()


def workload(name):
    from paper_1305_5639_b200 import inputs
    cfg = dict(inputs.CONFIGS[name])
    N, P, C, T = cfg["N"], cfg["P"], cfg["C"], cfg["T"]
    B = N * cfg["Nb"] if cfg.get("Nb") else N * (N + 1) // 2       # rectangle (cross workload) or packed triangle
    cfg["name"] = name
    cfg["n_baseline"] = B
    cfg["cmacs_per_call"] = C * T * B * P * P
    cfg["ops_per_call"] = 8 * cfg["cmacs_per_call"]
    elt = 2 if cfg["dtype"] == "ci8" else 4
    cfg["in_bytes"] = T * C * (N + cfg.get("Nb", 0)) * P * elt
    cfg["out_bytes"] = C * B * P * P * 8
    return cfg


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(bf16=float(p["bf16_tflops"]), bf16_sustained=float(p.get("bf16_tflops_sustained", p["bf16_tflops"])),
                    hbm=float(p["hbm_gbs"]), source="measured")
    return dict(bf16=FALLBACK_BF16_TFLOPS, bf16_sustained=1400.0, hbm=FALLBACK_HBM_GBS, source="fallback")


# ------------------------------------------------------------------------------------------------
# clocks: sample nvidia-smi DURING the timed region
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thr = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thr = threading.Thread(target=self._pump, daemon=True)
        self.thr.start()

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        inside = [r for (ts, r) in self.rows if t0 <= ts <= t1 + 0.1] or [r for (_, r) in self.rows[-3:]]
        sm, smax, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in inside:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); pw.append(float(f[2]))
            except (ValueError, IndexError):
                continue
            for k, nm in enumerate(names):
                if len(f) > 3 + k and f[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# CPU oracle legs (the ONLY places bench.py touches oracle/)
# ------------------------------------------------------------------------------------------------
def oracle_sample_rate(cfg, x_host, min_seconds, xb_host=None):
    """Times oracle.xengine on whole channels of `x_host` ([T, n, N, P, 2] numpy) -> (CMAC/s, seconds, channels)."""
    import oracle
    n = x_host.shape[1]
    cm_per_chan = cfg["cmacs_per_call"] // cfg["C"]
    done, secs = 0, 0.0
    while True:
        t0 = time.perf_counter()
        if xb_host is None:
            oracle.xengine(x_host)
        else:
            oracle.xengine_cross(x_host, xb_host)
        secs += time.perf_counter() - t0
        done += n
        if secs >= min_seconds or done >= 64 * n:
            break
    return done * cm_per_chan / secs, secs, done


def cpu_sample_input(cfg, n_chan):
    """Bounded sample of the workload for the oracle: `n_chan` whole channels (all baselines, full T) of call 0,
    generated on the CPU with the workload's own recipe."""
    from paper_1305_5639_b200 import inputs
    return inputs.make_input(cfg, call=0, device="cpu", C=n_chan).numpy()


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    cfg = workload(args.workload)
    cores = oracle.max_threads()
    n_chan = max(1, min(cfg["C"], cores))
    x = cpu_sample_input(cfg, n_chan)
    xb = None
    if cfg.get("Nb"):
        from paper_1305_5639_b200 import inputs
        xb = inputs.make_input_b(cfg, call=0, device="cpu", C=n_chan).numpy()
    run = (lambda: oracle.xengine(x)) if xb is None else (lambda: oracle.xengine_cross(x, xb))
    cm_per_chan = cfg["cmacs_per_call"] // cfg["C"]
    for _ in range(max(0, min(args.warmup, 1))):          # one warm-up pass is plenty for a CPU loop
        run()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        run()
    secs = time.perf_counter() - t0
    tops = 8.0 * args.steps * n_chan * cm_per_chan / secs / 1e12
    sample = "%d of %d channels of %s call 0 per step (all %d baselines x %d pol products, full T=%d)" % (
        n_chan, cfg["C"], cfg["name"], cfg["n_baseline"], cfg["P"] ** 2, cfg["T"])
    line = {
        "impl": "reference", "metric": METRIC, "value": tops, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "int64" if cfg["dtype"] == "ci8" else "f64", "data": "synthetic",
        "config": {"workload": describe(cfg), "sample": sample},
        "cpu_baseline": {"value": tops, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": tops, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def library_gemm_peak(torch, dtype, n=8192, secs=2.0):
    """cuBLAS GEMM n^3 of the kernel's dtype (torch._int_mm / torch.matmul): best of 10 (burst) and back to back
    for `secs` (sustained), in TOPS (2 n^3 ops).  What a dense contraction reaches on THIS box under its power cap."""
    if dtype == "ci8":
        a = torch.randint(-127, 128, (n, n), dtype=torch.int8, device="cuda")
        b = torch.randint(-127, 128, (n, n), dtype=torch.int8, device="cuda")
        f = lambda: torch._int_mm(a, b)
    else:
        a = torch.randn((n, n), dtype=torch.float16, device="cuda")
        b = torch.randn((n, n), dtype=torch.float16, device="cuda")
        f = lambda: torch.matmul(a, b)
    for _ in range(3):
        f()
    torch.cuda.synchronize()
    best = float("inf")
    for _ in range(10):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(); f(); e1.record()
        torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0, k = time.time(), 0
    e0.record()
    while time.time() - t0 < secs:
        for _ in range(20):
            f()
        k += 20
        torch.cuda.synchronize()
    e1.record()
    torch.cuda.synchronize()
    ops = 2.0 * n ** 3
    return {"burst": ops / best / 1e9, "sustained": ops * k / e0.elapsed_time(e1) / 1e9,
            "unit": "TOPS" if dtype == "ci8" else "TFLOP/s",
            "how": "torch %s %d^3, best of 10 / back to back for %.0f s" % ("_int_mm" if dtype == "ci8" else "matmul fp16", n, secs)}


def describe(cfg):
    if cfg.get("Nb"):
        return ("%s: rectangle of %d x %d stations (cross-correlations only, PAPER.md:79), %d pol, %d channels, T=%d samples/call, "
                "complex %s -> %s [c][i][j][p][q]" % (cfg["name"], cfg["N"], cfg["Nb"], cfg["P"], cfg["C"], cfg["T"],
                                                      "int8" if cfg["dtype"] == "ci8" else "fp16",
                                                      "int32" if cfg["dtype"] == "ci8" else "fp32"))
    return ("%s: N=%d stations, %d pol, %d channels, T=%d samples/call, %d call(s) integrated (accumulate 0,1,..), "
            "complex %s -> %s packed triangle" % (cfg["name"], cfg["N"], cfg["P"], cfg["C"], cfg["T"], cfg["calls"],
                                                    "int8" if cfg["dtype"] == "ci8" else "fp16",
                                                    "int32" if cfg["dtype"] == "ci8" else "fp32"))


def max_over_ranks(value, dist=None, world=1, device="cpu"):
    """MAX over all ranks of a per-rank scalar (the contract's timing reduction); identity at world == 1."""
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(units_per_rank_step, steps, world, total_ms):
    """Whole-job throughput: the units ALL ranks processed (replicas: world x the same count) / the slowest rank's time."""
    return world * steps * units_per_rank_step / (total_ms * 1e-3)


# ------------------------------------------------------------------------------------------------
# piece (a): the standalone corner-turn kernel, HBM-bound (read in + write two planes)
# ------------------------------------------------------------------------------------------------
def run_corner_turn(args):
    import torch
    from paper_1305_5639_b200 import binding, inputs
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    cfg = workload(args.workload)
    pk = peaks()
    x = inputs.make_input(cfg, call=0, device="cuda")
    h = binding.Correlator(cfg["N"], cfg["P"], cfg["C"], cfg["T"], cfg["dtype"])
    ws = torch.empty((h.workspace_bytes,), dtype=torch.uint8, device="cuda")
    K, W = args.steps, max(args.warmup, 3)
    for _ in range(W):
        h.corner_turn(x, ws)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    for a, b in ev:
        a.record(); h.corner_turn(x, ws); b.record()
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in ev) / K
    nbytes = cfg["in_bytes"] + h.workspace_bytes          # read the input once, write ws and ws_rot
    gbs = nbytes / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": "corner_turn_gbs", "value": gbs, "unit": "GB/s", "n_gpus": 1, "steps": K, "warmup": W,
                      "ms_per_step": ms, "higher_is_better": True, "dtype": "u8", "data": "synthetic",
                      "config": {"workload": describe(cfg), "l2": "input + workspace (%.0f MiB) larger than L2" % (nbytes / 2 ** 20)},
                      "gpu_launches": K,
                      "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm"], "unit": "GB/s", "frac": gbs / pk["hbm"],
                                   "traffic": None, "kernel": "cturn::corner_turn_kernel", "kernel_ms": ms,
                                   "algorithmic_bytes_per_launch": nbytes}}), flush=True)


def run_fengine(args):
    """corr_fengine alone: HBM-bound (1 byte read + 2 bytes written per real sample)."""
    import torch
    from paper_1305_5639_b200 import binding
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    pk = peaks()
    M, A = 512, 8192
    g = torch.Generator(device="cuda"); g.manual_seed(1700)
    s = torch.clamp(torch.round(torch.randn((M, A * 256), generator=g, device="cuda") * 20.0), -127, 127).to(torch.int8)
    out = binding.fengine(s)
    K, W = args.steps, max(args.warmup, 3)
    for _ in range(W):
        binding.fengine(s, out)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    for a, b in ev:
        a.record(); binding.fengine(s, out); b.record()
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in ev) / K
    nbytes = s.numel() + out.numel() * 2
    gbs = nbytes / (ms * 1e-3) / 1e9
    print(json.dumps({"metric": "fengine_gbs", "value": gbs, "unit": "GB/s", "n_gpus": 1, "steps": K, "warmup": W,
                      "ms_per_step": ms, "higher_is_better": True, "dtype": "f32", "data": "synthetic",
                      "config": {"workload": "F-engine: %d streams x %d spectra of 256 real int8 samples (sigma 20) -> 128 complex fp16 "
                                             "channels in the X-engine layout" % (M, A),
                                 "l2": "input + output (%.0f MiB) larger than L2" % (nbytes / 2 ** 20),
                                 "gsamples_per_s": s.numel() / (ms * 1e-3) / 1e9},
                      "gpu_launches": K,
                      "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm"], "unit": "GB/s", "frac": gbs / pk["hbm"],
                                   "traffic": None, "kernel": "feng::fengine_kernel", "kernel_ms": ms,
                                   "algorithmic_bytes_per_launch": nbytes}}), flush=True)


# ------------------------------------------------------------------------------------------------
# native arm
# ------------------------------------------------------------------------------------------------
def run_native(args):
    import torch
    import torch.distributed as dist
    from paper_1305_5639_b200 import binding, inputs

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the X-engine has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    binding.lib()                                   # raises if libcorr.so is missing / cannot be built

    cfg = workload(args.workload)
    sharded = args.shard == "channels" and world > 1
    if sharded:
        # this rank owns a contiguous block of channels: a smaller, otherwise identical problem with its own output slab
        from paper_1305_5639_b200.shard import channel_range
        c0, c1 = channel_range(cfg["C"], world, rank)
        frac = (c1 - c0) / cfg["C"]
        for key in ("cmacs_per_call", "ops_per_call", "in_bytes", "out_bytes"):
            cfg[key] = int(cfg[key] * frac)
        cfg["C_total"], cfg["C"] = cfg["C"], c1 - c0
        cfg["seed"] = cfg["seed"] + 7 * rank            # each slab gets its own noise
    N, P, C, T, dtype, calls = cfg["N"], cfg["P"], cfg["C"], cfg["T"], cfg["dtype"], cfg["calls"]
    K, W = args.steps, max(args.warmup, 3)
    pk = peaks()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # every rank is an independent replica on its own seeded inputs (replicas only; no sharding)
    xs = [inputs.make_input(cfg, call=k, device="cuda") for k in range(calls)]
    cross = bool(cfg.get("Nb"))
    xbs = [inputs.make_input_b(cfg, call=k, device="cuda") for k in range(calls)] if cross else None
    h = binding.CrossCorrelator(N, cfg["Nb"], P, C, T, dtype) if cross else binding.Correlator(N, P, C, T, dtype)
    if args.kernel != "auto":
        h.set_kernel(args.kernel)
    kernel = h.kernel
    if not h.uses_tensor_cores and args.kernel != "simt":
        raise RuntimeError("workload %s does not run on the tcgen05 kernel" % cfg["name"])
    out = h.empty_output()
    # inputs smaller than L2 (126 MB) are re-read from DRAM only if L2 is flushed between steps
    flush = None
    in_total = cfg["in_bytes"] * calls
    if in_total < 512 * 2 ** 20:
        flush = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device="cuda")

    def step(ev=None):
        for k in range(calls):
            if ev is not None:
                ev[2 * k].record()
            if cross:
                h.xengine_cross(xs[k], xbs[k], out, accumulate=k > 0)
            else:
                h.xengine(xs[k], out, accumulate=k > 0)
            if ev is not None:
                ev[2 * k + 1].record()

    for _ in range(W):
        if flush is not None:
            flush.fill_(1)
        step()
    launches_per_call = h.last_launch_count
    barrier()

    # ---- timed region: device-resident inputs ---------------------------------------------------
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(2 * calls)] for _ in range(K)]
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    barrier()
    w0 = time.time()
    for s in range(K):
        if flush is not None:
            flush.fill_(s & 1)
        step(evs[s])
    barrier()
    w1 = time.time()
    clocks = sampler.stop(w0, w1) if rank == 0 else None
    call_ms = [evs[s][2 * k].elapsed_time(evs[s][2 * k + 1]) for s in range(K) for k in range(calls)]
    step_ms = [sum(call_ms[s * calls:(s + 1) * calls]) for s in range(K)]
    total_ms = sum(step_ms)          # device time of exactly K steps (flush kernels excluded)
    total_ms = max_over_ranks(total_ms, dist, world, "cuda")
    ops_step = cfg["ops_per_call"] * calls
    if sharded:
        # strong scaling: the job is ONE workload; sum the ranks' (nearly equal) shares
        t_ops = torch.tensor([float(ops_step)], dtype=torch.float64, device="cuda")
        dist.all_reduce(t_ops, op=dist.ReduceOp.SUM)
        value = whole_job_value(float(t_ops.item()), K, 1, total_ms) / 1e12
    else:
        value = whole_job_value(ops_step, K, world, total_ms) / 1e12
    kernel_ms = sum(call_ms) / len(call_ms)          # average launch duration of the dominant (only) kernel

    # ---- e2e: HOST pinned buffers through corr_xengine_host --------------------------------------
    e2e = None
    if not args.no_e2e and not cross:          # the host-buffer entry point exists for corr_xengine only
        Ke = args.e2e_steps or min(K, 5)
        xh = [x.cpu().pin_memory() for x in xs]
        oh = torch.empty(h.output_shape(), dtype=out.dtype).pin_memory()

        def host_step():
            for k in range(calls):
                h.xengine_host(xh[k], oh if k == calls - 1 else None, accumulate=k > 0)

        host_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(Ke):
            host_step()                  # blocking: returns after the D2H copy has completed
        barrier()
        te = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e = {"value": world * Ke * ops_step / float(te.item()) / 1e12, "unit": UNIT,
               "h2d_bytes_per_step": cfg["in_bytes"] * calls, "d2h_bytes_per_step": cfg["out_bytes"],
               "steps": Ke, "ms_per_step": 1e3 * float(te.item()) / Ke}
        if not torch.equal(oh.cuda(), out):
            raise RuntimeError("host-buffer leg and device leg disagree")
        del xh, oh

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel ----------------------------------------------------------
    ratio = NOMINAL_RATIO[dtype]
    # a kernel timed back to back for longer than ~0.25 s runs under the 1 kW power cap: sustained peak; else burst
    sustained = total_ms > 250.0
    peak = (pk["bf16_sustained"] if sustained else pk["bf16"]) * ratio
    achieved = cfg["ops_per_call"] / (kernel_ms * 1e-3) / 1e12
    acc_calls = calls - 1
    bytes_call = cfg["in_bytes"] + cfg["out_bytes"] * (1.0 + acc_calls / calls)      # avg over the step's calls
    roofline = {
        "bound": "tensor", "achieved": achieved, "peak": peak, "unit": "TOPS" if dtype == "ci8" else "TFLOP/s",
        "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES.get(cfg["name"]),
        "kernel": {"single": "xtc::xengine_direct_kernel<%d>", "pair": "xtc::xengine_pair_kernel<%d, 1>",
                   "quad": "xtc::xengine_pair_kernel<%d, 2>", "simt": "xsimt::xengine_simt_kernel<%d>"}[kernel]
                  % (1 if dtype == "ci8" else 2), "kernel_ms": kernel_ms,
        "peak_source": "%s bf16 %s %.1f TFLOP/s x nominal %s/bf16 ratio %.0f" % (
            pk["source"], "sustained" if sustained else "burst", pk["bf16_sustained"] if sustained else pk["bf16"], dtype, ratio),
        "frac_of_burst": achieved / (pk["bf16"] * ratio),
        "frac_of_sustained": achieved / (pk["bf16_sustained"] * ratio),
        "frac_of_nominal": achieved / (2250.0 * ratio),
        "algorithmic_ops_per_launch": cfg["ops_per_call"],
        "hbm": {"algorithmic_bytes_per_launch": bytes_call, "achieved_gbs": bytes_call / (kernel_ms * 1e-3) / 1e9,
                "peak_gbs": pk["hbm"], "frac": bytes_call / (kernel_ms * 1e-3) / 1e9 / pk["hbm"]},
    }

    # ---- the library GEMM of the same dtype, same protocol as MEASURED_PEAKS.json (context, not the denominator) --
    if world == 1 and not args.no_gemm_peak:
        roofline["library_gemm_8192"] = library_gemm_peak(torch, dtype)

    # ---- CPU oracle on a bounded sample (rank 0, N = 1 only) ------------------------------------------
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        cores = oracle.max_threads()
        n_chan = max(1, min(C, cores))
        x_host = xs[0][:, :n_chan].contiguous().cpu().numpy()      # the same bytes the GPU consumed
        xb_host = xbs[0][:, :n_chan].contiguous().cpu().numpy() if cross else None
        rate, secs, done = oracle_sample_rate(cfg, x_host, min_seconds=10.0, xb_host=xb_host)
        cpu = {"value": 8.0 * rate / 1e12, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": "channels 0..%d of call 0 (all %d baselines x %d pol products, full T=%d), %d channel passes in %.1f s"
                         % (n_chan - 1, cfg["n_baseline"], P * P, T, done, secs),
               "gcmac_per_s": rate / 1e9}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
        "dtype": "s8 x s8 -> s32" if dtype == "ci8" else "f16 x f16 -> f32", "data": "synthetic",
        "config": {"workload": describe(cfg), "l2": ("flushed between steps" if flush is not None else
                                                     "inputs (%.0f MiB per step) larger than L2" % (in_total / 2 ** 20)),
                   "parallelism": ("channels sharded over %d ranks, no collective" % world) if sharded else "replicas only (x%d)" % world, "visibilities_per_s": world * K * C * cfg["n_baseline"] * P * P
                   / (total_ms * 1e-3)},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_call * calls * K,
        "roofline": roofline, "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.piece == "corner_turn":
        run_corner_turn(args)
    elif args.piece == "fengine":
        run_fengine(args)
    else:
        run_native(args)


if __name__ == "__main__":
    main()
