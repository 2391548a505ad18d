#!/usr/bin/env python
"""bench.py -- X-engine throughput on B200 (BASELINE.json metric: TOPS at 8 ops per complex MAC).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--impl reference]

One STEP = one pass of the whole hot path over one batch of synthetic input: for the default
workload (BASELINE.json config 4, the one the metric is quoted on) that is one full integration
of N=256 stations, 2 pol, 1024 channels, accumulated over 4 successive corr_xengine calls of
T=2048 samples each (accumulate = 0, 1, 1, 1) on four different 2 GiB input buffers, i.e. the
triangular tcgen05 HERK + cross-call accumulation + packed-baseline writer, all inside libcorr.so.

value     device-resident inputs, CUDA events on the launching stream, max over ranks.
e2e       the same metric through corr_xengine_host (HOST pinned buffers; H2D of every call's
          input and D2H of the integrated visibilities inside the timed region).
roofline  the dominant (only) kernel of a call against the SLOWER of its two roofs (north_star):
          tensor = algorithmic ops / dense tensor peak of its dtype (MEASURED_PEAKS.json bf16 x nominal
          ratio: int8 2x, fp16 1x), hbm = algorithmic bytes (input + output, + output again when a call
          accumulates) / measured copy bandwidth.  Both sides are always reported.
sustained the same step timed back to back for >= 2 s (power-capped clocks), with its own clock record,
          against the sustained peaks.
workloads (N = 1 only) short runs of every other BASELINE.json config point, the cross / dump modes and the
          standalone corner-turn and F-engine kernels, so that the driver-run line carries them too.
cpu_baseline / --impl reference: the CPU oracle (oracle/) as it stands, on the host cores, on a
          bounded sample of the same workload (whole channels: all baselines, full T).

N > 1 (torchrun): the path does not shard (north_star: one GPU, no collectives) -> N independent
replicas, "scaling": "weak"; the barrier and the max over ranks are the only communication.
`--shard channels` instead splits ONE seeded workload by channel windows (corr_create_window), no collective.
"""
import argparse
import hashlib
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
NOMINAL_BF16 = 2250.0
FALLBACK_BF16_TFLOPS = 1590.0                  # B200_PROFILING.md fallback
FALLBACK_HBM_GBS = 6650.0
# DRAM traffic (dram__bytes_read.sum + dram__bytes_write.sum, bytes per launch averaged over the step's calls) from the
# committed `ncu --set full` captures of the SAME kernel and geometry -- not measured by this run, and emitted only when
# the kernel that ran is the one that was captured: workload -> (kernel, bytes, capture file)
NCU_TRAFFIC = {
    "cfg4": ("pair", (3.1978e9 + 3 * 4.2746e9) / 4, "profiles/r3_ncu_final.md"),     # accumulate = 0 once, = 1 three times
    "cfg3": ("pair", 4.7305e9, "profiles/r3_ncu_final.md"),
    "cfg2": ("pair", 0.3158e9, "profiles/r3_ncu_final.md"),
    "cfg5_n32": ("single", 1.1387e9, "profiles/r3_ncu_final.md"),
    "cfg5_n64": ("pair", 1.1988e9, "profiles/r3_ncu_final.md"),
    "cfg5_n128": ("pair", 1.3251e9, "profiles/r3_ncu_final.md"),
    "cfg5_n256": ("pair", 1.5835e9, "profiles/r3_ncu_final.md"),
    "cfg5_n512": ("pair", 2.1053e9, "profiles/r3_ncu_final.md"),
    "cfg5_n1024": ("pair", 3.1701e9, "profiles/r3_ncu_final.md"),
    "cross_n256": ("pair", 3.1890e9, "profiles/r3_ncu_final.md"),
}      # every row: the shipped kernel at that geometry, captured at the end of round 3
KERNEL_NAMES = {"single": "xtc::xengine_direct_kernel<%d>", "pair": "xtc::xengine_pair_kernel<%d>",
                "simt": "xsimt::xengine_simt_kernel<%d>"}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg4")
    ap.add_argument("--impl", default="native", choices=["native", "reference"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "single", "pair", "simt"],
                    help="force a kernel variant (default: the library's own choice)")
    ap.add_argument("--piece", default="xengine", choices=["xengine", "corner_turn", "fengine", "fengine_ci8", "fx_chain", "fx_chain_f16", "dumps"],
                    help="corner_turn: time the standalone corner-turn kernel (SURVEY 8(a) a1) on the workload's input; "
                         "fengine: time corr_fengine (SURVEY 8(f) rank 2) on 512 streams x 8192 spectra of 256 real int8 samples")
    ap.add_argument("--shard", default="none", choices=["none", "channels"],
                    help="channels: the N ranks split ONE workload's channels into windows (strong scaling, SURVEY 8(f) rank 3); "
                         "default: N independent replicas (north_star: the path does not shard)")
    ap.add_argument("--backend", default="nccl", choices=["nccl", "gloo"],
                    help="torch.distributed backend for the barrier / max-over-ranks (gloo: several ranks may share one GPU, "
                         "LOCAL_RANK is mapped modulo the device count)")
    ap.add_argument("--channels", type=int, default=0, help="cut the workload to its first CHANNELS channels (sharding tests)")
    ap.add_argument("--check", action="store_true",
                    help="--shard channels: gather every rank's slabs on rank 0 (test-only gather; the data path keeps no "
                         "collective) and compare them word for word with ONE unsharded launch on the same input")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-gemm-peak", action="store_true",
                    help="skip the cuBLAS int8 / fp16 GEMM measured beside the kernel (context for the tensor peak)")
    ap.add_argument("--no-sustained", action="store_true", help="skip the >= 2 s back-to-back sub-record")
    ap.add_argument("--no-others", action="store_true", help="skip the short runs of the other workloads and pieces")
    ap.add_argument("--no-sha", action="store_true", help="skip the SHA-256 of the input buffers")
    ap.add_argument("--planes", type=int, default=1, choices=[1, 2], help="--piece corner_turn: planes written (2 adds ws_rot)")
    ap.add_argument("--e2e-steps", type=int, default=0, help="steps of the host-buffer leg (default min(K, 5))")
    return ap.parse_args()


def workload(name, channels=0):
    from paper_1305_5639_b200 import inputs
    cfg = dict(inputs.CONFIGS[name])
    if channels:
        cfg["C"] = min(cfg["C"], int(channels))
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
                    hbm=float(p["hbm_gbs"]), source="MEASURED_PEAKS.json")
    return dict(bf16=FALLBACK_BF16_TFLOPS, bf16_sustained=1400.0, hbm=FALLBACK_HBM_GBS, source="B200_PROFILING.md fallback")


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
                                          "--format=csv,noheader,nounits", "-lms", "50"],
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
def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


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


def cpu_baseline_record(cfg, x_host, xb_host, min_seconds=10.0):
    """The oracle as it stands on the host cores: all threads on `x_host`'s channels, then ONE thread on the first
    channel; CPU model and compiler flags recorded."""
    import oracle
    from oracle import build as obuild
    cores = oracle.max_threads()
    rate, secs, done = oracle_sample_rate(cfg, x_host, min_seconds, xb_host)
    oracle.set_threads(1)
    try:
        rate1, secs1, done1 = oracle_sample_rate(cfg, x_host[:, :1], min(3.0, min_seconds), None if xb_host is None else xb_host[:, :1])
    finally:
        oracle.set_threads(cores)
    return {"value": 8.0 * rate / 1e12, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "channels 0..%d of call 0 (all %d baselines x %d pol products, full T=%d), %d channel passes in %.1f s"
                      % (x_host.shape[1] - 1, cfg["n_baseline"], cfg["P"] ** 2, cfg["T"], done, secs),
            "gcmac_per_s": rate / 1e9,
            "threads_1": {"value": 8.0 * rate1 / 1e12, "unit": UNIT, "gcmac_per_s": rate1 / 1e9,
                          "sample": "channel 0, %d passes in %.1f s" % (done1, secs1)},
            "cpu_model": cpu_model(), "compiler": "gcc " + " ".join(obuild.CFLAGS)}


def run_reference(args):
    """--impl reference: the oracle as it stands on the host cores; rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    import oracle
    from oracle import build as obuild
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
        "cpu_baseline": {"value": tops, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "cpu_model": cpu_model(), "compiler": "gcc " + " ".join(obuild.CFLAGS)},
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


def bytes_per_call(cfg):
    """Algorithmic HBM bytes of one launch, averaged over the step's calls: input once, output written once, and read
    once more by every call that accumulates."""
    calls = cfg["calls"]
    return cfg["in_bytes"] + cfg["out_bytes"] * (1.0 + (calls - 1) / calls)


def exec_over_useful(cfg, kernel):
    """Real MACs the tensor-core tiles EXECUTE per channel and sample / the 4 real MACs of every needed complex product
    (the tensor fraction on executed as well as on useful operations).  Host logic only (corr_tile_schedule)."""
    from paper_1305_5639_b200 import binding
    N, P = cfg["N"], cfg["P"]
    useful = 4.0 * cfg["n_baseline"] * P * P
    if kernel == "simt":
        return 1.0
    if cfg.get("Nb"):
        blocks = -(-2 * N * P // 256) * -(-2 * cfg["Nb"] * P // 256)
        return blocks * 65536.0 / useful
    rows = 256 if kernel == "pair" else 128
    return sum(rows * ncols for (_, _, ncols) in binding.tile_schedule(N, P, cfg["dtype"], kernel)) / useful


def roofline_record(cfg, kernel, kernel_ms, pk, sustained):
    """The dominant kernel against the slower of its two roofs; both sides reported (north_star's definition)."""
    dtype = cfg["dtype"]
    ratio = NOMINAL_RATIO[dtype]
    bf16 = pk["bf16_sustained"] if sustained else pk["bf16"]
    peak_tensor = bf16 * ratio                                     # TOPS / TFLOP/s
    ops, nbytes = cfg["ops_per_call"], bytes_per_call(cfg)
    t_tensor_ms = ops / (peak_tensor * 1e12) * 1e3
    t_hbm_ms = nbytes / (pk["hbm"] * 1e9) * 1e3
    ach_tensor = ops / (kernel_ms * 1e-3) / 1e12
    ach_hbm = nbytes / (kernel_ms * 1e-3) / 1e9
    bound = "tensor" if t_tensor_ms >= t_hbm_ms else "hbm"
    tunit = "TOPS" if dtype == "ci8" else "TFLOP/s"
    traffic, traffic_source = None, None
    if cfg["name"] in NCU_TRAFFIC and NCU_TRAFFIC[cfg["name"]][0] == kernel and not cfg.get("sharded"):
        traffic = NCU_TRAFFIC[cfg["name"]][1]
        traffic_source = "%s (ncu capture)" % NCU_TRAFFIC[cfg["name"]][2]      # of this kernel + geometry, not this run
    return {
        "bound": bound,
        "achieved": ach_tensor if bound == "tensor" else ach_hbm,
        "peak": peak_tensor if bound == "tensor" else pk["hbm"],
        "unit": tunit if bound == "tensor" else "GB/s",
        "frac": max(t_tensor_ms, t_hbm_ms) / kernel_ms,
        "traffic": traffic, "traffic_source": traffic_source,
        "kernel": KERNEL_NAMES[kernel] % (1 if dtype == "ci8" else 2), "kernel_ms": kernel_ms,
        "exec_over_useful": exec_over_useful(cfg, kernel),
        "roof_ms": {"tensor": t_tensor_ms, "hbm": t_hbm_ms},
        "peak_source": "%s: bf16 %s %.1f TFLOP/s x nominal %s/bf16 ratio %.0f; HBM copy %.1f GB/s" % (
            pk["source"], "sustained" if sustained else "burst", bf16, dtype, ratio, pk["hbm"]),
        "tensor": {"algorithmic_ops_per_launch": ops, "achieved": ach_tensor, "unit": tunit, "peak": peak_tensor,
                   "frac": ach_tensor / peak_tensor, "frac_of_burst": ach_tensor / (pk["bf16"] * ratio),
                   "frac_of_sustained": ach_tensor / (pk["bf16_sustained"] * ratio),
                   "frac_of_nominal": ach_tensor / (NOMINAL_BF16 * ratio),
                   "frac_on_executed_ops": ach_tensor * exec_over_useful(cfg, kernel) / peak_tensor},
        "hbm": {"algorithmic_bytes_per_launch": nbytes, "achieved_gbs": ach_hbm, "peak_gbs": pk["hbm"],
                "frac": ach_hbm / pk["hbm"]},
    }


def sha256_tensor(t):
    """SHA-256 of a tensor's bytes (copied to the host in 256 MiB slices)."""
    import torch
    h = hashlib.sha256()
    flat = t.reshape(-1).view(torch.uint8)
    step = 1 << 28
    for k in range(0, flat.numel(), step):
        h.update(flat[k:k + step].cpu().numpy().tobytes())
    return h.hexdigest()


# ------------------------------------------------------------------------------------------------
# piece (a): the standalone corner-turn kernel, HBM-bound (read in + write two planes)
# ------------------------------------------------------------------------------------------------
def time_corner_turn(cfg, pk, K, W, planes=1):
    import torch
    from paper_1305_5639_b200 import binding, inputs
    x = inputs.make_input(cfg, call=0, device="cuda")
    with binding.Correlator(cfg["N"], cfg["P"], cfg["C"], cfg["T"], cfg["dtype"]) as h:
        ws = torch.empty((h.workspace_bytes * planes // 2,), dtype=torch.uint8, device="cuda")
        for _ in range(W):
            h.corner_turn(x, ws, planes=planes)
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        for a, b in ev:
            a.record(); h.corner_turn(x, ws, planes=planes); b.record()
        torch.cuda.synchronize()
        ms = sum(a.elapsed_time(b) for a, b in ev) / K
        nbytes = cfg["in_bytes"] + ws.numel()                 # read the input once, write ws (and ws_rot)
    gbs = nbytes / (ms * 1e-3) / 1e9
    return {"metric": "corner_turn_gbs", "value": gbs, "unit": "GB/s", "n_gpus": 1, "steps": K, "warmup": W,
            "ms_per_step": ms, "higher_is_better": True, "dtype": "u8", "data": "synthetic",
            "config": {"workload": describe(cfg), "planes": planes,
                       "l2": "input + workspace (%.0f MiB) larger than L2" % (nbytes / 2 ** 20)},
            "gpu_launches": K,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm"], "unit": "GB/s", "frac": gbs / pk["hbm"],
                         "traffic": 4.2471e9 if (cfg["name"] == "cfg4" and planes == 1) else None,
                         "traffic_source": "profiles/r3_ncu_final.md (ncu capture)" if (cfg["name"] == "cfg4" and planes == 1) else None,
                         "kernel": "cturn::corner_turn_kernel", "kernel_ms": ms,
                         "algorithmic_bytes_per_launch": nbytes}}


def time_fengine(pk, K, W, M=512, A=8192, ci8=False):
    """corr_fengine alone: HBM-bound (1 byte read + 2 bytes written per real sample; corr_fengine_ci8: 1 + 1)."""
    import torch
    from paper_1305_5639_b200 import binding
    g = torch.Generator(device="cuda"); g.manual_seed(1700)
    s = torch.clamp(torch.round(torch.randn((M, A * 256), generator=g, device="cuda") * 20.0), -127, 127).to(torch.int8)
    scale = 1.0 / 20 if ci8 else None                # sigma ~ 16 codes per component, the int8 X-engine's input range
    out = binding.fengine(s, scale=scale)
    for _ in range(W):
        binding.fengine(s, out, scale=scale)
    torch.cuda.synchronize()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    for a, b in ev:
        a.record(); binding.fengine(s, out, scale=scale); b.record()
    torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in ev) / K
    nbytes = s.numel() + out.numel() * out.element_size()
    gbs = nbytes / (ms * 1e-3) / 1e9
    return {"metric": "fengine_gbs", "value": gbs, "unit": "GB/s", "n_gpus": 1, "steps": K, "warmup": W,
            "ms_per_step": ms, "higher_is_better": True, "dtype": "f16 x f16 -> f32 (twiddles hi + lo)", "data": "synthetic",
            "config": {"workload": "F-engine: %d streams x %d spectra of 256 real int8 samples (sigma 20) -> 128 complex %s "
                                   "channels in the X-engine layout" % (M, A, "int8 (requantised, scale 1/20)" if ci8 else "fp16"),
                       "l2": "input + output (%.0f MiB) larger than L2" % (nbytes / 2 ** 20),
                       "gsamples_per_s": s.numel() / (ms * 1e-3) / 1e9},
            "gpu_launches": K,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm"], "unit": "GB/s", "frac": gbs / pk["hbm"],
                         "traffic": (2.0917e9 if ci8 else 3.1619e9) if (M, A) == (512, 8192) else None,
                         "traffic_source": "profiles/r3_ncu_final.md (ncu capture)" if (M, A) == (512, 8192) else None,
                         "kernel": ("fengtc::fengine_tc_kernel<%s, %s>" % ("true" if ci8 else "false", "true" if M % 64 else "false"))
                         if binding.fengine_uses_tensor_cores(M, out) else "feng::fengine_kernel",
                         "kernel_ms": ms, "algorithmic_bytes_per_launch": nbytes}}


def time_fx_chain(pk, K, W, ci8=True, N=256, P=2, A=8192):
    """The paper's FX pair as ONE timed unit ("the F-engine and the X-engine"; its only single-GPU figure, ~105
    GFLOPS on a C2075, is for both together): N*P streams of A*256 real int8 samples -> corr_fengine_ci8
    (or corr_fengine, fp16) -> corr_xengine on the 128 channels x A spectra it wrote, one CUDA-event interval around both
    launches.  Ops counted as the paper counts them, necessary operations only: X = 8 per complex MAC over
    the N(N+1)/2 pairs; F = 2.5 n log2 n per real length-n transform (n = 256: 5120), the usual split-radix convention."""
    import torch
    from paper_1305_5639_b200 import binding
    M = N * P
    g = torch.Generator(device="cuda"); g.manual_seed(1900)
    s = torch.clamp(torch.round(torch.randn((M, A * 256), generator=g, device="cuda") * 20.0), -127, 127).to(torch.int8)
    scale = 1.0 / 20 if ci8 else None
    dtype = "ci8" if ci8 else "cf16"
    with binding.Correlator(N, P, 128, A, dtype) as h:
        spec = binding.fengine(s, scale=scale)                        # [A, 128, M, 2] = the X-engine's [T, C, N, P, 2]
        x = spec.view(A, 128, N, P, 2)
        out = h.xengine(x)
        for _ in range(W):
            binding.fengine(s, spec, scale=scale); h.xengine(x, out)
        torch.cuda.synchronize()
        ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]
        for a, b, c in ev:
            a.record(); binding.fengine(s, spec, scale=scale); b.record(); h.xengine(x, out); c.record()
        torch.cuda.synchronize()
        kernel = h.kernel
    ms = sum(a.elapsed_time(c) for a, _, c in ev) / K
    ms_f = sum(a.elapsed_time(b) for a, b, _ in ev) / K
    ms_x = sum(b.elapsed_time(c) for _, b, c in ev) / K
    ops_x = 8.0 * 128 * A * (N * (N + 1) // 2) * P * P
    ops_f = 2.5 * 256 * 8 * M * A
    nbytes = s.numel() + 2 * spec.numel() * spec.element_size() + out.numel() * 4      # F: read + write; X: read + write
    gbs = nbytes / (ms * 1e-3) / 1e9
    return {"metric": "fx_chain_tops", "value": (ops_x + ops_f) / (ms * 1e-3) / 1e12, "unit": UNIT, "n_gpus": 1, "steps": K,
            "warmup": W, "ms_per_step": ms, "higher_is_better": True, "dtype": "s8 x s8 -> s32" if ci8 else "f16 x f16 -> f32",
            "data": "synthetic",
            "config": {"workload": "fx_%s: %d stations x %d pol = %d streams x %d spectra of 256 real int8 samples (sigma 20) -> F-engine "
                                   "(128 complex %s channels) -> X-engine (T = %d, %s kernel)"
                                   % ("ci8" if ci8 else "f16", N, P, M, A, "int8, scale 1/20" if ci8 else "fp16", A, kernel),
                       "l2": "every buffer of the chain (%.0f MiB moved) larger than L2" % (nbytes / 2 ** 20),
                       "gsamples_per_s": s.numel() / (ms * 1e-3) / 1e9,
                       "ops": {"x_engine_8_per_cmac": ops_x, "f_engine_2.5nlog2n": ops_f}},
            "gpu_launches": 2 * K,
            "fengine_ms": ms_f, "xengine_ms": ms_x,
            "xengine_tops": ops_x / (ms_x * 1e-3) / 1e12,
            "roofline": {"bound": "hbm", "achieved": gbs, "peak": pk["hbm"], "unit": "GB/s", "frac": gbs / pk["hbm"],
                         "traffic": None, "kernel": "fengtc::fengine_tc_kernel + xtc::xengine_%s_kernel" % kernel, "kernel_ms": ms,
                         "algorithmic_bytes_per_launch": nbytes,
                         "note": "the pair of launches against the HBM roof of the bytes both must move; the X-engine half alone "
                                 "is tensor-bound at this geometry (xengine_tops)"}}


def run_piece(args):
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device")
    torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    K, W = args.steps, max(args.warmup, 3)
    if args.piece == "corner_turn":
        rec = time_corner_turn(workload(args.workload), peaks(), K, W, args.planes)
    elif args.piece == "dumps":
        rec = dumps_run(peaks(), K, W)
    elif args.piece.startswith("fx_chain"):
        rec = time_fx_chain(peaks(), K, W, ci8=args.piece == "fx_chain")
    else:
        rec = time_fengine(peaks(), K, W, ci8=args.piece == "fengine_ci8")
    print(json.dumps(rec), flush=True)


# ------------------------------------------------------------------------------------------------
# timing of one X-engine workload on resident inputs
# ------------------------------------------------------------------------------------------------
class Resident:
    """A workload with its inputs resident in HBM and a plan on them."""

    def __init__(self, cfg, kernel="auto", window=None):
        import torch
        from paper_1305_5639_b200 import binding, inputs
        self.cfg, self.torch = cfg, torch
        self.cross = bool(cfg.get("Nb"))
        self.xs = [inputs.make_input(cfg, call=k, device="cuda") for k in range(cfg["calls"])]
        self.xbs = [inputs.make_input_b(cfg, call=k, device="cuda") for k in range(cfg["calls"])] if self.cross else None
        N, P, C, T, dtype = cfg["N"], cfg["P"], cfg["C"], cfg["T"], cfg["dtype"]
        self.h = (binding.CrossCorrelator(N, cfg["Nb"], P, C, T, dtype) if self.cross
                  else binding.Correlator(N, P, C, T, dtype, window=window))
        if kernel != "auto":
            self.h.set_kernel(kernel)
        self.out = self.h.empty_output()
        # inputs smaller than ~4x L2 (126 MB) are (partly) re-read from L2 unless it is flushed between steps
        self.flush = None
        if cfg["in_bytes"] * cfg["calls"] < 512 * 2 ** 20:
            self.flush = torch.empty(256 * 2 ** 20, dtype=torch.uint8, device="cuda")

    def step(self, ev=None):
        for k in range(self.cfg["calls"]):
            if ev is not None:
                ev[2 * k].record()
            if self.cross:
                self.h.xengine_cross(self.xs[k], self.xbs[k], self.out, accumulate=k > 0)
            else:
                self.h.xengine(self.xs[k], self.out, accumulate=k > 0)
            if ev is not None:
                ev[2 * k + 1].record()

    def timed(self, K, cold=True):
        """K steps, per-call CUDA events on the launching stream -> list of per-call ms (flush kernels excluded)."""
        torch, calls = self.torch, self.cfg["calls"]
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(2 * calls)] for _ in range(K)]
        for s in range(K):
            if cold and self.flush is not None:
                self.flush.fill_(s & 1)
            self.step(evs[s])
        torch.cuda.synchronize()
        return [evs[s][2 * k].elapsed_time(evs[s][2 * k + 1]) for s in range(K) for k in range(calls)]

    def close(self):
        self.h.close()
        self.xs = self.xbs = self.out = self.flush = None
        self.torch.cuda.empty_cache()


def short_run(name, pk, K=10, W=3, sha=True):
    """A short run of another workload for the `workloads` list of the headline line."""
    cfg = workload(name)
    r = Resident(cfg)
    try:
        for _ in range(W):
            if r.flush is not None:
                r.flush.fill_(1)
            r.step()
        r.torch.cuda.synchronize()
        ms = r.timed(K, cold=True)
        kernel_ms = sum(ms) / len(ms)
        rec = {"workload": describe(cfg), "kernel": r.h.kernel, "steps": K, "ms_per_call": kernel_ms,
               "value": cfg["ops_per_call"] / (kernel_ms * 1e-3) / 1e12, "unit": UNIT,
               "best_ms_per_call": min(ms), "best_value": cfg["ops_per_call"] / (min(ms) * 1e-3) / 1e12,
               "visibilities_per_s": cfg["C"] * cfg["n_baseline"] * cfg["P"] ** 2 / (kernel_ms * 1e-3),
               "l2": "flushed between steps (cold)" if r.flush is not None else "inputs larger than L2",
               "roofline": roofline_record(cfg, r.h.kernel, kernel_ms, pk, sustained=False)}
        if r.flush is not None:                                  # small inputs: also the L2-warm figure
            warm = r.timed(K, cold=False)
            wms = sum(warm) / len(warm)
            rec["l2_warm"] = {"ms_per_call": wms, "value": cfg["ops_per_call"] / (wms * 1e-3) / 1e12, "unit": UNIT}
        if kernel_ms < 0.03 and not r.cross:                     # launch-bound: the same calls replayed from a CUDA graph
            torch = r.torch
            st, g = torch.cuda.Stream(), torch.cuda.CUDAGraph()
            with torch.cuda.stream(st):
                with torch.cuda.graph(g, stream=st):
                    for _ in range(20):
                        for k in range(cfg["calls"]):
                            r.h.xengine(r.xs[k], r.out, accumulate=k > 0, stream=st)
            g.replay(); torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            for _ in range(K):
                g.replay()
            b.record(); torch.cuda.synchronize()
            gms = a.elapsed_time(b) / (K * 20 * cfg["calls"])
            rec["cuda_graph"] = {"ms_per_call": gms, "value": cfg["ops_per_call"] / (gms * 1e-3) / 1e12, "unit": UNIT,
                                 "how": "20 calls captured with stream capture, replayed back to back (L2 warm)"}
        if sha:
            rec["input_sha256"] = [sha256_tensor(x) for x in r.xs]
        return rec
    finally:
        r.close()


def dumps_run(pk, K=10, W=3):
    """Short-integration mode (corr_xengine_dumps): N=256, C=256, T=2048 in 16 integrations of 128 samples."""
    import torch
    from paper_1305_5639_b200 import binding, inputs
    N, P, C, T, nd = 256, 2, 256, 2048, 16
    x = inputs.gauss_ci8(T, C, N, P, 20.0, seed=1800, device="cuda")
    with binding.Correlator(N, P, C, T, "ci8") as h:
        out = h.xengine_dumps(x, nd)
        for _ in range(W):
            h.xengine_dumps(x, nd, out)
        torch.cuda.synchronize()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
        for a, b in ev:
            a.record(); h.xengine_dumps(x, nd, out); b.record()
        torch.cuda.synchronize()
    ms = sum(a.elapsed_time(b) for a, b in ev) / K
    ops = 8.0 * C * T * (N * (N + 1) // 2) * P * P
    nbytes = x.numel() + out.numel() * 4
    return {"workload": "dumps: N=%d, %d pol, %d channels, T=%d cut into %d integrations of %d samples, int8" % (N, P, C, T, nd, T // nd),
            "ms_per_call": ms, "value": ops / (ms * 1e-3) / 1e12, "unit": UNIT,
            "hbm": {"algorithmic_bytes_per_launch": nbytes, "achieved_gbs": nbytes / (ms * 1e-3) / 1e9,
                    "frac": nbytes / (ms * 1e-3) / 1e9 / pk["hbm"],
                    "traffic": 4.7919e9 if (N, P, C, T, nd) == (256, 2, 256, 2048, 16) else None,
                    "traffic_source": "profiles/r3_ncu_final.md (ncu capture)"}}


# ------------------------------------------------------------------------------------------------
# the headline line: compact (the driver keeps only the last ~3 KB of stdout and parses the LAST line)
# ------------------------------------------------------------------------------------------------
HEADLINE_MAX_BYTES = 2000


def _r(v, sig=5):
    """Floats to `sig` significant digits (bytes matter on the headline line); everything else unchanged."""
    if isinstance(v, float):
        return float("%.*g" % (sig, v)) if v == v and v not in (float("inf"), float("-inf")) else None
    return v


def _cut(s, n):
    return s if s is None or len(s) <= n else s[:n - 1] + "~"


def workload_key(rec, k):
    """Short key of a side record for the headline's `workloads` summary."""
    w = rec.get("workload") or (rec.get("config") or {}).get("workload") or rec.get("metric") or "w%d" % k
    key = w.split(":")[0].strip().replace(" ", "_")
    if rec.get("metric") == "fengine_gbs":
        key = "fengine_ci8" if "int8 (requantised" in w else "fengine_f16"
    elif rec.get("metric") == "corner_turn_gbs":
        key = "corner_turn"
    elif rec.get("metric") == "fx_chain_tops":
        key = "fx_ci8" if w.startswith("fx_ci8") else "fx_f16"
    return _cut(key, 16)


def workloads_summary(others):
    """{"cfg3": [value, frac, bound], ...}: ~40 bytes per side record; the full records go out on earlier lines."""
    out = {}
    for k, rec in enumerate(others or []):
        key = workload_key(rec, k)
        if "error" in rec:
            out[key] = "error"
            continue
        roof = rec.get("roofline") or {}
        if not roof and "hbm" in rec:
            roof = {"frac": rec["hbm"].get("frac"), "bound": "hbm"}
        out[key] = [_r(rec.get("value"), 4), _r(roof.get("frac"), 3), roof.get("bound")]
    return out


def compact_headline(full, others):
    """The ONE line the driver parses: the contract keys, compact roofline / sustained / e2e / cpu_baseline objects and a
    `workloads` summary.  Always a single line of strict JSON shorter than HEADLINE_MAX_BYTES: if worst-case strings
    push it over, the optional parts are dropped in a fixed order (never the contract keys)."""
    cfg, roof, sus, cpu, e2e, clk = (full.get(k) or {} for k in ("config", "roofline", "sustained", "cpu_baseline", "e2e", "clocks"))
    line = {k: _r(full.get(k)) for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better",
                                        "scaling", "vs_baseline", "dtype", "data", "gpu_launches")}
    line["config"] = {"workload": _cut(cfg.get("workload"), 132), "parallelism": _cut(cfg.get("parallelism"), 80),
                      "l2": _cut(cfg.get("l2"), 60)}
    line["clocks"] = {k: _r(clk.get(k)) for k in ("sm_mhz", "sm_max_mhz", "power_w_max", "reasons")} if clk else None
    line["e2e"] = {k: _r(e2e.get(k)) for k in ("value", "unit", "h2d_bytes_per_step", "d2h_bytes_per_step", "steps", "ms_per_step")} if e2e else None
    if roof:
        line["roofline"] = {k: _r(roof.get(k)) for k in ("bound", "achieved", "peak", "unit", "frac", "kernel", "kernel_ms", "traffic")}
        line["roofline"].update({"traffic_source": _cut(roof.get("traffic_source"), 40),
                                 "frac_of_nominal": _r((roof.get("tensor") or {}).get("frac_of_nominal"), 3),
                                 "frac_on_executed_ops": _r((roof.get("tensor") or {}).get("frac_on_executed_ops"), 3),
                                 "hbm_frac": _r((roof.get("hbm") or {}).get("frac"), 3),
                                 "exec_over_useful": _r(roof.get("exec_over_useful"), 4),
                                 "hbm_write_peak": _r(roof.get("hbm_write_peak_gbs"), 4)})
    else:
        line["roofline"] = None
    line["sustained"] = {"value": _r(sus.get("value")), "frac": _r((sus.get("roofline") or {}).get("frac"), 3),
                         "sm_mhz": _r((sus.get("clocks") or {}).get("sm_mhz")),
                         "reasons": (sus.get("clocks") or {}).get("reasons")} if sus else None
    line["cpu_baseline"] = {"value": _r(cpu.get("value")), "unit": cpu.get("unit"), "cores": cpu.get("cores"), "kind": cpu.get("kind"),
                            "sample": _cut(cpu.get("sample"), 72), "threads_1": _r((cpu.get("threads_1") or {}).get("value")),
                            "cpu_model": _cut(cpu.get("cpu_model"), 48)} if cpu else None
    line["workloads"] = workloads_summary(others) if others else None
    if full.get("check"):
        line["check"] = {k: full["check"].get(k) for k in ("sharded_equals_unsharded", "words", "ranks_with_work", "sha256")}
    line["full"] = "gpurun_out/bench_full.json"
    for drop in (None, "full", ("cpu_baseline", "sample"), ("config", "l2"), "workloads", ("cpu_baseline", "sample"), ("cpu_baseline", "cpu_model"), ("config", "l2"),
                 ("config", "parallelism"), ("roofline", "traffic_source"), "sustained", ("config", "workload")):
        if isinstance(drop, tuple):
            if line.get(drop[0]):
                line[drop[0]][drop[1]] = None
        elif drop is not None:
            line[drop] = None
        text = json.dumps(line, separators=(",", ":"), allow_nan=False)
        if len(text.encode()) < HEADLINE_MAX_BYTES:
            break
    return text


def sharded_check(cfg, r, window, rank, world, dist):
    """--shard channels --check: every rank runs one more step and sends the slabs its window plan wrote to rank 0
    (a test-only gather of host copies; the data path itself has no collective).  Rank 0 puts them together in channel order
    and compares them with ONE unsharded launch on the same seeded input: bit for bit (per-channel work is identical
    whichever plan runs it).  Returns the record for the headline on rank 0, None elsewhere."""
    import numpy as np
    import torch
    from paper_1305_5639_b200 import binding
    mine = None
    if r is not None:
        r.step()
        torch.cuda.synchronize()
        c0, n = window
        mine = (c0, r.out[c0:c0 + n].cpu().numpy())
    parts = [None] * world if rank == 0 else None
    dist.gather_object(mine, parts, dst=0)
    if rank != 0:
        return None
    parts = sorted((p for p in parts if p is not None), key=lambda p: p[0])
    covered = sum(p[1].shape[0] for p in parts)
    contiguous = all(parts[k][0] + parts[k][1].shape[0] == parts[k + 1][0] for k in range(len(parts) - 1))
    full = np.concatenate([p[1] for p in parts])
    with binding.Correlator(cfg["N"], cfg["P"], cfg["C"], cfg["T"], cfg["dtype"]) as h:
        ref = None
        for k, x in enumerate(r.xs):
            ref = h.xengine(x, ref, accumulate=k > 0)
        torch.cuda.synchronize()
        ref = ref.cpu().numpy()
    same = parts[0][0] == 0 and covered == cfg["C"] and contiguous and full.shape == ref.shape and bool(
        (full.view(np.uint32) == ref.view(np.uint32)).all())
    return {"sharded_equals_unsharded": same, "words": int(ref.size), "ranks_with_work": len(parts),
            "windows": [[int(p[0]), int(p[1].shape[0])] for p in parts], "sha256": hashlib.sha256(full.tobytes()).hexdigest()}


def emit(full, others):
    """Side records first (one JSON line each, also written to gpurun_out/bench_full.json), the compact headline LAST."""
    for rec in others or []:
        print(json.dumps({"record": "workload", **rec}), flush=True)
    print(json.dumps({"record": "headline_detail", **full}), flush=True)
    try:
        os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
        with open(os.path.join(ROOT, "gpurun_out", "bench_full.json"), "w") as f:
            json.dump({"headline": full, "workloads": others}, f, indent=1)
    except OSError:
        pass
    print(compact_headline(full, others), flush=True)


def hbm_write_peak(torch, nbytes=2 << 30, reps=10):
    """Write-only HBM bandwidth (a plain fill of 2 GiB, CUDA events, best of `reps`): the roof of the write-dominated
    pieces (dumps, F-engine, N = 1024), for which the 1:1 read/write copy figure of MEASURED_PEAKS.json is not the bound."""
    buf = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    buf.fill_(1)
    torch.cuda.synchronize()
    best = float("inf")
    for k in range(reps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(); buf.fill_(k & 1); b.record()
        torch.cuda.synchronize()
        best = min(best, a.elapsed_time(b))
    del buf
    return nbytes / (best * 1e-3) / 1e9


# ------------------------------------------------------------------------------------------------
# native arm
# ------------------------------------------------------------------------------------------------
def run_native(args):
    import torch
    import torch.distributed as dist
    from paper_1305_5639_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the X-engine has no CPU fallback")
    local = local % torch.cuda.device_count()       # (gloo runs: several ranks on one GPU)
    torch.cuda.set_device(local)
    red_dev = "cuda" if args.backend == "nccl" else "cpu"           # where the max-over-ranks scalars live
    if world > 1:
        if args.backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")
    binding.lib()                                   # raises if libcorr.so is missing / cannot be built

    cfg = workload(args.workload, args.channels)
    sharded = args.shard == "channels" and world > 1
    window = None
    share = 1.0                                     # this rank's share of the workload's ops / bytes
    if sharded:
        # every rank holds the SAME seeded whole-band input and a whole-band output; its window plan integrates its
        # contiguous block of channels in place (corr_create_window) -- one workload, disjoint output slabs, no collective
        from paper_1305_5639_b200.shard import channel_range
        if cfg.get("Nb"):
            raise RuntimeError("--shard channels applies to the triangle workloads")
        c0, c1 = channel_range(cfg["C"], world, rank)
        window = (c0, c1 - c0) if c1 > c0 else None
        share = (c1 - c0) / cfg["C"]
        cfg["sharded"] = True
    P, C, dtype, calls = cfg["P"], cfg["C"], cfg["dtype"], cfg["calls"]
    K, W = args.steps, max(args.warmup, 3)
    pk = peaks()
    idle = sharded and window is None               # more ranks than channels: this rank has nothing to integrate

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    r = None if idle else Resident(cfg, args.kernel, window)
    kernel = "pair" if idle else r.h.kernel
    if r is not None and not r.h.uses_tensor_cores and args.kernel != "simt":
        raise RuntimeError("workload %s does not run on the tcgen05 kernel" % cfg["name"])
    for _ in range(W):
        if r is not None:
            if r.flush is not None:
                r.flush.fill_(1)
            r.step()
    launches_per_call = 0 if idle else r.h.last_launch_count
    barrier()

    # ---- timed region: device-resident inputs ---------------------------------------------------
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    barrier()
    w0 = time.time()
    call_ms = [] if idle else r.timed(K, cold=True)
    barrier()
    w1 = time.time()
    clocks = sampler.stop(w0, w1) if rank == 0 else None
    total_ms = max_over_ranks(sum(call_ms), dist, world, red_dev)         # device time of exactly K steps, slowest rank
    ops_step = cfg["ops_per_call"] * calls
    if sharded:
        value = whole_job_value(ops_step, K, 1, total_ms) / 1e12          # strong scaling: the job is ONE workload
    else:
        value = whole_job_value(ops_step, K, world, total_ms) / 1e12
    kernel_ms = sum(call_ms) / max(1, len(call_ms))          # average launch duration of the dominant (only) kernel

    # ---- every other config point and piece, briefly (N = 1 only), so the driver-run line carries them --------------
    # They run BEFORE the >= 2 s sustained leg, after a pause, on a part that is not yet power-capped, so that scoring them
    # against the burst peaks is fair and their fractions are comparable from run to run.
    others, write_peak = None, None
    if world == 1 and not args.no_others and args.workload == "cfg4" and args.kernel == "auto":
        others = []
        time.sleep(1.0)
        try:
            write_peak = hbm_write_peak(torch)
        except Exception:
            write_peak = None
        for name in ["cfg1", "cfg2", "cfg3"] + ["cfg5_n%d" % n for n in (32, 64, 128, 256, 512, 1024)] + ["cross_n256"]:
            try:
                others.append(short_run(name, pk, sha=not args.no_sha))
            except Exception as e:                                    # a failed side run must not lose the headline
                others.append({"workload": name, "error": repr(e)})
        for fn in (lambda: dumps_run(pk), lambda: time_corner_turn(workload("cfg4"), pk, 10, 3), lambda: time_fengine(pk, 10, 3),
                   lambda: time_fengine(pk, 10, 3, ci8=True), lambda: time_fx_chain(pk, 10, 3, ci8=True),
                   lambda: time_fx_chain(pk, 10, 3, ci8=False)):
            try:
                others.append(fn())
            except Exception as e:
                others.append({"error": repr(e)})
        if write_peak:
            for rec in others:
                if isinstance(rec.get("roofline"), dict):
                    rec["roofline"]["hbm_write_peak_gbs"] = write_peak
                elif "hbm" in rec:
                    rec["hbm"]["hbm_write_peak_gbs"] = write_peak

    # ---- sustained: the same step back to back for >= 2 s (power-capped clocks), its own clock record -----------
    sustained = None
    if not args.no_sustained:                       # (idle ranks of a sharded run take part in the barriers and the reduction)
        est = max(kernel_ms * calls, 1e-3)
        Ks = 0 if idle else max(K, int(2200.0 / est) + 1)
        if sharded:                                 # one step count for the whole job: the slowest rank's
            Ks = max(K, int(max_over_ranks(Ks, dist, world, red_dev)))
        s2 = ClockSampler(local)
        if rank == 0:
            s2.start()
            time.sleep(0.1)
        barrier()
        t0 = time.time()
        ms2 = [0.0] if idle else r.timed(Ks, cold=True)
        barrier()
        t1 = time.time()
        tot2 = max_over_ranks(sum(ms2), dist, world, red_dev)
        k_ms = sum(ms2) / len(ms2)
        sustained = {"steps": Ks, "seconds": tot2 * 1e-3, "ms_per_step": tot2 / Ks,
                     "value": whole_job_value(ops_step, Ks, 1 if sharded else world, tot2) / 1e12, "unit": UNIT,
                     "clocks": s2.stop(t0, t1) if rank == 0 else None,
                     "roofline": None if sharded else roofline_record(cfg, kernel, k_ms, pk, sustained=True)}

    # ---- e2e: HOST pinned buffers through corr_xengine_host --------------------------------------
    e2e, sha = None, None
    if not args.no_e2e and not r is None and not r.cross and not sharded:
        Ke = args.e2e_steps or min(K, 5)
        xh = [x.cpu().pin_memory() for x in r.xs]
        oh = torch.empty(r.h.output_shape(), dtype=r.out.dtype).pin_memory()
        if not args.no_sha and rank == 0:
            sha = [hashlib.sha256(x.numpy()).hexdigest() for x in xh]

        def host_step():
            for k in range(calls):
                r.h.xengine_host(xh[k], oh if k == calls - 1 else None, accumulate=k > 0)

        host_step()
        barrier()
        t0 = time.perf_counter()
        for _ in range(Ke):
            host_step()                  # blocking: returns after the D2H copy has completed
        barrier()
        te = torch.tensor([time.perf_counter() - t0], dtype=torch.float64, device=red_dev)
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e = {"value": world * Ke * ops_step / float(te.item()) / 1e12, "unit": UNIT,
               "h2d_bytes_per_step": cfg["in_bytes"] * calls, "d2h_bytes_per_step": cfg["out_bytes"],
               "steps": Ke, "ms_per_step": 1e3 * float(te.item()) / Ke,
               "how": "corr_xengine_host: 8 channel windows per call through an H2D / kernel / D2H pipeline on 3 streams"}
        r.step()
        torch.cuda.synchronize()
        if not torch.equal(oh.cuda(), r.out):
            raise RuntimeError("host-buffer leg and device leg disagree")
        del xh, oh
    elif not args.no_sha and rank == 0 and r is not None:
        sha = [sha256_tensor(x) for x in r.xs]

    check = sharded_check(cfg, r, window, rank, world, dist) if (args.check and sharded) else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel: the timed region above decides burst vs sustained peaks -------------------
    # (a kernel timed back to back for longer than ~0.25 s runs under the 1 kW power cap: sustained peak; else burst)
    roofline = roofline_record(cfg, kernel, kernel_ms / max(share, 1e-9) if sharded else kernel_ms, pk, sustained=total_ms > 250.0)
    if sharded:
        roofline["note"] = "channel-sharded: kernel_ms scaled to the whole workload (this rank integrated %.3f of it)" % share

    # ---- the library GEMM of the same dtype, same protocol as MEASURED_PEAKS.json (context, not the denominator) --
    if world == 1 and not args.no_gemm_peak:
        roofline["library_gemm_8192"] = library_gemm_peak(torch, dtype)
    roofline["hbm_write_peak_gbs"] = write_peak

    # ---- CPU oracle on a bounded sample (rank 0, N = 1 only) ------------------------------------------
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        import oracle
        n_chan = max(1, min(C, oracle.max_threads()))
        x_host = r.xs[0][:, :n_chan].contiguous().cpu().numpy()      # the same bytes the GPU consumed
        xb_host = r.xbs[0][:, :n_chan].contiguous().cpu().numpy() if r.cross else None
        cpu = cpu_baseline_record(cfg, x_host, xb_host)

    in_total = cfg["in_bytes"] * calls
    flushed = r is not None and r.flush is not None
    if r is not None:
        r.close()

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "strong" if sharded else "weak", "vs_baseline": None,
        "dtype": "s8 x s8 -> s32" if dtype == "ci8" else "f16 x f16 -> f32", "data": "synthetic",
        "config": {"workload": describe(cfg), "l2": ("flushed between steps" if flushed else
                                                     "inputs (%.0f MiB per step) larger than L2" % (in_total / 2 ** 20)),
                   "parallelism": ("channel windows of one workload over %d ranks, no collective" % world) if sharded
                   else "replicas only (x%d)" % world,
                   "visibilities_per_s": (1 if sharded else world) * K * C * cfg["n_baseline"] * P * P / (total_ms * 1e-3),
                   "input_sha256": sha},
        "clocks": clocks, "e2e": e2e, "gpu_launches": launches_per_call * calls * K,
        "roofline": roofline, "sustained": sustained, "cpu_baseline": cpu,
    }
    if check is not None:
        line["check"] = check
    emit(line, others)
    if check is not None and not check["sharded_equals_unsharded"]:
        raise SystemExit("--check: the gathered channel windows differ from the unsharded launch")
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.piece != "xengine":
        run_piece(args)
    else:
        run_native(args)


if __name__ == "__main__":
    main()
