"""`bench.py --shard channels` with REAL processes on the CUDA window path ("orthogonal
correlation triangles separating frequency channels prior to the CMAC stage", PAPER.md:63-69 independent correlation nodes).

Only one GPU is available, so the ranks share it (gloo for the barrier and the max over ranks, LOCAL_RANK modulo the device
count); their kernels never wait on one another.  Every rank integrates its channel window of ONE seeded workload in place
through corr_create_window; `--check` gathers the slabs on rank 0 and compares them bit for bit with one unsharded launch.
This test then ties that result to the oracle: the same unsharded launch done here has the same SHA-256, and sampled
channels of it equal oracle.xengine word for word.  Three ranks on a two-channel cut exercise the idle-rank path.
Measured on ONE GPU only: no scaling figure is taken from this.
"""
import hashlib
import json
import os
import subprocess
import sys

import numpy as np
import pytest
import torch

from paper_1305_5639_b200 import inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("nproc,channels", [(2, 0), (3, 2)])
def test_bench_shard_channels_real_processes(oracle, nproc, channels):
    if not torch.cuda.is_available():
        pytest.fail("GPU tests need a CUDA device (there is no CPU fallback)")
    port = 34100 + (os.getpid() + 7 * nproc) % 1500
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(nproc),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"),
           "--gpus", str(nproc), "--shard", "channels", "--workload", "cfg2", "--backend", "gloo", "--check",
           "--steps", "2", "--warmup", "3", "--no-cpu-baseline", "--no-gemm-peak", "--no-sha"]
    if channels:
        cmd += ["--channels", str(channels), "--no-sustained"]
    res = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=900)
    assert res.returncode == 0, (res.stdout[-1500:], res.stderr[-3000:])
    line = json.loads(res.stdout.strip().splitlines()[-1])
    cfg = dict(inputs.CONFIGS["cfg2"])
    C = channels or cfg["C"]
    assert line["n_gpus"] == nproc and line["scaling"] == "strong" and line["value"] > 0
    chk = line["check"]
    assert chk["sharded_equals_unsharded"] is True
    assert chk["ranks_with_work"] == min(nproc, C)
    assert chk["words"] == C * (cfg["N"] * (cfg["N"] + 1) // 2) * cfg["P"] ** 2 * 2

    # the same unsharded launch here: same bytes as the gathered windows, and equal to the oracle on sampled channels
    from paper_1305_5639_b200 import binding
    x = inputs.make_input(cfg, call=0, device="cuda", C=C)
    with binding.Correlator(cfg["N"], cfg["P"], C, cfg["T"], cfg["dtype"]) as h:
        got = h.xengine(x)
        torch.cuda.synchronize()
    got = got.cpu().numpy()
    assert hashlib.sha256(got.tobytes()).hexdigest() == chk["sha256"]
    chans = sorted({0, C // 2, C - 1})
    want = oracle.xengine(x[:, chans].contiguous().cpu().numpy())
    assert (got[chans].astype(np.int64) == want).all()
