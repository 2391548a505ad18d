"""The N > 1 path of bench.py on CPU: two gloo ranks (world_size 2).

The X-engine does not shard (north_star: one GPU, no collectives): ranks are independent replicas and
the only communication is the contract's barrier plus the MAX over ranks of the timed device milliseconds.  These
tests run that host logic with the gloo backend, and the `--impl reference` arm under torchrun (rank 0 prints the
one JSON line, the other rank exits 0 without work).
"""
import json
import os
import subprocess
import sys

import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    per_rank_ms = [10.0, 12.5][rank]                     # the slower rank decides
    total = bench.max_over_ranks(per_rank_ms, dist, world, "cpu")
    value = bench.whole_job_value(1000.0, 4, world, total)
    dist.barrier()
    out.put((rank, total, value))
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_value_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, total, value in got:
        assert total == 12.5                                      # MAX over ranks, seen by every rank
        assert value == 2 * 4 * 1000.0 / 12.5e-3                  # both replicas' units over the slowest rank's time


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.25) == 3.25
    assert bench.whole_job_value(10.0, 5, 1, 1000.0) == 50.0


def test_reference_arm_under_torchrun_prints_one_line():
    port = 31500 + os.getpid() % 2000
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--steps", "1",
           "--warmup", "0", "--workload", "cfg1"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert res.returncode == 0, res.stderr[-2000:]
    lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["cpu_baseline"]["kind"] == "oracle" and d["e2e"]["h2d_bytes_per_step"] == 0


# ---- channel sharding: host logic + equivalence to the unsharded result, world_size 2 on gloo ----
def test_channel_ranges_partition_the_channels():
    from paper_1305_5639_b200.shard import channel_range
    for C in (0, 1, 5, 64, 1000, 1024):
        for world in (1, 2, 3, 8):
            parts = [channel_range(C, world, r) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == C
            assert all(parts[r][1] == parts[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in parts]
            assert max(sizes) - min(sizes) <= 1


def _shard_worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import numpy as np
    import torch
    import oracle
    from paper_1305_5639_b200 import inputs
    from paper_1305_5639_b200.shard import channel_range
    dist.init_process_group("gloo", rank=rank, world_size=world)
    T, C, N, P = 40, 7, 5, 2
    x = inputs.gauss_ci8(T, C, N, P, 30.0, seed=123)                 # every rank derives the same stream from the seed
    c0, c1 = channel_range(C, world, rank)
    mine = torch.from_numpy(oracle.xengine(x[:, c0:c1].contiguous().numpy()))     # this rank's output slab
    slabs = [None] * world
    dist.all_gather_object(slabs, (c0, c1, mine))                    # test-only gather; the data path has no collective
    full = torch.cat([s[2] for s in sorted(slabs, key=lambda s: s[0])])
    want = torch.from_numpy(oracle.xengine(x.numpy()))
    out.put((rank, bool((full == want).all()), (c0, c1)))
    dist.destroy_process_group()


def test_channel_sharded_slabs_equal_the_unsharded_result_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33500 + os.getpid() % 2000
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [g[1] for g in got] == [True, True]
    assert got[0][2] == (0, 4) and got[1][2] == (4, 7)
