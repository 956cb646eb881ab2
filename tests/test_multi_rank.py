"""Host logic of the N > 1 launch of bench.py, on CPU with the gloo backend (world_size 2).

The hot path does not shard (BASELINE.json north_star: "no multi-GPU sharding"):
N ranks are N independent replicas, there is no collective on the data path, and the only exchanges are
bench.py's barrier and the max-over-ranks of the timings.  These tests cover exactly that logic.
"""
import json
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, ROOT)
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, world, device="cpu")        # rank 1 is the slow one
    val = bench.whole_job_gcells(world, units_per_replica_step=3_000_000_000, steps=2, seconds=ms * 1e-3)
    dist.barrier()
    out.put((rank, ms, val))
    dist.destroy_process_group()


def test_max_over_ranks_and_replica_aggregate_gloo_world2():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, val in got:
        assert ms == 15.0                                    # the slowest rank's time, on every rank
        assert abs(val - 2 * 3.0 * 2 / 15e-3) < 1e-9         # 2 replicas x 3 Gcell x 2 steps / 15 ms
    assert torch.__version__


def test_reference_arm_under_torchrun_prints_one_line_from_rank0():
    """`bench.py --impl reference` launched as the driver launches it for N = 2: rank 0 runs the oracle on a
    bounded sample and prints the one JSON line, rank 1 exits 0 without work."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--workload", "config1"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(l) for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    line = lines[0]
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and line["e2e"]["h2d_bytes_per_step"] == 0
    assert line["metric"] == "cell-updates/sec" and line["unit"] == "Gcell/s"
