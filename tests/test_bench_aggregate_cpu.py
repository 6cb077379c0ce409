"""Multi-GPU path of bench.py on CPU: the codec has no exchange step ("replicas only",
DESIGN.md 8), so the only cross-rank logic is the max-over-ranks timing and the whole-job
throughput.  Run with gloo, world size 2."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    mine = [1.0 + rank, 5.0 - rank, 2.5]                      # per-rank times (ms)
    red = bench.reduce_max_over_ranks(mine)
    thr = bench.whole_job_throughput(8192, world, red[0])
    out.put((rank, red, thr))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, red, thr in res:
        assert red == [2.0, 5.0, 2.5]                          # slowest rank wins, element-wise
        assert abs(thr - 2 * 8192 / 2.0e-3) < 1e-6            # all ranks' tokens / slowest step


def test_single_process_is_identity():
    import bench
    assert bench.reduce_max_over_ranks([3.0, 1.0]) == [3.0, 1.0]
    assert bench.whole_job_throughput(100, 1, 10.0) == 100 / 0.01


def test_reference_arm_prints_the_contract_line():
    """`bench.py --impl reference` (the oracle on host cores) on the Tiny config: one JSON line with the contract's keys."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--impl", "reference", "--config", "tiny", "--ref-rows", "64",
                          "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=300, cwd=root)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
                "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in line, key
    assert line["impl"] == "reference" and line["value"] > 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["config"]["workload"] == "tiny"
