"""The N > 1 path of bench.py on CPU: two gloo ranks (replicas only).  Checks the
max-over-ranks timing exchange, the aggregate throughput and that the reference arm prints one line
from rank 0 only."""
import json
import os
import subprocess
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, ms_e2e = bench.max_over_ranks([10.0 + 5.0 * rank, 30.0 - 7.0 * rank], world, torch.device("cpu"))
    out.put((rank, ms, ms_e2e, bench.aggregate_throughput(200000, 4, ms, world)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_timing_is_max_over_ranks_and_throughput_is_aggregate():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, ms_e2e, value in res:
        assert ms == 15.0 and ms_e2e == 30.0                      # the slowest rank's time on every rank
        assert value == 2 * 200000 * 4 / 15e-3                     # both replicas' events in that time


def test_reference_arm_prints_from_rank0_only():
    env = dict(os.environ, WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT="29999")
    outs = []
    for rank in (0, 1):
        r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "1",
                            "--gpus", "2", "--steps", "1", "--warmup", "0"], env=dict(env, RANK=str(rank), LOCAL_RANK=str(rank)),
                           capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr
        outs.append(r.stdout.strip())
    line = json.loads(outs[0])
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["value"] > 0
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["cpu_baseline"]["kind"] == "oracle"
    assert outs[1] == ""
