"""The N > 1 path of bench.py on the CPU: two gloo ranks, whole-job aggregation (time = max over
ranks, units = sum over ranks).  The hot path itself shards with no exchange step."""
import os
import socket
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, units = bench.aggregate_over_ranks(10.0 + 5.0 * rank, 1000.0 * (rank + 1), dist)
    q.put((rank, ms, units))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregation_gloo():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, ms, units in res:
        assert ms == 15.0 and units == 3000.0


def test_single_rank_passthrough():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.aggregate_over_ranks(3.0, 7.0, None) == (3.0, 7.0)
    fl = bench.flops_per_unit({"Nr": 33, "Nt": 48, "Np": 96, "L": 43})
    assert sum(fl.values()) == (2 * 33 + 4 * 48 + 2 * 96 + 13) + 5 * (2 * 43 + 1)


def test_gpus_2_without_torchrun_starts_two_ranks():
    """`python bench.py --gpus 2` launched plainly (no torchrun, WORLD_SIZE unset) must start the two ranks itself.  Driven end
    to end on the CPU through the reference arm: both ranks rendezvous over gloo, rank 0 alone runs the oracle and prints the
    one JSON line with n_gpus = 2."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2", "--config", "1",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.strip().splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
