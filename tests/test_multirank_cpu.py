"""N > 1 path on CPU (gloo, world_size 2): bench.py runs one independent replica per rank, so
the only cross-rank logic is the reduction of time (MAX) and work (SUM) and the rule that rank 0 alone prints."""
import json
import os
import socket
import subprocess
import sys

import pytest

torch = pytest.importorskip("torch")
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms, nch = bench.reduce_over_ranks(dist, torch.device("cpu"), 10.0 + 5.0 * rank, 1000 * (rank + 1))
    # every rank builds a different replica (seed + rank)
    args = bench.parse.__globals__["argparse"].Namespace(config="tiny", grid=4, pair_prob=0.0)
    p = bench.make_workload(args, seed_offset=rank)
    seeds = [None] * world
    dist.all_gather_object(seeds, int(p.seed))
    out[rank] = (ms, nch, seeds)
    dist.destroy_process_group()


def test_time_is_max_and_work_is_sum_over_ranks():
    import torch.multiprocessing as mp
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    for rank in range(world):
        ms, nch, seeds = res[rank]
        assert ms == 15.0 and nch == 3000.0
        assert seeds[0] != seeds[1]


def test_reference_arm_prints_on_rank_zero_only():
    port = _free_port()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
           "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
           "--steps", "1", "--warmup", "0", "--config", "tiny", "--grid", "4"]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["n_gpus"] == 2 and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["cpu_baseline"]["kind"] == "oracle"
