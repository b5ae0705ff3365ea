"""N > 1 path on CPU (gloo, world_size 2): the reduction of time (MAX) and work (SUM), the rule that rank 0 alone prints,
and the k-sharded evaluation: ranges that partition the k points, stores that together hold every
ordered term exactly once, and the exchange of the owned slices."""
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


def _sharded_worker(rank, world, port, out):
    import numpy as np
    import torch.distributed as dist
    import paper_2511_03683_b200 as ephc
    from paper_2511_03683_b200.sharded import ShardedSolver
    from ephc_inputs import make_problem
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p = make_problem("si", grid=(12, 12, 12), pair_prob=0.3, seed=3)      # the same problem on every rank
    S = ShardedSolver(p, dist, torch.device("cpu"), flags=ephc.HOST_ONLY)
    g = S.h.export_gather()                                               # this rank's ordered terms
    lo, hi = S.h.owned_states()
    assert (lo, hi) == (S.ranges[rank][0] * p.nb, S.ranges[rank][1] * p.nb)
    assert np.all((g["dest"] >= lo) & (g["dest"] < hi))
    # this rank's piece of I from its own store (numpy, Eq. 2 as printed), then the library's exchange of the pieces
    f, N = p.f, p.N
    fa, fb, Nq = f[g["dest"]], f[g["partner"]], N[g["iq"].astype(np.int64) * p.nnu + g["nu"]]
    o_, i_ = fa * (1 - fb), fb * (1 - fa)
    F = np.where(g["kind"] == 1, o_ * (Nq + 1) - i_ * Nq, o_ * Nq - i_ * (Nq + 1))
    I = np.zeros(p.ns)
    np.add.at(I, g["dest"], np.where(g["diag"] == 1, 0.0, -g["w"] * F))
    It = torch.from_numpy(I)
    S.x(It)
    F3 = torch.from_numpy(np.tile(np.where((np.arange(p.ns) >= lo) & (np.arange(p.ns) < hi), float(rank + 1), -1.0), 3))
    S.x(F3, 3)
    out[rank] = dict(ranges=S.ranges, terms=np.stack([g[k] for k in ("dest", "partner", "iq", "nu", "kind", "diag")]),
                     w=g["w"], I=It.numpy().copy(), F3=F3.numpy().copy(), rows=S.h.export_rows()["dest"])
    dist.destroy_process_group()


def test_k_sharded_stores_partition_the_ordered_terms():
    import numpy as np
    import torch.multiprocessing as mp
    import oracle
    import paper_2511_03683_b200 as ephc
    from ephc_inputs import make_problem
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_sharded_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    p = make_problem("si", grid=(12, 12, 12), pair_prob=0.3, seed=3)
    ranges = res[0]["ranges"]
    assert ranges == res[1]["ranges"] and ranges[0][0] == 0 and ranges[0][1] == ranges[1][0] and ranges[1][1] == p.nk
    assert 0 < ranges[0][1] < p.nk
    # union of the two ranks' ordered terms == the single-rank two-sided store, as multisets
    h = ephc.build_channels(p, flags=ephc.HOST_ONLY)
    g = h.export_gather()
    full = np.stack([g[k] for k in ("dest", "partner", "iq", "nu", "kind", "diag")]).astype(np.int64)
    both = np.concatenate([res[0]["terms"], res[1]["terms"]], axis=1).astype(np.int64)
    wb = np.concatenate([res[0]["w"], res[1]["w"]])
    assert full.shape == both.shape
    of, ob = np.lexsort(full[::-1]), np.lexsort(both[::-1])
    assert np.array_equal(full[:, of], both[:, ob]) and np.array_equal(g["w"][of], wb[ob])
    # the exchanged pieces are the oracle's collision integral on both ranks; the 3-component exchange too
    Io = oracle.OracleList(p).collision(p.f, p.N)
    for r in range(world):
        assert np.abs(res[r]["I"] - Io).max() <= 1e-12 * np.abs(Io).max()
        s0 = ranges[0][1] * p.nb
        exp = np.tile(np.where(np.arange(p.ns) < s0, 1.0, 2.0), 3)
        assert np.array_equal(res[r]["F3"], exp)
        lo, hi = ranges[r][0] * p.nb, ranges[r][1] * p.nb
        assert np.all((res[r]["rows"] >= lo) & (res[r]["rows"] < hi))      # the row store is sharded with the gather store
