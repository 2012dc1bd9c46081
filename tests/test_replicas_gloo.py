"""N > 1 path (replicas only): the cross-rank reduction bench.py uses, run with
two gloo processes on CPU."""
import os
import socket

import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1104_3998_b200 import replicas as R
from paper_1104_3998_b200 import workloads as W


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p = W.make_params(0)
    p["seed"] = R.replica_seed(p["seed"], rank)
    parts = W.make_particles(p)
    n_local = sum(a[0].shape[0] for a in parts)
    ms, n = R.reduce_replicas(10.0 + 5.0 * rank, n_local)
    q.put((rank, ms, n, float(parts[0][0][0]), R.throughput(n, 4, ms)))
    dist.destroy_process_group()


def test_two_replicas_reduce_max_time_and_sum_units():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    n1 = 2 * 128 * 64
    for rank, ms, n, x0, thr in res:
        assert ms == 15.0 and n == 2 * n1
        assert abs(thr - 2 * n1 * 4 / 15e-3) < 1e-6 * thr
    assert res[0][3] != res[1][3]          # different seeds: independent replicas


def test_single_process_is_identity():
    assert R.reduce_replicas(3.0, 7) == (3.0, 7.0)
