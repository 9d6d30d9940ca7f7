"""The N > 1 path of bench.py on CPU: world_size-2 gloo processes run its distributed plumbing (rendezvous on
127.0.0.1, barrier, max-over-ranks timing, batch sharding with no data-path collective)."""
import os
import socket
import sys

import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import bench
    r, w = bench.dist_init("gloo")
    assert (r, w) == (rank, world) and bench.dist_env() == (rank, rank, world)
    per, total = bench.shard_units(4, w)
    bench.barrier(w)
    slowest = bench.max_over_ranks(10.0 + 5.0 * rank, w)       # rank 1 is the slow one
    bench.barrier(w)
    q.put((rank, per, total, slowest))
    import torch.distributed as dist
    dist.destroy_process_group()


def test_world2_gloo_max_over_ranks_and_sharding():
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
    assert res == [(0, 4, 8, 15.0), (1, 4, 8, 15.0)]


def test_single_process_plumbing_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.shard_units(4, 1) == (4, 4)
    bf, units, byt, comp = bench.work_model(1 << 16, 1240, 1240, 39, 78, 81, 121, 4)
    assert comp == 4 * 65536 * 4 * 6 * 39 + 65536 * 4 * 2 * 121
    # every transform has N/2 log2 N butterflies: 8 of the 16 stages in the column passes, 8 in the fused rows
    transforms = 4 * ((4 * 81 + 121) + (3 * 81 + 2 * 121))
    assert sum(bf.values()) == transforms * 32768 * 16
    assert bf["pointwise"] == bf["ntt_fwd"] + bf["ntt_inv"]
    assert all(v >= 0 for v in units.values()) and all(v >= 0 for v in byt.values())
