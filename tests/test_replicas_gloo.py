"""N > 1 is "replicas only": ranks share nothing on the data path; the only
cross-rank step of bench.py is the max-over-ranks time and the whole-job sum.  Covered here with
world_size 2 on the gloo backend (CPU)."""
import os
import socket
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    import bench
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        # rank r measured (r + 1) * 2 ms for the same per-rank work
        ms = bench.max_over_ranks(2.0 * (rank + 1), world, device="cpu")
        out.put((rank, ms, bench.aggregate_value(10**9, world, ms * 1e-3)))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_replicas_world2_max_time_and_aggregate():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=100) for _ in procs)
    for p in procs:
        p.join(timeout=30)
        assert p.exitcode == 0
    for rank, ms, gflops in res:
        assert ms == 4.0                      # the slowest rank's time, on every rank
        assert gflops == pytest.approx(2 * 1.0 / 4e-3)  # 2 ranks x 1 Gadd / 4 ms


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(3.5, 1) == 3.5
    assert bench.aggregate_value(2 * 10**9, 1, 1.0) == 2.0


def test_gpus_flag_must_agree_with_the_launcher():
    """`python bench.py --gpus 8` without torchrun would silently time one GPU: refused."""
    sys.path.insert(0, ROOT)
    import bench
    bench.check_world(1, 1)
    bench.check_world(4, 4)
    with pytest.raises(SystemExit):
        bench.check_world(8, 1)
