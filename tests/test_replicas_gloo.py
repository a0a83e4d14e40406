"""N > 1 host logic on CPU: two gloo ranks, max-over-ranks timing and whole-job aggregation."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    import torch.distributed as dist
    from paper_2510_13726_b200 import replicas as R
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ms_local = 10.0 + 5.0 * rank          # rank 1 is the slow one
    dist.barrier()
    ms = R.max_over_ranks(ms_local)
    out[rank] = (ms, R.aggregate_mlups(1000, 20, ms, world))
    dist.destroy_process_group()


def test_two_rank_aggregation():
    world, port = 2, _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 15.0
    assert abs(res[0][1] - 2 * 1000 * 20 / 15e3) < 1e-12


def test_single_process_identity():
    from paper_2510_13726_b200 import replicas as R
    assert R.max_over_ranks(3.5) == 3.5
    assert R.aggregate_mlups(10 ** 6, 10, 1.0, 1) == 10 ** 4
