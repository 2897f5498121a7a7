"""The N>1 path of bench.py on CPU: world_size 2 over gloo (one process per rank, 127.0.0.1 rendezvous)."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2606_15789_b200.dist import Ranks
    r = Ranks("gloo")
    r.barrier()
    t = 1.0 + rank                         # rank 1 is the slow one
    out[rank] = (r.max_over_ranks(t), r.aggregate(10.0, t), r.batch_seed(500))
    r.barrier()
    r.close()


def test_weak_scaling_timing_contract_world2():
    port = _free_port()
    with mp.Manager() as m:
        out = m.dict()
        mp.spawn(_worker, args=(2, port, out), nprocs=2, join=True)
        res = dict(out)
    assert res[0][0] == res[1][0] == 2.0                 # MAX over ranks
    assert res[0][1] == res[1][1] == 2 * 10.0 / 2.0      # whole-job units / slowest time
    assert res[0][2] != res[1][2]                        # each rank has its own batch


def test_single_process_is_identity():
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK"):
        os.environ.pop(k, None)
    from paper_2606_15789_b200.dist import Ranks
    r = Ranks()
    assert r.world == 1 and r.max_over_ranks(3.5) == 3.5 and r.aggregate(7.0, 2.0) == 3.5
