"""World-size-2 CPU test (gloo) of the N>1 host logic: the path does not shard, so the only
cross-rank logic is the barrier + max-over-ranks timing + whole-job aggregation bench.py uses."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2602_06688_b200.replicas import Replicas
    r = Replicas(backend="gloo")
    r.barrier()
    # rank 0 took 2 s for 4 frames, rank 1 took 3 s for 4 frames
    secs = 2.0 + rank
    out = (r.rank, r.world, r.max_over_ranks(secs), r.sum_over_ranks(4.0),
           r.whole_job_throughput(4.0, secs), r.seed_offset())
    r.barrier()
    r.close()
    q.put(out)


def test_two_replicas_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(i, 2, port, q)) for i in range(2)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[0] for r in res] == [0, 1] and all(r[1] == 2 for r in res)
    for r in res:
        assert r[2] == 3.0            # slowest rank
        assert r[3] == 8.0            # frames of the whole job
        assert abs(r[4] - 8.0 / 3.0) < 1e-12
    assert res[0][5] != res[1][5]     # different sources per replica


def test_single_process_is_identity():
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    from paper_2602_06688_b200.replicas import Replicas
    r = Replicas()
    assert not r.distributed and r.max_over_ranks(1.5) == 1.5 and r.whole_job_throughput(3, 1.5) == 2.0
    r.barrier()
    r.close()
