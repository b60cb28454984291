"""Host logic of the N-replica path on CPU: frame sharding and the max-over-ranks aggregation, world_size 2, gloo."""
import os
import socket

import pytest


def test_shard_frames_partitions_the_stream():
    from paper_1412_6367_b200.dist import shard_frames
    for total in (0, 1, 7, 1024, 1025):
        for world in (1, 2, 3, 8):
            blocks = [shard_frames(total, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == total
            for (a0, a1), (b0, b1) in zip(blocks, blocks[1:]):
                assert a1 == b0
            sizes = [b - a for a, b in blocks]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_frames(10, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    from paper_1412_6367_b200 import dist
    r, lr, w = dist.init(backend="gloo")
    start, stop = dist.shard_frames(101, r, w)
    dist.barrier()
    # rank 1 is "slower": the job time is the max, the job units the sum
    fps, ms = dist.aggregate_throughput(stop - start, 10.0 * (r + 1))
    q.put((r, start, stop, fps, ms))
    dist.finalize()


def test_two_rank_gloo_aggregation():
    import torch.multiprocessing as mp
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
    (r0, s0, e0, fps0, ms0), (r1, s1, e1, fps1, ms1) = res
    assert (s0, e0, s1, e1) == (0, 51, 51, 101)
    assert ms0 == ms1 == 20.0
    assert fps0 == fps1 == pytest.approx(101 / 0.020)
