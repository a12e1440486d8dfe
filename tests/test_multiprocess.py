"""World-size-2 gloo test (CPU) of the N > 1 host logic of bench.py: the slices of a batch are
sharded over ranks with no data-path collective; only the timings are max-reduced and the
per-rank pieces, when gathered, are exactly the single-process batch."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2412_07631_b200 import workload as wl


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, S, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = wl.CONFIGS["c0"]
    lo, cnt = wl.shard_slices(S, rank, world)
    X0, B = wl.make_slices(cfg, S=lo + cnt)
    mine = torch.from_numpy(np.ascontiguousarray(B[:, lo:lo + cnt].T))      # (cnt, m)
    # what bench.py reduces: per-rank times -> max; per-rank slice counts -> sum
    t = torch.tensor([10.0 + rank, 5.0 - rank], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    n = torch.tensor([cnt], dtype=torch.int64)
    dist.all_reduce(n, op=dist.ReduceOp.SUM)
    pieces = [None] * world
    dist.all_gather_object(pieces, (lo, mine.numpy()))
    if rank == 0:
        out.put((t.tolist(), int(n.item()), pieces))
    dist.barrier()
    dist.destroy_process_group()


def test_slice_sharding_world2():
    S, world = 5, 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, S, q)) for r in range(world)]
    for p in procs:
        p.start()
    t, n, pieces = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert t == [11.0, 5.0] and n == S
    _, B = wl.make_slices(wl.CONFIGS["c0"], S=S)
    got = np.concatenate([pc for _, pc in sorted(pieces, key=lambda x: x[0])], axis=0).T
    assert np.array_equal(got, B)


def test_shard_slices_partition():
    for S in (0, 1, 7, 8, 1024):
        for world in (1, 2, 3, 8):
            spans = [wl.shard_slices(S, r, world) for r in range(world)]
            assert sum(c for _, c in spans) == S
            assert spans[0][0] == 0 and all(spans[i][0] + spans[i][1] == spans[i + 1][0] for i in range(world - 1))
            assert max(c for _, c in spans) - min(c for _, c in spans) <= 1
