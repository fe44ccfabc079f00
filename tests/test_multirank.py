"""World-size-2 test of the N > 1 path on CPU (gloo): the event stream is sharded by Philox counter offset
(paper_2312_02898_b200.shard), ranks exchange nothing on the data path, and the max-over-ranks timing reduction of
bench.py works.  The sampler here is the oracle's (CPU); the GPU tests check the same offset property on the
CUDA sampler bit for bit."""
import os
import socket

import numpy as np
import pytest


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, nevt, out):
    import torch
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import paper_2312_02898_b200 as mg
    import workloads
    from oracle import oracle as O
    cfg = workloads.CONFIGS["ggttg"]
    first, n = mg.shard(nevt, rank, world)
    mom = O.load(False).rambo(cfg["seed"], n, cfg["masses_final"], cfg["sqrt_s"], first_event=first)
    gathered = [torch.zeros(mom.shape, dtype=torch.float64) for _ in range(world)]
    dist.all_gather(gathered, torch.from_numpy(mom))           # test-only exchange: the data path has none
    # batch-unweighting statistics of the shards: max / sum / sum of squares combine with one all-reduce
    orc = O.load(False)
    me = orc.me_batch(cfg["proc"], mom)
    prod, st = orc.weight_max(me, np.full(n, 2.0))
    st = mg.allreduce_weight_stats(torch.from_numpy(st.copy()))
    if rank == 0:
        np.save(out + ".stats", st.numpy())
    t = torch.tensor([0.5 + rank], dtype=torch.float64)        # per-rank timing -> max over ranks, as bench.py does
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.barrier()
    if rank == 0:
        np.save(out, np.concatenate([g.numpy() for g in gathered]))
        with open(out + ".t", "w") as fh:
            fh.write(repr(float(t[0])))
    dist.destroy_process_group()


def test_two_ranks_shard_the_event_stream(tmp_path):
    import torch.multiprocessing as mp
    import workloads
    from oracle import oracle as O
    world, nevt = 2, 257
    out = str(tmp_path / "gathered.npy")
    mp.spawn(_worker, args=(world, _free_port(), nevt, out), nprocs=world, join=True)
    cfg = workloads.CONFIGS["ggttg"]
    whole = O.load(False).rambo(cfg["seed"], world * nevt, cfg["masses_final"], cfg["sqrt_s"])
    assert np.array_equal(np.load(out), whole)
    assert float(open(out + ".t").read()) == 1.5
    orc = O.load(False)
    prod = 2.0 * orc.me_batch(cfg["proc"], whole)
    st = np.load(out + ".stats.npy")
    assert st[0] == prod.max() and abs(st[1] / prod.sum() - 1) < 1e-13 and abs(st[2] / (prod * prod).sum() - 1) < 1e-13


def test_shard_arguments():
    import paper_2312_02898_b200 as mg
    assert mg.shard(100, 0, 1) == (0, 100) and mg.shard(100, 3, 8) == (300, 100)
    with pytest.raises(ValueError):
        mg.shard(100, 2, 2)
