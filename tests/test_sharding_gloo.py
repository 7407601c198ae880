"""world_size-2 gloo test of the multi-GPU host logic on CPU: two ranks trace disjoint id shards
(with the oracle standing in for the device), merge with the product's reduction, and rank 0 must
hold exactly the single-range result."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, n_total, ret):
    sys.path.insert(0, ROOT)
    import sas_workloads as W
    from oracle import oracle as O
    from paper_2501_06054_b200.sharding import shard_ids, merge_detectors
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    c = W.config(0)
    first, n = shard_ids(n_total, rank, world)
    out = O.trace_range(c["instrument"], c["model"], c["seed"], first, n, dump=False)
    ts = [torch.from_numpy(out["sum_p"]), torch.from_numpy(out["sum_p2"]),
          torch.from_numpy(out["counts"].astype(np.int64))]
    merge_detectors(ts, dst=0)
    if rank == 0:
        ret["sum_p"], ret["counts"] = ts[0].numpy().copy(), ts[2].numpy().copy()
    ret[f"range{rank}"] = (first, n)
    dist.destroy_process_group()


def test_two_rank_shards_merge_to_the_single_range_result():
    import sas_workloads as W
    from oracle import oracle as O
    n_total = 60001
    mgr = mp.Manager()
    ret = mgr.dict()
    port = 29500 + os.getpid() % 2000
    mp.spawn(_worker, args=(2, port, n_total, ret), nprocs=2, join=True)
    c = W.config(0)
    ref = O.trace_range(c["instrument"], c["model"], c["seed"], 0, n_total, dump=False)
    assert ret["range0"] == (0, 30001) and ret["range1"] == (30001, 30000)
    assert np.array_equal(ret["counts"], ref["counts"].astype(np.int64))
    assert np.allclose(ret["sum_p"], ref["sum_p"], rtol=1e-13, atol=0)


def _batch_worker(rank, world, port, n_each, ret):
    sys.path.insert(0, ROOT)
    import sas_workloads as W
    from oracle import oracle as O
    from paper_2501_06054_b200.sharding import shard_ids, merge_detectors
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    c = W.batch_config(12, n_each, 20250110)
    first, n = shard_ids(n_each, rank, world)          # the id range this rank passes to sas_trace_batch_range
    sp, cn = [], []
    for e in range(12):
        out = O.trace_range(c["instruments"][e], c["models"][e], c["seed"], first, n, exp_index=e, dump=False)
        sp.append(out["sum_p"])
        cn.append(out["counts"].astype(np.int64))
    ts = [torch.from_numpy(np.stack(sp)), torch.from_numpy(np.stack(cn))]
    merge_detectors(ts, dst=0)
    if rank == 0:
        ret["sum_p"], ret["counts"] = ts[0].numpy().copy(), ts[1].numpy().copy()
    dist.destroy_process_group()


def test_two_rank_batch_shards_merge_to_the_single_range_result():
    """The batched path shards by id range like a single experiment (sas_trace_batch_range):
    the union of the two ranks' ranges of each of 12 experiments is the one-range detector, exactly in N."""
    import sas_workloads as W
    from oracle import oracle as O
    n_each = 20001
    mgr = mp.Manager()
    ret = mgr.dict()
    port = 31500 + os.getpid() % 2000
    mp.spawn(_batch_worker, args=(2, port, n_each, ret), nprocs=2, join=True)
    c = W.batch_config(12, n_each, 20250110)
    for e in range(12):
        ref = O.trace_range(c["instruments"][e], c["models"][e], c["seed"], 0, n_each, exp_index=e, dump=False)
        assert np.array_equal(ret["counts"][e], ref["counts"].astype(np.int64)), e
        assert np.allclose(ret["sum_p"][e], ref["sum_p"], rtol=1e-13, atol=0), e


def test_shard_ids_cover_the_range_exactly():
    from paper_2501_06054_b200.sharding import shard_ids, weak_shard
    for n, w in ((10, 3), (7, 8), (10**9, 8), (0, 2)):
        spans = [shard_ids(n, r, w) for r in range(w)]
        assert spans[0][0] == 0 and sum(s[1] for s in spans) == n
        for a, b in zip(spans, spans[1:]):
            assert a[0] + a[1] == b[0]
    assert weak_shard(100, 3) == (300, 100)
