"""Host-side logic of the N>1 path on CPU: gloo, world size 2.  Each rank runs the oracle on its
shard of config 1 (the GPU path shards the same way in bench.py), the counters are all-reduced,
and the result must equal the single-rank histogram bit for bit."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, mode, out):
    for p in (ROOT, os.path.join(ROOT, "oracle")):
        if p not in sys.path:
            sys.path.insert(0, p)
    import oracle as orc
    from paper_2506_15812_b200 import sharding, workloads as wl
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = sharding.shard_config(wl.config(1, n_override=1001), rank, world, mode)
    res = orc.run_config(cfg, nthreads=1)
    counts = torch.from_numpy(res["counts"].astype(np.int64))
    summary = torch.from_numpy(res["summary"].astype(np.int64))
    sharding.allreduce_counters(dist, counts, summary)
    if rank == 0:
        np.save(out, np.concatenate([counts.numpy().ravel(), summary.numpy().ravel()]))
    dist.barrier()
    dist.destroy_process_group()


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_strong_sharding_reproduces_single_rank_histogram(tmp_path):
    import oracle as orc
    from paper_2506_15812_b200 import sharding, workloads as wl
    out = str(tmp_path / "r.npy")
    mp.spawn(_worker, args=(2, _free_port(), "strong", out), nprocs=2, join=True)
    got = np.load(out)
    ref = orc.run_config(wl.config(1, n_override=1001), nthreads=1)
    exp = np.concatenate([ref["counts"].astype(np.int64).ravel(), ref["summary"].astype(np.int64).ravel()])
    assert np.array_equal(got, exp)
    # the shards tile the index range exactly
    a, b = (sharding.shard_config(wl.config(1, n_override=1001), r, 2, "strong").groups[0] for r in (0, 1))
    assert a.first_index == 0 and a.n_ions + b.n_ions == 1001 and b.first_index == a.n_ions


def test_weak_sharding_uses_disjoint_counters(tmp_path):
    import oracle as orc
    from paper_2506_15812_b200 import sharding, workloads as wl
    out = str(tmp_path / "r.npy")
    mp.spawn(_worker, args=(2, _free_port(), "weak", out), nprocs=2, join=True)
    got = np.load(out)
    tot = np.zeros_like(got)
    for r in (0, 1):
        cfg = sharding.shard_config(wl.config(1, n_override=1001), r, 2, "weak")
        assert cfg.groups[0].first_index == r << 40
        ref = orc.run_config(cfg, nthreads=1)
        tot += np.concatenate([ref["counts"].astype(np.int64).ravel(), ref["summary"].astype(np.int64).ravel()])
    assert np.array_equal(got, tot)
    assert got[-6:-1].sum() == 2 * 1001          # counting invariant over both ranks
