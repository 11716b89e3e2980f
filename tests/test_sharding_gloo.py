"""world_size-2 (and 3) gloo tests of the multi-GPU host logic on CPU: contiguous sharding covers
every unit exactly once, and the cross-rank "best hypothesis" pick equals the single-process result.
Per-rank results come from the oracle (this is test infrastructure: no GPU here)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import hg_workloads as W
from paper_2402_18008_b200.sharding import combine_best, shard_range


def test_shard_range_partitions():
    for n in (0, 1, 7, 64, 1 << 20, (1 << 26) + 3):
        for world in (1, 2, 3, 8):
            edges = [shard_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            for a, b in zip(edges[:-1], edges[1:]):
                assert a[1] == b[0]
            sizes = [e - b for b, e in edges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(10, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_hyp, tie, q):
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = W.ransac_workload(n_pts=256, n_hyp=n_hyp, seed=99)
        idx = wl["hyp_idx"].numpy()
        if tie:                                    # the global best also appears in the last shard
            full = oracle.ransac(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), idx, 3.0)
            idx = np.concatenate([idx, idx[full["best_index"]][None]], axis=0)
        b, e = shard_range(idx.shape[0], rank, world)
        out = oracle.ransac(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), idx[b:e], 3.0)
        gi = out["best_index"] + b if out["best_index"] >= 0 else -1
        cnt, gidx, H = combine_best(torch.tensor([out["best_count"]], dtype=torch.int32),
                                    torch.tensor([gi], dtype=torch.int64),
                                    torch.from_numpy(out["best_H"]).to(torch.float32))
        ref = oracle.ransac(wl["src_xy"].numpy(), wl["dst_xy"].numpy(), idx, 3.0)
        ok = (int(cnt) == ref["best_count"] and int(gidx) == ref["best_index"]
              and np.allclose(H.numpy(), ref["best_H"], atol=1e-6) if ref["best_index"] >= 0 else int(gidx) == -1)
        q.put((rank, bool(ok), int(cnt), int(gidx)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,n_hyp,tie", [(2, 300, False), (2, 300, True), (3, 2, False)])
def test_combine_best_over_gloo(world, n_hyp, tie):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_hyp, tie, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = [q.get(timeout=180) for _ in range(world)]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(r[1] for r in res), res
    assert len({(r[2], r[3]) for r in res}) == 1           # every rank holds the same answer


def test_bench_gpus_n_starts_n_ranks_or_fails_loudly():
    """bench.py --gpus N (launch logic only, no GPU): without a launcher and N > 1 it re-executes itself under
    torch.distributed.run with N ranks on 127.0.0.1; it refuses when fewer than N devices exist (a 1-GPU box must not print an
    n_gpus: 1 line for --gpus 2); a launcher's WORLD_SIZE is respected and must agree with --gpus."""
    import argparse
    import sys
    import bench
    a = lambda gpus, impl="ours": argparse.Namespace(gpus=gpus, impl=impl)
    argv = ["--gpus", "2", "--steps", "3", "--warmup", "3"]
    cmd = bench.self_launch_if_needed(a(2), argv, env={}, device_count=8)
    assert cmd[:3] == [sys.executable, "-m", "torch.distributed.run"] and "--nnodes=1" in cmd
    assert cmd[cmd.index("--nproc-per-node") + 1] == "2" and cmd[cmd.index("--master-addr") + 1] == "127.0.0.1"
    assert 0 < int(cmd[cmd.index("--master-port") + 1]) < 65536
    assert cmd[-len(argv) - 1].endswith("bench.py") and cmd[-len(argv):] == argv
    assert bench.self_launch_if_needed(a(1), ["--gpus", "1"], env={}, device_count=1) is None            # one GPU: this process
    assert bench.self_launch_if_needed(a(2), argv, env={"WORLD_SIZE": "2"}, device_count=8) is None       # already launched
    assert bench.self_launch_if_needed(a(4, "reference"), argv, env={}, device_count=0) is None           # the oracle arm: rank 0 only
    with pytest.raises(SystemExit) as e:
        bench.self_launch_if_needed(a(2), argv, env={}, device_count=1)
    assert "only 1 CUDA device" in str(e.value)
    with pytest.raises(SystemExit):
        bench.self_launch_if_needed(a(8), argv, env={"WORLD_SIZE": "2"}, device_count=8)
