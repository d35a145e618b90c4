"""Multi-GPU path on CPU (world size 2, gloo): the path shards by chain with no data-path collective
(DESIGN.md "Multi-GPU"), so what there is to test is the host logic of bench.py:
rank r must get exactly rows [r B, (r+1) B) of the world*B batch (states, chain ids that key the RNG,
per-chain temperatures), and the reported rate must be all ranks' proposals over the MAX of the ranks' times."""
import dataclasses
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    import amh_inputs as gi
    import bench
    dist.init_process_group("gloo", init_method="tcp://127.0.0.1:%d" % port, rank=rank, world_size=world)
    try:
        for cid in (0, 4):
            cfg = dataclasses.replace(gi.CONFIGS[cid], B=6, L=10)
            off, s0, kw = bench.shard(cfg, rank, world)
            assert off == rank * cfg.B and kw["chain_offset"] == off
            mine = torch.from_numpy(s0)
            parts = [torch.empty_like(mine) for _ in range(world)]
            dist.all_gather(parts, mine)
            whole = gi.initial_states(world * cfg.B, cfg.n, seed=1)           # what one GPU would run
            assert np.array_equal(torch.cat(parts).numpy(), whole)
            if cfg.replicas:
                t = torch.from_numpy(kw["per_chain_T"])
                tp = [torch.empty_like(t) for _ in range(world)]
                dist.all_gather(tp, t)
                assert np.array_equal(torch.cat(tp).numpy(),
                                      gi.per_chain_temperature(world * cfg.B, cfg.replicas, cfg.t_start, cfg.t_end))
        # timing: max over ranks, whole-job units
        ms = torch.tensor([100.0 * (rank + 1)], dtype=torch.float64)
        dist.all_reduce(ms, op=dist.ReduceOp.MAX)
        assert ms.item() == 100.0 * world
        rate = bench.job_rate(world, 1000, 2, ms.item())
        assert abs(rate - world * 1000 * 2 / (0.1 * world)) < 1e-9
        q.put((rank, "ok"))
    except Exception as e:                                                     # pragma: no cover
        q.put((rank, repr(e)))
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(180)
def test_chain_sharding_world_size_2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=150) for _ in procs)
    for p in procs:
        p.join(timeout=30)
    assert res == {0: "ok", 1: "ok"}, res
