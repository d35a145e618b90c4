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


@pytest.mark.timeout(300)
def test_bench_gpus_2_starts_two_ranks_itself():
    # `bench.py --gpus 2` WITHOUT a launcher environment must start the two ranks itself (torch.distributed.run on 127.0.0.1)
    # and report n_gpus = the ranks that ran; --dry-run takes the same launcher and sharding path with gloo and no kernels
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--dry-run", "--config", "0"],
                         capture_output=True, text=True, env=env, timeout=280)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads([x for x in out.stdout.splitlines() if x.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["dry_run"] is True
    B = 32
    assert [r[:3] for r in line["shards"]] == [[0, 0, B], [1, B, 2 * B]]
    assert line["shards"][0][3] != line["shards"][1][3]                       # the ranks hold different chains
    assert line["config"]["parallelism"] == "chains sharded x2"
    # one rank: no launcher, n_gpus 1
    out1 = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "1", "--dry-run", "--config", "0"],
                          capture_output=True, text=True, env=env, timeout=120)
    l1 = json.loads([x for x in out1.stdout.splitlines() if x.startswith("{")][-1])
    assert l1["n_gpus"] == 1 and l1["shards"] == [line["shards"][0]]
