"""N>1 host logic of bench.py on CPU: world_size-2 gloo (batch-sharded replicas, no
data-path collective).  Checks the max-over-ranks timing reduction, the per-rank seed split and that
the two ranks' shards are distinct slices of the job."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import gspn_inputs as gi
    from dataclasses import replace
    # timing reduction: the job's time is the slowest rank's
    t = bench.max_over_ranks(10.0 + rank, world, torch.device("cpu"))
    # weak scaling: every rank owns B images drawn from its own seed (bench.main: seed + 1000*rank)
    base = gi.small_config("dist", 2, 4, 6, 5, 2, seed=7)
    cfg = replace(base, seed=base.seed + 1000 * rank)
    x = gi.make_inputs(cfg, "f32")["x"]
    gathered = [torch.empty_like(x) for _ in range(world)]
    dist.all_gather(gathered, x)
    units = torch.tensor([cfg.n], dtype=torch.int64)
    dist.all_reduce(units)
    if rank == 0:
        out.put((t, bool(torch.equal(gathered[0], gathered[1])), int(units.item()), base.n))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_two_rank_gloo_timing_and_sharding():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = out.get(timeout=100)
    for p in procs:
        p.join(30)
        assert p.exitcode == 0
    t, same, units, n = res
    assert t == 11.0                 # max over ranks
    assert not same                  # ranks hold different shards
    assert units == 2 * n            # whole-job units = sum over ranks
