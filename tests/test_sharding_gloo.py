"""N > 1 host logic on CPU: world_size-2 `gloo` process group (samples shard across ranks with
no data-path collective; only timing/flags are reduced)."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2607_00095_b200 import sharding as SH  # noqa: E402


def test_shard_range_partitions_exactly():
    for total in (0, 1, 2, 7, 1024, 1025):
        for world in (1, 2, 3, 8):
            spans = [SH.shard_range(total, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == total
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [hi - lo for lo, hi in spans]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        SH.shard_range(4, 2, 2)
    assert SH.throughput(2048, 3, 6.0) == pytest.approx(2048 * 3 / 6e-3)
    assert SH.reduce_timing(None, None, 2.5, 10, True) == (2.5, 10, True)


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, total: int, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        dev = torch.device("cpu")
        lo, hi = SH.shard_range(total, rank, world)
        # each rank "projects" its slice: the result of sample b is a function of b only (block independence)
        local = (torch.arange(lo, hi, dtype=torch.float64)[:, None] * torch.ones(1, 3, dtype=torch.float64)) ** 2
        full = SH.gather_slices(dist, dev, local, total, rank, world)
        dist.barrier()
        ms, units, ok = SH.reduce_timing(dist, dev, 10.0 + 5.0 * rank, hi - lo, rank != 1)
        ms2, units2, ok2 = SH.reduce_timing(dist, dev, 1.0, hi - lo, True)
        q.put((rank, full.tolist(), ms, units, ok, ms2, units2, ok2, SH.rank_seed(1005, rank)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("total", [5, 8])
def test_world_size_2_gloo(total):
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, total, q)) for r in range(world)]
    for p in procs:
        p.start()
    outs = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    expect = [[float(b * b)] * 3 for b in range(total)]
    for rank, full, ms, units, ok, ms2, units2, ok2, seed in outs:
        assert full == expect                      # every rank sees all slices, in order, unpadded
        assert ms == 15.0 and units == total       # max over ranks, sum over ranks
        assert ok is False                         # one rank reported non-convergence
        assert (ms2, units2, ok2) == (1.0, total, True)
        assert seed == 1005 + 1000 * rank


def test_bench_gpus_flag_self_launches_ranks_and_reduces_through_sharding():
    """`python bench.py --gpus 2` with no torchrun environment re-execs itself under torch.distributed.run and
    reduces through sharding.reduce_timing — exercised here on CPU (gloo, no GPU work)."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--backend", "gloo", "--selftest-dist"],
                         capture_output=True, text=True, timeout=300, env=env)
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                                    # rank 0 alone prints
    rec = json.loads(lines[0])
    assert rec["n_gpus"] == 2 and rec["units"] == 200 and rec["max_ms"] == 11.0 and rec["ok"] is True
