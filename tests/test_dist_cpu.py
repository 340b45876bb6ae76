"""Host-side plumbing of `bench.py --gpus N` on CPU: two gloo ranks.

The path shards by whole frames with no data-path collective; what crosses ranks is control only:
a barrier on both sides of the timed region, a MAX over the per-rank device times and SUMs of the
units processed.  These tests run that plumbing with world_size 2 over gloo on 127.0.0.1, and the
reference arm's "rank 0 alone prints" rule through the real bench.py entry point."""
import json
import os
import socket
import subprocess
import sys

import pytest
import torch.multiprocessing as mp

from paper_1001_4309_b200 import dist as D
from paper_1001_4309_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      LOCAL_RANK=str(rank), WORLD_SIZE=str(world))
    info = D.rank_info()
    assert (info.rank, info.local_rank, info.world) == (rank, rank, world)
    assert D.init(info, "gloo") is True
    D.barrier(info)
    # rank r "processes" its shard of 7 frames of 4 views in (r + 1) * 0.5 s
    lo, hi = D.shard_range(7, info.rank, info.world)
    units = (hi - lo) * 4
    secs = 0.5 * (rank + 1)
    total, slowest, value = D.aggregate_throughput(info, units, secs)
    mx = D.max_over_ranks(info, float(rank))
    sm = D.sum_over_ranks(info, 10.0 + rank)
    D.barrier(info)
    D.finalize(info)
    out.put((rank, lo, hi, total, slowest, value, mx, sm))


def test_two_gloo_ranks_aggregate_like_bench():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, lo0, hi0, *a0), (r1, lo1, hi1, *a1) = res
    assert (lo0, hi0, lo1, hi1) == (0, 4, 4, 7)            # block partition, first rank takes the extra
    assert a0 == a1                                         # every rank sees the same aggregates
    total, slowest, value, mx, sm = a0
    assert total == 28.0 and slowest == 1.0 and value == 28.0   # all units / slowest rank's time
    assert mx == 1.0 and sm == 21.0


def test_single_rank_needs_no_process_group():
    info = D.rank_info({})
    assert info.world == 1 and info.is_root
    assert D.init(info, "gloo") is False
    D.barrier(info)
    assert D.aggregate_throughput(info, 8, 2.0) == (8.0, 2.0, 4.0)
    D.finalize(info)


@pytest.mark.parametrize("n,world", [(256, 2), (7, 4), (3, 8), (0, 2)])
def test_shard_range_partitions_every_unit_once(n, world):
    seen = []
    for r in range(world):
        lo, hi = W.shard_range(n, r, world)
        assert 0 <= lo <= hi <= n
        seen.extend(range(lo, hi))
    assert seen == list(range(n))
    sizes = [W.shard_range(n, r, world)[1] - W.shard_range(n, r, world)[0] for r in range(world)]
    assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        W.shard_range(n, world, world)


def _json_lines(text):
    return [json.loads(l) for l in text.splitlines() if l.startswith("{")]


def test_bare_bench_starts_its_own_ranks():
    """`python bench.py --impl reference --gpus 2` with no WORLD_SIZE in the environment launches two
    ranks itself (one process each, rendezvous on 127.0.0.1); both join the process group, rank 0 alone
    works and prints ONE JSON line, rank 1 exits 0 without output."""
    env = {k: v for k, v in os.environ.items()
           if k not in ("RANK", "LOCAL_RANK", "WORLD_SIZE", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--steps", "2", "--warmup", "1", "--config", "1"],
                       env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr
    lines = _json_lines(r.stdout)
    assert len(lines) == 1
    line = lines[0]
    assert line["impl"] == "reference" and line["n_gpus"] == 2 and line["ranks_joined"] == 2
    assert line["unit"] == "reconstructions/s" and line["value"] > 0
    assert line["cpu_baseline"]["kind"] == "oracle" and "caveat" in line["cpu_baseline"]
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["gpu_launches"] == 0


def test_reference_arm_under_a_torchrun_style_launch():
    """The driver's launch: every rank started with RANK / WORLD_SIZE / MASTER_* in its environment.
    Rank 1 joins, waits for rank 0 and exits 0 with empty stdout; rank 0 prints the line."""
    port = _free_port()
    procs = []
    for rank in (0, 1):
        env = dict(os.environ, RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference",
                                       "--gpus", "2", "--steps", "1", "--warmup", "0", "--config", "1"],
                                      env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    outs = [p.communicate(timeout=600) for p in procs]
    assert [p.returncode for p in procs] == [0, 0], outs
    assert outs[1][0].strip() == ""
    line = _json_lines(outs[0][0])[-1]
    assert line["impl"] == "reference" and line["ranks_joined"] == 2


def test_world_size_must_match_gpus():
    env = dict(os.environ, RANK="0", LOCAL_RANK="0", WORLD_SIZE="3", MASTER_ADDR="127.0.0.1",
               MASTER_PORT=str(_free_port()))
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2"],
                       env=env, capture_output=True, text=True, timeout=120)
    assert r.returncode != 0 and "WORLD_SIZE" in (r.stderr + r.stdout)
