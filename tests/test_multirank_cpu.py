"""World-size-2 gloo test of the benchmark's multi-rank host logic: frame ownership, the
strong-scaling tile split, and the max-over-ranks reduction behind the reported whole-job throughput."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2602_12949_b200 import dist as D


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        r, w, l = D.env_rank_world()
        frames = D.frame_of_rank(r, w)
        ms = 0.2 + 0.05 * rank                       # rank 1 is the slow one
        ms_max = D.reduce_max(ms)
        lo, hi = D.texel_range_of_rank(1920 * 1080, r, w)
        q.put((rank, frames, ms_max, lo, hi, D.whole_job_gqps(1920 * 1080, w, ms_max)))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
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
    assert [r[1] for r in res] == [[0], [1]]                       # one distinct frame per rank (weak scaling)
    assert all(abs(r[2] - 0.25) < 1e-12 for r in res)              # every rank sees the max
    assert res[0][3] == 0 and res[0][4] == res[1][3] and res[1][4] == 1920 * 1080   # contiguous, disjoint, complete
    assert res[0][4] % 128 == 0
    assert np.isclose(res[0][5], 2 * 1920 * 1080 / 0.25e-3 / 1e9)


def test_tile_split_covers_everything():
    for n in (1, 127, 128, 129, 2073600, 12345677):
        for world in (1, 2, 3, 8):
            spans = [D.texel_range_of_rank(n, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            for a, b in zip(spans, spans[1:]):
                assert a[1] == b[0] and a[0] <= a[1]
            assert all(s[0] % 128 == 0 for s in spans)


def test_single_process_defaults(monkeypatch):
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        monkeypatch.delenv(k, raising=False)
    assert D.env_rank_world() == (0, 1, 0)
    assert D.reduce_max(1.5) == 1.5
    with pytest.raises(ValueError):
        D.frame_of_rank(2, 2)


def test_bench_launches_its_own_ranks_and_broadcasts_the_parameters():
    """`python bench.py --gpus 2` outside torchrun starts two ranks itself (torch.distributed.run, 127.0.0.1); --dry runs
    the plumbing of the GPU arm over gloo: parameters built on rank 0 only and broadcast, weak / strong split, max over
    ranks, ONE JSON line."""
    import json
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    for scaling, per_rank, total in (("weak", [4096, 4096], 8192), ("strong", [2048, 2048], 4096)):
        res = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--dry", "--scaling", scaling],
                             capture_output=True, text=True, env=env, timeout=600)
        assert res.returncode == 0, res.stderr[-3000:]
        lines = [l for l in res.stdout.splitlines() if l.startswith("{")]
        assert len(lines) == 1, res.stdout
        d = json.loads(lines[0])
        assert d["dry"] is True and d["n_gpus"] == 2 and d["scaling"] == scaling
        assert d["texels_per_rank"] == per_rank and d["texels_per_step"] == total
        assert d["param_checksums"][0] == d["param_checksums"][1] != 0.0            # rank 1 got rank 0's parameters
        assert d["value"] > 0


def test_row_split_covers_the_image():
    for h in (1, 3, 4, 5, 540, 1080, 2160, 4099):
        for world in (1, 2, 3, 8):
            spans = [D.row_range_of_rank(h, r, world) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == h
            for a, b in zip(spans, spans[1:]):
                assert a[1] == b[0] and a[0] <= a[1]
            assert all(s[0] % 4 == 0 for s in spans)
