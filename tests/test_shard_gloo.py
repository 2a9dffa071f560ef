"""CPU tests of the N > 1 path's host logic: window / time partition, shard-edge run merging against
the oracle's clustering of the whole stream, and a world_size-2 gloo run of the reduce / gather steps bench.py uses."""
import os
import socket
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from gwsynth import rng
from oracle import gwo
from paper_2201_11133_b200 import shard


def test_plan_windows_covers_once():
    for n, w in [(1024, 1), (1024, 8), (7, 3), (2, 4), (0, 2)]:
        p = shard.plan_windows(n, w)
        assert len(p) == w and p[0][0] == 0 and p[-1][1] == n
        assert all(a[1] == b[0] for a, b in zip(p, p[1:]))
        assert max(e - s for s, e in p) - min(e - s for s, e in p) <= 1


def test_plan_time_warmup_and_alignment():
    sh = shard.plan_time(14745600, 4, receptive_field=2047, max_lag=32 * 4096, align=4096)
    assert sh[0].start == 0 and sh[-1].end == 14745600 and sh[0].warm_start == 0
    for a, b in zip(sh, sh[1:]):
        assert a.end == b.start and b.start % 4096 == 0
        assert b.warm_start == b.start - 2046 and b.l1_start == max(0, b.warm_start - 32 * 4096)


def _runs(pbar, theta, lmin, t0=0):
    n, recs = gwo.triggers(pbar, theta, lmin, t0=t0, cap=1 << 16)
    assert n == len(recs)
    return [(r[1], r[2]) for r in recs]


def test_merge_shard_runs_equals_unsharded_oracle():
    N = 50000
    base = rng.uniform01(3, 0, np.arange(N // 37 + 1, dtype=np.uint64))
    pbar = np.repeat(np.where(base < 0.45, 0.2, 0.8), 37)[:N].astype(np.float64)
    for world in (2, 3, 7):
        for lmin in (1, 50, 200):
            want = _runs(pbar, 0.5, lmin)
            bounds = [(s.start, s.end) for s in shard.plan_time(N, world, receptive_field=16, align=1)]
            per = [_runs(pbar[a:b], 0.5, 1, t0=a) for a, b in bounds]
            assert shard.merge_shard_runs(per, bounds, lmin) == want
    # a run that spans a whole shard and both its edges
    pbar[:] = 0.2
    pbar[100:40000] = 0.9
    bounds = [(s.start, s.end) for s in shard.plan_time(N, 5, receptive_field=16)]
    per = [_runs(pbar[a:b], 0.5, 1, t0=a) for a, b in bounds]
    assert shard.merge_shard_runs(per, bounds, 2048) == [(100, 40000)]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        mine = shard.plan_windows(1024, world)[rank]
        t = shard.reduce_step_time(10.0 + rank, dist)                     # max over ranks
        N = 20000
        pbar = np.full(N, 0.2)
        pbar[9000:11500] = 0.9                                            # crosses the edge between the two ranks
        b = [(s.start, s.end) for s in shard.plan_time(N, world, receptive_field=16)]
        n, recs = gwo.triggers(pbar[b[rank][0]:b[rank][1]], 0.5, 1, t0=b[rank][0])
        allruns = shard.gather_objects([(r[1], r[2]) for r in recs], dist)
        merged = shard.merge_shard_runs(allruns, b, 2048)
        q.put((rank, mine, t, merged))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo():
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got[0][1] == (0, 512) and got[1][1] == (512, 1024)
    assert got[0][2] == got[1][2] == 11.0
    assert got[0][3] == got[1][3] == [(9000, 11500)]


def test_shard_stream_args_and_edge_merge():
    a = shard.shard_stream_args(1000, 0, 400, receptive_field=16, max_lag=100)
    assert a["shard"] == (0, 0) and a["n_total"] == 400 and a["tail_indices"][0] == 1000 - 115 and a["tail_indices"][-1] == 999
    b = shard.shard_stream_args(1000, 400, 1000, receptive_field=16, max_lag=100)
    assert b["shard"] == (400, 15) and b["first_pushed"] == 385 and b["n_total"] == 615
    assert b["tail_indices"] == list(range(385 - 115, 385))
    c = shard.shard_stream_args(128 * 100, 128 * 50, 128 * 100, receptive_field=2047, max_lag=4096, align=128)
    assert c["shard"] == (6400, 2048) and c["n_total"] % 128 == 0
    L, R = shard.EDGE_LEFT, shard.EDGE_RIGHT
    recs = [(0, 390, 400, 0.9, 0.8, 1 | R), (0, 400, 450, 0.7, 0.6, 2 | L),          # joined: 60 samples
            (0, 100, 130, 0.9, 0.9, 3),                                              # an inner run, long enough
            (0, 0, 5, 0.9, 0.9, 1 | L),                                              # touches the stream start, too short
            (1, 395, 400, 0.9, 0.9, 1 | R), (1, 400, 600, 0.8, 0.8, 1 | L | R), (1, 600, 610, 0.6, 0.6, 4 | L),   # three shards
            (2, 390, 400, 0.9, 0.9, 1 | R), (2, 401, 450, 0.9, 0.9, 1)]              # not adjacent: not joined
    got = shard.merge_edge_records(recs, 30)
    assert [(r[0], r[1], r[2], r[5]) for r in got] == [(0, 100, 130, 3), (0, 390, 450, 3), (1, 395, 610, 5), (2, 401, 450, 1)]
    assert abs(got[1][4] - (0.8 * 10 + 0.6 * 50) / 60) < 1e-12 and got[1][3] == 0.9
