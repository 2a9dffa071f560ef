"""Time shards through gwi_stream_* (-m gpu): SURVEY.md section 8(e), PAPER.md:63 (one rank per GPU, the data sharded).

Every "rank" runs its span of one stream through its own gwi_stream handle in shard mode (include/gwi.h:
gwi_stream_set_shard): R_f - 1 warm-up samples in front, the slides primed with the L1 samples that precede the span
in the GLOBAL stream, runs that touch a shard edge reported whatever their length.  The ranks' records, joined by
shard.merge_edge_records, must be the unsharded stream's list exactly, and every kept probability must equal the
unsharded one bit for bit.  The ranks run one after the other on cuda:0 (they do not wait on one another); the
world_size-2 process-group plumbing of the same helpers is tested on CPU in tests/test_shard_gloo.py.
"""
import os

import numpy as np
import pytest

import gwsynth as gs
from oracle import gwo
from paper_2201_11133_b200 import shard
from tests.helpers import trig_tuples
from tests.test_gpu_t2 import FS, LMIN, _hand_lists, _instance

pytestmark = pytest.mark.gpu


def _unsharded(gms, x, lags, theta, lmin, chunk):
    import torch
    import paper_2201_11133_b200 as gwi
    N = x.shape[1]
    st = gwi.Stream(gms, N, chunk, theta, lmin, lags=lags, capacity=1 << 16, want_pbar=True)
    xt = torch.from_numpy(x)
    if lags:
        st.prime(xt[1, N - st.tail_samples:].contiguous())
    for p in range(0, N, chunk):
        st.push(xt[0, p:p + chunk].contiguous().cuda(), xt[1, p:p + chunk].contiguous().cuda())
    n, recs = st.finish()
    pb = st.pbar.cpu().numpy()
    st.close()
    return [(r.slide, r.start, r.end, r.peak_p, r.mean_p, r.model_mask) for r in recs], pb


def _sharded(gms, x, lags, theta, lmin, chunk, world, align=1, backend=None):
    import torch
    import paper_2201_11133_b200 as gwi
    N = x.shape[1]
    rf = gms[0].receptive_field
    xt = torch.from_numpy(x)
    allrecs, pbs = [], []
    for sh in shard.plan_time(N, world, rf, max(lags) if lags else 0, align=align):
        a = shard.shard_stream_args(N, sh.start, sh.end, rf, max(lags) if lags else 0, align=align)
        st = gwi.Stream(gms, a["n_total"], chunk, theta, lmin, lags=lags, capacity=1 << 16, want_pbar=True, shard=a["shard"])
        if backend is not None:
            assert st.backend == backend
        if lags:
            assert len(a["tail_indices"]) == st.tail_samples
            st.prime(xt[1, torch.tensor(a["tail_indices"])].contiguous())
        p0 = a["first_pushed"]
        for p in range(p0, sh.end, chunk):
            q = min(p + chunk, sh.end)
            st.push(xt[0, p:q].contiguous().cuda(), xt[1, p:q].contiguous().cuda())
        n, recs = st.finish()
        assert n == len(recs)
        for r in recs:
            assert sh.start <= r.start < r.end <= sh.end
            assert bool(r.model_mask & gwi.EDGE_LEFT) == (r.start == sh.start) and bool(r.model_mask & gwi.EDGE_RIGHT) == (r.end == sh.end)
        allrecs += [(r.slide, r.start, r.end, r.peak_p, r.mean_p, r.model_mask) for r in recs]
        pbs.append(st.pbar.cpu().numpy())
        st.close()
    return allrecs, np.concatenate(pbs, axis=1)


def _models(tmp, arch, tensors_list, tag):
    import paper_2201_11133_b200 as gwi
    gms = []
    for i, t in enumerate(tensors_list):
        path = os.path.join(str(tmp), f"sh_{tag}_{i}.gwim")
        gs.write_model(path, arch, t)
        gms.append(gwi.load_model(path, gwi.FP16, 0))
    return gms


def test_time_shards_exact_triggers_narrow_kernel(tmpdir_s):
    """P16 plateau instance (tests/test_gpu_t2.py) cut into 2 and 3 shards, one cut inside a plateau: joined records ==
    unsharded records == the hand-computed intersections, with slides (the primed L1 prefix wraps around the GLOBAL stream)."""
    import paper_2201_11133_b200 as gwi
    arch = gs.CFG1_ARCH
    gms = _models(tmpdir_s, arch, [gs.p16_tensors(arch, block=i, r=3 * i, q=(i, 8 + i), hid=(2 * i, 2 * i + 1)) for i in range(2)], "n")
    N, kstar = 40 * FS, 5
    edge = N // 2                                       # the 2-shard cut falls inside the "edge" plateau
    ph, pl = _instance(N, kstar, edge)
    x = np.stack([gs.plateau_square_wave(N, ph, -2, np.float16), gs.plateau_square_wave(N, pl, -3, np.float16)])
    lags = [FS, kstar * FS, 39 * FS]
    want = _hand_lists(ph, pl, lags, N)
    ref, pb_ref = _unsharded(gms, x, lags, 0.5, LMIN, 30000)
    assert [(r[0], r[1], r[2]) for r in ref] == want and (0, edge - 1000, edge + 2500) in want
    for world in (2, 3):
        recs, pb = _sharded(gms, x, lags, 0.5, LMIN, 30000, world, backend=gwi.BACKEND_NARROW)
        got = shard.merge_edge_records(recs, LMIN)
        assert [(r[0], r[1], r[2]) for r in got] == want, world
        assert np.array_equal(pb, pb_ref)
        for g, r in zip(got, ref):
            assert abs(g[3] - r[3]) <= 1e-6 and abs(g[4] - r[4]) <= 1e-5 and g[5] == r[5]


def test_time_shards_many_short_runs_random_ensemble(tmpdir_s):
    """Random 4-model ensemble thresholded at its median with L_min = 3 (thousands of runs, many cut by shard edges)."""
    arch = gs.CFG1_ARCH
    gms = _models(tmpdir_s, arch, [gs.xavier_tensors(arch, s) for s in range(4)], "r")
    N = 100_000
    x = gs.stream_noise(61, 0, N, dtype=np.float16)
    _, pb0 = _unsharded(gms, x, [], 0.5, 3, N)
    theta = float(np.median(pb0[0]))
    for lags in ([], [4096, 20000]):
        ref, pb_ref = _unsharded(gms, x, lags, theta, 3, 17000)
        assert len(ref) > 1000
        for world in (2, 5):
            recs, pb = _sharded(gms, x, lags, theta, 3, 17000, world)
            got = shard.merge_edge_records(recs, 3)
            assert [(r[0], r[1], r[2]) for r in got] == [(r[0], r[1], r[2]) for r in ref]
            assert np.array_equal(pb, pb_ref)


@pytest.mark.parametrize("lags", [[], [FS]])
def test_time_shards_paper_scale_tensor_core(tmpdir_s, lags):
    """The tensor-core back ends in shard mode (warm-up rounded to whole 128-sample tiles for the slide back end)."""
    import paper_2201_11133_b200 as gwi
    arch = gs.PAPER_ARCH
    gms = _models(tmpdir_s, arch, [gs.xavier_tensors(arch, 0)], "t")
    N = 128 * 600
    x = gs.stream_noise(63, 0, N, dtype=np.float16)
    _, pb0 = _unsharded(gms, x, [], 0.5, 5, N)
    theta = float(np.median(pb0[0]))
    ref, pb_ref = _unsharded(gms, x, lags, theta, 5, 20000)
    recs, pb = _sharded(gms, x, lags, theta, 5, 20000, 2, align=128,
                        backend=gwi.BACKEND_TENSOR_SLIDES if lags else gwi.BACKEND_TENSOR)
    got = shard.merge_edge_records(recs, 5)
    assert [(r[0], r[1], r[2]) for r in got] == [(r[0], r[1], r[2]) for r in ref] and len(ref) > 100
    assert np.array_equal(pb, pb_ref)


def _rank_worker(rank, world, port, tmp, q):
    """One process per rank (both on cuda:0, as the single-GPU box allows: the ranks' kernels do not wait on one
    another): its span through the library in shard mode, gloo gather of the records, join on every rank."""
    import torch
    import torch.distributed as dist
    import paper_2201_11133_b200 as gwi
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        arch = gs.CFG1_ARCH
        path = os.path.join(tmp, f"rank{rank}.gwim")
        gs.write_model(path, arch, gs.p16_tensors(arch, block=2, r=7, q=(3, 4), hid=(5, 6)))
        gm = gwi.load_model(path, gwi.FP16, 0)
        N, kstar = 40 * FS, 5
        ph, pl = _instance(N, kstar, N // 2)
        x = torch.from_numpy(np.stack([gs.plateau_square_wave(N, ph, -2, np.float16), gs.plateau_square_wave(N, pl, -3, np.float16)]))
        lags = [FS, kstar * FS]
        sh = shard.plan_time(N, world, gm.receptive_field, max(lags))[rank]
        a = shard.shard_stream_args(N, sh.start, sh.end, gm.receptive_field, max(lags))
        st = gwi.Stream([gm], a["n_total"], 50000, 0.5, LMIN, lags=lags, capacity=4096, shard=a["shard"])
        st.prime(x[1, torch.tensor(a["tail_indices"])].contiguous())
        for p in range(a["first_pushed"], sh.end, 50000):
            e = min(p + 50000, sh.end)
            st.push(x[0, p:e].contiguous().cuda(), x[1, p:e].contiguous().cuda())
        n, recs = st.finish()
        st.close()
        mine = [(r.slide, r.start, r.end, r.peak_p, r.mean_p, r.model_mask) for r in recs]
        allr = [r for part in shard.gather_objects(mine, dist) for r in part]
        got = [(r[0], r[1], r[2]) for r in shard.merge_edge_records(allr, LMIN)]
        q.put((rank, got, got == _hand_lists(ph, pl, lags, N)))
    finally:
        dist.destroy_process_group()


def test_two_rank_processes_time_sharded_stream(tmpdir_s):
    import socket
    import torch.multiprocessing as mp
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_rank_worker, args=(r, 2, port, str(tmpdir_s), q)) for r in range(2)]
    for p in ps:
        p.start()
    got = sorted(q.get(timeout=300) for _ in ps)
    for p in ps:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert got[0][2] and got[1][2] and got[0][1] == got[1][1] and len(got[0][1]) >= 6
