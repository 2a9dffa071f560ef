"""GPU parity of gwi_ensemble_triggers against the oracle's trigger stage: tier T1, BIT-EXACT (-m gpu).

Both sides get the same fp32 probability arrays; the mean is the fixed fp32 expression; (slide,start,end) and the
count must agree exactly for any theta and L_min; peak/mean to fp32 tolerance; the mean array bit for bit.
"""
import numpy as np
import pytest

import gwsynth as gs
from gwsynth import rng
from oracle import gwo
from tests.helpers import trig_tuples

pytestmark = pytest.mark.gpu


def _oracle(ps, theta, lmin, slide=0, t0=0):
    pb = gwo.ensemble_mean_f32(ps)
    n, recs = gwo.triggers(pb.astype(np.float64), float(np.float32(theta)), lmin, slide=slide, t0=t0,
                           pm=[p.astype(np.float64) for p in ps])
    return pb, n, recs


def _gpu(ps, theta, lmin, **kw):
    import torch
    import paper_2201_11133_b200 as gwi
    return gwi.ensemble_triggers([torch.from_numpy(p).cuda() for p in ps], theta, lmin, want_pbar=True, **kw)


def _noisy(seed, N, M=4, corr=64):
    """plateaus of random level + noise, so that runs of many lengths exist"""
    out = []
    base = rng.uniform01(seed, 0, np.arange(N // corr + 1, dtype=np.uint64))
    lvl = np.repeat(np.where(base < 0.5, 0.3, 0.7), corr)[:N]
    for m in range(M):
        out.append((lvl + 0.25 * (rng.uniform01(seed, 1 + m, np.arange(N, dtype=np.uint64)) - 0.5)).astype(np.float32))
    return out


@pytest.mark.parametrize("N,lmin,theta", [(11, 3, 0.5), (1, 1, 0.5), (31, 1, 0.5), (32, 2, 0.5), (33, 5, 0.45),
                                          (4096, 64, 0.5), (100003, 100, 0.5), (100003, 1, 0.52), (1 << 20, 2048, 0.5),
                                          (300000, 300001, 0.0), (5000, 1, 1.0), (5000, 1, 0.0)])
def test_t1_bit_exact(N, lmin, theta):
    ps = _noisy(N + lmin, N)
    pb, n, recs = _oracle(ps, theta, lmin, slide=3, t0=1000)
    gn, grecs, gpb = _gpu(ps, theta, lmin, slide_id=3, t0=1000, capacity=max(n, 1) + 5)
    assert np.array_equal(gpb.cpu().numpy(), pb)                          # fp32 mean, bit for bit
    assert gn == n
    assert trig_tuples(grecs) == [(r[0], r[1], r[2]) for r in recs]
    for g, o in zip(grecs, recs):
        assert abs(g.peak_p - o[3]) <= 1e-6 and abs(g.mean_p - o[4]) <= 1e-5 and g.model_mask == o[5]


def test_p13_fixture_on_gpu():
    ps = [np.array([.6, .6, .4, .6, .6, .6, .5, .7, .7, .7, .7], dtype=np.float32)] * 4
    n, recs, _ = _gpu(ps, 0.5, 3)
    assert n == 2 and [(r.start, r.end) for r in recs] == [(3, 6), (7, 11)]


def test_adversarial_runs():
    L = 40
    for ln in (L - 1, L, L + 1):
        for pos in (0, 7, 31, 32, 33, 1023 * 32 - 3, 8192 - 20, 8192, 32768 - 5):
            N = 70000
            a = np.zeros(N, dtype=np.float32) + 0.25
            a[pos:pos + ln] = 0.75
            a[N - ln:] = 0.75
            pb, n, recs = _oracle([a], 0.5, L)
            gn, grecs, _ = _gpu([a], 0.5, L)
            assert gn == n and trig_tuples(grecs) == [(r[0], r[1], r[2]) for r in recs], (ln, pos)
    ones = np.full(3 * 8192 * 32 + 17, 0.9, dtype=np.float32)           # all-ones: walks by 8192-sample blocks
    gn, grecs, _ = _gpu([ones], 0.5, 2048)
    assert gn == 1 and (grecs[0].start, grecs[0].end) == (0, len(ones))
    gn, _, _ = _gpu([np.zeros(100000, dtype=np.float32)], 0.5, 1)
    assert gn == 0
    un = np.full(1001, 0.9, dtype=np.float32)[1:]                          # 4-byte but not 16-byte aligned view
    import torch
    import paper_2201_11133_b200 as gwi
    t = torch.from_numpy(np.full(1001, 0.9, dtype=np.float32)).cuda()[1:]
    n, recs, _ = gwi.ensemble_triggers([t], 0.5, 10)
    assert n == 1 and (recs[0].start, recs[0].end) == (0, 1000)


@pytest.mark.parametrize("chunk", [1, 100, 2048, 4096 * 3 + 7])
def test_chunked_with_carry_equals_whole(chunk):
    import torch
    import paper_2201_11133_b200 as gwi
    from paper_2201_11133_b200.binding import new_carry
    N, lmin = (3000 if chunk == 1 else 60000), 150
    ps = _noisy(77, N, corr=128)
    pb, n, recs = _oracle(ps, 0.5, lmin)
    assert n >= 3
    carry = new_carry(0)
    got = []
    dev = [torch.from_numpy(p).cuda() for p in ps]
    for s in range(0, N, chunk):
        e = min(s + chunk, N)
        cn, crecs, _ = gwi.ensemble_triggers([d[s:e] for d in dev], 0.5, lmin, t0=s, last_chunk=(e == N), carry=carry,
                                             capacity=64)
        assert cn == len(crecs)
        got += crecs
    assert trig_tuples(got) == [(r[0], r[1], r[2]) for r in recs]
    for g, o in zip(got, recs):
        assert abs(g.peak_p - o[3]) <= 1e-6 and abs(g.mean_p - o[4]) <= 1e-5 and g.model_mask == o[5]


def test_capacity_overflow_gives_valid_prefix():
    import paper_2201_11133_b200 as gwi
    ps = _noisy(5, 50000, corr=32)
    pb, n, recs = _oracle(ps, 0.5, 8)
    assert n > 10
    with pytest.raises(gwi.GwiError) as e:
        _gpu(ps, 0.5, 8, capacity=7)
    assert e.value.status == 7 and e.value.count == n
    assert trig_tuples(e.value.records) == [(r[0], r[1], r[2]) for r in recs[:7]]


@pytest.mark.parametrize("N,lmin,M", [(1, 1, 1), (10, 11, 2), (5000, 1, 4), (100003, 100, 4), (300000, 2048, 4),
                                      (40000, 4097, 3), (70000, 16384, 2), (1 << 20, 2048, 4)])
def test_threshold_sweep_equals_per_threshold_clustering(N, lmin, M):
    """gwi_threshold_sweep (one sliding-window-minimum pass) against the oracle's trigger count at every threshold."""
    import torch
    import paper_2201_11133_b200 as gwi
    ps = _noisy(N + lmin + M, N, M=M, corr=max(16, min(lmin // 2, 700)))
    pb = gwo.ensemble_mean_f32(ps).astype(np.float64)
    th = np.unique(np.concatenate([np.linspace(0.0, 0.9998, 97), [0.3, 0.5, 0.7, float(pb.min()), float(pb.max())]])
                   .astype(np.float32))
    got = gwi.threshold_sweep([torch.from_numpy(p).cuda() for p in ps], th, lmin).cpu().numpy()
    want = [gwo.triggers(pb, float(t), lmin, cap=1)[0] for t in th]
    assert got.tolist() == want
    if N >= 5000:
        assert max(want) > 0
