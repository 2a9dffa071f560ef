"""Pins for the oracle's trigger stage (P13 worked example, P14 brute force, P15 nesting argument, P16 closed form).

Expected values: tests/golden/p13_clustering.txt (hand-computed), an O(N*L_min) sliding-window definition written
here in numpy ("t lies inside a trigger iff some all-ones window of length L_min covers it"), and the plateau
intersections of P16, computed from the plateau lists by interval arithmetic.  Nothing comes from the CUDA path.
"""
import os

import numpy as np
import pytest

import gwsynth as gs
from gwsynth import rng
from oracle import gwo

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def test_p13_worked_example():
    with open(os.path.join(GOLD, "p13_clustering.txt")) as f:
        rows = [l.split() for l in f if l.strip() and not l.startswith("#")]
    pbar = np.array([float(v) for v in rows[0]])
    theta, lmin = float(rows[1][0]), int(rows[1][1])
    want = [(int(a), int(b)) for a, b in rows[2:]]
    n, recs = gwo.triggers(pbar, theta, lmin, slide=5, t0=0)
    assert n == len(want) and [(r[1], r[2]) for r in recs] == want and all(r[0] == 5 for r in recs)
    assert abs(recs[0][3] - 0.6) < 1e-15 and abs(recs[1][3] - 0.7) < 1e-15          # peak
    assert abs(recs[0][4] - 0.6) < 1e-15                                             # mean
    n2, recs2 = gwo.triggers(pbar, theta, lmin, t0=1000)
    assert [(r[1], r[2]) for r in recs2] == [(a + 1000, b + 1000) for a, b in want]
    # capacity: count is the total, only `cap` records are written
    n3, recs3 = gwo.triggers(pbar, theta, lmin, cap=1)
    assert n3 == 2 and len(recs3) == 1 and (recs3[0][1], recs3[0][2]) == want[0]


def _brute(a, lmin):
    """Sliding-window definition: covered[t] iff exists s <= t < s+lmin with a[s:s+lmin] all ones (or, for runs
    clipped by the array, never: a run shorter than lmin does not qualify even at the edges -- reading A21 counts
    the TRUNCATED length).  Returns the maximal covered intervals."""
    N = len(a)
    cov = np.zeros(N, dtype=bool)
    for s in range(0, N - lmin + 1):
        if a[s:s + lmin].all():
            cov[s:s + lmin] = True
    out, t = [], 0
    while t < N:
        if cov[t]:
            s = t
            while t < N and cov[t]:
                t += 1
            out.append((s, t))
        else:
            t += 1
    return out


def _traces():
    L = 5
    yield np.zeros(40, dtype=bool), L
    yield np.ones(40, dtype=bool), L
    yield np.ones(3, dtype=bool), L                 # shorter than L_min altogether
    for ln in (L - 1, L, L + 1):
        for pos in (0, 7, 31, 32, 33):              # 32-sample word boundary
            a = np.zeros(64, dtype=bool)
            a[pos:pos + ln] = True
            yield a, L
        a = np.zeros(64, dtype=bool)
        a[64 - ln:] = True                          # touching the end
        yield a, L
    for big in (1023, 1024, 1025):                  # 1024-block boundary
        a = np.zeros(2100, dtype=bool)
        a[big - 3:big + 4] = True
        yield a, 7
        yield a, 8
    for seed in range(40):
        N = 50 + 13 * seed
        u = rng.uniform01(900 + seed, 0, np.arange(N, dtype=np.uint64))
        yield u < (0.55 + 0.01 * seed), 1 + seed % 6


def test_p14_brute_force():
    for a, lmin in _traces():
        pbar = np.where(a, 0.75, 0.25)
        n, recs = gwo.triggers(pbar, 0.5, lmin)
        assert n == len(recs)
        assert [(r[1], r[2]) for r in recs] == _brute(a, lmin), (a.astype(int).tolist(), lmin)


def test_p14_strict_threshold_and_param_edges():
    p = np.array([0.5, 0.5, 0.5000001, 0.6, 0.5, 1.0, 1.0])
    assert [(r[1], r[2]) for r in gwo.triggers(p, 0.5, 1)[1]] == [(2, 4), (5, 7)]
    assert gwo.triggers(p, 1.0, 1)[0] == 0                      # nothing is > 1
    assert [(r[1], r[2]) for r in gwo.triggers(p, 0.0, 1)[1]] == [(0, 7)]
    assert gwo.triggers(p, 0.0, 8)[0] == 0                      # L_min = N + 1
    m = [np.array([0.9, 0.1, 0.9]), np.array([0.2, 0.2, 0.9])]
    pb = gwo.ensemble_mean(m)
    n, r = gwo.triggers(pb, 0.5, 1, pm=m)
    assert [(x[1], x[2], x[5]) for x in r] == [(0, 1, 0b01), (2, 3, 0b11)]


def test_p15_nesting_argument_on_random_traces():
    """If the lists at theta-delta and theta+delta agree, any pbar' within delta of pbar gives that same list."""
    delta, theta, lmin = 0.05, 0.5, 4
    robust = 0
    for seed in range(300):
        N = 120
        base = rng.uniform01(5000 + seed, 0, np.arange(N // 8, dtype=np.uint64))
        p = np.repeat(np.where(base < 0.5, 0.15, 0.85), 8) + 0.2 * (rng.uniform01(5000 + seed, 1, np.arange(N, dtype=np.uint64)) - 0.5)
        lo = [(r[1], r[2]) for r in gwo.triggers(p, theta - delta, lmin)[1]]
        hi = [(r[1], r[2]) for r in gwo.triggers(p, theta + delta, lmin)[1]]
        if lo != hi:
            continue
        robust += 1
        pert = p + delta * (2 * rng.uniform01(6000 + seed, 2, np.arange(N, dtype=np.uint64)) - 1) * 0.999
        assert [(r[1], r[2]) for r in gwo.triggers(pert, theta, lmin)[1]] == lo
    assert robust > 50


# ---- P16 sign pass-through model: end-to-end closed form including slides ---------------------------------
def p16_model_tensors():
    a = gs.Arch(n_branch=2, c_in=1, R=1, S=2, k=2, dil=(1,), Hh=2)
    t = gs.zero_tensors(a)
    for b in range(2):
        t[f"b{b}.W_in"][:] = 1.0
        t[f"b{b}.l0.Wf"][0, 0] = [0.0, 1.0]         # f = x[t]; Wg = 0 -> z = tanh(x)/2
        t[f"b{b}.l0.Ws"][:, 0] = [2.0, -2.0]        # u = (T+, T-), T = tanh(x)
    t["W1"][0] = [1, -1, 1, -1]                     # v0 = ReLU(T_H + T_L)
    t["W1"][1] = [-1, 1, -1, 1]                     # v1 = ReLU(-(T_H + T_L))
    t["W2"][:] = [8.0, -8.0]                        # y = 8 (T_H + T_L)
    return a, t


def _intersections(ph, pl, lag, N, lmin):
    """plateau intersections of H1 with L1 delayed circularly by lag, as maximal runs in [0,N) of length >= lmin"""
    on = np.zeros(N, dtype=bool)
    h = np.zeros(N, dtype=bool)
    l = np.zeros(N, dtype=bool)
    for s, e in ph:
        h[s:e] = True
    for s, e in pl:
        l[s:e] = True
    on = h & np.roll(l, lag)
    out, t = [], 0
    while t < N:
        if on[t]:
            s = t
            while t < N and on[t]:
                t += 1
            if t - s >= lmin:
                out.append((s, t))
        else:
            t += 1
    return out


def test_p16_sign_pass_through(tmpdir_s):
    a, t = p16_model_tensors()
    path = os.path.join(str(tmpdir_s), "p16.gwim")
    gs.write_model(path, a, t)
    m = gwo.Model(path)
    fs, lmin = 64, 32                               # scaled-down "second" and L_min = fs/2
    N = 20 * fs
    ph = [(100, 100 + 31), (200, 200 + 32), (300, 300 + 33), (500, 700), (900, 1000), (N - 20, N)]
    pl = [(90, 140), (190, 240), (290, 340), (500 - 2 * fs, 700 - 2 * fs - 50), (900, 1000), (0, 30)]
    x = np.stack([gs.plateau_square_wave(N, ph, -2, np.float64), gs.plateau_square_wave(N, pl, -3, np.float64)])
    p, u = m.stream(x, want_u=True)
    # closed form of the logit: y = 8 (tanh xH + tanh xL)
    y = 8.0 * (np.tanh(x[0]) + np.tanh(x[1]))
    assert np.max(np.abs(p - 1.0 / (1.0 + np.exp(-y)))) < 1e-12
    vals = sorted(set(np.round(y, 1)))
    assert vals == [-15.7, -1.9, -1.6, 12.2]
    for lag_s in (0, 1, 2, 5):
        lag = lag_s * fs
        pk = m.head_slide(u, lag)
        n, recs = gwo.triggers(gwo.ensemble_mean([pk] * 4), 0.5, lmin, slide=lag_s)
        want = _intersections(ph, pl, lag, N, lmin)
        assert [(r[1], r[2]) for r in recs] == want, lag_s
        # P15 robustness: margins are >> 2e-3, so theta +- 2e-3 gives the same list
        for th in (0.5 - 2e-3, 0.5 + 2e-3):
            assert [(r[1], r[2]) for r in gwo.triggers(pk, th, lmin)[1]] == want
    assert len(_intersections(ph, pl, 0, N, lmin)) >= 3 and _intersections(ph, pl, 2 * fs, N, lmin) != _intersections(ph, pl, 0, N, lmin)


# ---- peak_p / mean_p on a NON-constant run, and the fixed fp32 mean expression (values worked by hand) --------
def test_peak_and_mean_on_non_constant_runs():
    """p = [.1, .6, .9, .7, .2, .8, .55, .3], theta = .5, L_min = 2: runs [1,4) and [5,7).  On [1,4) the maximum (.9) is
    neither the first (.6), the last (.7) nor the minimum (.6); mean = 2.2/3.  On [5,7): peak .8 (first), mean 1.35/2."""
    p = np.array([.1, .6, .9, .7, .2, .8, .55, .3])
    n, recs = gwo.triggers(p, 0.5, 2)
    assert n == 2 and [(r[1], r[2]) for r in recs] == [(1, 4), (5, 7)]
    assert recs[0][3] == 0.9 and abs(recs[0][4] - 2.2 / 3) < 1e-15
    assert recs[1][3] == 0.8 and abs(recs[1][4] - 0.675) < 1e-15
    # the peak at the last sample of a run that touches the stream end
    n, recs = gwo.triggers(np.array([.6, .7, .95]), 0.5, 1, t0=10)
    assert [(r[1], r[2], r[3]) for r in recs] == [(10, 13, 0.95)]


def test_ensemble_mean_f32_is_the_fixed_order_expression():
    """(((p0+p1)+p2)+p3)/(float)M with IEEE round-to-nearest-even adds and ONE correctly rounded division (tier T1).
    Expected bit patterns derived by hand, t = 2^-24 (half an ulp of 1.0f):
      (1, t, t, t): 1+t ties to even -> 1, three times; 1/4 = 0.25                          = 0x3e800000
      (t, t, t, 1): t+t = 2t, +t = 3t (exact), 3t+1 = 1 + 1.5 ulp -> tie to even = 1+2^-22; /4   = 0x3e800002
        (an fp64 sum rounded once, (1+3t)/4 = 0.25 + 1.5 ulp(0.25), would also give 0x3e800002 for BOTH orders)
      (2.5, 2.5, 0) / 3: 5/3 correctly rounded                                               = 0x3fd55555
        (5 * float(1/3), a reciprocal multiply, gives 0x3fd55556)"""
    t = np.float32(2.0 ** -24)
    one = np.float32(1.0)

    def bits(v):
        return int(np.asarray(v, dtype=np.float32).view(np.uint32)[0])

    a = gwo.ensemble_mean_f32([np.array([v], dtype=np.float32) for v in (one, t, t, t)])
    b = gwo.ensemble_mean_f32([np.array([v], dtype=np.float32) for v in (t, t, t, one)])
    c = gwo.ensemble_mean_f32([np.array([v], dtype=np.float32) for v in (2.5, 2.5, 0.0)])
    assert bits(a) == 0x3e800000 and bits(b) == 0x3e800002 and bits(c) == 0x3fd55555
