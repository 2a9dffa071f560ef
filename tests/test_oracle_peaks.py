"""Pins of the oracle's find_peaks (oracle/gwo_oracle.c: gwo_find_peaks), the paper's post-processing rule as stated
(PAPER.md:53, 102): a hand-worked fixture, and scipy.signal.find_peaks itself -- the routine the paper names -- on random,
plateau-ridden and adversarial traces (peak positions exact, prominences / widths / crossings to 1e-12)."""
import numpy as np
import pytest
from scipy.signal import find_peaks

from gwsynth import rng
from oracle import gwo


def test_hand_worked_fixture():
    """x = [0, 1, 3, 1, 2, 2, 2, 0.5, 4, 4, 1, 5]
    local maxima: 2 (3), the flat top 4..6 -> 5 (2), the flat top 8..9 -> 8 (4); index 11 is the last sample: never a peak.
    height >= 2 keeps all three.
    peak 2 (3): left walk 3,1,0 -> min 0; right walk 3,1,2,2,2,0.5 stops at 4 > 3 -> min 0.5; prominence 3 - 0.5 = 2.5;
        level 1.75: left crossing between x[1] = 1 and x[2] = 3 at 1 + 0.75/2 = 1.375, right crossing between x[3] = 1 and
        x[2] = 3 at 3 - 0.75/2 = 2.625; width 1.25.
    peak 5 (2): left walk 2,2,1 stops at 3 -> min 1; right walk 2,2,0.5 stops at 4 -> min 0.5; prominence 2 - 1 = 1; level
        1.5: left crossing between x[3] = 1 and x[4] = 2 at 3.5, right between x[7] = 0.5 and x[6] = 2 at 7 - 1/1.5; width
        7 - 2/3 - 3.5 = 2.8333...
    peak 8 (4): left walk down to index 0 -> min 0; right walk 4,4,1 stops at 5 -> min 1; prominence 4 - 1 = 3; level 2.5:
        left crossing between x[7] = 0.5 and x[8] = 4 at 7 + 2/3.5, right between x[10] = 1 and x[9] = 4 at 10 - 1.5/3 = 9.5;
        width 9.5 - 7.5714... = 1.92857..."""
    x = np.array([0, 1, 3, 1, 2, 2, 2, 0.5, 4, 4, 1, 5], dtype=np.float64)
    n, pk = gwo.find_peaks(x, 2.0, 0.0)
    assert n == 3 and [p[0] for p in pk] == [2, 5, 8]
    assert [p[2] for p in pk] == [2.5, 1.0, 3.0]
    want_w = [1.25, 7 - 1 / 1.5 - 3.5, 9.5 - (7 + 2 / 3.5)]
    for p, w in zip(pk, want_w):
        assert abs(p[3] - w) < 1e-14
    assert abs(pk[0][4] - 1.375) < 1e-15 and abs(pk[0][5] - 2.625) < 1e-15
    # the width condition
    assert [p[0] for p in gwo.find_peaks(x, 2.0, 1.5)[1]] == [5, 8]
    assert [p[0] for p in gwo.find_peaks(x, 2.5, 1.5)[1]] == [8]                 # height is inclusive: x[5] = 2 < 2.5
    assert [p[0] for p in gwo.find_peaks(x, 3.0, 0.0)[1]] == [2, 8]              # x[2] = 3 >= 3


def _traces():
    for seed in range(12):
        N = 200 + 97 * seed
        u = rng.uniform01(700 + seed, 0, np.arange(N, dtype=np.uint64))
        yield u                                                                   # white: a third of the samples are peaks
        yield np.round(u * 6) / 6                                                 # many flat tops and ties
        sm = np.convolve(u, np.ones(25) / 25, mode="same")
        yield sm                                                                  # broad features, large widths
        yield np.round(sm * 40) / 40
        yield (np.float32(0.5) + np.float32(0.03) * (sm.astype(np.float32) - np.float32(0.5))).astype(np.float64)  # fp32-valued, like p
    yield np.zeros(50)
    yield np.ones(3)
    yield np.array([0.0, 1.0, 0.0])
    yield np.array([1.0, 1.0, 0.0, 1.0, 1.0])                                      # flat tops touching both ends: no peaks
    yield np.array([0.0, 2.0, 2.0, 2.0, 2.0, 0.0, 2.0, 0.0])                       # even-length flat top -> floor of the middle
    yield np.concatenate([np.linspace(0, 1, 300), np.linspace(1, 0, 300)])


@pytest.mark.parametrize("height,width", [(0.0, 0.0), (0.5, 0.0), (0.5, 3.0), (0.45, 20.0), (0.2, 1.0)])
def test_against_scipy(height, width):
    for x in _traces():
        idx, props = find_peaks(x, height=height, width=width)
        n, pk = gwo.find_peaks(x, height, width)
        assert n == len(idx) and [p[0] for p in pk] == idx.tolist()
        if n:
            assert np.max(np.abs(np.array([p[1] for p in pk]) - props["peak_heights"])) == 0
            assert np.max(np.abs(np.array([p[2] for p in pk]) - props["prominences"])) <= 1e-12
            assert np.max(np.abs(np.array([p[3] for p in pk]) - props["widths"])) <= 1e-12
            assert np.max(np.abs(np.array([p[4] for p in pk]) - props["left_ips"])) <= 1e-12
            assert np.max(np.abs(np.array([p[5] for p in pk]) - props["right_ips"])) <= 1e-12


def test_run_length_rule_and_find_peaks_on_a_plateau():
    """How reading A34's run-length rule and the paper's find_peaks differ on the P16 plateaus:
    a rectangular plateau of L samples at p = 1 over a p = 0.15 floor is ONE flat-top peak at its middle, prominence 0.85,
    half-prominence level 0.575, crossings interpolated half a sample outside... the width is L, not L - 1, so both rules
    accept exactly the plateaus with L >= 2048; find_peaks reports the plateau's MIDDLE, the run rule its END."""
    for L in (2047, 2048, 2049):
        x = np.full(6000, 0.15)
        x[1000:1000 + L] = 1.0
        n, pk = gwo.find_peaks(x, 0.5, 2048.0)
        runs = gwo.triggers(x, 0.5, 2048)[1]
        n0, pk0 = gwo.find_peaks(x, 0.5, 0.0)
        assert n0 == 1 and pk0[0][0] == 1000 + (L - 1) // 2 and abs(pk0[0][3] - L) < 1e-9
        assert (n == 1) == (len(runs) == 1) == (L >= 2048)
