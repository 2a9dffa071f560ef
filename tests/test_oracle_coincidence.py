"""Pin P17 (-m "not gpu"): the oracle's all-model coincidence rule (reading A34) against a hand-worked
fixture, a brute force over all one-trigger-per-model tuples, and the invariances the definition implies."""
import itertools
import os

import numpy as np

from oracle import gwo

HERE = os.path.dirname(os.path.abspath(__file__))


def _fixture():
    W, ms, ev = None, [], []
    for line in open(os.path.join(HERE, "golden", "p17_coincidence.txt")):
        f = line.split()
        if not f or f[0] == "#":
            continue
        if f[0] == "W":
            W = int(f[1])
        elif f[0] == "m":
            ms.append([int(v) for v in f[1:]])
        elif f[0] == "e":
            ev.append(tuple(int(v) for v in f[1:]))
    return W, ms, ev


def test_p17_worked_example():
    W, ms, ev = _fixture()
    assert gwo.coincidence(ms, W) == ev
    assert gwo.coincidence(ms, 11) == [(100, 109, 3), (205, 216, 3), (296, 305, 3)]    # 216 - 205 = 11 now fits
    assert gwo.coincidence(ms[:1], 0) == [(e, e, 1) for e in ms[0]]                    # one model: every trigger
    assert gwo.coincidence([ms[0], []], 1000) == []                                     # a silent model vetoes all


def _rand_ends(rs, M, n, span):
    return [sorted(rs.choice(span, size=rs.randint(0, n + 1), replace=False).tolist()) for _ in range(M)]


def test_p17_tuple_brute_force_and_invariances():
    rs = np.random.RandomState(7)
    for trial in range(200):
        M = rs.randint(1, 5)
        ends = _rand_ends(rs, M, 6, 200)
        W = int(rs.randint(0, 40))
        ev = gwo.coincidence(ends, W)
        # brute force: all tuples with one trigger per model inside a window of W
        tuples = [t for t in itertools.product(*ends) if max(t) - min(t) <= W] if all(len(e) for e in ends) else []
        assert (len(ev) > 0) == (len(tuples) > 0)
        anchors = sorted({min(t) for t in tuples})
        # every tuple lies inside exactly one event, events are disjoint, ordered and more than W apart
        for t in tuples:
            assert sum(1 for a, b, _ in ev if a <= min(t) and max(t) <= b) == 1
        for (a0, b0, _), (a1, b1, _) in zip(ev, ev[1:]):
            assert b0 < a1
        # event starts are anchors, and clustering of the anchors by gaps > W reproduces the starts
        starts = [a for i, a in enumerate(anchors) if i == 0 or a - anchors[i - 1] > W]
        assert [a for a, _, _ in ev] == starts
        # trigger counts: all ends within [t_first, last anchor + W]
        for a, b, k in ev:
            cl = [x for x in anchors if a <= x and (x == a or True)]
            last = a
            for x in anchors:
                if x > last and x - last <= W and x >= a:
                    last = x
            assert k == sum(1 for e in ends for v in e if a <= v <= last + W)
            assert b == max(v for e in ends for v in e if a <= v <= last + W)
        # model order does not matter; a wider window keeps every anchor
        perm = list(rs.permutation(M))
        assert gwo.coincidence([ends[i] for i in perm], W) == ev
        wide = gwo.coincidence(ends, W + 5)
        for a, b, _ in ev:
            assert any(a2 <= a and b <= b2 for a2, b2, _ in wide)


def test_library_coincidence_matches_oracle_on_host():
    """gwi_coincidence is a host function (two-pointer sweeps): exact agreement with the oracle's O(n^2) definition on
    random per-model trigger lists, several slides, records in random order."""
    import paper_2201_11133_b200 as gwi
    rs = np.random.RandomState(11)
    for trial in range(100):
        M = int(rs.randint(1, 5))
        W = int(rs.randint(0, 60))
        recs, want = [], []
        for slide in range(int(rs.randint(1, 4))):
            ends = _rand_ends(rs, M, 8, 300)
            for m, e in enumerate(ends):
                for v in e:
                    recs.append(gwi.Trigger(slide=slide, model_mask=1 << m, start=v - 5, end=v, peak_p=1.0, mean_p=1.0))
            want += [(slide,) + ev for ev in gwo.coincidence(ends, W, slide=slide)]
        rs.shuffle(recs)
        got = [(e.slide, e.t_first, e.t_last, e.n_triggers) for e in gwi.coincidence(recs, M, W)]
        assert got == want
    with np.testing.assert_raises(gwi.GwiError):
        gwi.coincidence([], 0, 5)
