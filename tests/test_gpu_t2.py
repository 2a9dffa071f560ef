"""Tier T2 of trigger parity on the GPU (-m gpu): strain -> triggers END TO END through the fused kernels, exact.

north_star: "trigger lists must match exactly"; SURVEY.md section 8(c) "Two tiers of trigger parity": T2 is required on
delta-robust instances (pin P15) and pin P16 (the sign pass-through model) supplies non-vacuous ones.  Here P16's model
is placed inside the widths the fast kernels take (gwsynth.p16_tensors: all other channels and blocks are zero and
contribute nothing), so that k_tiny / k_tiny_heads (config-1 widths) and k_stack / k_head_tc (paper-scale widths)
themselves produce non-empty trigger lists, which are compared with

  (1) the plateau intersections worked out by interval arithmetic from the plateau lists (no network involved),
  (2) the oracle's list computed from the ORACLE's own probabilities (gwo.Model.stream / head_slide / triggers),
  (3) the P15 guard: the oracle's lists at theta -+ 2e-3 are identical, so the instance is provably robust.

Plateaus (width >= 0.5 s = 2048 samples): lengths 2047 / 2048 / 2049, one cut by a chunk boundary, one
that aligns only at lag k*, one truncated by the stream end, one that exists only through the circular wrap of a slide.
"""
import os

import numpy as np
import pytest

import gwsynth as gs
from oracle import gwo
from tests.helpers import trig_tuples

pytestmark = pytest.mark.gpu

FS = 4096
LMIN = 2048


def _runs(on, lmin):
    out, t, N = [], 0, len(on)
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


def _hand_lists(ph, pl, lags, N, shift=0):
    """expected (slide, start, end): H1 plateaus AND L1 plateaus delayed circularly by the lag; `shift` = the model reads
    its input `shift` samples in the past (zero history before t = 0: not a plateau)."""
    h = np.zeros(N, dtype=bool)
    l = np.zeros(N, dtype=bool)
    for s, e in ph:
        h[s:e] = True
    for s, e in pl:
        l[s:e] = True
    if shift:
        h = np.concatenate([np.zeros(shift, dtype=bool), h[:-shift]])
        l = np.concatenate([np.zeros(shift, dtype=bool), l[:-shift]])
    out = []
    for k, lag in enumerate([0] + list(lags)):
        out += [(k, s, e) for s, e in _runs(h & np.roll(l, lag), LMIN)]
    return out


def _instance(N, kstar, edge, a=10000):
    """plateau lists for a stream of N samples; `edge` = a sample index that is a chunk boundary of the pushes."""
    lag = kstar * FS
    e0 = N - 20000                                     # the plateau that aligns only at lag k*
    ph = [(a, a + 2047), (2 * a, 2 * a + 2048), (3 * a, 3 * a + 2049), (edge - 2000, edge + 3000),
          (e0, e0 + 3000), (0, 5000), (N - 2500, N)]
    pl = [(a - 1000, a + 3000), (2 * a - 1000, 2 * a + 3000), (3 * a - 1000, 3 * a + 3000), (edge - 1000, edge + 2500),
          (e0 - lag, e0 + 3000 - lag), (N - 3000, N)]
    assert 3 * a + 3100 < edge - 2000 and e0 - lag > edge + 3000 + 100 and a - 1000 >= 5000
    return ph, pl


_ORACLE_CACHE = {}


def _oracle_lists(oms, x, lags, theta, key=None):
    if key is not None and key in _ORACLE_CACHE:
        return _ORACLE_CACHE[key]
    per = []
    for om in oms:
        p0, u = om.stream(x.astype(np.float64), want_u=True)
        per.append([p0] + [om.head_slide(u, lag) for lag in lags])
    pbar = np.stack([gwo.ensemble_mean([per[m][k] for m in range(len(oms))]) for k in range(1 + len(lags))])
    out = {}
    for th in (theta - 2e-3, theta, theta + 2e-3):
        lst = []
        for k in range(pbar.shape[0]):
            _, recs = gwo.triggers(pbar[k], th, LMIN, slide=k)
            lst += [(r[0], r[1], r[2]) for r in recs]
        out[th] = lst
    if key is not None:
        _ORACLE_CACHE[key] = (pbar, out)
    return pbar, out


def _push_all(gms, x, chunks, lags, host, backend):
    import torch
    import paper_2201_11133_b200 as gwi
    N = x.shape[1]
    st = gwi.Stream(gms, N, max(chunks), 0.5, LMIN, lags=lags, capacity=1024, want_pbar=True)
    assert st.backend == backend, st.backend
    xt = torch.from_numpy(x)
    st.prime(xt[1, N - st.tail_samples:].contiguous())
    pos, keep = 0, []
    for n in chunks:
        a, b = xt[0, pos:pos + n].contiguous(), xt[1, pos:pos + n].contiguous()
        a, b = (a.pin_memory(), b.pin_memory()) if host else (a.cuda(), b.cuda())
        keep.append((a, b))
        st.push(a, b)
        pos += n
    n, recs = st.finish()
    pbar = st.pbar.cpu().numpy()
    st.close()
    return n, recs, pbar


def _models(tmp, arch, placements, tag):
    import paper_2201_11133_b200 as gwi
    oms, gms = [], []
    for i, kw in enumerate(placements):
        path = os.path.join(str(tmp), f"p16_{tag}_{i}.gwim")
        gs.write_model(path, arch, gs.p16_tensors(arch, **kw))
        oms.append(gwo.Model(path, round_fp16=True))
        gms.append(gwi.load_model(path, gwi.FP16, 0))
    return oms, gms


def _check(oms, gms, x, ph, pl, lags, chunks, host, backend, shift=0, ptol=2e-3, key=None):
    N = x.shape[1]
    want = _hand_lists(ph, pl, lags, N, shift)
    pbar_o, lists = _oracle_lists(oms, x, lags, 0.5, key)
    # the oracle from its own probabilities gives the hand-computed list, and the instance is delta-robust (P15)
    assert lists[0.5] == want
    assert lists[0.5 - 2e-3] == want and lists[0.5 + 2e-3] == want
    n, recs, pbar = _push_all(gms, x, chunks, lags, host, backend)
    got = trig_tuples(recs)
    assert n == len(got) and got == want, (got, want)
    assert np.max(np.abs(pbar - pbar_o)) <= ptol
    return want


@pytest.mark.parametrize("host", [False, True])
def test_t2_narrow_kernel_exact_triggers(tmpdir_s, host):
    """k_tiny + k_tiny_heads (R16/S32/Hh32, d = 1,2,4,8), 4-model ensemble whose members hold the pass-through in
    different blocks / channels, FP16 mode, ragged chunks, lags 1 s, 2 s, k* = 5 s and 39 s."""
    import paper_2201_11133_b200 as gwi
    place = [dict(block=0, r=0, q=(0, 1), hid=(0, 1)), dict(block=1, r=5, q=(7, 30), hid=(31, 2)),
             dict(block=2, r=15, q=(31, 16), hid=(9, 20)), dict(block=3, r=8, q=(12, 13), hid=(17, 16))]
    oms, gms = _models(tmpdir_s, gs.CFG1_ARCH, place, "n")
    N, kstar, edge = 40 * FS, 5, 50000
    ph, pl = _instance(N, kstar, edge)
    x = np.stack([gs.plateau_square_wave(N, ph, -2, np.float16), gs.plateau_square_wave(N, pl, -3, np.float16)])
    lags = [FS, 2 * FS, kstar * FS, 39 * FS]
    chunks = [20000, 30000, 1, 13333, 4096, N - 67430]
    assert sum(chunks) == N and sum(chunks[:2]) == edge
    want = _check(oms, gms, x, ph, pl, lags, chunks, host, gwi.BACKEND_NARROW)
    by_slide = {k: [w for w in want if w[0] == k] for k in range(5)}
    assert (0, 20000, 22048) in want and (0, 30000, 32049) in want and not any(w[1] == 10000 for w in want)
    assert (0, edge - 1000, edge + 2500) in want and (0, N - 2500, N) in want
    assert (3, N - 20000, N - 17000) in want and not any(w[1] == N - 20000 for k in (0, 1, 2, 4) for w in by_slide[k])
    assert (1, 1096, 4096) in want                      # exists only through the circular wrap (primed tail)


def test_t2_narrow_kernel_past_tap(tmpdir_s):
    """The pass-through on the PAST tap of the d = 8 block: every plateau moves 8 samples later (dilated tap index)."""
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, gs.CFG1_ARCH, [dict(block=3, r=3, q=(4, 5), hid=(6, 7), past=True)], "np")
    N, kstar, edge = 40 * FS, 5, 50000
    ph, pl = _instance(N, kstar, edge)
    ph = [p for p in ph if p[0] != 0]                    # a plateau at t = 0 would touch the p = 0.5 zero-history samples
    x = np.stack([gs.plateau_square_wave(N, ph, -2, np.float16), gs.plateau_square_wave(N, pl, -3, np.float16)])
    _check(oms, gms, x, ph, pl, [kstar * FS], [edge, N - edge], False, gwi.BACKEND_NARROW, shift=8)


@pytest.mark.parametrize("lags,host", [([], False), ([FS, 2 * FS], False), ([FS, 2 * FS], True)])
def test_t2_tensor_core_kernel_exact_triggers(tmpdir_s, lags, host):
    """k_stack + k_head_tc (R64/S128/Hh128, 2 x 10 dilations) with the pass-through in block 13 (d = 8, second stack),
    residual channel 37; zero lag only = the segment back end, with lags = the all-lag head back end."""
    import torch
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, gs.PAPER_ARCH, [dict(block=13, r=37, q=(127, 64), hid=(100, 3))], "t")
    assert all(g.uses_tensor_cores for g in gms)
    N, kstar, edge = 16 * FS, 2, 26112
    ph, pl = _instance(N, kstar, edge, a=6000)
    x = np.stack([gs.plateau_square_wave(N, ph, -2, np.float16), gs.plateau_square_wave(N, pl, -3, np.float16)])
    chunks = [20000, 6112, 1, 13333, 4096, N - 43542]
    assert sum(chunks) == N and sum(chunks[:2]) == edge
    all_lags = [FS, 2 * FS]
    if not lags:
        # zero lag only: no priming; the expected list is the zero-lag part of the slide instance's
        st = gwi.Stream(gms, N, max(chunks), 0.5, LMIN, capacity=1024, want_pbar=True)
        assert st.backend == gwi.BACKEND_TENSOR
        xt, pos = torch.from_numpy(x).cuda(), 0
        for n in chunks:
            st.push(xt[0, pos:pos + n].contiguous(), xt[1, pos:pos + n].contiguous())
            pos += n
        n, recs = st.finish()
        pbar = st.pbar.cpu().numpy()
        st.close()
        want = _hand_lists(ph, pl, [], N)
        pbar_o, lists = _oracle_lists(oms, x, all_lags, 0.5, key="tc")
        for th in lists:
            assert [w for w in lists[th] if w[0] == 0] == want
        assert trig_tuples(recs) == want and n == len(want) and len(want) >= 4
        assert np.max(np.abs(pbar[0] - pbar_o[0])) <= 2e-3
        return
    want = _check(oms, gms, x, ph, pl, lags, chunks, host, gwi.BACKEND_TENSOR_SLIDES, key="tc")
    assert (2, N - 20000, N - 17000) in want and (1, 1096, 4096) in want and (0, 12000, 14048) in want
    assert not any(w[1] == 6000 for w in want)


def test_t2_tensor_core_kernel_past_tap_d512(tmpdir_s):
    """The pass-through on the PAST tap of a d = 512 block: the plateaus move 512 samples later, which only holds if
    the kernel's L2-resident history ring of whole past tiles delivers the right rows."""
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, gs.PAPER_ARCH, [dict(block=19, r=63, q=(5, 6), hid=(7, 8), past=True)], "tp")
    N, kstar, edge = 16 * FS, 2, 26112
    ph, pl = _instance(N, kstar, edge, a=6000)
    ph = [p for p in ph if p[0] != 0]
    x = np.stack([gs.plateau_square_wave(N, ph, -2, np.float16), gs.plateau_square_wave(N, pl, -3, np.float16)])
    _check(oms, gms, x, ph, pl, [kstar * FS], [edge, N - edge], False, gwi.BACKEND_TENSOR_SLIDES, shift=512)
