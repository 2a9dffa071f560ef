"""GPU parity of the streaming ensemble driver (gwi_stream_*) against the oracle (-m gpu).

Rows a-1, a-2, a-7..a-11 of SURVEY.md section 8: one causal pass over a stream pushed in ragged chunks (device and
pinned-host pushes), per-layer history carried across chunks, circular time slides on branch features, ensemble mean,
threshold, run clustering across chunk boundaries, records sorted by (slide, start).

Oracle side: gwo.Model.stream (direct definition over the whole stream), gwo.Model.head_slide (reading A24),
gwo.ensemble_mean, gwo.triggers.  Bars: FP32 mode 1e-5, FP16 mode 2e-3 on the mean probabilities; trigger lists exact
on delta-robust instances (P15: the oracle's lists at theta +- delta coincide); chunked == unchunked bit for bit.
"""
import os

import numpy as np
import pytest

import gwsynth as gs
from oracle import gwo
from tests.helpers import trig_tuples

pytestmark = pytest.mark.gpu

ARCH = gs.CFG1_ARCH


def _models(tmp, seeds, prec, bias="zero", arch=ARCH):
    import paper_2201_11133_b200 as gwi
    oms, gms = [], []
    for s in seeds:
        path = os.path.join(str(tmp), f"m{s}_{bias}_{arch.R}.gwim")
        gs.make_model_file(path, arch, s, bias=bias)
        oms.append(gwo.Model(path, round_fp16=(prec == gwi.FP16)))
        gms.append(gwi.load_model(path, prec, 0))
    return oms, gms


def _oracle_slides(oms, x, lags):
    """-> pbar [1+len(lags)][N] float64 by the definition."""
    N = x.shape[1]
    per = []
    for om in oms:
        p0, u = om.stream(x.astype(np.float64), want_u=True)
        ps = [p0] + [om.head_slide(u, lag) for lag in lags]
        per.append(ps)
    return np.stack([gwo.ensemble_mean([per[m][k] for m in range(len(oms))]) for k in range(1 + len(lags))])


def _oracle_triggers(pbar, theta, lmin):
    out = []
    for k in range(pbar.shape[0]):
        _, recs = gwo.triggers(pbar[k], theta, lmin, slide=k)
        out += [(r[0], r[1], r[2]) for r in recs]
    return out


def _run_stream(gms, x, chunks, lags, theta, lmin, host=False, max_chunk=None):
    import torch
    import paper_2201_11133_b200 as gwi
    N = x.shape[1]
    st = gwi.Stream(gms, N, max_chunk or max(chunks), theta, lmin, lags=lags, capacity=4096, want_pbar=True)
    xt = torch.from_numpy(x)
    if lags:
        nt = st.tail_samples
        assert nt == min(N, max(lags) + gms[0].receptive_field - 1)
        st.prime(xt[1, N - nt:].contiguous())
    pos = 0
    keep = []
    for n in chunks:
        a, b = xt[0, pos:pos + n].contiguous(), xt[1, pos:pos + n].contiguous()
        if host:
            a, b = a.pin_memory(), b.pin_memory()
        else:
            a, b = a.cuda(), b.cuda()
        keep.append((a, b))
        st.push(a, b)
        pos += n
    assert pos == N and st.samples_done == N
    n, recs = st.finish()
    pbar = st.pbar.cpu().numpy()
    st.close()
    return n, recs, pbar


def _ragged(N, seed, lo, hi):
    rs = np.random.RandomState(seed)
    out, left = [], N
    while left > 0:
        n = int(min(left, rs.randint(lo, hi)))
        out.append(n)
        left -= n
    return out


@pytest.mark.parametrize("prec_name,tol,bias", [("FP32", 1e-5, "zero"), ("FP32", 1e-5, "random"), ("FP16", 2e-3, "zero")])
def test_stream_ensemble_slides_parity(tmpdir_s, prec_name, tol, bias):
    import paper_2201_11133_b200 as gwi
    prec = getattr(gwi, prec_name)
    oms, gms = _models(tmpdir_s, [0, 1, 2, 3], prec, bias=bias)
    N = 3 * 4096 + 777
    dt = np.float16 if prec == gwi.FP16 else np.float32
    x = gs.stream_noise(1, 0, N, dtype=dt)
    lags = [4096, 2 * 4096, 5000]
    want = _oracle_slides(oms, x, lags)
    chunks = _ragged(N, 3, 1, 3000)
    n, recs, pbar = _run_stream(gms, x, chunks, lags, 0.5, 8, max_chunk=3000)
    err = np.max(np.abs(pbar - want))
    assert err <= tol, err
    got = trig_tuples(recs)
    assert n == len(got)
    # tier T1: the list equals the oracle's clustering of the GPU's own mean, exactly, for every input.  (Random weights
    # are never delta-robust at L_min = 8 -- SURVEY.md 8(c); tier T2, strain -> triggers against the oracle's own
    # probabilities, is tests/test_gpu_t2.py.)
    assert got == _oracle_triggers(pbar.astype(np.float64), float(np.float32(0.5)), 8)
    assert got == sorted(got)


def test_chunked_equals_unchunked_bitwise_and_host_push(tmpdir_s):
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0, 1], gwi.FP16)
    N = 40000
    x = gs.stream_noise(7, 0, N, dtype=np.float16)
    lags = [4096]
    n0, r0, p0 = _run_stream(gms, x, [N], lags, 0.5, 16)
    n1, r1, p1 = _run_stream(gms, x, _ragged(N, 5, 1, 9000), lags, 0.5, 16, max_chunk=9000)
    n2, r2, p2 = _run_stream(gms, x, _ragged(N, 6, 2000, 9000), lags, 0.5, 16, host=True, max_chunk=9000)
    assert np.array_equal(p0, p1) and np.array_equal(p0, p2)
    assert trig_tuples(r0) == trig_tuples(r1) == trig_tuples(r2) and n0 == n1 == n2
    for a, b in zip(r0, r1):
        assert a.peak_p == b.peak_p and abs(a.mean_p - b.mean_p) <= 1e-6 and a.model_mask == b.model_mask


def test_stream_equals_stitched_windows(tmpdir_s):
    """Reading A15 on the GPU: the last 2048 outputs of each 1 s window taken every 0.5 s equal the stream pass."""
    import torch
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0], gwi.FP32)
    N = 6 * 2048
    x = gs.stream_noise(9, 0, N, dtype=np.float32)
    _, _, pbar = _run_stream(gms, x, [5000, N - 5000], [], 0.5, 2048)
    nwin = (N - 4096) // 2048 + 1
    wins = np.stack([x[:, i * 2048:i * 2048 + 4096].T for i in range(nwin)])
    pw = gms[0].infer(torch.from_numpy(np.ascontiguousarray(wins)).cuda()).cpu().numpy()
    assert np.max(np.abs(pw[0] - pbar[0, :4096])) <= 1e-6
    for i in range(1, nwin):
        assert np.max(np.abs(pw[i, 2048:] - pbar[0, i * 2048 + 2048:i * 2048 + 4096])) <= 1e-6


def test_stream_triggers_with_plateaus_cross_chunks(tmpdir_s):
    """Tier T1 on many runs of many lengths: random Xavier models thresholded at the median of the oracle's mean, runs cut
    by ragged chunk boundaries, clustered by the GPU and by the oracle on the GPU's own mean."""
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0, 1, 2, 3], gwi.FP32)
    N = 30000
    x = gs.stream_noise(11, 0, N, dtype=np.float32)
    want = _oracle_slides(oms, x, [])
    theta = float(np.median(want[0]))           # half of the samples above: many runs of many lengths
    n, recs, pbar = _run_stream(gms, x, _ragged(N, 8, 100, 2500), [], theta, 3, max_chunk=2500)
    got = trig_tuples(recs)
    assert got == _oracle_triggers(pbar.astype(np.float64), float(np.float32(theta)), 3)
    assert len(got) > 20
    assert np.max(np.abs(pbar - want)) <= 1e-5


def test_stream_argument_errors(tmpdir_s):
    import torch
    import paper_2201_11133_b200 as gwi
    _, gms = _models(tmpdir_s, [0], gwi.FP32)
    st = gwi.Stream(gms, 1000, 500, lags=[100])
    x = torch.zeros(500, dtype=torch.float32, device="cuda")
    with pytest.raises(gwi.GwiError):      # slides need priming
        st.push(x, x)
    st.prime(torch.zeros(st.tail_samples, dtype=torch.float32))
    st.push(x, x)
    with pytest.raises(gwi.GwiError):      # finish before the stream is complete
        st.finish()
    with pytest.raises(gwi.GwiError):      # chunk larger than max_chunk
        st.push(torch.zeros(501, dtype=torch.float32, device="cuda"), torch.zeros(501, dtype=torch.float32, device="cuda"))
    st.push(x, x)
    with pytest.raises(gwi.GwiError):      # more than n_total
        st.push(x, x)
    n, recs = st.finish()
    assert n == len(recs)
    with pytest.raises(gwi.GwiError):      # a lag must be >= 1 (lags >= n_total wrap: test_stream_degenerate_sizes)
        gwi.Stream(gms, 1000, 500, lags=[0])


def test_full_hour_sampled_against_oracle(tmpdir_s):
    """configs[2] at full size, in the launch configuration bench.py times (one 1 h push, 4 models, FP16): the mean
    probability on sampled spans against the oracle evaluated on those spans alone (valid R_f - 1 samples in)."""
    import torch
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0, 1, 2, 3], gwi.FP16)
    N = 3600 * 4096
    g = torch.Generator().manual_seed(5)
    xt = torch.randn((2, N), generator=g).to(torch.float16)
    st = gwi.Stream(gms, N, N, 0.5, 2048, capacity=4096, want_pbar=True)
    xd = xt.cuda()
    st.push(xd[0], xd[1])
    n, recs = st.finish()
    x = xt.numpy()
    rf = gms[0].receptive_field
    for s0 in [0, 111, 4096 * 1800 - 7, N - 5000]:
        span = x[:, s0:s0 + 5000].astype(np.float64)
        want = gwo.ensemble_mean([om.stream(span) for om in oms])
        got = st.pbar[0, s0:s0 + 5000].cpu().numpy()
        lo = 0 if s0 == 0 else rf - 1
        assert np.max(np.abs(got[lo:] - want[lo:])) <= 2e-3
    pb = st.pbar[0].cpu().numpy()
    assert np.isfinite(pb).all() and 0.0 <= pb.min() and pb.max() <= 1.0
    st.close()


@pytest.mark.parametrize("prec_name,tol", [("FP16", 2e-3), ("FP32", 1e-5)])
@pytest.mark.parametrize("N,chunks,lags", [(1, [1], []), (5, [1, 1, 1, 1, 1], [3]), (17, [16, 1], [16]),
                                           (113, [112, 1], []), (225, [1, 111, 113], [1, 224]),
                                           (4096, [4096], [4095]),
                                           (300, [100, 200], [307, 600, 1203])])      # lags >= N wrap (k fs >= N)
def test_stream_degenerate_sizes(tmpdir_s, prec_name, tol, N, chunks, lags):
    """Streams shorter than the receptive field / the kernel halo / one tile, one-sample chunks, lags next to N."""
    import paper_2201_11133_b200 as gwi
    prec = getattr(gwi, prec_name)
    oms, gms = _models(tmpdir_s, [0, 1], prec, bias="random")
    dt = np.float16 if prec == gwi.FP16 else np.float32
    x = gs.stream_noise(21, 0, N, dtype=dt)
    want = _oracle_slides(oms, x, lags)
    n, recs, pbar = _run_stream(gms, x, chunks, lags, 0.5, 1)
    assert np.max(np.abs(pbar - want)) <= tol
    assert trig_tuples(recs) == _oracle_triggers(pbar.astype(np.float64), float(np.float32(0.5)), 1)


def test_stream_generic_path_paper_scale_fp32(tmpdir_s):
    """The generic back end (any architecture) on the paper-scale model: carried per-layer history over dilations up
    to 512, chunks shorter than the receptive field."""
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0], gwi.FP32, bias="random", arch=gs.PAPER_ARCH)
    N = 5000
    x = gs.stream_noise(23, 0, N, dtype=np.float32)
    want = _oracle_slides(oms, x, [4096])
    n, recs, pbar = _run_stream(gms, x, _ragged(N, 4, 100, 900), [4096], 0.5, 4, max_chunk=900)
    assert np.max(np.abs(pbar - want)) <= 1e-5


def test_stream_paper_scale_tensor_core_back_end(tmpdir_s):
    """FP16 stream of paper-scale models: segments with recomputed warm-up through the fused tcgen05 kernel.  Parity
    with the oracle's one-pass definition, and chunked == unchunked bit for bit."""
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0, 1], gwi.FP16, arch=gs.PAPER_ARCH)
    assert all(g.uses_tensor_cores for g in gms)
    N = 40000
    x = gs.stream_noise(31, 0, N, dtype=np.float16)
    want = _oracle_slides(oms, x, [])
    n0, r0, p0 = _run_stream(gms, x, [N], [], 0.5, 16)
    assert np.max(np.abs(p0 - want)) <= 2e-3
    n1, r1, p1 = _run_stream(gms, x, _ragged(N, 2, 1000, 17000), [], 0.5, 16, max_chunk=17000)
    assert np.array_equal(p0, p1)
    assert trig_tuples(r0) == trig_tuples(r1)
    assert trig_tuples(r0) == _oracle_triggers(p0.astype(np.float64), float(np.float32(0.5)), 16)


def test_per_model_rule_and_coincidence(tmpdir_s):
    """The paper's decision rule (reading A34) end to end: per-model triggers from the stream in
    GWI_RULE_PER_MODEL mode, all-model coincidence on the host, against the oracle on the same probabilities."""
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0, 1, 2], gwi.FP16)
    N = 30000
    x = gs.stream_noise(41, 0, N, dtype=np.float16)
    st = gwi.Stream(gms, N, 7000, 0.5, 3, lags=[4096], capacity=1 << 16, want_pbar=True, rule=gwi.RULE_PER_MODEL)
    import torch
    xt = torch.from_numpy(x)
    st.prime(xt[1, N - st.tail_samples:].contiguous())
    pos = 0
    for n in _ragged(N, 9, 500, 7000):
        st.push(xt[0, pos:pos + n].contiguous().cuda(), xt[1, pos:pos + n].contiguous().cuda())
        pos += n
    cnt, recs = st.finish()
    p = st.pbar.cpu().numpy()                                   # [slide][model][N]
    st.close()
    assert cnt == len(recs) and cnt > 10
    # per-model probabilities against the oracle's definition
    for m, om in enumerate(oms):
        p0, u = om.stream(x.astype(np.float64), want_u=True)
        assert np.max(np.abs(p[0, m] - p0)) <= 2e-3
        assert np.max(np.abs(p[1, m] - om.head_slide(u, 4096))) <= 2e-3
    # threshold at each model's own median so that every model has many runs
    # (records were produced with theta = 0.5; compare those against the oracle's clustering of the same arrays)
    want_recs = []
    for k in range(2):
        for m in range(3):
            _, rr = gwo.triggers(p[k, m].astype(np.float64), float(np.float32(0.5)), 3, slide=k)
            want_recs += [(k, 1 << m, r[1], r[2]) for r in rr]
    got_recs = sorted((r.slide, r.model_mask, r.start, r.end) for r in recs)
    assert got_recs == sorted(want_recs)
    # coincidence within 0.5 s
    ev = gwi.coincidence(recs, 3, 2048)
    want_ev = []
    for k in range(2):
        ends = [[r[3] for r in want_recs if r[0] == k and r[1] == 1 << m] for m in range(3)]
        want_ev += [(k,) + e for e in gwo.coincidence(ends, 2048, slide=k)]
    assert [(e.slide, e.t_first, e.t_last, e.n_triggers) for e in ev] == want_ev


def test_config3_recipe_32_slides(tmpdir_s):
    """BASELINE.json configs[3] recipe at a size the oracle finishes: coloured-then-whitened noise (reading A27), the
    4-model ensemble, circular lags k x 1 s for k = 1..32 (reading A24, A25), all slides in one pass."""
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0, 1, 2, 3], gwi.FP16)
    N = 33 * 4096 + 1234
    x = np.stack([gs.coloured_whitened_noise(2 + d, d, N, seg_len=1 << 16) for d in range(2)])
    assert x.dtype == np.float16 and abs(float(x.astype(np.float64).std()) - 1.0) < 0.05
    lags = [k * 4096 for k in range(1, 33)]
    want = _oracle_slides(oms, x, lags)
    n, recs, pbar = _run_stream(gms, x, _ragged(N, 12, 9000, 40000), lags, 0.5, 64, max_chunk=40000)
    assert np.max(np.abs(pbar - want)) <= 2e-3
    got = trig_tuples(recs)
    assert got == _oracle_triggers(pbar.astype(np.float64), float(np.float32(0.5)), 64) and got == sorted(got)


@pytest.mark.parametrize("impl", ["1", "2"])
def test_config3_recipe_with_the_other_head_kernels(impl):
    """The slide heads have three implementations for regular lag lists (csrc/gwi_heads.cu: the tensor-path diagonal kernel
    is the default, GWI_HEADS_IMPL=1 the element-wise diagonal kernel, 2 the thread-per-item comb kernel).  The switch is read
    once per process, so the configs[3] parity test runs again in a child process under each of the other two."""
    import subprocess
    import sys
    env = dict(os.environ, GWI_HEADS_IMPL=impl)
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    r = subprocess.run([sys.executable, "-m", "pytest", "tests/test_gpu_stream.py", "-m", "gpu", "-x", "-q", "-k",
                        "test_config3_recipe_32_slides"], cwd=root, env=env, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0 and "1 passed" in r.stdout, r.stdout[-2000:] + r.stderr[-2000:]


def test_stream_narrow_arch_40_regular_lags_two_passes(tmpdir_s):
    """More regular lags than one pass of the comb heads holds (34): the diagonal kernel in two passes of 21 and 20 lags,
    on chunk lengths that are not multiples of its 16-row blocks."""
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0, 1, 2], gwi.FP16)
    N = 41 * 256 + 3000 + 7
    x = gs.stream_noise(36, 0, N, dtype=np.float16)
    lags = [k * 256 for k in range(1, 41)]
    want = _oracle_slides(oms, x, lags)
    n, recs, pbar = _run_stream(gms, x, _ragged(N, 4, 1000, 5000), lags, 0.5, 40, max_chunk=5000)
    assert np.max(np.abs(pbar - want)) <= 2e-3
    assert trig_tuples(recs) == _oracle_triggers(pbar.astype(np.float64), float(np.float32(0.5)), 40)


def test_stream_paper_scale_slides_tensor_core_back_end(tmpdir_s):
    """FP16 stream of paper-scale models WITH time slides: chunks re-blocked into whole segments, L1 feature tiles kept
    as history, one tcgen05 head launch per lag.  Parity with the oracle; chunked == unchunked bit for bit."""
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0, 1], gwi.FP16, arch=gs.PAPER_ARCH)
    N = 128 * 300
    x = gs.stream_noise(33, 0, N, dtype=np.float16)
    lags = [4096, 12800]
    want = _oracle_slides(oms, x, lags)
    n0, r0, p0 = _run_stream(gms, x, [N], lags, 0.5, 16)
    assert np.max(np.abs(p0 - want)) <= 2e-3
    n1, r1, p1 = _run_stream(gms, x, _ragged(N, 3, 1, 20000), lags, 0.5, 16, max_chunk=20000)
    assert np.array_equal(p0, p1)
    assert trig_tuples(r0) == trig_tuples(r1)
    assert trig_tuples(r0) == _oracle_triggers(p0.astype(np.float64), float(np.float32(0.5)), 16)


@pytest.mark.parametrize("seeds,G,K,check", [([0, 1], 2048, 7, None), ([0], 1024, 36, [0, 1, 2, 17, 18, 19, 34, 35])])
def test_stream_paper_scale_regular_lags_comb_heads(tmpdir_s, seeds, G, K, check):
    """Paper-scale models with a regular lag list k x G: the half-head rows v from the tensor cores, then the comb-scheduled
    element-wise heads fused with the ensemble mean and the threshold (one pass for 7 slides, two passes of 18 for 36).
    Parity of pbar with the oracle on every slide (on a spread of slides for the long list), triggers from pbar."""
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, seeds, gwi.FP16, arch=gs.PAPER_ARCH)
    # long enough for the largest lag plus several ragged chunks; the oracle costs about a minute per model per 40 000
    # samples on the GPU box's host cores, so the two-model case takes the shorter stream
    N = 128 * 320 if (K - 1) * G > 128 * 150 else 128 * 200
    x = gs.stream_noise(35, 0, N, dtype=np.float16)
    lags = [k * G for k in range(1, K)]
    n, recs, pbar = _run_stream(gms, x, _ragged(N, 4, 3000, 16000), lags, 0.5, 16, max_chunk=16000)
    ks = list(range(K)) if check is None else check
    want = _oracle_slides(oms, x, [lags[k - 1] for k in ks if k > 0])
    assert ks[0] == 0 and np.max(np.abs(pbar[ks] - want)) <= 2e-3
    got = trig_tuples(recs)
    assert got == _oracle_triggers(pbar.astype(np.float64), float(np.float32(0.5)), 16)
    # the same stream in one push: bit-identical
    n1, r1, p1 = _run_stream(gms, x, [N], lags, 0.5, 16)
    assert np.array_equal(pbar, p1) and trig_tuples(r1) == got


@pytest.mark.parametrize("lags", [[], [4096, 12800]])
def test_paper_scale_long_block_segment_choice(tmpdir_s, lags):
    """A block long enough that the tensor-core back ends pick segments longer than the minimum (pick_seg: > 296
    minimum-length segments per launch): one 6 M-sample push against the same stream in 1 M-sample pushes (minimum-length
    segments) bit for bit, and sampled spans against the oracle evaluated on those spans alone."""
    import torch
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0], gwi.FP16, arch=gs.PAPER_ARCH)
    N = 128 * 46872
    g = torch.Generator().manual_seed(11)
    xt = torch.randn((2, N), generator=g).to(torch.float16)
    xd = xt.cuda()
    outs = []
    for chunk in (N, 1 << 20):
        st = gwi.Stream(gms, N, chunk, 0.5, 2048, lags=lags, capacity=4096, want_pbar=True)
        if lags:
            st.prime(xd[1, N - st.tail_samples:].contiguous())
        for p in range(0, N, chunk):
            st.push(xd[0, p:p + chunk].contiguous(), xd[1, p:p + chunk].contiguous())
        n, recs = st.finish()
        outs.append((n, trig_tuples(recs), st.pbar.cpu().numpy()))
        st.close()
    assert outs[0][0] == outs[1][0] and outs[0][1] == outs[1][1]
    assert np.array_equal(outs[0][2], outs[1][2])
    pb = outs[0][2]
    assert np.isfinite(pb).all() and 0.0 <= pb.min() and pb.max() <= 1.0
    x = xt.numpy()
    rf = gms[0].receptive_field
    for s0 in [0, 40578 - 2100, 2_999_000, N - rf - 300]:
        span = x[:, s0:s0 + rf + 300].astype(np.float64)
        want = oms[0].stream(span)
        lo = 0 if s0 == 0 else rf - 1
        got = pb[0, s0:s0 + rf + 300]
        assert np.max(np.abs(got[lo:] - want[lo:])) <= 2e-3


@pytest.mark.parametrize("lags", [[], [4096, 12800]])
def test_paper_scale_host_push_equals_device_push(tmpdir_s, lags):
    """The tensor-core back ends fed through gwi_stream_push_host (pinned host chunks, side-stream copies into the
    staging buffers: the path bench.py's month legs use) against one device push, bit for bit."""
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0], gwi.FP16, arch=gs.PAPER_ARCH)
    N = 128 * 330
    x = gs.stream_noise(41, 0, N, dtype=np.float16)
    n0, r0, p0 = _run_stream(gms, x, [N], lags, 0.5, 16)
    n1, r1, p1 = _run_stream(gms, x, _ragged(N, 8, 3000, 15000), lags, 0.5, 16, host=True, max_chunk=15000)
    assert np.array_equal(p0, p1)
    assert n0 == n1 and trig_tuples(r0) == trig_tuples(r1)


def test_config4_month_recipe_hour_chunks_from_host(tmpdir_s):
    """BASELINE.json configs[4] recipe (SURVEY.md 8(d) cfg 5): one-hour chunks, chunk c detector d
    seeded (5, d, c), the 20 seeded A26 chirps, pushed from pinned host memory through gwi_stream_push_host.  The stream
    is month-chunks 0, 1 and the two chunks that hold the first two injections (4 h; the oracle cannot do 744).  The mean
    probability is compared with the oracle on the sub-spans BASELINE.md names: the start of chunk 0, the 0 -> 1 chunk
    boundary +- 2 s, the two injection sites; the trigger list is the oracle's clustering of the GPU's mean (T1) and,
    where the oracle's own spans allow a statement, empty as SURVEY.md 8(c) predicts for random weights."""
    import torch
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0, 1, 2, 3], gwi.FP16)
    n = gs.CFG5_CHUNK
    inj = gs.cfg5_injections()
    assert len(inj) == 20
    cA, cB = inj[0][0] // n, inj[1][0] // n
    assert 1 < cA < cB
    month_chunks = [0, 1, cA, cB]
    N = len(month_chunks) * n
    st = gwi.Stream(gms, N, n, 0.5, 2048, capacity=4096, want_pbar=True)
    assert st.backend == gwi.BACKEND_NARROW
    host = []
    for c in month_chunks:
        xc = torch.from_numpy(gs.cfg5_chunk(c, injections=inj))
        host.append((xc[0].contiguous().pin_memory(), xc[1].contiguous().pin_memory()))
        st.push(*host[-1])
    cnt, recs = st.finish()
    pb = st.pbar[0].cpu().numpy()
    st.close()
    x = np.concatenate([np.stack([h.numpy(), l.numpy()]) for h, l in host], axis=1)
    rf = gms[0].receptive_field
    spans = [(0, 8192), (n - 2 * 4096, n + 2 * 4096)]
    for j, c in ((0, 2), (1, 3)):
        loc = inj[j][0] - month_chunks[c] * n + c * n           # the chirp's end inside the 4 h stream
        spans.append((max(loc - 6000, c * n), min(loc + 2000, (c + 1) * n)))
        w = gs.chirp_waveform(inj[j][1])
        assert np.abs(x[:, max(loc - len(w), c * n):loc].astype(np.float64)).max() > 0   # the chirp lies in the chunk
    for a, b in spans:
        span = x[:, a:b].astype(np.float64)
        want = gwo.ensemble_mean([om.stream(span) for om in oms])
        lo = 0 if a == 0 else rf - 1
        assert np.max(np.abs(pb[a + lo:b] - want[lo:])) <= 2e-3, (a, b)
        # no oracle sample of these spans stays above theta + delta for 0.5 s: no trigger can lie inside them
        assert gwo.triggers(want[lo:], 0.5 - 2e-3, 2048)[0] == 0
    got = trig_tuples(recs)
    assert cnt == len(got)
    assert got == _oracle_triggers(pb[None].astype(np.float64), float(np.float32(0.5)), 2048)
    assert all(not (s < b and e > a) for _, s, e in got for a, b in spans)


def test_paper_scale_slides_one_push_larger_than_the_internal_block(tmpdir_s):
    """A single push far larger than the tensor-core back end's internal block (sub <= 2^24 samples) with time slides:
    the push is consumed in pieces, so the pending-sample and remainder buffers cannot overflow whatever max_chunk is.
    One 40.1 M-sample push against the same stream in 4 M-sample pushes, bit for bit."""
    import torch
    import paper_2201_11133_b200 as gwi
    oms, gms = _models(tmpdir_s, [0], gwi.FP16, arch=gs.PAPER_ARCH)
    N = 128 * 313_500                                   # 40 128 000 samples
    g = torch.Generator().manual_seed(13)
    xd = torch.randn((2, N), generator=g).to(torch.float16).cuda()
    lags = [4096]
    outs = []
    for chunk in (N, 1 << 22):
        st = gwi.Stream(gms, N, chunk, 0.5, 2048, lags=lags, capacity=4096, want_pbar=True)
        assert st.backend == gwi.BACKEND_TENSOR_SLIDES
        st.prime(xd[1, N - st.tail_samples:].contiguous())
        for p in range(0, N, chunk):
            st.push(xd[0, p:p + chunk].contiguous(), xd[1, p:p + chunk].contiguous())
        n, recs = st.finish()
        outs.append((n, trig_tuples(recs), st.pbar.clone()))
        st.close()
    assert outs[0][0] == outs[1][0] and outs[0][1] == outs[1][1]
    assert torch.equal(outs[0][2], outs[1][2])
    pb = outs[0][2]
    assert bool(torch.isfinite(pb).all()) and float(pb.min()) >= 0.0 and float(pb.max()) <= 1.0
    x = xd.cpu().numpy()
    rf = gms[0].receptive_field
    for s0 in [(1 << 24) - 1000, N - rf - 300]:         # across the internal block edge, and the stream's end
        span = x[:, s0:s0 + rf + 300].astype(np.float64)
        want = oms[0].stream(span)
        got = pb[0, s0:s0 + rf + 300].cpu().numpy()
        assert np.max(np.abs(got[rf - 1:] - want[rf - 1:])) <= 2e-3


@pytest.mark.parametrize("arch_name", ["cfg1", "generic"])
def test_prime_then_host_push_without_host_sync(tmpdir_s, arch_name):
    """C-ABI ordering: gwi_stream_prime leaves its kernels running on the caller's stream while they read the tail out
    of staging buffer 0; the first gwi_stream_push_host copies into that buffer on the side stream and has to wait
    for them.  No host synchronisation between the two calls; result equal to the synchronised run bit for bit."""
    import torch
    import paper_2201_11133_b200 as gwi
    prec = gwi.FP16 if arch_name == "cfg1" else gwi.FP32
    oms, gms = _models(tmpdir_s, [0, 1, 2, 3], prec)
    dt = np.float16 if prec == gwi.FP16 else np.float32
    N = 400_000
    x = torch.from_numpy(gs.stream_noise(51, 0, N, dtype=dt))
    lags = [300_000]                                    # a long tail: the prime kernels run for a while
    res = []
    for sync in (True, False):
        st = gwi.Stream(gms, N, N, 0.5, 16, lags=lags, capacity=1 << 16, want_pbar=True)
        tail = x[1, N - st.tail_samples:].contiguous().pin_memory()
        h, l = x[0].contiguous().pin_memory(), x[1].contiguous().pin_memory()
        st.prime(tail, sync=sync)
        st.push(h, l)
        n, recs = st.finish()
        res.append((n, trig_tuples(recs), st.pbar.clone()))
        st.close()
    assert res[0][0] == res[1][0] and res[0][1] == res[1][1] and torch.equal(res[0][2], res[1][2])
