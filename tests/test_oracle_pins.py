"""Pins for the oracle (oracle/gwo_oracle.c): what the definition and the mathematics fix, independent of it.

Every test cites the pin id of DESIGN.md section "Pins" (= SURVEY.md 8(c) C.4).  None of the expected values
below comes from the oracle or from the CUDA path: they are hand-computed fixtures (tests/golden), closed
forms, invariants, numpy library routines (numpy.convolve) or brute-force definitions.
"""
import math
import os

import numpy as np
import pytest

import gwsynth as gs
from gwsynth import rng
from oracle import gwo

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rand(seed, stream, n):
    return rng.normal(seed, stream, 0, n)


def _model(tmpdir_s, name, arch, tensors, fp16=False):
    path = os.path.join(str(tmpdir_s), name + ".gwim")
    gs.write_model(path, arch, tensors)
    return gwo.Model(path, round_fp16=fp16)


@pytest.fixture(scope="module")
def small(tmpdir_s):
    """config-1 architecture (R_f = 16) with random biases, two branches."""
    a = gs.CFG1_ARCH
    t = gs.xavier_tensors(a, seed=7, bias="random")
    return a, t, _model(tmpdir_s, "small", a, t)


# ---- P1 causality / P2 receptive-field extent -----------------------------------------------------------
def test_p1_p2_causality_and_receptive_field(small):
    a, _, m = small
    T, t0 = 96, 40
    x = np.stack([_rand(11, 0, T), _rand(11, 1, T)])
    p0, u0 = m.forward(x, want_u=True)
    for c in range(2):
        y = x.copy()
        y[c, t0] += 0.75
        p1, u1 = m.forward(y, want_u=True)
        Rf = a.receptive_field
        assert Rf == 16 == m.receptive_field
        # P1: nothing before t0 changes, bit for bit
        assert np.array_equal(p0[:t0], p1[:t0]) and np.array_equal(u0[:, :, :t0], u1[:, :, :t0])
        # P2: nothing at t >= t0 + R_f changes; t0 + R_f - 1 does (generic weights)
        assert np.array_equal(p0[t0 + Rf:], p1[t0 + Rf:]) and np.array_equal(u0[:, :, t0 + Rf:], u1[:, :, t0 + Rf:])
        assert u0[c, :, t0 + Rf - 1].tolist() != u1[c, :, t0 + Rf - 1].tolist()
        assert p0[t0] != p1[t0]
        # branch independence (P9a): the other branch's features are untouched everywhere
        assert np.array_equal(u0[1 - c], u1[1 - c])


def test_p2_paper_scale_receptive_field_value():
    assert gs.PAPER_ARCH.receptive_field == 2047 and gs.PAPER_ARCH.L == 20
    assert gs.PAPER_ARCH.flops_per_timestep() == 2359808 and gs.CFG1_ARCH.flops_per_timestep() == 32896


# ---- P3 linearity of one conv layer, bias at padded positions -------------------------------------------
def test_p3_linearity_and_bias():
    T, Cin, Cout, k, d = 50, 3, 4, 2, 5
    W = _rand(3, 0, Cout * Cin * k).reshape(Cout, Cin, k)
    x = _rand(3, 1, Cin * T).reshape(Cin, T)
    y = _rand(3, 2, Cin * T).reshape(Cin, T)
    al, be = 1.7, -0.3
    lhs = gwo.conv1d_causal(al * x + be * y, W, None, d)
    rhs = al * gwo.conv1d_causal(x, W, None, d) + be * gwo.conv1d_causal(y, W, None, d)
    assert np.max(np.abs(lhs - rhs)) < 1e-14
    b = _rand(3, 3, Cout)
    z = gwo.conv1d_causal(np.zeros((Cin, T)), W, b, d)
    assert np.array_equal(z, np.repeat(b[:, None], T, axis=1))      # conv(0) == b at EVERY t (reading A4)


# ---- P4 dilation <-> polyphase, shift equivariance -------------------------------------------------------
def test_p4_polyphase_and_shift():
    T, Cin, Cout, k, d = 60, 2, 3, 2, 4
    W = _rand(4, 0, Cout * Cin * k).reshape(Cout, Cin, k)
    b = _rand(4, 1, Cout)
    x = _rand(4, 2, Cin * T).reshape(Cin, T)
    y = gwo.conv1d_causal(x, W, b, d)
    for rho in range(d):
        yp = gwo.conv1d_causal(np.ascontiguousarray(x[:, rho::d]), W, b, 1)
        assert np.array_equal(y[:, rho::d], yp)
    tau = 7
    xs = np.concatenate([np.zeros((Cin, tau)), x[:, :-tau]], axis=1)
    ys = gwo.conv1d_causal(xs, W, None, d)
    y0 = gwo.conv1d_causal(x, W, None, d)
    assert np.array_equal(ys[:, tau:], y0[:, :-tau])


# ---- P12 one layer against numpy.convolve (textbook FIR) -------------------------------------------------
@pytest.mark.parametrize("k,d", [(2, 1), (2, 3), (3, 2), (2, 64)])
def test_p12_numpy_convolve(k, d):
    T, Cin, Cout = 40, 2, 2
    W = _rand(5, k * 10 + d, Cout * Cin * k).reshape(Cout, Cin, k)
    x = _rand(5, 99, Cin * T).reshape(Cin, T)
    y = gwo.conv1d_causal(x, W, None, d)
    ref = np.zeros((Cout, T))
    for o in range(Cout):
        for c in range(Cin):
            h = np.zeros((k - 1) * d + 1)          # impulse response: tap j sits (k-1-j)*d samples in the past
            for j in range(k):
                h[(k - 1 - j) * d] = W[o, c, j]
            ref[o] += np.convolve(x[c], h)[:T]
    assert np.max(np.abs(y - ref)) < 1e-13


# ---- P5 / P6 hand-worked examples ------------------------------------------------------------------------
def _load_table(name):
    rows = []
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                rows.append([float(v) for v in line.split()])
    return rows


def test_p5_worked_example_A(tmpdir_s):
    a = gs.Arch(n_branch=2, c_in=1, R=1, S=1, k=2, dil=(1,), Hh=1)
    t = gs.zero_tensors(a)
    t["b0.W_in"][:] = 1.0
    t["b1.W_in"][:] = 1.0
    t["b0.l0.Wf"][0, 0] = [0.5, 1.0]          # [past, current]
    t["b0.l0.Ws"][0, 0] = 2.0
    t["b1.l0.Wf"][0, 0] = [-1.0, 1.0]
    t["b1.l0.Wg"][0, 0] = [0.0, 1.0]
    t["b1.l0.Ws"][0, 0] = 1.0
    t["b1.l0.bs"][0] = 0.1
    t["W1"][0] = [1.0, 2.0]
    t["b1"][0] = -0.5
    t["W2"][0] = 3.0
    t["b2"][0] = -1.0
    m = _model(tmpdir_s, "p5", a, t)
    x = np.array([[1, -1, 2, 0], [0, 1, 1, -2]], dtype=np.float64)
    p, u = m.forward(x, want_u=True)
    tab = np.array(_load_table("p5_worked_example_A.txt"))
    # bs = 0.1 is stored as fp32 in the model file (0.1f - 0.1 = 1.5e-9): tolerance 1e-6 as the fixture states
    assert np.max(np.abs(u[0, 0] - tab[:, 1])) < 1e-6
    assert np.max(np.abs(u[1, 0] - tab[:, 2])) < 1e-6
    assert np.max(np.abs(p - tab[:, 5])) < 1e-6
    # the two spot values the fixture quotes for z_L
    assert abs(math.tanh(1) / (1 + math.exp(-1)) - 0.556770) < 1e-6
    # window API (channels-last) gives the same numbers: pins the [B][T][C] de-interleave
    pw = m.infer_windows(np.ascontiguousarray(x.T)[None])
    assert np.array_equal(pw[0], p)


def test_p6_worked_example_B(tmpdir_s):
    a = gs.Arch(n_branch=1, c_in=1, R=1, S=1, k=2, dil=(1, 2), Hh=1)
    t = gs.zero_tensors(a)
    t["b0.W_in"][:] = 1.0
    t["b0.l0.Wf"][0, 0] = [1.0, 1.0]
    t["b0.l0.Wr"][0, 0] = 2.0
    t["b0.l0.Ws"][0, 0] = 1.0
    t["b0.l1.Wf"][0, 0] = [1.0, 0.0]          # past tap only
    t["b0.l1.bg"][0] = math.log(3.0)
    t["b0.l1.Ws"][0, 0] = 1.0
    m = _model(tmpdir_s, "p6", a, t)
    x = np.array([[1, -1, 2, 0, 0.5, -2]], dtype=np.float64)
    u, h = m.branch(0, x, dump_h=True)
    tab = np.array(_load_table("p6_worked_example_B.txt"))
    assert np.max(np.abs(h[1, 0] - tab[:, 1])) < 1e-6     # ln 3 is stored as fp32: 2e-8 effect
    assert np.max(np.abs(u[0] - tab[:, 2])) < 1e-6


# ---- P7 degenerate closed forms --------------------------------------------------------------------------
def test_p7_closed_forms(tmpdir_s, small):
    a, t, m = small
    T = 40
    x = np.stack([_rand(21, 0, T), _rand(21, 1, T)])
    # (i) everything zero except b2 -> p == sigma(b2)
    z = gs.zero_tensors(a)
    z["b2"][0] = 0.7
    mz = _model(tmpdir_s, "p7i", a, z)
    assert np.allclose(mz.forward(x), 1.0 / (1.0 + math.exp(-float(np.float32(0.7)))), atol=1e-15)
    # (ii) zero input, zero biases -> p == 0.5 exactly, no triggers under strict '>'
    t0 = gs.xavier_tensors(a, seed=3, bias="zero")
    m0 = _model(tmpdir_s, "p7ii", a, t0)
    p = m0.forward(np.zeros((2, T)))
    assert np.all(p == 0.5)
    assert gwo.triggers(p, 0.5, 1)[0] == 0
    # (iii) negating W2, b2 maps p -> 1 - p
    tn = {k: v.copy() for k, v in t.items()}
    tn["W2"] *= -1
    tn["b2"] *= -1
    mn = _model(tmpdir_s, "p7iii", a, tn)
    assert np.max(np.abs(mn.forward(x) + m.forward(x) - 1.0)) < 1e-15
    # (iv) f, g -> +inf gives z -> 1: one block, bf = bg = 40, Ws = 1 -> u = S ones * R
    a1 = gs.Arch(n_branch=1, c_in=1, R=3, S=2, k=2, dil=(1,), Hh=1)
    t1 = gs.zero_tensors(a1)
    t1["b0.l0.bf"][:] = 40.0
    t1["b0.l0.bg"][:] = 40.0
    t1["b0.l0.Ws"][:] = 1.0
    m1 = _model(tmpdir_s, "p7iv", a1, t1)
    assert np.allclose(m1.branch(0, np.zeros((1, 5))), 3.0, atol=1e-12)
    # (v) dilation >= T: the past tap only reads padding -> same as a 1x1 with the current-tap weights
    W = _rand(22, 0, 2 * 2 * 2).reshape(2, 2, 2)
    xx = _rand(22, 1, 2 * 10).reshape(2, 10)
    assert np.array_equal(gwo.conv1d_causal(xx, W, None, 10), gwo.conv1d_causal(xx, W[:, :, 1:], None, 1))


# ---- P8 windowed + stitching == one stream pass ----------------------------------------------------------
def test_p8_windowed_equals_stream(small):
    a, _, m = small
    Wn, stride = 64, 32                        # R_f - 1 = 15 <= Wn - stride = 32
    N = stride * 9 + Wn
    x = np.stack([_rand(31, 0, N), _rand(31, 1, N)])
    ps = m.stream(x)
    nwin = (N - Wn) // stride + 1
    wins = np.stack([x[:, w * stride:w * stride + Wn].T for w in range(nwin)])       # [B][T][2]
    pw = m.infer_windows(wins)
    st = np.empty(N)
    st[:Wn] = pw[0]
    for w in range(1, nwin):                   # reading A15: the LAST `stride` outputs are authoritative
        st[w * stride + Wn - stride:w * stride + Wn] = pw[w, Wn - stride:]
    assert np.array_equal(st, ps)
    # negative test: taking each window's FIRST half (zero-padded warm-up) must differ
    bad = np.empty(N)
    for w in range(nwin):
        bad[w * stride:w * stride + stride] = pw[w, :stride]
    assert np.max(np.abs(bad[stride:nwin * stride] - ps[stride:nwin * stride])) > 1e-6
    # segmented evaluation (memory bound) is bit-identical to the whole pass, any segment length
    for seg in (1, 17, 100, N):
        assert np.array_equal(m.stream(x, seg=seg), ps)


# ---- P9 slide reuse ---------------------------------------------------------------------------------------
def test_p9_slide_equals_rolled_input_outside_seams(small):
    a, _, m = small
    N, lag = 200, 37
    x = np.stack([_rand(41, 0, N), _rand(41, 1, N)])
    _, u = m.stream(x, want_u=True)
    pk = m.head_slide(u, lag)
    xr = np.stack([x[0], np.roll(x[1], lag)])          # L1 delayed: L1'[t] = L1[t - lag] (circular, A24)
    pr = m.forward(xr)
    Rf = a.receptive_field
    seam = np.zeros(N, dtype=bool)
    seam[0:Rf - 1] = True
    seam[lag:lag + Rf - 1] = True
    assert np.max(np.abs(pk[~seam] - pr[~seam])) < 1e-14
    assert np.max(np.abs(pk[seam] - pr[seam])) > 1e-6   # and the seams are exactly where they differ
    assert np.array_equal(m.head_slide(u, 0), m.stream(x))
    assert np.array_equal(m.head_slide(u, lag + 3 * N), pk)     # lag wraps modulo N


# ---- P10 channel-permutation equivariance -----------------------------------------------------------------
def test_p10_channel_permutation(tmpdir_s, small):
    a, t, m = small
    T = 48
    x = np.stack([_rand(51, 0, T), _rand(51, 1, T)])
    pr = np.argsort(_rand(52, 0, a.R))
    ps_ = np.argsort(_rand(52, 1, a.S))
    ph = np.argsort(_rand(52, 2, a.Hh))
    q = {}
    for b in range(a.n_branch):
        q[f"b{b}.W_in"] = t[f"b{b}.W_in"][pr]
        q[f"b{b}.b_in"] = t[f"b{b}.b_in"][pr]
        for i in range(a.L):
            n = f"b{b}.l{i}."
            for w in ("Wf", "Wg", "Wr"):
                q[n + w] = t[n + w][pr][:, pr]
            for w in ("bf", "bg", "br"):
                q[n + w] = t[n + w][pr]
            q[n + "Ws"] = t[n + "Ws"][ps_][:, pr]
            q[n + "bs"] = t[n + "bs"][ps_]
    cat = np.concatenate([ps_ + b * a.S for b in range(a.n_branch)])
    q["W1"] = t["W1"][ph][:, cat]
    q["b1"] = t["b1"][ph]
    q["W2"] = t["W2"][ph]
    q["b2"] = t["b2"]
    mq = _model(tmpdir_s, "p10", a, q)
    assert np.max(np.abs(mq.forward(x) - m.forward(x))) < 1e-13


# ---- P11 batch independence; ensemble of copies ------------------------------------------------------------
def test_p11_batch_independence(small):
    a, _, m = small
    B, T = 5, 33
    x = np.stack([_rand(61, c, B * T).reshape(B, T) for c in range(2)], axis=-1)       # [B][T][2]
    p = m.infer_windows(x)
    perm = [3, 0, 4, 1, 2]
    assert np.array_equal(m.infer_windows(x[perm]), p[perm])
    assert np.array_equal(m.infer_windows(x[2:3])[0], p[2])
    assert np.array_equal(m.forward(np.ascontiguousarray(x[1].T)), p[1])
    pbar = gwo.ensemble_mean([p[0]] * 4)
    assert np.array_equal(pbar, p[0])
    pf = [p[i].astype(np.float32) for i in range(4)]
    want = ((pf[0] + pf[1]) + pf[2]) + pf[3]
    assert np.array_equal(gwo.ensemble_mean_f32(pf), want / np.float32(4))
    assert np.max(np.abs(gwo.ensemble_mean([p[i] for i in range(4)]) - p[:4].mean(axis=0))) < 1e-15


# ---- fp16 rounding helper against numpy's IEEE binary16 ---------------------------------------------------
def test_round_half_matches_numpy_float16():
    v = np.concatenate([_rand(71, 0, 4000) * 3, _rand(71, 1, 500) * 1e-6, _rand(71, 2, 500) * 3e4,
                        [0.0, -0.0, 65504.0, 65519.9, 65520.0, -7e4, 2.0 ** -24, 2.0 ** -25, 1.5 * 2.0 ** -25,
                         2.0 ** -14, 1 + 2.0 ** -11, 1 + 3 * 2.0 ** -11, 5.96e-8, 6.1e-5]])
    with np.errstate(over="ignore"):
        want = v.astype(np.float32).astype(np.float16).astype(np.float64)
    got = gwo.round_half(v)
    assert np.array_equal(got, want)


def test_model_fp16_rounding_is_applied(tmpdir_s, small):
    a, t, m = small
    path = os.path.join(str(tmpdir_s), "r16.gwim")
    t16 = {k: v.astype(np.float16).astype(np.float32) for k, v in t.items()}
    gs.write_model(path, a, t16)
    path0 = os.path.join(str(tmpdir_s), "small.gwim")
    x = np.stack([_rand(81, 0, 30), _rand(81, 1, 30)])
    assert np.array_equal(gwo.Model(path, False).forward(x), gwo.Model(path0, True).forward(x))
    assert not np.array_equal(gwo.Model(path0, False).forward(x), gwo.Model(path0, True).forward(x))
