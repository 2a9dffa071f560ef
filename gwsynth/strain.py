"""Seeded synthetic strain (inputs only; DESIGN.md section "Inputs" gives the recipe and the stand-in statement).

All Gaussian samples are drawn in fp64 from the counter generator (rng.normal) with
    generator stream = detector index (0: H1, 1: L1),  counter = sample index,
then rounded ONCE to the stored dtype. Oracle and CUDA path both read the stored values.
"""
import numpy as np

from . import rng

FS = 4096  # Hz


def white_noise(seed, det, start, count):
    return rng.normal(seed, det, start, count)


def cfg1_windows(seed=1, B=8, T=4096):
    """BASELINE.json configs[0]: B windows x T samples x 2 detectors of i.i.d. N(0,1), fp32, layout (B,T,2)."""
    x = np.empty((B, T, 2), dtype=np.float32)
    for c in range(2):
        x[:, :, c] = white_noise(seed, c, 0, B * T).reshape(B, T).astype(np.float32)
    return x


def chirp_waveform(tau_s, f0=30.0, f1=300.0, fs=FS):
    """Reading A26: hann(t/tau) * sin(2 pi (f0 t + (f1-f0) t^2 / (2 tau))), unit amplitude, len = round(tau*fs)."""
    n = int(round(tau_s * fs))
    t = np.arange(n) / fs
    hann = 0.5 - 0.5 * np.cos(2.0 * np.pi * np.arange(n) / max(n - 1, 1))
    return hann * np.sin(2.0 * np.pi * (f0 * t + (f1 - f0) * t * t / (2.0 * tau_s)))


def _inject(x2, end_idx, tau_s, snr):
    """Add the same chirp to both detector rows of x2[2][n] so that sqrt(sum_det sum_t s^2) = snr."""
    w = chirp_waveform(tau_s)
    amp = snr / np.sqrt(2.0 * np.sum(w * w))
    s0 = end_idx - len(w)
    for c in range(2):
        x2[c, s0:end_idx] += amp * w


def cfg2_windows(seed=1, B=1024, T=4096, inject_frac=0.10, dtype=np.float16):
    """BASELINE.json configs[1]: (B,T,2) N(0,1) noise; a seeded 10 % of windows carry an A26 chirp
    (tau ~ U(0.2,1) s, network SNR ~ U(8,20), end placed at a seeded time fully inside the window),
    added in fp64 before the single rounding to `dtype`. Returns (x, injected_window_indices)."""
    xs = np.empty((2, B * T), dtype=np.float64)
    for c in range(2):
        xs[c] = white_noise(seed, c, 0, B * T)
    n_inj = int(round(inject_frac * B))
    order = np.argsort(rng.u64(seed, 100, np.arange(B, dtype=np.uint64)), kind="stable")
    inj = np.sort(order[:n_inj])
    for j, b in enumerate(inj):
        u = rng.uniform01(seed, 101, np.arange(3 * j, 3 * j + 3, dtype=np.uint64))
        tau = 0.2 + 0.8 * u[0]
        snr = 8.0 + 12.0 * u[1]
        n = int(round(tau * FS))
        end = n + int(u[2] * (T - n + 1))
        end = min(max(end, n), T)
        _inject(xs[:, b * T:(b + 1) * T], end, tau, snr)
    x = np.empty((B, T, 2), dtype=dtype)
    for c in range(2):
        x[:, :, c] = xs[c].reshape(B, T).astype(dtype)
    return x, inj


def stream_noise(seed, start, count, dtype=np.float16, injections=()):
    """Planar [2][count] stream of N(0,1) for global sample indices start..start+count-1 (configs 3 and 5).
    injections: iterable of (end_global_index, tau_s, snr) chirps; the part inside this range is added."""
    xs = np.empty((2, count), dtype=np.float64)
    for c in range(2):
        xs[c] = white_noise(seed, c, start, count)
    for end_g, tau, snr in injections:
        w = chirp_waveform(tau)
        amp = snr / np.sqrt(2.0 * np.sum(w * w))
        s0 = end_g - len(w)
        lo, hi = max(s0, start), min(end_g, start + count)
        if lo < hi:
            for c in range(2):
                xs[c, lo - start:hi - start] += amp * w[lo - s0:hi - s0]
    return xs.astype(dtype)


def coloured_whitened_noise(seed, det, n, seg_len=4096 * FS, dtype=np.float16):
    """Reading A27 (config 4; harness only, never timed). Per segment of `seg_len` samples (4096 s, the paper's
    segment length): synthesise Gaussian noise with one-sided PSD S(f) = (40/max(f,10))^4 + 1 in
    the frequency domain, whiten by a Welch estimate (2 s Hann, 50 % overlap, mean) of that segment, scale
    to unit standard deviation."""
    out = np.empty(n, dtype=np.float64)
    pos = 0
    seg = 0
    while pos < n:
        m = min(seg_len, n - pos)
        m_even = m + (m & 1)
        w = rng.normal(seed, 1000 + det, seg * (seg_len + 2), m_even)
        f = np.fft.rfftfreq(m_even, 1.0 / FS)
        psd = (40.0 / np.maximum(f, 10.0)) ** 4 + 1.0
        col = np.fft.irfft(np.fft.rfft(w) * np.sqrt(psd), m_even)
        nper = min(2 * FS, m_even)
        step = nper // 2
        win = np.hanning(nper)
        acc = np.zeros(nper // 2 + 1)
        cnt = 0
        for s0 in range(0, m_even - nper + 1, step):
            acc += np.abs(np.fft.rfft(col[s0:s0 + nper] * win)) ** 2
            cnt += 1
        welch = acc / max(cnt, 1)
        fw = np.fft.rfftfreq(nper, 1.0 / FS)
        est = np.interp(f, fw, welch)
        wh = np.fft.irfft(np.fft.rfft(col) / np.sqrt(np.maximum(est, 1e-300)), m_even)[:m]
        out[pos:pos + m] = wh / np.std(wh)
        pos += m
        seg += 1
    return out.astype(dtype)


def plateau_square_wave(n, plateaus, low, dtype=np.float32):
    """Pin P16 input: +1 on each [s, e) in `plateaus`, `low` elsewhere (H1: low=-2, L1: low=-3)."""
    x = np.full(n, float(low), dtype=np.float64)
    for s, e in plateaus:
        x[max(s, 0):min(e, n)] = 1.0
    return x.astype(dtype)


CFG5_CHUNK = 3600 * FS  # BASELINE.json configs[4]: one-hour chunks


def cfg5_injections(seed=5, n_chunks=744, n_inj=20, chunk=CFG5_CHUNK):
    """The 20 seeded A26 chirps of configs[4]: [(end_global_index, tau_s, snr)] sorted by time; tau ~ U(0.2,1) s,
    network SNR ~ U(8,20), the chirp's end uniform over the stream (whole chirp inside it)."""
    total = n_chunks * chunk
    out = []
    for j in range(n_inj):
        u = rng.uniform01(seed, 200, np.arange(3 * j, 3 * j + 3, dtype=np.uint64))
        tau, snr = 0.2 + 0.8 * u[0], 8.0 + 12.0 * u[1]
        n = int(round(tau * FS))
        out.append((n + int(u[2] * (total - n)), float(tau), float(snr)))
    return sorted(out)


def cfg5_chunk(c, seed=5, injections=(), n=CFG5_CHUNK, chunk=CFG5_CHUNK, dtype=np.float16):
    """configs[4] chunk c: planar [2][n] N(0,1), detector d drawn from the generator keyed (seed, stream = 16 + 2c + d,
    counter = sample index inside the chunk) -- "seed (5, d, c)" of SURVEY.md 8(d) -- plus the parts of `injections`
    (global indices) that fall inside [c * chunk, c * chunk + n); rounded once to `dtype`."""
    xs = np.empty((2, n), dtype=np.float64)
    for d in range(2):
        xs[d] = rng.normal(seed, 16 + 2 * c + d, 0, n)
    start = c * chunk
    for end_g, tau, snr in injections:
        w = chirp_waveform(tau)
        amp = snr / np.sqrt(2.0 * np.sum(w * w))
        s0 = end_g - len(w)
        lo, hi = max(s0, start), min(end_g, start + n)
        if lo < hi:
            for d in range(2):
                xs[d, lo - start:hi - start] += amp * w[lo - s0:hi - s0]
    return xs.astype(dtype)
