"""Pin P18 (-m "not gpu"): the oracle of the whitening front end (reading A35) against what fixes it from
outside: scipy's Welch estimator (step 1), flatness of the output spectrum for noise of a known colour (steps 2-3: a
missing square root or a wrong interpolation fails it), unit standard deviation (step 4), invariance under scaling."""
import numpy as np
import scipy.signal

from gwsynth import rng
from oracle import gwo_whiten as ow


def _coloured(seed, n, fs=4096.0):
    w = rng.normal(seed, 7, 0, n)
    f = np.fft.rfftfreq(n, 1.0 / fs)
    psd = 10.0 ** (2.0 * f / f[-1])                   # smooth, a factor 100 across the band
    return np.fft.irfft(np.fft.rfft(w) * np.sqrt(psd), n), psd


def test_p18_welch_equals_scipy():
    x = rng.normal(3, 0, 0, 1 << 15)
    nper = 1024
    P = ow.welch_psd(x, nper)
    win = 0.5 - 0.5 * np.cos(2 * np.pi * np.arange(nper) / (nper - 1))
    _, S = scipy.signal.welch(x, fs=1.0, window=win, nperseg=nper, noverlap=nper // 2, detrend=False,
                              return_onesided=False, scaling="spectrum", average="mean")
    S = S[:nper // 2 + 1] * (win.sum() ** 2)           # scipy divides the periodogram by (sum w)^2
    assert np.max(np.abs(P / S - 1.0)) < 1e-10


def test_p18_output_is_white_and_unit_variance():
    n, nper = 1 << 18, 8192
    x, psd = _coloured(5, n)
    assert psd.max() / psd.min() > 99.0                # the input is far from white
    y = ow.whiten(x, nper)
    assert abs(np.std(y) - 1.0) < 1e-12
    Py = ow.welch_psd(y, nper)[8:-8]                    # away from DC / Nyquist window leakage
    q = np.array([np.mean(b) for b in np.array_split(Py, 16)])
    assert q.max() / q.min() < 1.08                    # flat within the statistical scatter of 16 band averages
    # a version that divides by the PSD instead of its square root is not flat
    Yw = np.fft.irfft(np.fft.rfft(x) / np.maximum(np.interp(np.arange(n // 2 + 1) * nper / n, np.arange(nper // 2 + 1),
                                                            ow.welch_psd(x, nper)), 1e-300), n)
    qin = np.array([np.mean(b) for b in np.array_split(ow.welch_psd(x, nper)[8:-8], 16)])
    assert qin.max() / qin.min() > 10.0                # the same band statistic on the unwhitened input is far from flat
    qw = np.array([np.mean(b) for b in np.array_split(ow.welch_psd(Yw, nper)[8:-8], 16)])
    assert qw.max() / qw.min() > 10.0


def test_p18_scale_invariance_and_interpolation_identity():
    x, _ = _coloured(9, 1 << 14)
    a = ow.whiten(x, 2048)
    b = ow.whiten(37.5 * x, 2048)
    assert np.max(np.abs(a - b)) < 1e-9
    # nper == n: one frame, no interpolation; the result divides the spectrum by |rfft(x w)|
    n = 4096
    xs = x[:n]
    w = 0.5 - 0.5 * np.cos(2 * np.pi * np.arange(n) / (n - 1))
    y = np.fft.irfft(np.fft.rfft(xs) / np.abs(np.fft.rfft(xs * w)), n)
    y = y / np.std(y)
    assert np.max(np.abs(ow.whiten(xs, n) - y)) < 1e-9
