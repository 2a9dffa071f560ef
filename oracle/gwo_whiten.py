"""Oracle of the whitening front end.  TEST INFRASTRUCTURE, NOT THE PRODUCT.

PAPER.md:43: "We used advanced LIGO data to compute power spectral density (PSDs) estimates ... We used these PSDs to
whiten ... advanced LIGO strain data ... we normalized the standard deviation ... to one."  The paper names no
parameters; reading A35 fixes them.  Plain numpy, FP64, step by step:

  1. Welch estimate of the segment's own PSD: frames of `nper` samples every nper/2 samples (the frames that fit),
     each multiplied by the symmetric Hann window, P[j] = mean over frames of |rfft(frame)[j]|^2   (no scaling constant:
     step 4 removes every constant factor)
  2. P interpolated linearly from the nper/2+1 frame frequencies to the n/2+1 frequencies of the whole segment
  3. Y = rfft(x) / sqrt(P_interp),  y = irfft(Y)
  4. out = y / std(y)            (population standard deviation)

Only tests/ may import this module.  It shares nothing with paper_2201_11133_b200/ or gwsynth/.
"""
import numpy as np


def welch_psd(x, nper):
    x = np.asarray(x, dtype=np.float64)
    step = nper // 2
    i = np.arange(nper, dtype=np.float64)
    w = 0.5 - 0.5 * np.cos(2.0 * np.pi * i / (nper - 1))
    acc = np.zeros(nper // 2 + 1)
    k = 0
    s0 = 0
    while s0 + nper <= len(x):
        acc += np.abs(np.fft.rfft(x[s0:s0 + nper] * w)) ** 2
        k += 1
        s0 += step
    return acc / k


def whiten(x, nper):
    """x: one segment (even length n >= nper, nper even) -> whitened, unit standard deviation, float64."""
    x = np.asarray(x, dtype=np.float64)
    n = len(x)
    assert n % 2 == 0 and nper % 2 == 0 and 4 <= nper <= n
    P = welch_psd(x, nper)
    pos = np.arange(n // 2 + 1, dtype=np.float64) * nper / n          # position on the frame-frequency grid
    j = np.minimum(np.floor(pos).astype(np.int64), nper // 2 - 1)
    frac = pos - j
    Pi = P[j] * (1.0 - frac) + P[j + 1] * frac
    y = np.fft.irfft(np.fft.rfft(x) / np.sqrt(np.maximum(Pi, 1e-300)), n)
    return y / np.sqrt(np.mean((y - np.mean(y)) ** 2))
