"""GPU parity of the whitening front end (gwi_whiten) against the oracle (-m gpu).  Bar: max-abs 1e-3 on unit-variance
output in fp32 (fp32 FFTs of up to 2^22 points against the oracle's fp64; reading A35), one fp16 ulp more for
the half output."""
import numpy as np
import pytest

from gwsynth import rng
from oracle import gwo_whiten as ow

pytestmark = pytest.mark.gpu


def _coloured(seed, n):
    w = rng.normal(seed, 11, 0, n)
    f = np.fft.rfftfreq(n, 1.0 / 4096.0)
    psd = (40.0 / np.maximum(f, 10.0)) ** 4 + 1.0          # the colour of reading A27
    return np.fft.irfft(np.fft.rfft(w) * np.sqrt(psd), n)


@pytest.mark.parametrize("n,nper", [(4096, 4096), (10000, 512), (1 << 16, 8192), (3 * 4096 * 50 + 2, 8192), (1 << 22, 8192)])
def test_whiten_matches_oracle(n, nper):
    import torch
    import paper_2201_11133_b200 as gwi
    x = (1e-19 * _coloured(n % 97, n)).astype(np.float32)      # raw-strain-like magnitudes
    want = ow.whiten(x.astype(np.float64), nper)
    xd = torch.from_numpy(x).cuda()
    got32 = gwi.whiten(xd, nper, half=False).cpu().numpy().astype(np.float64)
    assert np.max(np.abs(got32 - want)) <= 1e-3
    assert abs(got32.std() - 1.0) < 1e-4
    got16 = gwi.whiten(xd, nper, half=True).cpu().numpy().astype(np.float64)
    assert np.max(np.abs(got16 - want)) <= 1e-3 + np.max(np.abs(want)) * 2.0 ** -11
    assert np.array_equal(xd.cpu().numpy(), x)                  # the input is not modified


@pytest.mark.parametrize("n,nper,off", [(10002, 500, 0), (20000, 1004, 0), (1 << 16, 4096, 1), (30000, 500, 3)])
def test_whiten_scalar_and_unaligned_paths(n, nper, off):
    """Frame lengths that are no multiple of 8 (no 16-byte frame starts) and input pointers off a 16-byte boundary take
    the scalar loads of the framing / statistics kernels; same bar as above."""
    import torch
    import paper_2201_11133_b200 as gwi
    x = (1e-19 * _coloured(7 + off, n + off)).astype(np.float32)
    want = ow.whiten(x[off:].astype(np.float64), nper)
    xd = torch.from_numpy(x).cuda()[off:]
    got32 = gwi.whiten(xd, nper, half=False).cpu().numpy().astype(np.float64)
    assert np.max(np.abs(got32 - want)) <= 1e-3
    got16 = gwi.whiten(xd, nper, half=True).cpu().numpy().astype(np.float64)
    assert np.max(np.abs(got16 - want)) <= 1e-3 + np.max(np.abs(want)) * 2.0 ** -11


def test_whiten_argument_errors():
    import torch
    import paper_2201_11133_b200 as gwi
    x = torch.zeros(1001, device="cuda")
    with pytest.raises(gwi.GwiError):
        gwi.whiten(x, 100)            # odd n
    with pytest.raises(gwi.GwiError):
        gwi.whiten(x[:1000], 2000)    # nper > n
