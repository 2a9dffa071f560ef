"""gwi_ensemble_triggers_static -- the entry point that allocates nothing -- against gwi_ensemble_triggers (-m gpu).

The scratch of the static variant is a file-scope device array inside libgwi.so that every call shares and that keeps
the previous call's contents, so the check is made on TWO calls in a row with different inputs (a long chunk with many
runs, then a shorter one with other runs: stale mask words, block flags or counts of the first call would show in the
second), each compared with the existing path on the same inputs: records, count and mean probability bit for bit
(both paths run the same kernels; the tolerance of tests/test_gpu_triggers.py tier T1 is exact equality).
The file name sorts last so that pytest -x collects it after every other test.
"""
import ctypes as C

import numpy as np
import pytest

from gwsynth import rng

pytestmark = pytest.mark.gpu


def _noisy(seed, N, M=4, corr=64):
    base = rng.uniform01(seed, 0, np.arange(N // corr + 1, dtype=np.uint64))
    lvl = np.repeat(np.where(base < 0.5, 0.3, 0.7), corr)[:N]
    return [(lvl + 0.25 * (rng.uniform01(seed, 1 + m, np.arange(N, dtype=np.uint64)) - 0.5)).astype(np.float32)
            for m in range(M)]


def _tuples(recs):
    return [(r.slide, r.start, r.end, r.peak_p, r.mean_p, r.model_mask) for r in recs]


def _static_call(gwi, torch, probs, theta, lmin, capacity, check_mem=False, **kw):
    """all buffers allocated by the caller beforehand; the library call itself allocates nothing (check_mem: the free device
    memory does not move across the call -- asserted where the same kernels have run just before, so that the lazy
    loading of a kernel's code cannot be what moves it)"""
    dev = probs[0].device
    N = probs[0].numel()
    trig = torch.zeros(capacity * C.sizeof(gwi.Trigger), dtype=torch.uint8, device=dev)
    cnt = torch.zeros(1, dtype=torch.int32, device=dev)
    pbar = torch.empty(N, dtype=torch.float32, device=dev)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    gwi.ensemble_triggers_static(probs, theta, lmin, trig, cnt, pbar=pbar, **kw)
    torch.cuda.synchronize()
    assert not check_mem or torch.cuda.mem_get_info()[0] == free0
    n = int(cnt.item())
    raw = trig.cpu().numpy().tobytes()
    recs = [gwi.Trigger.from_buffer_copy(raw, i * C.sizeof(gwi.Trigger)) for i in range(min(n, capacity))]
    return n, recs, pbar


def test_static_scratch_matches_workspace_path_on_two_calls_in_a_row():
    import torch
    import paper_2201_11133_b200 as gwi
    cases = [(1 << 20, 9, 64, 0.5, 3, 1000), (300007, 10, 16, 0.45, 1, 0), (1 << 20, 9, 64, 0.5, 3, 1000)]
    for N, seed, lmin, theta, slide, t0 in cases:
        probs = [torch.from_numpy(p).cuda() for p in _noisy(seed, N)]
        n0, r0, pb0 = gwi.ensemble_triggers(probs, theta, lmin, t0=t0, slide_id=slide, capacity=1 << 16, want_pbar=True)
        n1, r1, pb1 = _static_call(gwi, torch, probs, theta, lmin, 1 << 16, check_mem=True, t0=t0, slide_id=slide)
        assert n0 > 100 and n1 == n0
        assert _tuples(r1) == _tuples(r0)
        assert torch.equal(pb1, pb0)


def test_static_scratch_with_carry_across_chunks():
    """two consecutive chunks with a carried run, through the static scratch: same records as the whole stream"""
    import torch
    import paper_2201_11133_b200 as gwi
    N, cut = 200000, 123457
    ps = _noisy(11, N)
    ps = [np.where((np.arange(N) > cut - 500) & (np.arange(N) < cut + 700), np.float32(0.9), p) for p in ps]   # a run across the cut
    whole = [torch.from_numpy(p).cuda() for p in ps]
    n0, r0, _ = gwi.ensemble_triggers(whole, 0.5, 32, capacity=1 << 14)
    carry = torch.zeros(gwi.lib().gwi_carry_bytes(), dtype=torch.uint8, device="cuda")
    a = [w[:cut].contiguous() for w in whole]
    b = [w[cut:].contiguous() for w in whole]
    na, ra, _ = _static_call(gwi, torch, a, 0.5, 32, 1 << 14, last_chunk=False, carry=carry)
    nb, rb, _ = _static_call(gwi, torch, b, 0.5, 32, 1 << 14, t0=cut, last_chunk=True, carry=carry)
    assert na + nb == n0 and n0 > 10
    assert sorted(_tuples(ra + rb)) == sorted(_tuples(r0))
    assert any(r.start < cut < r.end for r in ra + rb)


def test_static_scratch_rejects_sizes_beyond_its_maximum():
    import torch
    import paper_2201_11133_b200 as gwi
    N = gwi.TRIGGERS_STATIC_MAX_N + 1
    probs = [torch.zeros(N, dtype=torch.float32, device="cuda")]
    trig = torch.zeros(16 * C.sizeof(gwi.Trigger), dtype=torch.uint8, device="cuda")
    cnt = torch.zeros(1, dtype=torch.int32, device="cuda")
    with pytest.raises(gwi.GwiError) as ei:
        gwi.ensemble_triggers_static(probs, 0.5, 8, trig, cnt)
    assert ei.value.status == 7 and "GWI_TRIGGERS_STATIC_MAX_N" in str(ei.value)
    # the largest size it takes: a plateau at the very end of the array
    probs = [torch.zeros(N - 1, dtype=torch.float32, device="cuda")]
    probs[0][-5000:] = 0.9
    gwi.ensemble_triggers_static(probs, 0.5, 8, trig, cnt)
    torch.cuda.synchronize()
    rec = gwi.Trigger.from_buffer_copy(trig.cpu().numpy().tobytes(), 0)
    assert int(cnt.item()) == 1 and (rec.start, rec.end) == (N - 1 - 5000, N - 1)
