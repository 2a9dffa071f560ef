"""GPU parity of gwi_infer against the FP64 oracle, element by element, through the C-ABI (-m gpu).

Tolerances (BASELINE.json north_star): max-abs 1e-5 on probabilities in FP32 mode, 2e-3 in FP16 mode.
"""
import numpy as np
import pytest

import gwsynth as gs
from tests.helpers import model_pair, rand_windows

pytestmark = pytest.mark.gpu

TOL32, TOL16 = 1e-5, 2e-3


def _run(gm, x):
    import torch
    xt = torch.from_numpy(x).cuda()
    p = gm.infer(xt)
    torch.cuda.synchronize()
    return p.cpu().numpy().astype(np.float64)


def test_config1_fp32(tmpdir_s):
    """BASELINE.json configs[0]: tiny model, seed-0 Xavier weights, 8 x 4096 x 2 N(0,1) seed 1, FP32."""
    import paper_2201_11133_b200 as gwi
    a = gs.CFG1_ARCH
    om, gm = model_pair(tmpdir_s, "cfg1", a, gs.xavier_tensors(a, 0), gwi.FP32)
    x = gs.cfg1_windows(seed=1, B=8, T=4096)
    want = om.infer_windows(x)
    got = _run(gm, x)
    assert got.shape == (8, 4096)
    assert np.max(np.abs(got - want)) <= TOL32
    assert 0.3 < want.mean() < 0.7 and want.std() > 1e-3        # the comparison is not vacuous


@pytest.mark.parametrize("T", [1, 15, 16, 17, 127, 128, 129, 5000])
@pytest.mark.parametrize("B", [1, 3])
def test_shape_matrix_fp32_random_bias(tmpdir_s, T, B):
    import paper_2201_11133_b200 as gwi
    a = gs.CFG1_ARCH
    om, gm = model_pair(tmpdir_s, "sm_rb", a, gs.xavier_tensors(a, 5, bias="random"), gwi.FP32)
    x = rand_windows(100 + T, B, T)
    assert np.max(np.abs(_run(gm, x) - om.infer_windows(x))) <= TOL32


@pytest.mark.parametrize("arch", [
    gs.Arch(n_branch=1, c_in=2, R=16, S=32, k=2, dil=(1, 2, 4, 8), Hh=32),       # A1 variant: one 2-channel stack
    gs.Arch(n_branch=2, c_in=1, R=24, S=40, k=2, dil=(1, 2, 4), Hh=24),          # odd widths
    gs.Arch(n_branch=2, c_in=1, R=8, S=8, k=3, dil=(1, 3, 9), Hh=8),             # k = 3
    gs.Arch(n_branch=2, c_in=1, R=16, S=32, k=2, dil=(1, 300, 2), Hh=32),        # dilation > T (P7-v)
    gs.Arch(n_branch=2, c_in=1, R=1, S=1, k=2, dil=(1,), Hh=1),                  # degenerate widths
], ids=["single-stack", "odd-width", "k3", "dil-gt-T", "width1"])
def test_architecture_variants_fp32(tmpdir_s, arch):
    import paper_2201_11133_b200 as gwi
    om, gm = model_pair(tmpdir_s, "var", arch, gs.xavier_tensors(arch, 9, bias="random"), gwi.FP32)
    x = rand_windows(7, 2, 200)
    assert np.max(np.abs(_run(gm, x) - om.infer_windows(x))) <= TOL32


def test_paper_scale_fp32_small_batch(tmpdir_s):
    import paper_2201_11133_b200 as gwi
    a = gs.PAPER_ARCH
    om, gm = model_pair(tmpdir_s, "paper32", a, gs.xavier_tensors(a, 0, bias="random"), gwi.FP32)
    x = rand_windows(3, 2, 4096)
    want = om.infer_windows(x)
    got = _run(gm, x)
    assert np.max(np.abs(got - want)) <= TOL32
    assert want.std() > 1e-2


def test_config1_arch_fp16_mode(tmpdir_s):
    """FP16 mode on an architecture the tensor-core kernel does not cover: generic kernel on fp16-rounded operands."""
    import paper_2201_11133_b200 as gwi
    a = gs.CFG1_ARCH
    om, gm = model_pair(tmpdir_s, "cfg1h", a, gs.xavier_tensors(a, 0, bias="random"), gwi.FP16)
    x = rand_windows(1, 4, 1000, dtype=np.float16)
    want = om.infer_windows(x.astype(np.float64))
    assert np.max(np.abs(_run(gm, x) - want)) <= TOL16


def test_p5_worked_example_on_gpu(tmpdir_s):
    """The hand-computed fixture checked directly against the CUDA path too (not only via the oracle)."""
    import os
    import paper_2201_11133_b200 as gwi
    a = gs.Arch(n_branch=2, c_in=1, R=1, S=1, k=2, dil=(1,), Hh=1)
    t = gs.zero_tensors(a)
    t["b0.W_in"][:] = 1.0
    t["b1.W_in"][:] = 1.0
    t["b0.l0.Wf"][0, 0] = [0.5, 1.0]
    t["b0.l0.Ws"][0, 0] = 2.0
    t["b1.l0.Wf"][0, 0] = [-1.0, 1.0]
    t["b1.l0.Wg"][0, 0] = [0.0, 1.0]
    t["b1.l0.Ws"][0, 0] = 1.0
    t["b1.l0.bs"][0] = 0.1
    t["W1"][0] = [1.0, 2.0]
    t["b1"][0] = -0.5
    t["W2"][0] = 3.0
    t["b2"][0] = -1.0
    _, gm = model_pair(tmpdir_s, "p5gpu", a, t, gwi.FP32)
    x = np.array([[[1, 0], [-1, 1], [2, 1], [0, -2]]], dtype=np.float32)
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "p5_worked_example_A.txt"))
            if l.strip() and not l.startswith("#")]
    want = np.array([float(r[5]) for r in rows])
    assert np.max(np.abs(_run(gm, x)[0] - want)) < 2e-6


def test_error_paths(tmpdir_s):
    import torch
    import paper_2201_11133_b200 as gwi
    a = gs.CFG1_ARCH
    _, gm = model_pair(tmpdir_s, "err", a, gs.xavier_tensors(a, 0), gwi.FP32)
    with pytest.raises(gwi.GwiError) as e:
        gm.infer(torch.zeros((1, 8, 2), dtype=torch.float32))            # host tensor: no CPU fallback
    assert e.value.status == 1
    with pytest.raises(gwi.GwiError):
        gm.infer(torch.zeros((1, 8, 3), dtype=torch.float32, device="cuda"))
    p = gm.infer(torch.zeros((0, 8, 2), dtype=torch.float32, device="cuda"))   # B = 0 is a no-op
    assert p.shape == (0, 8)
    bad = tmpdir_s / "bad.gwim"
    bad.write_bytes(b"NOPE" + b"\0" * 100)
    with pytest.raises(gwi.GwiError) as e:
        gwi.load_model(str(bad))
    assert e.value.status == 3
