"""Shared helpers of the GPU parity tests (no arithmetic of the method here)."""
import os

import numpy as np

import gwsynth as gs
from oracle import gwo


def model_pair(tmpdir, name, arch, tensors, precision):
    """Write the GWIM file once; load it in the oracle (own parser) and in the CUDA library (own parser)."""
    import paper_2201_11133_b200 as gwi
    path = os.path.join(str(tmpdir), name + ".gwim")
    gs.write_model(path, arch, tensors)
    om = gwo.Model(path, round_fp16=(precision == gwi.FP16))
    gm = gwi.load_model(path, precision, 0)
    return om, gm


def rand_windows(seed, B, T, C=2, dtype=np.float32):
    x = np.empty((B, T, C), dtype=dtype)
    for c in range(C):
        x[:, :, c] = gs.white_noise(seed, c, 0, B * T).reshape(B, T).astype(dtype)
    return x


def trig_tuples(recs):
    return [(r.slide, r.start, r.end) for r in recs]
