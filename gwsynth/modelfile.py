"""GWIM v1 model file: writer, python reader (for tests that perturb weights) and seeded weight generators.

File layout (little-endian), DESIGN.md section "Model file":
    bytes 0..3   magic "GWIM"
    int32        version (=1), n_branch, c_in, R, S, k, L, Hh, dtype (=0: fp32)
    int32[L]     dilations d_1..d_L
    fp32 tensors, C order, in the order given by tensor_specs():
      per branch b:  W_in[R][c_in], b_in[R],
                     per block i: Wf[R][R][k], bf[R], Wg[R][R][k], bg[R], Wr[R][R], br[R], Ws[S][R], bs[S]
      head:          W1[Hh][n_branch*S], b1[Hh], W2[Hh], b2[1]
Tap index j = k-1 multiplies the CURRENT sample, tap j the sample (k-1-j)*d in the past (reading A5).

The oracle (oracle/gwo_oracle.c) and the CUDA library (paper_2201_11133_b200/csrc/model.cpp) each parse
this format with their own code; nothing here is imported by either.
"""
from dataclasses import dataclass, field
import struct
import numpy as np

from . import rng

MAGIC = b"GWIM"
VERSION = 1


@dataclass(frozen=True)
class Arch:
    n_branch: int = 2
    c_in: int = 1
    R: int = 16
    S: int = 32
    k: int = 2
    dil: tuple = (1, 2, 4, 8)
    Hh: int = 32

    @property
    def L(self):
        return len(self.dil)

    @property
    def receptive_field(self):
        return 1 + (self.k - 1) * sum(self.dil)

    def flops_per_timestep(self):
        """Multiply-add = 2 flops; the count DESIGN.md uses for roofline figures."""
        R, S, k = self.R, self.S, self.k
        per_branch = 2 * self.c_in * R + self.L * (4 * k * R * R + 2 * R * R + 2 * R * S)
        head = 2 * self.n_branch * S * self.Hh + 2 * self.Hh
        return self.n_branch * per_branch + head


# BASELINE.json configs[0] (and 2-4): 4 blocks, k=2, d=1,2,4,8, 16 residual / 32 skip channels, per branch.
CFG1_ARCH = Arch(n_branch=2, c_in=1, R=16, S=32, k=2, dil=(1, 2, 4, 8), Hh=32)
# BASELINE.json configs[1] default (PAPER.md gives no layer spec): 2 stacks x 10 blocks, d=1..512, 64/128.
PAPER_ARCH = Arch(n_branch=2, c_in=1, R=64, S=128, k=2, dil=tuple([1 << i for i in range(10)] * 2), Hh=128)


def tensor_specs(a: Arch):
    """[(name, shape, fan_in, fan_out)] in file order. fan = channels * taps (Xavier convention)."""
    out = []
    for b in range(a.n_branch):
        p = f"b{b}."
        out.append((p + "W_in", (a.R, a.c_in), a.c_in, a.R))
        out.append((p + "b_in", (a.R,), 0, 0))
        for i in range(a.L):
            q = f"{p}l{i}."
            out.append((q + "Wf", (a.R, a.R, a.k), a.R * a.k, a.R * a.k))
            out.append((q + "bf", (a.R,), 0, 0))
            out.append((q + "Wg", (a.R, a.R, a.k), a.R * a.k, a.R * a.k))
            out.append((q + "bg", (a.R,), 0, 0))
            out.append((q + "Wr", (a.R, a.R), a.R, a.R))
            out.append((q + "br", (a.R,), 0, 0))
            out.append((q + "Ws", (a.S, a.R), a.R, a.S))
            out.append((q + "bs", (a.S,), 0, 0))
    out.append(("W1", (a.Hh, a.n_branch * a.S), a.n_branch * a.S, a.Hh))
    out.append(("b1", (a.Hh,), 0, 0))
    out.append(("W2", (a.Hh,), a.Hh, 1))
    out.append(("b2", (1,), 0, 0))
    return out


def zero_tensors(a: Arch):
    return {n: np.zeros(s, dtype=np.float32) for n, s, _, _ in tensor_specs(a)}


def xavier_tensors(a: Arch, seed: int, bias: str = "zero"):
    """Xavier-uniform weights U(-a, a), a = sqrt(6/(fan_in+fan_out)); draws in file order, tensor number
    = generator stream, flat C index = generator counter. bias: "zero" (headline configs, Keras default)
    or "random" (U(-0.5, 0.5); the dedicated parity test, so a kernel that drops a bias cannot pass)."""
    t = {}
    for sid, (name, shape, fi, fo) in enumerate(tensor_specs(a)):
        n = int(np.prod(shape))
        u = rng.uniform01(seed, sid, np.arange(n, dtype=np.uint64))
        if fi == 0:  # a bias
            v = (u - 0.5) if bias == "random" else np.zeros(n)
        else:
            lim = np.sqrt(6.0 / (fi + fo))
            v = (2.0 * u - 1.0) * lim
        t[name] = v.astype(np.float32).reshape(shape)
    return t


def write_model(path, a: Arch, tensors):
    with open(path, "wb") as f:
        f.write(MAGIC)
        f.write(struct.pack("<9i", VERSION, a.n_branch, a.c_in, a.R, a.S, a.k, a.L, a.Hh, 0))
        f.write(struct.pack(f"<{a.L}i", *a.dil))
        for name, shape, _, _ in tensor_specs(a):
            arr = np.ascontiguousarray(np.asarray(tensors[name], dtype=np.float32))
            if arr.shape != tuple(shape):
                raise ValueError(f"{name}: shape {arr.shape} != {shape}")
            f.write(arr.astype("<f4").tobytes())


def read_model(path):
    with open(path, "rb") as f:
        raw = f.read()
    if raw[:4] != MAGIC:
        raise ValueError("bad magic")
    ver, nb, cin, R, S, k, L, Hh, dt = struct.unpack_from("<9i", raw, 4)
    if ver != VERSION or dt != 0:
        raise ValueError("unsupported version/dtype")
    dil = struct.unpack_from(f"<{L}i", raw, 40)
    a = Arch(nb, cin, R, S, k, tuple(dil), Hh)
    off = 40 + 4 * L
    t = {}
    for name, shape, _, _ in tensor_specs(a):
        n = int(np.prod(shape))
        t[name] = np.frombuffer(raw, dtype="<f4", count=n, offset=off).reshape(shape).copy()
        off += 4 * n
    if off != len(raw):
        raise ValueError("trailing bytes")
    return a, t


def make_model_file(path, a: Arch, seed: int, bias: str = "zero"):
    t = xavier_tensors(a, seed, bias)
    write_model(path, a, t)
    return t


def p16_tensors(a: Arch, block=0, r=0, q=(0, 1), hid=(0, 1), gamma=8.0, past=False):
    """Pin P16's sign pass-through model placed inside any two-branch
    architecture: every weight and bias is zero except
        lift      W_in[r] = 1                                   -> h[r][t] = x[t]
        `block`   Wf[r][r] = (0,1) (or (1,0) with past=True)    -> f[r][t] = x[t] (or x[t - d_block]); g = 0
                  Ws[q0][r] = +2, Ws[q1][r] = -2                -> u[q0] = ReLU(T), u[q1] = ReLU(-T), T = tanh(f)
        head      W1[hid0] = (+1,-1 | +1,-1) on (q0,q1) of both branches, W1[hid1] = its negation, W2 = (gamma,-gamma)
    so that y[t] = gamma * (T_H1[t] + T_L1[t]).  All other blocks have f = g = 0, z = 0 and contribute nothing; Wr = 0
    keeps h = x through the stack.  Only weight placement -- none of the method's arithmetic happens here."""
    assert a.n_branch == 2 and a.c_in == 1 and a.k == 2
    t = zero_tensors(a)
    for b in range(2):
        t[f"b{b}.W_in"][r, 0] = 1.0
        t[f"b{b}.l{block}.Wf"][r, r] = [1.0, 0.0] if past else [0.0, 1.0]
        t[f"b{b}.l{block}.Ws"][q[0], r] = 2.0
        t[f"b{b}.l{block}.Ws"][q[1], r] = -2.0
        for s, qq in zip((1.0, -1.0), q):
            t["W1"][hid[0], b * a.S + qq] = s
            t["W1"][hid[1], b * a.S + qq] = -s
    t["W2"][hid[0]] = gamma
    t["W2"][hid[1]] = -gamma
    return t
