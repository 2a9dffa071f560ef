"""ctypes loader for the oracle (oracle/gwo_oracle.c).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this.
It contains no arithmetic of its own: every number comes out of gwo_oracle.c.  Argument marshalling only.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gwo_oracle.c")
_LIB = os.path.join(_HERE, "libgwo_oracle.so")

_dp = C.POINTER(C.c_double)
_fp = C.POINTER(C.c_float)


class Trigger(C.Structure):
    _fields_ = [("slide", C.c_int32), ("model_mask", C.c_int32), ("start", C.c_int64), ("end", C.c_int64),
                ("peak_p", C.c_double), ("mean_p", C.c_double)]


class Peak(C.Structure):
    _fields_ = [("index", C.c_int64), ("height", C.c_double), ("prominence", C.c_double), ("width", C.c_double),
                ("left_ip", C.c_double), ("right_ip", C.c_double)]


class Event(C.Structure):
    _fields_ = [("t_first", C.c_int64), ("t_last", C.c_int64), ("n_triggers", C.c_int32), ("slide", C.c_int32)]


def build(force=False):
    """gcc -O2 -fopenmp -ffp-contract=off: no FMA contraction, so the sums are the ones the source spells."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC", _SRC,
                               "-o", _LIB, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.gwo_round_half.restype = C.c_double
        L.gwo_round_half.argtypes = [C.c_double]
        L.gwo_load_model.restype = C.c_int
        L.gwo_load_model.argtypes = [C.c_char_p, C.c_int, C.POINTER(C.c_void_p)]
        L.gwo_free_model.argtypes = [C.c_void_p]
        L.gwo_model_info.argtypes = [C.c_void_p] + [C.POINTER(C.c_int32)] * 8
        L.gwo_conv1d_causal.argtypes = [_dp, C.c_int, C.c_int, C.c_int, C.c_int, _dp, _dp, C.c_long, _dp]
        L.gwo_branch.argtypes = [C.c_void_p, C.c_int, _dp, C.c_long, _dp, _dp]
        L.gwo_forward.argtypes = [C.c_void_p, _dp, C.c_long, _dp, _dp]
        L.gwo_infer_windows.argtypes = [C.c_void_p, _dp, C.c_long, C.c_long, _dp]
        L.gwo_stream.argtypes = [C.c_void_p, _dp, C.c_long, C.c_long, _dp, _dp]
        L.gwo_head_slide.argtypes = [C.c_void_p, _dp, C.c_long, C.c_long, _dp]
        L.gwo_ensemble_mean.argtypes = [C.POINTER(_dp), C.c_int, C.c_long, _dp]
        L.gwo_ensemble_mean_f32.argtypes = [C.POINTER(_fp), C.c_int, C.c_long, _fp]
        L.gwo_triggers.restype = C.c_long
        L.gwo_triggers.argtypes = [_dp, C.c_long, C.c_double, C.c_long, C.c_int, C.c_long, C.POINTER(_dp), C.c_int,
                                   C.POINTER(Trigger), C.c_long]
        L.gwo_coincidence.restype = C.c_long
        L.gwo_coincidence.argtypes = [C.POINTER(C.POINTER(C.c_long)), C.POINTER(C.c_int), C.c_int, C.c_long, C.c_int,
                                      C.POINTER(Event), C.c_long]
        L.gwo_find_peaks.restype = C.c_long
        L.gwo_find_peaks.argtypes = [_dp, C.c_long, C.c_double, C.c_double, C.POINTER(Peak), C.c_long]
        L.gwo_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(_dp)


def round_half(x):
    """Element-wise float -> binary16 (RNE) -> double, by the oracle's own routine."""
    L = lib()
    x = np.asarray(x, dtype=np.float64)
    return np.array([L.gwo_round_half(float(v)) for v in x.ravel()]).reshape(x.shape)


class Model:
    """Handle on a gwo_model loaded from a GWIM file. round_fp16=True rounds every weight to binary16 (RNE)."""

    def __init__(self, path, round_fp16=False):
        self._h = C.c_void_p()
        rc = lib().gwo_load_model(os.fsencode(path), int(round_fp16), C.byref(self._h))
        if rc != 0:
            raise IOError(f"gwo_load_model({path}) -> {rc}")
        v = [C.c_int32() for _ in range(8)]
        lib().gwo_model_info(self._h, *[C.byref(x) for x in v])
        (self.n_branch, self.c_in, self.R, self.S, self.k, self.L, self.Hh, self.receptive_field) = [x.value for x in v]

    def close(self):
        if self._h:
            lib().gwo_free_model(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def branch(self, b, x, dump_h=False):
        """x: [c_in][T] -> u [S][T] (and h_dump [L+1][R][T] if asked)."""
        x, xp = _d(x)
        T = x.shape[-1]
        u = np.empty((self.S, T))
        h = np.empty((self.L + 1, self.R, T)) if dump_h else None
        lib().gwo_branch(self._h, b, xp, T, u.ctypes.data_as(_dp), h.ctypes.data_as(_dp) if dump_h else None)
        return (u, h) if dump_h else u

    def forward(self, x, want_u=False):
        """x: [n_branch*c_in][T] planar -> p [T] (and u [n_branch][S][T])."""
        x, xp = _d(x)
        T = x.shape[-1]
        p = np.empty(T)
        u = np.empty((self.n_branch, self.S, T)) if want_u else None
        lib().gwo_forward(self._h, xp, T, p.ctypes.data_as(_dp), u.ctypes.data_as(_dp) if want_u else None)
        return (p, u) if want_u else p

    def infer_windows(self, x):
        """x: [B][T][C] channels-last -> p [B][T]."""
        x, xp = _d(x)
        B, T, Cc = x.shape
        assert Cc == self.n_branch * self.c_in
        p = np.empty((B, T))
        lib().gwo_infer_windows(self._h, xp, B, T, p.ctypes.data_as(_dp))
        return p

    def stream(self, x, seg=0, want_u=False):
        """x: [C][N] planar -> p_stream [N]; seg = segment length of the halo-extended evaluation (0: whole)."""
        x, xp = _d(x)
        N = x.shape[-1]
        p = np.empty(N)
        u = np.empty((self.n_branch, self.S, N)) if want_u else None
        lib().gwo_stream(self._h, xp, N, seg, p.ctypes.data_as(_dp), u.ctypes.data_as(_dp) if want_u else None)
        return (p, u) if want_u else p

    def head_slide(self, u, lag):
        u, up = _d(u)
        N = u.shape[-1]
        p = np.empty(N)
        lib().gwo_head_slide(self._h, up, N, int(lag), p.ctypes.data_as(_dp))
        return p


def conv1d_causal(x, W, b, d):
    """x [Cin][T], W [Cout][Cin][k], b [Cout] or None -> y [Cout][T]."""
    x, xp = _d(x)
    W, Wp = _d(W)
    Cout, Cin, k = W.shape
    T = x.shape[-1]
    y = np.empty((Cout, T))
    if b is not None:
        b, bp = _d(b)
    else:
        bp = None
    lib().gwo_conv1d_causal(xp, Cin, Cout, k, int(d), Wp, bp, T, y.ctypes.data_as(_dp))
    return y


def ensemble_mean(ps):
    arrs = [np.ascontiguousarray(p, dtype=np.float64) for p in ps]
    N = arrs[0].shape[0]
    ptrs = (_dp * len(arrs))(*[a.ctypes.data_as(_dp) for a in arrs])
    out = np.empty(N)
    lib().gwo_ensemble_mean(ptrs, len(arrs), N, out.ctypes.data_as(_dp))
    return out


def ensemble_mean_f32(ps):
    arrs = [np.ascontiguousarray(p, dtype=np.float32) for p in ps]
    N = arrs[0].shape[0]
    ptrs = (_fp * len(arrs))(*[a.ctypes.data_as(_fp) for a in arrs])
    out = np.empty(N, dtype=np.float32)
    lib().gwo_ensemble_mean_f32(ptrs, len(arrs), N, out.ctypes.data_as(_fp))
    return out


def triggers(pbar, theta, Lmin, slide=0, t0=0, pm=None, cap=1 << 16):
    """-> (total_count, [(slide, start, end, peak_p, mean_p, model_mask)])."""
    pbar, pp = _d(pbar)
    N = pbar.shape[0]
    out = (Trigger * cap)()
    if pm is not None:
        arrs = [np.ascontiguousarray(p, dtype=np.float64) for p in pm]
        ptrs = (_dp * len(arrs))(*[a.ctypes.data_as(_dp) for a in arrs])
        M = len(arrs)
    else:
        ptrs, M = None, 0
    n = lib().gwo_triggers(pp, N, float(theta), int(Lmin), int(slide), int(t0), ptrs, M, out, cap)
    recs = [(o.slide, o.start, o.end, o.peak_p, o.mean_p, o.model_mask) for o in out[:min(n, cap)]]
    return n, recs


def num_threads():
    return lib().gwo_num_threads()


def coincidence(ends, window, slide=0, cap=1 << 14):
    """ends: list (one per model) of lists of trigger end times -> [(t_first, t_last, n_triggers)] (reading A34)."""
    M = len(ends)
    arrs = [(C.c_long * max(len(e), 1))(*[int(v) for v in e]) for e in ends]
    ptrs = (C.POINTER(C.c_long) * M)(*[C.cast(a, C.POINTER(C.c_long)) for a in arrs])
    n = (C.c_int * M)(*[len(e) for e in ends])
    out = (Event * cap)()
    k = lib().gwo_coincidence(ptrs, n, M, int(window), int(slide), out, cap)
    return [(o.t_first, o.t_last, o.n_triggers) for o in out[:min(k, cap)]]


def find_peaks(x, height, width, cap=1 << 16):
    """SciPy's find_peaks(x, height=height, width=width) restated -> (count, [(index, height,
    prominence, width, left_ip, right_ip)])."""
    x, xp = _d(x)
    out = (Peak * cap)()
    n = lib().gwo_find_peaks(xp, x.shape[0], float(height), float(width), out, cap)
    return n, [(o.index, o.height, o.prominence, o.width, o.left_ip, o.right_ip) for o in out[:min(n, cap)]]
