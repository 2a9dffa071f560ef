"""ctypes binding of libgwi.so.  Same names as include/gwi.h; marshalling only."""
import ctypes as C
import os

import torch

from . import build as _build

FP32, FP16 = 0, 1
STATUS_NAMES = {0: "GWI_OK", 1: "GWI_ERR_ARG", 2: "GWI_ERR_IO", 3: "GWI_ERR_FORMAT", 4: "GWI_ERR_UNSUPPORTED",
                5: "GWI_ERR_CUDA", 6: "GWI_ERR_NOMEM", 7: "GWI_ERR_CAPACITY"}
EXPORTED_SYMBOLS = ["gwi_load_model", "gwi_free_model", "gwi_model_info", "gwi_model_uses_tensor_cores",
                    "gwi_infer_workspace_bytes", "gwi_infer", "gwi_carry_bytes", "gwi_triggers_workspace_bytes",
                    "gwi_ensemble_triggers", "gwi_ensemble_triggers_static", "gwi_last_error", "gwi_version", "gwi_launch_count", "gwi_stream_create",
                    "gwi_stream_tail_samples", "gwi_stream_prime", "gwi_stream_push", "gwi_stream_push_host",
                    "gwi_stream_finish", "gwi_stream_samples_done", "gwi_stream_backend", "gwi_stream_set_shard", "gwi_stream_destroy", "gwi_stream_set_rule",
                    "gwi_coincidence", "gwi_find_peaks_workspace_bytes", "gwi_find_peaks", "gwi_sweep_workspace_bytes", "gwi_threshold_sweep", "gwi_whiten_workspace_bytes",
                    "gwi_whiten"]


class GwiError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


class Trigger(C.Structure):
    _fields_ = [("slide", C.c_int32), ("model_mask", C.c_int32), ("start", C.c_int64), ("end", C.c_int64),
                ("peak_p", C.c_float), ("mean_p", C.c_float)]


_lib = None


def lib():
    """Load (building if stale and nvcc is present) the shared library.  Raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    try:
        path = _build.build()
    except Exception:
        if not os.path.exists(path):
            raise
    L = C.CDLL(path)
    vp, i32p = C.c_void_p, C.POINTER(C.c_int32)
    L.gwi_load_model.restype = C.c_int
    L.gwi_load_model.argtypes = [C.c_char_p, C.c_int, C.c_int, C.POINTER(vp)]
    L.gwi_free_model.restype = None
    L.gwi_free_model.argtypes = [vp]
    L.gwi_model_info.restype = C.c_int
    L.gwi_model_info.argtypes = [vp] + [i32p] * 8
    L.gwi_model_uses_tensor_cores.restype = C.c_int
    L.gwi_model_uses_tensor_cores.argtypes = [vp]
    L.gwi_infer_workspace_bytes.restype = C.c_size_t
    L.gwi_infer_workspace_bytes.argtypes = [vp, C.c_int64, C.c_int32]
    L.gwi_infer.restype = C.c_int
    L.gwi_infer.argtypes = [vp, vp, C.c_int64, C.c_int32, vp, vp, C.c_size_t, vp]
    L.gwi_carry_bytes.restype = C.c_size_t
    L.gwi_triggers_workspace_bytes.restype = C.c_size_t
    L.gwi_triggers_workspace_bytes.argtypes = [C.c_int64]
    L.gwi_ensemble_triggers.restype = C.c_int
    L.gwi_ensemble_triggers.argtypes = [C.POINTER(vp), C.c_int32, C.c_int64, C.c_int64, C.c_float, C.c_int64, C.c_int32,
                                        C.c_int, vp, vp, C.c_int32, vp, vp, vp, C.c_size_t, vp]
    L.gwi_ensemble_triggers_static.restype = C.c_int
    L.gwi_ensemble_triggers_static.argtypes = [C.POINTER(vp), C.c_int32, C.c_int64, C.c_int64, C.c_float, C.c_int64, C.c_int32,
                                               C.c_int, vp, vp, C.c_int32, vp, vp, vp]
    L.gwi_stream_create.restype = C.c_int
    L.gwi_stream_create.argtypes = [C.POINTER(vp), C.c_int32, C.POINTER(C.c_int64), C.c_int32, C.c_int64, C.c_int64,
                                    C.c_float, C.c_int64, C.c_int32, vp, C.POINTER(vp)]
    L.gwi_stream_tail_samples.restype = C.c_int64
    L.gwi_stream_tail_samples.argtypes = [vp]
    L.gwi_stream_prime.restype = C.c_int
    L.gwi_stream_prime.argtypes = [vp, vp, C.c_int64, vp]
    L.gwi_stream_push.restype = C.c_int
    L.gwi_stream_push.argtypes = [vp, vp, vp, C.c_int64, vp]
    L.gwi_stream_push_host.restype = C.c_int
    L.gwi_stream_push_host.argtypes = [vp, vp, vp, C.c_int64, vp]
    L.gwi_stream_finish.restype = C.c_int
    L.gwi_stream_finish.argtypes = [vp, vp, C.c_int32, i32p, vp]
    L.gwi_stream_samples_done.restype = C.c_int64
    L.gwi_stream_samples_done.argtypes = [vp]
    L.gwi_stream_set_shard.restype = C.c_int
    L.gwi_stream_set_shard.argtypes = [vp, C.c_int64, C.c_int64]
    L.gwi_stream_backend.restype = C.c_int
    L.gwi_stream_backend.argtypes = [vp]
    L.gwi_stream_destroy.restype = None
    L.gwi_stream_destroy.argtypes = [vp]
    L.gwi_stream_set_rule.restype = C.c_int
    L.gwi_stream_set_rule.argtypes = [vp, C.c_int]
    L.gwi_coincidence.restype = C.c_int
    L.gwi_coincidence.argtypes = [vp, C.c_int32, C.c_int32, C.c_int64, vp, C.c_int32, i32p]
    L.gwi_find_peaks_workspace_bytes.restype = C.c_size_t
    L.gwi_find_peaks_workspace_bytes.argtypes = [C.c_int64, C.c_int32]
    L.gwi_find_peaks.restype = C.c_int
    L.gwi_find_peaks.argtypes = [vp, C.c_int64, C.c_float, C.c_double, vp, C.c_int32, vp, vp, C.c_size_t, vp]
    L.gwi_sweep_workspace_bytes.restype = C.c_size_t
    L.gwi_sweep_workspace_bytes.argtypes = [C.c_int32]
    L.gwi_threshold_sweep.restype = C.c_int
    L.gwi_threshold_sweep.argtypes = [C.POINTER(vp), C.c_int32, C.c_int64, vp, C.c_int32, C.c_int64, vp, vp, C.c_size_t, vp]
    L.gwi_whiten_workspace_bytes.restype = C.c_size_t
    L.gwi_whiten_workspace_bytes.argtypes = [C.c_int64, C.c_int32]
    L.gwi_whiten.restype = C.c_int
    L.gwi_whiten.argtypes = [vp, C.c_int64, C.c_int32, vp, C.c_int, vp, C.c_size_t, vp]
    L.gwi_last_error.restype = C.c_char_p
    L.gwi_version.restype = C.c_int
    L.gwi_launch_count.restype = C.c_int64
    _lib = L
    return L


def last_error():
    return lib().gwi_last_error().decode()


def version():
    return lib().gwi_version()


def launch_count():
    return lib().gwi_launch_count()


def _check(st):
    if st != 0:
        raise GwiError(st, last_error())


def _stream_ptr(device):
    return C.c_void_p(torch.cuda.current_stream(device).cuda_stream)


class Model:
    """Handle on a gwi_model (gwi_load_model / gwi_free_model)."""

    def __init__(self, path, precision=FP32, device=0):
        self._h = C.c_void_p()
        self.device = int(device)
        self.precision = precision
        _check(lib().gwi_load_model(os.fsencode(path), int(precision), self.device, C.byref(self._h)))
        v = [C.c_int32() for _ in range(8)]
        _check(lib().gwi_model_info(self._h, *[C.byref(x) for x in v]))
        (self.n_branch, self.c_in, self.R, self.S, self.k, self.L, self.Hh, self.receptive_field) = [x.value for x in v]
        self.uses_tensor_cores = bool(lib().gwi_model_uses_tensor_cores(self._h))
        self._ws = None

    def close(self):
        if self._h:
            lib().gwi_free_model(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def workspace_bytes(self, B, T):
        return lib().gwi_infer_workspace_bytes(self._h, int(B), int(T))

    def infer(self, strain, out=None):
        """gwi_infer: strain [B][T][C] device tensor (float32 in FP32 mode, float16 in FP16 mode) -> prob [B][T]."""
        return infer(self, strain, out)


def load_model(path, precision=FP32, device=0):
    return Model(path, precision, device)


def infer(model, strain, out=None):
    if not strain.is_cuda:
        raise GwiError(1, "strain must be a CUDA tensor (no CPU fallback)")
    want = torch.float16 if model.precision == FP16 else torch.float32
    if strain.dtype != want or strain.dim() != 3 or strain.shape[2] != model.n_branch * model.c_in:
        raise GwiError(1, f"strain must be [B][T][{model.n_branch * model.c_in}] {want}")
    strain = strain.contiguous()
    B, T, _ = strain.shape
    if out is None:
        out = torch.empty((B, T), dtype=torch.float32, device=strain.device)
    need = model.workspace_bytes(B, T)
    if model._ws is None or model._ws.numel() < need:
        model._ws = torch.empty(max(need, 256), dtype=torch.uint8, device=strain.device)
    _check(lib().gwi_infer(model._h, C.c_void_p(strain.data_ptr()), B, T, C.c_void_p(out.data_ptr()),
                           C.c_void_p(model._ws.data_ptr()), model._ws.numel(), _stream_ptr(strain.device)))
    return out


def ensemble_triggers(probs, threshold, min_len, t0=0, slide_id=0, last_chunk=True, carry=None, capacity=4096,
                      want_pbar=False, sync=True):
    """gwi_ensemble_triggers on a list of [N] float32 device tensors.
    Returns (count, [Trigger...], pbar or None); raises GwiError(GWI_ERR_CAPACITY) when count > capacity
    (the exception carries .count and .records with the valid prefix)."""
    dev = probs[0].device
    if not probs[0].is_cuda:
        raise GwiError(1, "probabilities must be CUDA tensors (no CPU fallback)")
    probs = [p.contiguous() for p in probs]
    N = probs[0].numel()
    ptrs = (C.c_void_p * len(probs))(*[p.data_ptr() for p in probs])
    trig = torch.zeros(max(capacity, 1) * C.sizeof(Trigger), dtype=torch.uint8, device=dev)
    cnt = torch.zeros(1, dtype=torch.int32, device=dev)
    pbar = torch.empty(N, dtype=torch.float32, device=dev) if want_pbar else None
    wsb = lib().gwi_triggers_workspace_bytes(N)
    ws = torch.empty(max(wsb, 256), dtype=torch.uint8, device=dev)
    _check(lib().gwi_ensemble_triggers(ptrs, len(probs), N, int(t0), float(threshold), int(min_len), int(slide_id),
                                       int(bool(last_chunk)), C.c_void_p(carry.data_ptr()) if carry is not None else None,
                                       C.c_void_p(trig.data_ptr()), int(capacity), C.c_void_p(cnt.data_ptr()),
                                       C.c_void_p(pbar.data_ptr()) if pbar is not None else None,
                                       C.c_void_p(ws.data_ptr()), ws.numel(), _stream_ptr(dev)))
    if not sync:
        return cnt, trig, pbar
    n = int(cnt.item())
    raw = trig.cpu().numpy().tobytes()
    recs = [Trigger.from_buffer_copy(raw, i * C.sizeof(Trigger)) for i in range(min(n, capacity))]
    if n > capacity:
        e = GwiError(7, f"{n} triggers > capacity {capacity}")
        e.count, e.records = n, recs
        raise e
    return n, recs, pbar


TRIGGERS_STATIC_MAX_N = 1 << 24


def ensemble_triggers_static(probs, threshold, min_len, trig, cnt, t0=0, slide_id=0, last_chunk=True, carry=None, pbar=None):
    """gwi_ensemble_triggers_static: the call that allocates nothing.  Every buffer is the caller's: probs = list of [N]
    float32 device tensors (contiguous), trig = uint8 device tensor of capacity * sizeof(Trigger) bytes, cnt = int32[1],
    pbar = optional float32 [N].  Asynchronous on the current stream; N <= TRIGGERS_STATIC_MAX_N."""
    dev = probs[0].device
    if not probs[0].is_cuda:
        raise GwiError(1, "probabilities must be CUDA tensors (no CPU fallback)")
    N = probs[0].numel()
    ptrs = (C.c_void_p * len(probs))(*[p.data_ptr() for p in probs])
    with torch.cuda.device(dev):
        _check(lib().gwi_ensemble_triggers_static(ptrs, len(probs), N, int(t0), float(threshold), int(min_len), int(slide_id),
                                                  int(bool(last_chunk)), C.c_void_p(carry.data_ptr()) if carry is not None else None,
                                                  C.c_void_p(trig.data_ptr()), trig.numel() // C.sizeof(Trigger),
                                                  C.c_void_p(cnt.data_ptr()),
                                                  C.c_void_p(pbar.data_ptr()) if pbar is not None else None, _stream_ptr(dev)))


def threshold_sweep(probs, thresholds, min_len):
    """gwi_threshold_sweep: probs = list of [N] float32 device tensors, thresholds ascending -> int64 device tensor [K]."""
    dev = probs[0].device
    probs = [p.contiguous() for p in probs]
    N = probs[0].numel()
    ptrs = (C.c_void_p * len(probs))(*[p.data_ptr() for p in probs])
    th = torch.as_tensor(thresholds, dtype=torch.float32).to(dev).contiguous()
    K = th.numel()
    counts = torch.zeros(K, dtype=torch.int64, device=dev)
    ws = torch.empty(max(lib().gwi_sweep_workspace_bytes(K), 256), dtype=torch.uint8, device=dev)
    _check(lib().gwi_threshold_sweep(ptrs, len(probs), N, C.c_void_p(th.data_ptr()), K, int(min_len),
                                     C.c_void_p(counts.data_ptr()), C.c_void_p(ws.data_ptr()), ws.numel(), _stream_ptr(dev)))
    return counts


class Peak(C.Structure):
    _fields_ = [("index", C.c_int64), ("height", C.c_float), ("prominence", C.c_float), ("width", C.c_double),
                ("left_ip", C.c_double), ("right_ip", C.c_double)]


def find_peaks(x, height, min_width, capacity=65536, sync=True):
    """gwi_find_peaks on a [N] float32 device tensor -> (count, [Peak...]) sorted by index; raises GwiError(GWI_ERR_CAPACITY)
    when count > capacity.  sync=False: nothing is read back, returns the device tensors (count int32[1], records as bytes)."""
    if not x.is_cuda or x.dtype != torch.float32:
        raise GwiError(1, "x must be a float32 CUDA tensor (no CPU fallback)")
    x = x.contiguous()
    N = x.numel()
    out = torch.zeros(max(capacity, 1) * C.sizeof(Peak), dtype=torch.uint8, device=x.device)
    cnt = torch.zeros(1, dtype=torch.int32, device=x.device)
    ws = torch.empty(max(lib().gwi_find_peaks_workspace_bytes(N, int(capacity)), 256), dtype=torch.uint8, device=x.device)
    _check(lib().gwi_find_peaks(C.c_void_p(x.data_ptr()), N, float(height), float(min_width), C.c_void_p(out.data_ptr()),
                                int(capacity), C.c_void_p(cnt.data_ptr()), C.c_void_p(ws.data_ptr()), ws.numel(), _stream_ptr(x.device)))
    if not sync:
        return cnt, out
    n = int(cnt.item())
    if n > capacity:
        raise GwiError(7, f"{n} peaks > capacity {capacity}")
    raw = out.cpu().numpy().tobytes()
    return n, [Peak.from_buffer_copy(raw, i * C.sizeof(Peak)) for i in range(n)]


def whiten(raw, nper, half=True):
    """gwi_whiten: raw [n] float32 device tensor -> whitened unit-variance [n] tensor (float16 or float32)."""
    raw = raw.contiguous()
    n = raw.numel()
    out = torch.empty(n, dtype=torch.float16 if half else torch.float32, device=raw.device)
    ws = torch.empty(max(lib().gwi_whiten_workspace_bytes(n, int(nper)), 256), dtype=torch.uint8, device=raw.device)
    _check(lib().gwi_whiten(C.c_void_p(raw.data_ptr()), n, int(nper), C.c_void_p(out.data_ptr()), int(bool(half)),
                            C.c_void_p(ws.data_ptr()), ws.numel(), _stream_ptr(raw.device)))
    return out


def new_carry(device=0):
    return torch.zeros(lib().gwi_carry_bytes(), dtype=torch.uint8, device=f"cuda:{device}" if isinstance(device, int) else device)


RULE_MEAN, RULE_PER_MODEL = 0, 1
EDGE_LEFT, EDGE_RIGHT = 1 << 30, 1 << 29
BACKEND_GENERIC, BACKEND_NARROW, BACKEND_TENSOR, BACKEND_TENSOR_SLIDES = 0, 1, 2, 3


class Event(C.Structure):
    _fields_ = [("t_first", C.c_int64), ("t_last", C.c_int64), ("n_triggers", C.c_int32), ("slide", C.c_int32)]


def coincidence(records, n_models, window, capacity=4096):
    """gwi_coincidence on a list of Trigger records (per-model rule) -> [Event...] sorted by (slide, t_first)."""
    arr = (Trigger * max(len(records), 1))(*records)
    out = (Event * max(capacity, 1))()
    n = C.c_int32(0)
    _check(lib().gwi_coincidence(arr, len(records), int(n_models), int(window), out, int(capacity), C.byref(n)))
    return [Event.from_buffer_copy(out[i]) for i in range(n.value)]


class Stream:
    """Handle on a gwi_stream (gwi_stream_create ... gwi_stream_destroy).  Marshalling only.

    models: list of Model (same architecture / precision); lags: lags in samples; n_total: stream length;
    max_chunk: largest push; want_pbar: keep the mean probability of every slide ([1+n_lags][n_total] float32 device
    tensor in .pbar) for parity tests."""

    def __init__(self, models, n_total, max_chunk, threshold=0.5, min_len=2048, lags=(), capacity=4096, want_pbar=False,
                 rule=RULE_MEAN, shard=None):
        """shard = (t_first, warmup): time-shard mode (gwi_stream_set_shard); n_total then counts the warm-up samples too
        and .pbar covers the kept samples only."""
        self.models = list(models)
        self.device = torch.device("cuda", self.models[0].device)
        self.dtype = torch.float16 if self.models[0].precision == FP16 else torch.float32
        self.capacity = int(capacity)
        n_kept = int(n_total) - (int(shard[1]) if shard else 0)
        shape = (1 + len(lags), n_kept) if rule == RULE_MEAN else (1 + len(lags), len(self.models), n_kept)
        self.pbar = torch.zeros(shape, dtype=torch.float32, device=self.device) if want_pbar else None
        mp = (C.c_void_p * len(self.models))(*[m._h for m in self.models])
        lg = (C.c_int64 * max(len(lags), 1))(*[int(v) for v in lags])
        self._h = C.c_void_p()
        _check(lib().gwi_stream_create(mp, len(self.models), lg, len(lags), int(n_total), int(max_chunk), float(threshold),
                                       int(min_len), self.capacity,
                                       C.c_void_p(self.pbar.data_ptr()) if want_pbar else None, C.byref(self._h)))
        if rule != RULE_MEAN:
            _check(lib().gwi_stream_set_rule(self._h, int(rule)))
        if shard is not None:
            _check(lib().gwi_stream_set_shard(self._h, int(shard[0]), int(shard[1])))

    @property
    def tail_samples(self):
        return lib().gwi_stream_tail_samples(self._h)

    def prime(self, l1_tail, sync=True):
        """l1_tail: the last .tail_samples samples of L1 (torch tensor on the host or the device).  sync=False leaves the
        call asynchronous, as the C-ABI is (the caller then keeps l1_tail alive until the stream has been synchronised)."""
        assert l1_tail.dtype == self.dtype and l1_tail.is_contiguous()
        _check(lib().gwi_stream_prime(self._h, C.c_void_p(l1_tail.data_ptr()), l1_tail.shape[-1], _stream_ptr(self.device)))
        if sync:
            torch.cuda.current_stream(self.device).synchronize()   # the caller may free a host tail right away

    def push(self, h1, l1):
        """h1, l1: [n] tensors of the stream dtype; device tensors -> gwi_stream_push, host tensors (pin them) ->
        gwi_stream_push_host."""
        assert h1.dtype == self.dtype and l1.dtype == self.dtype and h1.is_contiguous() and l1.is_contiguous()
        f = lib().gwi_stream_push if h1.is_cuda else lib().gwi_stream_push_host
        _check(f(self._h, C.c_void_p(h1.data_ptr()), C.c_void_p(l1.data_ptr()), h1.shape[-1], _stream_ptr(self.device)))

    @property
    def backend(self):
        return lib().gwi_stream_backend(self._h)

    @property
    def samples_done(self):
        return lib().gwi_stream_samples_done(self._h)

    def finish(self):
        """-> (count, [Trigger...]) sorted by (slide, start)."""
        buf = (Trigger * max(self.capacity, 1))()
        n = C.c_int32(0)
        st = lib().gwi_stream_finish(self._h, buf, self.capacity, C.byref(n), _stream_ptr(self.device))
        recs = [Trigger.from_buffer_copy(buf[i]) for i in range(min(n.value, self.capacity))]
        if st == 7:
            e = GwiError(7, last_error())
            e.count, e.records = n.value, recs
            raise e
        _check(st)
        return n.value, recs

    def close(self):
        if self._h:
            lib().gwi_stream_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
