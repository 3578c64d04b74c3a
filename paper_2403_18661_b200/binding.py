"""Thin ctypes binding of include/aframe.h: argument marshalling only.

Every step of the path runs in the CUDA kernels of libaframe_b200.so; torch is used for device
memory and streams.  There is no CPU fallback: if the shared library is missing or no sm_100 device
is present, calls fail loudly.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libaframe_b200.so")

OK, EINVAL, ESHAPE, ENOMEM, ECUDA, ESTATE, EUNSUPPORTED = range(7)
FP32, BF16, F16 = 0, 1, 2
_DT = {torch.float32: FP32, torch.bfloat16: BF16, torch.float16: F16}
_STATUS = {0: "AFRAME_OK", 1: "AFRAME_EINVAL", 2: "AFRAME_ESHAPE", 3: "AFRAME_ENOMEM", 4: "AFRAME_ECUDA",
           5: "AFRAME_ESTATE", 6: "AFRAME_EUNSUPPORTED"}


class AframeError(RuntimeError):
    def __init__(self, status, msg=""):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


class aframe_config(C.Structure):
    _fields_ = [("size", C.c_uint32), ("n_channels", C.c_int32), ("fs", C.c_double),
                ("welch_nfft", C.c_int32), ("welch_hop", C.c_int32), ("filter_len", C.c_int32),
                ("n_design", C.c_int32), ("f_lo", C.c_double), ("f_hi", C.c_double),
                ("kernel_len", C.c_int32), ("stride", C.c_int32), ("psd_len", C.c_int64),
                ("psd_update", C.c_int64), ("strain_scale_log2", C.c_int32), ("precision", C.c_int32),
                ("welch_average", C.c_int32), ("stream_full_forward", C.c_int32)]


class aframe_stage_plan(C.Structure):
    _fields_ = [("first_layer", C.c_int32), ("n_layers", C.c_int32), ("T", C.c_int32), ("C", C.c_int32), ("head", C.c_int32),
                ("tail", C.c_int32), ("packed", C.c_int32), ("P", C.c_int32), ("spare_slots", C.c_int32),
                ("e_head", C.c_int32 * 16), ("e_tail", C.c_int32 * 16), ("tbox", C.c_int32 * 16)]


EXPORTS = {
    "aframe_config_default": (C.c_int, [C.POINTER(aframe_config)]),
    "aframe_create": (C.c_int, [C.POINTER(aframe_config), C.c_void_p, C.POINTER(C.c_void_p)]),
    "aframe_destroy": (None, [C.c_void_p]),
    "aframe_last_error": (C.c_char_p, [C.c_void_p]),
    "aframe_psd_welch": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p]),
    "aframe_psd_welch_static": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p]),
    "aframe_psd_welch_static_max_floats": (C.c_int64, []),
    "aframe_whiten": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_void_p, C.c_int64, C.c_int]),
    "aframe_filter_taps": (C.c_int, [C.c_void_p, C.c_void_p]),
    "aframe_rfft8192": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]),
    "aframe_irfft8192": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]),
    "aframe_whiten_rolling": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_void_p, C.c_int64, C.c_int,
                                        C.POINTER(C.c_int64)]),
    "aframe_weights_load": (C.c_int, [C.c_void_p, C.c_char_p, C.c_size_t, C.POINTER(C.c_void_p)]),
    "aframe_weights_free": (None, [C.c_void_p]),
    "aframe_forward": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p]),
    "aframe_forward_strided": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int64, C.c_int64,
                                         C.POINTER(C.c_int64), C.c_int64, C.c_void_p]),
    "aframe_stream_create": (C.c_int, [C.c_void_p, C.c_void_p, C.POINTER(C.c_void_p)]),
    "aframe_stream_reset": (C.c_int, [C.c_void_p]),
    "aframe_stream_destroy": (None, [C.c_void_p]),
    "aframe_stream_step": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "aframe_launch_count": (C.c_int64, [C.c_void_p]),
    "aframe_tensor_macs": (C.c_double, [C.c_void_p]),
    "aframe_whiten_batch": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_void_p, C.c_int]),
    "aframe_far": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.c_int64, C.c_double, C.c_void_p, C.c_void_p]),
    "aframe_postprocess": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_int32, C.c_int32,
                                     C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_int64)]),
    "aframe_stream_graph_replays": (C.c_int64, [C.c_void_p]),
    "aframe_stream_incremental": (C.c_int32, [C.c_void_p]),
    "aframe_describe_stream_plan": (C.c_int, [C.c_char_p, C.c_size_t, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_int32),
                                              C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int32), C.POINTER(C.c_int32)]),
    "aframe_describe_shared_plan": (C.c_int, [C.c_char_p, C.c_size_t, C.c_int32, C.c_int32, C.c_int32, C.c_int64, C.POINTER(C.c_int32),
                                              C.POINTER(aframe_stage_plan), C.c_int32, C.POINTER(C.c_int32)]),
    "aframe_score_timeslides": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64, C.c_int64,
                                          C.POINTER(C.c_int64), C.c_int32, C.c_int64, C.c_void_p]),
    "aframe_score_timeslides_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_int64, C.c_int64,
                                               C.c_int64, C.POINTER(C.c_int64), C.c_int32, C.c_int64, C.c_void_p]),
    "aframe_profile": (C.c_int, [C.c_void_p, C.c_int]),
    "aframe_profile_layers": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p, C.POINTER(C.c_float), C.c_int32]),
    "aframe_profile_read": (C.c_int, [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]),
}
PROF_KINDS = ("welch", "design", "whiten", "stem", "conv", "head", "stream", "gather")

_lib = None


def load_library():
    """dlopen the C-ABI library and declare every prototype of include/aframe.h."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2403_18661_b200.build` "
                              "(or __graft_entry__.build()); there is no fallback path")
        lib = C.CDLL(LIB_PATH)
        for name, (res, args) in EXPORTS.items():
            fn = getattr(lib, name)
            fn.restype, fn.argtypes = res, args
        _lib = lib
    return _lib


def describe_shared_plan(blob: bytes, kernel_len=3072, n_channels=2, window_spacing=128, n_windows=4096):
    """aframe_describe_shared_plan (host arithmetic only: works without a GPU).  Returns (first_stage_blocks, [stage dicts])."""
    lib = load_library()
    s1 = C.c_int32(0)
    n = C.c_int32(0)
    arr = (aframe_stage_plan * 8)()
    st = lib.aframe_describe_shared_plan(blob, len(blob), int(kernel_len), int(n_channels), int(window_spacing), int(n_windows),
                                         C.byref(s1), arr, 8, C.byref(n))
    if st != OK:
        raise AframeError(st, "aframe_describe_shared_plan")
    out = []
    for i in range(n.value):
        a = arr[i]
        nl = min(a.n_layers, 16)
        out.append(dict(first_layer=a.first_layer, n_layers=a.n_layers, T=a.T, C=a.C, head=a.head, tail=a.tail, packed=bool(a.packed),
                        P=a.P, spare_slots=a.spare_slots, e_head=list(a.e_head[:nl]), e_tail=list(a.e_tail[:nl]), tbox=list(a.tbox[:nl])))
    return s1.value, out


def describe_stream_plan(blob: bytes, kernel_len=3072, n_channels=2, stride=128):
    """aframe_describe_stream_plan (host arithmetic only).  Returns a list of dicts (t_out, head, tail, new) per layer, [] if
    the table / stride does not qualify for the incremental network."""
    lib = load_library()
    n = C.c_int32(0)
    cap = 256
    arrs = [(C.c_int32 * cap)() for _ in range(4)]
    st = lib.aframe_describe_stream_plan(blob, len(blob), int(kernel_len), int(n_channels), int(stride), cap, C.byref(n), *arrs)
    if st != OK:
        raise AframeError(st, "aframe_describe_stream_plan")
    return [dict(t_out=arrs[0][i], head=arrs[1][i], tail=arrs[2][i], new=arrs[3][i]) for i in range(min(n.value, cap))]


def default_config(**overrides) -> aframe_config:
    cfg = aframe_config()
    load_library().aframe_config_default(C.byref(cfg))
    for k, v in overrides.items():
        if not hasattr(cfg, k):
            raise AttributeError(k)
        setattr(cfg, k, v)
    return cfg


def _ptr(t: torch.Tensor):
    return C.c_void_p(t.data_ptr())


def _need(t, dtype, what):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{what}: expected a contiguous CUDA tensor of {dtype}")


class Weights:
    def __init__(self, ctx, handle):
        self.ctx, self.handle = ctx, handle

    def free(self):
        if self.handle:
            load_library().aframe_weights_free(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


class Context:
    """aframe_ctx bound to a torch CUDA stream (default: the current stream)."""

    def __init__(self, cfg: aframe_config | None = None, stream: torch.cuda.Stream | None = None, **overrides):
        self.lib = load_library()
        self.cfg = cfg if cfg is not None else default_config(**overrides)
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        h = C.c_void_p()
        st = self.lib.aframe_create(C.byref(self.cfg), C.c_void_p(self.stream.cuda_stream), C.byref(h))
        if st != OK:
            raise AframeError(st, "aframe_create")
        self.handle = h

    def close(self):
        if getattr(self, "handle", None):
            self.lib.aframe_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st):
        if st != OK:
            raise AframeError(st, self.lib.aframe_last_error(self.handle).decode())

    @property
    def n_freq(self):
        return self.cfg.welch_nfft // 2 + 1

    def launch_count(self):
        return int(self.lib.aframe_launch_count(self.handle))

    def tensor_macs(self):
        return float(self.lib.aframe_tensor_macs(self.handle))

    # ---- O-1
    def psd_welch(self, strain: torch.Tensor, out: torch.Tensor | None = None):
        _need(strain, torch.float32, "strain")
        c, n = strain.shape
        if out is None:
            out = torch.empty((c, self.n_freq), dtype=torch.float32, device=strain.device)
        self._check(self.lib.aframe_psd_welch(self.handle, _ptr(strain), n, strain.stride(0), _ptr(out)))
        return out

    def psd_welch_static(self, strain: torch.Tensor, out: torch.Tensor):
        """aframe_psd_welch_static: the same PSD with its scratch in a fixed device array (the call allocates nothing, so
        `out` is the caller's)."""
        _need(strain, torch.float32, "strain"); _need(out, torch.float32, "out")
        c, n = strain.shape
        if tuple(out.shape) != (c, self.n_freq) or not out.is_contiguous():
            raise ValueError("out must be a contiguous [C][welch_nfft / 2 + 1] tensor")
        self._check(self.lib.aframe_psd_welch_static(self.handle, _ptr(strain), n, strain.stride(0), _ptr(out)))
        return out

    # ---- O-2 / O-3
    def whiten(self, strain, psd, out=None, out_dtype=torch.float32):
        _need(strain, torch.float32, "strain"); _need(psd, torch.float32, "psd")
        c, n = strain.shape
        n_out = max(n - self.cfg.filter_len, 0)
        if out is None:
            out = torch.empty((c, max(n_out, 1)), dtype=out_dtype, device=strain.device)
        prec = _DT[out.dtype]
        self._check(self.lib.aframe_whiten(self.handle, _ptr(strain), n, strain.stride(0), _ptr(psd), _ptr(out),
                                           out.stride(0), prec))
        return out[:, :n_out]

    def rfft8192(self, x, out=None):
        """x [batch][8192] float32 CUDA -> one-sided spectrum [batch][4097][2] (re, im)."""
        _need(x, torch.float32, "x")
        if out is None:
            out = torch.empty((x.shape[0], 4097, 2), dtype=torch.float32, device=x.device)
        self._check(self.lib.aframe_rfft8192(self.handle, _ptr(x), x.shape[0], _ptr(out)))
        return out

    def irfft8192(self, spec, out=None):
        """spec [batch][4097][2] float32 CUDA -> [batch][8192] real rows (1/8192 included)."""
        _need(spec, torch.float32, "spec")
        if out is None:
            out = torch.empty((spec.shape[0], 8192), dtype=torch.float32, device=spec.device)
        self._check(self.lib.aframe_irfft8192(self.handle, _ptr(spec), spec.shape[0], _ptr(out)))
        return out

    def filter_taps(self):
        out = torch.empty((self.cfg.n_channels, self.cfg.filter_len + 1), dtype=torch.float32, device="cuda")
        self._check(self.lib.aframe_filter_taps(self.handle, _ptr(out)))
        return out

    def whiten_rolling(self, strain, out=None, out_dtype=torch.float32):
        _need(strain, torch.float32, "strain")
        c, n = strain.shape
        if out is None:
            out = torch.empty((c, max(n, 1)), dtype=out_dtype, device=strain.device)
        prec = _DT[out.dtype]
        n_out = C.c_int64(0)
        self._check(self.lib.aframe_whiten_rolling(self.handle, _ptr(strain), n, strain.stride(0), _ptr(out),
                                                   out.stride(0), prec, C.byref(n_out)))
        return out[:, : n_out.value]

    # ---- weights / O-5
    def load_weights(self, blob: bytes) -> Weights:
        h = C.c_void_p()
        self._check(self.lib.aframe_weights_load(self.handle, blob, len(blob), C.byref(h)))
        return Weights(self, h)

    def forward(self, weights: Weights, windows, scores=None):
        _need(windows, torch.float32, "windows")
        b = windows.shape[0]
        if scores is None:
            scores = torch.empty((b,), dtype=torch.float32, device=windows.device)
        self._check(self.lib.aframe_forward(self.handle, weights.handle, _ptr(windows), b, _ptr(scores)))
        return scores

    def forward_strided(self, weights: Weights, white, first, n_windows, chan_shift=None, scores=None):
        if not (white.is_cuda and white.is_contiguous() and white.dtype in _DT):
            raise TypeError("white: expected a contiguous CUDA tensor of float32, bfloat16 or float16")
        if scores is None:
            scores = torch.empty((n_windows,), dtype=torch.float32, device=white.device)
        shifts = None
        if chan_shift is not None:
            shifts = (C.c_int64 * self.cfg.n_channels)(*[int(v) for v in chan_shift])
        prec = _DT[white.dtype]
        self._check(self.lib.aframe_forward_strided(self.handle, weights.handle, _ptr(white), prec, white.stride(0),
                                                    int(first), shifts, int(n_windows), _ptr(scores)))
        return scores

    # ---- configs[3]: whiten once, score every timeslide
    def score_timeslides(self, weights: Weights, strain, first, n_windows, slide_shifts, batch=4096, scores=None):
        """strain: CUDA tensor (device entry point) or pinned/pageable CPU tensor (host entry point,
        copies inside the call, synchronises).  Returns scores [n_slides][n_windows] on the same side."""
        if not (isinstance(strain, torch.Tensor) and strain.dtype == torch.float32 and strain.stride(1) == 1):
            raise TypeError("strain: expected a float32 tensor [C][N] with unit inner stride")
        c, n = strain.shape
        ns = len(slide_shifts)
        sh = (C.c_int64 * ns)(*[int(v) for v in slide_shifts])
        if scores is None:
            scores = torch.empty((ns, n_windows), dtype=torch.float32, device=strain.device,
                                 pin_memory=not strain.is_cuda)
        fn = self.lib.aframe_score_timeslides if strain.is_cuda else self.lib.aframe_score_timeslides_host
        self._check(fn(self.handle, weights.handle, _ptr(strain), n, strain.stride(0), int(first), int(n_windows), sh, ns,
                       int(batch), _ptr(scores)))
        return scores

    # ---- NEXT-1: top-hat integration + clustering
    def postprocess(self, scores, n_int=16, n_cluster=128):
        """scores [n_series][n] (or [n]) float32 CUDA -> (integrated [n_series][n], trig_value, trig_index [n_series][n_trig])."""
        _need(scores, torch.float32, "scores")
        s2 = scores if scores.dim() == 2 else scores[None]
        ns, n = s2.shape
        n_trig = -(-n // n_cluster)
        integ = torch.empty((ns, n), dtype=torch.float32, device=scores.device)
        val = torch.empty((ns, n_trig), dtype=torch.float32, device=scores.device)
        idx = torch.empty((ns, n_trig), dtype=torch.int64, device=scores.device)
        nt = C.c_int64(0)
        self._check(self.lib.aframe_postprocess(self.handle, _ptr(s2), ns, n, s2.stride(0), int(n_int), int(n_cluster),
                                                _ptr(integ), _ptr(val), _ptr(idx), C.byref(nt)))
        assert nt.value == n_trig
        return integ, val, idx

    # ---- NEXT-4
    def whiten_batch(self, strain, n_psd, out_dtype=torch.float32):
        """strain [B][C][n] float32 CUDA -> [B][C][n - n_psd - filter_len]: own PSD (first n_psd samples) per row."""
        _need(strain, torch.float32, "strain")
        b, c, n = strain.shape
        if c != self.cfg.n_channels:
            raise ValueError("strain must be [B][n_channels][n]")
        n_out = n - int(n_psd) - self.cfg.filter_len
        out = torch.empty((b, c, max(n_out, 1)), dtype=out_dtype, device=strain.device)
        prec = _DT[out_dtype]
        self._check(self.lib.aframe_whiten_batch(self.handle, _ptr(strain), b, n, int(n_psd), _ptr(out), prec))
        return out

    def far(self, background, events, livetime_s):
        """counts[i] = #{background > events[i]} (int64), far = counts / livetime_s (float64, 1/s)."""
        _need(events, torch.float32, "events")
        if background.numel():
            _need(background, torch.float32, "background")
        counts = torch.empty((events.numel(),), dtype=torch.int64, device=events.device)
        far = torch.empty((events.numel(),), dtype=torch.float64, device=events.device)
        self._check(self.lib.aframe_far(self.handle, _ptr(background) if background.numel() else None, background.numel(),
                                        _ptr(events), events.numel(), float(livetime_s), _ptr(counts), _ptr(far)))
        return counts, far

    # ---- per-stage device timing
    def profile(self, enable: bool):
        self._check(self.lib.aframe_profile(self.handle, 1 if enable else 0))

    def profile_layers(self, weights, windows, n_layers):
        _need(windows, torch.float32, "windows")
        scores = torch.empty((windows.shape[0],), dtype=torch.float32, device=windows.device)
        ms = (C.c_float * n_layers)()
        self._check(self.lib.aframe_profile_layers(self.handle, weights.handle, _ptr(windows), windows.shape[0], _ptr(scores),
                                                   ms, n_layers))
        return list(ms), scores

    def profile_read(self):
        ms = (C.c_double * 8)()
        nl = (C.c_int64 * 8)()
        self._check(self.lib.aframe_profile_read(self.handle, ms, nl))
        return {k: (ms[i], int(nl[i])) for i, k in enumerate(PROF_KINDS)}

    # ---- O-6
    def stream_create(self, weights: Weights):
        return Stream(self, weights)


class Stream:
    def __init__(self, ctx: Context, weights: Weights):
        self.ctx, self.weights = ctx, weights
        h = C.c_void_p()
        ctx._check(ctx.lib.aframe_stream_create(ctx.handle, weights.handle, C.byref(h)))
        self.handle = h
        self.score = torch.zeros(1, dtype=torch.float32, device="cuda")
        self.n_scores = torch.zeros(1, dtype=torch.int32, device="cuda")

    def reset(self):
        self.ctx._check(self.ctx.lib.aframe_stream_reset(self.handle))

    @property
    def uses_graph(self):
        return int(self.ctx.lib.aframe_stream_graph_replays(self.handle)) > 0

    @property
    def incremental(self):
        """CTAs of the cluster that runs the incremental network, 0 = one full forward per update."""
        return int(self.ctx.lib.aframe_stream_incremental(self.handle))

    def step(self, new_samples: torch.Tensor):
        """Enqueue one update; results land in self.score / self.n_scores (device tensors)."""
        _need(new_samples, torch.float32, "new_samples")
        self.ctx._check(self.ctx.lib.aframe_stream_step(self.ctx.handle, _ptr(new_samples), self.handle,
                                                        _ptr(self.score), _ptr(self.n_scores)))

    def close(self):
        if getattr(self, "handle", None):
            self.ctx.lib.aframe_stream_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
