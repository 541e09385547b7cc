"""ctypes binding with the same names as the C ABI (include/bg_moe.h).  Marshalling only."""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import torch

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("BG_MOE_LIB") or os.path.join(HERE, "libbg_moe.so")

BG_OK, BG_ERR_INVALID_ARG, BG_ERR_UNSUPPORTED, BG_ERR_CUDA, BG_ERR_NOMEM, BG_ERR_NO_WEIGHTS = 0, -1, -2, -3, -4, -5

EXPORTS = ["bg_moe_create", "bg_moe_destroy", "bg_moe_set_weights", "bg_moe_route", "bg_moe_permute",
           "bg_moe_expert_ffn", "bg_moe_unpermute", "bg_moe_combined_forward", "bg_moe_combined_forward_host",
           "bg_moe_debug_views", "bg_moe_profile_enable", "bg_moe_profile_read", "bg_moe_launch_count", "bg_moe_workspace_bytes", "bg_moe_strerror",
           "bg_moe_last_error", "bg_moe_set_debug", "bg_moe_set_weights_offloaded", "bg_moe_ring_bytes_per_call", "bg_moe_set_precision", "bg_moe_debug_fp8_views", "bg_moe_debug_fp8_down_views", "bg_moe_combined_forward_segments", "bg_moe_fit_roofline", "bg_moe_workspace_bytes_for", "bg_moe_choose_tokens",
           "bg_moe_route_logits_noalloc", "bg_moe_noalloc_last_error", "bg_moe_host_input_sync", "bg_moe_debug_ffn_views", "bg_moe_set_ring_skip_empty"]


class BgMoeConfig(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int32) for n in ("d", "f", "E", "k", "max_tokens", "gate_fn", "device")]


class BgMoeSegment(ctypes.Structure):
    _fields_ = [("hidden", ctypes.c_void_p), ("out", ctypes.c_void_p), ("n_tokens", ctypes.c_int32)]


class BgMoeError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"bg_moe status {status}: {msg}")
        self.status = status


_lib = None


def load_library() -> ctypes.CDLL:
    """Loads libbg_moe.so; raises (no fallback) if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2606_21712_b200.build` "
                              "(there is no CPU fallback)")
        lib = ctypes.CDLL(LIB_PATH)
        vp, i32, i64 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64
        lib.bg_moe_create.argtypes = [ctypes.POINTER(BgMoeConfig), ctypes.POINTER(vp)]
        lib.bg_moe_destroy.argtypes = [vp]
        lib.bg_moe_set_weights.argtypes = [vp] * 7
        lib.bg_moe_set_debug.argtypes = [vp, i32, i32, i32]
        lib.bg_moe_set_weights_offloaded.argtypes = [vp, vp, vp, vp, vp, vp, i32, vp]
        lib.bg_moe_ring_bytes_per_call.argtypes = [vp]
        lib.bg_moe_set_ring_skip_empty.argtypes = [vp, i32]
        lib.bg_moe_ring_bytes_per_call.restype = i64
        lib.bg_moe_set_precision.argtypes = [vp, i32, vp]
        lib.bg_moe_debug_fp8_views.argtypes = [vp] + [ctypes.POINTER(vp)] * 6
        lib.bg_moe_debug_fp8_down_views.argtypes = [vp] + [ctypes.POINTER(vp)] * 5
        lib.bg_moe_route.argtypes = [vp, vp, i32, vp, vp, vp, vp, vp, vp, vp]
        lib.bg_moe_permute.argtypes = [vp, vp, i32, vp, vp, vp, vp, vp, vp]
        lib.bg_moe_expert_ffn.argtypes = [vp, vp, vp, i32, vp, vp]
        lib.bg_moe_unpermute.argtypes = [vp, vp, vp, vp, i32, vp, vp]
        lib.bg_moe_combined_forward.argtypes = [vp, vp, i32, vp, vp]
        lib.bg_moe_combined_forward_host.argtypes = [vp, vp, i32, vp, vp]
        lib.bg_moe_host_input_sync.argtypes = [vp]
        lib.bg_moe_debug_ffn_views.argtypes = [vp] + [ctypes.POINTER(vp)] * 2
        lib.bg_moe_debug_views.argtypes = [vp] + [ctypes.POINTER(vp)] * 7
        lib.bg_moe_profile_enable.argtypes = [vp, ctypes.c_int]
        lib.bg_moe_profile_read.argtypes = [vp, ctypes.POINTER(ctypes.c_float)]
        lib.bg_moe_launch_count.argtypes = [vp]
        lib.bg_moe_launch_count.restype = i64
        lib.bg_moe_workspace_bytes.argtypes = [vp]
        lib.bg_moe_workspace_bytes.restype = i64
        lib.bg_moe_strerror.argtypes = [ctypes.c_int]
        lib.bg_moe_strerror.restype = ctypes.c_char_p
        lib.bg_moe_last_error.argtypes = [vp]
        lib.bg_moe_last_error.restype = ctypes.c_char_p
        lib.bg_moe_route_logits_noalloc.argtypes = [vp, i32, i32, i32, vp, vp, vp, vp, vp]
        lib.bg_moe_noalloc_last_error.argtypes = []
        lib.bg_moe_noalloc_last_error.restype = ctypes.c_char_p
        _lib = lib
    return _lib


def _ptr(t: Optional[torch.Tensor]):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def _chk(t: torch.Tensor, dtype, shape, what: str, cuda: bool = True):
    """Every tensor that crosses the C ABI as a raw pointer: dtype, device, contiguity and shape are checked here
    (the library only sees addresses)."""
    assert isinstance(t, torch.Tensor), f"{what}: tensor expected"
    assert t.dtype == dtype, f"{what}: dtype {t.dtype}, expected {dtype}"
    assert t.is_cuda == cuda, f"{what}: must be a {'CUDA' if cuda else 'CPU'} tensor"
    assert t.is_contiguous(), f"{what}: must be contiguous"
    assert tuple(t.shape) == tuple(shape), f"{what}: shape {tuple(t.shape)}, expected {tuple(shape)}"


def _stream(stream: Optional[torch.cuda.Stream]):
    s = torch.cuda.current_stream() if stream is None else stream
    return ctypes.c_void_p(s.cuda_stream)


class MoELayer:
    """One combined MoE layer context (`bg_moe_ctx`).  Methods mirror the C entry points."""

    def __init__(self, d: int, f: int, E: int, k: int, max_tokens: int, device: int = 0, gate_fn: int = 0):
        self.lib = load_library()
        self.d, self.f, self.E, self.k, self.max_tokens, self.device = d, f, E, k, max_tokens, device
        self._ctx = ctypes.c_void_p()
        cfg = BgMoeConfig(d, f, E, k, max_tokens, gate_fn, device)
        self._check(self.lib.bg_moe_create(ctypes.byref(cfg), ctypes.byref(self._ctx)), ctx=False)
        self._weights = None

    # ------------------------------------------------------------------ helpers
    def _check(self, rc: int, ctx: bool = True):
        if rc != BG_OK:
            msg = self.lib.bg_moe_strerror(rc).decode()
            if ctx and rc == BG_ERR_CUDA and self._ctx:
                msg += " -- " + self.lib.bg_moe_last_error(self._ctx).decode()
            raise BgMoeError(rc, msg)

    def _dev(self):
        return torch.device("cuda", self.device)

    def close(self):
        if getattr(self, "_ctx", None):
            self.lib.bg_moe_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def launch_count(self) -> int:
        return int(self.lib.bg_moe_launch_count(self._ctx))

    @property
    def workspace_bytes(self) -> int:
        return int(self.lib.bg_moe_workspace_bytes(self._ctx))

    # ------------------------------------------------------------------ C ABI mirrors
    def set_debug(self, static_tile_feed: bool = False, supergroup_token_tiles: int = 0, router_form: int = 0):
        """bg_moe_set_debug: scheduler / router-form switches used by the tests only."""
        self._check(self.lib.bg_moe_set_debug(self._ctx, int(static_tile_feed), int(supergroup_token_tiles),
                                              int(router_form)))

    def set_weights(self, W_r, b_r, W_gate, W_up, W_down, stream=None):
        assert W_r.dtype == torch.float32 and W_r.shape == (self.d, self.E) and W_r.is_contiguous() and W_r.is_cuda
        assert b_r is None or (b_r.dtype == torch.float32 and b_r.shape == (self.E,) and b_r.is_contiguous()
                               and b_r.is_cuda)
        for w, shp in ((W_gate, (self.E, self.d, self.f)), (W_up, (self.E, self.d, self.f)),
                       (W_down, (self.E, self.f, self.d))):
            assert w.dtype == torch.bfloat16 and tuple(w.shape) == shp and w.is_contiguous() and w.is_cuda
        self._weights = (W_r, b_r, W_gate, W_up, W_down)          # keep the borrowed tensors alive
        self._check(self.lib.bg_moe_set_weights(self._ctx, _ptr(W_r), _ptr(b_r), _ptr(W_gate), _ptr(W_up),
                                                _ptr(W_down), _stream(stream)))

    def set_weights_offloaded(self, W_r, b_r, W_gate_host, W_up_host, W_down_host, ring_experts: int, stream=None):
        """bg_moe_set_weights_offloaded: expert weights stay in (pinned) host memory and are streamed through a
        device ring of `ring_experts` expert slots while the grouped GEMMs run."""
        assert W_r.dtype == torch.float32 and W_r.shape == (self.d, self.E) and W_r.is_contiguous() and W_r.is_cuda
        assert b_r is None or (b_r.dtype == torch.float32 and b_r.shape == (self.E,) and b_r.is_contiguous()
                               and b_r.is_cuda)
        for w, shp in ((W_gate_host, (self.E, self.d, self.f)), (W_up_host, (self.E, self.d, self.f)),
                       (W_down_host, (self.E, self.f, self.d))):
            assert w.dtype == torch.bfloat16 and tuple(w.shape) == shp and w.is_contiguous() and not w.is_cuda
            assert w.is_pinned(), "offloaded expert weights must be in pinned host memory"
        self._weights = (W_r, b_r, W_gate_host, W_up_host, W_down_host)
        self._check(self.lib.bg_moe_set_weights_offloaded(self._ctx, _ptr(W_r), _ptr(b_r), _ptr(W_gate_host),
                                                          _ptr(W_up_host), _ptr(W_down_host), int(ring_experts),
                                                          _stream(stream)))

    def set_precision(self, precision: int, stream=None):
        """bg_moe_set_precision: 0 = bf16, 1 = FP8 (e4m3) gate/up GEMM; quantises the resident weights."""
        self._check(self.lib.bg_moe_set_precision(self._ctx, int(precision), _stream(stream)))

    def fp8_views(self, T: int) -> dict:
        """FP8 artefacts of the last fused call, copied out of the library's buffers (codes as uint8)."""
        ptrs = [ctypes.c_void_p() for _ in range(6)]
        self._check(self.lib.bg_moe_debug_fp8_views(self._ctx, *[ctypes.byref(p) for p in ptrs]))
        R = T * self.k
        spec = [("xq_perm", "|u1", (R, self.d)), ("sx_perm", "<f4", (R,)), ("q_gate", "|u1", (self.E, self.f, self.d)),
                ("sw_gate", "<f4", (self.E, self.f)), ("q_up", "|u1", (self.E, self.f, self.d)),
                ("sw_up", "<f4", (self.E, self.f))]
        out = {}
        for p, (name, ts, shape) in zip(ptrs, spec):
            out[name] = torch.as_tensor(_DeviceArray(p.value, shape, ts), device=self._dev()).clone()
        return out

    def fp8_down_views(self, T: int) -> dict:
        """Precision-2 artefacts of the last fused call (H as bf16, codes as uint8)."""
        ptrs = [ctypes.c_void_p() for _ in range(5)]
        self._check(self.lib.bg_moe_debug_fp8_down_views(self._ctx, *[ctypes.byref(p) for p in ptrs]))
        R = T * self.k
        spec = [("H", "<u2", (R, self.f)), ("hq", "|u1", (R, self.f)), ("sh_perm", "<f4", (R,)),
                ("q_down", "|u1", (self.E, self.d, self.f)), ("sw_down", "<f4", (self.E, self.d))]
        out = {}
        for p, (name, ts, shape) in zip(ptrs, spec):
            t = torch.as_tensor(_DeviceArray(p.value, shape, ts), device=self._dev()).clone()
            out[name] = t.view(torch.bfloat16) if name == "H" else t
        return out

    def ffn_views(self, T: int, rows=None) -> dict:
        """bg_moe_debug_ffn_views: H bf16 [T*k, f] and Y bf16 [T*k, d] of the last fused call (expert order), copied out
        of the workspace; rows = (r0, r1) copies only that row range."""
        ptrs = [ctypes.c_void_p() for _ in range(2)]
        self._check(self.lib.bg_moe_debug_ffn_views(self._ctx, *[ctypes.byref(p) for p in ptrs]))
        R = T * self.k
        r0, r1 = (0, R) if rows is None else rows
        out = {}
        for p, (name, width) in zip(ptrs, (("H", self.f), ("Y", self.d))):
            t = torch.as_tensor(_DeviceArray(p.value, (R, width), "<u2"), device=self._dev())
            out[name] = t[r0:r1].clone().view(torch.bfloat16)
        return out

    def set_ring_skip_empty(self, enable: bool = True):
        """bg_moe_set_ring_skip_empty: offloaded weights only -- copy just the experts that received rows (one host
        synchronisation per call)."""
        self._check(self.lib.bg_moe_set_ring_skip_empty(self._ctx, int(bool(enable))))

    @property
    def ring_bytes_per_call(self) -> int:
        return int(self.lib.bg_moe_ring_bytes_per_call(self._ctx))

    def _alloc_stream(self, stream):
        """Outputs are allocated under the stream the call runs on (caching-allocator reuse is stream-ordered)."""
        return torch.cuda.stream(stream) if stream is not None else torch.cuda.stream(torch.cuda.current_stream())

    def route(self, hidden, logits_in=None, want_logits=True, stream=None):
        T = hidden.shape[0] if hidden is not None else logits_in.shape[0]
        if hidden is not None:
            _chk(hidden, torch.bfloat16, (T, self.d), "hidden")
        if logits_in is not None:
            _chk(logits_in, torch.float32, (T, self.E), "logits_in")
        dev = self._dev()
        logits = torch.empty(T, self.E, dtype=torch.float32, device=dev) if want_logits else None
        idx = torch.empty(T, self.k, dtype=torch.int32, device=dev)
        w = torch.empty(T, self.k, dtype=torch.float32, device=dev)
        counts = torch.empty(self.E, dtype=torch.int32, device=dev)
        offsets = torch.empty(self.E + 1, dtype=torch.int32, device=dev)
        self._check(self.lib.bg_moe_route(self._ctx, _ptr(hidden), T, _ptr(logits_in), _ptr(logits), _ptr(idx),
                                          _ptr(w), _ptr(counts), _ptr(offsets), _stream(stream)))
        return dict(logits=logits, idx=idx, w=w, counts=counts, offsets=offsets)

    def permute(self, hidden, topk_idx, offsets, gather=True, stream=None):
        T = topk_idx.shape[0]
        _chk(topk_idx, torch.int32, (T, self.k), "topk_idx")
        _chk(offsets, torch.int32, (self.E + 1,), "offsets")
        if gather:
            _chk(hidden, torch.bfloat16, (T, self.d), "hidden")
        dev = self._dev()
        row_src = torch.empty(T * self.k, dtype=torch.int32, device=dev)
        inv_perm = torch.empty(T * self.k, dtype=torch.int32, device=dev)
        x_perm = torch.empty(T * self.k, self.d, dtype=torch.bfloat16, device=dev) if gather else None
        self._check(self.lib.bg_moe_permute(self._ctx, _ptr(hidden), T, _ptr(topk_idx), _ptr(offsets), _ptr(row_src),
                                            _ptr(inv_perm), _ptr(x_perm), _stream(stream)))
        return dict(row_src=row_src, inv_perm=inv_perm, x_perm=x_perm)

    def expert_ffn(self, x_perm, offsets, T=None, stream=None):
        T = x_perm.shape[0] // self.k if T is None else T
        _chk(x_perm, torch.bfloat16, (T * self.k, self.d), "x_perm")
        _chk(offsets, torch.int32, (self.E + 1,), "offsets")
        y = torch.empty(T * self.k, self.d, dtype=torch.bfloat16, device=self._dev())
        self._check(self.lib.bg_moe_expert_ffn(self._ctx, _ptr(x_perm), _ptr(offsets), T, _ptr(y), _stream(stream)))
        return y

    def unpermute(self, y_perm, inv_perm, topk_w, stream=None):
        T = topk_w.shape[0]
        _chk(y_perm, torch.bfloat16, (T * self.k, self.d), "y_perm")
        _chk(inv_perm, torch.int32, (T * self.k,), "inv_perm")
        _chk(topk_w, torch.float32, (T, self.k), "topk_w")
        out = torch.empty(T, self.d, dtype=torch.bfloat16, device=self._dev())
        self._check(self.lib.bg_moe_unpermute(self._ctx, _ptr(y_perm), _ptr(inv_perm), _ptr(topk_w), T, _ptr(out),
                                              _stream(stream)))
        return out

    def combined_forward(self, hidden, out=None, stream=None):
        T = hidden.shape[0]
        _chk(hidden, torch.bfloat16, (T, self.d), "hidden")
        if out is None:
            with self._alloc_stream(stream):
                out = torch.empty(T, self.d, dtype=torch.bfloat16, device=self._dev())
        else:
            _chk(out, torch.bfloat16, (T, self.d), "out")
        self._check(self.lib.bg_moe_combined_forward(self._ctx, _ptr(hidden), T, _ptr(out), _stream(stream)))
        return out

    def combined_forward_host(self, hidden_host, out_host=None, stream=None):
        """hidden_host / out_host: CPU (ideally pinned) bf16 tensors.  The copies run on streams the context owns;
        `stream` waits for the download.  Keep hidden_host alive and unmodified until host_input_sync() (or a
        synchronize on `stream`) -- the upload is asynchronous and torch's host allocator does not know of it."""
        T = hidden_host.shape[0]
        _chk(hidden_host, torch.bfloat16, (T, self.d), "hidden_host", cuda=False)
        if out_host is None:
            out_host = torch.empty(T, self.d, dtype=torch.bfloat16).pin_memory()
        else:
            _chk(out_host, torch.bfloat16, (T, self.d), "out_host", cuda=False)
        self._check(self.lib.bg_moe_combined_forward_host(self._ctx, _ptr(hidden_host), T, _ptr(out_host),
                                                          _stream(stream)))
        return out_host

    def host_input_sync(self):
        """bg_moe_host_input_sync: blocks until the last combined_forward_host's upload has finished."""
        self._check(self.lib.bg_moe_host_input_sync(self._ctx))

    def build_segments(self, hidden_segments, out_segments):
        """The bg_moe_segment array for a list of per-coroutine tensors (marshalling only; reusable)."""
        n = len(hidden_segments)
        arr = (BgMoeSegment * max(n, 1))()
        for i, (h, o) in enumerate(zip(hidden_segments, out_segments)):
            assert h.dtype == torch.bfloat16 and h.is_cuda and h.is_contiguous() and h.shape[1] == self.d
            assert o.dtype == torch.bfloat16 and o.is_cuda and o.is_contiguous() and o.shape == h.shape
            arr[i].hidden = h.data_ptr() if h.shape[0] else None
            arr[i].out = o.data_ptr() if o.shape[0] else None
            arr[i].n_tokens = h.shape[0]
        return arr, n

    def combined_forward_segments(self, hidden_segments, out_segments=None, stream=None, table=None):
        """bg_moe_combined_forward_segments: zero-copy COMBINE.  hidden_segments: list of CUDA bf16 tensors
        [n_s, d] (the yielded coroutines' buffers; n_s may be 0); returns the list of per-segment outputs.
        `table` = a (array, n) pair from build_segments for the same tensors skips the marshalling."""
        if out_segments is None:
            out_segments = [torch.empty_like(h) for h in hidden_segments]
        arr, n = table if table is not None else self.build_segments(hidden_segments, out_segments)
        self.lib.bg_moe_combined_forward_segments.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32,
                                                              ctypes.c_void_p]
        self._check(self.lib.bg_moe_combined_forward_segments(self._ctx, ctypes.cast(arr, ctypes.c_void_p),
                                                              ctypes.c_int32(n), _stream(stream)))
        return out_segments

    STAGES = ("router", "gather", "gateup_swiglu", "down", "unpermute")

    def profile_enable(self, on: bool = True):
        self._check(self.lib.bg_moe_profile_enable(self._ctx, int(on)))

    def profile_read(self) -> dict:
        """Per-kernel milliseconds of the last fused call made while profiling was enabled."""
        buf = (ctypes.c_float * len(self.STAGES))()
        self._check(self.lib.bg_moe_profile_read(self._ctx, buf))
        return dict(zip(self.STAGES, [float(x) for x in buf]))

    def debug_views(self, T: int) -> dict:
        """Routing artefacts of the last fused call, as torch tensors copied out of the workspace."""
        ptrs = [ctypes.c_void_p() for _ in range(7)]
        self._check(self.lib.bg_moe_debug_views(self._ctx, *[ctypes.byref(p) for p in ptrs]))
        R = T * self.k
        spec = [("logits", torch.float32, (T, self.E)), ("idx", torch.int32, (T, self.k)),
                ("w", torch.float32, (T, self.k)), ("counts", torch.int32, (self.E,)),
                ("offsets", torch.int32, (self.E + 1,)), ("row_src", torch.int32, (R,)),
                ("inv_perm", torch.int32, (R,))]
        out = {}
        typestr = {torch.float32: "<f4", torch.int32: "<i4"}
        for p, (name, dt, shape) in zip(ptrs, spec):
            n = 1
            for s in shape:
                n *= s
            if n == 0:
                out[name] = torch.empty(shape, dtype=dt, device=self._dev())
                continue
            view = _DeviceArray(p.value, shape, typestr[dt])
            out[name] = torch.as_tensor(view, device=self._dev()).clone()
        return out


class _DeviceArray:
    """Zero-copy view of library-owned device memory through `__cuda_array_interface__`."""

    def __init__(self, ptr: int, shape, typestr: str):
        self.__cuda_array_interface__ = {"shape": tuple(shape), "typestr": typestr, "data": (ptr, False),
                                         "version": 2, "strides": None}


# ---------------------------------------------------------------------- planning (host only)
class BgMoeFit(ctypes.Structure):
    _fields_ = [(n, ctypes.c_double) for n in ("t_floor_ms", "t0_ms", "ms_per_token", "ridge_tokens", "rms_rel_err")]

    def as_dict(self) -> dict:
        return {n: float(getattr(self, n)) for n, _ in self._fields_}


def _plan_check(lib, rc: int):
    if rc != BG_OK:
        raise BgMoeError(rc, lib.bg_moe_strerror(rc).decode())


def fit_roofline(tokens, ms) -> BgMoeFit:
    """bg_moe_fit_roofline: module-level roofline t(T) = max(t_floor, t0 + s T) fitted to measured points."""
    lib = load_library()
    n = len(tokens)
    tok = (ctypes.c_int32 * n)(*[int(t) for t in tokens])
    y = (ctypes.c_double * n)(*[float(v) for v in ms])
    fit = BgMoeFit()
    lib.bg_moe_fit_roofline.restype = ctypes.c_int
    _plan_check(lib, lib.bg_moe_fit_roofline(tok, y, ctypes.c_int32(n), ctypes.byref(fit)))
    return fit


def workspace_bytes_for(d: int, f: int, E: int, k: int, tokens: int) -> int:
    """bg_moe_workspace_bytes_for: device workspace of a context with max_tokens = tokens."""
    lib = load_library()
    cfg = BgMoeConfig(d, f, E, k, 0, 0, 0)
    out = ctypes.c_int64()
    _plan_check(lib, lib.bg_moe_workspace_bytes_for(ctypes.byref(cfg), ctypes.c_int32(tokens), ctypes.byref(out)))
    return int(out.value)


def choose_tokens(d: int, f: int, E: int, k: int, fit: BgMoeFit, target_util: float, memory_budget_bytes: int,
                  granularity: int = 1):
    """bg_moe_choose_tokens: (B_moe, reached) -- see include/bg_moe.h."""
    lib = load_library()
    cfg = BgMoeConfig(d, f, E, k, 0, 0, 0)
    tok, reached = ctypes.c_int32(), ctypes.c_int32()
    _plan_check(lib, lib.bg_moe_choose_tokens(ctypes.byref(cfg), ctypes.byref(fit), ctypes.c_double(target_util),
                                              ctypes.c_int64(memory_budget_bytes), ctypes.c_int32(granularity),
                                              ctypes.byref(tok), ctypes.byref(reached)))
    return int(tok.value), bool(reached.value)


# ---------------------------------------------------------------------- routing without allocation
NOALLOC_MAX_TOKENS = 16384   # BG_MOE_NOALLOC_MAX_TOKENS of include/bg_moe.h


def route_logits_noalloc(logits, k: int, topk_idx, topk_w, counts, offsets, stream=None) -> None:
    """bg_moe_route_logits_noalloc: top-k + gates + histogram + exclusive scan from fp32 logits [T,E], for callers
    that may not allocate device memory (a runtime that owns all of HBM through its own pools, or a latency-critical
    section where cudaMalloc's device-wide serialisation is banned).  No context and no workspace: the library's
    scratch is a fixed array in its own image, which is why T <= NOALLOC_MAX_TOKENS, and why calls that may run
    concurrently on one GPU must be ordered by the caller (they share that array).  In keeping with that, this
    wrapper allocates nothing either: ALL four outputs are passed in (topk_idx int32 [T,k], topk_w fp32 [T,k],
    counts int32 [E], offsets int32 [E+1]) and are overwritten.  Runs on the device of `logits`, asynchronously on
    `stream` (default: torch's current stream).  Make the first call on a device during set-up, outside any
    stream capture."""
    lib = load_library()
    assert isinstance(logits, torch.Tensor) and logits.dim() == 2, "logits: [T,E] tensor expected"
    T, E = logits.shape
    _chk(logits, torch.float32, (T, E), "logits")
    _chk(topk_idx, torch.int32, (T, k), "topk_idx")
    _chk(topk_w, torch.float32, (T, k), "topk_w")
    _chk(counts, torch.int32, (E,), "counts")
    _chk(offsets, torch.int32, (E + 1,), "offsets")
    for t in (topk_idx, topk_w, counts, offsets):
        assert t.device == logits.device, "all tensors must live on the device of `logits`"
    with torch.cuda.device(logits.device):
        rc = lib.bg_moe_route_logits_noalloc(_ptr(logits), T, E, k, _ptr(topk_idx), _ptr(topk_w), _ptr(counts),
                                             _ptr(offsets), _stream(stream))
        if rc != BG_OK:
            raise BgMoeError(rc, lib.bg_moe_strerror(rc).decode() + " -- " + lib.bg_moe_noalloc_last_error().decode())
