"""CPU oracle for the combined MoE layer -- TEST INFRASTRUCTURE, not a product path.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this package.  It shares no code with
`paper_2606_21712_b200/` and imports nothing from it.  The arithmetic lives in
`bgo_oracle.cpp` (C++17, fp64, OpenMP over independent rows only); this file is the
`ctypes` marshalling around it.  See the header of `bgo_oracle.cpp` for the definition
it follows (PAPER.md:244 `h_out <- MoE(h_combined, l)`; BASELINE.json `north_star`) and
for what pins it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bgo_oracle.cpp")
_LIB = os.path.join(_HERE, "libbgo_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle (g++ -O3 -march=native -fopenmp).  Building is not using."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["g++", "-O3", "-march=native", "-std=c++17", "-fopenmp", "-fPIC", "-shared",
               "-ffp-contract=off", "-o", _LIB + ".tmp", _SRC]
        subprocess.run(cmd, check=True)
        os.replace(_LIB + ".tmp", _LIB)
    return _LIB


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB)
    return _lib


def num_threads() -> int:
    return int(lib().bgo_num_threads())


def _u16(t) -> np.ndarray:
    """torch bf16 tensor (CPU) or uint16/int16 ndarray -> contiguous uint16 ndarray (bit view)."""
    if isinstance(t, np.ndarray):
        assert t.dtype in (np.uint16, np.int16)
        return np.ascontiguousarray(t).view(np.uint16)
    import torch
    assert t.dtype == torch.bfloat16 and t.device.type == "cpu"
    return t.contiguous().view(torch.int16).numpy().view(np.uint16)


def _f32(t) -> Optional[np.ndarray]:
    if t is None:
        return None
    if not isinstance(t, np.ndarray):
        t = t.detach().cpu().numpy()
    return np.ascontiguousarray(t, dtype=np.float32)


def _i32(t) -> np.ndarray:
    if not isinstance(t, np.ndarray):
        t = t.detach().cpu().numpy()
    return np.ascontiguousarray(t, dtype=np.int32)


def _p(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


def _check(rc: int, what: str):
    if rc != 0:
        raise ValueError(f"oracle {what} rejected its arguments (rc={rc})")


def router_logits(hidden, W_r, b_r=None) -> np.ndarray:
    h, W = _u16(hidden), _f32(W_r)
    T, d = h.shape
    E = W.shape[1]
    assert W.shape[0] == d
    b = _f32(b_r)
    out = np.empty((T, E), np.float32)
    _check(lib().bgo_router_logits(_p(h), _p(W), _p(b), T, d, E, _p(out)), "router_logits")
    return out


def topk_gate(logits, k: int):
    L = _f32(logits)
    T, E = L.shape
    idx = np.empty((T, k), np.int32)
    w = np.empty((T, k), np.float32)
    _check(lib().bgo_topk_gate(_p(L), T, E, k, _p(idx), _p(w)), "topk_gate")
    return idx, w


def hist_scan_perm(idx, E: int):
    idx = _i32(idx)
    T, k = idx.shape
    counts = np.empty(E, np.int32)
    offsets = np.empty(E + 1, np.int32)
    row_src = np.empty(T * k, np.int32)
    inv_perm = np.empty(T * k, np.int32)
    _check(lib().bgo_hist_scan_perm(_p(idx), T, k, E, _p(counts), _p(offsets), _p(row_src), _p(inv_perm)),
           "hist_scan_perm")
    return counts, offsets, row_src, inv_perm


def gather(hidden, row_src, k: int) -> np.ndarray:
    h, rs = _u16(hidden), _i32(row_src)
    T, d = h.shape
    assert rs.shape[0] == T * k
    x = np.empty((T * k, d), np.uint16)
    _check(lib().bgo_gather(_p(h), _p(rs), T, k, d, _p(x)), "gather")
    return x


def expert_ffn(x_perm, offsets, W_gate, W_up, W_down) -> np.ndarray:
    x, off = _u16(x_perm), _i32(offsets)
    Wg, Wu, Wd = _u16(W_gate), _u16(W_up), _u16(W_down)
    R, d = x.shape
    E, d2, f = Wg.shape
    assert d2 == d and Wu.shape == (E, d, f) and Wd.shape == (E, f, d) and off.shape[0] == E + 1
    y = np.empty((R, d), np.float64)
    _check(lib().bgo_expert_ffn(_p(x), _p(off), _p(Wg), _p(Wu), _p(Wd), R, d, f, E, _p(y)), "expert_ffn")
    return y


def unpermute(y_perm, inv_perm, w) -> np.ndarray:
    y = np.ascontiguousarray(y_perm, dtype=np.float64)
    ip, w = _i32(inv_perm), _f32(w)
    T, k = w.shape
    d = y.shape[1]
    assert ip.shape[0] == T * k and y.shape[0] == T * k
    out = np.empty((T, d), np.float64)
    _check(lib().bgo_unpermute(_p(y), _p(ip), _p(w), T, k, d, _p(out)), "unpermute")
    return out


def forward_batched(hidden, W_r, b_r, W_gate, W_up, W_down, k: int, logits_in=None) -> dict:
    h, W = _u16(hidden), _f32(W_r)
    Wg, Wu, Wd = _u16(W_gate), _u16(W_up), _u16(W_down)
    T, d = h.shape
    E, _, f = Wg.shape
    b, Lin = _f32(b_r), _f32(logits_in)
    res = dict(logits=np.empty((T, E), np.float32), idx=np.empty((T, k), np.int32),
               w=np.empty((T, k), np.float32), counts=np.empty(E, np.int32),
               offsets=np.empty(E + 1, np.int32), row_src=np.empty(T * k, np.int32),
               inv_perm=np.empty(T * k, np.int32), out=np.empty((T, d), np.float64))
    _check(lib().bgo_forward_batched(_p(h), _p(W), _p(b), _p(Wg), _p(Wu), _p(Wd), T, d, E, k, f, _p(Lin),
                                     _p(res["logits"]), _p(res["idx"]), _p(res["w"]), _p(res["counts"]),
                                     _p(res["offsets"]), _p(res["row_src"]), _p(res["inv_perm"]),
                                     _p(res["out"])), "forward_batched")
    return res


def forward_tokens(hidden, W_r, b_r, W_gate, W_up, W_down, k: int, tokens, logits_in=None) -> np.ndarray:
    """Per-token brute force (the plain definition) for the listed tokens -> fp64 [n_tok, d]."""
    h, W = _u16(hidden), _f32(W_r)
    Wg, Wu, Wd = _u16(W_gate), _u16(W_up), _u16(W_down)
    T, d = h.shape
    E, _, f = Wg.shape
    b, Lin = _f32(b_r), _f32(logits_in)
    tok = _i32(np.asarray(tokens))
    out = np.empty((tok.shape[0], d), np.float64)
    _check(lib().bgo_forward_tokens(_p(h), _p(W), _p(b), _p(Wg), _p(Wu), _p(Wd), T, d, E, k, f, _p(tok),
                                    tok.shape[0], _p(Lin), _p(out)), "forward_tokens")
    return out
