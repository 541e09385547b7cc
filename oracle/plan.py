"""CPU oracle for the planning helpers (module-level roofline fit, B_moe choice) -- TEST INFRASTRUCTURE.

Plain numpy / pure-Python restatement of what include/bg_moe.h defines for bg_moe_fit_roofline and
bg_moe_choose_tokens, following PAPER.md:261 (§5.1: "a module-level roofline model enables static planning
for batch accumulation ... select the largest feasible module batch size that remains within memory
constraints") and PAPER.md:353 (§5.4: the module is profiled "over multiple batch sizes" and the results
are fitted "to roofline-style models that predict runtime as a function of batch size").  The paper
gives no formula; the reading taken (R6) is the two-segment roofline
    t(T) = max(t_floor, t0 + s*T),      u(T) = min(1, s*T / t(T)).
Pinned in tests/test_plan.py by exact synthetic data (parameters recovered), by the closed forms
T_flat = ceil(u*t_floor/s), T_line = ceil(u*t0/((1-u)*s)), and by monotonicity.  Shares no code with the
library; only tests import it.

workspace_bytes() is the memory side: the sum of the slabs DESIGN.md §4 lists for the context's workspace, each
rounded up to 1 KB, written out from that list (it is the oracle's own arithmetic, not a call into the library).
Pinned in tests/test_plan.py by a hand-computed small case, by its exact linear growth per 128 tokens and by what
the slabs must at least hold.
"""
from __future__ import annotations

import math

import numpy as np


def model_ms(fit: dict, T: float) -> float:
    return max(fit["t_floor_ms"], fit["t0_ms"] + fit["ms_per_token"] * T)


def fit_roofline(tokens, ms) -> dict:
    """Every split 'first j points flat, the rest on a line' (1 <= j <= n-2); flat = mean, line = numpy's
    least-squares polynomial of degree 1; smallest sum of squared relative errors wins (lowest j on ties)."""
    x = np.asarray(tokens, dtype=np.float64)
    y = np.asarray(ms, dtype=np.float64)
    n = len(x)
    assert n >= 3 and np.all(np.diff(x) > 0) and np.all(y > 0)
    best, best_fit = math.inf, None
    for j in range(1, n - 1):
        flat = float(np.mean(y[:j]))
        slope, icpt = np.polyfit(x[j:], y[j:], 1)
        if not slope > 0:
            continue
        fit = {"t_floor_ms": flat, "t0_ms": float(icpt), "ms_per_token": float(slope),
               "ridge_tokens": float((flat - icpt) / slope)}
        rel = np.array([(model_ms(fit, xi) - yi) / yi for xi, yi in zip(x, y)])
        sse = float(np.sum(rel * rel))
        fit["rms_rel_err"] = math.sqrt(sse / n)
        if sse < best:
            best, best_fit = sse, fit
    if best_fit is None:
        raise ValueError("no split with a positive slope")
    return best_fit


def utilisation(fit: dict, T: float) -> float:
    return min(1.0, fit["ms_per_token"] * T / model_ms(fit, T))


def choose_tokens(fit: dict, target_util: float, memory_budget_bytes: int, granularity: int, bytes_for, t_limit: int):
    """Linear scan over the multiples of `granularity` up to t_limit: the largest one whose workspace
    (bytes_for(T), a callable) fits, and the first one whose utilisation reaches the target."""
    t_mem = 0
    T = granularity
    while T <= t_limit and bytes_for(T) <= memory_budget_bytes:
        t_mem = T
        T += granularity
    if t_mem == 0:
        raise MemoryError("not even one granule fits")
    T = granularity
    while T <= t_mem:
        if utilisation(fit, T) >= target_util:
            return T, True
        T += granularity
    return t_mem, False


def _kb(n: int) -> int:
    return -(-n // 1024) * 1024


def workspace_bytes(d: int, f: int, E: int, k: int, tokens: int) -> int:
    """Device workspace of a context with max_tokens = tokens ("Library workspace"): every slab is
    rounded up to a multiple of 1 KB.  T = max(tokens, 1), R = T k, tiles = ceil(T / 128)."""
    T = max(int(tokens), 1)
    R = T * k
    tiles = -(-T // 128)
    E16 = -(-E // 16) * 16
    slabs = [
        4 * T * E,                   # logits [T,E] f32
        4 * R, 4 * R,                # topk_idx, topk_w [T,k]
        2 * 3 * d * E16,             # W_r pieces [3][d][ceil16(E)] bf16
        4 * E, 4 * (E + 1),          # counts [E], offsets [E+1]
        4 * tiles * E,               # per-tile histograms
        4 * tiles * E,               # per-tile bases
        4 * R,                       # tile-local ranks
        4 * R, 4 * R,                # row_src, inv_perm
        4 * R,                       # w_perm f32
        2 * R * d,                   # x_perm bf16
        2 * R * f,                   # H bf16
        2 * R * d,                   # Y bf16
        2 * 2 * T * d,               # host entry point: two [T,d] bf16 staging slots in ...
        2 * 2 * T * d,               # ... and two out
        8 * T + 8 * T + 4 * (T + 1), # segment table: hidden pointers, out pointers, start offsets
        64,                          # counters
    ]
    return sum(_kb(b) for b in slabs)
