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
