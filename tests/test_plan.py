"""Planning helpers (bg_moe_fit_roofline, bg_moe_workspace_bytes_for, bg_moe_choose_tokens): host-only
entry points of the C ABI, checked on CPU against oracle/plan.py and against closed forms."""
import math

import numpy as np
import pytest

import paper_2606_21712_b200 as pk
from oracle import plan as oplan

C3 = dict(d=2048, f=768, E=128, k=8)


def synth(t_floor, t0, s, tokens):
    return [max(t_floor, t0 + s * T) for T in tokens]


# ---- oracle pins (closed forms; nothing here calls the library)
def test_oracle_fit_recovers_exact_piecewise_data():
    tokens = [64, 256, 1024, 4096, 16384, 32768]
    fit = oplan.fit_roofline(tokens, synth(0.25, 0.05, 7.5e-5, tokens))
    assert abs(fit["t_floor_ms"] - 0.25) < 1e-12 and abs(fit["t0_ms"] - 0.05) < 1e-9
    assert abs(fit["ms_per_token"] - 7.5e-5) < 1e-12 and fit["rms_rel_err"] < 1e-9
    assert abs(fit["ridge_tokens"] - (0.25 - 0.05) / 7.5e-5) < 1e-3


def test_oracle_choice_matches_closed_forms():
    fit = {"t_floor_ms": 0.25, "t0_ms": 0.05, "ms_per_token": 7.5e-5}
    big = 1 << 60
    # target reached on the flat part: s T / t_floor >= u  <=>  T >= u t_floor / s
    T, ok = oplan.choose_tokens(fit, 0.5, big, 1, lambda T: 0, 100000)
    assert ok and T == math.ceil(0.5 * 0.25 / 7.5e-5)
    # target reached on the line: s T / (t0 + s T) >= u  <=>  T >= u t0 / ((1-u) s)
    T, ok = oplan.choose_tokens(fit, 0.95, big, 1, lambda T: 0, 100000)
    assert ok and T == math.ceil(0.95 * 0.05 / (0.05 * 7.5e-5))
    # memory cap binds: bytes_for(T) = 1000 T, budget 5 MB -> 5000 tokens, utilisation target not reached
    T, ok = oplan.choose_tokens(fit, 0.95, 5_000_000, 8, lambda T: 1000 * T, 100000)
    assert not ok and T == 5000
    us = [oplan.utilisation(fit, T) for T in range(1, 50000, 97)]
    assert all(b >= a for a, b in zip(us, us[1:])) and us[-1] < 1.0


# ---- the library against the oracle
@pytest.mark.parametrize("seed", [0, 1, 2, 3])
def test_fit_matches_oracle_on_noisy_data(seed):
    rng = np.random.default_rng(seed)
    tokens = [64, 256, 1024, 4096, 8192, 16384, 32768]
    ms = [v * (1 + 0.03 * rng.standard_normal()) for v in synth(0.23, 0.06, 7.4e-5, tokens)]
    got = pk.fit_roofline(tokens, ms).as_dict()
    ref = oplan.fit_roofline(tokens, ms)
    for key in ref:
        assert abs(got[key] - ref[key]) <= 1e-9 * max(1.0, abs(ref[key])), (key, got[key], ref[key])


def test_fit_of_the_measured_c3_sweep():
    """The round-1 C3 sweep: the fit must put the ridge between T=1024 and T=4096 and
    reproduce every point within 10 %."""
    tokens = [64, 256, 1024, 4096, 16384, 32768]
    ms = [0.226, 0.236, 0.255, 0.414, 1.272, 2.477]
    fit = pk.fit_roofline(tokens, ms).as_dict()
    assert 1024 < fit["ridge_tokens"] < 4096 and fit["rms_rel_err"] < 0.10
    ref = oplan.fit_roofline(tokens, ms)
    assert abs(fit["ms_per_token"] - ref["ms_per_token"]) < 1e-12


def test_fit_rejects_bad_input():
    with pytest.raises(pk.BgMoeError):
        pk.fit_roofline([1, 2], [1.0, 2.0])                      # n < 3
    with pytest.raises(pk.BgMoeError):
        pk.fit_roofline([1, 3, 2], [1.0, 2.0, 3.0])              # not increasing
    with pytest.raises(pk.BgMoeError):
        pk.fit_roofline([1, 2, 3], [3.0, 2.0, 1.0])              # no positive slope


def test_workspace_bytes_monotone_and_dominated_by_activations():
    prev = 0
    for T in (0, 1, 64, 1000, 4096, 32768):
        b = pk.workspace_bytes_for(tokens=T, **C3)
        assert b >= prev
        prev = b
    R = 32768 * C3["k"]
    # x_perm + Y + H, plus the host entry point's two staging slots each way (4 x [T,d] bf16)
    act = R * (2 * C3["d"] + C3["f"]) * 2 + 4 * 32768 * C3["d"] * 2
    assert act <= prev <= 1.1 * act + (64 << 20)


@pytest.mark.parametrize("target,budget,gran", [(0.5, 8 << 30, 1), (0.8, 8 << 30, 64), (0.9, 1 << 30, 128),
                                                (0.95, 300 << 20, 16), (0.3, 64 << 20, 8)])
def test_choice_matches_oracle(target, budget, gran):
    tokens = [64, 256, 1024, 4096, 16384, 32768]
    fit = pk.fit_roofline(tokens, [0.226, 0.236, 0.255, 0.414, 1.272, 2.477])
    ref = oplan.choose_tokens(fit.as_dict(), target, budget, gran, lambda T: pk.workspace_bytes_for(tokens=T, **C3),
                              t_limit=200000)
    got = pk.choose_tokens(fit=fit, target_util=target, memory_budget_bytes=budget, granularity=gran, **C3)
    assert got == ref


def test_choice_errors():
    fit = pk.fit_roofline([64, 1024, 16384, 32768], [0.2, 0.25, 1.2, 2.4])
    with pytest.raises(pk.BgMoeError) as e:
        pk.choose_tokens(fit=fit, target_util=0.5, memory_budget_bytes=1024, granularity=64, **C3)
    assert e.value.status == pk.BG_ERR_NOMEM
    with pytest.raises(pk.BgMoeError):
        pk.choose_tokens(fit=fit, target_util=1.5, memory_budget_bytes=1 << 30, granularity=64, **C3)
