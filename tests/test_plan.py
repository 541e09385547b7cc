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


def test_oracle_workspace_closed_form_pins():
    """oracle/plan.py:workspace_bytes against arithmetic done by hand (nothing here calls the library)."""
    # d = f = 64, E = 4, k = 2, T = 1: every slab but four fits its first KB.  19 slabs; pieces = 2*3*64*16 = 6144 B
    # (6 KB); x_perm = Y = 2*2*64 = 256 B; H = 256 B; so 18 slabs of 1 KB + 6 KB
    assert oplan.workspace_bytes(64, 64, 4, 2, 1) == 18 * 1024 + 6 * 1024
    assert oplan.workspace_bytes(64, 64, 4, 2, 0) == oplan.workspace_bytes(64, 64, 4, 2, 1)     # T = 0 sized as T = 1
    # once every token-proportional slab is a whole number of KB per 128 tokens, growth is exactly linear:
    # per token: logits 4E + six 4-byte [R] tables (idx, w, rank, row_src, inv_perm, w_perm) 24k + (x, Y) 4kd + H 2kf + staging 8d + segment table 20
    # + tiles 8E/128
    d, f, E, k = 2048, 768, 128, 8
    per_token = 4 * E + 24 * k + 4 * k * d + 2 * k * f + 8 * d + 20 + 8 * E // 128
    a, b = oplan.workspace_bytes(d, f, E, k, 128 * 1024), oplan.workspace_bytes(d, f, E, k, 128 * 2048)
    assert b - a == per_token * 128 * 1024
    # lower bound: the three activation slabs alone
    assert oplan.workspace_bytes(d, f, E, k, 32768) > 32768 * k * (4 * d + 2 * f)


# ---- the library against the oracle
@pytest.mark.parametrize("d,f,E,k", [(2048, 768, 128, 8), (4096, 14336, 8, 2), (7168, 2048, 256, 8), (512, 1024, 8, 2),
                                     (192, 200, 5, 5), (64, 64, 1, 1), (4096, 1408, 64, 6)])
def test_workspace_bytes_match_the_oracle_closed_form(d, f, E, k):
    for T in (0, 1, 7, 64, 127, 128, 129, 1000, 4096, 16384, 32768, 100001):
        assert pk.workspace_bytes_for(d=d, f=f, E=E, k=k, tokens=T) == oplan.workspace_bytes(d, f, E, k, T), T


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
    # both sides of the choice come from the oracle: its own fit of the points and its own workspace closed form
    ref = oplan.choose_tokens(oplan.fit_roofline(tokens, [0.226, 0.236, 0.255, 0.414, 1.272, 2.477]), target, budget, gran,
                              lambda T: oplan.workspace_bytes(tokens=T, **C3), t_limit=200000)
    got = pk.choose_tokens(fit=fit, target_util=target, memory_budget_bytes=budget, granularity=gran, **C3)
    assert got == ref


def test_choice_errors():
    fit = pk.fit_roofline([64, 1024, 16384, 32768], [0.2, 0.25, 1.2, 2.4])
    with pytest.raises(pk.BgMoeError) as e:
        pk.choose_tokens(fit=fit, target_util=0.5, memory_budget_bytes=1024, granularity=64, **C3)
    assert e.value.status == pk.BG_ERR_NOMEM
    with pytest.raises(pk.BgMoeError):
        pk.choose_tokens(fit=fit, target_util=1.5, memory_budget_bytes=1 << 30, granularity=64, **C3)


@pytest.mark.gpu
def test_plan_on_a_sweep_measured_on_this_gpu():
    """(f)-3 on the GPU box: time the fused chain over the C3 combine-size sweep bench.py measures (CUDA events on the
    launching stream), fit the module-level roofline with the library and with the oracle on the SAME measured
    points, and choose B_moe both ways; the workspace the planner predicts is what a context really allocates."""
    import torch
    import workloads as wl
    tokens = [64, 256, 1024, 4096, 8192, 16384]
    base = wl.C3
    lay = wl.make_layer(base.with_T(max(tokens)), "cuda")
    layer = pk.MoELayer(base.d, base.f, base.E, base.k, max(tokens))
    layer.set_weights(lay["W_r"], lay["b_r"], lay["W_gate"], lay["W_up"], lay["W_down"])
    assert layer.workspace_bytes == oplan.workspace_bytes(base.d, base.f, base.E, base.k, max(tokens))
    ms = []
    st = torch.cuda.current_stream()
    for T in tokens:
        h = lay["hidden"][:T].contiguous()
        out = torch.empty_like(h)
        for _ in range(3):
            layer.combined_forward(h, out)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(st)
        for _ in range(10):
            layer.combined_forward(h, out)
        e1.record(st)
        torch.cuda.synchronize()
        ms.append(e0.elapsed_time(e1) / 10)
    got = pk.fit_roofline(tokens, ms)
    ref = oplan.fit_roofline(tokens, ms)
    for key in ref:
        assert abs(got.as_dict()[key] - ref[key]) <= 1e-9 * max(1.0, abs(ref[key])), (key, got.as_dict()[key], ref[key])
    assert all(b > a * 0.9 for a, b in zip(ms, ms[1:])), ms                 # a sweep, not noise
    assert ms[-1] > 2 * ms[0] and got.as_dict()["ms_per_token"] > 0           # compute-bound tail is visible
    for target, budget, gran in [(0.5, 8 << 30, 64), (0.8, 8 << 30, 64), (0.9, 1 << 30, 128), (0.95, 300 << 20, 16)]:
        want = oplan.choose_tokens(ref, target, budget, gran, lambda T: oplan.workspace_bytes(tokens=T, **C3), t_limit=400000)
        assert pk.choose_tokens(fit=got, target_util=target, memory_budget_bytes=budget, granularity=gran, **C3) == want
    print(f"[plan] measured sweep {dict(zip(tokens, [round(m, 4) for m in ms]))} -> {got.as_dict()}")
