"""Pins for the CPU oracle (`oracle/`), CPU only.

Every check compares the oracle with something OTHER than itself: closed forms, numpy
library routines (fp64 matmul, stable argsort), pure-Python brute force on tiny inputs, or
invariants stated in BASELINE.json `north_star` / SURVEY.md §8(c).  A dropped term, a wrong
sign or index, a transposed operand or a swapped gate/up in the oracle fails at least one.
"""
import math
import os

import numpy as np
import pytest
import torch

import oracle
import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def bf16_to_f64(t: torch.Tensor) -> np.ndarray:
    return t.to(torch.float64).numpy()


def small_layer(**kw):
    return wl.make_layer(wl.small_config(**kw))


# ----------------------------------------------------------------------------- paper fixtures
def _read_kv(name):
    kv = {}
    for line in open(os.path.join(GOLD, name)):
        if line.startswith("#") or not line.strip():
            continue
        a, b = line.split()
        kv[a] = float(b)
    return kv


def test_paper_hidden_state_is_two_bytes_per_element():
    """~7 MB for 512 x 7168-dim hidden states => 2-byte elements (bf16)."""
    kv = _read_kv("paper_hidden_state_bytes.txt")
    h = wl.make_hidden(wl.MoEConfig("p", 9, T=int(kv["sequences"]), d=int(kv["dim"]), E=2, k=1, f=8))
    nbytes = h.numel() * h.element_size()
    assert h.dtype == torch.bfloat16 and h.is_contiguous()
    assert abs(nbytes / 2**20 - kv["approx_megabytes"]) < 0.5      # 7.0 MiB; 4-byte would be 14
    assert wl.C4.d == int(kv["dim"])


def test_paper_saturation_tokens_is_in_sweep():
    kv = _read_kv("paper_saturation_tokens.txt")
    assert int(kv["tokens_at_moe_gate"]) in wl.C3_SWEEP_T
    assert wl.C5.T == int(kv["tokens_at_moe_gate"])
    assert sum(wl.segment_lengths(wl.C5)) == wl.C5.T


# ----------------------------------------------------------------------------- a1 router logits
def test_router_one_hot_and_zero_rows_closed_form():
    cfg = wl.small_config(T=5, d=32, E=7)
    W_r, _ = wl.make_router(cfg)
    b = torch.linspace(-1, 1, cfg.E)
    h = torch.zeros(cfg.T, cfg.d, dtype=torch.bfloat16)
    h[1, 3] = 1.0
    h[2, 31] = 1.0
    h[3, 0] = -2.0
    L = oracle.router_logits(h, W_r, None)
    Wn = W_r.numpy()
    assert np.array_equal(L[0], np.zeros(cfg.E, np.float32))
    assert np.array_equal(L[1], Wn[3])            # one-hot row j => W_r[j,:] exactly
    assert np.array_equal(L[2], Wn[31])
    assert np.array_equal(L[3], -2.0 * Wn[0])
    Lb = oracle.router_logits(h, W_r, b)
    assert np.array_equal(Lb[0], b.numpy())       # zero row => bias
    assert np.allclose(Lb[1], Wn[3].astype(np.float64) + b.numpy(), rtol=0, atol=1e-7)


def test_router_matches_numpy_fp64_matmul_and_is_not_transposed():
    cfg = wl.small_config(T=33, d=40, E=9)
    h = wl.make_hidden(cfg)
    W_r, _ = wl.make_router(cfg)
    L = oracle.router_logits(h, W_r)
    ref = bf16_to_f64(h) @ W_r.to(torch.float64).numpy()
    assert np.allclose(L, ref, rtol=0, atol=2e-6)
    assert np.array_equal(L, ref.astype(np.float32)) or np.max(np.abs(L - ref)) < 2e-7
    # linearity: L(2h) = 2 L(h) exactly (power-of-two scale commutes with every rounding)
    L2 = oracle.router_logits((h.float() * 2).to(torch.bfloat16), W_r)
    assert np.array_equal(L2, 2 * L)


# ----------------------------------------------------------------------------- a2 top-k + gates
def brute_topk(L: np.ndarray, k: int) -> np.ndarray:
    """Full stable sort of (-L, e) per token (numpy mergesort is stable => ties keep lower e first)."""
    out = np.empty((L.shape[0], k), np.int32)
    for t in range(L.shape[0]):
        order = np.argsort(-L[t].astype(np.float64), kind="stable")
        out[t] = order[:k]
    return out


@pytest.mark.parametrize("E,k", [(8, 2), (6, 6), (5, 1), (130, 8), (256, 8), (33, 3)])
def test_topk_matches_stable_sort_bruteforce(E, k):
    rng = np.random.default_rng(E * 100 + k)
    L = rng.standard_normal((97, E)).astype(np.float32)
    L[3] = 0.25                                   # all equal
    L[4, :] = np.round(L[4] * 2) / 2              # many duplicates
    idx, w = oracle.topk_gate(L, k)
    assert np.array_equal(idx, brute_topk(L, k))
    assert np.array_equal(idx[3], np.arange(k))   # all-equal logits => experts 0..k-1 in order
    for t in range(L.shape[0]):
        assert len(set(idx[t].tolist())) == k     # k distinct experts per token


def test_topk_known_answer_distinct_integers_and_signed_zero_tie():
    L = np.array([[3, 9, 1, 7, 5, -2]], np.float32)
    idx, w = oracle.topk_gate(L, 3)
    assert idx.tolist() == [[1, 3, 4]]
    e = np.exp(np.array([0.0, -2.0, -4.0]))
    assert np.allclose(w[0], e / e.sum(), rtol=1e-7)
    Lz = np.array([[-1.0, -0.0, 0.0, -5.0]], np.float32)     # -0.0 == +0.0: tie -> lower index
    idx, _ = oracle.topk_gate(Lz, 2)
    assert idx.tolist() == [[1, 2]]
    idx, _ = oracle.topk_gate(L, 6)                          # k = E: a permutation of all experts
    assert sorted(idx[0].tolist()) == list(range(6))
    assert idx.tolist() == [[1, 3, 4, 0, 2, 5]]


@pytest.mark.parametrize("E,k", [(8, 2), (64, 6), (128, 8), (4, 4)])
def test_gate_weights_softmax_renorm(E, k):
    rng = np.random.default_rng(E + k)
    L = (rng.standard_normal((64, E)) * 2).astype(np.float32)
    idx, w = oracle.topk_gate(L, k)
    assert np.all(np.abs(w.astype(np.float64).sum(1) - 1) <= 4 * k * 2.0**-24)   # sums to 1
    # "softmax over all E, then renormalise over the top-k" is the same function (S2)
    Ld = L.astype(np.float64)
    full = np.exp(Ld - Ld.max(1, keepdims=True))
    full /= full.sum(1, keepdims=True)
    sel = np.take_along_axis(full, idx.astype(np.int64), 1)
    assert np.allclose(w, sel / sel.sum(1, keepdims=True), rtol=0, atol=1e-6)
    if k == E:                                                 # k=E: the full softmax itself
        assert np.allclose(w, sel, rtol=0, atol=1e-6)
    assert np.all(np.diff(w, axis=1) <= 0)                     # slots ordered by logit descending


def test_gate_weights_special_cases():
    L = np.random.default_rng(1).standard_normal((10, 12)).astype(np.float32)
    _, w1 = oracle.topk_gate(L, 1)
    assert np.array_equal(w1, np.ones((10, 1), np.float32))    # k=1 => exactly 1.0f
    _, we = oracle.topk_gate(np.full((3, 8), -1.5, np.float32), 4)
    assert np.array_equal(we, np.full((3, 4), 0.25, np.float32))   # equal logits => 1/k
    with pytest.raises(ValueError):
        oracle.topk_gate(L, 13)                                # k > E rejected


# ----------------------------------------------------------------------------- a3-a5 hist / scan / perm
@pytest.mark.parametrize("T,E,k", [(1, 4, 2), (97, 8, 2), (300, 130, 8), (64, 256, 8), (50, 3, 3)])
def test_hist_scan_perm_invariants_and_stable_sort(T, E, k):
    rng = np.random.default_rng(T + E)
    L = rng.standard_normal((T, E)).astype(np.float32)
    L[:, 0] -= 100.0 if E > 4 else 0.0                          # make expert 0 empty when possible
    idx, _ = oracle.topk_gate(L, k)
    counts, offsets, row_src, inv_perm = oracle.hist_scan_perm(idx, E)
    R = T * k
    assert counts.sum() == R                                    # counts sum to T*k
    assert np.array_equal(counts, np.bincount(idx.ravel(), minlength=E))
    if E > 4:
        assert counts[0] == 0
    assert offsets[0] == 0 and offsets[E] == R
    assert np.array_equal(np.diff(offsets), counts)
    assert np.array_equal(np.sort(row_src), np.arange(R))       # bijection on [0,R)
    assert np.array_equal(inv_perm[row_src], np.arange(R))      # inv_perm o row_src = id
    flat = idx.ravel()
    assert np.all(np.diff(flat[row_src]) >= 0)                  # expert-contiguous
    assert np.array_equal(row_src, np.argsort(flat, kind="stable"))   # == stable sort by expert
    for e in range(E):                                          # stable: ascending inside each expert
        seg = row_src[offsets[e]:offsets[e + 1]]
        assert np.all(np.diff(seg) > 0)
        assert np.all(flat[seg] == e)


def test_hist_rejects_out_of_range_expert():
    with pytest.raises(ValueError):
        oracle.hist_scan_perm(np.array([[0, 5]], np.int32), 4)


def test_gather_copies_rows():
    cfg = wl.small_config(T=7, d=16, E=4, k=2)
    h = wl.make_hidden(cfg)
    row_src = np.array([3, 0, 13, 1, 2, 12, 5, 4, 6, 7, 8, 9, 10, 11], np.int32)
    x = oracle.gather(h, row_src, 2)
    hb = h.view(torch.int16).numpy().view(np.uint16)
    for r, i in enumerate(row_src):
        assert np.array_equal(x[r], hb[i // 2])


# ----------------------------------------------------------------------------- a7/a8 expert FFN
def np_swiglu(x64, Wg64, Wu64, Wd64):
    g = x64 @ Wg64
    u = x64 @ Wu64
    return ((g / (1 + np.exp(-g))) * u) @ Wd64


def test_e1_k1_is_dense_swiglu_ffn_numpy():
    """E=1,k=1: the layer equals a dense SwiGLU FFN (gate weight exactly 1)."""
    lay = small_layer(T=19, d=48, E=1, k=1, f=80)
    res = oracle.forward_batched(lay["hidden"], lay["W_r"], None, lay["W_gate"], lay["W_up"], lay["W_down"], 1)
    ref = np_swiglu(bf16_to_f64(lay["hidden"]), bf16_to_f64(lay["W_gate"][0]), bf16_to_f64(lay["W_up"][0]),
                    bf16_to_f64(lay["W_down"][0]))
    assert np.array_equal(res["w"], np.ones((19, 1), np.float32))
    assert np.allclose(res["out"], ref, rtol=1e-12, atol=1e-15)
    assert np.max(np.abs(ref)) > 1e-4


def test_expert_ffn_pure_python_triple_loop_tiny():
    """Separately written naive loops (math.exp, python floats) on a tiny shape, 2 experts."""
    lay = small_layer(T=3, d=8, E=2, k=1, f=8)
    x = lay["hidden"]
    offsets = np.array([0, 2, 3], np.int32)
    y = oracle.expert_ffn(x, offsets, lay["W_gate"], lay["W_up"], lay["W_down"])
    X = bf16_to_f64(x).tolist()
    for r in range(3):
        e = 0 if r < 2 else 1
        Wg = bf16_to_f64(lay["W_gate"][e]).tolist()
        Wu = bf16_to_f64(lay["W_up"][e]).tolist()
        Wd = bf16_to_f64(lay["W_down"][e]).tolist()
        h = []
        for c in range(8):
            g = sum(X[r][j] * Wg[j][c] for j in range(8))
            u = sum(X[r][j] * Wu[j][c] for j in range(8))
            h.append(g / (1.0 + math.exp(-g)) * u)
        for j in range(8):
            yy = sum(h[c] * Wd[c][j] for c in range(8))
            assert y[r, j] == pytest.approx(yy, rel=1e-12, abs=1e-300)


def test_expert_ffn_one_hot_zero_scaling_and_operand_order():
    lay = small_layer(T=4, d=16, E=3, k=1, f=24)
    x = torch.zeros(4, 16, dtype=torch.bfloat16)
    x[1, 5] = 1.0            # row 1 -> expert 1 (offsets below)
    x[3, 2] = 1.0            # row 3 -> expert 2
    offsets = np.array([0, 1, 2, 4], np.int32)
    Wg, Wu, Wd = lay["W_gate"], lay["W_up"], lay["W_down"]
    y = oracle.expert_ffn(x, offsets, Wg, Wu, Wd)
    assert np.all(y[0] == 0) and np.all(y[2] == 0)              # zero input => zero
    for r, e, j in [(1, 1, 5), (3, 2, 2)]:                      # one-hot closed form
        g = bf16_to_f64(Wg[e][j])
        u = bf16_to_f64(Wu[e][j])
        ref = ((g / (1 + np.exp(-g))) * u) @ bf16_to_f64(Wd[e])
        assert np.allclose(y[r], ref, rtol=1e-12, atol=0)
    xr = wl.make_hidden(wl.small_config(T=4, d=16))
    y1 = oracle.expert_ffn(xr, offsets, Wg, Wu, Wd)
    y2 = oracle.expert_ffn(xr, offsets, Wg, Wu, (Wd.float() * 2).to(torch.bfloat16))
    assert np.array_equal(y2, 2 * y1)                           # W_down*2 doubles exactly
    ys = oracle.expert_ffn(xr, offsets, Wu, Wg, Wd)             # swapped gate/up must differ
    assert np.max(np.abs(ys - y1)) > 1e-3 * np.max(np.abs(y1))
    # and equals numpy with the operands swapped the same way (silu on the FIRST matrix)
    ref_sw = np_swiglu(bf16_to_f64(xr[2:4]), bf16_to_f64(Wu[2]), bf16_to_f64(Wg[2]), bf16_to_f64(Wd[2]))
    assert np.allclose(ys[2:4], ref_sw, rtol=1e-12, atol=1e-18)
    ref = np_swiglu(bf16_to_f64(xr[2:4]), bf16_to_f64(Wg[2]), bf16_to_f64(Wu[2]), bf16_to_f64(Wd[2]))
    assert np.allclose(y1[2:4], ref, rtol=1e-12, atol=1e-18)


# ----------------------------------------------------------------------------- a9 un-permute
def test_unpermute_closed_form():
    T, k, d, E = 11, 3, 5, 6
    L = np.random.default_rng(0).standard_normal((T, E)).astype(np.float32)
    idx, w = oracle.topk_gate(L, k)
    _, _, _, inv_perm = oracle.hist_scan_perm(idx, E)
    Y = np.repeat(np.arange(T * k, dtype=np.float64)[:, None], d, 1)        # Y[r,:] = r
    out = oracle.unpermute(Y, inv_perm, w)
    ref = (w.astype(np.float64) * inv_perm.reshape(T, k)).sum(1)
    assert np.allclose(out, np.repeat(ref[:, None], d, 1), rtol=1e-14)


# ----------------------------------------------------------------------------- whole layer
@pytest.mark.parametrize("T,d,E,k,f", [(40, 32, 6, 2, 48), (9, 24, 5, 5, 16), (64, 64, 16, 4, 40)])
def test_bruteforce_per_token_equals_batched(T, d, E, k, f):
    lay = small_layer(T=T, d=d, E=E, k=k, f=f)
    args = (lay["hidden"], lay["W_r"], None, lay["W_gate"], lay["W_up"], lay["W_down"], k)
    res = oracle.forward_batched(*args)
    bf = oracle.forward_tokens(*args, tokens=np.arange(T))
    assert np.allclose(res["out"], bf, rtol=1e-12, atol=1e-18)
    assert np.max(np.abs(bf)) > 0


def test_whole_layer_against_numpy_definition():
    """Independent numpy restatement of the definition (argsort routing, fp64 matmuls)."""
    T, d, E, k, f = 24, 32, 5, 2, 40
    lay = small_layer(T=T, d=d, E=E, k=k, f=f)
    b = torch.tensor([0.3, -0.2, 0.0, 0.5, -0.4])
    res = oracle.forward_batched(lay["hidden"], lay["W_r"], b, lay["W_gate"], lay["W_up"], lay["W_down"], k)
    X = bf16_to_f64(lay["hidden"])
    L = (X @ lay["W_r"].to(torch.float64).numpy() + b.to(torch.float64).numpy()).astype(np.float32)
    assert np.allclose(res["logits"], L, atol=1e-6, rtol=0)
    ref = np.zeros((T, d))
    for t in range(T):
        Lt = res["logits"][t].astype(np.float64)
        order = np.argsort(-Lt, kind="stable")[:k]
        ws = np.exp(Lt[order] - Lt[order[0]])
        ws = (ws / ws.sum()).astype(np.float32).astype(np.float64)
        for s, e in enumerate(order):
            ref[t] += ws[s] * np_swiglu(X[t:t + 1], bf16_to_f64(lay["W_gate"][e]), bf16_to_f64(lay["W_up"][e]),
                                        bf16_to_f64(lay["W_down"][e]))[0]
    assert np.allclose(res["out"], ref, rtol=1e-11, atol=1e-16)


def test_combine_invariance_concat_split_and_segment_order():
    """combining is a concatenation and does not affect correctness."""
    cfg = wl.small_config(T=30, d=32, E=6, k=2, f=24)
    lay = wl.make_layer(cfg)
    args = lambda h: (h, lay["W_r"], None, lay["W_gate"], lay["W_up"], lay["W_down"], 2)
    h = lay["hidden"]
    full = oracle.forward_batched(*args(h))["out"]
    a = oracle.forward_batched(*args(h[:11]))["out"]
    b = oracle.forward_batched(*args(h[11:]))["out"]
    assert np.array_equal(np.concatenate([a, b]), full)          # exact in the oracle
    perm = np.random.default_rng(5).permutation(30)
    shuf = oracle.forward_batched(*args(h[torch.from_numpy(perm)]))["out"]
    assert np.array_equal(shuf, full[perm])
    hd = h.clone()
    hd[7] = hd[2]                                                # duplicate tokens => identical rows
    dup = oracle.forward_batched(*args(hd))["out"]
    assert np.array_equal(dup[7], dup[2])


def test_logits_in_overrides_router():
    lay = small_layer(T=12, d=16, E=4, k=2, f=16)
    L = np.random.default_rng(2).standard_normal((12, 4)).astype(np.float32)
    res = oracle.forward_batched(lay["hidden"], lay["W_r"], None, lay["W_gate"], lay["W_up"], lay["W_down"], 2,
                                 logits_in=L)
    assert np.array_equal(res["logits"], L)
    assert np.array_equal(res["idx"], brute_topk(L, 2))
    bf = oracle.forward_tokens(lay["hidden"], lay["W_r"], None, lay["W_gate"], lay["W_up"], lay["W_down"], 2,
                               tokens=[5, 0, 11], logits_in=L)
    assert np.allclose(bf, res["out"][[5, 0, 11]], rtol=1e-12, atol=1e-18)


# ----------------------------------------------------------------------------- workloads recipe
def test_c1_config_matches_baseline_and_is_seeded():
    lay = wl.make_layer(wl.C1)
    assert lay["hidden"].shape == (256, 512) and lay["W_gate"].shape == (8, 512, 1024)
    assert lay["W_down"].shape == (8, 1024, 512) and lay["W_r"].shape == (512, 8)
    assert lay["hidden"].dtype == torch.bfloat16 and lay["W_r"].dtype == torch.float32
    assert abs(lay["hidden"].float().std().item() - 1.0) < 0.02
    assert abs(lay["W_gate"].float().std().item() - 0.02) < 0.001
    assert abs(lay["W_r"].std().item() - 1 / math.sqrt(512)) < 0.002
    assert torch.equal(wl.make_hidden(wl.C1), lay["hidden"])     # deterministic
    assert sum(wl.segment_lengths(wl.C1)) == 256


def test_c4_zipf_bias_shape():
    W_r, b_r = wl.make_router(wl.MoEConfig("z", 3, T=8, d=64, E=256, k=8, f=8, zipf_s=1.1))
    assert b_r.shape == (256,) and b_r.max().item() == 0.0
    assert b_r.min().item() == pytest.approx(-1.1 * math.log(256), rel=1e-6)
    assert len(set(b_r.tolist())) == 256
