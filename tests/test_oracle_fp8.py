"""Pins of the FP8 oracle (oracle/fp8.py, readings F1-F4 of DESIGN.md §2) -- CPU only.

The paper runs FP8 MoE GEMMs and gives no recipe; every pin below fixes the oracle to
something other than itself: the OCP e4m3 format's closed form and fixed points, hand-computed rounding cases,
torch's own float8_e4m3fn conversion, invariants, a pure-Python loop, and the bf16 oracle on exactly representable
data."""
import numpy as np
import torch

import oracle
from oracle import fp8


def test_decode_table_matches_the_format():
    t = fp8.e4m3_decode_table()
    # fixed points of OCP e4m3 (no infinities, one NaN code per sign, largest finite 448)
    assert t[0x00] == 0.0 and t[0x38] == 1.0 and t[0x7E] == 448.0 and t[0xFE] == -448.0
    assert t[0x01] == 2.0 ** -9 and t[0x07] == 7 * 2.0 ** -9 and t[0x08] == 2.0 ** -6
    assert t[0x40] == 2.0 and t[0x3C] == 1.5 and t[0xB8] == -1.0
    assert np.isnan(t[0x7F]) and np.isnan(t[0xFF])
    fin = np.array([c for c in range(256) if c & 0x7F != 0x7F], dtype=np.uint8)
    # torch's bit-level view of the same codes (a library routine)
    ref = torch.from_numpy(fin.copy()).view(torch.float8_e4m3fn).to(torch.float64).numpy()
    assert np.array_equal(t[fin], ref)
    # strictly increasing in the positive codes
    assert np.all(np.diff(t[0:0x7F]) > 0)


def test_encode_is_the_inverse_of_decode_on_every_finite_code():
    fin = np.array([c for c in range(256) if c & 0x7F != 0x7F], dtype=np.uint8)
    vals = fp8.e4m3_decode(fin)
    back = fp8.e4m3_encode(vals)
    # -0.0 encodes to 0x80, +0.0 to 0x00
    assert np.array_equal(back, fin)


def test_rounding_ties_to_even_and_saturation():
    # between 1.0 (mantissa 000) and 1.125 (001): 1.0625 is a tie -> even mantissa 000
    # between 1.125 (001) and 1.25 (010): 1.1875 is a tie -> 010
    # 464 is the midpoint of 448 and the non-existent 480: rounds to 448; anything larger saturates
    # subnormals: 1.5 * 2^-9 ties to 2 * 2^-9; 0.5 * 2^-9 ties to 0; 7.5 * 2^-9 ties to 8 * 2^-9 = 2^-6 (first normal)
    x = np.array([1.0625, 1.1875, 1.0626, 464.0, 480.0, 1e9, -1e9, 1.5 * 2.0 ** -9, 0.5 * 2.0 ** -9,
                  7.5 * 2.0 ** -9, 0.51 * 2.0 ** -9, -0.3])
    got = fp8.e4m3_decode(fp8.e4m3_encode(x))
    want = np.array([1.0, 1.25, 1.125, 448.0, 448.0, 448.0, -448.0, 2 * 2.0 ** -9, 0.0, 2.0 ** -6, 2.0 ** -9, -0.3125])
    assert np.array_equal(got, want)


def test_encode_agrees_with_torch_in_range():
    rng = np.random.default_rng(0)
    x = np.concatenate([rng.standard_normal(20000) * s for s in (1e-3, 0.05, 1.0, 30.0, 150.0)]).astype(np.float32)
    x = x[np.abs(x) <= 448.0]
    mine = fp8.e4m3_decode(fp8.e4m3_encode(x))
    ref = torch.from_numpy(x).to(torch.float8_e4m3fn).to(torch.float64).numpy()
    assert np.array_equal(mine, ref)


def test_quantise_rows_scale_properties():
    rng = np.random.default_rng(1)
    x = torch.from_numpy(rng.standard_normal((37, 200)).astype(np.float32)).to(torch.bfloat16).float().numpy()
    x[5] = 0.0                                            # zero row: scale 1, codes 0
    q, sx = fp8.quantize_rows(x)
    assert sx[5] == 1.0 and not q[5].any()
    # the row maximum maps to +-448 exactly
    deq = fp8.e4m3_decode(q) * sx[:, None]
    for r in range(37):
        if r != 5:
            j = np.argmax(np.abs(x[r]))
            assert abs(fp8.e4m3_decode(q[r, j])) == 448.0
    # relative error of quantise-dequantise <= 2^-4 in the normal range (3 mantissa bits, RNE), plus fp32 scale rounding
    big = np.abs(x) >= (2.0 ** -6) * sx[:, None] * 1.01
    rel = np.abs(deq - x)[big] / np.abs(x)[big]
    assert rel.max() <= 2.0 ** -4 * 1.001
    # scale invariance: a power of two on the row changes the scale, never the codes
    q2, sx2 = fp8.quantize_rows(x * 8.0)
    assert np.array_equal(q2, q) and np.array_equal(sx2[np.arange(37) != 5], (sx * 8.0)[np.arange(37) != 5])


def test_weight_channel_quantisation_layout_and_scales():
    rng = np.random.default_rng(2)
    W = (rng.standard_normal((3, 40, 24)) * 0.02).astype(np.float32)
    W[1, :, 7] = 0.0
    q, sw = fp8.quantize_weight_channels(W)
    assert q.shape == (3, 24, 40) and sw.shape == (3, 24)              # [E, N, K], k contiguous
    assert sw[1, 7] == 1.0 and not q[1, 7].any()
    # the same thing as quantising every output channel as a row
    for e in range(3):
        qr, sr = fp8.quantize_rows(np.ascontiguousarray(W[e].T))
        assert np.array_equal(qr, q[e]) and np.array_equal(sr, sw[e])


def test_w8a8_gemm_against_a_pure_python_loop():
    rng = np.random.default_rng(3)
    R, d, f, E = 7, 16, 8, 2
    bf = lambda a: torch.from_numpy(a.astype(np.float32)).to(torch.bfloat16).float().numpy()
    x, Wg, Wu, Wd = bf(rng.standard_normal((R, d))), bf(rng.standard_normal((E, d, f)) * 0.3), \
        bf(rng.standard_normal((E, d, f)) * 0.3), bf(rng.standard_normal((E, f, d)) * 0.3)
    off = np.array([0, 4, 7])
    res = fp8.expert_ffn_fp8_gateup(x, off, Wg, Wu, Wd)
    tab = fp8.e4m3_decode_table()
    for r in range(R):
        e = 0 if r < 4 else 1
        h = []
        for n in range(f):
            g = sum(tab[res["xq"][r, k]] * tab[res["gq"][e, n, k]] for k in range(d)) * float(res["sx"][r]) * float(res["sg"][e, n])
            u = sum(tab[res["xq"][r, k]] * tab[res["uq"][e, n, k]] for k in range(d)) * float(res["sx"][r]) * float(res["su"][e, n])
            h.append(g / (1.0 + np.exp(-g)) * u)
        for j in range(d):
            yj = sum(h[n] * float(Wd[e, n, j]) for n in range(f))
            assert abs(yj - res["y"][r, j]) <= 1e-12 * max(1.0, abs(yj))


def test_exactly_representable_data_reduces_to_the_bf16_oracle():
    """If every x[r,:] / sx[r] and W[:,n] / sw[n] is an e4m3 value, quantisation is lossless and the FP8 path must
    equal the bf16 oracle's expert FFN (bgo_oracle.cpp) -- a textbook special case that pins the scale handling."""
    rng = np.random.default_rng(4)
    R, d, f, E = 24, 32, 16, 3
    grid = fp8.e4m3_decode(np.array([c for c in range(0x30, 0x46)], dtype=np.uint8))      # e4m3 values 0.5 .. 3.25
    x = rng.choice(grid, size=(R, d)) * rng.choice([-1.0, 1.0], size=(R, d))
    Wg = rng.choice(grid, size=(E, d, f)) * rng.choice([-1.0, 1.0], size=(E, d, f)) / 64.0
    Wu = rng.choice(grid, size=(E, d, f)) * rng.choice([-1.0, 1.0], size=(E, d, f)) / 64.0
    Wd = (rng.standard_normal((E, f, d)) * 0.1)
    # make every row / channel maximum a value whose scale amax / 448 is a power of two times an e4m3 grid step:
    # put 3.5 = 448 / 128 in each row and channel, so sx = sw = 2^-7 (resp. 2^-13) exactly
    x[:, 0] = 3.5
    Wg[:, 0, :] = 3.5 / 64.0
    Wu[:, 0, :] = 3.5 / 64.0
    tb = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to(torch.bfloat16)
    xb, Wgb, Wub, Wdb = tb(x), tb(Wg), tb(Wu), tb(Wd)
    assert np.array_equal(xb.float().numpy(), x.astype(np.float32))                        # bf16 holds them exactly
    off = np.array([0, 10, 10, 24], dtype=np.int32)
    res = fp8.expert_ffn_fp8_gateup(xb.float().numpy(), off, Wgb.float().numpy(), Wub.float().numpy(), Wdb.float().numpy())
    assert np.all(res["sx"] == np.float32(2.0 ** -7))
    ref = oracle.expert_ffn(xb, off, Wgb, Wub, Wdb)
    assert np.max(np.abs(res["y"] - ref)) <= 1e-12 * np.max(np.abs(ref))


def test_round_bf16_matches_torch():
    rng = np.random.default_rng(6)
    x = np.concatenate([rng.standard_normal(50000) * s for s in (1e-4, 1.0, 300.0)]).astype(np.float32)
    x = np.concatenate([x, np.array([1.00390625, 1.01171875, -1.00390625, 0.0, -0.0], np.float32)])   # exact ties
    ref = torch.from_numpy(x).to(torch.bfloat16).float().numpy()
    assert np.array_equal(fp8.round_bf16(x).view(np.uint32), ref.view(np.uint32))


def test_down_fp8_against_a_pure_python_loop_and_lossless_case():
    rng = np.random.default_rng(7)
    R, f, d, E = 6, 12, 8, 2
    H = fp8.round_bf16(rng.standard_normal((R, f)))
    Wd = fp8.round_bf16(rng.standard_normal((E, f, d)) * 0.2)
    off = np.array([0, 2, 6])
    res = fp8.down_fp8(H, off, Wd)
    tab = fp8.e4m3_decode_table()
    for r in range(R):
        e = 0 if r < 2 else 1
        for j in range(d):
            acc = sum(tab[res["hq"][r, n]] * tab[res["dq"][e, j, n]] for n in range(f))
            want = acc * float(res["sh"][r]) * float(res["sd"][e, j])
            assert abs(want - res["y"][r, j]) <= 1e-12 * max(1.0, abs(want))
    # lossless case: values on the e4m3 grid with power-of-two scales -> the plain fp64 product
    grid = fp8.e4m3_decode(np.arange(0x30, 0x46, dtype=np.uint8))
    H = rng.choice(grid, size=(R, f)) * rng.choice([-1.0, 1.0], size=(R, f))
    H[:, 0] = 3.5
    Wd = rng.choice(grid, size=(E, f, d)) * rng.choice([-1.0, 1.0], size=(E, f, d)) / 32.0
    Wd[:, 0, :] = 3.5 / 32.0
    res = fp8.down_fp8(H.astype(np.float32), off, Wd.astype(np.float32))
    for e, (r0, r1) in enumerate(((0, 2), (2, 6))):
        assert np.max(np.abs(res["y"][r0:r1] - H[r0:r1] @ Wd[e])) <= 1e-12
