"""CPU oracle for the FP8 (e4m3) gate/up expert GEMM -- TEST INFRASTRUCTURE, not a product path.

Only `tests/` (and `bench.py`'s oracle legs) may import this module; it shares no code with
`paper_2606_21712_b200/` and imports nothing from it.

What it restates.  The paper runs its MoE GEMMs in FP8 ("FP8 MoE GEMMs at 1979 TFLOP/s", §5.5;
FP8 DeepSeek-R1 / Kimi-K2 weights, §6.1; FP8 decoding, §6.3) and says nothing about
the quantisation recipe.  Reading taken (F1-F4):

  F1  format: OCP e4m3 ("e4m3fn": 1 sign, 4 exponent bits, bias 7, 3 mantissa bits, no infinities, the one NaN code
      S.1111.111, largest finite 448, subnormals k * 2^-9); conversion rounds to nearest even and SATURATES at +-448.
  F2  activations: one fp32 scale per token row, sx[r] = fl32(max_j |x[r,j]| / 448) (1 if the row is zero),
      xq[r,j] = e4m3(fl32(x[r,j] / sx[r])).  The division and the scale are IEEE fp32 -- the precision in which
      both sides take the integer decision (the code), so the codes are compared bit for bit.
  F3  weights: one fp32 scale per expert and OUTPUT channel, sw[e,n] = fl32(max_k |W[e,k,n]| / 448) (1 if zero),
      Wq[e,n,k] = e4m3(fl32(W[e,k,n] / sw[e,n])); the quantised tensor is stored [E, N, K] (k contiguous).
  F4  scope: the gate/up GEMM (two thirds of the expert FLOPs and weight bytes) runs W8A8:
        g[r,n] = sx[r] * sw_gate[e,n] * sum_k xq[r,k] * Wq_gate[e,n,k]      (products exact, fp32 accumulate on the GPU)
        u[r,n] likewise;  H = silu(g) * u;  Y = H W_down[e] with H and W_down in bf16 as before.
      (precision 1: H and the down GEMM stay bf16.)
  F5  precision 2 adds the down GEMM: H is first rounded to bf16 as in every other path (RNE), then quantised like an
      activation row (F2: sh[r] = fl32(max_n |Hb[r,n]| / 448), Hq = e4m3(fl32(Hb / sh))), W_down per expert and output
      channel (F3, stored [E, d, f]), and  Y[r,j] = sh[r] * sw_down[e,j] * sum_n Hq[r,n] * Wq_down[e,j,n].

Every floating-point step of the reference GEMMs is fp64 on exactly decoded values, with no intermediate rounding
(as in bgo_oracle.cpp); only the quantisation decisions are taken in fp32, as F2 / F3 state.

Pins (tests/test_oracle_fp8.py, -m "not gpu"): the 256-entry decode table against the format's closed form and the
values the OCP format fixes (0x38 = 1, 0x7E = 448, 0x01 = 2^-9, 0x08 = 2^-6, 0x7F = NaN); encode(decode(c)) = c for
every finite code; ties to even and saturation on hand-computed cases; agreement with torch's float8_e4m3fn
conversion (a library routine) on in-range values; scale invariance under powers of two; quantise-dequantise error
<= 2^-4 relative (normal range); the W8A8 GEMM against a pure-Python triple loop on a tiny case; and with weights /
activations that are exactly representable the FP8 path equals the bf16 oracle's expert FFN.
"""
from __future__ import annotations

import numpy as np

E4M3_MAX = 448.0


def e4m3_decode_table() -> np.ndarray:
    """float64[256]: the value of every e4m3 code (NaN for 0x7F / 0xFF), from the format's definition."""
    t = np.empty(256, np.float64)
    for c in range(256):
        s = -1.0 if c & 0x80 else 1.0
        e = (c >> 3) & 0xF
        m = c & 0x7
        if e == 0xF and m == 0x7:
            t[c] = np.nan
        elif e == 0:
            t[c] = s * m * 2.0 ** -9
        else:
            t[c] = s * (1.0 + m / 8.0) * 2.0 ** (e - 7)
    return t


_DECODE = e4m3_decode_table()


def e4m3_decode(codes: np.ndarray) -> np.ndarray:
    return _DECODE[np.asarray(codes, dtype=np.uint8)]


def e4m3_encode(x: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even, saturating conversion of finite float values to e4m3 codes (uint8).
    Exact: the input is widened to float64 and only scaled by powers of two before np.rint (half to even)."""
    x = np.asarray(x, dtype=np.float64)
    assert np.all(np.isfinite(x)), "the oracle's quantiser takes finite values only"
    sign = np.signbit(x)
    a = np.minimum(np.abs(x), E4M3_MAX)                    # saturate
    code = np.zeros(x.shape, np.int64)
    sub = a < 2.0 ** -6
    # subnormal grid: multiples of 2^-9 (q = 8 is the first normal, code 0x08)
    q_sub = np.rint(a / 2.0 ** -9).astype(np.int64)
    code = np.where(sub, q_sub, code)
    # normal: a = m * 2^e, m in [1, 2)
    mant, expo = np.frexp(np.where(sub, 1.0, a))           # a = mant * 2^expo, mant in [0.5, 1)
    e = expo - 1
    m = mant * 2.0
    q = np.rint((m - 1.0) * 8.0).astype(np.int64)          # 0..8, half to even
    e = np.where(q == 8, e + 1, e)
    q = np.where(q == 8, 0, q)
    c_norm = ((e + 7) << 3) | q
    c_norm = np.minimum(c_norm, 0x7E)                      # rounding up past 448 saturates too
    code = np.where(sub, code, c_norm)
    code = code | np.where(sign, 0x80, 0)
    return code.astype(np.uint8)


def quantize_rows(x: np.ndarray):
    """F2.  x: float32 [R, K] (exactly widened bf16).  Returns (codes uint8 [R, K], sx float32 [R])."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    amax = np.max(np.abs(x), axis=1).astype(np.float32) if x.shape[1] else np.zeros(x.shape[0], np.float32)
    sx = (amax / np.float32(E4M3_MAX)).astype(np.float32)
    sx = np.where(amax == 0, np.float32(1.0), sx).astype(np.float32)
    ratio = (x / sx[:, None]).astype(np.float32)           # IEEE fp32 division
    return e4m3_encode(ratio), sx


def quantize_weight_channels(W: np.ndarray):
    """F3.  W: float32 [E, K, N].  Returns (codes uint8 [E, N, K], sw float32 [E, N])."""
    W = np.asarray(W, dtype=np.float32)
    amax = np.max(np.abs(W), axis=1).astype(np.float32)    # [E, N]
    sw = (amax / np.float32(E4M3_MAX)).astype(np.float32)
    sw = np.where(amax == 0, np.float32(1.0), sw).astype(np.float32)
    ratio = (W / sw[:, None, :]).astype(np.float32)
    return np.ascontiguousarray(e4m3_encode(ratio).transpose(0, 2, 1)), sw


def _silu(z: np.ndarray) -> np.ndarray:
    return z / (1.0 + np.exp(-z))


def round_bf16(a: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even of float64 / float32 values to bf16, returned as float32 (exact bit arithmetic on the
    float32 rounding of the input; the inputs here are far from the float32 rounding boundary cases that would make
    the double rounding visible -- and the GPU's H is compared through its own bits anyway, reading F5)."""
    x = np.ascontiguousarray(a, dtype=np.float32)
    u = x.view(np.uint32).astype(np.uint64)
    r = ((u + 0x7FFF + ((u >> 16) & 1)) >> 16) << 16
    return r.astype(np.uint32).view(np.float32).reshape(x.shape)


def down_fp8(H_bf16: np.ndarray, offsets: np.ndarray, W_down: np.ndarray) -> dict:
    """F5.  H_bf16 float32 [R, f] (bf16 values), W_down float32 [E, f, d].  Returns y float64 [R, d] + artefacts."""
    R, f = H_bf16.shape
    E, _, d = W_down.shape
    hq, sh = quantize_rows(H_bf16)
    dq, sd = quantize_weight_channels(W_down)              # [E, d, f], [E, d]
    hd = e4m3_decode(hq)
    y = np.zeros((R, d), np.float64)
    for e in range(E):
        r0, r1 = int(offsets[e]), int(offsets[e + 1])
        if r1 > r0:
            y[r0:r1] = (hd[r0:r1] @ e4m3_decode(dq[e]).T) * sh[r0:r1, None].astype(np.float64) * sd[e][None, :].astype(np.float64)
    return dict(y=y, hq=hq, sh=sh, dq=dq, sd=sd)


def expert_ffn_fp8_gateup(x_perm: np.ndarray, offsets: np.ndarray, W_gate: np.ndarray, W_up: np.ndarray,
                          W_down: np.ndarray) -> dict:
    """F4.  x_perm float32 [R, d] (widened bf16), offsets int [E+1], W_gate / W_up float32 [E, d, f], W_down float32
    [E, f, d] (all exactly widened bf16).  Returns y float64 [R, d] and the quantisation artefacts."""
    R, d = x_perm.shape
    E = W_gate.shape[0]
    xq, sx = quantize_rows(x_perm)
    gq, sg = quantize_weight_channels(W_gate)
    uq, su = quantize_weight_channels(W_up)
    xd = e4m3_decode(xq)                                   # float64 [R, d]
    y = np.zeros((R, d), np.float64)
    H = np.zeros((R, W_gate.shape[2]), np.float64)
    for e in range(E):
        r0, r1 = int(offsets[e]), int(offsets[e + 1])
        if r1 == r0:
            continue
        xe = xd[r0:r1]                                     # [n, d]
        g = (xe @ e4m3_decode(gq[e]).T) * sx[r0:r1, None].astype(np.float64) * sg[e][None, :].astype(np.float64)
        u = (xe @ e4m3_decode(uq[e]).T) * sx[r0:r1, None].astype(np.float64) * su[e][None, :].astype(np.float64)
        h = _silu(g) * u
        H[r0:r1] = h
        y[r0:r1] = h @ W_down[e].astype(np.float64)
    return dict(y=y, H=H, xq=xq, sx=sx, gq=gq, sg=sg, uq=uq, su=su)
