"""GPU parity at BASELINE.json's FULL sizes (configs C2..C5), in the launch configuration bench.py
times (one fused `bg_moe_combined_forward` on a context sized for T).

Routing artefacts are checked in full against the oracle (bit-exact given the GPU's fp32 logits) and
so is the WHOLE `[T,d]` output: the oracle's per-token brute force runs over every token (fp64, routed
by the GPU's logits, reading S5), so every (expert, feature tile, token tile) of both grouped GEMMs has
all of its rows compared.  The oracle needs ~3-50 s per config on the box's host
cores; each test prints what it took.  Properties that hold at any size (counts sum to T*k, permutation
is a bijection, segments expert-contiguous and stable) are checked on the whole tensors too.

Inputs are generated on the GPU by torch's seeded Philox generator (workloads.py, device="cuda");
the oracle receives host copies of exactly those bits.
"""
import time

import numpy as np
import pytest
import torch

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

MAX_TOL, L2_TOL = 2e-2, 5e-3


def run_fullsize(cfg: wl.MoEConfig, shuffle_segments: bool = False, via_segments: bool = False):
    from paper_2606_21712_b200 import MoELayer
    lay = wl.make_layer(cfg, "cuda")
    hidden = lay["hidden"]
    if shuffle_segments:                       # reading S17: segment order must not matter
        segs = wl.segment_lengths(cfg)
        starts = np.concatenate([[0], np.cumsum(segs)[:-1]])
        order = np.random.default_rng(17).permutation(len(segs))
        rows = np.concatenate([np.arange(starts[i], starts[i] + segs[i]) for i in order])
        hidden = hidden[torch.from_numpy(rows).cuda()].contiguous()
    layer = MoELayer(cfg.d, cfg.f, cfg.E, cfg.k, cfg.T)
    layer.set_weights(lay["W_r"], lay["b_r"], lay["W_gate"], lay["W_up"], lay["W_down"])
    out = layer.combined_forward(hidden)
    out2 = layer.combined_forward(hidden)
    torch.cuda.synchronize()
    assert torch.equal(out, out2), "fused path is not bitwise deterministic"
    v = layer.debug_views(cfg.T)
    if via_segments:
        # zero-copy COMBINE at full size: the config's own coroutine list -- C5: 30 prefill segments
        # of 512 rows + 1024 single-token decode segments = 1054 -- each in its own allocation, in both router forms.
        # Every routing artefact and the output must carry the bits of the concatenated call; what is then checked
        # against the oracle below is the SEGMENT path's result.
        lengths = wl.segment_lengths(cfg)
        assert sum(lengths) == cfg.T
        segs, pos = [], 0
        for n in lengths:
            segs.append(hidden[pos:pos + n].clone())
            pos += n
        for form in (1, 2, 0):
            layer.set_debug(router_form=form)
            outs = layer.combined_forward_segments(segs)
            torch.cuda.synchronize()
            vs = layer.debug_views(cfg.T)
            for key in ("logits", "idx", "w", "counts", "offsets", "row_src", "inv_perm"):
                assert torch.equal(v[key], vs[key]), f"segments, router form {form}: {key} differs"
            seg_out = torch.cat(outs, dim=0)
            assert torch.equal(seg_out, out), f"segments, router form {form}: output differs from the concatenated call"
        print(f"[fullsize] {cfg.name}: {len(lengths)} segments, bit-identical to the concatenated call in all router forms")
        out, v = seg_out, vs
    T, k, E, R = cfg.T, cfg.k, cfg.E, cfg.T * cfg.k

    # ---- routing: whole tensors, bit-exact given the GPU's logits
    L = v["logits"].cpu().numpy()
    o_idx, o_w = oracle.topk_gate(L, k)
    assert np.array_equal(v["idx"].cpu().numpy(), o_idx)
    assert np.max(np.abs(v["w"].cpu().numpy() - o_w)) <= 2e-6
    o_counts, o_offsets, o_rs, o_ip = oracle.hist_scan_perm(o_idx, E)
    counts = v["counts"].cpu().numpy()
    assert np.array_equal(counts, o_counts) and counts.sum() == R
    assert np.array_equal(v["offsets"].cpu().numpy(), o_offsets)
    row_src, inv_perm = v["row_src"].cpu().numpy(), v["inv_perm"].cpu().numpy()
    assert np.array_equal(row_src, o_rs) and np.array_equal(inv_perm, o_ip)
    assert np.array_equal(np.sort(row_src), np.arange(R))                 # bijection
    assert np.array_equal(inv_perm[row_src], np.arange(R))

    # ---- outputs: every token, per-token brute force routed by the GPU's logits (reading S5)
    toks = np.arange(T, dtype=np.int32)
    cpu = {kk: (vv.cpu() if isinstance(vv, torch.Tensor) else vv) for kk, vv in lay.items()}
    cpu["hidden"] = hidden.cpu()
    # logits: the oracle's own fp64-accumulated logits, whole tensor
    own = oracle.router_logits(cpu["hidden"], cpu["W_r"], cpu["b_r"])
    assert np.all(np.abs(L - own) <= 1e-4 * np.maximum(1.0, np.abs(own))), "router logits out of tolerance"
    t0 = time.perf_counter()
    ref = oracle.forward_tokens(cpu["hidden"], cpu["W_r"], cpu["b_r"], cpu["W_gate"], cpu["W_up"], cpu["W_down"], k,
                                toks, logits_in=L)
    oracle_s = time.perf_counter() - t0
    got = out.to(torch.float64).cpu().numpy()
    assert np.all(np.isfinite(got))
    scale = np.abs(ref).max()
    max_err = np.abs(got - ref).max()
    l2 = np.linalg.norm(got - ref) / np.linalg.norm(ref)
    assert max_err <= MAX_TOL * scale, f"{cfg.name}: max|err| {max_err:.3e} vs {MAX_TOL}*{scale:.3e}"
    assert l2 <= L2_TOL, f"{cfg.name}: rel L2 {l2:.3e}"
    # every token row on its own too (a single wrong row is invisible in a global norm)
    row_l2 = np.linalg.norm(got - ref, axis=1) / np.maximum(np.linalg.norm(ref, axis=1), 1e-30)
    assert row_l2.max() <= 4 * L2_TOL, f"{cfg.name}: worst row rel L2 {row_l2.max():.3e} (token {row_l2.argmax()})"
    # token tiles of the grouped GEMMs (256-row cap): all of them are covered by construction
    n_tiles = int(np.ceil(counts[counts > 0] / 256).sum())
    print(f"[fullsize] {cfg.name}: whole tensor {T}x{cfg.d} checked, {n_tiles} (expert, token-tile) pairs all covered, "
          f"oracle {oracle_s:.1f} s on {oracle.num_threads()} threads, max_err/max|ref| {max_err / scale:.2e}, "
          f"relL2 {l2:.2e}, worst row relL2 {row_l2.max():.2e}")
    return dict(counts=counts, n_checked=len(toks), max_err=max_err / scale, l2=l2, oracle_s=oracle_s)


def test_c2_mixtral_full():
    r = run_fullsize(wl.C2)
    assert r["counts"].min() > 800 and r["counts"].max() < 1250          # near-uniform load


def test_c3_finegrained_T4096_full():
    r = run_fullsize(wl.C3)
    assert r["counts"].min() >= 150 and r["counts"].max() <= 400


@pytest.mark.parametrize("T", [64, 1024, 16384, 32768])
def test_c3_sweep_points(T):
    run_fullsize(wl.C3.with_T(T))


def test_c4_zipf_skewed_full():
    r = run_fullsize(wl.C4)
    c = r["counts"]
    assert (c == 0).sum() >= 20, "the Zipf bias should leave many experts empty"
    assert c.max() >= 4000, "and give a few hot experts most tokens"
    assert ((c > 0) & (c <= 2)).sum() >= 10, "with many experts at 1-2 rows"


def test_c5_mixed_prefill_decode_full():
    run_fullsize(wl.C5)


def test_c5_zero_copy_segments_full():
    run_fullsize(wl.C5, via_segments=True)


def test_c5_segment_order_shuffled():
    run_fullsize(wl.C5, shuffle_segments=True)
