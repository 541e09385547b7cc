"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element.

Bars (BASELINE.json north_star):
  * routing artefacts (idx, counts, offsets, row_src, inv_perm) bit-exact given the same fp32 logits;
  * logits |L_gpu - L_ref| <= 1e-4 * max(1,|L|); gate weights |w_gpu - w_ref| <= 2e-6;
  * expert outputs max|err| <= 2e-2 * max|ref| and relative L2 <= 5e-3 (bf16 I/O, fp32 accumulate).
"""
import numpy as np
import pytest
import torch

import oracle
import workloads as wl

pytestmark = pytest.mark.gpu

MAX_TOL, L2_TOL = 2e-2, 5e-3


def to_dev(lay):
    dev = torch.device("cuda", 0)
    return {k: (v.to(dev) if isinstance(v, torch.Tensor) else v) for k, v in lay.items()}


def make(cfg, max_tokens=None):
    from paper_2606_21712_b200 import MoELayer
    lay = wl.make_layer(cfg)
    g = to_dev(lay)
    layer = MoELayer(cfg.d, cfg.f, cfg.E, cfg.k, max_tokens or max(cfg.T, 1))
    layer.set_weights(g["W_r"], g["b_r"], g["W_gate"], g["W_up"], g["W_down"])
    return lay, g, layer


def check_out(out_gpu: torch.Tensor, ref: np.ndarray, what=""):
    got = out_gpu.to(torch.float64).cpu().numpy()
    assert np.all(np.isfinite(got)), f"{what}: non-finite output"
    scale = np.max(np.abs(ref))
    err = np.abs(got - ref)
    max_err = err.max() if err.size else 0.0
    l2 = np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-300) if err.size else 0.0
    assert max_err <= MAX_TOL * scale, f"{what}: max|err| {max_err:.3e} > {MAX_TOL}*max|ref| ({scale:.3e}); relL2 {l2:.3e}"
    assert l2 <= L2_TOL, f"{what}: relative L2 {l2:.3e} > {L2_TOL}"
    return max_err / max(scale, 1e-300), l2


def check_routing_against_oracle(logits_gpu, idx, w, counts, offsets, row_src, inv_perm, E, k):
    """Feed the GPU's fp32 logits to the oracle's top-k / hist / scan / perm: integers bit-exact."""
    L = logits_gpu.cpu().numpy()
    o_idx, o_w = oracle.topk_gate(L, k)
    assert np.array_equal(idx.cpu().numpy(), o_idx), "topk_idx differs from the oracle on the same logits"
    assert np.max(np.abs(w.cpu().numpy() - o_w)) <= 2e-6 if o_w.size else True
    assert np.all(np.abs(w.cpu().numpy().astype(np.float64).sum(1) - 1) <= 4 * k * 2.0**-24)
    o_counts, o_offsets, o_rs, o_ip = oracle.hist_scan_perm(o_idx, E)
    assert np.array_equal(counts.cpu().numpy(), o_counts)
    assert np.array_equal(offsets.cpu().numpy(), o_offsets)
    if row_src is not None:
        assert np.array_equal(row_src.cpu().numpy(), o_rs)
        assert np.array_equal(inv_perm.cpu().numpy(), o_ip)
    return o_idx, o_w, o_counts, o_offsets, o_rs, o_ip


ROUTE_SHAPES = [
    # T, d, E, k
    (256, 512, 8, 2), (1, 64, 4, 2), (127, 128, 8, 2), (129, 96, 33, 3), (300, 256, 128, 8),
    (64, 128, 256, 8), (200, 72, 5, 5), (77, 64, 1, 1), (513, 320, 64, 6), (1000, 64, 16, 1),
]


@pytest.mark.parametrize("T,d,E,k", ROUTE_SHAPES)
def test_route_and_permute_parity(T, d, E, k):
    cfg = wl.small_config(T=T, d=d, E=E, k=k, f=64, index=11)
    lay, g, layer = make(cfg)
    r = layer.route(g["hidden"])
    Lref = oracle.router_logits(lay["hidden"], lay["W_r"], lay["b_r"])
    Lg = r["logits"].cpu().numpy()
    assert np.all(np.abs(Lg - Lref) <= 1e-4 * np.maximum(1.0, np.abs(Lref))), "router logits out of tolerance"
    p = layer.permute(g["hidden"], r["idx"], r["offsets"])
    check_routing_against_oracle(r["logits"], r["idx"], r["w"], r["counts"], r["offsets"], p["row_src"],
                                 p["inv_perm"], E, k)
    xo = oracle.gather(lay["hidden"], p["row_src"].cpu().numpy(), k)
    xg = p["x_perm"].view(torch.int16).cpu().numpy().view(np.uint16)
    assert np.array_equal(xg, xo), "gathered rows differ"
    torch.cuda.synchronize()


def test_route_logits_in_ties_and_bias():
    """Reverse direction of S5: oracle-made logits (with exact ties, +-0) go INTO the GPU top-k."""
    T, E, k = 333, 40, 4
    rng = np.random.default_rng(3)
    L = rng.standard_normal((T, E)).astype(np.float32)
    L[0] = 0.5                       # all equal -> experts 0..k-1
    L[1] = np.round(L[1])            # many duplicates
    L[2, :4] = [0.0, -0.0, 0.0, -0.0]
    L[2, 4:] = -1.0
    L[3, ::2] = L[3, 1::2]           # pairwise ties
    cfg = wl.small_config(T=T, d=64, E=E, k=k, f=64, index=12)
    lay, g, layer = make(cfg)
    r = layer.route(None, logits_in=torch.from_numpy(L).cuda())
    assert torch.equal(r["logits"].cpu(), torch.from_numpy(L))
    o_idx, *_ = check_routing_against_oracle(r["logits"], r["idx"], r["w"], r["counts"], r["offsets"], None, None,
                                             E, k)
    assert o_idx[0].tolist() == [0, 1, 2, 3] and o_idx[2].tolist() == [0, 1, 2, 3]
    # Zipf-style bias (reading S7): used for selection and gates
    b = torch.linspace(-3, 0, E)
    layer.set_weights(g["W_r"], b.cuda(), g["W_gate"], g["W_up"], g["W_down"])
    r = layer.route(g["hidden"])
    Lref = oracle.router_logits(lay["hidden"], lay["W_r"], b)
    assert np.all(np.abs(r["logits"].cpu().numpy() - Lref) <= 1e-4 * np.maximum(1.0, np.abs(Lref)))
    check_routing_against_oracle(r["logits"], r["idx"], r["w"], r["counts"], r["offsets"], None, None, E, k)


@pytest.mark.parametrize("T,E,k", [(300, 5, 4), (129, 8, 8), (1000, 200, 8), (77, 3, 3), (513, 256, 2), (64, 1, 1)])
def test_permute_accepts_duplicate_experts_in_a_token(T, E, k):
    """bg_moe_permute sorts ANY caller-supplied index list (include/bg_moe.h): a token may name one expert in
    several slots.  Each entry must get its own row, lower slot first -- the plain stable counting sort of the
    oracle -- and the gathered rows must follow."""
    rng = np.random.default_rng(100 + T)
    idx = rng.integers(0, E, size=(T, k)).astype(np.int32)
    idx[0, :] = idx[0, 0]                        # one token, the same expert in every slot
    if T > 130:
        idx[127, :2] = idx[128, :2] = 0          # duplicates on both sides of a tile boundary
    assert k == 1 or any(len(set(r)) < k for r in idx.tolist())
    o_counts, o_offsets, o_rs, o_ip = oracle.hist_scan_perm(idx, E)
    cfg = wl.small_config(T=T, d=64, E=E, k=k, f=64, index=14)
    lay = wl.make_layer(cfg)
    from paper_2606_21712_b200 import MoELayer
    layer = MoELayer(64, 64, E, k, T)
    hidden = lay["hidden"].cuda()
    p = layer.permute(hidden, torch.from_numpy(idx).cuda(), torch.from_numpy(o_offsets).cuda())
    torch.cuda.synchronize()
    rs, ip = p["row_src"].cpu().numpy(), p["inv_perm"].cpu().numpy()
    assert np.array_equal(np.sort(ip), np.arange(T * k)), "inv_perm is not a bijection"
    assert np.array_equal(rs, o_rs) and np.array_equal(ip, o_ip)
    xo = oracle.gather(lay["hidden"], o_rs, k)
    xg = p["x_perm"].view(torch.int16).cpu().numpy().view(np.uint16)
    assert np.array_equal(xg, xo), "gathered rows differ"


def test_one_expert_gets_everything_and_empty_experts():
    T, E, k = 500, 16, 2
    L = np.full((T, E), -5.0, np.float32)
    L[:, 7] = 3.0
    L[:, 9] = 1.0                      # every token -> experts (7, 9); 14 experts empty
    cfg = wl.small_config(T=T, d=64, E=E, k=k, f=64, index=13)
    lay, g, layer = make(cfg)
    r = layer.route(None, logits_in=torch.from_numpy(L).cuda())
    p = layer.permute(g["hidden"], r["idx"], r["offsets"])
    check_routing_against_oracle(r["logits"], r["idx"], r["w"], r["counts"], r["offsets"], p["row_src"],
                                 p["inv_perm"], E, k)
    c = r["counts"].cpu().numpy()
    assert c[7] == T and c[9] == T and c.sum() == 2 * T


FFN_SHAPES = [
    # R rows per expert list, d, f
    ([64] * 8, 512, 1024),             # C1-like: half-filled tiles
    ([128, 256, 130, 1, 0, 127, 129, 3], 256, 384),   # ragged: tails, empty expert, multi-tile
    ([300], 64, 64),                   # minimum d, f; one expert
    ([5, 0, 0, 700, 2], 192, 200),     # f not a multiple of 128, K not a multiple of 64
    ([33, 90], 1024, 136),             # N tail of 8
    ([256, 257, 512, 16, 17, 1, 0, 255, 513], 128, 256),   # token-tile boundaries: 1 / 2 / 3 tiles, 16-row steps
]


@pytest.mark.parametrize("rows,d,f", FFN_SHAPES)
def test_expert_ffn_parity(rows, d, f):
    E = len(rows)
    R = sum(rows)
    cfg = wl.MoEConfig("ffn", 14, T=R, d=d, E=E, k=1, f=f)
    lay, g, layer = make(cfg)
    offsets = np.concatenate([[0], np.cumsum(rows)]).astype(np.int32)
    x = lay["hidden"]                                   # [R, d] rows already "expert-contiguous"
    y = layer.expert_ffn(g["hidden"], torch.from_numpy(offsets).cuda(), T=R)
    torch.cuda.synchronize()
    ref = oracle.expert_ffn(x, offsets, lay["W_gate"], lay["W_up"], lay["W_down"])
    m, l2 = check_out(y, ref, f"expert_ffn rows={rows} d={d} f={f}")
    # per-expert check too: a wrong expert's weights would still pass a global norm only by luck
    for e in range(E):
        if rows[e]:
            check_out(y[offsets[e]:offsets[e + 1]], ref[offsets[e]:offsets[e + 1]], f"expert {e}")


@pytest.mark.parametrize("env", [dict(supergroup_token_tiles=2), dict(supergroup_token_tiles=1),
                                 dict(static_tile_feed=True), dict(static_tile_feed=True, supergroup_token_tiles=2)],
                         ids=["supergroups-of-2", "supergroups-of-1", "static-feed", "static-feed-supergroups"])
def test_expert_ffn_scheduler_variants(env):
    """The same FFN through (i) the pair kernel's super-group tile order, which production shapes only
    reach with experts of several thousand rows (forced here on experts of 3-5 token tiles) and (ii) the
    static tile feed (the default is the dynamic ticket feed); both selected through bg_moe_set_debug."""
    rows = [1300, 0, 700, 257, 16, 1, 64, 65]
    d, f = 192, 320
    E, R = len(rows), sum(rows)
    cfg = wl.MoEConfig("ffn-sched", 15, T=R, d=d, E=E, k=1, f=f)
    lay, g, layer = make(cfg)
    layer.set_debug(**env)
    offsets = np.concatenate([[0], np.cumsum(rows)]).astype(np.int32)
    y = layer.expert_ffn(g["hidden"], torch.from_numpy(offsets).cuda(), T=R)
    torch.cuda.synchronize()
    ref = oracle.expert_ffn(lay["hidden"], offsets, lay["W_gate"], lay["W_up"], lay["W_down"])
    check_out(y, ref, f"expert_ffn {env}")
    for e in range(E):
        if rows[e]:
            check_out(y[offsets[e]:offsets[e + 1]], ref[offsets[e]:offsets[e + 1]], f"expert {e} {env}")


def test_expert_ffn_skewed_load():
    """Zipf-like load (config C4's structure at test size): 200 experts of 1..32 rows, a dozen of 1500-2600 rows
    (several token tiles each), mid-size single-tile experts and empty ones, interleaved by expert index."""
    rng = np.random.default_rng(11)
    rows = [0] * 256
    for e in range(0, 200):
        rows[e] = int(rng.integers(1, 33))
    rows[3] = 1; rows[4] = 32; rows[5] = 16; rows[6] = 17; rows[7] = 8; rows[8] = 9; rows[9] = 15
    for e in range(200, 212):
        rows[e] = int(rng.integers(1500, 2600))
    for e in range(212, 230):
        rows[e] = int(rng.integers(33, 257))
    order = rng.permutation(256)
    rows = [rows[i] for i in order]
    d, f = 512, 256
    E, R = len(rows), sum(rows)
    cfg = wl.MoEConfig("ffn-skewed", 16, T=R, d=d, E=E, k=1, f=f)
    lay, g, layer = make(cfg)
    offsets = np.concatenate([[0], np.cumsum(rows)]).astype(np.int32)
    outs = [layer.expert_ffn(g["hidden"], torch.from_numpy(offsets).cuda(), T=R) for _ in range(3)]
    torch.cuda.synchronize()
    assert torch.equal(outs[0], outs[1]) and torch.equal(outs[0], outs[2])     # the tile feed is dynamic: repeat
    ref = oracle.expert_ffn(lay["hidden"], offsets, lay["W_gate"], lay["W_up"], lay["W_down"])
    check_out(outs[0], ref, "expert_ffn skewed")
    for e in range(E):
        if rows[e]:
            check_out(outs[0][offsets[e]:offsets[e + 1]], ref[offsets[e]:offsets[e + 1]], f"expert {e} ({rows[e]} rows)")
    layer.set_debug(static_tile_feed=True)
    assert torch.equal(layer.expert_ffn(g["hidden"], torch.from_numpy(offsets).cuda(), T=R), outs[0])


def test_unpermute_parity():
    T, k, d, E = 257, 3, 136, 7
    rng = np.random.default_rng(4)
    L = rng.standard_normal((T, E)).astype(np.float32)
    idx, w = oracle.topk_gate(L, k)
    _, _, _, inv_perm = oracle.hist_scan_perm(idx, E)
    cfg = wl.small_config(T=T, d=d, E=E, k=k, f=64, index=15)
    lay, g, layer = make(cfg)
    y = (torch.randn(T * k, d, generator=torch.Generator().manual_seed(1)) * 0.3).to(torch.bfloat16)
    out = layer.unpermute(y.cuda(), torch.from_numpy(inv_perm).cuda(), torch.from_numpy(w).cuda())
    ref = oracle.unpermute(y.to(torch.float64).numpy(), inv_perm, w)
    got = out.to(torch.float64).cpu().numpy()
    # only the final RNE to bf16 (2^-9 relative) plus fp32 summation noise
    assert np.all(np.abs(got - ref) <= 2.0**-8 * np.abs(ref) + 1e-6)


FUSED_SHAPES = [
    wl.C1,
    wl.small_config(T=1, d=64, E=4, k=2, f=64, index=21, name="T1"),
    wl.small_config(T=127, d=128, E=8, k=2, f=256, index=22, name="T127"),
    wl.small_config(T=129, d=256, E=5, k=5, f=192, index=23, name="k=E"),
    wl.small_config(T=384, d=512, E=1, k=1, f=512, index=24, name="dense"),
    wl.small_config(T=600, d=256, E=130, k=8, f=128, index=25, name="E130"),
    wl.small_config(T=96, d=320, E=256, k=8, f=200, index=26, name="E256-sparse"),
]


@pytest.mark.parametrize("cfg", FUSED_SHAPES, ids=lambda c: c.name)
def test_fused_forward_parity(cfg):
    lay, g, layer = make(cfg)
    n0 = layer.launch_count
    out = layer.combined_forward(g["hidden"])
    torch.cuda.synchronize()
    assert layer.launch_count - n0 == 5          # fused router, gather (+ permutation), 2 GEMMs, reduce
    v = layer.debug_views(cfg.T)
    check_routing_against_oracle(v["logits"], v["idx"], v["w"], v["counts"], v["offsets"], v["row_src"],
                                 v["inv_perm"], cfg.E, cfg.k)
    # expert outputs: oracle routed by the GPU's logits (reading S5), fp64, no intermediate rounding
    ref = oracle.forward_batched(lay["hidden"], lay["W_r"], lay["b_r"], lay["W_gate"], lay["W_up"], lay["W_down"],
                                 cfg.k, logits_in=v["logits"].cpu().numpy())
    m, l2 = check_out(out, ref["out"], cfg.name)
    # and the oracle's own logits agree with the GPU's
    own = oracle.router_logits(lay["hidden"], lay["W_r"], lay["b_r"])
    assert np.all(np.abs(v["logits"].cpu().numpy() - own) <= 1e-4 * np.maximum(1.0, np.abs(own)))


def test_fused_equals_split_and_is_deterministic():
    cfg = wl.small_config(T=700, d=256, E=12, k=3, f=320, index=27)
    lay, g, layer = make(cfg)
    out1 = layer.combined_forward(g["hidden"])
    out2 = layer.combined_forward(g["hidden"])
    assert torch.equal(out1, out2), "fused path is not bitwise deterministic run to run"
    r = layer.route(g["hidden"])
    p = layer.permute(g["hidden"], r["idx"], r["offsets"])
    y = layer.expert_ffn(p["x_perm"], r["offsets"])
    out_split = layer.unpermute(y, p["inv_perm"], r["w"])
    torch.cuda.synchronize()
    ref = oracle.forward_batched(lay["hidden"], lay["W_r"], None, lay["W_gate"], lay["W_up"], lay["W_down"], cfg.k,
                                 logits_in=r["logits"].cpu().numpy())["out"]
    check_out(out_split, ref, "split")
    check_out(out1, ref, "fused")
    # the two differ only in where the gate weight is applied (before vs after Y's bf16 rounding)
    a, b = out1.float(), out_split.float()
    assert (a - b).abs().max().item() <= 2e-2 * b.abs().max().item()


def test_combine_invariance_on_gpu():
    """forward(concat(S1,S2)) == concat(forward(S1), forward(S2)), row for row."""
    cfg = wl.small_config(T=300, d=128, E=8, k=2, f=128, index=28)
    lay, g, layer = make(cfg)
    h = g["hidden"]
    full = layer.combined_forward(h).clone()
    a = layer.combined_forward(h[:111].contiguous()).clone()
    b = layer.combined_forward(h[111:].contiguous()).clone()
    assert torch.equal(torch.cat([a, b]), full), "per-row results depend on what the row was combined with"
    perm = torch.randperm(300, generator=torch.Generator().manual_seed(2)).cuda()
    shuf = layer.combined_forward(h[perm].contiguous())
    assert torch.equal(shuf, full[perm])


@pytest.mark.parametrize("d,E,k", [(2048, 128, 8), (4096, 16, 2), (7168, 256, 8)], ids=["d2048", "d4096", "d7168"])
def test_combine_invariance_large_d(d, E, k):
    """the router's K partition (cluster of router_nch(d) CTAs, partials added in chunk order) is a
    function of d only, so the fp32 logits of a row -- and everything downstream -- cannot depend on how many
    tokens it was combined with.  T=4096 against its two halves and against single 128-token tiles, at the d of
    C3 / C2,C5 / C4 (2 / 4 / 4 K chunks: router_nch caps at 4)."""
    cfg = wl.small_config(T=4096, d=d, E=E, k=k, f=128, index=33)
    lay, g, layer = make(cfg)
    h = g["hidden"]
    full = layer.combined_forward(h).clone()
    L_full = layer.debug_views(4096)["logits"].clone()
    outs, Ls = [], []
    for lo, hi in ((0, 2048), (2048, 4096)):
        outs.append(layer.combined_forward(h[lo:hi].contiguous()).clone())
        Ls.append(layer.debug_views(hi - lo)["logits"].clone())
    assert torch.equal(torch.cat(Ls), L_full), "router logits depend on the combined-batch size"
    assert torch.equal(torch.cat(outs), full), "outputs depend on the combined-batch size"
    for lo, hi in ((0, 1), (130, 257), (4000, 4096)):
        o = layer.combined_forward(h[lo:hi].contiguous())
        assert torch.equal(layer.debug_views(hi - lo)["logits"], L_full[lo:hi])
        assert torch.equal(o, full[lo:hi])
    own = oracle.router_logits(lay["hidden"], lay["W_r"], lay["b_r"])
    assert np.all(np.abs(L_full.cpu().numpy() - own) <= 1e-4 * np.maximum(1.0, np.abs(own)))


@pytest.mark.parametrize("T,d,E,k", [(1000, 2048, 128, 8), (333, 4096, 8, 2), (700, 1024, 64, 6), (130, 2048, 33, 3),
                                     (19000, 2048, 128, 8)])
def test_router_forms_are_bit_identical(T, d, E, k):
    """The router's cluster form (K chunks on the CTAs of a cluster, partials reduced through DSMEM) and its
    sequential form (one CTA, one TMEM accumulator per chunk) add the same partial sums in the same order:
    logits, indices, gates and every routing table must agree bit for bit, and match the oracle."""
    cfg = wl.small_config(T=T, d=d, E=E, k=k, f=64, index=36)
    lay, g, layer = make(cfg)
    res = {}
    for form in (1, 2):
        layer.set_debug(router_form=form)
        r = layer.route(g["hidden"])
        p = layer.permute(g["hidden"], r["idx"], r["offsets"], gather=False)
        res[form] = {**r, **{kk: p[kk] for kk in ("row_src", "inv_perm")}}
    for key in ("logits", "idx", "w", "counts", "offsets", "row_src", "inv_perm"):
        assert torch.equal(res[1][key], res[2][key]), f"{key} differs between the router forms"
    r = res[1]
    check_routing_against_oracle(r["logits"], r["idx"], r["w"], r["counts"], r["offsets"], r["row_src"],
                                 r["inv_perm"], E, k)
    own = oracle.router_logits(lay["hidden"], lay["W_r"], lay["b_r"])
    assert np.all(np.abs(r["logits"].cpu().numpy() - own) <= 1e-4 * np.maximum(1.0, np.abs(own)))


def test_host_entry_point_and_zero_tokens():
    cfg = wl.small_config(T=200, d=128, E=8, k=2, f=128, index=29)
    lay, g, layer = make(cfg)
    dev_out = layer.combined_forward(g["hidden"])
    h_pinned = lay["hidden"].pin_memory()     # referenced until the upload is done (include/bg_moe.h: lifetime rule)
    host_out = layer.combined_forward_host(h_pinned)
    layer.host_input_sync()                   # the upload is finished: the input may be overwritten ...
    h_pinned.zero_()
    torch.cuda.synchronize()
    assert torch.equal(host_out, dev_out.cpu())   # ... without touching the result
    # pipelined back-to-back host calls with different inputs and sizes (two staging slots, the context's own
    # copy / compute streams): every result must equal the device-pointer path on the same rows
    gen = torch.Generator().manual_seed(5)
    ins, outs, refs = [], [], []
    for i in range(7):
        T = [200, 64, 200, 1, 129, 200, 37][i]
        hi = (torch.randn(T, cfg.d, generator=gen) * (1 + i)).to(torch.bfloat16).pin_memory()
        ins.append(hi)
        outs.append(layer.combined_forward_host(hi))
    torch.cuda.current_stream().synchronize()          # the caller's stream waited for every download
    for hi, ho in zip(ins, outs):
        refs.append(layer.combined_forward(hi.cuda()).cpu())
    for i, (ho, r) in enumerate(zip(outs, refs)):
        assert torch.equal(ho, r), f"host call {i} differs from the device-pointer path"
    # a device-pointer call right after host calls (and the reverse) is ordered correctly
    a = layer.combined_forward_host(ins[0])
    b = layer.combined_forward(g["hidden"])
    c = layer.combined_forward_host(ins[2])
    torch.cuda.synchronize()
    assert torch.equal(a, refs[0]) and torch.equal(b, dev_out) and torch.equal(c, refs[2])
    empty = torch.empty(0, cfg.d, dtype=torch.bfloat16, device="cuda")
    assert layer.combined_forward(empty).shape == (0, cfg.d)          # T == 0: BG_OK, no-op
    r = layer.route(empty)
    assert r["counts"].sum().item() == 0 and r["offsets"].abs().sum().item() == 0


def test_argument_errors():
    from paper_2606_21712_b200 import MoELayer, BgMoeError, BG_ERR_INVALID_ARG, BG_ERR_UNSUPPORTED, BG_ERR_NO_WEIGHTS
    with pytest.raises(BgMoeError) as ei:
        MoELayer(512, 1024, 300, 2, 16)          # E > 256
    assert ei.value.status == BG_ERR_UNSUPPORTED
    with pytest.raises(BgMoeError) as ei:
        MoELayer(512, 1024, 8, 9, 16)            # k > E
    assert ei.value.status == BG_ERR_INVALID_ARG
    with pytest.raises(BgMoeError) as ei:
        MoELayer(100, 1024, 8, 2, 16)            # d not a multiple of 8
    assert ei.value.status == BG_ERR_INVALID_ARG
    layer = MoELayer(64, 64, 4, 2, 16)
    h = torch.zeros(32, 64, dtype=torch.bfloat16, device="cuda")
    with pytest.raises(BgMoeError) as ei:
        layer.combined_forward(h[:8].contiguous())   # weights not set
    assert ei.value.status == BG_ERR_NO_WEIGHTS
    cfg = wl.small_config(T=16, d=64, E=4, k=2, f=64, index=30)
    g = to_dev(wl.make_layer(cfg))
    layer.set_weights(g["W_r"], None, g["W_gate"], g["W_up"], g["W_down"])
    with pytest.raises(BgMoeError) as ei:
        layer.combined_forward(h)                # T > max_tokens
    assert ei.value.status == BG_ERR_INVALID_ARG


def test_context_survives_failed_and_degenerate_calls():
    """the tile-feed and tiles-done counters must be zero at every launch whatever the
    previous calls did.  The fused router's last tile zeroes the GEMM ticket counters, the split FFN zeroes
    them on the stream, and a CUDA failure marks the context so that the next call re-zeroes everything.  Here:
    rejected calls (T > max_tokens, misaligned pointer), a split FFN that draws zero tiles (all experts empty) and
    one with fewer tiles than clusters, interleaved with fused calls that must stay bit-identical."""
    from paper_2606_21712_b200 import BgMoeError
    cfg = wl.small_config(T=300, d=256, E=12, k=3, f=192, index=34)
    lay, g, layer = make(cfg)
    first = layer.combined_forward(g["hidden"]).clone()
    x = torch.zeros(cfg.T * cfg.k + 8, cfg.d, dtype=torch.bfloat16, device="cuda")
    empty_off = torch.zeros(cfg.E + 1, dtype=torch.int32, device="cuda")     # all experts empty: zero tiles drawn
    layer.expert_ffn(x[:cfg.T * cfg.k], empty_off, T=cfg.T)
    assert torch.equal(layer.combined_forward(g["hidden"]), first)
    with pytest.raises(BgMoeError):
        layer.combined_forward(torch.zeros(cfg.T + 1, cfg.d, dtype=torch.bfloat16, device="cuda"))   # T > max_tokens
    with pytest.raises(BgMoeError):
        layer.expert_ffn(x.view(-1)[4:4 + cfg.T * cfg.k * cfg.d].view(cfg.T * cfg.k, cfg.d), empty_off, T=cfg.T)  # 8-byte aligned
    one_off = torch.zeros(cfg.E + 1, dtype=torch.int32, device="cuda")
    one_off[3:] = 5                                                          # one expert, 5 rows: 1-2 tiles
    layer.expert_ffn(x[:cfg.T * cfg.k], one_off, T=cfg.T)
    for _ in range(3):
        assert torch.equal(layer.combined_forward(g["hidden"]), first)
    torch.cuda.synchronize()


def test_non_finite_logits_are_memory_safe():
    """Reading S4: non-finite logits are out of contract; the routing kernels must still produce in-range, distinct
    expert indices and a valid permutation (memory safety), whatever the values."""
    T, E, k = 257, 40, 4
    rng = np.random.default_rng(8)
    L = rng.standard_normal((T, E)).astype(np.float32)
    L[0, :] = -np.inf
    L[1, ::3] = np.inf
    L[2, 5] = np.nan
    L[3, :] = np.nan
    L[4, :10] = -np.inf
    cfg = wl.small_config(T=T, d=64, E=E, k=k, f=64, index=35)
    lay, g, layer = make(cfg)
    r = layer.route(None, logits_in=torch.from_numpy(L).cuda())
    idx = r["idx"].cpu().numpy()
    assert idx.min() >= 0 and idx.max() < E
    assert all(len(set(row)) == k for row in idx.tolist())
    p = layer.permute(g["hidden"], r["idx"], r["offsets"])
    rs = p["row_src"].cpu().numpy()
    assert np.array_equal(np.sort(rs), np.arange(T * k))
    assert r["counts"].sum().item() == T * k
    # rows without non-finite entries still match the oracle bit for bit
    fin = np.isfinite(L).all(axis=1)
    o_idx, _ = oracle.topk_gate(L[fin], k)
    assert np.array_equal(idx[fin], o_idx)


@pytest.mark.parametrize("ring_experts", [2, 4, 6, 16], ids=lambda r: f"ring{r}")
def test_offloaded_weights_ring_buffer_equals_resident(ring_experts):
    """SURVEY §8(f)-4 / PAPER.md:317-325: expert weights in pinned host memory, streamed through a device ring of
    `ring_experts` slots (two halves) while the grouped GEMMs run.  The result must be bit-identical to the
    resident path (same kernels, the experts merely arrive in chunks) and match the oracle; chunk sizes 1, 2, 3
    (11 experts: a ragged last chunk) and a ring larger than the layer; repeated calls reuse the ring halves."""
    cfg = wl.small_config(T=600, d=256, E=11, k=3, f=192, index=37)
    lay, g, layer = make(cfg)
    ref = layer.combined_forward(g["hidden"]).clone()
    h2 = g["hidden"].flip(0).contiguous()
    ref2 = layer.combined_forward(h2).clone()
    pinned = [lay[n].pin_memory() for n in ("W_gate", "W_up", "W_down")]
    layer.set_weights_offloaded(g["W_r"], g["b_r"], *pinned, ring_experts=ring_experts)
    a = layer.combined_forward(g["hidden"]).clone()
    b = layer.combined_forward(h2).clone()
    c = layer.combined_forward(g["hidden"]).clone()
    torch.cuda.synchronize()
    assert layer.ring_bytes_per_call == 6 * cfg.d * cfg.f * cfg.E * 2 // 2
    assert torch.equal(a, ref) and torch.equal(b, ref2) and torch.equal(c, ref)
    L = layer.debug_views(cfg.T)["logits"].cpu().numpy()
    o = oracle.forward_batched(lay["hidden"], lay["W_r"], lay["b_r"], lay["W_gate"], lay["W_up"], lay["W_down"], cfg.k,
                               logits_in=L)["out"]
    check_out(c, o, f"ring of {ring_experts}")
    # host entry point and zero-copy segments ride the same ring
    h_pinned = lay["hidden"].pin_memory()     # kept referenced until the synchronize below
    host_out = layer.combined_forward_host(h_pinned)
    segs = [g["hidden"][:100].clone(), g["hidden"][100:].clone()]
    outs = layer.combined_forward_segments(segs)
    torch.cuda.synchronize()
    assert torch.equal(host_out, ref.cpu()) and torch.equal(torch.cat(outs), ref)
    # back to resident weights on the same context
    layer.set_weights(g["W_r"], g["b_r"], g["W_gate"], g["W_up"], g["W_down"])
    assert torch.equal(layer.combined_forward(g["hidden"]), ref)


@pytest.mark.parametrize("ring_experts", [2, 6, 32])
def test_ring_buffer_skips_experts_without_rows(ring_experts):
    """bg_moe_set_ring_skip_empty: on a skewed layer -- a router bias that starves most
    experts, as BASELINE config C4's Zipf bias does -- only the experts that received rows are copied into the ring
    (the byte counter says exactly which), whole chunks of empty experts are skipped, and the result keeps the bits
    of the resident path; switching the option off copies everything again."""
    cfg = wl.small_config(T=500, d=256, E=19, k=2, f=192, index=38)
    lay, g, layer = make(cfg)
    b = torch.full((cfg.E,), -40.0)
    live = [0, 1, 5, 6, 7, 13, 18]                       # runs of 2, 3, 1, 1 experts; chunks of 3 / 16 with none at all
    b[live] = 0.0
    layer.set_weights(g["W_r"], b.cuda(), g["W_gate"], g["W_up"], g["W_down"])
    ref = layer.combined_forward(g["hidden"]).clone()
    counts = layer.debug_views(cfg.T)["counts"].cpu().numpy()
    assert set(np.nonzero(counts)[0].tolist()) <= set(live) and (counts == 0).sum() >= cfg.E - len(live)
    n_live = int((counts > 0).sum())
    pinned = [lay[n].pin_memory() for n in ("W_gate", "W_up", "W_down")]
    layer.set_weights_offloaded(g["W_r"], b.cuda(), *pinned, ring_experts=ring_experts)
    per_expert = 6 * cfg.d * cfg.f
    a = layer.combined_forward(g["hidden"]).clone()
    torch.cuda.synchronize()
    assert layer.ring_bytes_per_call == per_expert * cfg.E and torch.equal(a, ref)      # default: every expert
    layer.set_ring_skip_empty(True)
    h2 = g["hidden"].flip(0).contiguous()
    for x in (g["hidden"], h2, g["hidden"]):
        got = layer.combined_forward(x).clone()
        torch.cuda.synchronize()
        c = layer.debug_views(cfg.T)["counts"].cpu().numpy()
        assert layer.ring_bytes_per_call == per_expert * int((c > 0).sum()), "copied bytes != non-empty experts"
        if x is g["hidden"]:
            assert torch.equal(got, ref), "skip-empty ring differs from the resident path"
    assert layer.ring_bytes_per_call == per_expert * n_live
    # segments and the host entry point ride the same path
    segs = [g["hidden"][:77].clone(), g["hidden"][77:].clone()]
    outs = layer.combined_forward_segments(segs)
    h_pinned = lay["hidden"].pin_memory()
    host_out = layer.combined_forward_host(h_pinned)
    torch.cuda.synchronize()
    assert torch.equal(torch.cat(outs), ref) and torch.equal(host_out, ref.cpu())
    layer.set_ring_skip_empty(False)
    assert torch.equal(layer.combined_forward(g["hidden"]), ref)
    torch.cuda.synchronize()
    assert layer.ring_bytes_per_call == per_expert * cfg.E
    L = layer.debug_views(cfg.T)["logits"].cpu().numpy()
    o = oracle.forward_batched(lay["hidden"], lay["W_r"], b, lay["W_gate"], lay["W_up"], lay["W_down"], cfg.k,
                               logits_in=L)["out"]
    check_out(ref, o, "skewed layer")


def test_failed_ring_allocation_leaves_no_half_state():
    """A bg_moe_set_weights_offloaded call that cannot get its ring must leave the context either as it was
    (resident weights) or without weights (BG_ERR_NO_WEIGHTS from the next forward) -- never with a freed ring and
    the old chunk size.  The impossible request is a ring of 2 x 256 experts of 3 x 268 MB (~412 GB); the host
    pointers are never read because no forward succeeds while they are installed... except the small first ring,
    which is only installed, not run."""
    import ctypes
    from paper_2606_21712_b200 import MoELayer, BgMoeError, BG_ERR_NO_WEIGHTS, BG_ERR_NOMEM
    d, f, E, k = 8192, 16384, 256, 2
    layer = MoELayer(d, f, E, k, 8)
    W_r = torch.zeros(d, E, device="cuda")
    fake = torch.zeros(64, dtype=torch.uint8).pin_memory()          # stands for three 69 GB host tensors: never read
    hp = ctypes.c_void_p(fake.data_ptr())
    st = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    call = lambda ring: layer.lib.bg_moe_set_weights_offloaded(layer._ctx, ctypes.c_void_p(W_r.data_ptr()), None, hp, hp,
                                                               hp, ring, st)
    assert call(2) == 0                                             # 1.6 GB ring: fits
    assert call(512) == BG_ERR_NOMEM                                # 2 x 256 experts: cannot fit
    x = torch.zeros(8, d, dtype=torch.bfloat16, device="cuda")
    with pytest.raises(BgMoeError) as ei:
        layer.combined_forward(x)
    assert ei.value.status == BG_ERR_NO_WEIGHTS
    torch.cuda.synchronize()
    layer.close()
    # resident weights survive a failed switch to a ring
    cfg = wl.small_config(T=100, d=128, E=8, k=2, f=128, index=41)
    lay, g, small = make(cfg)
    ref = small.combined_forward(g["hidden"]).clone()
    rc = small.lib.bg_moe_set_weights_offloaded(small._ctx, ctypes.c_void_p(g["W_r"].data_ptr()), None, hp, hp, hp, 1, st)
    assert rc == -1                                                 # odd ring: refused, nothing touched
    assert torch.equal(small.combined_forward(g["hidden"]), ref)


def test_planned_workspace_equals_allocated_workspace():
    """bg_moe_workspace_bytes_for (host-only planner) must predict what bg_moe_create allocates."""
    import paper_2606_21712_b200 as pk
    for (d, f, E, k, T) in [(512, 1024, 8, 2, 256), (2048, 768, 128, 8, 4096), (192, 200, 5, 5, 1000)]:
        layer = pk.MoELayer(d, f, E, k, T)
        assert layer.lib.bg_moe_workspace_bytes(layer._ctx) == pk.workspace_bytes_for(d, f, E, k, T)
        layer.close()


@pytest.mark.parametrize("lengths", [
    [256],                                   # one segment = the contiguous case
    [16] * 16,                               # C1's 16 coroutines x 16 tokens
    [100, 0, 1, 1, 1, 57, 0, 96],            # ragged, single-token (decode) and empty segments
    [1] * 256,                               # every token its own coroutine
    [130, 126],                              # a boundary inside a 128-token router tile, off the 8-row grid
], ids=["one", "16x16", "ragged", "all-decode", "straddle"])
def test_zero_copy_segments_equal_the_concatenation(lengths):
    """bg_moe_combined_forward_segments: COMBINE = concatenation, so the
    segment path must give bit-identical routing artefacts and outputs to the fused call on the concatenated
    tensor, and that result is checked against the oracle."""
    cfg = wl.C1
    assert sum(lengths) == cfg.T
    lay, g, layer = make(cfg)
    ref_out = layer.combined_forward(g["hidden"]).clone()
    v0 = {k: x.clone() for k, x in layer.debug_views(cfg.T).items()}
    torch.cuda.synchronize()
    # every segment in its own allocation (not views of one buffer), in list order
    segs, pos = [], 0
    for n in lengths:
        segs.append(g["hidden"][pos:pos + n].clone())
        pos += n
    n0 = layer.launch_count
    outs = layer.combined_forward_segments(segs)
    torch.cuda.synchronize()
    assert layer.launch_count - n0 == 5
    v1 = layer.debug_views(cfg.T)
    for key in ("logits", "idx", "w", "counts", "offsets", "row_src", "inv_perm"):
        assert torch.equal(v0[key], v1[key]), key
    got = torch.cat(outs, dim=0)
    assert torch.equal(got, ref_out), "segment path differs from the concatenated path"
    L = v1["logits"].cpu().numpy()
    ref = oracle.forward_batched(lay["hidden"], lay["W_r"], lay["b_r"], lay["W_gate"], lay["W_up"], lay["W_down"],
                                 cfg.k, logits_in=L)["out"]
    check_out(got, ref, f"segments {lengths[:4]}...")


@pytest.mark.parametrize("router_form", [1, 2], ids=["sequential", "cluster"])
@pytest.mark.parametrize("T,d,E,k", [(700, 2048, 128, 8), (333, 4096, 8, 2), (600, 7168, 256, 8), (1500, 1024, 40, 4)])
def test_zero_copy_segments_large_d_both_router_forms(T, d, E, k, router_form):
    """The segment path where the router splits K over several chunks (d >= 1024: router_nch(d) = 2 or 4), in BOTH
    router forms -- the cluster form with its DSMEM reduce-scatter and the sequential form with one TMEM accumulator
    per chunk read their token rows through the segment table here (C1's d = 512 has one chunk).
    Segments: a boundary inside a 128-token router tile and off the 8-row grid, empty segments, single-token
    (decode) segments, ragged tails.  Bit-identical to the concatenated call on every routing artefact and on the
    output, and that output against the oracle."""
    lengths = [130, 0, 1, 1, 57, 0]
    rest = T - sum(lengths)
    lengths += [rest // 2 + 3, 0, rest - rest // 2 - 3]
    assert sum(lengths) == T and min(lengths) == 0
    cfg = wl.small_config(T=T, d=d, E=E, k=k, f=128, index=60 + E % 7)
    lay, g, layer = make(cfg)
    layer.set_debug(router_form=router_form)
    ref_out = layer.combined_forward(g["hidden"]).clone()
    v0 = {kk: x.clone() for kk, x in layer.debug_views(T).items()}
    torch.cuda.synchronize()
    segs, pos = [], 0
    for n in lengths:
        segs.append(g["hidden"][pos:pos + n].clone())      # every segment in its own allocation
        pos += n
    outs = layer.combined_forward_segments(segs)
    torch.cuda.synchronize()
    v1 = layer.debug_views(T)
    for key in ("logits", "idx", "w", "counts", "offsets", "row_src", "inv_perm"):
        assert torch.equal(v0[key], v1[key]), key
    got = torch.cat(outs, dim=0)
    assert torch.equal(got, ref_out), "segment path differs from the concatenated path"
    L = v1["logits"].cpu().numpy()
    own = oracle.router_logits(lay["hidden"], lay["W_r"], lay["b_r"])
    assert np.all(np.abs(L - own) <= 1e-4 * np.maximum(1.0, np.abs(own)))
    check_routing_against_oracle(v1["logits"], v1["idx"], v1["w"], v1["counts"], v1["offsets"], v1["row_src"],
                                 v1["inv_perm"], E, k)
    ref = oracle.forward_batched(lay["hidden"], lay["W_r"], lay["b_r"], lay["W_gate"], lay["W_up"], lay["W_down"],
                                 k, logits_in=L)["out"]
    check_out(got, ref, f"segments d={d} form={router_form}")


@pytest.mark.parametrize("precision", [1, 2])
def test_fp8_through_segments_and_host_entry_points(precision):
    """The FP8 path through the other two fused entry points: the quantising gather has its own
    segment-table branch and the host pipeline runs the same chain on its own streams -- both must give the bits of
    the device-pointer FP8 call."""
    cfg = wl.small_config(T=700, d=256, E=12, k=3, f=256, index=66)
    lay, g, layer = make(cfg)
    bf16_out = layer.combined_forward(g["hidden"]).clone()
    layer.set_precision(precision)
    ref = layer.combined_forward(g["hidden"]).clone()
    assert not torch.equal(ref, bf16_out)
    lengths = [130, 0, 1, 1, 57, 0, 300, 211]
    segs, pos = [], 0
    for n in lengths:
        segs.append(g["hidden"][pos:pos + n].clone())
        pos += n
    outs = layer.combined_forward_segments(segs)
    h_pinned = lay["hidden"].pin_memory()
    host_out = layer.combined_forward_host(h_pinned)
    torch.cuda.synchronize()
    assert torch.equal(torch.cat(outs), ref), "FP8 segments differ from the FP8 device-pointer call"
    assert torch.equal(host_out, ref.cpu()), "FP8 host entry point differs from the FP8 device-pointer call"


def test_zero_copy_segments_argument_errors_and_empty_batch():
    import ctypes
    from paper_2606_21712_b200.binding import BgMoeSegment, BG_ERR_INVALID_ARG
    cfg = wl.C1
    lay, g, layer = make(cfg)
    assert layer.combined_forward_segments([]) == []                      # no segments: BG_OK, nothing launched
    empty = torch.empty(0, cfg.d, dtype=torch.bfloat16, device="cuda")
    n0 = layer.launch_count
    layer.combined_forward_segments([empty, empty])
    assert layer.launch_count == n0
    too_many = [g["hidden"], g["hidden"][:1].clone()]                     # T + 1 tokens > max_tokens
    with pytest.raises(Exception) as e:
        layer.combined_forward_segments(too_many)
    assert getattr(e.value, "status", None) == BG_ERR_INVALID_ARG


def _guarded(rows, cols, dtype=torch.bfloat16, guard=8):
    """A [rows, cols] view in the middle of a larger buffer whose other rows hold a sentinel."""
    full = torch.full((rows + 2 * guard, cols), 123.0, dtype=dtype, device="cuda")
    return full, full[guard:guard + rows], guard


def _guards_intact(full, rows, guard):
    return bool((full[:guard] == 123.0).all()) and bool((full[guard + rows:] == 123.0).all())


def test_no_writes_outside_the_output_buffers():
    """Bounds check of our own (compute-sanitizer is not available on the GPU pool): every caller-owned
    output sits between sentinel rows; ragged experts, a ragged last router tile and a column count that is
    not a multiple of 64 exercise the masked stores of both GEMM epilogues, the gather and the un-permute."""
    import ctypes
    from paper_2606_21712_b200.binding import _ptr, _stream
    cfg = wl.small_config(T=333, d=200, E=7, k=3, f=136, index=21)
    lay, g, layer = make(cfg)
    T, R = cfg.T, cfg.T * cfg.k
    # fused call
    full_o, out, gd = _guarded(T, cfg.d)
    layer.combined_forward(g["hidden"], out)
    torch.cuda.synchronize()
    assert _guards_intact(full_o, T, gd)
    ref = layer.combined_forward(g["hidden"]).clone()
    assert torch.equal(out, ref)
    # split calls on guarded buffers
    r = layer.route(g["hidden"])
    full_x, x_perm, _ = _guarded(R, cfg.d)
    full_rs = torch.full((R + 16,), -77, dtype=torch.int32, device="cuda")
    full_ip = torch.full((R + 16,), -77, dtype=torch.int32, device="cuda")
    layer._check(layer.lib.bg_moe_permute(layer._ctx, _ptr(g["hidden"]), T, _ptr(r["idx"]), _ptr(r["offsets"]),
                                          _ptr(full_rs[8:8 + R]), _ptr(full_ip[8:8 + R]), _ptr(x_perm), _stream(None)))
    full_y, y_perm, _ = _guarded(R, cfg.d)
    layer._check(layer.lib.bg_moe_expert_ffn(layer._ctx, _ptr(x_perm), _ptr(r["offsets"]), T, _ptr(y_perm), _stream(None)))
    full_o2, out2, _ = _guarded(T, cfg.d)
    layer._check(layer.lib.bg_moe_unpermute(layer._ctx, _ptr(y_perm), _ptr(full_ip[8:8 + R]), _ptr(r["w"]), T,
                                            _ptr(out2), _stream(None)))
    torch.cuda.synchronize()
    assert _guards_intact(full_x, R, gd) and _guards_intact(full_y, R, gd) and _guards_intact(full_o2, T, gd)
    for t_ in (full_rs, full_ip):
        assert bool((t_[:8] == -77).all()) and bool((t_[8 + R:] == -77).all())
    # zero-copy segments: each coroutine's output between its own sentinels
    lengths = [100, 1, 0, 232]
    segs, outs, fulls, pos = [], [], [], 0
    for n in lengths:
        segs.append(g["hidden"][pos:pos + n].clone())
        full, view, _ = _guarded(n, cfg.d)
        fulls.append(full)
        outs.append(view)
        pos += n
    layer.combined_forward_segments(segs, outs)
    torch.cuda.synchronize()
    assert all(_guards_intact(f_, n, gd) for f_, n in zip(fulls, lengths))
    assert torch.equal(torch.cat(outs, 0), ref)


def test_dynamic_tile_feed_rearms_across_many_launches():
    """The pair GEMMs draw tiles from ticket counters that the last cluster of a launch re-arms.  Many
    back-to-back launches with changing token counts (hence changing tile counts, including fewer tiles than
    clusters) must neither hang nor change results: every call is compared bit for bit with the first result
    for that token count."""
    cfg = wl.small_config(T=700, d=256, E=16, k=4, f=192, index=31)
    lay, g, layer = make(cfg)
    first = {}
    rng = np.random.default_rng(0)
    for it in range(120):
        T = int(rng.choice([1, 3, 64, 129, 300, 700]))
        out = layer.combined_forward(g["hidden"][:T].contiguous())
        if it % 10 == 9:
            torch.cuda.synchronize()
        if T in first:
            assert torch.equal(out, first[T]), f"launch {it}, T={T}: result changed"
        else:
            first[T] = out.clone()
    last = layer.combined_forward(g["hidden"])            # T = 700 once more: its logits feed the oracle
    torch.cuda.synchronize()
    assert torch.equal(last, first[700])
    L = layer.debug_views(700)["logits"].cpu().numpy()
    ref = oracle.forward_batched(lay["hidden"], lay["W_r"], lay["b_r"], lay["W_gate"], lay["W_up"], lay["W_down"],
                                 cfg.k, logits_in=L)["out"]
    check_out(first[700], ref, "T=700 after 120 launches")
