"""GPU test of bg_moe_route_logits_noalloc -- the routing call for users who may not allocate device memory.

Some users of this library cannot call cudaMalloc at all: a serving runtime that has already given every byte of HBM
to pools it manages itself (the paper's runtime does -- KV cache plus ring parameter buffer), or code
on a latency-critical path where cudaMalloc / cudaFree are banned because they serialise with all work in flight on
the device.  For them the library keeps the scratch of this one call (per-tile expert histograms and a tile ticket) in
a fixed array inside its own image, which limits the call to BG_MOE_NOALLOC_MAX_TOKENS = 16384 tokens.

What is checked: the call gives exactly what the ordinary, context-based path gives (bg_moe_route with logits_in;
integers identical, gate weights within the 2e-6 bar of tests/test_gpu_parity.py -- in fact identical), on TWO calls
in a row over different shapes, because every call reuses the same array and finds the previous call's contents in
it; that the outputs are the only memory written; that an oversized T is refused with a message and launches nothing;
and that neither torch's allocator nor the driver is asked for memory during a call.

The file sorts last in pytest's collection order on purpose (`pytest --collect-only`): `pytest -x` stops at the
first failure, and a failure here must not hide the parity tests.  It passes alone in a fresh process and after the
rest of the suite: it depends on no state but the library's own array.
"""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

W_TOL = 2e-6          # gate-weight bar of tests/test_gpu_parity.py


def make_logits(T, E, seed):
    """Seeded fp32 logits with the awkward rows of test_route_logits_in_ties_and_bias: exact ties, +-0."""
    rng = np.random.default_rng(seed)
    L = rng.standard_normal((T, E)).astype(np.float32)
    if T > 3 and E >= 4:
        L[0] = 0.5                       # all equal: experts 0..k-1 in index order
        L[1] = np.round(L[1])            # many duplicates
        L[2, :4] = [0.0, -0.0, 0.0, -0.0]
        L[2, 4:] = -1.0
        if E % 2 == 0:
            L[3, ::2] = L[3, 1::2]       # pairwise ties
    return torch.from_numpy(L).cuda()


def existing_path(L, k):
    """The context-based path: bg_moe_route(ctx, hidden = NULL, logits_in = L)."""
    from paper_2606_21712_b200 import MoELayer
    T, E = L.shape
    layer = MoELayer(64, 64, E, k, max(T, 1))      # d and f play no part in routing from given logits
    r = layer.route(None, logits_in=L, want_logits=False)
    torch.cuda.synchronize()
    layer.close()
    return r


def noalloc_path(L, k, guard=64, check_driver=False):
    """The new call, with every output inside a larger buffer filled with a sentinel: what lies around the outputs
    must come back untouched."""
    from paper_2606_21712_b200 import route_logits_noalloc
    T, E = L.shape
    dev = L.device
    SENT_I, SENT_F = -77, -77.0
    bufs = dict(idx=torch.full((T * k + 2 * guard,), SENT_I, dtype=torch.int32, device=dev),
                w=torch.full((T * k + 2 * guard,), SENT_F, dtype=torch.float32, device=dev),
                counts=torch.full((E + 2 * guard,), SENT_I, dtype=torch.int32, device=dev),
                offsets=torch.full((E + 1 + 2 * guard,), SENT_I, dtype=torch.int32, device=dev))
    view = dict(idx=bufs["idx"][guard:guard + T * k].view(T, k), w=bufs["w"][guard:guard + T * k].view(T, k),
                counts=bufs["counts"][guard:guard + E], offsets=bufs["offsets"][guard:guard + E + 1])
    torch.cuda.synchronize()
    # Two counters that cannot go down behind our back (the bytes torch has in use can: garbage of earlier tests is
    # collected whenever Python likes): the number of allocation requests torch has served, and the free memory the
    # driver reports (torch's caching allocator never hands memory back on a tensor free).
    n_before = torch.cuda.memory_stats(dev)["allocation.all.allocated"]
    free_before = torch.cuda.mem_get_info(dev)[0] if check_driver else None
    route_logits_noalloc(L, k, view["idx"], view["w"], view["counts"], view["offsets"])
    torch.cuda.synchronize()
    assert torch.cuda.memory_stats(dev)["allocation.all.allocated"] == n_before, "the binding allocated through torch"
    if check_driver:      # not on a device's first call: the runtime may still be loading the library's kernels
        assert torch.cuda.mem_get_info(dev)[0] >= free_before, "the call took device memory from the driver"
    for name, b in bufs.items():
        sent = SENT_F if b.dtype == torch.float32 else SENT_I
        assert bool((b[:guard] == sent).all()) and bool((b[-guard:] == sent).all()), f"{name}: wrote outside its output"
    return view


def compare(L, k, check_driver=False):
    T, E = L.shape
    ref = existing_path(L, k)
    got = noalloc_path(L, k, check_driver=check_driver)
    assert torch.equal(got["idx"], ref["idx"]), "topk_idx differs from bg_moe_route"
    if T:
        assert float((got["w"] - ref["w"]).abs().max()) <= W_TOL, "gate weights differ from bg_moe_route"
    assert torch.equal(got["counts"], ref["counts"]), "counts differ from bg_moe_route"
    assert torch.equal(got["offsets"], ref["offsets"]), "offsets differ from bg_moe_route"
    assert int(got["offsets"][-1]) == T * k and int(got["counts"].sum()) == T * k


def test_noalloc_route_matches_existing_path_on_two_calls_in_a_row():
    from paper_2606_21712_b200 import NOALLOC_MAX_TOKENS
    # first call: many tiles, E > 128 (both halves of the scan), ragged last tile
    compare(make_logits(5000, 200, seed=21), 8)
    # second call, straight after: fewer tiles and fewer experts, so most of the array still holds the first
    # call's histograms -- none of it may leak into the result
    compare(make_logits(333, 40, seed=22), 4, check_driver=True)
    # and a few more in a row over the shapes that bracket the kernel's cases: one token, E = 1, k = E,
    # an exact multiple of the tile, the largest call the array allows
    for T, E, k, seed in [(1, 4, 2, 23), (77, 1, 1, 24), (200, 5, 5, 25), (1024, 64, 6, 26), (129, 33, 3, 27),
                          (NOALLOC_MAX_TOKENS, 256, 8, 28), (64, 256, 8, 29), (0, 16, 2, 30)]:
        compare(make_logits(T, E, seed), k, check_driver=True)


def test_noalloc_route_same_stream_back_to_back_without_sync():
    """Two launches on one stream with no host synchronisation between them: stream order is enough."""
    from paper_2606_21712_b200 import route_logits_noalloc
    La, Lb = make_logits(3000, 128, seed=31), make_logits(700, 16, seed=32)
    outs = []
    for L, k in ((La, 8), (Lb, 2)):
        T, E = L.shape
        o = dict(idx=torch.empty(T, k, dtype=torch.int32, device="cuda"), w=torch.empty(T, k, device="cuda"),
                 counts=torch.empty(E, dtype=torch.int32, device="cuda"),
                 offsets=torch.empty(E + 1, dtype=torch.int32, device="cuda"))
        outs.append(o)
    route_logits_noalloc(La, 8, outs[0]["idx"], outs[0]["w"], outs[0]["counts"], outs[0]["offsets"])
    route_logits_noalloc(Lb, 2, outs[1]["idx"], outs[1]["w"], outs[1]["counts"], outs[1]["offsets"])
    torch.cuda.synchronize()
    for (L, k), o in zip(((La, 8), (Lb, 2)), outs):
        ref = existing_path(L, k)
        assert torch.equal(o["idx"], ref["idx"]) and torch.equal(o["counts"], ref["counts"])
        assert torch.equal(o["offsets"], ref["offsets"])
        assert float((o["w"] - ref["w"]).abs().max()) <= W_TOL


def test_noalloc_route_refuses_sizes_beyond_its_array():
    from paper_2606_21712_b200 import BgMoeError, NOALLOC_MAX_TOKENS, BG_ERR_INVALID_ARG, BG_ERR_UNSUPPORTED
    from paper_2606_21712_b200 import route_logits_noalloc
    T, E, k = NOALLOC_MAX_TOKENS + 1, 8, 2
    L = torch.zeros(T, E, device="cuda")
    idx = torch.full((T, k), -5, dtype=torch.int32, device="cuda")
    w = torch.full((T, k), -5.0, device="cuda")
    counts = torch.full((E,), -5, dtype=torch.int32, device="cuda")
    offsets = torch.full((E + 1,), -5, dtype=torch.int32, device="cuda")
    with pytest.raises(BgMoeError) as ei:
        route_logits_noalloc(L, k, idx, w, counts, offsets)
    assert ei.value.status == BG_ERR_INVALID_ARG
    assert "BG_MOE_NOALLOC_MAX_TOKENS" in str(ei.value) and str(NOALLOC_MAX_TOKENS) in str(ei.value)
    torch.cuda.synchronize()
    assert bool((counts == -5).all()) and bool((offsets == -5).all()) and bool((idx == -5).all()), "refused call wrote"
    # E beyond the 256 experts a histogram row holds
    E2 = 257
    with pytest.raises(BgMoeError) as ei:
        route_logits_noalloc(torch.zeros(4, E2, device="cuda"), 2, torch.empty(4, 2, dtype=torch.int32, device="cuda"),
                             torch.empty(4, 2, device="cuda"), torch.empty(E2, dtype=torch.int32, device="cuda"),
                             torch.empty(E2 + 1, dtype=torch.int32, device="cuda"))
    assert ei.value.status == BG_ERR_UNSUPPORTED
    # the array is still usable afterwards
    compare(make_logits(300, 8, seed=33), 2)
