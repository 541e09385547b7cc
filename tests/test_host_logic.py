"""CPU-only checks of the host logic: the C-ABI library loads and exports every symbol the header
declares, fails loudly without a GPU (no CPU fallback), the roofline arithmetic, and the
multi-rank (replicas-only) plumbing of bench.py under gloo with world_size 2."""
import ctypes
import os
import re
import socket
import sys

import pytest
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
import workloads as wl  # noqa: E402


def declared_symbols():
    hdr = open(os.path.join(ROOT, "include", "bg_moe.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return sorted(set(re.findall(r"\b(bg_moe_[a-z0-9_]+)\s*\(", hdr)))


def test_library_exports_every_declared_symbol():
    from paper_2606_21712_b200 import load_library
    from paper_2606_21712_b200.binding import EXPORTS
    lib = load_library()
    syms = declared_symbols()
    assert len(syms) >= 14
    for name in syms:
        assert hasattr(lib, name), f"{name} is declared in include/bg_moe.h but not exported"
    assert sorted(EXPORTS) == syms, "binding.EXPORTS and the header disagree"


def test_strerror_and_null_handling_without_gpu():
    from paper_2606_21712_b200 import load_library
    lib = load_library()
    assert lib.bg_moe_strerror(0) == b"ok"
    assert b"invalid" in lib.bg_moe_strerror(-1)
    assert b"unknown" in lib.bg_moe_strerror(-99)
    assert lib.bg_moe_create(None, None) == -1                     # NULL arguments: error code, no crash
    assert lib.bg_moe_destroy(None) == 0
    assert lib.bg_moe_launch_count(None) == 0


def test_noalloc_route_checks_its_limits_before_touching_the_gpu():
    """bg_moe_route_logits_noalloc refuses what its fixed scratch array cannot hold, with a message, before any CUDA
    call (so this runs without a GPU)."""
    from paper_2606_21712_b200 import load_library, NOALLOC_MAX_TOKENS
    lib = load_library()
    hdr = open(os.path.join(ROOT, "include", "bg_moe.h")).read()
    assert int(re.search(r"#define\s+BG_MOE_NOALLOC_MAX_TOKENS\s+(\d+)", hdr).group(1)) == NOALLOC_MAX_TOKENS
    one = ctypes.c_void_p(256)            # never dereferenced: the size check comes first
    assert lib.bg_moe_route_logits_noalloc(one, NOALLOC_MAX_TOKENS + 1, 8, 2, one, one, one, one, None) == -1
    msg = lib.bg_moe_noalloc_last_error().decode()
    assert "BG_MOE_NOALLOC_MAX_TOKENS" in msg and str(NOALLOC_MAX_TOKENS + 1) in msg
    assert lib.bg_moe_route_logits_noalloc(one, 16, 257, 2, one, one, one, one, None) == -2      # E > 256
    assert lib.bg_moe_route_logits_noalloc(one, 16, 8, 9, one, one, one, one, None) == -1        # k > E
    assert lib.bg_moe_route_logits_noalloc(one, 16, 16, 9, one, one, one, one, None) == -2       # k > 8
    assert lib.bg_moe_route_logits_noalloc(one, -1, 8, 2, one, one, one, one, None) == -1
    assert lib.bg_moe_route_logits_noalloc(one, 16, 8, 2, one, one, None, one, None) == -1       # counts NULL
    assert lib.bg_moe_route_logits_noalloc(None, 16, 8, 2, one, one, one, one, None) == -1       # logits NULL
    # and its translation unit calls no allocating routine at all
    src = open(os.path.join(ROOT, "paper_2606_21712_b200", "csrc", "route_noalloc.cu")).read()
    assert not re.search(r"\b(cudaMalloc\w*|cudaFree\w*|cudaHostAlloc|cuMemAlloc\w*|malloc|new)\s*[\(\[]", src)
    assert "cudaGetSymbolAddress" in src and "static __device__ __align__(256)" in src


@pytest.mark.skipif(torch.cuda.is_available(), reason="checks the no-GPU failure mode")
def test_no_cpu_fallback_create_fails_loudly():
    from paper_2606_21712_b200 import MoELayer, BgMoeError
    with pytest.raises(BgMoeError) as ei:
        MoELayer(512, 1024, 8, 2, 256)
    assert ei.value.status in (-2, -3)                              # unsupported device / CUDA error


def test_product_does_not_import_oracle():
    """The product path may not route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2606_21712_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "bgo_" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_2606_21712_b200" not in txt and "from paper_2606_21712_b200" not in txt
            assert "csrc" not in txt or f.endswith(".cpp")           # the header comment names it only


def test_roofline_arithmetic_matches_survey_table():
    """F = 6Tkdf + 2TdE, B_min = 4Td + 4dE + 6df*E_act."""
    assert wl.C2.flops() / 1e9 == pytest.approx(2886, rel=2e-3)
    assert wl.C2.min_bytes() / 1e6 == pytest.approx(2886, rel=2e-3)
    assert wl.C3.flops() / 1e9 == pytest.approx(311, rel=5e-3)
    assert wl.C3.min_bytes() / 1e6 == pytest.approx(1243, rel=2e-3)
    assert wl.C3.with_T(32768).flops() / 1e9 == pytest.approx(2491, rel=2e-3)
    assert wl.C4.flops() / 1e9 == pytest.approx(5802, rel=2e-3)
    assert wl.C4.min_bytes(194) / 1e6 == pytest.approx(17330, rel=1e-2)
    assert wl.C5.flops() / 1e9 == pytest.approx(3410, rel=2e-3)
    assert wl.C5.min_bytes() / 1e6 == pytest.approx(2484, rel=2e-3)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _gloo_worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    ms = bench.max_over_ranks(10.0 + 5.0 * rank, dist, "cpu")        # rank 1 is the slow one
    dist.barrier()
    q.put((rank, ms, bench.whole_job_rate(4096, world, ms)))
    dist.destroy_process_group()


def test_replicas_timing_is_max_over_ranks_gloo_world2():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [15.0, 15.0]                        # both ranks report the max
    assert res[0][2] == pytest.approx(2 * 4096 / 15e-3)                # whole-job units / slowest time


def test_single_rank_helpers():
    import bench
    assert bench.max_over_ranks(3.5, None, "cpu") == 3.5
    assert bench.whole_job_rate(100, 4, 1000.0) == 400.0
    n = bench.oracle_tokens_per_step(wl.C2, 1.0, 16)
    assert 16 <= n <= wl.C2.T
