"""Seeded synthetic inputs for the combined MoE layer (BASELINE.json `configs[0..4]`).

This module serves BOTH the CPU oracle (`oracle/`) and the CUDA path
(`paper_2606_21712_b200/`).  It holds none of the method's arithmetic: it only
draws random tensors of the shapes / distributions the configs name and rounds
them to bf16 where the layer takes bf16.  It imports neither side.

The tensors stand in for the paper's LongBench / GSM8K / ChatBotArena /
production-trace workloads: the MoE layer is
token-content-agnostic, so only the shapes (T, d, E, k, f), the value
distributions and the prefill/decode length mix matter.

Recipe (DESIGN.md §"Input recipe"):
  seed(tensor) = 260621712 + 100*config_index + tensor_index
  hidden   bf16 [T,d]   ~ N(0, 1)            (C5 decode rows: std 2)        tensor_index 0
  W_r      fp32 [d,E]   ~ N(0, 1/sqrt(d))                                   tensor_index 1
  W_gate   bf16 [E,d,f] ~ N(0, 0.02)                                        tensor_index 2
  W_up     bf16 [E,d,f] ~ N(0, 0.02)                                        tensor_index 3
  W_down   bf16 [E,f,d] ~ N(0, 0.02)                                        tensor_index 4
  b_r      fp32 [E]     C4 only: -1.1*ln(rank_e), rank a seeded permutation  tensor_index 5
The second parameter of N(.,.) is the standard deviation (reading S15).
Expert weights are drawn expert by expert (seed + 1000*(e+1)) so that the
22.5 GB of C4 never needs a 45 GB fp32 temporary, and so that a test can
materialise a single expert.

`device="cpu"` uses torch's CPU generator; `device="cuda"` uses torch's CUDA
Philox generator (different bits from the CPU stream, but the same bits for
every consumer in the process: the oracle receives a host copy of exactly what
the GPU path reads).
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import torch

BASE_SEED = 260621712


@dataclasses.dataclass(frozen=True)
class MoEConfig:
    name: str
    index: int          # position in BASELINE.json configs (seed stream)
    T: int              # combined tokens
    d: int              # hidden
    E: int              # experts
    k: int              # top-k
    f: int              # expert intermediate
    zipf_s: float = 0.0  # C4: per-expert Zipf bias exponent (0 = no bias)
    # C5: (n_prefill_segments, prefill_len, n_decode_rows, decode_std)
    mix: Optional[tuple] = None

    @property
    def R(self) -> int:
        return self.T * self.k

    def with_T(self, T: int) -> "MoEConfig":
        return dataclasses.replace(self, T=T, name=f"{self.name.split('@')[0]}@T{T}")

    def flops(self) -> float:
        """F = 6*T*k*d*f + 2*T*d*E; useful rows only."""
        return 6.0 * self.T * self.k * self.d * self.f + 2.0 * self.T * self.d * self.E

    def min_bytes(self, E_active: Optional[int] = None) -> float:
        """B_min = 4*T*d + 4*d*E + 6*d*f*E_active."""
        ea = self.E if E_active is None else E_active
        return 4.0 * self.T * self.d + 4.0 * self.d * self.E + 6.0 * self.d * self.f * ea


C1 = MoEConfig("C1-tiny", 0, T=256, d=512, E=8, k=2, f=1024)
C2 = MoEConfig("C2-mixtral", 1, T=4096, d=4096, E=8, k=2, f=14336)
C3 = MoEConfig("C3-finegrained", 2, T=4096, d=2048, E=128, k=8, f=768)
C3_SWEEP_T = (64, 256, 1024, 4096, 16384, 32768)
C4 = MoEConfig("C4-dsv3-zipf", 3, T=8192, d=7168, E=256, k=8, f=2048, zipf_s=1.1)
C5 = MoEConfig("C5-mixed", 4, T=16384, d=4096, E=64, k=6, f=1408,
               mix=(30, 512, 1024, 2.0))

CONFIGS = {"C1": C1, "C2": C2, "C3": C3, "C4": C4, "C5": C5}


def _gen(device: str, seed: int) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed)
    return g


def _seed(cfg: MoEConfig, tensor_index: int) -> int:
    return BASE_SEED + 100 * cfg.index + tensor_index


def make_hidden(cfg: MoEConfig, device: str = "cpu") -> torch.Tensor:
    """`hidden [T,d]` bf16: the COMBINE result (Alg. 1 l.7)."""
    g = _gen(device, _seed(cfg, 0))
    h = torch.randn(cfg.T, cfg.d, generator=g, device=device, dtype=torch.float32)
    if cfg.mix is not None:
        n_pre, pre_len, n_dec, dec_std = cfg.mix
        n_prefill_rows = min(n_pre * pre_len, cfg.T)
        # prefill segments first, then single-row decode segments (reading S17)
        h[n_prefill_rows:] *= dec_std
    return h.to(torch.bfloat16)


def segment_lengths(cfg: MoEConfig) -> list:
    """Per-coroutine token counts whose concatenation is `hidden` (a0 COMBINE)."""
    if cfg.mix is not None:
        n_pre, pre_len, n_dec, _ = cfg.mix
        return [pre_len] * n_pre + [1] * n_dec
    if cfg.index == 0:
        return [16] * 16
    return [cfg.T]


def make_router(cfg: MoEConfig, device: str = "cpu"):
    """`W_r [d,E]` fp32 and `b_r [E]` fp32 (None unless the config has a Zipf bias)."""
    g = _gen(device, _seed(cfg, 1))
    W_r = torch.randn(cfg.d, cfg.E, generator=g, device=device, dtype=torch.float32)
    W_r *= 1.0 / math.sqrt(cfg.d)
    b_r = None
    if cfg.zipf_s > 0:
        gp = _gen("cpu", _seed(cfg, 5))
        rank = torch.randperm(cfg.E, generator=gp) + 1          # rank_e in 1..E
        b_r = (-cfg.zipf_s * torch.log(rank.to(torch.float64))).to(torch.float32).to(device)
    return W_r, b_r


def make_expert_weight(cfg: MoEConfig, which: str, e: int, device: str = "cpu") -> torch.Tensor:
    """One expert's matrix: which in {"gate","up"} -> [d,f]; "down" -> [f,d]; bf16."""
    ti = {"gate": 2, "up": 3, "down": 4}[which]
    shape = (cfg.f, cfg.d) if which == "down" else (cfg.d, cfg.f)
    g = _gen(device, _seed(cfg, ti) + 1000 * (e + 1))
    w = torch.randn(*shape, generator=g, device=device, dtype=torch.float32)
    w *= 0.02
    return w.to(torch.bfloat16)


def make_expert_weights(cfg: MoEConfig, device: str = "cpu"):
    """`W_gate, W_up [E,d,f]`, `W_down [E,f,d]`, bf16, row-major (reading S14)."""
    Wg = torch.empty(cfg.E, cfg.d, cfg.f, dtype=torch.bfloat16, device=device)
    Wu = torch.empty(cfg.E, cfg.d, cfg.f, dtype=torch.bfloat16, device=device)
    Wd = torch.empty(cfg.E, cfg.f, cfg.d, dtype=torch.bfloat16, device=device)
    for e in range(cfg.E):
        Wg[e] = make_expert_weight(cfg, "gate", e, device)
        Wu[e] = make_expert_weight(cfg, "up", e, device)
        Wd[e] = make_expert_weight(cfg, "down", e, device)
    return Wg, Wu, Wd


def make_layer(cfg: MoEConfig, device: str = "cpu") -> dict:
    hidden = make_hidden(cfg, device)
    W_r, b_r = make_router(cfg, device)
    Wg, Wu, Wd = make_expert_weights(cfg, device)
    return dict(cfg=cfg, hidden=hidden, W_r=W_r, b_r=b_r, W_gate=Wg, W_up=Wu, W_down=Wd)


def small_config(T=48, d=64, E=6, k=2, f=96, index=7, name="small") -> MoEConfig:
    """Ad-hoc config for unit tests (same recipe, its own seed stream)."""
    return MoEConfig(name, index, T=T, d=d, E=E, k=k, f=f)
