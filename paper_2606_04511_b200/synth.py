"""Seeded synthetic inputs for the SparDA decode hot path (shared by tests, bench and smoke).

This module holds NONE of the method's arithmetic: it only draws random tensors with the shapes,
value distributions and layouts of BASELINE.json's configs (recipe in DESIGN.md "Inputs").  The
pooled keys are part of the method (Eq.2) and are therefore NOT produced here: the CUDA path
pools with its own kernel, the oracle with its own loop.

Recipe per layer (reading q15): bias[r, j, :] ~ N(0, sigma) one D-vector per (row, block);
K0, V, F, Q, F0cur ~ N(0, 1); K = bf16(K0 + bias) (bias on keys only, so block scores separate);
everything rounded to bf16 once.  KV is emitted in the ABI layout [R][Nb][2][S][D] (R = B*Hkv,
plane 0 = K, plane 1 = V), F [R][D], Q [B][Hq][D].  Draw order is fixed: bias, K0, V, F, Q, F0cur.
The generator is torch's Philox (CUDA) or mt19937 (CPU) seeded with seed*1000003 + layer; the two
devices give different streams, so a test that feeds both the oracle and the GPU generates ONCE and
copies the bytes.
"""
from __future__ import annotations

from dataclasses import dataclass, replace

import torch


@dataclass(frozen=True)
class DecodeConfig:
    name: str
    batch: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    n_blocks: int          # context = n_blocks * block_size tokens
    topk: int
    n_layers: int = 1
    bias_std: float = 1.5
    seed: int = 0
    block_size: int = 64

    @property
    def rows(self) -> int:
        return self.batch * self.n_kv_heads

    @property
    def group(self) -> int:
        return self.n_q_heads // self.n_kv_heads

    @property
    def context(self) -> int:
        return self.n_blocks * self.block_size

    @property
    def block_bytes(self) -> int:
        """K + V bytes of one block of one KV head (32 KiB at D=128)."""
        return 2 * self.block_size * self.head_dim * 2

    @property
    def kv_bytes_per_layer(self) -> int:
        return self.rows * self.n_blocks * self.block_bytes

    @property
    def gather_bytes_per_layer(self) -> int:
        return self.rows * self.topk * self.block_bytes

    @property
    def kpool_bytes_per_layer(self) -> int:
        return self.rows * self.n_blocks * self.head_dim * 2

    def with_(self, **kw) -> "DecodeConfig":
        return replace(self, **kw)


@dataclass(frozen=True)
class PrefillConfig:
    name: str
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    seq_len: int           # T query positions; Nb = T / block_size pooled keys
    topk: int
    chunk: int = 2048
    bias_std: float = 1.5
    seed: int = 5
    block_size: int = 64

    @property
    def n_blocks(self) -> int:
        return self.seq_len // self.block_size

    def with_(self, **kw) -> "PrefillConfig":
        return replace(self, **kw)


# BASELINE.json configs[0..4]
CFG1_TINY = DecodeConfig("cfg1_tiny", batch=1, n_q_heads=4, n_kv_heads=1, head_dim=64, n_blocks=64, topk=8,
                         bias_std=2.0, seed=0)
CFG2_32K = DecodeConfig("cfg2_32k", batch=8, n_q_heads=32, n_kv_heads=2, head_dim=128, n_blocks=512, topk=64,
                        seed=2)
CFG3_128K = DecodeConfig("cfg3_128k_pipeline", batch=4, n_q_heads=32, n_kv_heads=2, head_dim=128, n_blocks=2048,
                         topk=64, n_layers=32, seed=3)
CFG4_128K = DecodeConfig("cfg4_128k_offload", batch=32, n_q_heads=32, n_kv_heads=2, head_dim=128, n_blocks=2048,
                         topk=64, n_layers=32, seed=4)
CFG5_PREFILL = PrefillConfig("cfg5_prefill_32k", n_q_heads=32, n_kv_heads=2, head_dim=128, seq_len=32768, topk=64)

CONFIGS = {c.name: c for c in (CFG1_TINY, CFG2_32K, CFG3_128K, CFG4_128K, CFG5_PREFILL)}


def _gen(device, seed: int, layer: int) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(seed * 1000003 + layer)
    return g


def _randn(shape, g, device):
    return torch.randn(shape, generator=g, device=device, dtype=torch.float32)


def decode_layer(cfg: DecodeConfig, layer: int = 0, device="cpu", rows: slice | None = None) -> dict:
    """One layer's inputs.  Returns bf16 tensors on ``device``:
    kv [R][Nb][2][S][D], F [R][D], Q [B][Hq][D], F0cur [R][D].

    ``rows`` is not supported for partial generation (draws are whole-tensor); callers that need to
    bound memory generate layer by layer."""
    assert rows is None
    R, Nb, S, D = cfg.rows, cfg.n_blocks, cfg.block_size, cfg.head_dim
    g = _gen(device, cfg.seed, layer)
    bias = _randn((R, Nb, 1, D), g, device) * cfg.bias_std
    kv = torch.empty((R, Nb, 2, S, D), dtype=torch.bfloat16, device=device)
    k0 = _randn((R, Nb, S, D), g, device)
    kv[:, :, 0] = (k0 + bias).to(torch.bfloat16)
    del k0, bias
    kv[:, :, 1] = _randn((R, Nb, S, D), g, device).to(torch.bfloat16)
    F = _randn((R, D), g, device).to(torch.bfloat16)
    Q = _randn((cfg.batch, cfg.n_q_heads, D), g, device).to(torch.bfloat16)
    F0 = _randn((R, D), g, device).to(torch.bfloat16)
    return {"kv": kv, "F": F, "Q": Q, "F0cur": F0}


def prefill_inputs(cfg: PrefillConfig, device="cpu") -> dict:
    """Config-5 inputs: keys K [Hkv][Nb][S][D] (biased per block, to be pooled by the caller's side of
    the method), Forecast F [Hkv][T][D], comparison queries Q [Hq][T][D]; all bf16."""
    Hkv, Hq, T, Nb, S, D = cfg.n_kv_heads, cfg.n_q_heads, cfg.seq_len, cfg.n_blocks, cfg.block_size, cfg.head_dim
    g = _gen(device, cfg.seed, 0)
    bias = _randn((Hkv, Nb, 1, D), g, device) * cfg.bias_std
    kv = torch.empty((Hkv, Nb, 2, S, D), dtype=torch.bfloat16, device=device)
    kv[:, :, 0] = (_randn((Hkv, Nb, S, D), g, device) + bias).to(torch.bfloat16)
    kv[:, :, 1] = _randn((Hkv, Nb, S, D), g, device).to(torch.bfloat16)
    F = _randn((Hkv, T, D), g, device).to(torch.bfloat16)
    Q = _randn((Hq, T, D), g, device).to(torch.bfloat16)
    return {"kv": kv, "F": F, "Q": Q}
