"""Seeded generators: tensors, group maps, router bias.  No method arithmetic lives here.

Recipe:
  * every tensor comes from its own `torch.Generator().manual_seed(1000*seed + tensor_id)`, is
    sampled in fp32 on the CPU and cast to bf16 (round-to-nearest-even); the same host buffers go
    to the oracle and (copied) to the GPU;
  * x ~ N(0,1);  W_router, W1, W3, W2 ~ N(0, 0.02);
  * group maps: literal (cfg 0) / balanced seeded permutation / uneven sizes 2..8 / identity;
  * router skew: rank = seeded permutation of 1..E, bias_e = -s * c * sigma * ln(rank_e) with
    sigma = 0.02*sqrt(D) (std of a logit) and c = 0.55; s = 0 -> no bias (None).
"""
from __future__ import annotations

import math
from types import SimpleNamespace

import numpy as np
import torch

from .configs import LayerConfig

TID_X, TID_WR, TID_RANK, TID_GMAP, TID_W1, TID_W3, TID_W2 = 1, 2, 3, 4, 5, 6, 7
SKEW_C = 0.55
W_STD = 0.02


def _gen(seed: int, tensor_id: int) -> torch.Generator:
    g = torch.Generator(device="cpu")
    g.manual_seed(1000 * seed + tensor_id)
    return g


def bf16_bits(t: torch.Tensor) -> np.ndarray:
    """View a CPU bf16 tensor as a uint16 numpy array (the storage format of both C ABIs)."""
    assert t.dtype == torch.bfloat16 and t.device.type == "cpu"
    return t.contiguous().view(torch.uint16).numpy()


def make_group_map(cfg: LayerConfig, seed: int = 0) -> torch.Tensor:
    """Group map g: expert -> united group, 0-based, int32 [E] (Eq. 2)."""
    E, G = cfg.E, cfg.G
    if cfg.gmap_kind == "fixed":
        gm = torch.tensor(cfg.fixed_gmap, dtype=torch.int32)
        assert gm.numel() == E
        return gm
    if cfg.gmap_kind == "identity":
        assert G == E
        return torch.arange(E, dtype=torch.int32)
    perm = torch.randperm(E, generator=_gen(seed, TID_GMAP))
    gm = torch.empty(E, dtype=torch.int32)
    if cfg.gmap_kind == "balanced":
        # sizes differ by at most 1, so the capacity cap ceil(E/G) of PAPER.md:145 holds
        gm[perm] = (torch.arange(E) % G).to(torch.int32)
        return gm
    if cfg.gmap_kind == "uneven":
        # BJ:configs[3]: group sizes 2..8 summing to E
        assert 2 * G <= E <= 8 * G
        g = _gen(seed, TID_GMAP + 100)
        sizes = [2] * G
        while sum(sizes) < E:
            u = int(torch.randint(0, G, (1,), generator=g))
            if sizes[u] < 8:
                sizes[u] += 1
        pos = 0
        for u, n in enumerate(sizes):
            gm[perm[pos:pos + n]] = u
            pos += n
        return gm
    raise ValueError(cfg.gmap_kind)


def make_router_bias(E: int, D: int, zipf_s: float, seed: int = 0):
    """Per-expert logit bias producing a Zipf-like load skew (PAPER.md:58 shapes it); f32 [E] or None."""
    if zipf_s == 0.0:
        return None
    rank = torch.randperm(E, generator=_gen(seed, TID_RANK)) + 1
    sigma = W_STD * math.sqrt(D)
    return (-zipf_s * SKEW_C * sigma * torch.log(rank.to(torch.float64))).to(torch.float32)


def make_cold_mask(E: int, frac_cold: float, seed: int = 0) -> torch.Tensor:
    """Partial-brownout input: i32 [E], 1 = cold.  The round(frac_cold * E) experts that the
    skew recipe above loads least (largest Zipf rank) are cold -- the paper's cold experts are the rarely
    activated ones; its threshold criterion itself is in its reference [7] (A9)."""
    rank = torch.randperm(E, generator=_gen(seed, TID_RANK)) + 1
    n_cold = int(round(frac_cold * E))
    return (rank > E - n_cold).to(torch.int32)


def _randn_bf16(shape, std: float, gen: torch.Generator) -> torch.Tensor:
    """N(0, std) sampled in fp32, cast to bf16; the leading dim is drawn slice by slice to bound memory."""
    out = torch.empty(shape, dtype=torch.bfloat16)
    if len(shape) <= 2:
        out.copy_(torch.randn(shape, generator=gen, dtype=torch.float32) * std)
        return out
    for i in range(shape[0]):
        out[i].copy_(torch.randn(shape[1:], generator=gen, dtype=torch.float32) * std)
    return out


def make_layer(cfg: LayerConfig, seed: int = 0, weights: bool = True) -> SimpleNamespace:
    """All inputs of one layer call as CPU tensors.

    x [T,D] bf16, W_router [E,D] bf16, router_bias [E] f32 | None, group_map [E] i32,
    W1, W3 [G+S,F,D] bf16, W2 [G+S,D,F] bf16 (united experts first, then the S shared experts).
    """
    T, D, F, E, G, S = cfg.T, cfg.D, cfg.F, cfg.E, cfg.G, cfg.S
    L = SimpleNamespace(cfg=cfg, seed=seed)
    L.x = _randn_bf16((T, D), 1.0, _gen(seed, TID_X))
    L.W_router = _randn_bf16((E, D), W_STD, _gen(seed, TID_WR))
    L.router_bias = make_router_bias(E, D, cfg.zipf_s, seed)
    L.group_map = make_group_map(cfg, seed)
    if weights:
        L.W1 = _randn_bf16((G + S, F, D), W_STD, _gen(seed, TID_W1))
        L.W3 = _randn_bf16((G + S, F, D), W_STD, _gen(seed, TID_W3))
        L.W2 = _randn_bf16((G + S, D, F), W_STD, _gen(seed, TID_W2))
    else:
        L.W1 = L.W3 = L.W2 = None
    return L


def identity_variant(cfg: LayerConfig) -> LayerConfig:
    """The ungrouped comparison run: G = E, identity map (zero brownout)."""
    return cfg.with_(name=cfg.name + "_ungrouped", G=cfg.E, gmap_kind="identity", fixed_gmap=())
