"""Config registry: the five workloads of BASELINE.json `configs[0..4]`.

Notation (SURVEY.md top): T tokens, D = d_model, F = d_ff, E routed experts, K = top-k,
G united groups, S always-on shared experts, zipf_s = router skew exponent.
"""
from __future__ import annotations

from dataclasses import dataclass, replace
from typing import Iterator


@dataclass(frozen=True)
class LayerConfig:
    name: str
    T: int
    D: int
    F: int
    E: int
    K: int
    G: int
    S: int = 0
    zipf_s: float = 0.0
    # 'fixed'    : gmap given literally (cfg 0)
    # 'balanced' : seeded permutation, gmap[perm[i]] = i mod G  (sizes differ by <= 1; cap ceil(E/G))
    # 'uneven'   : seeded sizes in [2, 8] summing to E (cfg 3)
    # 'identity' : gmap[e] = e, G == E  (zero brownout)
    gmap_kind: str = "balanced"
    fixed_gmap: tuple = ()

    def with_(self, **kw) -> "LayerConfig":
        return replace(self, **kw)


CONFIGS = {
    # BJ:configs[0]  tiny correctness layer
    "tiny": LayerConfig("tiny", T=64, D=256, F=512, E=8, K=2, G=4, gmap_kind="fixed",
                        fixed_gmap=(0, 0, 1, 1, 2, 2, 3, 3)),
    # BJ:configs[1]  Mixtral-8x7B-shaped decode layer (HBM-bound, the headline bench workload)
    "decode": LayerConfig("decode", T=64, D=4096, F=14336, E=8, K=2, G=4, zipf_s=1.2),
    # BJ:configs[2]  Mixtral-8x7B-shaped prefill layer (tensor-bound)
    "prefill": LayerConfig("prefill", T=8192, D=4096, F=14336, E=8, K=2, G=4, zipf_s=1.2),
    # BJ:configs[3]  fine-grained layer with 2 always-on shared experts, uneven groups
    "finegrained": LayerConfig("finegrained", T=4096, D=2048, F=1408, E=64, K=6, G=16, S=2,
                               zipf_s=1.5, gmap_kind="uneven"),
}

SWEEP_G = (60, 30, 15, 8)
SWEEP_T = (1, 16, 256, 4096, 16384)
SWEEP_S = (0.0, 1.0, 2.0)


def sweep_points() -> Iterator[LayerConfig]:
    """BJ:configs[4]  brownout sweep at the Qwen-MoE-like shape (E=60, top-4)."""
    for G in SWEEP_G:
        for T in SWEEP_T:
            for s in SWEEP_S:
                yield LayerConfig(f"sweep_G{G}_T{T}_s{s:g}", T=T, D=2048, F=1408, E=60, K=4, G=G,
                                  zipf_s=s, gmap_kind="identity" if G == 60 else "balanced")


def get_config(name: str) -> LayerConfig:
    if name in CONFIGS:
        return CONFIGS[name]
    for c in sweep_points():
        if c.name == name:
            return c
    raise KeyError(name)
