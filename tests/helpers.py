"""Test helpers: an independent definition-form evaluator of PAPER.md:42 and small utilities.

`definition_form` is written directly from the layer definition h_t = sum_{i<=K} g_i(x_t) FFN_i(x_t)
 with every routed expert e replaced by its united expert gmap[e] (full
brownout).  It has no dedup, no histogram, no permutation and no shared code with oracle/ -- it is
the pin the grouped/permuted oracle is checked against.
"""
from __future__ import annotations

import numpy as np
import torch


def f64(t: torch.Tensor) -> np.ndarray:
    return t.to(torch.float64).numpy()


def silu(a):
    return a / (1.0 + np.exp(-a))


def ffn_def(x_t, W1, W3, W2):
    """SwiGLU FFN of one expert on one token in fp64 with library matmuls (reading A3)."""
    return W2 @ (silu(W1 @ x_t) * (W3 @ x_t))


def definition_form(x, W_router, bias, K, gmap, W1, W3, W2, S=0, tokens=None):
    """Per token: fp64 logits, sort, softmax over the top-K, sum w_i * FFN_{gmap[e_i]}(x_t) (+ shared).

    All arguments are fp64 numpy arrays (gmap int).  Returns (out [n,D], expert_ids [n,K], margin [n])
    where margin is the gap between the K-th and (K+1)-th logit (inf if K == E).
    """
    T, D = x.shape
    E = W_router.shape[0]
    G = W1.shape[0] - S
    toks = range(T) if tokens is None else tokens
    outs, ids, margins = [], [], []
    for t in toks:
        l = W_router @ x[t]
        if bias is not None:
            l = l + bias
        order = sorted(range(E), key=lambda e: (-l[e], e))
        sel = order[:K]
        margins.append(l[order[K - 1]] - l[order[K]] if K < E else np.inf)
        p = np.exp(l[sel] - l[sel[0]])
        w = p / p.sum()
        o = np.zeros(D)
        for i, e in enumerate(sel):
            u = int(gmap[e])
            o += w[i] * ffn_def(x[t], W1[u], W3[u], W2[u])
        for j in range(S):
            o += ffn_def(x[t], W1[G + j], W3[G + j], W2[G + j])
        outs.append(o)
        ids.append(sel)
    return np.array(outs), np.array(ids, dtype=np.int32), np.array(margins)


def bf16_tensor(a) -> torch.Tensor:
    """fp -> bf16 CPU tensor (round to nearest even)."""
    return torch.as_tensor(np.asarray(a, dtype=np.float32)).to(torch.bfloat16)


def rand_layer(rng: np.random.Generator, T, D, F, E, K, G, S=0, gmap=None, bias=False, wstd=0.05):
    """Small random bf16 layer for property tests (independent of bm_inputs' recipe)."""
    from types import SimpleNamespace
    L = SimpleNamespace(T=T, D=D, F=F, E=E, K=K, G=G, S=S)
    L.x = bf16_tensor(rng.standard_normal((T, D)))
    L.W_router = bf16_tensor(rng.standard_normal((E, D)) * 0.2)
    L.router_bias = torch.as_tensor(rng.standard_normal(E).astype(np.float32)) if bias else None
    if gmap is None:
        gmap = rng.integers(0, G, size=E)
    L.group_map = torch.as_tensor(np.asarray(gmap, dtype=np.int32))
    L.W1 = bf16_tensor(rng.standard_normal((G + S, F, D)) * wstd)
    L.W3 = bf16_tensor(rng.standard_normal((G + S, F, D)) * wstd)
    L.W2 = bf16_tensor(rng.standard_normal((G + S, D, F)) * wstd)
    return L


def oracle_layer(L, sel_tokens=None, want_logits=False):
    """Run the oracle end to end on a layer namespace; returns (routing, out fp64)."""
    import oracle
    from bm_inputs import bf16_bits
    K = L.K if hasattr(L, "K") else L.cfg.K
    G = L.G if hasattr(L, "G") else L.cfg.G
    S = L.S if hasattr(L, "S") else L.cfg.S
    bias = None if L.router_bias is None else L.router_bias.numpy()
    r = oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), bias, K, L.group_map.numpy(), G,
                     want_logits=want_logits)
    out = oracle.moe_forward(bf16_bits(L.x), r, bf16_bits(L.W1), bf16_bits(L.W3), bf16_bits(L.W2), S,
                             sel_tokens=sel_tokens)
    return r, out
