"""All-T restatement of F1-F2 with library matmuls (SURVEY.md 8(c) pins table, "Large shapes").

The plain oracle (oracle/bm_oracle.c) evaluates a few hundred tokens per second at the Mixtral shape, so at
T >= 4096 it covers a seeded token subset.  This module restates the same definition (PAPER.md:42 with united
experts; SwiGLU: DESIGN.md A3) group by group with torch CPU matmuls so that EVERY token of a full-size
config can be compared with the GPU output.  It is test infrastructure: it lives in tests/, shares no code with
oracle/ or with the CUDA path, and is itself pinned against the plain oracle (tests/test_restatement.py on
mid-size shapes, and on the sampled subset inside every full-size GPU test).

    for each group u (and shared expert G+j):  X_u = rows of x routed to u
        H = SiLU(X_u W1[u]^T) * (X_u W3[u]^T);   Y = H W2[u]^T
        out[t] += gate_w[t, s] * Y[row of (t, s)]            (shared experts: weight 1, every token)

`round_h` / `round_y` model the two bf16 roundings reading A12 allows the GPU (the intermediate h always; the
per-row expert output y on the prefill and matrix-vector paths): with them switched on, the remaining GPU
difference is the bf16 rounding of `out` and fp32 summation order.
"""
from __future__ import annotations

import numpy as np
import torch


def _bf16_round(t: torch.Tensor) -> torch.Tensor:
    return t.to(torch.bfloat16).to(t.dtype)


def layer_restatement(x, routing, W1, W3, W2, S=0, dtype=torch.float32, round_h=False, round_y=False,
                      row_block=4096, return_abs_y=False):
    """x [T,D], W1/W3 [G+S,F,D], W2 [G+S,D,F]: CPU bf16 tensors.  routing: the oracle's routing arrays (numpy).
    Returns out [T,D] float64; with return_abs_y also sum_s gate_w[t,s] * |y_s| [T,D] (the scale of a bf16
    rounding of the per-row expert outputs: each y_s moves by at most 2^-8 |y_s|)."""
    T, D = x.shape
    G = W1.shape[0] - S
    K = routing.group_ids.shape[1]
    out = torch.zeros((T, D), dtype=torch.float64)
    abs_y = torch.zeros((T, D), dtype=torch.float64) if return_abs_y else None
    gid = torch.as_tensor(np.asarray(routing.group_ids)).long()
    gw = torch.as_tensor(np.asarray(routing.gate_w)).double()
    nsl = torch.as_tensor(np.asarray(routing.n_slots)).long()
    valid = torch.arange(K)[None, :] < nsl[:, None]
    for u in range(G + S):
        if u < G:
            tok, slot = torch.nonzero((gid == u) & valid, as_tuple=True)     # token ascending
            if tok.numel() == 0:
                continue
            wts = gw[tok, slot]
        else:
            tok = torch.arange(T)
            wts = torch.ones(T, dtype=torch.float64)
        w1, w3, w2 = W1[u].to(dtype), W3[u].to(dtype), W2[u].to(dtype)
        for r0 in range(0, tok.numel(), row_block):
            tk = tok[r0:r0 + row_block]
            xu = x[tk].to(dtype)
            a = xu @ w1.T
            b = xu @ w3.T
            h = a / (1.0 + torch.exp(-a)) * b
            if round_h:
                h = _bf16_round(h)
            y = h @ w2.T
            if round_y:
                y = _bf16_round(y)
            out.index_add_(0, tk, y.double() * wts[r0:r0 + row_block, None])
            if return_abs_y:
                abs_y.index_add_(0, tk, y.double().abs() * wts[r0:r0 + row_block, None])
    return (out.numpy(), abs_y.numpy()) if return_abs_y else out.numpy()


def chunk_boundary_tokens(routing, T, S=0, chunk=128) -> set:
    """First and last token of every `chunk`-row piece of every group's row list (and of the token range, for
    shared experts): the rows at the edges of the GEMM tiles."""
    sel = set()
    offs = np.asarray(routing.offsets)
    rt = np.asarray(routing.row_token)
    for u in range(len(offs) - 1):
        lo, hi = int(offs[u]), int(offs[u + 1])
        for c0 in range(lo, hi, chunk):
            sel.add(int(rt[c0]))
            sel.add(int(rt[min(c0 + chunk, hi) - 1]))
    if S > 0:
        for c0 in range(0, T, chunk):
            sel.add(c0)
            sel.add(min(c0 + chunk, T) - 1)
    return sel
