"""Helpers for the -m gpu parity tests: run a layer through the C ABI (via the thin binding) and fetch
results as numpy; compare with the oracle."""
from __future__ import annotations

from types import SimpleNamespace

import numpy as np
import torch

import oracle
from bm_inputs import bf16_bits

ROUTING_INT_FIELDS = ["expert_ids", "group_ids", "n_slots", "counts", "offsets", "row_token", "row_slot", "slot_row"]


def layer_dims(L):
    if hasattr(L, "cfg"):
        c = L.cfg
        return c.K, c.G, c.S
    return L.K, L.G, L.S


def to_device(L):
    d = SimpleNamespace()
    for k in ("x", "W_router", "router_bias", "group_map", "W1", "W3", "W2"):
        v = getattr(L, k, None)
        setattr(d, k, None if v is None else v.cuda())
    return d


def gpu_route(L, d=None):
    import paper_2607_04164_b200 as bm
    K, G, S = layer_dims(L)
    d = d or to_device(L)
    T, D = L.x.shape
    E = L.W_router.shape[0]
    F = 8 if getattr(L, "W1", None) is None else L.W1.shape[1]
    ws = bm.alloc_workspace(T, D, F, E, K, G, S)
    r = bm.Routing(T, K, G)
    bm.bm_route(d.x, d.W_router, d.router_bias, K, d.group_map, G, r, ws)
    torch.cuda.synchronize()
    return r, ws, d


def routing_to_numpy(r, T):
    return SimpleNamespace(**{k: v.cpu().numpy() for k, v in r.view(T).items()})


def gpu_layer(L, path=0, d=None):
    """Returns (routing numpy namespace, out float64 numpy [T,D], device status bits)."""
    import paper_2607_04164_b200 as bm
    K, G, S = layer_dims(L)
    T, D = L.x.shape
    r, ws, d = gpu_route(L, d)
    out = torch.full((T, D), float("nan"), dtype=torch.bfloat16, device="cuda")
    bm.bm_moe_forward(d.x, r, d.W1, d.W3, d.W2, out, ws, S=S, path=path)
    torch.cuda.synchronize()
    status = bm.bm_device_status(ws)
    return routing_to_numpy(r, T), out.float().cpu().numpy().astype(np.float64), status


def oracle_route(L, want_logits=False):
    K, G, S = layer_dims(L)
    bias = None if L.router_bias is None else L.router_bias.numpy()
    return oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), bias, K, L.group_map.numpy(), G,
                        want_logits=want_logits)


def oracle_forward(L, r, sel_tokens=None):
    K, G, S = layer_dims(L)
    return oracle.moe_forward(bf16_bits(L.x), r, bf16_bits(L.W1), bf16_bits(L.W3), bf16_bits(L.W2), S,
                              sel_tokens=sel_tokens)


def assert_routing_equal(g, o):
    """Bit-exact integer routing arrays; gate weights within 1e-6 (expf ulps)."""
    for k in ROUTING_INT_FIELDS:
        a, b = getattr(g, k), getattr(o, k)
        assert a.shape == b.shape, (k, a.shape, b.shape)
        if not (a == b).all():
            bad = np.argwhere(a != b)
            raise AssertionError(f"routing field {k} differs at {len(bad)} places, first {bad[0]}: "
                                 f"gpu {a[tuple(bad[0])]} oracle {b[tuple(bad[0])]}")
    assert np.abs(g.gate_w.astype(np.float64) - o.gate_w.astype(np.float64)).max() <= 1e-6


def assert_out_close(out_gpu, out_oracle, rel_rms=1e-2):
    """BASELINE.json north_star: max|gpu - oracle| <= 2e-2 * (1 + |oracle|) elementwise.  That tolerance has an
    absolute floor of 0.02, which on small shapes (|out| ~ 0.02) would let a dropped term through, so the
    relative RMS error is bounded too: bf16 rounding of h, y and out gives ~2e-3."""
    assert np.isfinite(out_gpu).all(), "non-finite values in the GPU output"
    err = np.abs(out_gpu - out_oracle)
    tol = 2e-2 * (1.0 + np.abs(out_oracle))
    worst = (err / tol).max()
    assert worst <= 1.0, f"max err/tol = {worst:.3f} (max abs err {err.max():.4g}, max |oracle| {np.abs(out_oracle).max():.4g})"
    rms_o = float(np.sqrt(np.mean(np.square(out_oracle))))
    rms_e = float(np.sqrt(np.mean(np.square(err))))
    if rms_o > 0:
        assert rms_e <= rel_rms * rms_o, f"relative RMS error {rms_e / rms_o:.4g} > {rel_rms} (rms oracle {rms_o:.4g})"
    else:
        assert rms_e == 0.0
    return worst
