"""GPU parity (-m gpu) for SURVEY.md 8(f) rows: partial brownout (bm_route_partial + bm_moe_forward over stacked
weight sets) and united-weight construction (bm_unite_weights), against the oracle on the same seeded inputs."""
import numpy as np
import pytest
import torch

import oracle
from bm_inputs import LayerConfig, bf16_bits, make_layer
from gpu_helpers import ROUTING_INT_FIELDS, assert_out_close, assert_routing_equal, routing_to_numpy
from helpers import bf16_tensor

pytestmark = pytest.mark.gpu


def _orig(seed, E, F, D):
    g = torch.Generator().manual_seed(7000 + seed)
    mk = lambda *sh: (torch.randn(*sh, generator=g) * 0.02).to(torch.bfloat16)
    return mk(E, F, D), mk(E, F, D), mk(E, D, F)


def _run_partial(cfg, seed, cold, path=0):
    import paper_2607_04164_b200 as bm
    L = make_layer(cfg, seed)
    T, D, F, E, K, G, S = cfg.T, cfg.D, cfg.F, cfg.E, cfg.K, cfg.G, cfg.S
    Wo = _orig(seed, E, F, D)
    stack = lambda u, o: torch.cat([u[:G], o, u[G:G + S]], dim=0).contiguous()
    W1, W3, W2 = stack(L.W1, Wo[0]), stack(L.W3, Wo[1]), stack(L.W2, Wo[2])
    NS = G + E
    bias = None if L.router_bias is None else L.router_bias.numpy()
    o = oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), bias, K, L.group_map.numpy(), G, cold_mask=cold)
    ref = oracle.moe_forward(bf16_bits(L.x), o, bf16_bits(W1), bf16_bits(W3), bf16_bits(W2), S)
    ws = bm.alloc_workspace(T, D, F, E, K, NS, S)
    r = bm.Routing(T, K, NS)
    xd = L.x.cuda()
    bm.bm_route_partial(xd, L.W_router.cuda(), None if L.router_bias is None else L.router_bias.cuda(), K,
                        L.group_map.cuda(), G, torch.as_tensor(cold, dtype=torch.int32).cuda(), r, ws)
    out = torch.full((T, D), float("nan"), dtype=torch.bfloat16, device="cuda")
    bm.bm_moe_forward(xd, r, W1.cuda(), W3.cuda(), W2.cuda(), out, ws, S=S, path=path)
    torch.cuda.synchronize()
    assert bm.bm_device_status(ws) == 0
    assert r.c.G == NS
    assert_routing_equal(routing_to_numpy(r, T), o)
    return assert_out_close(out.float().cpu().numpy().astype(np.float64), ref), o


@pytest.mark.parametrize("path", [0, 1, 2])
@pytest.mark.parametrize("frac_cold", [0.0, 0.5, 1.0])
def test_partial_brownout_small(path, frac_cold):
    cfg = LayerConfig("pb", T=200, D=256, F=320, E=12, K=3, G=4, S=1, zipf_s=1.0)
    rng = np.random.default_rng(5)
    cold = (rng.random(cfg.E) < frac_cold).astype(np.int32)
    _, o = _run_partial(cfg, 0, cold, path)
    if frac_cold == 0.0:
        assert (o.counts[:cfg.G] == 0).all() and (o.n_slots == cfg.K).all()
    if frac_cold == 1.0:
        assert (o.counts[cfg.G:] == 0).all()


def test_partial_brownout_qwen_shape_prefill():
    # BJ:configs[4] shape (E=60, top-4) with the 20 least-loaded experts ... here: a seeded half of the experts cold
    cfg = LayerConfig("pbq", T=1500, D=2048, F=1408, E=60, K=4, G=15, zipf_s=1.0)
    rng = np.random.default_rng(6)
    cold = (rng.random(cfg.E) < 0.6).astype(np.int32)
    _run_partial(cfg, 1, cold)


def test_route_partial_argument_errors():
    import paper_2607_04164_b200 as bm
    from paper_2607_04164_b200.binding import BM_MAX_G
    cfg = LayerConfig("pb", T=8, D=64, F=64, E=8, K=2, G=4)
    L = make_layer(cfg, 0, weights=False)
    ws = bm.alloc_workspace(8, 64, 64, 8, 2, 12, 0)
    r = bm.Routing(8, 2, 12)
    with pytest.raises(bm.BmError) as ei:
        bm.bm_route_partial(L.x.cuda(), L.W_router.cuda(), None, 2, L.group_map.cuda(), 4, None, r, ws)
    assert ei.value.code == -1                                   # BM_ERR_NULL: cold_mask missing
    big = torch.zeros((400, 64), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(bm.BmError) as ei:                       # G + E > BM_MAX_G
        bm.bm_route_partial(L.x.cuda(), big, None, 2, torch.zeros(400, dtype=torch.int32, device="cuda"), 200,
                            torch.zeros(400, dtype=torch.int32, device="cuda"), r, ws)
    assert ei.value.code == -2


@pytest.mark.parametrize("E,G,shape", [(8, 4, (64, 40)), (60, 15, (1408, 2048)), (7, 3, (24, 8)), (5, 8, (16, 16))])
def test_unite_weights_matches_oracle(E, G, shape):
    import paper_2607_04164_b200 as bm
    rng = np.random.default_rng(E * 100 + G)
    W = bf16_tensor(rng.standard_normal((E,) + shape) * 0.02)
    gmap = rng.integers(0, G, size=E).astype(np.int32)
    if E >= G:
        gmap[:G] = np.arange(G)                                  # no empty group ...
    ref = oracle.unite_weights(bf16_bits(W), gmap, G)            # (E < G: some groups stay empty -> zeros)
    out = bm.bm_unite_weights(W.cuda(), torch.as_tensor(gmap).cuda(), G)
    torch.cuda.synchronize()
    got = out.float().cpu().numpy().astype(np.float64)
    # one rounding to bf16 (half an ulp = 2^-9 relative) on top of an fp32 sum of <= E exact bf16 values
    tol = 2.0 ** -8 * np.abs(ref) + 1e-30
    assert (np.abs(got - ref) <= tol).all()
    for u in range(G):
        if not (gmap == u).any():
            assert (got[u] == 0).all()
    # a singleton group returns its member bit-exactly
    for u in range(G):
        m = np.nonzero(gmap == u)[0]
        if len(m) == 1:
            assert (out[u].cpu().view(torch.uint16) == W[m[0]].view(torch.uint16)).all()
