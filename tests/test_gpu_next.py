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


@pytest.mark.parametrize("T", [1, 3, 16])
def test_partial_brownout_single_token_decode(T):
    # small batches: split router with the cold mask (+ fused permutation over G + E sets), matrix-vector forward
    cfg = LayerConfig("pbd", T=T, D=2048, F=1408, E=60, K=4, G=15, zipf_s=1.0)
    rng = np.random.default_rng(7 + T)
    cold = (rng.random(cfg.E) < 0.5).astype(np.int32)
    _run_partial(cfg, 2, cold)                                  # BM_PATH_AUTO
    _run_partial(cfg, 2, cold, 4)                               # BM_PATH_GEMV forced


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
                            torch.zeros(400, dtype=torch.int32, device="cuda"), bm.Routing(8, 2, 600), ws)
    assert ei.value.code == -2
    with pytest.raises(ValueError):                             # the binding refuses routing arrays of another size
        bm.bm_route_partial(L.x.cuda(), L.W_router.cuda(), None, 2, L.group_map.cuda(), 4,
                            torch.zeros(8, dtype=torch.int32, device="cuda"), bm.Routing(8, 2, 4), ws)


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


# ---------------------------------------------------------------------------------------------------
# calibration forward (NEXT-2)
# ---------------------------------------------------------------------------------------------------
def _calib_case(seed, T, D, F, E, K, G):
    cfg = LayerConfig("cal", T=T, D=D, F=F, E=E, K=K, G=G, zipf_s=1.0)
    L = make_layer(cfg, seed, weights=False)
    Wo = _orig(seed, E, F, D)
    return cfg, L, Wo


@pytest.mark.parametrize("T,D,F,E,K,G", [(96, 256, 320, 12, 3, 4), (700, 512, 264, 60, 4, 15), (5, 64, 64, 3, 1, 2)])
def test_expert_histogram_and_outputs(T, D, F, E, K, G):
    import paper_2607_04164_b200 as bm
    cfg, L, Wo = _calib_case(2, T, D, F, E, K, G)
    bias = None if L.router_bias is None else L.router_bias.numpy()
    o = oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), bias, K, L.group_map.numpy(), G)
    # routing frequency: exact
    w = bm.bm_expert_histogram(torch.as_tensor(o.expert_ids).cuda(), E)
    assert (w.cpu().numpy() == oracle.expert_histogram(o.expert_ids, E)).all()
    # all-expert outputs: the hot path's tolerance
    Y = bm.bm_expert_outputs(L.x.cuda(), Wo[0].cuda(), Wo[1].cuda(), Wo[2].cuda())
    torch.cuda.synchronize()
    ref = oracle.expert_outputs(bf16_bits(L.x), bf16_bits(Wo[0]), bf16_bits(Wo[1]), bf16_bits(Wo[2]))
    assert tuple(Y.shape) == (T, E, D)                          # token-major
    assert_out_close(Y.permute(1, 0, 2).float().cpu().numpy().astype(np.float64).reshape(E * T, D), ref.reshape(E * T, D))


@pytest.mark.parametrize("E,T,D", [(12, 96, 256), (60, 300, 512), (128, 40, 64), (3, 5, 8)])
def test_cosine_gram_matches_oracle(E, T, D):
    import paper_2607_04164_b200 as bm
    rng = np.random.default_rng(E)
    base = rng.standard_normal((4, T, D))
    mix = rng.standard_normal((E, 4)) * np.array([2.0, 1.0, 0.5, 0.25])        # correlated experts
    Y = bf16_tensor(np.tensordot(mix, base, axes=1) + 0.3 * rng.standard_normal((E, T, D)))
    if E >= 3:
        Y[1] = Y[0]                                                        # identical pair -> cos 1
        Y[2] = -Y[0]                                                       # negated -> cos -1
    Ytm = Y.permute(1, 0, 2).contiguous().cuda()                # the C ABI takes the token-major layout [T, E, D]
    gram, cos = bm.bm_cosine_gram(Ytm)
    torch.cuda.synchronize()
    g_ref, c_ref = oracle.cosine_matrix(Y.double().numpy())
    gram, cos = gram.cpu().numpy().astype(np.float64), cos.cpu().numpy().astype(np.float64)
    # same bf16 inputs on both sides: only the fp32 accumulation order differs (n terms, products exact in fp32 pairs)
    scale = np.sqrt(np.outer(np.diag(g_ref), np.diag(g_ref)))
    assert (np.abs(gram - g_ref) <= 1e-5 * scale).all()
    assert (np.abs(cos - c_ref) <= 2e-5).all()
    assert np.allclose(gram, gram.T, rtol=0, atol=1e-6 * scale.max())
    if E >= 3:
        assert abs(cos[0, 1] - 1) <= 2e-5 and abs(cos[0, 2] + 1) <= 2e-5
    # determinism: partial tiles are summed in a fixed order
    gram2, _ = bm.bm_cosine_gram(Ytm)
    assert (gram2.cpu().numpy() == gram.astype(np.float32)).all()


@pytest.mark.parametrize("E,G,T,D", [(12, 4, 96, 256), (60, 15, 200, 512), (5, 8, 7, 16)])
def test_group_mse_matches_oracle(E, G, T, D):
    import paper_2607_04164_b200 as bm
    rng = np.random.default_rng(E + G)
    Y = bf16_tensor(rng.standard_normal((E, T, D)))
    U = bf16_tensor(rng.standard_normal((G, T, D)) * 0.5)
    gmap = rng.integers(0, G, size=E).astype(np.int32)
    w = rng.integers(0, 50, size=E).astype(np.int32)
    w[gmap == gmap[0]] = 0                                                # one never-selected group (A20)
    mse, tot = bm.bm_group_mse(Y.permute(1, 0, 2).contiguous().cuda(), U.permute(1, 0, 2).contiguous().cuda(),
                               torch.as_tensor(w).cuda(), torch.as_tensor(gmap).cuda())
    torch.cuda.synchronize()
    m_ref, t_ref, _ = oracle.group_mse(Y.double().numpy(), U.double().numpy(), w, gmap, G)
    mse, tot = mse.cpu().numpy().astype(np.float64), float(tot.cpu()[0])
    assert (np.abs(mse - m_ref) <= 1e-4 * m_ref + 1e-6).all()              # same bf16 inputs; fp32 target and squares
    assert abs(tot - t_ref) <= 1e-4 * t_ref + 1e-6
    for r in range(G):
        if not (gmap == r).any():
            assert mse[r] == 0.0


def test_calibration_pipeline_end_to_end_against_oracle():
    """Routing frequency -> all-expert outputs -> united experts by parameter average (NEXT-3) -> their outputs ->
    Eq. 5-6, every stage on the GPU, against the fp64 oracle fed with the same inputs only."""
    import paper_2607_04164_b200 as bm
    T, D, F, E, K, G = 256, 256, 192, 16, 2, 4
    cfg, L, Wo = _calib_case(3, T, D, F, E, K, G)
    gmap = L.group_map.numpy()
    bias = L.router_bias.numpy()
    xd, gm = L.x.cuda(), L.group_map.cuda()
    ws = bm.alloc_workspace(T, D, F, E, K, G, 0)
    r = bm.Routing(T, K, G)
    bm.bm_route(xd, L.W_router.cuda(), L.router_bias.cuda(), K, gm, G, r, ws)
    w = bm.bm_expert_histogram(r.view(T)["expert_ids"], E)
    Wd = [t.cuda() for t in Wo]
    Y = bm.bm_expert_outputs(xd, *Wd)
    Ud = [bm.bm_unite_weights(t, gm, G) for t in Wd]
    U = bm.bm_expert_outputs(xd, *Ud)
    mse, tot = bm.bm_group_mse(Y, U, w, gm)
    gram, cos = bm.bm_cosine_gram(Y)
    torch.cuda.synchronize()
    # oracle chain (fp64; the united weights are rounded to bf16 as the GPU stores them -- A18)
    o = oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), bias, K, gmap, G)
    w_ref = oracle.expert_histogram(o.expert_ids, E)
    assert (w.cpu().numpy() == w_ref).all()
    Y_ref = oracle.expert_outputs(bf16_bits(L.x), *[bf16_bits(t) for t in Wo])
    Uw = [bf16_tensor(oracle.unite_weights(bf16_bits(t), gmap, G)) for t in Wo]
    U_ref = oracle.expert_outputs(bf16_bits(L.x), *[bf16_bits(t) for t in Uw])
    m_ref, t_ref, _ = oracle.group_mse(Y_ref, U_ref, w_ref, gmap, G)
    _, c_ref = oracle.cosine_matrix(Y_ref)
    # bf16 outputs on the GPU side: each y carries 2^-9 relative rounding noise -> 2e-2 relative on the MSE, 5e-3 on cos
    mse = mse.cpu().numpy().astype(np.float64)
    assert (np.abs(mse - m_ref) <= 2e-2 * m_ref + 1e-7).all(), (mse, m_ref)
    assert abs(float(tot.cpu()[0]) - t_ref) <= 2e-2 * t_ref + 1e-7
    assert np.abs(cos.cpu().numpy() - c_ref).max() <= 5e-3


# ---------------------------------------------------------------------------------------------------
# tensor parallelism over F (NEXT-4): the ranks emulated one after the other on one GPU
# ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("T,world", [(1, 2), (48, 2), (700, 4), (3000, 2)])     # T = 1: matrix-vector path, fp32 partial
def test_tensor_parallel_partials_sum_to_the_layer(T, world):
    import paper_2607_04164_b200 as bm
    from paper_2607_04164_b200.tp import shard_f
    cfg = LayerConfig("tp", T=T, D=512, F=1408, E=16, K=4, G=4, S=1, zipf_s=1.0)
    L = make_layer(cfg, 4)
    bias = L.router_bias.numpy()
    o = oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), bias, cfg.K, L.group_map.numpy(), cfg.G)
    ref = oracle.moe_forward(bf16_bits(L.x), o, bf16_bits(L.W1), bf16_bits(L.W3), bf16_bits(L.W2), cfg.S)
    xd = L.x.cuda()
    r = bm.Routing(T, cfg.K, cfg.G)
    total = torch.zeros((T, cfg.D), dtype=torch.float32, device="cuda")
    for rank in range(world):
        W1r, W3r, W2r = [t.cuda() for t in shard_f(L.W1, L.W3, L.W2, rank, world)]
        ws = bm.alloc_workspace(T, cfg.D, W1r.shape[1], cfg.E, cfg.K, cfg.G, cfg.S)
        bm.bm_route(xd, L.W_router.cuda(), L.router_bias.cuda(), cfg.K, L.group_map.cuda(), cfg.G, r, ws)
        part = torch.full((T, cfg.D), float("nan"), dtype=torch.float32, device="cuda")
        bm.bm_moe_forward_f32(xd, r, W1r, W3r, W2r, part, ws, S=cfg.S)
        total += part                                   # stands in for the NCCL all-reduce
        assert bm.bm_device_status(ws) == 0
    out = bm.bm_round_bf16(total)
    torch.cuda.synchronize()
    assert_routing_equal(routing_to_numpy(r, T), o)
    assert_out_close(out.float().cpu().numpy().astype(np.float64), ref)
    # one rank = the plain layer: tp_moe_forward without a process group is bm_moe_forward
    ws = bm.alloc_workspace(T, cfg.D, cfg.F, cfg.E, cfg.K, cfg.G, cfg.S)
    W = [t.cuda() for t in (L.W1, L.W3, L.W2)]
    a = torch.empty((T, cfg.D), dtype=torch.bfloat16, device="cuda")
    b = torch.empty_like(a)
    bm.tp_moe_forward(xd, r, *W, a, ws, S=cfg.S)
    bm.bm_moe_forward(xd, r, *W, b, ws, S=cfg.S)
    torch.cuda.synchronize()
    assert_out_close(a.float().cpu().numpy().astype(np.float64), ref)
    _, det = bm.bm_forward_info(T, cfg.K, cfg.G, cfg.S, cfg.D, cfg.F)
    if det:                                             # matrix-vector path: fixed summation order -> the same bits
        assert (a == b).all()
    else:                                               # fused combine, K + S = 5 sources: fp32 adds arrive in any order
        assert (a.float() - b.float()).abs().max() <= 2.0 ** -7 * b.float().abs().max()


def test_tp_moe_forward_under_a_real_nccl_process_group():
    """The collective call path of tensor parallelism (tp.py: bm_moe_forward_f32 -> dist.all_reduce -> bm_round_bf16)
    executed on hardware: a one-rank NCCL process group (one GPU per box here).  The sum over one rank is the rank's
    partial, so the result must equal the plain layer within the fp32-order tolerance; what this covers is that NCCL
    accepts the fp32 partial buffer on the library's stream and that the rounding pass follows it."""
    import os
    import torch.distributed as dist
    import paper_2607_04164_b200 as bm
    if dist.is_initialized():
        pytest.skip("a process group already exists in this process")
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", str(29600 + os.getpid() % 300))
    dist.init_process_group("nccl", rank=0, world_size=1, device_id=torch.device("cuda", 0))
    try:
        for T in (48, 700):
            cfg = LayerConfig("tpn", T=T, D=512, F=704, E=16, K=2, G=4, S=0, zipf_s=1.0)
            L = make_layer(cfg, 5)
            o = oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), L.router_bias.numpy(), cfg.K, L.group_map.numpy(), cfg.G)
            ref = oracle.moe_forward(bf16_bits(L.x), o, bf16_bits(L.W1), bf16_bits(L.W3), bf16_bits(L.W2), cfg.S)
            xd = L.x.cuda()
            r = bm.Routing(T, cfg.K, cfg.G)
            ws = bm.alloc_workspace(T, cfg.D, cfg.F, cfg.E, cfg.K, cfg.G, cfg.S)
            bm.bm_route(xd, L.W_router.cuda(), L.router_bias.cuda(), cfg.K, L.group_map.cuda(), cfg.G, r, ws)
            out = torch.full((T, cfg.D), float("nan"), dtype=torch.bfloat16, device="cuda")
            bm.tp_moe_forward(xd, r, L.W1.cuda(), L.W3.cuda(), L.W2.cuda(), out, ws, S=cfg.S)
            torch.cuda.synchronize()
            assert dist.get_world_size() == 1 and dist.get_backend() == "nccl"
            assert_out_close(out.float().cpu().numpy().astype(np.float64), ref)
    finally:
        dist.destroy_process_group()


def test_bench_device_layer_tensor_parallel_step_runs_and_matches_oracle():
    """bench.py's DeviceLayer with tp=(rank, world) (the `--parallel tp` arm): round 1's version raised AttributeError on
    the first step.  One rank of one: the F shard is the whole F, so the step must reproduce the layer."""
    import sys, os
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import bench
    from bm_inputs import CONFIGS
    import paper_2607_04164_b200 as bm
    cfg = CONFIGS["tiny"]
    layer = bench.DeviceLayer(cfg, seed=0, x_seed=0, keep_host_weights=True, tp=(0, 1))
    layer.step()
    torch.cuda.synchronize()
    L = layer.host
    o = oracle.route(bf16_bits(L.x), bf16_bits(L.W_router), None, cfg.K, L.group_map.numpy(), cfg.G)
    ref = oracle.moe_forward(bf16_bits(L.x), o, bf16_bits(L.W1), bf16_bits(L.W3), bf16_bits(L.W2), cfg.S)
    assert_out_close(layer.out.float().cpu().numpy().astype(np.float64), ref)
    assert bm.bm_device_status(layer.ws) == 0
