"""bm_route_static (include/bm.h): the routing step for callers that may not allocate -- its scratch is a fixed 2 MiB
file-scope device array inside the library instead of a caller workspace.  Checked against the existing path (bm_route
with a workspace) on the same inputs: the kernels are the same, so the integer arrays must be bit-equal and the gate
weights inside the routing tests' tolerance (tests/gpu_helpers.py: assert_routing_equal), on two calls in a row with
different data -- the array is shared by every call and keeps the last call's contents.

This file is named to be collected LAST (the suite runs with pytest -x) and depends on no state of other tests: it runs
alone in a fresh process as well as after the whole suite."""
import numpy as np
import pytest
import torch

from bm_inputs import LayerConfig, make_layer

SHAPES = [
    # T, D, E, K, G, zipf_s
    (1, 256, 8, 2, 4, 0.0),            # one CTA, split router off (E <= 8)
    (16, 2048, 60, 4, 15, 1.0),        # split router with arrival counters + fused permutation
    (257, 2048, 60, 4, 15, 1.0),       # latency router + one-CTA permutation
    (1000, 512, 64, 6, 16, 1.5),       # tensor-core filter + refinement, cluster permutation
    (3001, 264, 13, 5, 7, 1.0),        # throughput router (all E dots), ragged D
    (8192, 128, 200, 16, 97, 0.5),     # the limit: T = BM_STATIC_ROUTE_MAX_T, K = BM_MAX_K, three-kernel permutation
]


def _route_both(bm, L):
    from gpu_helpers import routing_to_numpy, to_device
    T, D = L.x.shape
    E = L.W_router.shape[0]
    K, G = L.cfg.K, L.cfg.G
    d = to_device(L)
    ws = bm.alloc_workspace(T, D, 8, E, K, G, 0)
    r_ref, r_new = bm.Routing(T, K, G), bm.Routing(T, K, G)
    for r in (r_ref, r_new):
        for arr in (r.expert_ids, r.group_ids, r.row_token, r.row_slot, r.slot_row, r.n_slots, r.counts, r.offsets):
            arr.fill_(-7)
    bm.bm_route(d.x, d.W_router, d.router_bias, K, d.group_map, G, r_ref, ws)
    bm.bm_route_static(d.x, d.W_router, d.router_bias, K, d.group_map, G, r_new)
    torch.cuda.synchronize()
    assert bm.bm_device_status(ws) == 0
    assert bm.bm_route_static_status() == 0
    return routing_to_numpy(r_ref, T), routing_to_numpy(r_new, T)


@pytest.mark.gpu
@pytest.mark.parametrize("T,D,E,K,G,s", SHAPES)
def test_route_static_matches_bm_route_on_two_calls_in_a_row(T, D, E, K, G, s):
    import paper_2607_04164_b200 as bm
    from gpu_helpers import assert_routing_equal
    cfg = LayerConfig("t", T=T, D=D, F=8, E=E, K=K, G=G, zipf_s=s, gmap_kind="balanced")
    for seed in (0, 1):                                   # second call: other data through the same shared array
        L = make_layer(cfg, seed, weights=False)
        ref, new = _route_both(bm, L)
        assert_routing_equal(new, ref)
        assert (new.gate_w == ref.gate_w).all()           # the same kernels: the same bits


@pytest.mark.gpu
def test_route_static_allocates_nothing_and_clears_what_the_last_call_left():
    import paper_2607_04164_b200 as bm
    from gpu_helpers import assert_routing_equal, routing_to_numpy, to_device
    cfg = LayerConfig("t", T=300, D=256, F=8, E=24, K=3, G=6, zipf_s=1.0, gmap_kind="balanced")
    L = make_layer(cfg, 3, weights=False)
    ref, new = _route_both(bm, L)                          # warm-up: module load, symbol lookup, shared-memory grants
    assert_routing_equal(new, ref)
    d = to_device(L)
    r = bm.Routing(300, 3, 6)
    bad = d.group_map.clone()
    bad[:] = 9
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    # a call that raises a status bit (group map outside [0, G)), then a clean call: the bit must not survive, and the
    # device's free memory must not move (no allocation by the entry point; torch allocates nothing in between either)
    bm.bm_route_static(d.x, d.W_router, d.router_bias, 3, bad, 6, r)
    assert bm.bm_route_static_status() & bm.BM_DEV_BAD_GROUP_MAP
    bm.bm_route_static(d.x, d.W_router, d.router_bias, 3, d.group_map, 6, r)
    assert bm.bm_route_static_status() == 0
    assert_routing_equal(routing_to_numpy(r, 300), ref)
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    # an empty batch is BM_OK (and is the documented set-up call)
    e = bm.Routing(0, 3, 6)
    bm.bm_route_static(d.x[:0], d.W_router, d.router_bias, 3, d.group_map, 6, e)
    torch.cuda.synchronize()
    assert int(e.counts.abs().sum()) == 0 and int(e.offsets.abs().sum()) == 0


def test_route_static_rejects_sizes_beyond_its_scratch_on_the_host():
    """The limit is checked before any device work (no GPU needed): BM_ERR_LIMIT, with a message that says why."""
    import ctypes
    import paper_2607_04164_b200 as bm
    from paper_2607_04164_b200.binding import BmRouting
    assert bm.BM_STATIC_ROUTE_MAX_T == 8192 and bm.BM_STATIC_ROUTE_BYTES == 2 << 20
    r = BmRouting()
    rc = bm.lib().bm_route_static(None, bm.BM_STATIC_ROUTE_MAX_T + 1, 64, None, None, 8, 2, None, 4, ctypes.byref(r), None)
    assert rc == bm.BM_ERR_LIMIT
    assert "BM_ERR_LIMIT" in bm.status_string(rc) and "scratch" in bm.status_string(rc)
    assert bm.lib().bm_route_static(None, 16, 64, None, None, 8, 2, None, 4, None, None) == -1      # BM_ERR_NULL
    assert bm.lib().bm_route_static(None, 16, 64, None, None, 8, 9, None, 4, ctypes.byref(r), None) == -2   # K > E
